"""Coordinate Descent by best-response look-ups (csrc/factors.cu; many starts per problem on library-built tables of two
and three mesh levels) against the oracle's plain CD on the K x K tables: cost, strategy and sweep count, bit for bit."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def _oracle_cd(w, init, cap):
    from concurrent.futures import ThreadPoolExecutor
    import os
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    S = init.shape[1]
    n = min(max(1, len(os.sched_getaffinity(0))), S)
    bounds = np.linspace(0, S, n + 1).astype(int)
    with ThreadPoolExecutor(n) as ex:
        parts = list(ex.map(lambda k: ref.coord_descent(T, np.ascontiguousarray(init[:, bounds[k]:bounds[k + 1]]), cap), range(n)))
    return tuple(np.concatenate([p[i] for p in parts], axis=1) for i in range(3)), T


@pytest.mark.parametrize("k", [2, 3, 5])
def test_configs_without_tables(adl, k):
    """autoddl_coord_descent(d_T = NULL) with 64 / 256 / 1024 starts: no K x K table is built at all"""
    w = cf.CONFIGS[k]()
    init = w.cd_init()
    got = adl.coord_descent(None, torch.from_numpy(init).cuda(), w.mesh, w.max_sweeps, net=w.net, d_layers=adl.layers_to_device(w.layers))
    torch.cuda.synchronize()
    want, _ = _oracle_cd(w, init, w.max_sweeps)
    for name, g, x in zip(("cd_cost", "cd_strategy", "cd_sweeps"), got, want):
        assert np.array_equal(g.cpu().numpy(), x), name


def test_random_workloads_both_routes(adl):
    rng = np.random.default_rng(31)
    for case in range(40):
        D = int(rng.choice([2, 2, 3]))
        sizes = tuple(int(x) for x in rng.choice([1, 2, 3, 4, 8], D))
        links = tuple(int(rng.integers(0, 2)) | (int(rng.choice([0, 0, 0x07, 0x0b, 0x15])) << 8) for _ in range(D))
        Bp = int(rng.choice([1, 2, 5])) if D == 3 else int(rng.choice([1, 3, 17, 300]))
        L = int(rng.choice([1, 2, 3, 9, 31, 32, 33, 64, 65, 97])) if D == 2 else int(rng.choice([1, 2, 5, 33]))
        S = int(rng.choice([32, 33, 64, 100]))
        if Bp * L * S > 200_000:
            Bp = max(1, 200_000 // (L * S))
        layers = cf.config4_batched(Bp=Bp, L=L, seed=int(rng.integers(0, 1000))).layers.copy()
        if rng.random() < 0.5:
            for p in range(Bp):
                for l in range(L):
                    if rng.random() < 0.3:
                        layers[p, l] = cf.attn(int(layers[p, l]["M"]), int(layers[p, l]["N"]), int(rng.integers(1, 4000)), 2,
                                               int(rng.integers(1, 40)), int(rng.integers(1, 40)))
        if rng.random() < 0.3:
            layers["max_split_rows"] = rng.integers(1, 40, size=layers.shape)
            layers["max_split_cols"] = rng.integers(1, 40, size=layers.shape)
        cap = int(rng.choice([0, 0, 10**7 * L, 10**9 * L]))
        w = cf.Workload("lookup-%d" % case, layers, cf.Mesh(sizes, links), cf.Net(cf.ALPHA_PS, (3, 40), cap, micro_batches=int(rng.choice([0, 1, 3]))),
                        S=S, seed=int(rng.integers(0, 1000)))
        init = w.cd_init()
        cap_sw = int(rng.choice([1, 2, 3, 64]))
        dl = adl.layers_to_device(w.layers)
        dinit = torch.from_numpy(init).cuda()
        a = adl.coord_descent(None, dinit, w.mesh, cap_sw, net=w.net, d_layers=dl)                 # look-ups, no tables
        o = adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=cap_sw)                           # tables + DP, then look-ups
        T, _, _ = adl.build_tables(dl, w.mesh, w.net)
        b = adl.coord_descent(T, dinit, w.mesh, cap_sw)                                            # gathers on the tables
        torch.cuda.synchronize()
        (occ, ocs, osw), oT = _oracle_cd(w, init, cap_sw)
        info = dict(case=case, sizes=sizes, links=links, Bp=Bp, L=L, S=S, cap=cap, cap_sw=cap_sw)
        for name, g, x in (("lookup.cost", a[0], occ), ("lookup.strategy", a[1], ocs), ("lookup.sweeps", a[2], osw),
                           ("search.cost", o["cd_cost"], occ), ("search.strategy", o["cd_strategy"], ocs), ("search.sweeps", o["cd_sweeps"], osw),
                           ("gather.cost", b[0], occ), ("gather.strategy", b[1], ocs), ("gather.sweeps", b[2], osw), ("T", o["T"], oT)):
            assert np.array_equal(g.cpu().numpy(), x), (name, info)


# ---- the same look-up scheme on K x K tables (K <= 64): caller-supplied tables, random ones with many ties -----------------
def _mesh_with_k(K):
    if K == 36:
        return cf.Mesh((4, 4), (cf.INTER, cf.INTRA))
    if K == 16:
        return cf.Mesh((2, 2, 2, 2), tuple(l | (0x03 << 8) for l in (cf.INTER, cf.INTER, cf.INTRA, cf.INTRA)))
    if K == 64:
        return cf.Mesh((2, 2, 2, 2), (cf.INTER | (0x0f << 8), cf.INTER | (0x0f << 8), cf.INTRA | (0x03 << 8), cf.INTRA | (0x03 << 8)))
    n = 6 if K == 28 else 8
    return cf.Mesh((2,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))


@pytest.mark.parametrize("K,L,Bp,S,hi,cap", [(36, 1, 2, 32, 5, 64), (36, 2, 3, 33, 1 << 40, 64), (16, 31, 2, 40, 3, 64), (28, 32, 1, 64, 4, 64),
                                             (45, 33, 2, 32, 6, 64), (45, 97, 1, 50, 1 << 45, 3), (64, 64, 2, 32, 4, 64),
                                             (64, 130, 1, 100, 9, 64), (36, 65, 5, 64, 3, 1)])
def test_lookup_cd_on_tables(adl, K, L, Bp, S, hi, cap):
    """trajectory, sweep count and result of the plain algorithm (R10: smallest-index argmin, Gauss-Seidel order, dirty
    layers) on random tables -- cells in [0, hi) for a small hi tie nearly every update --, also with a sweep cap"""
    mesh = _mesh_with_k(K)
    assert adl.num_signatures(mesh) == K
    rng = np.random.default_rng(K * 977 + L)
    T = rng.integers(0, hi, size=(Bp, L, K, K), dtype=np.int64)
    init = rng.integers(0, K, size=(Bp, S, L), dtype=np.int32)
    want = ref.coord_descent(T, init, cap)
    d_T, d_init = torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda()
    work = torch.empty(adl.workspace_bytes(Bp, L, S, mesh), dtype=torch.uint8, device="cuda")
    work.fill_(0xC3)
    got = adl.coord_descent(d_T, d_init, mesh, cap, work=work)          # best responses from the tiles + look-up sweeps
    plain = adl.coord_descent(d_T, d_init, mesh, cap)                   # no workspace: the gather kernel
    torch.cuda.synchronize()
    for name, g, q, x in zip(("cd_cost", "cd_strategy", "cd_sweeps"), got, plain, want):
        assert np.array_equal(g.cpu().numpy(), x), name
        assert np.array_equal(q.cpu().numpy(), x), name + " (gather kernel)"
