"""Parity of the CUDA path (through the C-ABI) against the CPU oracle: bit-exact, element by element.

Run with `pytest -m gpu` on a B200.  All costs are int64, all indices int32/uint8: the bar is equality.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf

pytestmark = pytest.mark.gpu

PEN = 1 << 50


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def _oracle_all(w, init):
    T, node, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    dc, ds = ref.chain_dp(T)
    cc, cs, sw = ref.coord_descent(T, init, w.max_sweeps)
    return T, node, mask, dc, ds, cc, cs, sw


def _gpu_all(adl, w, init):
    d_layers = adl.layers_to_device(w.layers)
    T, node, mask = adl.build_tables(d_layers, w.mesh, w.net)
    dc, ds = adl.chain_dp(T, w.mesh)
    cc, cs, sw = adl.coord_descent(T, torch.from_numpy(init).cuda(), w.mesh, w.max_sweeps)
    torch.cuda.synchronize()
    return [x.cpu().numpy() for x in (T, node, mask, dc, ds, cc, cs, sw)]


def _ncores():
    import os
    return max(1, len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))


def _oracle_slices(w, init, per=64):
    """the oracle's whole path on contiguous slices of the problems, fanned over the host cores (ctypes releases the GIL;
    the oracle itself stays single-threaded): yields (a, b, (T, node, mask, dp_cost, dp_strategy, cd_cost, cd_strategy,
    cd_sweeps)) slice by slice so that host memory stays bounded"""
    from concurrent.futures import ThreadPoolExecutor
    mesh, net = ref.mesh_of(w), ref.net_of(w)
    bounds = list(range(0, w.Bp, per)) + [w.Bp]

    def work(k):
        a, b = bounds[k], bounds[k + 1]
        T, node, mask = ref.build_tables(np.ascontiguousarray(w.layers[a:b]), mesh, net)
        dc, ds = ref.chain_dp(T)
        cc, cs, sw = ref.coord_descent(T, np.ascontiguousarray(init[a:b]), w.max_sweeps)
        return a, b, (T, node, mask, dc, ds, cc, cs, sw)

    ref.lib()
    n = _ncores()
    with ThreadPoolExecutor(n) as ex:
        for k0 in range(0, len(bounds) - 1, n):                     # one wave of slices at a time
            for r in ex.map(work, range(k0, min(k0 + n, len(bounds) - 1))):
                yield r


def _oracle_cd_all_starts(T, init, max_sweeps):
    """oracle CD of ONE problem over all its starts, the starts fanned over the host cores"""
    from concurrent.futures import ThreadPoolExecutor
    S = init.shape[1]
    n = min(_ncores(), S)
    bounds = np.linspace(0, S, n + 1).astype(int)
    with ThreadPoolExecutor(n) as ex:
        parts = list(ex.map(lambda k: ref.coord_descent(T, np.ascontiguousarray(init[:, bounds[k]:bounds[k + 1]]), max_sweeps), range(n)))
    return tuple(np.concatenate([p[i] for p in parts], axis=1) for i in range(3))


def _assert_same(got, want, names=("T", "node", "mask", "dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps")):
    for g, x, n in zip(got, want, names):
        assert g.shape == x.shape and g.dtype == x.dtype, n
        if not np.array_equal(g, x):
            bad = np.argwhere(g != x)
            raise AssertionError(f"{n}: {len(bad)} mismatches, first at {bad[0].tolist()}: got {g[tuple(bad[0])]} want {x[tuple(bad[0])]}")


@pytest.mark.parametrize("k", [1, 2, 3])
def test_configs_small_full(adl, k):
    w = cf.CONFIGS[k]()
    init = w.cd_init()
    _assert_same(_gpu_all(adl, w, init), _oracle_all(w, init))


def test_config5_k216(adl):
    """BASELINE.json configs[4] in full: tables, node, mask, DP and ALL 1024 CD starts against the oracle"""
    w = cf.config5_transformer96()
    init = w.cd_init()
    T, node, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    dc, ds = ref.chain_dp(T)
    _assert_same(_gpu_all(adl, w, init), (T, node, mask, dc, ds) + _oracle_cd_all_starts(T, init, w.max_sweeps))


def test_config5_all_starts_properties(adl):
    """all 1024 starts at full size: DP <= CD, cost == Cost(strategy), fixed point reached"""
    w = cf.config5_transformer96()
    init = torch.from_numpy(w.cd_init()).cuda()
    T, _, _ = adl.build_tables(adl.layers_to_device(w.layers), w.mesh, w.net)
    dc, ds = adl.chain_dp(T, w.mesh)
    cc, cs, sw = adl.coord_descent(T, init, w.mesh, w.max_sweeps)
    assert (cc >= dc[:, None]).all()
    assert int(dc[0]) == 294_284_438_784         # tests/golden/survey_crosscheck.txt config5_dp
    _check_costs(T, cs.reshape(1, -1, w.L), cc.reshape(1, -1))
    _check_costs(T, ds.reshape(1, 1, w.L), dc.reshape(1, 1))


def _check_costs(T, strat, cost):
    """Cost(s) = sum_l T[l][s_{l-1}][s_l] recomputed with torch gathers for [Bp, S, L] strategies"""
    Bp, S, L = strat.shape
    K = T.shape[-1]
    s = strat.long()
    prev = torch.cat([torch.zeros_like(s[..., :1]), s[..., :-1]], dim=-1)
    l = torch.arange(L, device=T.device).view(1, 1, L)
    p = torch.arange(Bp, device=T.device).view(Bp, 1, 1)
    flat = ((p * L + l) * K + prev) * K + s
    tot = T.reshape(-1)[flat.reshape(-1)].reshape(Bp, S, L).sum(-1)
    assert torch.equal(tot, cost)


def test_config4_reduced_full_compare(adl):
    w = cf.config4_batched(Bp=37, L=64)          # ragged: 37 problems
    init = w.cd_init()
    _assert_same(_gpu_all(adl, w, init), _oracle_all(w, init))


@pytest.mark.parametrize("L", [1, 2, 3, 7])
def test_config4_short_chains(adl, L):
    w = cf.config4_batched(Bp=5, L=L, seed=3)
    init = w.cd_init()
    _assert_same(_gpu_all(adl, w, init), _oracle_all(w, init))


def test_config4_full_size(adl):
    """BASELINE.json configs[3] at full size (4096 x 64, the launch configuration bench.py times): EVERY problem's tables,
    node costs, masks, DP optimum + strategy and CD cost + strategy + sweep count against the oracle, through the three
    separate kernels AND through the one-call path (fused kernel + CD from the compact factors)."""
    w = cf.config4_batched()
    init = w.cd_init()
    d_layers = adl.layers_to_device(w.layers)
    T, node, mask = adl.build_tables(d_layers, w.mesh, w.net)
    dc, ds = adl.chain_dp(T, w.mesh)
    cc, cs, sw = adl.coord_descent(T, torch.from_numpy(init).cuda(), w.mesh, w.max_sweeps)
    one = adl.search(d_layers, w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps, want_node_mask=True)
    dc2, ds2 = adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers)       # fused, no table written
    torch.cuda.synchronize()
    sep = (T, node, mask, dc, ds, cc, cs, sw)
    fused = tuple(one[k] for k in ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
    seen = 0
    for a, b, want in _oracle_slices(w, init):
        _assert_same([x[a:b].cpu().numpy() for x in sep], want)
        _assert_same([x[a:b].cpu().numpy() for x in fused], want)
        _assert_same([dc2[a:b].cpu().numpy(), ds2[a:b].cpu().numpy()], want[3:5], names=("dp_cost", "dp_strategy"))
        seen += b - a
    assert seen == 4096
    # properties at any size
    _check_costs(T, ds.view(4096, 1, 64), dc.view(4096, 1))
    _check_costs(T, cs, cc)
    assert (cc >= dc[:, None]).all()
    assert (dc < PEN).all()                      # no cap in config 4: always feasible
    assert (sw >= 1).all() and (sw <= w.max_sweeps).all()


def _random_tables(rng, Bp, L, K, hi):
    T = rng.integers(0, hi, size=(Bp, L, K, K)).astype(np.int64)
    T[rng.random(T.shape) < 0.08] += PEN
    return T


@pytest.mark.parametrize("K,L,Bp,hi", [(6, 1, 3, 10), (6, 9, 11, 4), (36, 2, 5, 3), (36, 65, 150, 7), (36, 33, 301, 10**9),
                                        (216, 2, 2, 5), (216, 11, 3, 10**10), (216, 90, 1, 3)])
def test_dp_cd_random_tables(adl, K, L, Bp, hi):
    """generic tables with heavy ties and penalties; L*K > 16384 exercises back-pointers in the workspace"""
    rng = np.random.default_rng(K * 1000 + L)
    T = _random_tables(rng, Bp, L, K, hi)
    S = 3
    init = rng.integers(0, K, size=(Bp, S, L)).astype(np.int32)
    mesh = cf.Mesh(tuple([2] * {6: 1, 36: 2, 216: 3}[K]), tuple([0] * {6: 1, 36: 2, 216: 3}[K]))
    dT = torch.from_numpy(T).cuda()
    dc, ds = adl.chain_dp(dT, mesh)
    cc, cs, sw = adl.coord_descent(dT, torch.from_numpy(init).cuda(), mesh, 64)
    odc, ods = ref.chain_dp(T)
    occ, ocs, osw = ref.coord_descent(T, init, 64)
    _assert_same([x.cpu().numpy() for x in (dc, ds, cc, cs, sw)], (odc, ods, occ, ocs, osw),
                 names=("dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps"))


def test_cd_sweep_cap(adl):
    rng = np.random.default_rng(5)
    T = _random_tables(rng, 4, 40, 36, 1000)
    init = rng.integers(0, 36, size=(4, 6, 40)).astype(np.int32)
    mesh = cf.Mesh((2, 2), (0, 0))
    for cap in (1, 2, 3):
        cc, cs, sw = adl.coord_descent(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), mesh, cap)
        occ, ocs, osw = ref.coord_descent(T, init, cap)
        _assert_same([x.cpu().numpy() for x in (cc, cs, sw)], (occ, ocs, osw), names=("cd_cost", "cd_strategy", "cd_sweeps"))


def test_fused_build_paths_and_search_host(adl):
    """d_T == NULL (tables built into the workspace) and the host-pointer end-to-end call"""
    w = cf.config4_batched(Bp=9, L=17, seed=2)
    init = w.cd_init()
    want = _oracle_all(w, init)
    d_layers = adl.layers_to_device(w.layers)
    dc, ds = adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers)
    cc, cs, sw = adl.coord_descent(None, torch.from_numpy(init).cuda(), w.mesh, w.max_sweeps, net=w.net, d_layers=d_layers)
    _assert_same([x.cpu().numpy() for x in (dc, ds, cc, cs, sw)], want[3:],
                 names=("dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
    out = adl.search_host(w, init, work)
    _assert_same([out["opt_cost"], out["strategy"], out["cd_cost"], out["cd_strategy"], out["cd_sweeps"]], want[3:],
                 names=("dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
    # pinned (device-mapped) host inputs are read by the kernels straight over PCIe, pageable ones are copied: same results
    for Bp2 in (9, 700):
        w2 = cf.config4_batched(Bp=Bp2, L=17, seed=2)
        init2 = w2.cd_init()
        want2 = _oracle_all(cf.Workload(w2.name, w2.layers[:9], w2.mesh, w2.net, S=w2.S, seed=2), init2[:9])
        h_layers = torch.from_numpy(np.ascontiguousarray(w2.layers).view(np.uint8).reshape(Bp2, 17, 64).copy()).pin_memory()
        h_init = torch.from_numpy(init2.copy()).pin_memory()
        w_pin = cf.Workload(w2.name, h_layers.numpy().view(cf.LAYER_DTYPE).reshape(Bp2, 17), w2.mesh, w2.net, S=w2.S, seed=2)
        work2 = torch.empty(adl.workspace_bytes(Bp2, 17, w2.S, w2.mesh), dtype=torch.uint8, device="cuda")
        pinned = adl.search_host(w_pin, h_init.numpy(), work2)
        pinned = {k: v.copy() for k, v in pinned.items()}
        pageable = adl.search_host(w2, init2, work2)
        for k in pinned:
            assert np.array_equal(pinned[k], pageable[k]), k
        _assert_same([pinned[k][:9] for k in ("opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")], want2[3:],
                     names=("dp_cost", "dp_strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
    w5 = cf.config5_transformer96()               # back-pointers in the workspace, no CD
    work = torch.empty(adl.workspace_bytes(w5.Bp, w5.L, 0, w5.mesh), dtype=torch.uint8, device="cuda")
    out = adl.search_host(w5, None, work)
    assert int(out["opt_cost"][0]) == 294_284_438_784


def _search_all(adl, w, init, **kw):
    """the one-call path (autoddl_search): on 2-level meshes tables and chain DP run as one fused kernel"""
    o = adl.search(adl.layers_to_device(w.layers), w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=w.max_sweeps,
                   want_node_mask=True, **kw)
    torch.cuda.synchronize()
    return [o[k].cpu().numpy() for k in ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")]


@pytest.mark.parametrize("k", [1, 2, 3, 5])
def test_search_one_call_configs(adl, k):
    """configs 1-3 (K = 36: fused build + DP kernel, GEMM and ATTN edges) and 5 (K = 216: three kernels)"""
    w = cf.CONFIGS[k]()
    init = w.cd_init()
    if k == 5:                                                   # all 1024 starts
        T, node, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
        dc, ds = ref.chain_dp(T)
        want = (T, node, mask, dc, ds) + _oracle_cd_all_starts(T, init, w.max_sweeps)
    else:
        want = _oracle_all(w, init)
    _assert_same(_search_all(adl, w, init), want)


def _fused_dp(adl, w):
    """chain DP through the fused build + DP kernel whatever the number of chains: with a workspace too small for the
    tables autoddl_chain_dp(d_T = NULL) has to run the tables through shared memory only"""
    d_layers = adl.layers_to_device(w.layers)
    small = torch.empty(148 * 28 * w.L * 36 + 4096, dtype=torch.uint8, device="cuda")
    assert small.numel() < w.Bp * w.L * 36 * 36 * 8
    dc, ds = adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers, work=small)
    torch.cuda.synchronize()
    return dc.cpu().numpy(), ds.cpu().numpy()


@pytest.mark.parametrize("Bp,L", [(1, 1), (3, 1), (5, 2), (7, 3), (5, 7), (1500, 3), (900, 5), (33, 64), (2, 300), (741, 86), (296, 500)])
def test_search_fused_shapes(adl, Bp, L):
    """fused kernel over ragged groups (L not a multiple of the group size), more chains than resident CTAs,
    single-layer chains, and a chain longer than any shared-memory back-pointer table would allow"""
    w = cf.config4_batched(Bp=Bp, L=L, seed=5)
    init = w.cd_init()
    nsamp = min(Bp, 40)
    idx = np.unique(np.concatenate([np.arange(min(Bp, 6)), np.random.default_rng(1).integers(0, Bp, nsamp), [Bp - 1]]))
    got = _search_all(adl, w, init)                              # fused for Bp >= 296, three kernels below
    ws = cf.Workload(w.name, np.ascontiguousarray(w.layers[idx]), w.mesh, w.net, S=w.S, seed=w.seed)
    want = _oracle_all(ws, np.ascontiguousarray(init[idx]))
    _assert_same([g[idx] for g in got], want)
    # all chains: fused DP (forced) == one-call path == the separate DP kernel on the same tables
    d_layers = adl.layers_to_device(w.layers)
    T, _, _ = adl.build_tables(d_layers, w.mesh, w.net)
    dc, ds = adl.chain_dp(T, w.mesh)
    assert np.array_equal(got[3], dc.cpu().numpy()) and np.array_equal(got[4], ds.cpu().numpy())
    assert np.array_equal(got[0], T.cpu().numpy())
    if Bp * L * 36 * 36 * 8 > 148 * 28 * L * 36 + 4096:
        fc, fs = _fused_dp(adl, w)
        assert np.array_equal(fc, dc.cpu().numpy()) and np.array_equal(fs, ds.cpu().numpy())


def test_search_mixed_kinds_and_unit_level(adl):
    """fused kernel with ATTN edges, ragged dims, split limits, a memory cap and a mesh level of size 1"""
    rng = np.random.default_rng(11)
    for sizes, links in [((3, 5), (1, 0)), ((1, 7), (1, 0)), ((8, 1), (1, 0))]:
        Bp, L = 310, 9
        layers = np.zeros((Bp, L), dtype=cf.LAYER_DTYPE)
        for p in range(Bp):
            for l in range(L):
                M, Kd, N = (int(x) for x in rng.integers(1, 3000, 3))
                if (l + p) % 3 == 1:
                    layers[p, l] = cf.attn(M, N, int(rng.integers(1, 3000)), 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)))
                else:
                    layers[p, l] = cf.gemm(M, Kd, N, 2, 4, 18, in_rows=int(rng.integers(1, 5000)), in_cols=int(rng.integers(1, 5000)),
                                           max_rows=int(rng.integers(1, 64)), max_cols=int(rng.integers(1, 64)))
        w = cf.Workload("mixed", layers, cf.Mesh(sizes, links), cf.Net(cf.ALPHA_PS, (3, 40), 150_000 * L), S=2, seed=2)
        init = w.cd_init()
        got = _search_all(adl, w, init)                          # 310 chains: the fused kernel
        idx = np.arange(0, Bp, 9)
        ws = cf.Workload(w.name, np.ascontiguousarray(w.layers[idx]), w.mesh, w.net, S=w.S, seed=w.seed)
        _assert_same([g[idx] for g in got], _oracle_all(ws, np.ascontiguousarray(init[idx])))
        fc, fs = _fused_dp(adl, w)
        assert np.array_equal(fc, got[3]) and np.array_equal(fs, got[4])
        d_layers = adl.layers_to_device(w.layers)
        T, _, _ = adl.build_tables(d_layers, w.mesh, w.net)
        dc, ds = adl.chain_dp(T, w.mesh)
        assert np.array_equal(got[0], T.cpu().numpy()) and np.array_equal(got[3], dc.cpu().numpy()) and np.array_equal(got[4], ds.cpu().numpy())


def test_search_without_tables_and_full_size(adl):
    """config 4 at full size through the fused kernel (the launch configuration bench.py times): sweep caps and the
    no-table route agree with the separate kernels on every chain (which test_config4_full_size holds to the oracle)"""
    w = cf.config4_batched()
    d_layers = adl.layers_to_device(w.layers)
    o = adl.search(d_layers, w.mesh, w.net, want_tables=True)
    dc2, ds2 = adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers)       # fused, no table written
    T, _, _ = adl.build_tables(d_layers, w.mesh, w.net)
    dc, ds = adl.chain_dp(T, w.mesh)
    torch.cuda.synchronize()
    assert torch.equal(o["T"], T) and torch.equal(o["opt_cost"], dc) and torch.equal(o["strategy"], ds)
    assert torch.equal(dc2, dc) and torch.equal(ds2, ds)
    # one call with CD: the first sweep runs inside the fused kernel, the CD kernel resumes at sweep 2
    init = torch.from_numpy(w.cd_init()).cuda()
    o3 = adl.search(d_layers, w.mesh, w.net, init=init, max_sweeps=w.max_sweeps)
    cc, cs, sw = adl.coord_descent(T, init, w.mesh, w.max_sweeps)
    torch.cuda.synchronize()
    assert torch.equal(o3["cd_cost"], cc) and torch.equal(o3["cd_strategy"], cs) and torch.equal(o3["cd_sweeps"], sw)
    assert torch.equal(o3["opt_cost"], dc) and torch.equal(o3["T"], T)
    for cap in (1, 2, 3):                                   # sweep cap below, at and above the resume point
        o4 = adl.search(d_layers, w.mesh, w.net, init=init, max_sweeps=cap)
        c4 = adl.coord_descent(T, init, w.mesh, cap)
        torch.cuda.synchronize()
        assert torch.equal(o4["cd_cost"], c4[0]) and torch.equal(o4["cd_strategy"], c4[1]) and torch.equal(o4["cd_sweeps"], c4[2])
    # (the oracle comparison of every chain of this configuration is test_config4_full_size)


@pytest.mark.parametrize("Bp,L,hi", [(1, 2, 5), (3, 7, 3), (2, 33, 10**9), (5, 100, 1000), (1, 864, 50), (1, 865, 50), (19, 5, 7)])
def test_dp_k216_cluster_and_fallback(adl, Bp, L, hi):
    """K = 216 chain DP: one 8-CTA cluster per chain (row blocks per CTA, partial minima exchanged over distributed
    shared memory) for few chains and L <= 864, the one-CTA kernel otherwise; many exact ties (small hi)"""
    rng = np.random.default_rng(Bp * 1000 + L)
    T = rng.integers(0, hi, size=(Bp, L, 216, 216)).astype(np.int64)
    T[:, 0] = T[:, 0, :1]
    mesh = cf.Mesh((2, 2, 2), (0, 0, 0))
    work = torch.empty(Bp * L * 216 + 4096, dtype=torch.uint8, device="cuda")
    dc, ds = adl.chain_dp(torch.from_numpy(T).cuda(), mesh, work=work)
    odc, ods = ref.chain_dp(T)
    _assert_same([dc.cpu().numpy(), ds.cpu().numpy()], (odc, ods), names=("dp_cost", "dp_strategy"))


def test_ragged_dims_and_mesh_with_unit_level(adl):
    """non-divisible tensor dims (ceil shards), a level of size 1 and a 3-level odd mesh"""
    rng = np.random.default_rng(9)
    for sizes, links in [((3, 5), (1, 0)), ((1, 7), (1, 0)), ((2, 3, 5), (1, 1, 0)), ((4,), (1,))]:
        L = 6
        recs = []
        for l in range(L):
            M, Kd, N = (int(x) for x in rng.integers(1, 3000, 3))
            if l % 3 == 1:
                recs.append(cf.attn(M, N, int(rng.integers(1, 3000)), 2, int(rng.integers(1, 40)), int(rng.integers(1, 40))))
            else:
                recs.append(cf.gemm(M, Kd, N, 2, 4, 18, in_rows=int(rng.integers(1, 5000)), in_cols=int(rng.integers(1, 5000)),
                                    max_rows=int(rng.integers(1, 64)), max_cols=int(rng.integers(1, 64))))
        layers = np.zeros((1, L), dtype=cf.LAYER_DTYPE)
        for l, r in enumerate(recs):
            layers[0, l] = r
        w = cf.Workload("ragged", layers, cf.Mesh(sizes, links), cf.Net(cf.ALPHA_PS, (3, 40), 150_000 * L), S=4, seed=1)
        init = w.cd_init()
        _assert_same(_gpu_all(adl, w, init), _oracle_all(w, init))


def test_large_dims_64bit(adl):
    """dims beyond 32 bits in bytes (the paper's 2^20 x 8192 fp32 activation)"""
    layers = np.zeros((1, 3), dtype=cf.LAYER_DTYPE)
    for l in range(3):
        layers[0, l] = cf.gemm(2**20, 8192, 8192 * 3, 4, 4, 16)
    w = cf.Workload("big", layers, cf.Mesh((4, 16), (1, 1)), cf.Net((0, 0), (1, 1), 0), S=2)
    init = w.cd_init()
    got = _gpu_all(adl, w, init)
    _assert_same(got, _oracle_all(w, init))
    assert got[0][0, 1, 1, 1] - got[1][0, 1, 1] == 15 * 2**30     # (S0,S1)->(S0,B): the paper's 15 GB


def test_errors(adl):
    import ctypes as C
    w = cf.config1_tiny()
    d_layers = adl.layers_to_device(w.layers)
    bad = cf.Mesh((2, 2, 2, 2), (0, 0, 0, 0))
    with pytest.raises(Exception):
        adl.num_signatures(bad)
    T, _, _ = adl.build_tables(d_layers, w.mesh, w.net)
    w5 = cf.config5_transformer96()
    T5 = torch.zeros((1, 480, 216, 216), dtype=torch.int64, device="cuda")
    with pytest.raises(adl.AutoddlError, match="workspace"):
        adl.chain_dp(T5, w5.mesh, work=torch.empty(256, dtype=torch.uint8, device="cuda"))
    with pytest.raises(adl.AutoddlError):
        adl.coord_descent(T, torch.zeros((1, 1, 4), dtype=torch.int32, device="cuda"), w.mesh, 0)
    m, n = adl.c_mesh(w.mesh), adl.c_net(w.net)
    rc = adl.lib().autoddl_build_tables(None, 1, 4, C.addressof(m), C.addressof(n), None, None, None, None)
    assert rc == -1 and b"NULL" in adl.lib().autoddl_last_error()
