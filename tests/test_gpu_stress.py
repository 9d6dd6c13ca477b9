"""Randomised differential test (`pytest -m gpu`): the one-call path (fused kernel for >= 296 chains, CD resume, class
representative rows) against the three separate kernels on ALL chains, and against the oracle on a sample, over random
meshes (1-3 levels, sizes 1..8, random allowed-row masks), chain counts around the fused-kernel thresholds (295/296,
739/740/741 = resident CTAs), chain lengths around the group size, mixed GEMM / ATTN kinds, split limits, memory caps,
1-3 starts, sweep caps 1, 2, 3, 64 and 0-17 micro-batches; a second generator covers four and five mesh levels.  Bit-exact.  (A 480-second run of the same generator, ~28,000 cases, is clean.)"""
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


@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_random_cases(adl, seed):
    rng = np.random.default_rng(seed)
    for case in range(150):
        D = int(rng.choice([1, 2, 2, 2, 3]))
        sizes = tuple(int(x) for x in rng.choice([1, 2, 3, 4, 5, 8], D))
        links = tuple(int(rng.integers(0, 2)) | (int(rng.choice([0, 0, 0x07, 0x0b, 0x3e, 0x15])) << 8) for _ in range(D))
        Bp = int(rng.choice([1, 2, 17, 295, 296, 300, 739, 740, 741, 1481, 2000])) if D == 2 else int(rng.choice([1, 3, 9]))
        L = int(rng.choice([1, 2, 3, 4, 5, 7, 8, 9, 16, 33, 63, 64, 65]))
        if D == 3: L = min(L, 9)
        if Bp * L > 60000: Bp = max(1, 60000 // L)
        S = int(rng.choice([1, 1, 2, 3]))
        layers = np.zeros((Bp, L), dtype=cf.LAYER_DTYPE)
        base = cf.config4_batched(Bp=Bp, L=L, seed=int(rng.integers(0, 1000))).layers
        layers[:] = base
        pa = float(rng.choice([0.0, 0.0, 0.3]))
        if pa > 0:
            for p in range(min(Bp, 400)):
                for l in range(L):
                    if rng.random() < pa:
                        layers[p, l] = cf.attn(int(layers[p, l]["M"]), int(layers[p, l]["N"]), int(rng.integers(1, 4000)), 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)))
        if rng.random() < 0.3:
            layers["max_split_rows"] = rng.integers(1, 40, size=layers.shape)
            layers["max_split_cols"] = rng.integers(1, 40, size=layers.shape)
        cap = int(rng.choice([0, 0, 10**7 * L, 10**9 * L]))
        w = cf.Workload("stress", layers, cf.Mesh(sizes, links), cf.Net(cf.ALPHA_PS, (3, 40), cap, micro_batches=int(rng.choice([0, 1, 1, 3, 17]))), S=S, seed=int(rng.integers(0, 1000)))
        init = w.cd_init()
        cap_sw = int(rng.choice([1, 2, 3, 64]))
        dl = adl.layers_to_device(w.layers)
        dinit = torch.from_numpy(init).cuda()
        T, node, mask = adl.build_tables(dl, w.mesh, w.net)
        work = torch.empty(adl.workspace_bytes(Bp, L, S, w.mesh), dtype=torch.uint8, device="cuda")
        dc, ds = adl.chain_dp(T, w.mesh, work=work)
        cc, cs, sw = adl.coord_descent(T, dinit, w.mesh, cap_sw)
        o = adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=cap_sw, want_node_mask=True)
        torch.cuda.synchronize()
        ok = all(torch.equal(a, b) for a, b in ((o["T"], T), (o["node"], node), (o["mask"], mask), (o["opt_cost"], dc), (o["strategy"], ds),
                                               (o["cd_cost"], cc), (o["cd_strategy"], cs), (o["cd_sweeps"], sw)))
        idx = np.unique(rng.integers(0, Bp, min(Bp, 3)))
        oT, on, om = ref.build_tables(np.ascontiguousarray(w.layers[idx]), ref.mesh_of(w), ref.net_of(w))
        odc, ods = ref.chain_dp(oT)
        occ, ocs, osw = ref.coord_descent(oT, np.ascontiguousarray(init[idx]), cap_sw)
        ok2 = (np.array_equal(T[idx].cpu().numpy(), oT) and np.array_equal(node[idx].cpu().numpy(), on) and np.array_equal(mask[idx].cpu().numpy(), om)
               and np.array_equal(dc[idx].cpu().numpy(), odc) and np.array_equal(ds[idx].cpu().numpy(), ods) and np.array_equal(cc[idx].cpu().numpy(), occ) and np.array_equal(cs[idx].cpu().numpy(), ocs)
               and np.array_equal(sw[idx].cpu().numpy(), osw))
        assert ok and ok2, dict(seed=seed, case=case, sizes=sizes, links=links, Bp=Bp, L=L, S=S, pa=pa, cap=cap, cap_sw=cap_sw,
                                one_call_equals_separate=ok, separate_equals_oracle=ok2)


@pytest.mark.parametrize("seed", [11, 12])
def test_random_deep_meshes(adl, seed):
    """four and five mesh levels (R26): random allowed-row sets with K <= 256, chain counts on both sides of the
    cluster / one-CTA switch of the single-chain DP (Bp * 8 <= 148), back-pointers in shared memory and in the workspace.
    (A 240-second run of this generator, 5,600 cases over 140 seeds, is clean.)"""
    rng = np.random.default_rng(seed)
    masks = [0x01, 0x03, 0x05, 0x06, 0x07, 0x0b, 0x0e, 0x15, 0x30, 0x0f, 0x38]
    for case in range(40):
        D = int(rng.choice([4, 5]))
        while True:
            allow = [int(rng.choice(masks)) for _ in range(D)]
            K = int(np.prod([bin(a).count("1") for a in allow]))
            if 2 <= K <= 256:
                break
        sizes = tuple(int(x) for x in rng.choice([1, 2, 2, 3, 4], D))
        links = tuple(int(rng.integers(0, 2)) | (a << 8) for a in allow)
        Bp = int(rng.choice([1, 2, 5, 18, 19, 40]))
        L = int(rng.choice([1, 2, 3, 5, 9, 17, 70]))
        if Bp * L * K * K > 3_000_000: Bp = max(1, 3_000_000 // (L * K * K))
        S = int(rng.choice([1, 2, 3]))
        layers = cf.config4_batched(Bp=Bp, L=L, seed=int(rng.integers(0, 1000))).layers.copy()
        if rng.random() < 0.5:
            for p in range(Bp):
                for l in range(L):
                    if rng.random() < 0.3:
                        layers[p, l] = cf.attn(int(layers[p, l]["M"]), int(layers[p, l]["N"]), int(rng.integers(1, 4000)), 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)))
        if rng.random() < 0.3:
            layers["max_split_rows"] = rng.integers(1, 40, size=layers.shape)
            layers["max_split_cols"] = rng.integers(1, 40, size=layers.shape)
        cap = int(rng.choice([0, 0, 10**7 * L, 10**9 * L]))
        w = cf.Workload("stress-deep", layers, cf.Mesh(sizes, links), cf.Net(cf.ALPHA_PS, (3, 40), cap, micro_batches=int(rng.choice([0, 1, 3]))), S=S, seed=int(rng.integers(0, 1000)))
        assert w.K == K
        init = w.cd_init()
        cap_sw = int(rng.choice([1, 2, 64]))
        dl = adl.layers_to_device(w.layers)
        dinit = torch.from_numpy(init).cuda()
        T, node, mask = adl.build_tables(dl, w.mesh, w.net)
        work = torch.empty(adl.workspace_bytes(Bp, L, S, w.mesh), dtype=torch.uint8, device="cuda")
        dc, ds = adl.chain_dp(T, w.mesh, work=work)
        cc, cs, sw = adl.coord_descent(T, dinit, w.mesh, cap_sw)
        o = adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=cap_sw, want_node_mask=True)
        torch.cuda.synchronize()
        ok = all(torch.equal(a, b) for a, b in ((o["T"], T), (o["node"], node), (o["mask"], mask), (o["opt_cost"], dc), (o["strategy"], ds),
                                               (o["cd_cost"], cc), (o["cd_strategy"], cs), (o["cd_sweeps"], sw)))
        idx = np.unique(rng.integers(0, Bp, min(Bp, 2)))
        oT, on, om = ref.build_tables(np.ascontiguousarray(w.layers[idx]), ref.mesh_of(w), ref.net_of(w))
        odc, ods = ref.chain_dp(oT)
        occ, ocs, osw = ref.coord_descent(oT, np.ascontiguousarray(init[idx]), cap_sw)
        ok2 = (np.array_equal(T[idx].cpu().numpy(), oT) and np.array_equal(node[idx].cpu().numpy(), on) and np.array_equal(mask[idx].cpu().numpy(), om)
               and np.array_equal(dc[idx].cpu().numpy(), odc) and np.array_equal(ds[idx].cpu().numpy(), ods) and np.array_equal(cc[idx].cpu().numpy(), occ)
               and np.array_equal(cs[idx].cpu().numpy(), ocs) and np.array_equal(sw[idx].cpu().numpy(), osw))
        assert ok and ok2, dict(seed=seed, case=case, sizes=sizes, links=links, K=K, Bp=Bp, L=L, S=S, cap=cap, cap_sw=cap_sw,
                                one_call_equals_separate=ok, separate_equals_oracle=ok2)


# ---- generators for the paths added late in round 2: class-space DP and look-up CD on the factors (A), the same two schemes
# on K x K tables with K <= 64 and the allocation-free entry point (B), the fused kernel with up to 9 starts (C).
# (A 600-second run of the three generators, 9,000 cases over seeds 1000..9993, is clean.)
def _rand_layers(rng, Bp, L):
    layers = cf.config4_batched(Bp=Bp, L=L, seed=int(rng.integers(0, 100000))).layers.copy()
    pa = float(rng.choice([0.0, 0.2, 0.4]))
    if pa > 0:
        for p in range(min(Bp, 64)):
            for l in range(L):
                if rng.random() < pa:
                    layers[p, l] = cf.attn(int(layers[p, l]["M"]), int(layers[p, l]["N"]), int(rng.integers(1, 4000)), 2,
                                           int(rng.integers(1, 40)), int(rng.integers(1, 40)))
    if rng.random() < 0.3:
        layers["max_split_rows"] = rng.integers(1, 40, size=layers.shape)
        layers["max_split_cols"] = rng.integers(1, 40, size=layers.shape)
    if rng.random() < 0.3:                                   # ragged dims
        for f in ("M", "Kd", "N"):
            layers[f] = rng.integers(1, 3000, size=layers.shape)
        layers["in_rows"], layers["in_cols"] = layers["M"], layers["Kd"]
    return layers


def _same(got, want, ctx):
    for name, g, o in zip(ctx["names"], got, want):
        assert np.array_equal(g.cpu().numpy(), o), dict(ctx, differs=name)


@pytest.mark.parametrize("seed", [21, 22])
def test_random_long_chains_on_factors(adl, seed):
    rng = np.random.default_rng(seed)
    for case in range(40):
        D = int(rng.choice([2, 2, 3]))
        sizes = tuple(int(x) for x in rng.choice([1, 2, 3, 4, 5, 8], D))
        links = tuple(int(rng.integers(0, 2)) | (int(rng.choice([0, 0, 0x07, 0x0b, 0x3e, 0x15])) << 8) for _ in range(D))
        Bp = int(rng.choice([1, 1, 2, 5, 64])) if D == 2 else int(rng.choice([1, 2]))
        L = int(rng.integers(32, 140)) if D == 2 else int(rng.integers(32, 60))
        S, cap_sw = int(rng.choice([1, 3, 32, 40])), int(rng.choice([1, 2, 3, 64]))
        cap = int(rng.choice([0, 0, 10**7 * L, 10**9 * L]))
        w = cf.Workload("fz", _rand_layers(rng, Bp, L), cf.Mesh(sizes, links),
                        cf.Net(cf.ALPHA_PS, (3, 40), cap, micro_batches=int(rng.choice([0, 1, 3]))), S=S, seed=int(rng.integers(0, 1000)))
        init = w.cd_init()
        ctx = dict(seed=seed, case=case, sizes=sizes, links=links, Bp=Bp, L=L, S=S, cap=cap, cap_sw=cap_sw,
                   names=("opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
        dl, dinit = adl.layers_to_device(w.layers), torch.from_numpy(init).cuda()
        work = torch.empty(adl.workspace_bytes(Bp, L, S, w.mesh), dtype=torch.uint8, device="cuda")
        work.fill_(int(rng.integers(0, 256)))
        o1 = adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=cap_sw, want_tables=False, work=work)
        o2 = adl.search(dl, w.mesh, w.net, init=dinit, max_sweeps=cap_sw, work=work)
        torch.cuda.synchronize()
        oT, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
        want = ref.chain_dp(oT) + ref.coord_descent(oT, init, cap_sw)
        assert np.array_equal(o2["T"].cpu().numpy(), oT), ctx
        _same([o1[k] for k in ctx["names"]], want, dict(ctx, path="no table"))
        _same([o2[k] for k in ctx["names"]], want, dict(ctx, path="tables wanted"))


def _mesh_with_k(K):
    if K == 6:
        return cf.Mesh((4,), (cf.INTRA,))
    if K == 36:
        return cf.Mesh((4, 4), (cf.INTER, cf.INTRA))
    if K == 16:
        return cf.Mesh((2, 2, 2, 2), tuple(l | (0x03 << 8) for l in (cf.INTER, cf.INTER, cf.INTRA, cf.INTRA)))
    if K == 64:
        return cf.Mesh((2, 2, 2, 2), (cf.INTER | (0x0f << 8), cf.INTER | (0x0f << 8), cf.INTRA | (0x03 << 8), cf.INTRA | (0x03 << 8)))
    n = {10: 3, 15: 4, 21: 5, 28: 6, 45: 8}[K]                # folded: n equal levels, (n + 2)(n + 1) / 2 signatures
    return cf.Mesh((2,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))


@pytest.mark.parametrize("seed", [31, 32])
def test_random_small_tables(adl, seed):
    rng = np.random.default_rng(seed)
    for case in range(60):
        K = int(rng.choice([6, 36, 16, 64, 28, 45, 10, 15, 21]))
        mesh = _mesh_with_k(K)
        assert adl.num_signatures(mesh) == K
        Bp, L = int(rng.choice([1, 2, 3, 64])), int(rng.choice([1, 2, 31, 32, 33, 40, 41, 48, 49, 97, 200]))
        S, cap_sw = int(rng.choice([1, 31, 32, 33, 64])), int(rng.choice([1, 2, 3, 64]))
        if Bp * L * K * K > 6e6:
            Bp = 1
        hi = int(rng.choice([2, 4, 9, 1 << 20, 1 << 50]))
        ctx = dict(seed=seed, case=case, K=K, Bp=Bp, L=L, S=S, hi=hi, cap_sw=cap_sw, names=("opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps"))
        T = rng.integers(0, hi, size=(Bp, L, K, K), dtype=np.int64)
        init = rng.integers(0, K, size=(Bp, S, L), dtype=np.int32)
        dT, dinit = torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda()
        work = torch.empty(adl.workspace_bytes(Bp, L, S, mesh), dtype=torch.uint8, device="cuda")
        work.fill_(int(rng.integers(0, 256)))
        got = adl.chain_dp(dT, mesh, work=work) + adl.coord_descent(dT, dinit, mesh, cap_sw, work=work)
        torch.cuda.synchronize()
        want = ref.chain_dp(T) + ref.coord_descent(T, init, cap_sw)
        _same(got, want, ctx)
        if 0 < adl.chain_dp_static_bytes(Bp, L, mesh) <= adl.STATIC_SCRATCH_BYTES:
            out = (torch.empty(Bp, dtype=torch.int64, device="cuda"), torch.empty((Bp, L), dtype=torch.int32, device="cuda"))
            adl.chain_dp_static(dT, mesh, out)
            torch.cuda.synchronize()
            _same(out, want[:2], dict(ctx, path="static scratch"))


@pytest.mark.parametrize("seed", [41])
def test_random_fused_many_starts(adl, seed):
    rng = np.random.default_rng(seed)
    for case in range(40):
        sizes = tuple(int(x) for x in rng.choice([1, 2, 3, 4, 5, 8, 16], 2))
        links = tuple(int(rng.integers(0, 2)) | (int(rng.choice([0, 0, 0x07, 0x0b, 0x3e, 0x15])) << 8) for _ in range(2))
        Bp, L = int(rng.choice([296, 300, 741, 1000, 4200])), int(rng.choice([1, 2, 3, 5, 8, 9, 17, 33, 64, 70]))
        S, cap_sw = int(rng.choice([1, 2, 4, 8, 9])), int(rng.choice([1, 2, 3, 4, 64]))
        if Bp * L > 40000:
            Bp = max(296, 40000 // L)
        cap = int(rng.choice([0, 0, 10**7 * L, 10**9 * L]))
        w = cf.Workload("fz", _rand_layers(rng, Bp, L), cf.Mesh(sizes, links),
                        cf.Net(cf.ALPHA_PS, (3, 40), cap, micro_batches=int(rng.choice([0, 1, 3]))), S=S, seed=int(rng.integers(0, 1000)))
        init = w.cd_init()
        names = ("T", "node", "mask", "opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")
        ctx = dict(seed=seed, case=case, sizes=sizes, links=links, Bp=Bp, L=L, S=S, cap=cap, cap_sw=cap_sw, names=names)
        o = adl.search(adl.layers_to_device(w.layers), w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=cap_sw, want_node_mask=True)
        torch.cuda.synchronize()
        idx = np.unique(np.concatenate([[0, Bp - 1], rng.integers(0, Bp, 6)]))
        oT, on, om = ref.build_tables(np.ascontiguousarray(w.layers[idx]), ref.mesh_of(w), ref.net_of(w))
        want = (oT, on, om) + ref.chain_dp(oT) + ref.coord_descent(oT, np.ascontiguousarray(init[idx]), cap_sw)
        _same([o[k][torch.from_numpy(idx).cuda()] for k in names], want, ctx)


@pytest.mark.parametrize("seed", [51])
def test_random_deep_and_folded_one_call(adl, seed):
    """the one-call path on folded, four- and five-level meshes (K <= 256): layer-parallel DP beside look-up or gather CD on
    side streams, with and without the tables wanted.  (A 900-second run of generators A-D on the final library, 11,880 cases over seeds 50000..61879, is clean.)"""
    rng = np.random.default_rng(seed)
    names = ("opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps")
    for case in range(40):
        kind = int(rng.integers(0, 3))
        if kind == 0:
            n, sz = int(rng.integers(3, 9)), int(rng.choice([2, 2, 3]))
            mesh = cf.Mesh((sz,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))
        elif kind == 1:
            masks = [int(rng.choice([0x03, 0x05, 0x07, 0x0b])) for _ in range(4)]
            mesh = cf.Mesh(tuple(int(x) for x in rng.choice([2, 2, 3, 4], 4)), tuple(int(rng.integers(0, 2)) | (m << 8) for m in masks))
        else:
            mesh = cf.Mesh((2, 2, 2, 2, 2), tuple(int(rng.integers(0, 2)) | (int(rng.choice([0x03, 0x07])) << 8) for _ in range(5)))
        K = adl.num_signatures(mesh)
        if K > 256:
            continue
        Bp, L = int(rng.choice([1, 2, 64])), int(rng.choice([1, 2, 9, 31, 32, 33, 48, 70]))
        S, cap_sw = int(rng.choice([1, 3, 32, 40])), int(rng.choice([1, 2, 3, 64]))
        if Bp * L * K * K > 3e6:
            Bp = 1
        if L * K * K > 3e6:
            L = 9
        cap = int(rng.choice([0, 0, 10**8 * L]))
        w = cf.Workload("fz", _rand_layers(rng, Bp, L), mesh, cf.Net(cf.ALPHA_PS, (3, 40), cap, micro_batches=int(rng.choice([0, 1, 3]))),
                        S=S, seed=int(rng.integers(0, 1000)))
        init = w.cd_init()
        ctx = dict(seed=seed, case=case, size=mesh.size, link=mesh.link, K=K, Bp=Bp, L=L, S=S, cap=cap, cap_sw=cap_sw, names=names)
        dl, dinit = adl.layers_to_device(w.layers), torch.from_numpy(init).cuda()
        work = torch.empty(adl.workspace_bytes(Bp, L, S, mesh), dtype=torch.uint8, device="cuda")
        work.fill_(int(rng.integers(0, 256)))
        o1 = adl.search(dl, mesh, w.net, init=dinit, max_sweeps=cap_sw, want_tables=False, work=work)
        o2 = adl.search(dl, mesh, w.net, init=dinit, max_sweeps=cap_sw, want_node_mask=True, work=work)
        torch.cuda.synchronize()
        oT, on, om = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
        want = ref.chain_dp(oT) + ref.coord_descent(oT, init, cap_sw)
        for nm, g, o in (("T", o2["T"], oT), ("node", o2["node"], on), ("mask", o2["mask"], om)):
            assert np.array_equal(g.cpu().numpy(), o), dict(ctx, differs=nm)
        _same([o1[k] for k in names], want, dict(ctx, path="no table"))
        _same([o2[k] for k in names], want, dict(ctx, path="tables wanted"))
