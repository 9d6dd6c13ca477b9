"""Parity of the CUDA Metropolis-Hastings kernel (autoddl_metropolis) against the oracle: bit-exact.

The kernel evaluates 32 proposals of a chain at once and commits them in order; the committed trajectory must be
the sequential one, so every output (best cost and strategy, final state, acceptance count) is compared
element by element.  `pytest -m gpu` on a B200."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf

pytestmark = pytest.mark.gpu
NAMES = ("best_cost", "best_strategy", "final_cost", "final_strategy", "accepted")


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def _same(got, want):
    for g, x, n in zip(got, want, NAMES):
        g = g.cpu().numpy()
        assert g.shape == x.shape and g.dtype == x.dtype, n
        if not np.array_equal(g, x):
            bad = np.argwhere(g != x)
            raise AssertionError(f"{n}: {len(bad)} mismatches, first at {bad[0].tolist()}: got {g[tuple(bad[0])]} want {x[tuple(bad[0])]}")


def _tau(T):
    return int(np.median(T[T < (1 << 50)])) // 8 + 1


@pytest.mark.parametrize("k,nsteps", [(1, 3000), (2, 2000), (3, 1500)])
def test_configs_small(adl, k, nsteps):
    w = cf.CONFIGS[k]()
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    init = w.cd_init()[:, :16]
    for tau in (0, _tau(T), (1 << 40) - 1):                          # greedy, typical, hot (every window full of changes)
        want = ref.metropolis(T, init, nsteps, tau, seed=k)
        got = adl.metropolis(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), w.mesh, nsteps, tau, seed=k)
        _same(got, want)


def test_config5_k216(adl):
    w = cf.config5_transformer96()
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    init = w.cd_init()[:, :6]
    tau = _tau(T)
    want = ref.metropolis(T, init, 4000, tau, seed=5)
    got = adl.metropolis(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), w.mesh, 4000, tau, seed=5)
    _same(got, want)


@pytest.mark.parametrize("K,L,Bp,S,nsteps,hi", [(6, 1, 3, 2, 500, 50), (6, 2, 5, 3, 777, 1000), (36, 3, 7, 2, 1000, 10**6),
                                                 (36, 64, 9, 5, 2500, 10**9), (216, 33, 2, 3, 1200, 10**4), (36, 300, 2, 2, 3000, 100)])
def test_random_tables(adl, K, L, Bp, S, nsteps, hi):
    """ragged window tails (nsteps not a multiple of 32), L < 3 (every step conflicts with every other), ties (small hi),
    chains that do not fill a block"""
    rng = np.random.default_rng(K * 1000 + L)
    T = rng.integers(0, hi, size=(Bp, L, K, K)).astype(np.int64)
    T[:, 0] = T[:, 0, :1]
    init = rng.integers(0, K, size=(Bp, S, L)).astype(np.int32)
    mesh = cf.Mesh((2,) * {6: 1, 36: 2, 216: 3}[K], (0,) * {6: 1, 36: 2, 216: 3}[K])
    for tau in (0, max(hi // 5, 1), hi * 50):
        want = ref.metropolis(T, init, nsteps, tau, seed=L)
        got = adl.metropolis(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), mesh, nsteps, tau, seed=L)
        _same(got, want)
    z = adl.metropolis(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), mesh, 0, 5, seed=1)     # no steps
    _same(z, ref.metropolis(T, init, 0, 5, seed=1))


def test_penalties_and_feasibility(adl):
    """cells carrying the 2^50 infeasibility penalty: uphill moves of >= 2^45 are never accepted"""
    w = cf.config3_transformer24()
    T, _, mask = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    assert (mask == 0).any()
    init = w.cd_init()[:, :8]
    want = ref.metropolis(T, init, 6000, (1 << 40) - 1, seed=3)
    got = adl.metropolis(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), w.mesh, 6000, (1 << 40) - 1, seed=3)
    _same(got, want)


def test_config4_full_size_sampled(adl):
    """BASELINE.json configs[3] at full size: 4096 chains on GPU-built tables.  The draws of a chain depend on its
    index, so the oracle replays the first 24 chains; properties are checked on all of them."""
    w = cf.config4_batched()
    d_layers = adl.layers_to_device(w.layers)
    T, _, _ = adl.build_tables(d_layers, w.mesh, w.net)
    init = w.cd_init()
    nsteps, tau = 2048, 20_000_000
    bc, bs, fc, fs, acc = adl.metropolis(T, torch.from_numpy(init).cuda(), w.mesh, nsteps, tau, seed=0)
    dc, _ = adl.chain_dp(T, w.mesh)
    torch.cuda.synchronize()
    n = 24
    oT, _, _ = ref.build_tables(w.layers[:n], ref.mesh_of(w), ref.net_of(w))
    want = ref.metropolis(oT, init[:n], nsteps, tau, seed=0)
    _same([x[:n] for x in (bc, bs, fc, fs, acc)], want)
    # properties on all chains: costs re-evaluate, optimum <= best <= final-or-start
    Bp, L, K = w.Bp, w.L, w.K
    ar = torch.arange(Bp, device="cuda")[:, None]
    for strat, cost in ((bs, bc), (fs, fc)):
        s = strat[:, 0].long()
        prev = torch.cat([torch.zeros((Bp, 1), dtype=torch.long, device="cuda"), s[:, :-1]], 1)
        lidx = torch.arange(L, device="cuda")[None, :]
        re = T[ar, lidx, prev, s].sum(1)
        assert torch.equal(re, cost[:, 0])
    assert (bc[:, 0] >= dc).all() and (bc <= fc).all() and (acc >= 0).all() and (acc <= nsteps).all()


@pytest.mark.parametrize("L", [1, 2, 3, 31, 97, 1000, 4099])
@pytest.mark.parametrize("sizes,links", [((4,), (1,)), ((2, 2, 2, 2), (0x03 << 8,) * 4), ((2, 2, 2, 2, 2), (0x07 << 8,) * 5)])
def test_draw_reduction_for_odd_lengths_and_k(adl, L, sizes, links):
    """the layer and signature draws are reduced modulo L and K by a multiply-high remainder in the kernel and by `%` in the
    oracle: chain lengths 1, primes, a value above 2^12, and K = 6, 16, 243 on random tables"""
    mesh = cf.Mesh(sizes, links)
    K = adl.num_signatures(mesh)
    L = min(L, 60_000_000 // (K * K))                            # K = 243: at most 1016 layers (480 MB of tables)
    rng = np.random.default_rng(L + K)
    T = rng.integers(0, 1000, size=(1, L, K, K)).astype(np.int64)
    init = rng.integers(0, K, size=(1, 5, L)).astype(np.int32)
    want = ref.metropolis(T, init, 3000, 400, seed=L)
    got = adl.metropolis(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), mesh, 3000, 400, seed=L)
    _same(got, want)
