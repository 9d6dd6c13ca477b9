"""Coordinate Descent from few starts on caller-supplied tables: the sweeps of a start run side by side
(coord_descent_wave_kernel).  Trajectory-dependent outputs -- result, cost and SWEEP COUNT -- must be those of the plain
sequential algorithm (oracle R10), also when a descent needs more sweeps than the block has warps (each warp then runs
several sweeps), when the cap cuts it short, and on tables whose updates nearly all tie."""
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


def _mesh(K):
    if K == 6:
        return cf.Mesh((4,), (cf.INTER,))
    if K == 36:
        return cf.Mesh((4, 4), (cf.INTER, cf.INTRA))
    if K == 216:
        return cf.Mesh((2, 2, 2), (cf.INTER, cf.INTER, cf.INTRA))
    if K == 81:
        return cf.Mesh((2, 2, 2, 2), (0x07 << 8,) * 4)
    if K == 243:
        return cf.CONFIGS[7]().mesh
    if K == 16:
        return cf.Mesh((2, 2, 2, 2), tuple(l | (0x03 << 8) for l in (cf.INTER, cf.INTER, cf.INTRA, cf.INTRA)))
    n = {28: 6, 36: 7, 45: 8}[K]
    return cf.Mesh((2,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))


def _backward_chain(K, L, Bp, rng, noise):
    """tables on which a change travels from the last layer to the first ONE layer per sweep: the coupling of a layer to
    its right neighbour (weight l + 2) beats the one to its left (l + 1), and only the last layer has a preference"""
    T = np.zeros((Bp, L, K, K), dtype=np.int64)
    eye = np.eye(K, dtype=np.int64)
    for l in range(L):
        T[:, l] = (1 - eye) * (l + 1) * 1000
    T[:, L - 1] += (np.arange(K) != 1).astype(np.int64)[None, None, :] * 10_000_000
    if noise:
        T += rng.integers(0, noise, size=T.shape, dtype=np.int64)
    return T


def _check(adl, K, T, init, cap):
    mesh = _mesh(K)
    assert adl.num_signatures(mesh) == K
    want = ref.coord_descent(T, init, cap)
    got = adl.coord_descent(torch.from_numpy(T).cuda(), torch.from_numpy(init).cuda(), mesh, cap)
    torch.cuda.synchronize()
    for name, g, x in zip(("cd_cost", "cd_strategy", "cd_sweeps"), got, want):
        assert np.array_equal(g.cpu().numpy(), x), name
    return want[2]


@pytest.mark.parametrize("K,L,Bp,S,cap,noise", [(6, 40, 1, 3, 64, 0), (6, 40, 1, 3, 20, 0), (36, 30, 1, 300, 64, 5), (16, 70, 2, 5, 200, 0),
                                                (28, 25, 1, 9, 64, 3), (243, 12, 1, 4, 64, 0), (216, 20, 3, 2, 9, 0), (6, 8, 1, 1, 64, 0)])
def test_descents_longer_than_the_block_has_warps(adl, K, L, Bp, S, cap, noise):
    rng = np.random.default_rng(K * 31 + L + cap)
    T = _backward_chain(K, L, Bp, rng, noise)
    init = rng.integers(0, K, size=(Bp, S, L), dtype=np.int32)
    init[:, 0] = 0                                           # the all-zero start: exactly one layer flips per sweep
    sweeps = _check(adl, K, T, init, cap)
    assert sweeps.max() == min(cap, L + 1)                   # the chain really is that long: every warp ran several sweeps


@pytest.mark.parametrize("K,L,Bp,S,hi,cap", [(243, 24, 1, 20, 1 << 40, 64), (216, 40, 1, 10, 50, 64), (81, 64, 1, 330, 1 << 35, 64),
                                             (6, 8, 3, 100, 3, 64), (36, 400, 2, 20, 1 << 40, 64), (36, 9, 1, 300, 7, 2),
                                             (45, 33, 7, 290, 4, 3), (6, 2000, 1, 8, 1 << 30, 64)])
def test_random_tables(adl, K, L, Bp, S, hi, cap):
    rng = np.random.default_rng(K * 131 + L)
    T = rng.integers(0, hi, size=(Bp, L, K, K), dtype=np.int64)
    init = rng.integers(0, K, size=(Bp, S, L), dtype=np.int32)
    _check(adl, K, T, init, cap)


@pytest.mark.parametrize("Bp,S,L,cap", [(100, 2, 64, 64), (70, 8, 24, 64), (300, 3, 40, 5), (65, 1, 9, 64)])
def test_resume_after_the_fused_kernel(adl, Bp, S, L, cap):
    """one call on a two-level mesh with more than 64 chains: the fused kernel runs sweeps 1 and 2, the sweep-parallel kernel
    resumes from sweep 3 (8 warps per start up to 296 starts, 4 beyond) -- same costs, strategies and sweep counts"""
    w = cf.config4_batched(Bp=Bp, L=L, seed=Bp + S)
    rng = np.random.default_rng(Bp * 7 + S)
    init = rng.integers(0, w.K, size=(Bp, S, L), dtype=np.int32)
    one = adl.search(adl.layers_to_device(w.layers), w.mesh, w.net, init=torch.from_numpy(init).cuda(), max_sweeps=cap)
    torch.cuda.synchronize()
    oT, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    want = ref.coord_descent(oT, init, cap)
    for name, x in zip(("cd_cost", "cd_strategy", "cd_sweeps"), want):
        assert np.array_equal(one[name].cpu().numpy(), x), name
    assert want[2].max() > 2 or cap <= 2                     # the resume kernel had sweeps to run
