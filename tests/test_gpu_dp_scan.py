"""Chain DP of few long chains in class space, parallel over the layers (csrc/chain_dp_scan.cu: class matrices, chunk products,
prefix vectors, per-chunk DP, walk) against the oracle's sequential DP (PAPER.md:225 exhaustive optimum,
R9 tie-break): optimum AND strategy bit-exact at chain lengths around every chunk boundary, on two and three mesh levels,
with attention layers (the invalid class), split limits, a memory cap (2^50 penalties in the sums) and several chains."""
import numpy as np
import pytest
import torch

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


def _chains(rng, Bp, L, ragged):
    layers = np.zeros((Bp, L), dtype=cf.LAYER_DTYPE)
    for p in range(Bp):
        M = int(rng.integers(300, 3000)) if ragged else 1024
        d = int(rng.integers(200, 3000)) if ragged else 512
        for l in range(L):
            n = int(rng.integers(200, 3000)) if ragged else 512 * int(rng.integers(1, 5))
            if l % 5 == 1:
                layers[p, l] = cf.attn(M, n, d, 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)))
            else:
                layers[p, l] = cf.gemm(M, d, n, 2, 4, 18, max_rows=int(rng.integers(2, 64)) if l % 7 == 3 else None)
            d = n
    return layers


def _check(adl, w):
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    want_c, want_s = ref.chain_dp(T)
    d_layers = adl.layers_to_device(w.layers)
    work = torch.empty(adl.workspace_bytes(w.Bp, w.L, 0, w.mesh), dtype=torch.uint8, device="cuda")
    work.fill_(0x5A)                                         # nothing may be read before it is written
    got_c, got_s = adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers, work=work)
    torch.cuda.synchronize()
    assert np.array_equal(got_c.cpu().numpy(), want_c)
    assert np.array_equal(got_s.cpu().numpy(), want_s)
    # and through the one-call path, which shares the factors with nothing else here
    out = adl.search(d_layers, w.mesh, w.net, want_tables=False, work=work)
    torch.cuda.synchronize()
    assert np.array_equal(out["opt_cost"].cpu().numpy(), want_c) and np.array_equal(out["strategy"].cpu().numpy(), want_s)


# two levels: chunks of 8 layers -> boundaries at L - 2 = 8 k
@pytest.mark.parametrize("L", [32, 33, 34, 35, 41, 42, 43, 50, 121])
def test_scan_dp_two_levels(adl, L):
    rng = np.random.default_rng(100 + L)
    for Bp, sizes, cap in [(1, (4, 8), 0), (3, (3, 5), 60_000 * L)]:
        w = cf.Workload("scan2", _chains(rng, Bp, L, ragged=True), cf.Mesh(sizes, (cf.INTER, cf.INTRA)),
                        cf.Net(cf.ALPHA_PS, (cf.BETA_300, cf.BETA_25), cap), S=1, seed=1)
        _check(adl, w)


# three levels: chunks of 8 layers below 256 layers, of 16 from there on
@pytest.mark.parametrize("L", [32, 34, 49, 257, 258, 259, 274])
def test_scan_dp_three_levels(adl, L):
    rng = np.random.default_rng(200 + L)
    Bp = 2 if L < 100 else 1
    w = cf.Workload("scan3", _chains(rng, Bp, L, ragged=L < 100), cf.Mesh((2, 3, 2), (cf.INTER, cf.INTER, cf.INTRA)),
                    cf.Net(cf.ALPHA_PS, (cf.BETA_300, cf.BETA_25), 40_000 * L if L == 49 else 0), S=1, seed=1)
    _check(adl, w)


def test_scan_dp_many_chains_and_fallbacks(adl):
    """64 chains still take the scan path, 65 the table kernels; 31 layers are below its threshold: all agree with the oracle"""
    rng = np.random.default_rng(7)
    for Bp, L in [(64, 40), (65, 40), (2, 31)]:
        w = cf.Workload("scan-many", _chains(rng, Bp, L, ragged=True), cf.Mesh((2, 2, 2), (cf.INTER, cf.INTER, cf.INTRA)),
                        cf.Net(cf.ALPHA_PS, (cf.BETA_300, cf.BETA_25), 0), S=1, seed=1)
        _check(adl, w)


# ---- the same scheme on K x K tables (any mesh, K <= 64): caller-supplied tables, so random ones with MANY ties --------------
def _mesh_with_k(K):
    """a mesh whose signature count is K (the tables themselves are random)"""
    if K == 36:
        return cf.Mesh((4, 4), (cf.INTER, cf.INTRA))
    if K == 16:                                              # four levels, two allowed rows each (R24, R26)
        return cf.Mesh((2, 2, 2, 2), tuple(l | (0x03 << 8) for l in (cf.INTER, cf.INTER, cf.INTRA, cf.INTRA)))
    if K == 64:                                              # four levels, 4 . 4 . 2 . 2 allowed rows
        return cf.Mesh((2, 2, 2, 2), (cf.INTER | (0x0f << 8), cf.INTER | (0x0f << 8), cf.INTRA | (0x03 << 8), cf.INTRA | (0x03 << 8)))
    if K in (28, 45):                                        # folded: six / eight equal levels (R28)
        n = 6 if K == 28 else 8
        return cf.Mesh((2,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))
    raise ValueError(K)


@pytest.mark.parametrize("K,L,Bp,hi", [(36, 32, 1, 4), (36, 33, 3, 1 << 40), (16, 41, 2, 3), (28, 40, 1, 5), (45, 57, 2, 1 << 45),
                                       (45, 220, 1, 7), (64, 49, 2, 4), (64, 130, 1, 1 << 50), (36, 64, 64, 6)])
def test_scan_dp_on_tables(adl, K, L, Bp, hi):
    """random tables; with cells in [0, hi) for a small hi nearly every minimum is tied: the back-pointers must be the
    sequential DP's (smallest i), chunk by chunk"""
    mesh = _mesh_with_k(K)
    assert adl.num_signatures(mesh) == K
    rng = np.random.default_rng(K * 1000 + L)
    T = rng.integers(0, hi, size=(Bp, L, K, K), dtype=np.int64)
    want_c, want_s = ref.chain_dp(T)
    d_T = torch.from_numpy(T).cuda()
    work = torch.empty(adl.workspace_bytes(Bp, L, 0, mesh), dtype=torch.uint8, device="cuda")
    work.fill_(0xA5)
    got_c, got_s = adl.chain_dp(d_T, mesh, work=work)
    torch.cuda.synchronize()
    assert np.array_equal(got_c.cpu().numpy(), want_c)
    assert np.array_equal(got_s.cpu().numpy(), want_s)
    # the kernel that runs when the workspace is too small for this path gives the same
    small = torch.empty(Bp * L * K + 4096, dtype=torch.uint8, device="cuda")
    c2, s2 = adl.chain_dp(d_T, mesh, work=small)
    assert torch.equal(c2, got_c) and torch.equal(s2, got_s)
