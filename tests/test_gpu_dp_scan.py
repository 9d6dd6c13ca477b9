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
