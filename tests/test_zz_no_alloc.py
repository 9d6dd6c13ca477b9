"""autoddl_chain_dp_static: the chain DP (R9 tie-break) with its scratch in the library's static device array
-- for callers that cannot call cudaMalloc -- against the existing path autoddl_chain_dp and the oracle, bit-exact (integer
work), on two calls in a row (the array keeps the first call's contents; the second call has another shape).  Collected
last on purpose (file name): a failure here hides no other test under pytest -x."""
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


def _folded_mesh(n):
    return cf.Mesh((2,) * n, (cf.INTER | cf.FOLD,) + (cf.INTER,) * (n - 1))


def test_static_scratch_chain_dp_two_calls_in_a_row(adl):
    cases = [(cf.Mesh((4, 4), (cf.INTER, cf.INTRA)), 36, 3, 97, 5),            # heavily tied cells
             (_folded_mesh(8), 45, 1, 220, 1 << 45),                            # config 11's shape, another K and L
             (cf.Mesh((4, 4), (cf.INTER, cf.INTRA)), 36, 3, 97, 5)]             # the first one again, after a different call
    for mesh, K, Bp, L, hi in cases:
        assert adl.num_signatures(mesh) == K
        need = adl.chain_dp_static_bytes(Bp, L, mesh)
        assert 0 < need <= adl.STATIC_SCRATCH_BYTES
        T = np.random.default_rng(K * 31 + L).integers(0, hi, size=(Bp, L, K, K), dtype=np.int64)
        d_T = torch.from_numpy(T).cuda()
        out = (torch.full((Bp,), -1, dtype=torch.int64, device="cuda"), torch.full((Bp, L), -1, dtype=torch.int32, device="cuda"))
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        adl.chain_dp_static(d_T, mesh, out)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before                          # (torch's view: the binding allocated nothing)
        work = torch.empty(adl.workspace_bytes(Bp, L, 0, mesh), dtype=torch.uint8, device="cuda")
        ec, es = adl.chain_dp(d_T, mesh, work=work)                             # the existing path
        torch.cuda.synchronize()
        assert torch.equal(out[0], ec) and torch.equal(out[1], es)
        oc, os_ = ref.chain_dp(T)
        assert np.array_equal(out[0].cpu().numpy(), oc) and np.array_equal(out[1].cpu().numpy(), os_)


def test_static_scratch_limits(adl):
    """sizes beyond the array and shapes outside the path are refused with a clear error, nothing is launched"""
    mesh64 = cf.Mesh((2, 2, 2, 2), (cf.INTER | (0x0f << 8), cf.INTER | (0x0f << 8), cf.INTRA | (0x03 << 8), cf.INTRA | (0x03 << 8)))
    Bp, L, K = 64, 128, 64
    assert adl.num_signatures(mesh64) == K
    assert adl.chain_dp_static_bytes(Bp, L, mesh64) > adl.STATIC_SCRATCH_BYTES
    d_T = torch.zeros((Bp, L, K, K), dtype=torch.int64, device="cuda")
    out = (torch.empty(Bp, dtype=torch.int64, device="cuda"), torch.empty((Bp, L), dtype=torch.int32, device="cuda"))
    with pytest.raises(RuntimeError, match="static array holds"):
        adl.chain_dp_static(d_T, mesh64, out)
    mesh36 = cf.Mesh((4, 4), (cf.INTER, cf.INTRA))
    with pytest.raises(RuntimeError, match="use autoddl_chain_dp"):             # L < 32
        adl.chain_dp_static(d_T[:1, :8, :36, :36].contiguous(), mesh36, (out[0][:1], out[1][:1, :8].contiguous()))
    assert adl.chain_dp_static_bytes(1, 8, mesh36) == 0
