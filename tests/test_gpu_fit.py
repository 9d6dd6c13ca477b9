"""Parity of autoddl_fit_alpha_beta against the oracle's least-squares solution (numpy lstsq, fp64).
Floating point: the tolerance is relative 1e-9 on exact data (both sides are accurate to ~1e-13 there; the normal
equations square the condition number, which the column scaling keeps near 1e2) and 1e-7 on noisy data."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def adl():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_2301_06813_b200 import binding
    binding.lib()
    return binding


def _data(rng, n, alpha, beta, noise):
    kind = rng.integers(0, 4, n).astype(np.int32)
    p = rng.choice([2, 3, 4, 8, 16, 32, 64], n).astype(np.int32)
    nbytes = (2 ** rng.uniform(10, 30, n)).astype(np.int64)
    X = ref.fit_design_matrix(kind, p, nbytes)
    t = X[:, 0] * alpha + X[:, 1] * beta
    if noise:
        t = t * (1 + noise * rng.standard_normal(n))
    return kind, p, nbytes, t


@pytest.mark.parametrize("n,noise,tol", [(2, 0.0, 1e-9), (7, 0.0, 1e-9), (1000, 0.0, 1e-9), (100_003, 0.05, 1e-7), (4_000_000, 0.02, 1e-7)])
def test_fit_matches_lstsq(adl, n, noise, tol):
    rng = np.random.default_rng(n)
    kind, p, nb, t = _data(rng, n, 5e-6, 1 / 25e9, noise)
    if n == 2:
        kind[:] = [ref.AG, ref.A2A]                       # two independent rows
        t = ref.fit_design_matrix(kind, p, nb) @ np.array([5e-6, 1 / 25e9])
    want = ref.fit_alpha_beta(kind, p, nb, t)
    got = adl.fit_alpha_beta(*(torch.from_numpy(x).cuda() for x in (kind, p, nb, t))).cpu().numpy()
    assert abs(got[0] / want[0] - 1) < tol and abs(got[1] / want[1] - 1) < tol, (got, want)
    again = adl.fit_alpha_beta(*(torch.from_numpy(x).cuda() for x in (kind, p, nb, t))).cpu().numpy()
    assert np.array_equal(got, again)                      # deterministic
