"""Pins of the oracle's alpha-beta calibration ("we can formulate a linear system in terms of alpha and
beta for each network, as shown in Table 2 ... least squares").  No GPU."""
import numpy as np

from oracle import ref


def _measurements(rng, n, alpha, beta, noise=0.0):
    kind = rng.integers(0, 4, n).astype(np.int32)
    p = rng.choice([2, 3, 4, 8, 16, 32, 64], n).astype(np.int32)
    nbytes = (2 ** rng.uniform(10, 30, n)).astype(np.int64)
    X = ref.fit_design_matrix(kind, p, nbytes)
    t = X[:, 0] * alpha + X[:, 1] * beta
    if noise:
        t = t * (1 + noise * rng.standard_normal(n))
    return kind, p, nbytes, t


def test_design_matrix_is_table2():
    # hand values, PAPER.md:104-106 with p = 4, n = 2^20: AG/RS (3, 786432); AR (7, 1572864); A2A (3, 1048576)
    X = ref.fit_design_matrix([ref.AG, ref.RS, ref.AR, ref.A2A], [4, 4, 4, 4], [2**20] * 4)
    assert X.tolist() == [[3, 786432], [3, 786432], [7, 1572864], [3, 1048576]]
    # consistent with the integer cost model when p divides n (R3)
    for k in (ref.AG, ref.RS, ref.AR, ref.A2A):
        a, b = ref.fit_design_matrix([k], [8], [2**20])[0]
        assert ref.collective(k, 2**20, 8, 5_000_000, 3) == a * 5_000_000 + b * 3


def test_exact_recovery_and_normal_equations():
    rng = np.random.default_rng(0)
    kind, p, nb, t = _measurements(rng, 5000, 5e-6, 1 / 25e9)
    a, b = ref.fit_alpha_beta(kind, p, nb, t)
    assert abs(a / 5e-6 - 1) < 1e-9 and abs(b * 25e9 - 1) < 1e-9
    # noisy data: the solution satisfies the normal equations X^T (X s - t) = 0 (the definition of least squares)
    kind, p, nb, t = _measurements(rng, 20000, 2e-5, 1 / 12.5e9, noise=0.05)
    a, b = ref.fit_alpha_beta(kind, p, nb, t)
    X = ref.fit_design_matrix(kind, p, nb)
    g = X.T @ (X @ np.array([a, b]) - t)
    scale = np.abs(X).T @ np.abs(t)
    assert (np.abs(g) < 1e-9 * scale).all()
    assert abs(a / 2e-5 - 1) < 0.2 and abs(b * 12.5e9 - 1) < 0.01
    # two measurements determine the line exactly
    a, b = ref.fit_alpha_beta([ref.AG, ref.A2A], [2, 2], [1000, 3000], [1 * 7.0 + 500 * 2.0, 1 * 7.0 + 3000 * 2.0])
    assert abs(a - 7) < 1e-9 and abs(b - 2) < 1e-12
