"""Pins of the oracle's Metropolis-Hastings sampler (R19-R22).  No GPU.

The sampler is an algorithm with random draws, so it is pinned by what the paper and the mathematics fix:
  M1  the counter-based generator is splitmix64 (known answer; an independent implementation in configs.py)
  M2  the integer -ln(u) agrees with libm and is monotone
  M3  the chain's stationary law is P(S) ~ exp(-Cost(S) / tau) on chains small enough to enumerate
  M4  limits: tau = 0 never goes uphill ("if a new strategy has a lower cost ... it is immediately accepted");
      a very hot chain accepts (almost) everything
  M5  bookkeeping: best = min over the trajectory, costs re-evaluate through Cost(S) (R8), DP optimum <= best
  M6  an independent Python replay of the whole procedure (floating-point acceptance) reproduces the trajectory
  M7  the acceptance frequency of an uphill move is exp(-dC / tau) (PAPER.md:233 min(1, P(S_new) / P(S_old)))
"""
import math

import numpy as np
import pytest

from oracle import ref
from paper_2301_06813_b200 import configs as cf

MASK = (1 << 64) - 1


def _random_problem(rng, L, K, hi):
    T = rng.integers(0, hi, size=(1, L, K, K)).astype(np.int64)
    T[0, 0] = T[0, 0, 0][None, :]                      # T[0][i][j] does not depend on i (no producer)
    return T


def _all_costs(T1):
    """Cost(S) of every strategy, by plain enumeration (numpy, independent of the oracle's chain_cost)"""
    L, K, _ = T1.shape
    costs = {}
    idx = np.zeros(L, dtype=np.int64)
    for flat in range(K ** L):
        x = flat
        for l in range(L - 1, -1, -1):
            idx[l] = x % K
            x //= K
        c, prev = 0, 0
        for l in range(L):
            c += int(T1[l, prev, idx[l]])
            prev = idx[l]
        costs[tuple(idx.tolist())] = c
    return costs


# ---- M1 -----------------------------------------------------------------------------------------------
def test_rng_is_splitmix64():
    assert ref.rng(0, 1) == 0xE220A8397B1DCDAF                     # published first output of splitmix64(0)
    g = cf.SplitMix64(12345)
    for n in range(1, 50):
        assert ref.rng(12345, n) == g.next()
    # counter-based: any n directly
    g = cf.SplitMix64(7)
    outs = [g.next() for _ in range(1000)]
    assert ref.rng(7, 1000) == outs[-1] and ref.rng(7, 500) == outs[499]


# ---- M2 -----------------------------------------------------------------------------------------------
def test_neglog_matches_libm_and_is_monotone():
    rng = np.random.default_rng(0)
    xs = [1, 2, 3, 4, 5, 7, 8, 2**16, 2**16 + 1, 2**31 - 1, 2**31, 2**31 + 1, 2**32 - 1, 2**32]
    xs += [int(v) for v in rng.integers(1, 2**32, 3000)]
    xs += [int(2 ** e) for e in rng.uniform(0, 32, 2000)]
    for x in xs:
        got = ref.neglog_q16(x)
        want = -math.log(x / 2**32) * 65536
        assert abs(got - want) <= 2.0, (x, got, want)                # 2 units of 2^-16: truncated log2, truncated ln 2
    assert ref.neglog_q16(2**32) == 0 and ref.neglog_q16(0) == -1 and ref.neglog_q16(2**32 + 1) == -1
    srt = sorted(set(xs))
    vals = [ref.neglog_q16(x) for x in srt]
    assert all(a >= b for a, b in zip(vals, vals[1:]))


# ---- M3 -----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,K,tau,seed", [(2, 6, 400, 1), (3, 6, 250, 2), (1, 6, 300, 3), (2, 36, 500, 4)])
def test_stationary_law_is_boltzmann(L, K, tau, seed):
    rng = np.random.default_rng(seed)
    T = _random_problem(rng, L, K, 1000)
    costs = _all_costs(T[0])
    nsteps = 400_000
    init = np.zeros((1, 1, L), np.int32)
    *_, trace = ref.metropolis(T, init, nsteps, tau, seed=seed, want_trace=True)
    tr = trace[0, 0, nsteps // 20:]                                  # drop burn-in
    # law of the cost under P(S) ~ exp(-Cost(S) / tau)
    w = {}
    for c in costs.values():
        w[c] = w.get(c, 0.0) + math.exp(-c / tau)
    Z = sum(w.values())
    vals, cnt = np.unique(tr, return_counts=True)
    emp = dict(zip(vals.tolist(), (cnt / len(tr)).tolist()))
    assert set(emp) <= set(w)                                        # only real costs are ever visited
    tv = 0.5 * sum(abs(emp.get(c, 0.0) - w[c] / Z) for c in w)
    assert tv < 0.03, tv
    mean_emp = float(tr.mean())
    mean_th = sum(c * w[c] for c in w) / Z
    assert abs(mean_emp - mean_th) < 0.03 * mean_th + 5


# ---- M4 -----------------------------------------------------------------------------------------------
def test_limits_greedy_and_hot():
    rng = np.random.default_rng(5)
    T = _random_problem(rng, 6, 36, 10**6)
    init = rng.integers(0, 36, size=(1, 3, 6)).astype(np.int32)
    bc, bs, fc, fs, acc, trace = ref.metropolis(T, init, 5000, 0, seed=9, want_trace=True)
    for r in range(3):
        c0 = ref.chain_cost(T[0], init[0, r])
        full = np.concatenate([[c0], trace[0, r]])
        assert (np.diff(full) <= 0).all()                            # tau = 0: never uphill
        assert bc[0, r] == fc[0, r] == full[-1]
    small = _random_problem(rng, 6, 36, 1000)
    *_, acc = ref.metropolis(small, init, 5000, (1 << 39), seed=9)
    assert (acc >= 4990).all()                                       # exp(-dC / tau) ~ 1 - 2e-9


# ---- M5 -----------------------------------------------------------------------------------------------
def test_bookkeeping_and_dp_bound():
    w = cf.config4_batched(Bp=3, L=12, seed=4)
    T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
    init = np.zeros((3, 4, 12), np.int32)
    init[:] = cf.Workload(w.name, w.layers, w.mesh, w.net, S=4, seed=4).cd_init()
    dp, _ = ref.chain_dp(T)
    tau = int(np.median(T[T < (1 << 50)])) // 4 + 1
    bc, bs, fc, fs, acc, trace = ref.metropolis(T, init, 3000, tau, seed=11, want_trace=True)
    for p in range(3):
        for r in range(4):
            c0 = ref.chain_cost(T[p], init[p, r])
            assert bc[p, r] == min(c0, int(trace[p, r].min()))
            assert ref.chain_cost(T[p], bs[p, r]) == bc[p, r]
            assert ref.chain_cost(T[p], fs[p, r]) == fc[p, r] == trace[p, r, -1]
            assert dp[p] <= bc[p, r]
            assert 0 < acc[p, r] <= 3000
    # chains are independent of how many run beside them: chain id = p * S + r
    b1 = ref.metropolis(T[:1], init[:1, :2], 3000, tau, seed=11)
    assert np.array_equal(b1[0], bc[:1, :2]) and np.array_equal(b1[3], fs[:1, :2])
    # zero steps: the start is returned
    z = ref.metropolis(T, init, 0, tau, seed=11)
    assert np.array_equal(z[1], init) and np.array_equal(z[3], init) and (z[4] == 0).all()


# ---- M6 -----------------------------------------------------------------------------------------------
def _py_rng(seed, n):
    z = (seed + n * 0x9E3779B97F4A7C15) & MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK
    return z ^ (z >> 31)


def test_python_replay_reproduces_the_trajectory():
    """PAPER.md:231-233 written out in Python with a floating-point acceptance test; draws whose uniform lies
    within 1e-4 (relative) of the acceptance probability are too close to call in floating point: there the replay
    follows the oracle (there must be very few of them)"""
    rng = np.random.default_rng(21)
    L, K, S, nsteps, tau, seed = 5, 36, 3, 4000, 700, 77
    T = _random_problem(rng, L, K, 3000)
    init = rng.integers(0, K, size=(1, S, L)).astype(np.int32)
    bc, bs, fc, fs, acc, trace = ref.metropolis(T, init, nsteps, tau, seed=seed, want_trace=True)
    T1 = T[0]
    compared = undecided = 0
    for r in range(S):
        s = init[0, r].tolist()
        cur = ref.chain_cost(T1, s)
        for t in range(nsteps):
            base = ((r << 32) + t) * 4
            l = _py_rng(seed, base + 1) % L
            c = _py_rng(seed, base + 2) % K
            u = ((_py_rng(seed, base + 3) >> 32) + 1) / 2**32
            new = list(s)
            new[l] = c
            cost_new = 0
            prev = 0
            for ll in range(L):                                    # Cost(S_new) from scratch, not incrementally
                cost_new += int(T1[ll, prev, new[ll]])
                prev = new[ll]
            d = cost_new - cur
            prob = 1.0 if d <= 0 else math.exp(-d / tau)
            if d > 0 and abs(u - prob) <= 1e-4 * prob + 1e-12:
                undecided += 1                                      # undecidable in floating point
                if trace[0, r, t] == cost_new:
                    s, cur = new, cost_new
                continue
            if u <= prob:
                s, cur = new, cost_new
            assert trace[0, r, t] == cur, (r, t)
            compared += 1
        assert s == fs[0, r].tolist() and cur == fc[0, r]
    assert undecided <= 5 and compared >= S * nsteps - 5


# ---- M7 -----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d,tau", [(100, 100), (1000, 250), (3, 1000), (5000, 700)])
def test_acceptance_frequency(d, tau):
    xs = np.random.default_rng(3).integers(1, 2**32 + 1, 200_000)
    acc = sum(1 for x in xs if tau * ref.neglog_q16(int(x)) >= (d << 16))
    p = math.exp(-d / tau)
    assert abs(acc / len(xs) - p) < 4 * math.sqrt(p * (1 - p) / len(xs)) + 2e-4
