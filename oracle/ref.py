"""ctypes loader for the CPU oracle (oracle/autoddl_ref.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, bench.py's cpu_baseline / --impl reference legs and __graft_entry__.smoke() may
import this.  It never touches the CUDA library and takes numpy (host) arrays only.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# AUTODDL_REF_SO: tests/test_oracle_mutations.py points the pins at a deliberately broken build of the oracle
_SO = os.environ.get("AUTODDL_REF_SO") or os.path.join(_HERE, "libautoddl_ref.so")
_SRC = os.path.join(_HERE, "autoddl_ref.cpp")


def build(force: bool = False) -> str:
    """Compile the oracle with plain g++ -O2 (never tuned)."""
    hdr = os.path.join(_HERE, "autoddl_ref.h")
    if os.environ.get("AUTODDL_REF_SO"):
        return _SO
    stale = (not os.path.exists(_SO)) or any(os.path.getmtime(f) > os.path.getmtime(_SO) for f in (_SRC, hdr))
    if force or stale:
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", _SO])
    return _SO


class RefMesh(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("size", C.c_int32 * 8), ("link", C.c_int32 * 8)]


class RefNet(C.Structure):
    _fields_ = [("alpha_ps", C.c_int64 * 2), ("beta_ps_per_byte", C.c_int64 * 2), ("mem_cap_bytes", C.c_int64),
                ("micro_batches", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        i64, i32, vp = C.c_int64, C.c_int32, C.c_void_p
        L.autoddl_ref_num_signatures.restype = C.c_int
        L.autoddl_ref_num_signatures.argtypes = [vp]
        L.autoddl_ref_collective.restype = i64
        L.autoddl_ref_collective.argtypes = [C.c_int, i64, i64, i64, i64]
        L.autoddl_ref_local_size.restype = i64
        L.autoddl_ref_local_size.argtypes = [i64, i64, vp, vp]
        L.autoddl_ref_sig_states.restype = C.c_int
        L.autoddl_ref_sig_states.argtypes = [C.c_int, C.c_int, vp, vp, vp, vp]
        L.autoddl_ref_reshard.restype = i64
        L.autoddl_ref_reshard.argtypes = [i64, i64, i64, vp, vp, vp, vp]
        L.autoddl_ref_edge_cost.restype = i64
        L.autoddl_ref_edge_cost.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp]
        L.autoddl_ref_node_cost.restype = i64
        L.autoddl_ref_node_cost.argtypes = [vp, C.c_int, vp, vp]
        L.autoddl_ref_feasible.restype = C.c_int
        L.autoddl_ref_feasible.argtypes = [vp, C.c_int, i32, vp, vp]
        L.autoddl_ref_layer_mem.restype = i64
        L.autoddl_ref_layer_mem.argtypes = [vp, C.c_int, vp]
        L.autoddl_ref_build_tables.restype = C.c_int
        L.autoddl_ref_build_tables.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp]
        L.autoddl_ref_chain_cost.restype = i64
        L.autoddl_ref_chain_cost.argtypes = [vp, i32, i32, vp]
        L.autoddl_ref_chain_dp.restype = C.c_int
        L.autoddl_ref_chain_dp.argtypes = [vp, i32, i32, i32, vp, vp]
        L.autoddl_ref_brute_force.restype = C.c_int
        L.autoddl_ref_brute_force.argtypes = [vp, i32, i32, vp, vp]
        L.autoddl_ref_coord_descent.restype = C.c_int
        L.autoddl_ref_coord_descent.argtypes = [vp, i32, i32, i32, vp, i32, i32, vp, vp, vp, vp]
        L.autoddl_ref_best_of_starts.restype = C.c_int
        L.autoddl_ref_best_of_starts.argtypes = [vp, i32, i32, vp, vp]
        L.autoddl_ref_segment_optima.restype = C.c_int
        L.autoddl_ref_segment_optima.argtypes = [vp, vp, vp, i32, i32, vp]
        L.autoddl_ref_stage_transfer.restype = C.c_int
        L.autoddl_ref_stage_transfer.argtypes = [vp, i32, vp, vp, vp]
        L.autoddl_ref_pipeline_partition.restype = C.c_int
        L.autoddl_ref_pipeline_partition.argtypes = [vp, vp, i32, i32, i32, vp, vp]
        L.autoddl_ref_segment_strategies.restype = C.c_int
        L.autoddl_ref_segment_strategies.argtypes = [vp, vp, vp, i32, i32, vp, i32, vp, vp]
        L.autoddl_ref_rng.restype = C.c_uint64
        L.autoddl_ref_rng.argtypes = [C.c_uint64, C.c_uint64]
        L.autoddl_ref_neglog_q16.restype = i64
        L.autoddl_ref_neglog_q16.argtypes = [C.c_uint64]
        L.autoddl_ref_metropolis.restype = C.c_int
        L.autoddl_ref_metropolis.argtypes = [vp, i32, i32, i32, vp, i32, i32, i64, C.c_uint64, vp, vp, vp, vp, vp, vp]
        _lib = L
    return _lib


def make_mesh(size, link) -> RefMesh:
    m = RefMesh()
    m.ndim = len(size)
    for d in range(len(size)):
        m.size[d] = int(size[d])
        m.link[d] = int(link[d])
    return m


def make_net(alpha_ps, beta_ps_per_byte, mem_cap_bytes=0, micro_batches=1) -> RefNet:
    n = RefNet()
    n.alpha_ps[0], n.alpha_ps[1] = int(alpha_ps[0]), int(alpha_ps[1])
    n.beta_ps_per_byte[0], n.beta_ps_per_byte[1] = int(beta_ps_per_byte[0]), int(beta_ps_per_byte[1])
    n.mem_cap_bytes = int(mem_cap_bytes)
    n.micro_batches = int(micro_batches)
    return n


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _st(v):
    return np.ascontiguousarray(np.asarray(v, dtype=np.int32))


def mesh_of(w) -> RefMesh:
    return make_mesh(w.mesh.size, w.mesh.link)


def net_of(w) -> RefNet:
    return make_net(w.net.alpha_ps, w.net.beta_ps_per_byte, w.net.mem_cap_bytes, getattr(w.net, "micro_batches", 1))


# ---- scalar pieces (for the pins) -------------------------------------------------------------
AG, RS, AR, A2A = 0, 1, 2, 3


def num_signatures(mesh: RefMesh) -> int:
    """K: 6^ndim for ndim <= 3; the product of the levels' allowed-row counts for ndim = 4, 5 (R26)"""
    return int(lib().autoddl_ref_num_signatures(C.addressof(mesh)))


def collective(which, n, p, alpha, beta) -> int:
    return int(lib().autoddl_ref_collective(which, n, p, alpha, beta))


def local_size(R, Cc, st, mesh: RefMesh) -> int:
    s = _st(st)
    return int(lib().autoddl_ref_local_size(R, Cc, _p(s), C.addressof(mesh)))


def sig_states(kind, sig, mesh: RefMesh):
    I = np.zeros(8, np.int32); W = np.zeros(8, np.int32); O = np.zeros(8, np.int32)
    v = lib().autoddl_ref_sig_states(kind, sig, C.addressof(mesh), _p(I), _p(W), _p(O))
    D = mesh.ndim
    return int(v), tuple(I[:D].tolist()), tuple(W[:D].tolist()), tuple(O[:D].tolist())


def reshard(rows, cols, eb, a, b, mesh: RefMesh, net: RefNet) -> int:
    aa, bb = _st(a), _st(b)
    return int(lib().autoddl_ref_reshard(rows, cols, eb, _p(aa), _p(bb), C.addressof(mesh), C.addressof(net)))


def edge_cost(prev_rec, cur_rec, i, j, mesh, net) -> int:
    a = np.ascontiguousarray(prev_rec).reshape(1); b = np.ascontiguousarray(cur_rec).reshape(1)
    return int(lib().autoddl_ref_edge_cost(_p(a), _p(b), i, j, C.addressof(mesh), C.addressof(net)))


def node_cost(rec, j, mesh, net) -> int:
    a = np.ascontiguousarray(rec).reshape(1)
    return int(lib().autoddl_ref_node_cost(_p(a), j, C.addressof(mesh), C.addressof(net)))


def feasible(rec, j, L, mesh, net) -> int:
    a = np.ascontiguousarray(rec).reshape(1)
    return int(lib().autoddl_ref_feasible(_p(a), j, L, C.addressof(mesh), C.addressof(net)))


def layer_mem(rec, j, mesh) -> int:
    a = np.ascontiguousarray(rec).reshape(1)
    return int(lib().autoddl_ref_layer_mem(_p(a), j, C.addressof(mesh)))


# ---- the three steps ---------------------------------------------------------------------------
def build_tables(layers: np.ndarray, mesh: RefMesh, net: RefNet):
    """layers: LAYER_DTYPE [Bp, L] -> T int64 [Bp,L,K,K], node int64 [Bp,L,K], mask uint8 [Bp,L,K]"""
    layers = np.ascontiguousarray(layers)
    Bp, L = layers.shape
    K = num_signatures(mesh)
    T = np.empty((Bp, L, K, K), np.int64)
    node = np.empty((Bp, L, K), np.int64)
    mask = np.empty((Bp, L, K), np.uint8)
    rc = lib().autoddl_ref_build_tables(_p(layers), Bp, L, C.addressof(mesh), C.addressof(net), _p(T), _p(node), _p(mask))
    assert rc == 0, rc
    return T, node, mask


def chain_cost(T1: np.ndarray, s) -> int:
    """T1: [L,K,K] of one problem"""
    T1 = np.ascontiguousarray(T1, dtype=np.int64)
    s = _st(s)
    return int(lib().autoddl_ref_chain_cost(_p(T1), T1.shape[0], T1.shape[1], _p(s)))


def chain_dp(T: np.ndarray):
    T = np.ascontiguousarray(T, dtype=np.int64)
    Bp, L, K, _ = T.shape
    cost = np.empty(Bp, np.int64)
    strat = np.empty((Bp, L), np.int32)
    rc = lib().autoddl_ref_chain_dp(_p(T), Bp, L, K, _p(cost), _p(strat))
    assert rc == 0, rc
    return cost, strat


def brute_force(T1: np.ndarray):
    T1 = np.ascontiguousarray(T1, dtype=np.int64)
    L, K, _ = T1.shape
    cost = np.empty(1, np.int64)
    strat = np.empty(L, np.int32)
    rc = lib().autoddl_ref_brute_force(_p(T1), L, K, _p(cost), _p(strat))
    assert rc == 0, rc
    return int(cost[0]), strat


def coord_descent(T: np.ndarray, init: np.ndarray, max_sweeps: int = 64, want_trace: bool = False):
    T = np.ascontiguousarray(T, dtype=np.int64)
    init = np.ascontiguousarray(init, dtype=np.int32)
    Bp, L, K, _ = T.shape
    S = init.shape[1]
    assert init.shape == (Bp, S, L)
    cost = np.empty((Bp, S), np.int64)
    strat = np.empty((Bp, S, L), np.int32)
    sweeps = np.empty((Bp, S), np.int32)
    trace = np.full((Bp, S, max_sweeps, L), -1, np.int64) if want_trace else None
    rc = lib().autoddl_ref_coord_descent(_p(T), Bp, L, K, _p(init), S, max_sweeps, _p(cost), _p(strat), _p(sweeps), _p(trace))
    assert rc == 0, rc
    if want_trace:
        return cost, strat, sweeps, trace
    return cost, strat, sweeps


def best_of_starts(cost: np.ndarray):
    """cost [Bp, S] -> (best cost [Bp], first start attaining it [Bp])"""
    cost = np.ascontiguousarray(cost, dtype=np.int64)
    Bp, S = cost.shape
    bc = np.empty(Bp, np.int64); bs = np.empty(Bp, np.int32)
    rc = lib().autoddl_ref_best_of_starts(_p(cost), Bp, S, _p(bc), _p(bs))
    assert rc == 0, rc
    return bc, bs


# ---- pipeline stages (R27) ----------------------------------------------------------
def segment_optima(T1: np.ndarray, node1: np.ndarray, mask1: np.ndarray) -> np.ndarray:
    """one problem: T1 [L,K,K], node1 [L,K], mask1 [L,K] -> tri [L, L+1] (C(a,b) for a < b, -1 elsewhere)"""
    T1 = np.ascontiguousarray(T1, dtype=np.int64); node1 = np.ascontiguousarray(node1, dtype=np.int64)
    mask1 = np.ascontiguousarray(mask1, dtype=np.uint8)
    L, K, _ = T1.shape
    tri = np.empty((L, L + 1), np.int64)
    rc = lib().autoddl_ref_segment_optima(_p(T1), _p(node1), _p(mask1), L, K, _p(tri))
    assert rc == 0, rc
    return tri


def stage_transfer(layers1: np.ndarray, mesh: RefMesh, net: RefNet) -> np.ndarray:
    layers1 = np.ascontiguousarray(layers1)
    L = layers1.shape[0]
    x = np.empty(L, np.int64)
    rc = lib().autoddl_ref_stage_transfer(_p(layers1), L, C.addressof(mesh), C.addressof(net), _p(x))
    assert rc == 0, rc
    return x


def pipeline_partition(tri: np.ndarray, xfer: np.ndarray, stages: int, objective: int):
    tri = np.ascontiguousarray(tri, dtype=np.int64); xfer = np.ascontiguousarray(xfer, dtype=np.int64)
    L = tri.shape[0]
    val = np.empty(1, np.int64); cuts = np.empty(stages + 1, np.int32)
    rc = lib().autoddl_ref_pipeline_partition(_p(tri), _p(xfer), L, stages, objective, _p(val), _p(cuts))
    assert rc == 0, rc
    return int(val[0]), cuts


def segment_strategies(T1, node1, mask1, cuts):
    T1 = np.ascontiguousarray(T1, dtype=np.int64); node1 = np.ascontiguousarray(node1, dtype=np.int64)
    mask1 = np.ascontiguousarray(mask1, dtype=np.uint8); cuts = np.ascontiguousarray(cuts, dtype=np.int32)
    L, K, _ = T1.shape
    stages = len(cuts) - 1
    sc = np.empty(stages, np.int64); st = np.empty(L, np.int32)
    rc = lib().autoddl_ref_segment_strategies(_p(T1), _p(node1), _p(mask1), L, K, _p(cuts), stages, _p(sc), _p(st))
    assert rc == 0, rc
    return sc, st


# ---- Metropolis-Hastings -------------------------------------------------------------
def rng(seed: int, n: int) -> int:
    return int(lib().autoddl_ref_rng(seed, n))


def neglog_q16(x: int) -> int:
    return int(lib().autoddl_ref_neglog_q16(x))


def metropolis(T: np.ndarray, init: np.ndarray, nsteps: int, tau_ps: int, seed: int = 0, want_trace: bool = False):
    """-> best_cost [Bp,S], best_strategy [Bp,S,L], final_cost [Bp,S], final_strategy [Bp,S,L], accepted [Bp,S] (, trace [Bp,S,nsteps])"""
    T = np.ascontiguousarray(T, dtype=np.int64)
    init = np.ascontiguousarray(init, dtype=np.int32)
    Bp, L, K, _ = T.shape
    S = init.shape[1]
    assert init.shape == (Bp, S, L)
    bc = np.empty((Bp, S), np.int64); fc = np.empty((Bp, S), np.int64)
    bs = np.empty((Bp, S, L), np.int32); fs = np.empty((Bp, S, L), np.int32)
    acc = np.empty((Bp, S), np.int32)
    trace = np.empty((Bp, S, nsteps), np.int64) if want_trace else None
    rc = lib().autoddl_ref_metropolis(_p(T), Bp, L, K, _p(init), S, nsteps, tau_ps, seed, _p(bc), _p(bs), _p(fc), _p(fs), _p(acc), _p(trace))
    assert rc == 0, rc
    if want_trace:
        return bc, bs, fc, fs, acc, trace
    return bc, bs, fc, fs, acc


# ---- alpha-beta calibration (Table 2) ---------------------------------------
def fit_design_matrix(kind: np.ndarray, p: np.ndarray, nbytes: np.ndarray) -> np.ndarray:
    """rows (A_i, B_i) of the linear system t_i = A_i alpha + B_i beta, Table 2 as printed (real-valued (p-1)/p n):
    AllGather / ReduceScatter: (p-1, (p-1)/p n); AllReduce: (2p-1, 2 (p-1)/p n); AlltoAll: (p-1, n)"""
    kind = np.asarray(kind); p = np.asarray(p, dtype=np.float64); n = np.asarray(nbytes, dtype=np.float64)
    A = np.where(kind == AR, 2 * p - 1, p - 1)
    B = np.where(kind == AR, 2 * (p - 1) / p * n, np.where(kind == A2A, n, (p - 1) / p * n))
    return np.stack([A, B], axis=1)


def fit_alpha_beta(kind, p, nbytes, t):
    """least-squares (alpha, beta) from timed collectives: the definition, solved by numpy.linalg.lstsq (SVD) in fp64"""
    X = fit_design_matrix(kind, p, nbytes)
    sol, *_ = np.linalg.lstsq(X, np.asarray(t, dtype=np.float64), rcond=None)
    return float(sol[0]), float(sol[1])
