"""Thin ctypes binding over the C-ABI library (include/autoddl.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of libautoddl.so.  torch is used for device memory
and streams.  There is no CPU fallback: if the library is missing or there is no CUDA device the
calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from .configs import LAYER_DTYPE, Workload

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libautoddl.so")

EXPORTS = [
    "autoddl_num_signatures", "autoddl_workspace_bytes", "autoddl_build_tables", "autoddl_chain_dp",
    "autoddl_chain_dp_static", "autoddl_chain_dp_static_bytes", "autoddl_coord_descent", "autoddl_metropolis", "autoddl_search", "autoddl_search_host", "autoddl_fit_workspace_bytes", "autoddl_fit_alpha_beta", "autoddl_best_of_starts", "autoddl_pipeline_workspace_bytes", "autoddl_segment_optima", "autoddl_stage_transfer",
    "autoddl_pipeline_partition", "autoddl_segment_strategies", "autoddl_copy_probe", "autoddl_store_probe", "autoddl_profile_mark", "autoddl_launch_count",
    "autoddl_last_error",
]


class AutoddlError(RuntimeError):
    pass


class CMesh(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("size", C.c_int32 * 8), ("link", C.c_int32 * 8)]


class CNet(C.Structure):
    _fields_ = [("alpha_ps", C.c_int64 * 2), ("beta_ps_per_byte", C.c_int64 * 2), ("mem_cap_bytes", C.c_int64),
                ("micro_batches", C.c_int64)]


_lib = None


def lib():
    """Loads libautoddl.so; raises if it has not been built (python -m paper_2301_06813_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise AutoddlError(f"{LIB_PATH} not found: build it with `python paper_2301_06813_b200/build.py` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t
        L.autoddl_num_signatures.restype = C.c_int
        L.autoddl_num_signatures.argtypes = [vp]
        L.autoddl_workspace_bytes.restype = sz
        L.autoddl_workspace_bytes.argtypes = [i32, i32, i32, vp]
        L.autoddl_build_tables.restype = C.c_int
        L.autoddl_build_tables.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp]
        L.autoddl_chain_dp.restype = C.c_int
        L.autoddl_chain_dp.argtypes = [vp, i32, i32, vp, vp, vp, vp, sz, vp, vp, vp]
        L.autoddl_chain_dp_static.restype = C.c_int
        L.autoddl_chain_dp_static.argtypes = [vp, i32, i32, vp, vp, vp, vp]
        L.autoddl_chain_dp_static_bytes.restype = sz
        L.autoddl_chain_dp_static_bytes.argtypes = [i32, i32, vp]
        L.autoddl_coord_descent.restype = C.c_int
        L.autoddl_coord_descent.argtypes = [vp, i32, i32, vp, vp, vp, vp, sz, vp, i32, i32, vp, vp, vp, vp]
        L.autoddl_metropolis.restype = C.c_int
        L.autoddl_metropolis.argtypes = [vp, i32, i32, vp, vp, i32, i32, i64, C.c_uint64, vp, vp, vp, vp, vp, vp]
        L.autoddl_search.restype = C.c_int
        L.autoddl_search.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp, vp, vp, i32, i32, vp, vp, vp, vp]
        L.autoddl_search_host.restype = C.c_int
        L.autoddl_search_host.argtypes = [vp, i32, i32, vp, vp, vp, i32, i32, vp, sz, vp, vp, vp, vp, vp, vp]
        L.autoddl_best_of_starts.restype = C.c_int
        L.autoddl_best_of_starts.argtypes = [vp, i32, i32, vp, vp, vp]
        L.autoddl_pipeline_workspace_bytes.restype = sz
        L.autoddl_pipeline_workspace_bytes.argtypes = [i32, i32, i32]
        L.autoddl_segment_optima.restype = C.c_int
        L.autoddl_segment_optima.argtypes = [vp, vp, vp, i32, vp, vp, vp]
        L.autoddl_stage_transfer.restype = C.c_int
        L.autoddl_stage_transfer.argtypes = [vp, i32, vp, vp, vp, vp]
        L.autoddl_pipeline_partition.restype = C.c_int
        L.autoddl_pipeline_partition.argtypes = [vp, vp, i32, i32, i32, vp, sz, vp, vp, vp]
        L.autoddl_segment_strategies.restype = C.c_int
        L.autoddl_segment_strategies.argtypes = [vp, vp, vp, i32, vp, vp, i32, vp, sz, vp, vp, vp]
        L.autoddl_store_probe.restype = C.c_int
        L.autoddl_store_probe.argtypes = [vp, i32, i32, i32, vp]
        L.autoddl_copy_probe.restype = C.c_int
        L.autoddl_copy_probe.argtypes = [vp, vp, sz, vp]
        L.autoddl_fit_workspace_bytes.restype = sz
        L.autoddl_fit_workspace_bytes.argtypes = []
        L.autoddl_fit_alpha_beta.restype = C.c_int
        L.autoddl_fit_alpha_beta.argtypes = [vp, vp, vp, vp, i64, vp, vp, sz, vp]
        L.autoddl_profile_mark.restype = C.c_int
        L.autoddl_profile_mark.argtypes = [vp]
        L.autoddl_launch_count.restype = i64
        L.autoddl_launch_count.argtypes = []
        L.autoddl_last_error.restype = C.c_char_p
        L.autoddl_last_error.argtypes = []
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise AutoddlError(f"autoddl error {rc}: {lib().autoddl_last_error().decode()}")


def c_mesh(mesh) -> CMesh:
    m = CMesh()
    m.ndim = len(mesh.size)                       # ndim outside 1..8 is rejected by the library
    for d in range(min(m.ndim, 8)):
        m.size[d] = int(mesh.size[d])
        m.link[d] = int(mesh.link[d])
    return m


def c_net(net) -> CNet:
    n = CNet()
    for c in range(2):
        n.alpha_ps[c] = int(net.alpha_ps[c])
        n.beta_ps_per_byte[c] = int(net.beta_ps_per_byte[c])
    n.mem_cap_bytes = int(net.mem_cap_bytes)
    n.micro_batches = int(getattr(net, "micro_batches", 1))
    return n


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _ptr(t, dtype=None, name="tensor"):
    """device pointer of a tensor the library will read or write as raw memory: it must live on a CUDA device, be
    contiguous and have exactly the dtype the C-ABI states (the library cannot see any of this)"""
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise AutoddlError(f"{name}: expected a CUDA tensor")
    if not t.is_contiguous():
        raise AutoddlError(f"{name}: tensor must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise AutoddlError(f"{name}: dtype {t.dtype}, the C-ABI needs {dtype}")
    return t.data_ptr()


def _hptr(a, dtype, name):
    """host pointer of a numpy array handed to the host entry point: C-contiguous, exact dtype"""
    if a is None:
        return None
    if not isinstance(a, np.ndarray) or not a.flags["C_CONTIGUOUS"]:
        raise AutoddlError(f"{name}: expected a C-contiguous numpy array")
    if a.dtype != dtype:
        raise AutoddlError(f"{name}: dtype {a.dtype}, the C-ABI needs {np.dtype(dtype)}")
    return a.ctypes.data


I64, I32, U8, F64 = torch.int64, torch.int32, torch.uint8, torch.float64


def layers_to_device(layers: np.ndarray, device="cuda") -> torch.Tensor:
    """LAYER_DTYPE [Bp, L] -> uint8 device tensor [Bp, L, 64]"""
    assert layers.dtype == LAYER_DTYPE
    raw = np.ascontiguousarray(layers).view(np.uint8).reshape(layers.shape + (64,))
    return torch.from_numpy(raw).to(device)


def num_signatures(mesh) -> int:
    m = c_mesh(mesh)
    k = lib().autoddl_num_signatures(C.addressof(m))
    if k < 0:
        _check(k)
    return k


def workspace_bytes(Bp: int, L: int, S: int, mesh) -> int:
    m = c_mesh(mesh)
    return int(lib().autoddl_workspace_bytes(Bp, L, S, C.addressof(m)))


def build_tables(d_layers: torch.Tensor, mesh, net, want_node_mask: bool = True, out=None):
    """(a1) -> T int64 [Bp,L,K,K], node int64 [Bp,L,K] | None, mask uint8 [Bp,L,K] | None (device tensors)"""
    Bp, L = d_layers.shape[0], d_layers.shape[1]
    K = num_signatures(mesh)
    dev = d_layers.device
    T = out if out is not None else torch.empty((Bp, L, K, K), dtype=torch.int64, device=dev)
    node = torch.empty((Bp, L, K), dtype=torch.int64, device=dev) if want_node_mask else None
    mask = torch.empty((Bp, L, K), dtype=torch.uint8, device=dev) if want_node_mask else None
    m, n = c_mesh(mesh), c_net(net)
    _check(lib().autoddl_build_tables(_ptr(d_layers, U8, "d_layers"), Bp, L, C.addressof(m), C.addressof(n), _ptr(T, I64, "T"),
                                      _ptr(node, I64, "node"), _ptr(mask, U8, "mask"), _stream()))
    return T, node, mask


def chain_dp(T: torch.Tensor | None, mesh, net=None, d_layers=None, work: torch.Tensor | None = None, out=None):
    """(a2) -> opt_cost int64 [Bp], strategy int32 [Bp, L] (device tensors)"""
    if T is not None:
        Bp, L = T.shape[0], T.shape[1]
        dev = T.device
    else:
        Bp, L = d_layers.shape[0], d_layers.shape[1]
        dev = d_layers.device
    if work is None:
        K = num_signatures(mesh)
        if T is None:
            need = workspace_bytes(Bp, L, 0, mesh)
        else:
            need = Bp * L * K + 256 if L * K > 16384 else 0
        work = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    if out is None:
        cost = torch.empty(Bp, dtype=torch.int64, device=dev)
        strat = torch.empty((Bp, L), dtype=torch.int32, device=dev)
    else:
        cost, strat = out
    m = c_mesh(mesh)
    n = c_net(net) if net is not None else None
    _check(lib().autoddl_chain_dp(_ptr(d_layers, U8, "d_layers"), Bp, L, C.addressof(m), C.addressof(n) if n is not None else None,
                                  _ptr(T, I64, "T"), _ptr(work, U8, "work"), work.numel(), _ptr(cost, I64, "opt_cost"),
                                  _ptr(strat, I32, "strategy"), _stream()))
    return cost, strat


def coord_descent(T: torch.Tensor | None, init: torch.Tensor, mesh, max_sweeps: int = 64, net=None, d_layers=None,
                  work: torch.Tensor | None = None, out=None):
    """(a3) init int32 [Bp,S,L] -> cost int64 [Bp,S], strategy int32 [Bp,S,L], sweeps int32 [Bp,S]"""
    Bp, S, L = init.shape
    dev = init.device
    if T is None and work is None:
        K = num_signatures(mesh)
        work = torch.empty(Bp * L * K * K * 8 + 256, dtype=torch.uint8, device=dev)
    if out is None:
        cost = torch.empty((Bp, S), dtype=torch.int64, device=dev)
        strat = torch.empty((Bp, S, L), dtype=torch.int32, device=dev)
        sweeps = torch.empty((Bp, S), dtype=torch.int32, device=dev)
    else:
        cost, strat, sweeps = out
    m = c_mesh(mesh)
    n = c_net(net) if net is not None else None
    _check(lib().autoddl_coord_descent(_ptr(d_layers, U8, "d_layers"), Bp, L, C.addressof(m), C.addressof(n) if n is not None else None,
                                       _ptr(T, I64, "T"), _ptr(work, U8, "work"), work.numel() if work is not None else 0,
                                       _ptr(init, I32, "init"), S, max_sweeps, _ptr(cost, I64, "cost"), _ptr(strat, I32, "strategy"),
                                       _ptr(sweeps, I32, "sweeps"), _stream()))
    return cost, strat, sweeps


def metropolis(T: torch.Tensor, init: torch.Tensor, mesh, nsteps: int, tau_ps: int, seed: int = 0, out=None):
    """Metropolis-Hastings chains on the tables -> best_cost [Bp,S], best_strategy [Bp,S,L], final_cost [Bp,S],
    final_strategy [Bp,S,L], accepted [Bp,S] (device tensors)"""
    Bp, S, L = init.shape
    dev = init.device
    if out is None:
        out = (torch.empty((Bp, S), dtype=torch.int64, device=dev), torch.empty((Bp, S, L), dtype=torch.int32, device=dev),
               torch.empty((Bp, S), dtype=torch.int64, device=dev), torch.empty((Bp, S, L), dtype=torch.int32, device=dev),
               torch.empty((Bp, S), dtype=torch.int32, device=dev))
    bc, bs, fc, fs, acc = out
    m = c_mesh(mesh)
    _check(lib().autoddl_metropolis(_ptr(T, I64, "T"), Bp, L, C.addressof(m), _ptr(init, I32, "init"), S, nsteps, tau_ps, seed,
                                    _ptr(bc, I64, "best_cost"), _ptr(bs, I32, "best_strategy"), _ptr(fc, I64, "final_cost"),
                                    _ptr(fs, I32, "final_strategy"), _ptr(acc, I32, "accepted"), _stream()))
    return out


def fit_alpha_beta(kind: torch.Tensor, p: torch.Tensor, nbytes: torch.Tensor, t: torch.Tensor, out=None, work=None):
    """alpha-beta calibration: kind int32 [N], p int32 [N], nbytes int64 [N], t float64 [N] (device) -> float64 [2] (device)"""
    N = kind.numel()
    dev = kind.device
    if out is None:
        out = torch.empty(2, dtype=torch.float64, device=dev)
    if work is None:
        work = torch.empty(int(lib().autoddl_fit_workspace_bytes()), dtype=torch.uint8, device=dev)
    _check(lib().autoddl_fit_alpha_beta(_ptr(kind, I32, "kind"), _ptr(p, I32, "p"), _ptr(nbytes, I64, "nbytes"), _ptr(t, F64, "t"), N,
                                        _ptr(out, F64, "out"), _ptr(work, U8, "work"), work.numel(), _stream()))
    return out


STATIC_SCRATCH_BYTES = 8 << 20   # AUTODDL_STATIC_SCRATCH_BYTES


def chain_dp_static_bytes(Bp: int, L: int, mesh) -> int:
    m = c_mesh(mesh)
    return int(lib().autoddl_chain_dp_static_bytes(Bp, L, C.addressof(m)))


def chain_dp_static(T: torch.Tensor, mesh, out):
    """(a2) on tables with K <= 64 with the scratch in the library's static device array (autoddl_chain_dp_static): no
    allocation here or in the library -- `out` = (opt_cost int64 [Bp], strategy int32 [Bp, L]) is the caller's."""
    Bp, L = T.shape[0], T.shape[1]
    m = c_mesh(mesh)
    _check(lib().autoddl_chain_dp_static(_ptr(T, I64, "T"), Bp, L, C.addressof(m), _ptr(out[0], I64, "opt_cost"),
                                         _ptr(out[1], I32, "strategy"), _stream()))
    return out


def best_of_starts(cost: torch.Tensor, out=None):
    """cost int64 [Bp, S] (device) -> best_cost int64 [Bp], best_start int32 [Bp]: smallest cost, smallest start on ties"""
    Bp, S = cost.shape
    if out is None:
        out = (torch.empty(Bp, dtype=torch.int64, device=cost.device), torch.empty(Bp, dtype=torch.int32, device=cost.device))
    _check(lib().autoddl_best_of_starts(_ptr(cost, I64, "cost"), Bp, S, _ptr(out[0], I64, "best_cost"), _ptr(out[1], I32, "best_start"), _stream()))
    return out


def pipeline_stages(d_layers1: torch.Tensor, T1: torch.Tensor, node1: torch.Tensor, mask1: torch.Tensor, mesh, net, stages: int,
                    objective: int = 1):
    """Pipeline-stage enumeration of ONE chain whose tables (T1 [L,K,K], node1 [L,K], mask1 [L,K]; d_layers1 [L,64]) were
    built on the stage sub-mesh `mesh`: -> dict(tri [L, L+1], xfer [L], value [1], cuts [stages+1], seg_cost [stages],
    strategy [L]) -- four kernels, no host synchronisation in between."""
    L, K = T1.shape[0], T1.shape[1]
    dev = T1.device
    m, n = c_mesh(mesh), c_net(net)
    tri = torch.empty((L, L + 1), dtype=torch.int64, device=dev)
    xfer = torch.empty(L, dtype=torch.int64, device=dev)
    value = torch.empty(1, dtype=torch.int64, device=dev)
    cuts = torch.empty(stages + 1, dtype=torch.int32, device=dev)
    seg_cost = torch.empty(stages, dtype=torch.int64, device=dev)
    strategy = torch.empty(L, dtype=torch.int32, device=dev)
    work = torch.empty(int(lib().autoddl_pipeline_workspace_bytes(L, K, stages)), dtype=torch.uint8, device=dev)
    _check(lib().autoddl_segment_optima(_ptr(T1, I64, "T"), _ptr(node1, I64, "node"), _ptr(mask1, U8, "mask"), L, C.addressof(m),
                                        _ptr(tri), _stream()))
    _check(lib().autoddl_stage_transfer(_ptr(d_layers1, U8, "d_layers"), L, C.addressof(m), C.addressof(n), _ptr(xfer), _stream()))
    _check(lib().autoddl_pipeline_partition(_ptr(tri), _ptr(xfer), L, stages, objective, _ptr(work), work.numel(), _ptr(value),
                                            _ptr(cuts), _stream()))
    _check(lib().autoddl_segment_strategies(_ptr(T1, I64, "T"), _ptr(node1, I64, "node"), _ptr(mask1, U8, "mask"), L, C.addressof(m),
                                            _ptr(cuts), stages, _ptr(work), work.numel(), _ptr(seg_cost), _ptr(strategy), _stream()))
    return dict(tri=tri, xfer=xfer, value=value, cuts=cuts, seg_cost=seg_cost, strategy=strategy)


def profile_mark(event: "torch.cuda.Event | None"):
    """the next search() records `event` between tables + DP and Coordinate Descent (the event must have been recorded
    once before so that its handle exists)"""
    _check(lib().autoddl_profile_mark(None if event is None else event.cuda_event))


def search(d_layers: torch.Tensor, mesh, net, init: torch.Tensor | None = None, max_sweeps: int = 64,
           want_tables: bool = True, want_node_mask: bool = False, work: torch.Tensor | None = None, out=None):
    """Whole path on device tensors in one call (autoddl_search).  Returns a dict with T (or None), node, mask,
    opt_cost, strategy and, when init is given, cd_cost, cd_strategy, cd_sweeps."""
    Bp, L = d_layers.shape[0], d_layers.shape[1]
    K = num_signatures(mesh)
    dev = d_layers.device
    o = dict(out) if out else {}
    if want_tables and "T" not in o:
        o["T"] = torch.empty((Bp, L, K, K), dtype=torch.int64, device=dev)
    if want_node_mask:
        o.setdefault("node", torch.empty((Bp, L, K), dtype=torch.int64, device=dev))
        o.setdefault("mask", torch.empty((Bp, L, K), dtype=torch.uint8, device=dev))
    o.setdefault("opt_cost", torch.empty(Bp, dtype=torch.int64, device=dev))
    o.setdefault("strategy", torch.empty((Bp, L), dtype=torch.int32, device=dev))
    S = 0
    if init is not None:
        S = init.shape[1]
        o.setdefault("cd_cost", torch.empty((Bp, S), dtype=torch.int64, device=dev))
        o.setdefault("cd_strategy", torch.empty((Bp, S, L), dtype=torch.int32, device=dev))
        o.setdefault("cd_sweeps", torch.empty((Bp, S), dtype=torch.int32, device=dev))
    if work is None:
        need = workspace_bytes(Bp, L, S, mesh)
        if o.get("T") is not None:
            need -= Bp * L * K * K * 8                       # tables go to T, not to the workspace
        work = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    m, n = c_mesh(mesh), c_net(net)
    _check(lib().autoddl_search(_ptr(d_layers, U8, "d_layers"), Bp, L, C.addressof(m), C.addressof(n), _ptr(o.get("T"), I64, "T"),
                                _ptr(o.get("node"), I64, "node"), _ptr(o.get("mask"), U8, "mask"), _ptr(work, U8, "work"),
                                work.numel() if work is not None else 0, _ptr(o["opt_cost"], I64, "opt_cost"),
                                _ptr(o["strategy"], I32, "strategy"), _ptr(init, I32, "init"), S, max_sweeps,
                                _ptr(o.get("cd_cost"), I64, "cd_cost"), _ptr(o.get("cd_strategy"), I32, "cd_strategy"),
                                _ptr(o.get("cd_sweeps"), I32, "cd_sweeps"), _stream()))
    return o


def search_host(w: Workload, init: np.ndarray | None, work: torch.Tensor, pinned=None):
    """End-to-end call with HOST inputs/outputs (numpy or pinned torch CPU tensors).  Returns a dict of numpy arrays."""
    layers = np.ascontiguousarray(w.layers)
    Bp, L = layers.shape
    S = 0 if init is None else init.shape[1]
    if pinned is None:
        pinned = alloc_host_outputs(Bp, L, S)
    m, n = c_mesh(w.mesh), c_net(w.net)
    ip = _hptr(init, np.int32, "init")
    _check(lib().autoddl_search_host(_hptr(layers, LAYER_DTYPE, "layers"), Bp, L, C.addressof(m), C.addressof(n), ip, S, w.max_sweeps,
                                     _ptr(work, U8, "work"), work.numel(),
                                     pinned["opt_cost"].data_ptr(), pinned["strategy"].data_ptr(),
                                     pinned["cd_cost"].data_ptr() if S else None,
                                     pinned["cd_strategy"].data_ptr() if S else None,
                                     pinned["cd_sweeps"].data_ptr() if S else None, _stream()))
    keys = ("opt_cost", "strategy") + (("cd_cost", "cd_strategy", "cd_sweeps") if S else ())
    return {k: pinned[k].numpy() for k in keys}         # no Coordinate Descent: no cd_* keys (nothing was written there)


def alloc_host_outputs(Bp: int, L: int, S: int, pin: bool = True):
    pin = pin and torch.cuda.is_available()
    mk = lambda shape, dt: torch.empty(shape, dtype=dt, pin_memory=pin)
    return {
        "opt_cost": mk((Bp,), torch.int64), "strategy": mk((Bp, L), torch.int32),
        "cd_cost": mk((Bp, max(S, 1)), torch.int64), "cd_strategy": mk((Bp, max(S, 1), L), torch.int32),
        "cd_sweeps": mk((Bp, max(S, 1)), torch.int32),
    }


def store_probe(T: torch.Tensor):
    """store-only kernel with the fused table writer's address pattern over T [Bp, L, K, K] int64 (overwrites it)"""
    Bp, L, K = T.shape[0], T.shape[1], T.shape[2]
    _check(lib().autoddl_store_probe(_ptr(T, I64, "T"), Bp, L, K, _stream()))


def copy_probe(src: torch.Tensor, dst: torch.Tensor):
    nbytes = src.numel() * src.element_size()
    _check(lib().autoddl_copy_probe(src.data_ptr(), dst.data_ptr(), nbytes, _stream()))


def launch_count() -> int:
    return int(lib().autoddl_launch_count())
