"""Compute calls straight through the C-ABI (ctypes on libautoddl.so, no binding.py wrapper in between): raw device
pointers from torch, host structs built here from include/autoddl.h's layout.  Results against the oracle."""
import ctypes as C
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ref
from paper_2301_06813_b200 import configs as cf

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


class Mesh(C.Structure):                                            # autoddl_mesh: ndim, size[8], link[8]
    _fields_ = [("ndim", C.c_int32), ("size", C.c_int32 * 8), ("link", C.c_int32 * 8)]


class Net(C.Structure):                                             # autoddl_net
    _fields_ = [("alpha_ps", C.c_int64 * 2), ("beta_ps_per_byte", C.c_int64 * 2), ("mem_cap_bytes", C.c_int64),
                ("micro_batches", C.c_int64)]


def test_three_steps_and_one_call_raw():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    lib = C.CDLL(os.path.join(ROOT, "paper_2301_06813_b200", "libautoddl.so"))
    vp, i32, sz = C.c_void_p, C.c_int32, C.c_size_t
    lib.autoddl_workspace_bytes.restype = sz
    lib.autoddl_workspace_bytes.argtypes = [i32, i32, i32, vp]
    lib.autoddl_build_tables.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp]
    lib.autoddl_chain_dp.argtypes = [vp, i32, i32, vp, vp, vp, vp, sz, vp, vp, vp]
    lib.autoddl_coord_descent.argtypes = [vp, i32, i32, vp, vp, vp, vp, sz, vp, i32, i32, vp, vp, vp, vp]
    lib.autoddl_search.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp, vp, vp, i32, i32, vp, vp, vp, vp]
    lib.autoddl_best_of_starts.argtypes = [vp, i32, i32, vp, vp, vp]
    lib.autoddl_last_error.restype = C.c_char_p
    for w in (cf.config3_transformer24(), cf.config4_batched(Bp=333, L=21, seed=6)):
        S = min(w.S, 5)
        init = np.ascontiguousarray(w.cd_init()[:, :S])
        Bp, L, K = w.Bp, w.L, w.K
        m = Mesh(); m.ndim = w.mesh.ndim
        for d in range(m.ndim):
            m.size[d], m.link[d] = w.mesh.size[d], w.mesh.link[d]
        n = Net()
        n.alpha_ps[0], n.alpha_ps[1] = w.net.alpha_ps
        n.beta_ps_per_byte[0], n.beta_ps_per_byte[1] = w.net.beta_ps_per_byte
        n.mem_cap_bytes, n.micro_batches = w.net.mem_cap_bytes, w.net.micro_batches
        dev = "cuda"
        d_layers = torch.from_numpy(np.ascontiguousarray(w.layers).view(np.uint8).reshape(Bp, L, 64).copy()).to(dev)
        d_init = torch.from_numpy(init).to(dev)
        T = torch.empty((Bp, L, K, K), dtype=torch.int64, device=dev)
        node = torch.empty((Bp, L, K), dtype=torch.int64, device=dev)
        mask = torch.empty((Bp, L, K), dtype=torch.uint8, device=dev)
        dc = torch.empty(Bp, dtype=torch.int64, device=dev); ds = torch.empty((Bp, L), dtype=torch.int32, device=dev)
        cc = torch.empty((Bp, S), dtype=torch.int64, device=dev); cs = torch.empty((Bp, S, L), dtype=torch.int32, device=dev)
        sw = torch.empty((Bp, S), dtype=torch.int32, device=dev)
        bc = torch.empty(Bp, dtype=torch.int64, device=dev); bs = torch.empty(Bp, dtype=torch.int32, device=dev)
        nbytes = lib.autoddl_workspace_bytes(Bp, L, S, C.addressof(m))
        assert nbytes > 0
        work = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        st = torch.cuda.current_stream().cuda_stream

        def ok(rc):
            assert rc == 0, lib.autoddl_last_error()

        ok(lib.autoddl_build_tables(d_layers.data_ptr(), Bp, L, C.addressof(m), C.addressof(n), T.data_ptr(), node.data_ptr(), mask.data_ptr(), st))
        ok(lib.autoddl_chain_dp(None, Bp, L, C.addressof(m), None, T.data_ptr(), work.data_ptr(), nbytes, dc.data_ptr(), ds.data_ptr(), st))
        ok(lib.autoddl_coord_descent(None, Bp, L, C.addressof(m), None, T.data_ptr(), None, 0, d_init.data_ptr(), S, w.max_sweeps,
                                     cc.data_ptr(), cs.data_ptr(), sw.data_ptr(), st))
        ok(lib.autoddl_best_of_starts(cc.data_ptr(), Bp, S, bc.data_ptr(), bs.data_ptr(), st))
        torch.cuda.synchronize()
        oT, on, om = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
        odc, ods = ref.chain_dp(oT)
        occ, ocs, osw = ref.coord_descent(oT, init, w.max_sweeps)
        obc, obs = ref.best_of_starts(occ)
        want = dict(T=oT, node=on, mask=om, dc=odc, ds=ods, cc=occ, cs=ocs, sw=osw, bc=obc, bs=obs)
        got = dict(T=T, node=node, mask=mask, dc=dc, ds=ds, cc=cc, cs=cs, sw=sw, bc=bc, bs=bs)
        for k in want:
            assert np.array_equal(got[k].cpu().numpy(), want[k]), (w.name, k)
        # the one-call entry point into fresh buffers
        for t in (T, node, mask, dc, ds, cc, cs, sw):
            t.zero_()
        ok(lib.autoddl_search(d_layers.data_ptr(), Bp, L, C.addressof(m), C.addressof(n), T.data_ptr(), node.data_ptr(), mask.data_ptr(),
                              work.data_ptr(), nbytes, dc.data_ptr(), ds.data_ptr(), d_init.data_ptr(), S, w.max_sweeps,
                              cc.data_ptr(), cs.data_ptr(), sw.data_ptr(), st))
        torch.cuda.synchronize()
        for k in ("T", "node", "mask", "dc", "ds", "cc", "cs", "sw"):
            assert np.array_equal(got[k].cpu().numpy(), want[k]), (w.name, "search", k)


def test_store_probe_covers_every_cell():
    """autoddl_store_probe (bench.py's write-pattern ceiling): every cell of [Bp][L][K][K] is written, nothing beyond it"""
    import torch
    from paper_2301_06813_b200 import binding as adl
    adl.lib()
    Bp, L, K = 301, 5, 36
    buf = torch.full((Bp * L * K * K + 64,), -7, dtype=torch.int64, device="cuda")
    T = buf[:Bp * L * K * K].view(Bp, L, K, K)
    adl.store_probe(T)
    torch.cuda.synchronize()
    cells = T.view(Bp, L, K * K // 2, 2)
    assert torch.equal(cells[..., 0], torch.arange(Bp, device="cuda").view(Bp, 1, 1).expand(Bp, L, K * K // 2))
    assert torch.equal(cells[..., 1], torch.arange(L, device="cuda").view(1, L, 1).expand(Bp, L, K * K // 2))
    assert bool((buf[Bp * L * K * K:] == -7).all())
