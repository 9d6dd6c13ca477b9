#!/usr/bin/env python
"""bench.py -- AutoDDL strategy-search hot path on B200 (contract: see DESIGN.md section 8).

One "step" = one pass of the whole hot path over one batch of synthetic input:
  (a1) cost tables -> (a2) chain DP -> (a3) coordinate descent
run through the library's one-call entry point autoddl_search: (a1) + (a2) + the first two sweeps of (a3) as ONE
fused kernel (one warp per chain: a tile's factors are evaluated in shared memory, expanded to HBM with 16-byte
streaming stores, and consumed by the DP and the CD sweeps from shared memory), then the CD kernel from sweep 3.  The three
stand-alone kernels (autoddl_build_tables, autoddl_chain_dp, autoddl_coord_descent) are timed in the same run
and reported under "kernels" / "parts" (the three numbers BASELINE.json's metric names).
Workload: BASELINE.json configs[3] (4096 independent chains x 64 GEMM layers, mesh 4 x 4, K = 36), the
configuration the metric is quoted on.  Inputs (layer records, CD starts) are resident in HBM for
`value`; `e2e` goes through autoddl_search_host with pinned HOST buffers (the kernels read the pinned inputs
over PCIe, results are copied back: host-to-device and device-to-host traffic inside the timed
region).  `--impl reference` times the CPU oracle (oracle/, plain single-threaded C++) instead.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
  torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...     (N > 1: one rank per GPU)
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2301_06813_b200 import configs as cf  # noqa: E402

METRIC = "SBP cost-table cells/s, min-plus DP cells/s, CD sweeps/s on 1 B200 vs HBM roofline"
FALLBACK_HBM_GBS = 6650.0       # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload_desc(w, extra=None):
    d = {
        "workload": "configs[3] batched random chains: %d problems x L=%d GEMM layers, dims log-uniform [256,16384], "
                    "fp16 act / fp32 wgrad, mesh 4x4 (inter 25 GB/s, intra 300 GB/s), K=%d, 1 CD start per problem"
                    % (w.Bp, w.L, w.K),
        "Bp_per_gpu": w.Bp, "L": w.L, "K": w.K, "cd_starts": w.S, "seed": w.seed,
        "cells_per_gpu": w.cells, "table_bytes_per_gpu": w.cells * 8,
        "l2": "tables (2.7 GB) exceed the 126 MB L2, so every step streams them through HBM; no explicit flush",
    }
    if extra:
        d.update(extra)
    return d


# ---------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py may execute oracle/)
# ---------------------------------------------------------------------------------------------------
def oracle_sample_run(w, nprob, repeat=1):
    """whole path of the oracle, as it stands, single thread, on the first nprob problems"""
    from oracle import ref
    mesh, net = ref.mesh_of(w), ref.net_of(w)
    layers = np.ascontiguousarray(w.layers[:nprob])
    init = np.ascontiguousarray(w.cd_init()[:nprob])
    t = {"build": 0.0, "dp": 0.0, "cd": 0.0}
    sweeps = 0
    for _ in range(repeat):
        t0 = time.perf_counter()
        T, _, _ = ref.build_tables(layers, mesh, net)
        t1 = time.perf_counter()
        ref.chain_dp(T)
        t2 = time.perf_counter()
        _, _, sw = ref.coord_descent(T, init, w.max_sweeps)
        t3 = time.perf_counter()
        t["build"] += t1 - t0
        t["dp"] += t2 - t1
        t["cd"] += t3 - t2
        sweeps += int(sw.sum())
    cells = nprob * w.L * w.K * w.K * repeat
    return cells, sweeps, t


def cpu_baseline(w, nprob=2048):
    cells, sweeps, t = oracle_sample_run(w, nprob)
    tot = t["build"] + t["dp"] + t["cd"]
    return {
        "value": cells / tot, "unit": "cells/s", "cores": 1, "kind": "oracle",
        "sample": "first %d of %d problems of the same workload, whole path (build + DP + CD), single-threaded "
                  "g++ -O2 oracle, %.1f s" % (nprob, w.Bp, tot),
        "parts": {"build_cells_per_s": cells / t["build"], "dp_cells_per_s": cells / t["dp"],
                  "cd_sweeps_per_s": sweeps / t["cd"]},
    }


def cpu_baseline_all_cores(w, nprob=2048):
    """the same oracle calls fanned out over the host cores: one thread per core, each on a contiguous
    slice of the problems; ctypes releases the GIL during the calls, the oracle itself stays single-threaded C++"""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import ref
    ncores = max(1, len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
    nthreads = min(ncores, nprob)
    mesh, net = ref.mesh_of(w), ref.net_of(w)
    init = w.cd_init()
    bounds = np.linspace(0, nprob, nthreads + 1).astype(int)

    def work(k):
        a, b = int(bounds[k]), int(bounds[k + 1])
        if a == b:
            return 0
        T, _, _ = ref.build_tables(np.ascontiguousarray(w.layers[a:b]), mesh, net)
        ref.chain_dp(T)
        _, _, sw = ref.coord_descent(T, np.ascontiguousarray(init[a:b]), w.max_sweeps)
        return int(sw.sum())

    ref.lib()
    t0 = time.perf_counter()
    with ThreadPoolExecutor(nthreads) as ex:
        list(ex.map(work, range(nthreads)))
    el = time.perf_counter() - t0
    return {"value": nprob * w.L * w.K * w.K / el, "unit": "cells/s", "cores": nthreads, "seconds": el,
            "sample": "first %d problems, whole path, one oracle thread per host core" % nprob}


def run_reference(args):
    """--impl reference: the CPU oracle on the box's host cores; each step is a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = cf.config4_batched()
    nprob = max(4, min(48, 48 * 200 // max(args.steps, 1)))      # whole run stays within a few minutes
    for _ in range(args.warmup):
        oracle_sample_run(w, 4)
    t0 = time.perf_counter()
    cells = 0
    parts = {"build": 0.0, "dp": 0.0, "cd": 0.0}
    sweeps = 0
    for _ in range(args.steps):
        c, s, t = oracle_sample_run(w, nprob)
        cells += c
        sweeps += s
        for k in parts:
            parts[k] += t[k]
    el = time.perf_counter() - t0
    val = cells / el
    sample = "each step = whole path on the first %d of %d problems, single-threaded oracle" % (nprob, w.Bp)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "cells/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic (seeded splitmix64)",
        "config": workload_desc(w, {"parallelism": "problems sharded over %d GPU(s), one all-gather of the result rows" % args.gpus,
                                    "scaling_mode": args.scaling}),
        "cpu_baseline": {"value": val, "unit": "cells/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "cells/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "parts": {"build_cells_per_s": cells / parts["build"], "dp_cells_per_s": cells / parts["dp"],
                  "cd_sweeps_per_s": sweeps / parts["cd"]},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def cuda_compute(adl, w, work=None, out=None):
    """(compute, best_of_starts) callables for shard.ShardedSearch backed by the CUDA path: compute uploads a shard once
    (cached by the identity of the numpy arrays: the timed loop calls it every step with the same shard) and runs the
    one-call entry point autoddl_search on it; best_of_starts is the library's reduction kernel."""
    import torch
    cache = {}

    def resident(a, to_dev):
        key = (id(a), a.shape)
        if key not in cache:
            cache[key] = (a, to_dev(a))                           # keeps `a` alive: ids are not reused
        return cache[key][1]

    def compute(layers, init):
        d_layers = resident(layers, adl.layers_to_device)
        d_init = None if init is None else resident(init, lambda x: torch.from_numpy(x).cuda())
        return adl.search(d_layers, w.mesh, w.net, init=d_init, max_sweeps=w.max_sweeps, work=work, out=out)

    return compute, adl.best_of_starts


def run_ours(args):
    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    sampler = ClockSampler(local) if rank == 0 else None          # from before the warm-up to after the end-to-end loop
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2301_06813_b200 import binding as adl
    from paper_2301_06813_b200.shard import ShardedSearch, shard_range
    adl.lib()

    # weak scaling (default): every rank searches its own 4096 problems (seed = rank); strong: the 4096 problems of seed 0
    # are split over the ranks.  Either way the step ends with ONE all-gather of the result rows; there is
    # no collective in the data path.
    strong = args.scaling == "strong"
    w_all = cf.config4_batched(seed=0 if strong else rank)
    plan = ShardedSearch(w_all.layers, w_all.cd_init(), mode="problems", local_shard=not strong)
    w = cf.Workload(w_all.name, plan.layers, w_all.mesh, w_all.net, S=w_all.S, seed=w_all.seed, max_sweeps=w_all.max_sweeps)
    init_np = plan.init
    d_layers = adl.layers_to_device(w.layers)
    d_init = torch.from_numpy(init_np).cuda()
    K, L, Bp, S = w.K, w.L, w.Bp, w.S
    T = torch.empty((Bp, L, K, K), dtype=torch.int64, device="cuda")
    dp_out = (torch.empty(Bp, dtype=torch.int64, device="cuda"), torch.empty((Bp, L), dtype=torch.int32, device="cuda"))
    cd_out = (torch.empty((Bp, S), dtype=torch.int64, device="cuda"), torch.empty((Bp, S, L), dtype=torch.int32, device="cuda"),
              torch.empty((Bp, S), dtype=torch.int32, device="cuda"))

    work = torch.empty(adl.workspace_bytes(Bp, L, S, w.mesh), dtype=torch.uint8, device="cuda")
    one_out = {"T": T, "opt_cost": dp_out[0], "strategy": dp_out[1], "cd_cost": cd_out[0], "cd_strategy": cd_out[1],
               "cd_sweeps": cd_out[2]}
    compute, best = cuda_compute(adl, w, work=work, out=one_out)
    results = {}

    def step(evs=None):
        """the whole path on this rank's shard in ONE library call (autoddl_search): the fused kernel (tables, chain DP,
        first two CD sweeps), then the CD kernel from sweep 3; then the exchange: all-gather of the result rows and the
        best-of-starts kernel.  evs[1] is recorded by the library between the two kernels (autoddl_profile_mark)."""
        if evs:
            adl.profile_mark(evs[1])
            evs[0].record()
        results.update(plan.run(compute, best))
        if evs: evs[2].record()

    def step_separate(evs):
        """the three stand-alone kernels, for the per-kernel numbers"""
        evs[0].record()
        adl.build_tables(d_layers, w.mesh, w.net, want_node_mask=False, out=T)
        evs[1].record()
        adl.chain_dp(T, w.mesh, out=dp_out)
        evs[2].record()
        adl.coord_descent(T, d_init, w.mesh, w.max_sweeps, out=cd_out)
        evs[3].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    total_sweeps = int(cd_out[2].sum().item())
    fused_sweeps = int(cd_out[2].clamp(max=2).sum().item())      # the fused kernel runs the first two sweeps of every start

    # ---- timed region: exactly K steps, CUDA events on the launching (current) stream ----------------
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    for e in evs:
        e[1].record()                                        # instantiate the handle the library records later
    e_start, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = adl.launch_count()
    barrier()
    e_start.record()
    for k in range(args.steps):
        step(evs[k])
    e_end.record()
    barrier()
    launches = adl.launch_count() - launches0
    ms_total = e_start.elapsed_time(e_end)
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms = {"fused": 0.0, "cd_resume": 0.0, "build": 0.0, "dp": 0.0, "cd": 0.0}
    for e in evs:
        ms["fused"] += e[0].elapsed_time(e[1]); ms["cd_resume"] += e[1].elapsed_time(e[2])
    # the stand-alone table builder and chain DP, same inputs, same run (outside the timed step region)
    evs2 = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    for _ in range(3):
        step_separate(evs2[0])
    torch.cuda.synchronize()
    for k in range(args.steps):
        step_separate(evs2[k])
    torch.cuda.synchronize()
    for e in evs2:
        ms["build"] += e[0].elapsed_time(e[1]); ms["dp"] += e[1].elapsed_time(e[2]); ms["cd"] += e[2].elapsed_time(e[3])
    # the one-call path with no table requested (nothing of (a1) reaches HBM): reported beside the step, not as the step
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    nt_out = {k: v for k, v in one_out.items() if k != "T"}
    for _ in range(3):
        adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers, work=work, out=dp_out)
    e0.record()
    for _ in range(args.steps):
        adl.chain_dp(None, w.mesh, net=w.net, d_layers=d_layers, work=work, out=dp_out)
    e1.record()
    torch.cuda.synchronize()
    ms["fused_no_table"] = e0.elapsed_time(e1)
    for k in ms:
        ms[k] /= args.steps
    ms_step = ms_total / args.steps
    cells = w.cells                                          # per rank
    value = world * cells / (ms_step * 1e-3)

    # ---- HBM copy peak by our own copy kernel, in the same run -------------------------------------------
    nb = 1 << 30
    a = torch.empty(nb, dtype=torch.uint8, device="cuda").random_(0, 255)
    b = torch.empty(nb, dtype=torch.uint8, device="cuda")
    best_ms = 1e9
    for i in range(13):
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(); adl.copy_probe(a, b); s1.record(); torch.cuda.synchronize()
        if i >= 3:
            best_ms = min(best_ms, s0.elapsed_time(s1))
    copy_gbs = 2 * nb / (best_ms * 1e-3) / 1e9
    del a, b
    # ---- the ceiling of the fused kernel's WRITE PATTERN: a store-only kernel with its addresses (one warp per chain, tile
    # after tile, 16-byte streaming stores), same run, same buffer; average of back-to-back launches like the step itself
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        adl.store_probe(T)
    s0.record()
    for _ in range(20):
        adl.store_probe(T)
    s1.record(); torch.cuda.synchronize()
    store_ms = s0.elapsed_time(s1) / 20
    store_gbs = w.cells * 8 / (store_ms * 1e-3) / 1e9

    # ---- end to end through the host-pointer C-ABI call (pinned host buffers, H2D + D2H timed) -----------
    pinned = adl.alloc_host_outputs(Bp, L, S)
    h_layers = torch.from_numpy(np.ascontiguousarray(w.layers).view(np.uint8).reshape(Bp, L, 64).copy()).pin_memory()
    h_init = torch.from_numpy(init_np.copy()).pin_memory()
    w_host = cf.Workload(w.name, h_layers.numpy().view(cf.LAYER_DTYPE).reshape(Bp, L), w.mesh, w.net, S=S, seed=w.seed)
    e2e_steps = max(3, min(args.steps, 50))
    for _ in range(3):
        adl.search_host(w_host, h_init.numpy(), work, pinned)
    barrier()
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record()
    for _ in range(e2e_steps):
        adl.search_host(w_host, h_init.numpy(), work, pinned)
    s1.record()
    barrier()
    e2e_ms = s0.elapsed_time(s1)
    if world > 1:
        t = torch.tensor([e2e_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    e2e_ms /= e2e_steps
    clocks = sampler.stop() if sampler else None
    h2d = h_layers.numel() + h_init.numel() * 4
    d2h = sum(v.numel() * v.element_size() for v in pinned.values())
    assert np.array_equal(pinned["opt_cost"].numpy(), dp_out[0].cpu().numpy())      # same answers through both routes
    off = plan.rank * Bp if not strong else shard_range(plan.n_total, plan.rank, world)[0]
    assert torch.equal(results["opt_cost"][off:off + Bp], dp_out[0])            # the gathered rows hold this rank's shard

    if rank == 0:
        peak, peak_src = measured_peak()
        table_bytes = cells * 8
        dp_bytes = (L - 1) * Bp * K * K * 8 + Bp * K * 8          # tile 0 contributes one row
        cd_alg_bytes = total_sweeps * 16 * K * L
        sweep1_bytes = fused_sweeps * 16 * K * L             # CD work done inside the fused launch (sweeps 1 and 2)
        # Bytes that MUST reach HBM per launch (what "roofline" means here): the fused kernel writes the tables (8 B per
        # cell) and reads 64 B per layer record; the chain DP and the first two CD sweeps run from shared memory and move
        # nothing.  SURVEY 8(d)'s per-unit figures (8 B/cell written + 8 B/cell read by the DP + 16 K L B per CD sweep)
        # count WORK; for the fused launch their sum is reported separately as work_units_*: it exceeds the HBM bytes
        # because fusion removed two of the three streams.
        fused_hbm = table_bytes + Bp * L * 64
        fused_work = table_bytes + dp_bytes + sweep1_bytes
        kernels = {
            "build_dp_cd2_fused": {"ms": ms["fused"], "cells_per_s": cells / (ms["fused"] * 1e-3),
                                   "hbm_GBps": fused_hbm / (ms["fused"] * 1e-3) / 1e9,
                                   "work_units_GBps": fused_work / (ms["fused"] * 1e-3) / 1e9, "in_step": True,
                                   "bound": "LSU data pipe (shared-memory loads + the global stores: ncu 81 %) / issue (67 %); hbm traffic "
                                            "= the 8 B/cell table write only (DP and the first two CD sweeps read the tile factors "
                                            "from shared memory)"},
            "coord_descent_resume": {"ms": ms["cd_resume"], "sweeps": total_sweeps - fused_sweeps,
                                     "sweeps_per_s": (total_sweeps - fused_sweeps) / (ms["cd_resume"] * 1e-3),
                                     "hbm_GBps": (cd_alg_bytes - sweep1_bytes) / (ms["cd_resume"] * 1e-3) / 1e9, "in_step": True,
                                     "bound": "latency of the dependent updates of the slowest chains; 16*K*L B per sweep, sweeps 3.. "
                                              "(plus the exchange: all-gather of result rows and best-of-starts, no-ops at 1 GPU)"},
            "build_tables": {"ms": ms["build"], "cells_per_s": cells / (ms["build"] * 1e-3),
                             "hbm_GBps": table_bytes / (ms["build"] * 1e-3) / 1e9, "in_step": False, "bound": "hbm (write 8 B/cell)"},
            "chain_dp": {"ms": ms["dp"], "cells_per_s": cells / (ms["dp"] * 1e-3),
                         "hbm_GBps": dp_bytes / (ms["dp"] * 1e-3) / 1e9, "in_step": False, "bound": "hbm (read 8 B/cell)"},
            "coord_descent": {"ms": ms["cd"], "sweeps_per_s": total_sweeps / (ms["cd"] * 1e-3), "sweeps": total_sweeps,
                              "hbm_GBps": cd_alg_bytes / (ms["cd"] * 1e-3) / 1e9, "in_step": False,
                              "bound": "hbm, random 64-byte granules (16*K*L B per sweep)"},
            "fused_no_table": {"ms": ms["fused_no_table"], "cells_per_s": cells / (ms["fused_no_table"] * 1e-3), "in_step": False,
                               "hbm_GBps": Bp * L * 64 / (ms["fused_no_table"] * 1e-3) / 1e9,
                               "bound": "autoddl_chain_dp(d_T = NULL): the same kernel with no table written (optimum + strategy "
                                        "only): shared-memory bandwidth / issue"},
        }
        for k in kernels.values():
            k["frac_of_peak"] = k["hbm_GBps"] / peak
        kernels["build_dp_cd2_fused"]["work_units_frac_of_peak"] = kernels["build_dp_cd2_fused"]["work_units_GBps"] / peak
        dom = max(("build_dp_cd2_fused", "coord_descent_resume"), key=lambda n: kernels[n]["ms"])
        traffic, traffic_src = None, None
        tpath = os.path.join(ROOT, "profiles", "traffic_r2.csv")       # per-launch DRAM bytes from a committed ncu --set full capture
        if os.path.exists(tpath):
            try:
                rows = dict(l.strip().split(",")[:2] for l in open(tpath).read().splitlines()[1:] if l.strip())
                traffic = float(rows[dom]) if dom in rows else None
                traffic_src = "profiles/traffic_r2.csv (committed ncu capture of the same command: dram__bytes_read.sum + dram__bytes_write.sum per launch; NOT measured in this run)"
                for name, k in kernels.items():
                    if name in rows:
                        k["dram_bytes_per_launch_ncu"] = float(rows[name])
                        k["dram_GBps"] = float(rows[name]) / (k["ms"] * 1e-3) / 1e9
                        k["dram_frac_of_peak"] = k["dram_GBps"] / peak
                        k["dram_source"] = "committed ncu capture (profiles/traffic_r2.csv) / this run's launch time"
            except Exception:
                traffic, traffic_src = None, None
        line = {
            "metric": METRIC, "value": value, "unit": "cells/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
            "dtype": "int64", "data": "synthetic (seeded splitmix64; shapes of BASELINE.json configs[3])",
            "config": workload_desc(w, {"parallelism": "problems sharded over %d GPU(s), one all-gather of the result rows" % world,
                                        "scaling_mode": args.scaling}),
            "parts": {"build_cells_per_s": world * kernels["build_tables"]["cells_per_s"],
                      "dp_cells_per_s": world * kernels["chain_dp"]["cells_per_s"],
                      "fused_build_dp_cd2_cells_per_s": world * kernels["build_dp_cd2_fused"]["cells_per_s"],
                      "cd_sweeps_per_s": world * kernels["coord_descent"]["sweeps_per_s"]},
            "kernels": kernels,
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["hbm_GBps"], "peak": peak, "unit": "GB/s",
                         "frac": kernels[dom]["hbm_GBps"] / peak, "traffic": traffic, "traffic_source": traffic_src,
                         "peak_source": peak_src, "copy_probe_GBps_same_run": copy_gbs,
                         "store_pattern_probe_GBps_same_run": store_gbs, "store_pattern_probe_ms": store_ms,
                         "frac_of_store_pattern_probe": (store_ms / kernels[dom]["ms"]) if dom == "build_dp_cd2_fused" else None,
                         "bytes_per_launch": fused_hbm if dom == "build_dp_cd2_fused" else cd_alg_bytes - sweep1_bytes,
                         "work_units_frac": kernels[dom].get("work_units_frac_of_peak"),
                         "note": "frac = bytes that must reach HBM per launch (8 B per cell written + 64 B per layer record read) / "
                                 "CUDA-event launch time / peak; work_units_frac counts SURVEY 8(d)'s per-unit bytes for all the work "
                                 "the fused launch does (tables + DP + two CD sweeps) and can exceed 1; store_pattern_probe = a store-only "
                                 "kernel with the fused kernel's write addresses (autoddl_store_probe), timed in this run: "
                                 "frac_of_store_pattern_probe = its time / the fused kernel's time"},
            "e2e": {"value": world * cells / (e2e_ms * 1e-3), "unit": "cells/s", "ms_per_step": e2e_ms,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps},
            "gpu_launches": launches,
            "clocks": clocks,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w)
            line["cpu_baseline"]["all_cores"] = cpu_baseline_all_cores(w)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# ---------------------------------------------------------------------------------------------------
# --configs: one JSON line per BASELINE.json config (the small ones are launch-bound: absolute microseconds)
# ---------------------------------------------------------------------------------------------------
def run_configs(args):
    """GPU kernel times and single-thread oracle times on configs 1, 2, 3, 5 (config 4 is the default run).  Also times
    the Metropolis-Hastings kernel and, on config 4, reports its proposals/s."""
    import torch
    from oracle import ref
    from paper_2301_06813_b200 import binding as adl
    adl.lib()
    torch.cuda.set_device(0)

    def gpu_us(fn, n=30):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n * 1e3

    for k in args.configs:
        w = cf.CONFIGS[k]() if k != 4 else cf.config4_batched()
        dl = adl.layers_to_device(w.layers)
        init_np = w.cd_init()
        init = torch.from_numpy(init_np).cuda()
        T, _, _ = adl.build_tables(dl, w.mesh, w.net, want_node_mask=False)
        work = torch.empty(adl.workspace_bytes(w.Bp, w.L, w.S, w.mesh), dtype=torch.uint8, device="cuda")
        dp = adl.chain_dp(T, w.mesh, work=work)
        cd = adl.coord_descent(T, init, w.mesh, w.max_sweeps)
        nsteps = 4096
        tau = 20_000_000
        mh = adl.metropolis(T, init, w.mesh, nsteps, tau, seed=0)
        one = adl.search(dl, w.mesh, w.net, init=init, max_sweeps=w.max_sweeps, work=work, out={"T": T})
        one_nt = adl.search(dl, w.mesh, w.net, init=init, max_sweeps=w.max_sweeps, want_tables=False, work=work)
        torch.cuda.synchronize()
        for key in ("opt_cost", "strategy", "cd_cost", "cd_strategy", "cd_sweeps"):
            assert torch.equal(one[key], one_nt[key]), key
        sweeps = int(cd[2].sum().item())
        g = {
            "build_us": gpu_us(lambda: adl.build_tables(dl, w.mesh, w.net, want_node_mask=False, out=T)),
            "dp_us": gpu_us(lambda: adl.chain_dp(T, w.mesh, work=work, out=dp)),
            "cd_us": gpu_us(lambda: adl.coord_descent(T, init, w.mesh, w.max_sweeps, out=cd)),          # no workspace: the gather kernel
            # with a workspace: K <= 64 and >= 32 starts take best responses from the tiles + look-up sweeps
            "cd_work_us": gpu_us(lambda: adl.coord_descent(T, init, w.mesh, w.max_sweeps, work=work, out=cd)),
            # d_T = NULL: no K x K table; with >= 32 starts per problem on 2 / 3 mesh levels factors -> best responses -> look-ups
            "cd_no_table_us": gpu_us(lambda: adl.coord_descent(None, init, w.mesh, w.max_sweeps, net=w.net, d_layers=dl, work=work, out=cd)),
            "search_us": gpu_us(lambda: adl.search(dl, w.mesh, w.net, init=init, max_sweeps=w.max_sweeps, work=work, out=one)),
            # the same with no table asked for (optimum, strategies and CD results only): long chains take the DP in class space
            "dp_no_table_us": gpu_us(lambda: adl.chain_dp(None, w.mesh, net=w.net, d_layers=dl, work=work, out=dp)),
            "search_no_table_us": gpu_us(lambda: adl.search(dl, w.mesh, w.net, init=init, max_sweeps=w.max_sweeps, want_tables=False,
                                                            work=work, out=one_nt)),
            "mh_us": gpu_us(lambda: adl.metropolis(T, init, w.mesh, nsteps, tau, seed=0, out=mh), n=5),
        }
        # the same call captured once into a CUDA graph and replayed (the small configs are launch-bound)
        graph, gs = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        torch.cuda.synchronize()
        with torch.cuda.stream(gs):
            with torch.cuda.graph(graph, stream=gs):
                adl.search(dl, w.mesh, w.net, init=init, max_sweeps=w.max_sweeps, work=work, out=one)
        g["search_graph_us"] = gpu_us(graph.replay)
        line = {"config": k, "name": w.name, "Bp": w.Bp, "L": w.L, "K": w.K, "S": w.S, "cells": w.cells, "cd_sweeps": sweeps,
                "gpu": g,
                "gpu_rates": {"build_cells_per_s": w.cells / g["build_us"] * 1e6, "dp_cells_per_s": w.cells / g["dp_us"] * 1e6,
                              "cd_sweeps_per_s": sweeps / g["cd_us"] * 1e6,
                              "mh_proposals_per_s": w.Bp * w.S * nsteps / g["mh_us"] * 1e6},
                "dp_optimum_ps": int(dp[0][0]), "best_cd_over_dp": float(cd[0].min(dim=1).values.double().div(dp[0].double()).mean()),
                "best_mh_over_dp": float(mh[0].min(dim=1).values.double().div(dp[0].double()).mean()),
                # random search with the same S samples (the starts themselves; zero proposals): PAPER.md Fig. 7's third arm
                "best_random_over_dp": float(adl.metropolis(T, init, w.mesh, 0, tau, seed=0)[0].min(dim=1).values.double()
                                             .div(dp[0].double()).mean()),
                "mh": {"nsteps": nsteps, "tau_ps": tau}}
        if w.Bp == 1 and w.L >= 8:
            # pipeline-stage enumeration (R27, 6.12) of the chain into 4 stages, objective max: segment optima for all
            # O(L^2) segments, stage-transfer costs, partition DP, strategies of the chosen segments -- four kernels
            Tn, nodeN, maskN = adl.build_tables(dl, w.mesh, w.net, want_node_mask=True)
            torch.cuda.synchronize()
            pipe = adl.pipeline_stages(dl[0], Tn[0], nodeN[0], maskN[0], w.mesh, w.net, 4, 1)
            g["pipeline_us"] = gpu_us(lambda: adl.pipeline_stages(dl[0], Tn[0], nodeN[0], maskN[0], w.mesh, w.net, 4, 1), n=5)
            line["pipeline"] = {"stages": 4, "objective": "max", "value_ps": int(pipe["value"][0]), "cuts": pipe["cuts"].tolist(),
                                "segments": w.L * (w.L + 1) // 2}
            if w.L * w.K * w.K <= 3_000_000:                 # the oracle's segment optima are O(L^2 K^2): bounded
                hT, hn, hm = Tn[0].cpu().numpy(), nodeN[0].cpu().numpy(), maskN[0].cpu().numpy()
                t0 = time.perf_counter()
                otri = ref.segment_optima(hT, hn, hm)
                oval, ocuts = ref.pipeline_partition(otri, ref.stage_transfer(w.layers[0], ref.mesh_of(w), ref.net_of(w)), 4, 1)
                line["pipeline"]["oracle_1core_us"] = (time.perf_counter() - t0) * 1e6
                assert int(oval) == line["pipeline"]["value_ps"] and [int(x) for x in ocuts] == line["pipeline"]["cuts"]
        if k == 6:                                           # the same chain on the unrestricted six-row space
            wu = cf.config6_paper_space(restricted=False)
            Tu, _, _ = adl.build_tables(dl, wu.mesh, wu.net, want_node_mask=False)
            line["dp_optimum_unrestricted_ps"] = int(adl.chain_dp(Tu, wu.mesh, work=work)[0][0])
            line["note"] = "rows {0,1,2} per prime sub-level: the paper's factorisation space (27 of 216 signatures)"
        if k != 4:                                           # oracle, one core (config 4's oracle numbers are in the default run)
            mesh, net = ref.mesh_of(w), ref.net_of(w)
            t0 = time.perf_counter(); oT, _, _ = ref.build_tables(w.layers, mesh, net)
            t1 = time.perf_counter(); ref.chain_dp(oT)
            t2 = time.perf_counter(); _, _, osw = ref.coord_descent(oT, init_np, w.max_sweeps)
            t3 = time.perf_counter()
            ms = min(nsteps, 256)
            ref.metropolis(oT, init_np, ms, tau, seed=0)
            t4 = time.perf_counter()
            line["oracle_1core"] = {"build_cells_per_s": w.cells / (t1 - t0), "dp_cells_per_s": w.cells / (t2 - t1),
                                    "cd_sweeps_per_s": int(osw.sum()) / (t3 - t2),
                                    "mh_proposals_per_s": w.Bp * w.S * ms / (t4 - t3), "cores": 1}
        print(json.dumps(line))
    # alpha-beta calibration (R23): least squares over N timed collectives, GPU kernel and oracle
    import numpy as np
    N = 1 << 20
    rng = np.random.default_rng(0)
    kind = rng.integers(0, 4, N).astype(np.int32)
    pp = rng.choice([2, 4, 8, 16], N).astype(np.int32)
    nb = (2 ** rng.uniform(10, 28, N)).astype(np.int64)
    tt = ref.fit_design_matrix(kind, pp, nb) @ np.array([5e-6, 4e-11]) * (1 + 0.01 * rng.standard_normal(N))
    dev = [torch.from_numpy(x).cuda() for x in (kind, pp, nb, tt)]
    got = adl.fit_alpha_beta(*dev)
    fit_us = gpu_us(lambda: adl.fit_alpha_beta(*dev, out=got))
    t0 = time.perf_counter()
    want = ref.fit_alpha_beta(kind, pp, nb, tt)
    oracle_us = (time.perf_counter() - t0) * 1e6
    g = got.cpu().numpy()
    print(json.dumps({"fit_alpha_beta": {"samples": N, "gpu_us": fit_us, "oracle_1core_us": oracle_us, "alpha_s": float(g[0]),
                                         "beta_s_per_byte": float(g[1]),
                                         "rel_diff_to_oracle": [abs(float(g[0] / want[0]) - 1), abs(float(g[1] / want[1]) - 1)],
                                         "hbm_GBps": N * 24 / (fit_us * 1e-6) / 1e9}}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scaling", choices=["weak", "strong"], default="weak",
                    help="N > 1: weak = every rank its own 4096 problems; strong = the 4096 problems of seed 0 split over the ranks")
    ap.add_argument("--configs", type=int, nargs="+", default=None,
                    help="per-config report (kernel microseconds, oracle rates) instead of the bench line, e.g. --configs 1 2 3 5")
    args = ap.parse_args()
    if args.configs:
        return run_configs(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
