#!/usr/bin/env python
"""bench.py -- one JSON line for the Vietoris-Rips hot path (filtration construction with clearing
+ apparent pairs) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

A "step" is one pass of the whole hot path (every row a3-a10 of DESIGN.md section 1) over one
workload: for d = 1..dim_max: rips_stage1(d) (fused enumerate + diameter + threshold + clearing +
apparent-pair test, then the onesweep filtration sort), rips_stage2(d) (pair partition + the sorts
of the small irregular / non-apparent lists), called
through the C ABI on a context whose distance matrix, key matrix, binomial table and clearing sets
are resident in HBM (one untimed rips_compute produced them).  `value` = candidate simplices
(sum over d of C(n, d+1)) per second, whole job.  `e2e` = the same count divided by the time of
rips_init (HOST distance matrix) + rips_compute (dim 0, both stages, reduction) + rips_barcodes
(HOST bars), copies inside the timed region.  The serial remainder (dim 0, reduction of the
non-apparent columns) is reported separately under "barcode".

Multi-GPU: replicas only -- every rank runs the same workload on its own
GPU, no data-path collective; timing is the max over ranks.

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample.
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
from math import comb

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "simplices/sec (filtration+clearing+apparent pairs)"
UNIT = "simplices/s"
RECORD_BYTES = 8  # packed column / pair record


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs[k-1]; 2 is the one the metric is quoted on")
    ap.add_argument("--n", type=int, default=None, help="point count override (config 6, the second workload of PAPER.md:719-729: n = 1000 .. 20000)")
    ap.add_argument("--mode", type=int, default=0, help="0 auto, 1 dense, 2 sparse (rips_set_mode)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="budget of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-scale-row", action="store_true",
                    help="skip the scale row (stage 1 + 2 at d = dim_max+1: the C(n, dim_max+2) simplices the config names)")
    ap.add_argument("--warmup-seconds", type=float, default=0.0,
                    help="keep warming up (beyond --warmup, which is honoured exactly by default) until this much time has "
                         "passed; the warm-ups actually run are printed as `warmup`")
    return ap.parse_args()


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload_dict(w, n_cand):
    thr = None if w.threshold == float("inf") else w.threshold
    return {"workload": w.name, "n": w.n, "dim_max": w.dim_max, "threshold": thr, "note": w.note,
            "candidates_per_step": n_cand,
            "l2": "no flush: the record arrays of the top dimension exceed the 126 MB L2"}


# ------------------------------------------------------------------------------------ CPU oracle leg
def oracle_sample(w, budget_s):
    """The oracle as it stands (stage 1 + stage 2 of every dimension) on a bounded sample: the lower
    dimensions completely, then slices of the top dimension's index range until the budget is used.
    Returns (simplices, seconds, cores, description)."""
    from oracle import oracle
    t_all = time.perf_counter()
    z = oracle.dim0(w.dist, w.n, w.threshold)
    cleared = z["t"]
    done, spent, parts = 0, 0.0, []
    for d in range(1, w.dim_max + 1):
        total = comb(w.n, d + 1)
        if d < w.dim_max:
            t0 = time.perf_counter()
            fd, fc, _ = oracle.stage1(w.dist, w.n, d, w.threshold, cleared)
            s2 = oracle.stage2(w.dist, w.n, d, fd, fc)
            spent += time.perf_counter() - t0
            done += total
            parts.append(f"d={d} all {total}")
            # clearing set of the next dimension (untimed: the reduction is not the hot path)
            red = oracle.reduce_columns(w.dist, w.n, d, w.threshold, s2["non_cidx"], s2["app_t"], s2["app_s"])
            cleared = np.sort(np.concatenate([s2["app_t"], red["t"]]))
        else:
            lo, chunk = 0, 2_000_000
            while lo < total and (spent < budget_s or lo == 0):
                hi = min(total, lo + chunk)
                t0 = time.perf_counter()
                fd, fc, _ = oracle.stage1(w.dist, w.n, d, w.threshold, cleared, lo, hi)
                oracle.stage2(w.dist, w.n, d, fd, fc)
                spent += time.perf_counter() - t0
                done += hi - lo
                lo = hi
            parts.append(f"d={d} candidates [0,{lo}) of {total}")
    desc = "oracle stage 1 + stage 2 (sort included): " + "; ".join(parts)
    return done, spent, oracle.num_threads(), desc, time.perf_counter() - t_all


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2003_07989_b200 import inputs
    w = inputs.config(args.config, args.n)
    n_cand = sum(comb(w.n, d + 1) for d in range(1, w.dim_max + 1))
    per_step = max(2.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(w, per_step / 4)
    tot_s, tot_t, cores, desc = 0, 0.0, 0, ""
    for _ in range(args.steps):
        s, t, cores, desc, _ = oracle_sample(w, per_step)
        tot_s += s
        tot_t += t
    value = tot_s / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": workload_dict(w, n_cand),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------ clocks sampler
class ClockSampler:
    """nvidia-smi sampled every 200 ms DURING the timed region (B200_PROFILING.md's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        with open(self.path) as f:
            for ln in f:
                p = [x.strip() for x in ln.split(",")]
                if len(p) < 9:
                    continue
                try:
                    sm.append(float(p[1])); smax.append(float(p[2])); power.append(float(p[3]))
                except ValueError:
                    continue
                for name, v in zip(names, p[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        os.unlink(self.path)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------ ranks
class Ranks:
    """One process per GPU (replicas only): rendezvous, barrier and the max over
    ranks of a device time.  backend "nccl" on the GPU box, "gloo" in the CPU test."""

    def __init__(self, backend="nccl", device=None):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        if self.world > 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29533")
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, rank=self.rank, world_size=self.world, **kw)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        if self.device is not None and self.device.type == "cuda":
            self.torch.cuda.synchronize()

    def max_over_ranks(self, x):
        if self.world == 1:
            return float(x)
        t = self.torch.tensor([float(x)], dtype=self.torch.float64, device=self.device or "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_rate(self, units_per_rank, ms):
        """units all ranks processed / the slowest rank's time"""
        return self.world * units_per_rank / (self.max_over_ranks(ms) * 1e-3)

    def close(self):
        if self.world > 1:
            self.dist.destroy_process_group()


# ------------------------------------------------------------------------------------ B200 arm
KERNELS = {  # rips_timings field -> kernel
    "enumerate_ms": "enumerate_apparent_kernel (a3-a5+a7 fused enumerate, filter, apparent test)",
    "sort_pass_ms": "onesweep_pass_kernel (a6 filtration sort)",
    "pair_sort_ms": "onesweep_pass_kernel (a9 pair partition by cofacet vertex)",
}


def algorithmic_bytes(field, st):
    """HBM bytes ONE launch of the kernel must move, from rips_stats of that dimension."""
    if field == "enumerate_ms":   # clearing bitmap read; one column record and one pair record written per slot
        if st["n_removed_by_diameter"] > 0 and st["n_slots"] == st["n_columns"] + st["n_cleared"] and st["n_slots"] < st["n_candidates"]:
            return 3 * RECORD_BYTES * st["n_slots"], 1    # sparse path: the simplex list read instead of a bitmap
        return st["n_candidates"] / 8 + 2 * RECORD_BYTES * st["n_slots"], 1
    if field == "sort_pass_ms":   # each pass reads and writes every record once
        return 2 * RECORD_BYTES * st["n_slots"], max(1, st["sort_passes"])
    if field == "pair_sort_ms":
        return 2 * RECORD_BYTES * st["n_slots"], max(1, st["pair_sort_passes"])
    raise KeyError(field)


def source_stamp():
    """sha256 over the kernel sources: profiles/traffic.json carries the stamp of the build it was captured from."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2003_07989_b200", "csrc")
    for f in sorted(os.listdir(d)):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def compute_all(g, w, reduce_upto):
    """dim 0, then per dimension stage 1, stage 2 and (up to reduce_upto) the reduction."""
    g.dim0()
    for d in range(1, w.dim_max + 1):
        g.stage1(d)
        g.stage2(d)
        if d <= reduce_upto:
            g.reduce(d)


def run_b200(args):
    import torch

    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the product has no CPU fallback"
    torch.cuda.set_device(local)
    ranks = Ranks("nccl", torch.device("cuda", local))
    rank, world, barrier = ranks.rank, ranks.world, ranks.barrier
    from paper_2003_07989_b200 import inputs, rips
    rips.lib()

    w = inputs.config(args.config, args.n)
    D = w.dim_max
    # config 3 (random matrix): the reduced columns of dimension 2 do not fit any device: its
    # barcodes stop at dimension 1; the hot path (stage 1 + stage 2) runs in every dimension
    reduce_upto = 1 if args.config == 3 else D
    if args.config == 6:      # the second workload measures the apparent fraction of dimension 1: stage 1 + stage 2 only
        reduce_upto = 0
    n_cand = sum(comb(w.n, d + 1) for d in range(1, D + 1))
    host = torch.from_numpy(w.dist).pin_memory()
    dev = host.cuda()
    wsize = rips.rips_workspace_bytes(w.n, D)
    free_b, _ = torch.cuda.mem_get_info()
    if args.config == 3:      # the reduced columns of its dimension 1 fill in: 42 GB of arena
        wsize = max(wsize, 72 << 30)
    # (allocated before the resident context, whose own workspace grows with what its reduction needs)
    workspace = torch.empty(min(wsize, int(free_b * 0.42)), dtype=torch.uint8, device="cuda")

    # ---- resident context; one full computation provides the clearing sets (and the barcode time)
    g = rips.Rips(dev, w.n, D, w.threshold)
    g.set_mode(args.mode)
    t0 = time.perf_counter()
    compute_all(g, w, reduce_upto)
    torch.cuda.synchronize()
    first_compute_ms = 1e3 * (time.perf_counter() - t0)
    stats = {d: g.stats(d) for d in range(0, D + 1)}

    def hot_step():
        for d in range(1, D + 1):
            g.stage1(d)
            g.stage2(d)

    # ---- clocks are sampled from the warm-up on (nvidia-smi needs ~0.2 s to start) through the timed region
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    t_w = time.perf_counter()
    n_w = 0
    while n_w < args.warmup or (time.perf_counter() - t_w < args.warmup_seconds and n_w < 200):
        hot_step()
        n_w += 1
    torch.cuda.synchronize()
    launches0 = g.kernel_launches()
    barrier()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    evs[0].record()
    for i in range(args.steps):      # nothing in the timed region waits for the device: the steps are enqueued back to back
        hot_step()
        evs[i + 1].record()
    barrier()
    elapsed_ms = evs[0].elapsed_time(evs[-1])
    step_ms = sorted(evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps))
    launches = g.kernel_launches() - launches0
    # the library's own CUDA events (per kernel) of the LAST timed step, then of a few more steps run one by one
    per_kernel = {k: 0.0 for k in KERNELS}
    per_kernel_dim = {k: {d: 0.0 for d in range(1, D + 1)} for k in KERNELS}
    n_prof = 0
    for rep in range(1 + 4):
        if rep:
            hot_step()
        for d in range(1, D + 1):
            t = g.timings(d)            # synchronises
            for k in KERNELS:
                per_kernel[k] += t[k]
                per_kernel_dim[k][d] += t[k]
        n_prof += 1
    clocks = sampler.stop() if rank == 0 else None
    ms_per_step = ranks.max_over_ranks(elapsed_ms) / args.steps
    value = world * n_cand / (ms_per_step * 1e-3)

    # ---- the step WITH the arrays the ABI promises (fp32 diameter + u64 index filtration, (t, s) pair arrays):
    # stage 1 + stage 2 + rips_filtration / rips_apparent_pairs / rips_nonapparent of every dimension
    lib, C = rips.lib(), rips.C
    def outputs():
        a, b, k = C.c_void_p(), C.c_void_p(), C.c_int64()
        for d in range(1, D + 1):
            for fn in ("rips_filtration", "rips_apparent_pairs", "rips_nonapparent"):
                rc = getattr(lib, fn)(g._h, d, C.byref(a), C.byref(b), C.byref(k))
                assert rc == 0, (fn, d, rc)
    with_out = []
    try:
        for i in range(2 + min(args.steps, 5)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); hot_step(); outputs(); e1.record()
            torch.cuda.synchronize()
            if i >= 2:
                with_out.append(e0.elapsed_time(e1))
        step_with_outputs = {"ms_per_step": statistics.median(with_out), "value": world * n_cand / (statistics.median(with_out) * 1e-3),
                             "unit": UNIT, "what": "stage 1 + stage 2 + rips_filtration + rips_apparent_pairs + rips_nonapparent of every "
                             "dimension (unpack / merge kernels materialise the fp32 + u64 arrays of include/rips.h)"}
    except rips.RipsError as e:
        step_with_outputs = {"unavailable": str(e)}

    # ---- roofline of the dominant kernel (largest share of the timed region)
    peak, peak_src = load_peaks()
    kernels = []
    for k, name in KERNELS.items():
        d_top = max(per_kernel_dim[k], key=lambda d: per_kernel_dim[k][d])
        b, nl = algorithmic_bytes(k, g.stats(d_top))
        ms_launch = per_kernel_dim[k][d_top] / n_prof / nl
        kernels.append({"kernel": name, "dim": d_top, "ms_per_step_all_dims": per_kernel[k] / n_prof,
                        "ms_per_launch": ms_launch, "launches_per_step": nl, "bytes_per_launch": b,
                        "gbs": (b / (ms_launch * 1e-3) / 1e9) if ms_launch > 0 else 0.0,
                        "frac_of_peak": (b / (ms_launch * 1e-3) / 1e9 / peak) if ms_launch > 0 else 0.0,
                        "share_of_step": per_kernel[k] / n_prof / ms_per_step})
    top = max(kernels, key=lambda r: r["ms_per_step_all_dims"])
    roofline = {"bound": "hbm", "kernel": top["kernel"], "dim": top["dim"], "achieved": top["gbs"], "peak": peak,
                "unit": "GB/s", "frac": top["frac_of_peak"], "traffic": None, "peak_source": peak_src,
                "bytes_per_launch": top["bytes_per_launch"], "ms_per_launch": top["ms_per_launch"],
                "nominal_peak_gbs": 8000.0, "frac_of_nominal": top["gbs"] / 8000.0,
                "kernels_ms_per_step": sum(r["ms_per_step_all_dims"] for r in kernels),
                "not_in_kernels_ms": ms_per_step - sum(r["ms_per_step_all_dims"] for r in kernels)}
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_file):
        with open(traffic_file) as f:
            tj = json.load(f)
        if tj.get("source_stamp") == source_stamp():   # captured from this very build; dropped silently once the kernels change
            key = f"cfg{args.config}:{top['kernel'].split(' ')[0]}:{'a9' if 'a9' in top['kernel'] else 'a6' if 'a6' in top['kernel'] else ''}"
            roofline["traffic"] = tj.get(key)
            inst = tj.get(key + ":inst")
            if inst and top["ms_per_launch"] > 0:
                # the fused kernel is bound by instruction issue, not by HBM: SMs x 4 schedulers x clock
                peak_inst = 148 * 4 * 1.965e9
                roofline["issue"] = {"warp_inst_per_launch": inst, "achieved_ginst_s": inst / (top["ms_per_launch"] * 1e-3) / 1e9,
                                     "peak_ginst_s": peak_inst / 1e9, "frac": inst / (top["ms_per_launch"] * 1e-3) / peak_inst,
                                     "note": "ncu smsp__inst_executed.sum / live duration; what actually binds this kernel"}
                roofline["bound_actual"] = "issue"
        else:
            roofline["traffic_note"] = "profiles/traffic.json was captured from other kernel sources: not quoted"

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region); the workspace is the
    # caller's (one torch allocation reused by every iteration: nothing allocates device memory inside)
    e2e_ms, d2h_bytes, parts = [], 0, None
    for i in range(args.e2e_steps + 1 if args.e2e_steps > 0 else 0):
        barrier()
        t0 = time.perf_counter()
        h = rips.Rips(host.numpy(), w.n, D, w.threshold, workspace=workspace)
        h.set_mode(args.mode)
        compute_all(h, w, reduce_upto)
        bars = [h.barcodes(d) for d in range(0, reduce_upto + 1)]
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        if i > 0:   # the first one warms up
            e2e_ms.append(1e3 * (t1 - t0))
        d2h_bytes = sum(b.nbytes for b in bars)
        tim = {d: h.timings(d) for d in range(0, D + 1)}
        parts = {"dim0_ms": tim[0]["dim0_ms"],
                 "hot_path_ms": sum(tim[d]["stage1_ms"] + tim[d]["stage2_ms"] for d in range(1, D + 1)),
                 "reduce_device_ms": sum(tim[d]["reduce_device_ms"] for d in range(1, D + 1)),
                 "reduce_host_ms": sum(tim[d]["reduce_host_ms"] for d in range(1, D + 1)),
                 "reduce_xfer_ms": sum(tim[d]["reduce_xfer_ms"] for d in range(1, D + 1)),
                 "reduce": {str(d): {k: h.stats(d)[k] for k in ("n_nonapparent", "n_additions", "n_reduce_serial", "n_reduce_displaced",
                                                                 "reduce_arena_bytes")} for d in range(1, reduce_upto + 1)},
                 "barcodes_of_dimensions": list(range(0, reduce_upto + 1)),
                 "workspace_bytes": int(workspace.numel()), "workspace_peak_bytes": h.workspace_in_use()[1],
                 "bars": {str(d): int(b.shape[0]) for d, b in enumerate(bars)}}
        h.free()
    e2e_t = statistics.median(e2e_ms) if e2e_ms else float("nan")
    e2e_t = ranks.max_over_ranks(e2e_t)
    e2e = {"value": world * n_cand / (e2e_t * 1e-3), "unit": UNIT, "ms": e2e_t,
           "h2d_bytes_per_step": int(host.numel() * 4), "d2h_bytes_per_step": int(d2h_bytes),
           "what": "rips_init(host matrix, caller's workspace) + dim 0 + per dimension stage 1, stage 2, reduction + rips_barcodes(host) + rips_free"}

    # ---- scale row: the same kernels one dimension up, on the simplices the config names
    scale = None
    if not args.no_scale_row and D + 1 <= 4 and reduce_upto == D:
        del workspace
        torch.cuda.empty_cache()
        need = 5 * 8 * comb(w.n, D + 2) + (1 << 30)
        free_b, _ = torch.cuda.mem_get_info()
        if need < free_b:
            reps = []
            for _ in range(3):
                barrier()
                e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
                e0.record(); g.stage1(D + 1); e1.record(); g.stage2(D + 1); e2.record()
                torch.cuda.synchronize()
                reps.append((e0.elapsed_time(e1), e1.elapsed_time(e2), g.timings(D + 1)))
            s1, s2, tm = min(reps, key=lambda r: r[0] + r[1])
            st = g.stats(D + 1)
            nbytes = 2 * RECORD_BYTES * st["n_slots"]
            scale = {"what": f"rips_stage1({D + 1}) + rips_stage2({D + 1}) with the pivots of dimension {D} as the clearing set",
                     "candidates": st["n_candidates"], "columns": st["n_columns"], "apparent": st["n_apparent"],
                     "stage1_ms": s1, "stage2_ms": s2,
                     "simplices_per_s": world * st["n_candidates"] / ((ranks.max_over_ranks(s1 + s2)) * 1e-3),
                     "fused_kernel_ms": tm["enumerate_ms"], "fused_kernel_gbs": (nbytes + st["n_candidates"] / 8) / tm["enumerate_ms"] / 1e6,
                     "fused_kernel_frac_of_peak": (nbytes + st["n_candidates"] / 8) / tm["enumerate_ms"] / 1e6 / peak,
                     "filtration_sort_pass_ms": tm["sort_pass_ms"] / max(1, st["sort_passes"]),
                     "filtration_sort_pass_gbs": nbytes / (tm["sort_pass_ms"] / max(1, st["sort_passes"])) / 1e6,
                     "filtration_sort_pass_frac_of_peak": nbytes / (tm["sort_pass_ms"] / max(1, st["sort_passes"])) / 1e6 / peak,
                     "pair_partition_pass_ms": tm["pair_sort_ms"] / max(1, st["pair_sort_passes"]),
                     "pair_partition_pass_gbs": nbytes / (tm["pair_sort_ms"] / max(1, st["pair_sort_passes"])) / 1e6,
                     "pair_partition_pass_frac_of_peak": nbytes / (tm["pair_sort_ms"] / max(1, st["pair_sort_passes"])) / 1e6 / peak,
                     "hbm_bytes": 4 * nbytes + st["n_candidates"] / 8,
                     "overall_gbs": (4 * nbytes + st["n_candidates"] / 8) / (s1 + s2) / 1e6,
                     "device_bytes": g.device_bytes()}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        s, t, cores, desc, _ = oracle_sample(w, args.cpu_seconds)
        cpu = {"value": s / t, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": t}
        # the same sample at one thread (a shorter one), and the oracle's barcodes single-threaded on what it finishes
        oracle.set_threads(1)
        s1, t1, _, desc1, _ = oracle_sample(w, max(3.0, args.cpu_seconds / 3))
        cpu["one_thread"] = {"value": s1 / t1, "unit": UNIT, "cores": 1, "sample": desc1, "seconds": t1}
        dlow = min(D, 2) if args.config != 3 else 1
        t0 = time.perf_counter()
        oracle.barcodes(w.dist, w.n, dlow, w.threshold, explicit=(args.config == 3)) if (args.config != 3 or args.cpu_seconds >= 60) else None
        cpu["barcodes_one_thread"] = {"seconds": time.perf_counter() - t0, "dimensions": f"0..{dlow}",
                                      "what": "oracle.barcodes (stage 1, stage 2, reduction) with one thread" +
                                              ("" if (args.config != 3 or args.cpu_seconds >= 60) else ": skipped (about 40 s; pass --cpu-seconds 60)")}
        oracle.set_threads(cores)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": n_w, "ms_per_step": ms_per_step, "ms_per_step_median": statistics.median(step_ms),
                "ms_per_step_best": step_ms[0], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
                "config": workload_dict(w, n_cand), "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
                "roofline": roofline, "cpu_baseline": cpu, "step_with_outputs": step_with_outputs,
                "kernels": kernels, "scale_row": scale,
                "barcode": {"end_to_end_ms": e2e_t, "first_compute_ms": first_compute_ms, **(parts or {})},
                "stats": {str(d): {k: stats[d][k] for k in ("n_candidates", "n_columns", "n_cleared",
                                                            "n_removed_by_diameter", "n_apparent", "n_regular",
                                                            "n_nonapparent", "n_slots", "sort_passes",
                                                            "pair_sort_passes", "key_bits", "index_bits")} for d in range(1, D + 1)},
                "device_bytes": g.device_bytes(), "parallelism": "replicas" if world > 1 else "single"}
        line["mode"] = {0: "auto", 1: "dense", 2: "sparse"}[args.mode] + (" (sparse path taken)" if stats[D]["n_slots"] != comb(w.n, D + 1) and stats[D]["n_removed_by_diameter"] > 0 and stats[D]["n_slots"] == stats[D]["n_columns"] + stats[D]["n_cleared"] else "")
        if args.config == 6:
            import math
            closed = 1 - (math.sqrt(math.pi) / 2) * math.exp(math.lgamma(w.n - 1) - math.lgamma(w.n - 0.5))
            line["apparent_fraction"] = {"measured": stats[1]["n_apparent"] / comb(w.n, 2), "closed_form": closed,
                                         "paper": {"10000": 0.991127743, "20000": 0.993733522}.get(str(w.n)),
                                         "what": "apparent pairs of dimension 1 / C(n,2) (PAPER.md:723, :729)"}
        print(json.dumps(line))
    g.free()
    ranks.close()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
