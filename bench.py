#!/usr/bin/env python
"""bench.py -- one H and one H^T (the whole hot path) per step on the
configuration BASELINE.json's metric is quoted on: config 3, 240^3 voxels x 9,216 transducers x
2,048 time samples (arc-array geometry), synthetic seeded phantom and data.

    python bench.py --gpus N --steps K --warmup W            (our arm, CUDA)
    python bench.py --impl reference --steps K --warmup W    (the fp64 oracle on host cores)

Prints ONE JSON line (DESIGN.md §7 explains every field).  Timing: CUDA events on the launching
stream, barrier + synchronize on both sides, max over ranks; L2 is flushed between steps.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ms per H and per H^T at 240^3 voxels x 9216 transducers x 2048 t (value = ms per H + H^T pair)"
# Algorithmic work per interpolation sample: 8 corners x 4 B gathered at L1 level; ~30 fp32 lane-operations
# (3 FMA position, 3 floor + 3 fraction, ~14 weights / lerps, 1 accumulate, rest bounds).
L1_BYTES_PER_SAMPLE = 32.0
LANE_OPS_PER_SAMPLE = 30.0
# B200 unit counts (guide): 148 SMs; L1 delivers 128 B per clock per SM; 128 fp32 lanes per SM
N_SM, L1_BYTES_PER_CLK, FP32_LANES = 148, 128, 128
# ncu captures of the SHIPPING marching kernels on the 512-transducer subset of config 3 (profiles/r2_march_counters.md
# names the commands and the library revision): `ncu -i ... --page raw --csv` dumps, parsed below for the per-sample counters
PROFILE_FWD = os.path.join(ROOT, "profiles", "r2_march_fwd_raw.csv")
PROFILE_BWD = os.path.join(ROOT, "profiles", "r2_march_bwd_raw.csv")
PROFILE_META = os.path.join(ROOT, "profiles", "r2_march_counters.json")


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    sm_mhz, hbm, src = 1965.0, 6650.0, "fallback of B200_PROFILING.md (clocks.max.sm 1965 MHz, 6.65 TB/s)"
    if os.path.exists(path):
        try:
            mp = json.load(open(path))
            sm_mhz = float(mp.get("sm_max_mhz", sm_mhz)); hbm = float(mp.get("hbm_gbs", hbm))
            src = "MEASURED_PEAKS.json (sm_max_mhz, hbm_gbs)"
        except Exception:
            pass
    return sm_mhz, hbm, src


def ncu_counters():
    """Per-sample counters of the two marching kernels from the committed ncu raw pages ({"error": ...} when unreadable)."""
    unit = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}

    def raw(path):
        rows = list(csv.reader(open(path)))
        return dict(zip(rows[0], rows[2])), dict(zip(rows[0], rows[1]))

    def num(d, k):
        return float(d[k].replace(",", ""))

    def dram(d, u):
        return sum(num(d, k) * unit.get(u[k], 1.0) for k in ("dram__bytes_read.sum", "dram__bytes_write.sum"))
    try:
        meta = json.load(open(PROFILE_META))
        ns = float(meta["in_box_samples_per_launch"])
        (f, uf), (b, ub) = raw(PROFILE_FWD), raw(PROFILE_BWD)
        return {"samples": ns, "revision": meta.get("library_revision"),
                "H_sectors_per_sample": num(f, "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum") / ns,
                "H_inst_per_sample": num(f, "smsp__inst_executed.sum") * 32.0 / ns,
                "H_dram_bytes_per_sample": dram(f, uf) / ns,
                "HT_red_lanes_per_sample": num(b, "l1tex__t_sectors_pipe_lsu_mem_global_op_red.sum") / ns,
                "HT_inst_per_sample": num(b, "smsp__inst_executed.sum") * 32.0 / ns,
                "HT_dram_bytes_per_sample": dram(b, ub) / ns}
    except Exception as ex:
        return {"error": f"{type(ex).__name__}: {ex}"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (profiling recipe's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu, self.proc, self.path = gpu_index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            sm, mx, reasons = [], [], set()
            for line in open(self.path):
                f = [s.strip() for s in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); mx.append(float(f[2]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            if sm:
                out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}
            os.unlink(self.path)
        except Exception:
            pass
        return out


def workload(args):
    from paper_1304_2017_b200 import workloads as wl
    w = wl.config(args.config)
    note = None
    if args.subset and args.subset < w.n_trans:
        _, w = w.seeded_subset(args.subset)
        note = f"DEBUG subset of {args.subset} transducers: not the BASELINE workload"
    if args.kband:
        from dataclasses import replace
        w = replace(w, kband=args.kband)
        note = ((note + "; ") if note else "") + (f"NON-BASELINE angular rule: B = {args.kband} time samples per rule (B = 1 is the paper's literal per-sample "
                                                  "Eq. 37; any B < 32 runs on the generic patch kernel, not the marching kernels)")
    return w, note


def dense_data(w):
    """The data vector H^T is timed on: dense seeded N(0,1), config 1's recipe (no band of 32 samples is all zero, so
    the kernel skips nothing; y = H x of the sparse vessel phantom would leave ~5 % of the samples in skipped bands)."""
    rng = np.random.default_rng(w.seed + 101)
    return rng.standard_normal((w.n_trans, w.nt)).astype(np.float32)


def oracle_step(w, x64, sample_q, n_threads=0):
    """One H + one H^T of the oracle on `sample_q` seeded transducers; returns (s_H, s_HT, n_trans)."""
    from oracle import oat_oracle as orc
    _, ws = w.seeded_subset(sample_q)
    kw = {"n_threads": n_threads} if n_threads else {}
    t0 = time.perf_counter()
    y = orc.project(ws, x64, **kw)
    t1 = time.perf_counter()
    orc.backproject(ws, y, **kw)
    t2 = time.perf_counter()
    return t1 - t0, t2 - t1, ws.n_trans


def parallelism_note(world, scaling):
    return "1 GPU" if world == 1 else (f"{world} GPUs, transducers sharded ({scaling}" +
                                       (f": {world}x denser views" if scaling == "weak" else ": rows of H partitioned") +
                                       "), H^T partial volumes all-reduced over NCCL")


def config_object(w, args, note, world):
    """The `config` of the JSON line: the workload and the step, nothing that depends on which arm runs it, so that the
    GPU arm and `--impl reference` print the same object."""
    return {"workload": f"{w.name}: {w.nx}x{w.ny}x{w.nz} voxels @ {w.spacing} mm, {w.n_trans} transducers/GPU, nt={w.nt}, h={w.surf_step}, B={w.kband}",
            "step": "one H (phantom x -> y) followed by one H^T (dense data of the same shape -> x)",
            "l2": "GPU arm: inputs resident in HBM, L2 flushed between steps (256 MB fill)", "note": note,
            "parallelism": parallelism_note(world, args.scaling)}


def oracle_sample_size(want, n_trans, threads):
    """The oracle parallelises over transducers only: a sample keeps every core busy when it is a multiple of the
    thread count."""
    sq = max(1, min(want, n_trans))
    if threads > 1 and sq >= threads:
        sq -= sq % threads
    return sq


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oat_oracle as orc
    w, note = workload(args)
    x64 = w.phantom().astype(np.float64)
    threads = orc.max_threads()
    sq = oracle_sample_size(args.ref_sample if args.ref_sample > 0 else threads, w.n_trans, threads)   # default: every host thread busy
    for _ in range(args.warmup):
        oracle_step(w, x64, min(threads, sq))
    th = tt = 0.0
    for _ in range(args.steps):
        a, b, nq = oracle_step(w, x64, sq)
        th += a; tt += b
    scale = w.n_trans / sq
    ms_h, ms_t = th / args.steps * 1e3 * scale, tt / args.steps * 1e3 * scale
    cores = min(threads, sq)
    sample = f"{sq} of {w.n_trans} transducers per step (seeded subset, {cores} threads busy), times scaled by {scale:.0f}x"
    metric = METRIC if (args.config == 3 and not args.subset) else f"ms per H and per H^T on {w.name} (value = ms per H + H^T pair)"
    line = {"impl": "reference", "metric": metric, "value": ms_h + ms_t, "unit": "ms", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_h + ms_t, "higher_is_better": False,
            "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_object(w, args, note, max(1, args.gpus)),
            "ms_H": ms_h, "ms_HT": ms_t,
            "cpu_baseline": {"value": ms_h + ms_t, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": ms_h + ms_t, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def timed(torch, stream, fn, reps=5):
    fn(); torch.cuda.synchronize()
    a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(reps):
        fn()
    b.record(stream); torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def run_ours(args):
    import torch
    import torch.distributed as dist
    from dataclasses import replace
    from paper_1304_2017_b200 import binding as oat, build, shard, workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")           # the communicator log (stderr) shows every rank
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()

    w_all, note = workload(args)
    w = w_all
    if world > 1 and args.scaling == "strong":              # rows of H partitioned: total work fixed
        w = replace(w_all, trans_xyz=shard.shard_transducers(w_all.trans_xyz, rank, world))
    elif world > 1:                                         # weak: N-times denser view sampling, per-GPU work fixed
        w = replace(w_all, trans_xyz=shard.weak_replica_transducers(w_all.trans_xyz, rank, world, 144))
    g = oat.oat_geometry_create(w, local)
    if args.project_variant != 4:                           # measurement aid: 5 = the tile-stationary projection kernel (not the default)
        oat.oat_set_variant(g, "project", args.project_variant)
        note = ((note + "; ") if note else "") + f"NON-DEFAULT projection kernel variant {args.project_variant} (include/oat_probe.h)"
    if args.backproject_variant != 4:                       # measurement aid: 0 = the generic patch kernel
        oat.oat_set_variant(g, "backproject", args.backproject_variant)
        note = ((note + "; ") if note else "") + f"NON-DEFAULT backprojection kernel variant {args.backproject_variant} (include/oat_probe.h)"
    x = torch.from_numpy(w.phantom()).cuda()
    y = torch.empty((w.n_trans, w.nt), dtype=torch.float32, device="cuda")
    ynoise = torch.from_numpy(dense_data(w)).cuda()
    xb = torch.empty_like(x)
    n_samples = oat.oat_num_surface_samples(g)              # per operator, this rank
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step(rec=None, kernel_ms=None):
        """One H + one H^T.  The timed loop (rec given) only enqueues: no host synchronisation between or inside steps.
        kernel_ms given (the untimed pass after the timed region): also reads the library's own event pair around the
        marching kernel after each operator, which waits for it (oat_last_kernel_ms synchronises on the event)."""
        flush.fill_(1)                                      # L2 flush between timed iterations
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)] if rec is not None else None
        if e: e[0].record(stream)
        oat.oat_project(g, x, y)
        kh = oat.oat_last_kernel_ms(g) if kernel_ms is not None else 0.0
        nl = oat.oat_last_launch_count(g)
        if e: e[1].record(stream)
        oat.oat_backproject(g, ynoise, xb)
        kt = oat.oat_last_kernel_ms(g) if kernel_ms is not None else 0.0
        nl += oat.oat_last_launch_count(g)
        if world > 1:
            shard.allreduce_volume(xb)                      # the path's one exchange step (H^T only)
        if e:
            e[2].record(stream)
            rec.append((e, nl))
        if kernel_ms is not None:
            kernel_ms.append((kh, kt))

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    rec = []
    t_begin = torch.cuda.Event(enable_timing=True); t_end = torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t_begin.record(stream)
    for _ in range(args.steps):
        step(rec)
    t_end.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    total_ms = t_begin.elapsed_time(t_end)
    ms_h = float(np.mean([r[0][0].elapsed_time(r[0][1]) for r in rec]))
    ms_t = float(np.mean([r[0][1].elapsed_time(r[0][2]) for r in rec]))
    launches = int(sum(r[1] for r in rec)) + args.steps      # + the L2-flush fill per step
    # kernel-only durations (the roofline's denominator): the library's event pair around the marching kernel, read in an
    # UNTIMED pass over the same inputs (same L2 flush) right after the timed region, so that the timed loop holds no host sync
    kms = []
    n_kernel_pass = max(1, min(args.steps, 5))
    for _ in range(n_kernel_pass):
        step(None, kms)
    torch.cuda.synchronize()
    k_h = float(np.mean([k[0] for k in kms])); k_t = float(np.mean([k[1] for k in kms]))
    vals = torch.tensor([total_ms, ms_h, ms_t, k_h, k_t], dtype=torch.float64, device="cuda")
    tot_samples = torch.tensor([float(n_samples)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot_samples, op=dist.ReduceOp.SUM)
    total_ms, ms_h, ms_t, k_h, k_t = [float(v) for v in vals.tolist()]
    ms_step = total_ms / args.steps

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region)
    e2e = None
    if args.e2e_steps > 0:
        hx = torch.from_numpy(w.phantom()).pin_memory()
        hy = torch.empty((w.n_trans, w.nt), dtype=torch.float32).pin_memory()
        hyn = torch.from_numpy(dense_data(w)).pin_memory()
        hxb = torch.empty_like(hx).pin_memory()
        n_e2e = args.e2e_steps
        oat.oat_project_host(g, hx, hy); oat.oat_backproject_host(g, hyn, hxb)     # warm-up
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            oat.oat_project_host(g, hx, hy)
            oat.oat_backproject_host(g, hyn, hxb)
        dt_e2e = (time.perf_counter() - t0) / n_e2e * 1e3
        v = torch.tensor([dt_e2e], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(v, op=dist.ReduceOp.MAX)
        bx, by = x.numel() * 4, y.numel() * 4
        e2e = {"value": float(v.item()), "unit": "ms", "h2d_bytes_per_step": bx + by, "d2h_bytes_per_step": by + bx,
               "steps": n_e2e, "api": "oat_project_host + oat_backproject_host (pinned host buffers)"}

    # ---- N > 1: the spherical-voxel pair behind the same transducer split (rows of H_sph per transducer: no exchange;
    # H_sph† sums over transducers: one all-reduce) -- the paper's own multi-GPU case (L243-245, Algs. 7-12), every rank runs it
    sph_sharded = None
    if world > 1 and not args.no_next:
        try:
            _, ws3_all = w_all.seeded_subset(256)
            ws3 = replace(ws3_all, trans_xyz=shard.shard_transducers(ws3_all.trans_xyz, rank, world))
            g3 = oat.oat_geometry_create(ws3, local)
            nf3 = 64
            oat.oat_sph_set(g3, nf3, 0.0, 0.078125)
            u3 = torch.empty((ws3.n_trans, nf3), dtype=torch.complex64, device="cuda")
            xs = torch.empty_like(x)

            def sph_pair():
                oat.oat_sph_project(g3, x, u3)
                oat.oat_sph_backproject(g3, u3, xs)
                shard.allreduce_volume(xs)
            sph_pair(); torch.cuda.synchronize(); dist.barrier()
            ms = timed(torch, stream, sph_pair, reps=2)
            vv = torch.tensor([ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(vv, op=dist.ReduceOp.MAX)
            sph_sharded = {"ms_pair": float(vv.item()), "n_trans_total": ws3_all.n_trans, "n_freq": nf3,
                           "split": f"{world} ranks, rows of H_sph partitioned, H_sph† partial volumes all-reduced"}
            g3.close()
        except Exception as ex:
            sph_sharded = {"error": str(ex)}

    if rank == 0:
        sm_mhz, hbm_gbs, peak_src = measured_peaks()
        clk = sm_mhz * 1e6
        peak_l1 = N_SM * L1_BYTES_PER_CLK * clk / 1e9        # GB/s
        peak_alu = N_SM * FP32_LANES * clk                    # lane-ops/s
        cnt = ncu_counters()

        def kernel_roofline(name, k_ms, dram_per_sample):
            ach = n_samples * L1_BYTES_PER_SAMPLE / (k_ms * 1e-3) / 1e9 if k_ms > 0 else 0.0
            ops = n_samples * LANE_OPS_PER_SAMPLE / (k_ms * 1e-3) if k_ms > 0 else 0.0
            return {"kernel": name, "kernel_ms": k_ms, "achieved": ach, "peak": peak_l1, "unit": "GB/s", "frac": ach / peak_l1,
                    "frac_alu": ops / peak_alu, "samples_per_sm_cycle": n_samples / (k_ms * 1e-3) / (N_SM * clk) if k_ms > 0 else None,
                    "traffic": dram_per_sample * n_samples if dram_per_sample is not None else None}
        march_h, march_t = oat.oat_uses_marching(g), oat.oat_uses_marching(g, backproject=True)
        name_h = "oat_march_fwd_kernel" if march_h else ("oat_tile_kernel" if args.project_variant == 5 else "oat_patch_kernel (generic)")
        name_t = "oat_march_bwd_kernel" if march_t else "oat_patch_kernel (generic)"
        # the committed ncu counters are of the marching kernels: they say nothing about another variant
        r_t = kernel_roofline(name_t + " (backproject)", k_t, cnt.get("HT_dram_bytes_per_sample") if march_t else None)
        r_h = kernel_roofline(name_h + " (project)", k_h, cnt.get("H_dram_bytes_per_sample") if march_h else None)
        r_t["bound_ncu"] = "l2 reduction rate (scattered RED.128 sectors) + issue slots" if march_t else None
        r_h["bound_ncu"] = "l2 latency (long scoreboard on the record load) under a 77 %-busy L1 data stage" if march_h else None
        dom, other = (r_t, r_h) if k_t >= k_h else (r_h, r_t)
        roofline = dict(dom)
        roofline.update({
            "bound": "l1",
            "bound_note": "'l1' names the SURVEY 8(d) ceiling the fraction is taken against (algorithmic bytes gathered at L1 level); it is an "
                          "algorithmic-bytes figure, not the unit that limits the kernel. ncu of the shipping kernels (profiles/r2_march_counters.md) names "
                          "that unit: see bound_ncu here and in other_kernel, and limiter_diagnostics for the probe rates of those units",
            "kernel_ms_source": f"library event pair around the kernel, mean of {n_kernel_pass} launches in an untimed pass right after the timed region "
                                "(same inputs, L2 flushed); the timed loop itself holds no host synchronisation",
            "kernel_share_of_step": dom["kernel_ms"] / ms_step if ms_step else None,
            "other_kernel": other,
            "algorithmic": f"SURVEY 8(d): {L1_BYTES_PER_SAMPLE:.0f} B gathered at L1 level (frac) and {LANE_OPS_PER_SAMPLE:.0f} fp32 lane-operations (frac_alu) per "
                           f"interpolation sample x {n_samples:.4g} in-box samples per launch; unique HBM bytes per launch = size(x) + size(y) = {(x.numel() + y.numel()) * 4:.4g} B",
            "peak_source": f"148 SM x 128 B/clk (L1) resp. 148 SM x 128 fp32 lanes, x max SM clock of {peak_src}; the L1-bytes ceiling is the tighter of the two",
            "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum of this kernel per launch: ncu --set full of the shipping kernel on the 512-transducer "
                            "subset of config 3 (profiles/r2_march_*_raw.csv), per in-box sample x this launch's samples; unit B",
            "ncu_counters": cnt})
        # Diagnostics, self-measured in this run by the library's own probe kernels (include/oat_probe.h).  NOT roofline
        # fractions: neighbouring rays share sectors, so the kernels can exceed the scattered-access rates.
        diag = {"note": "self-measured probe rates of the two hardware paths ncu names as the kernels' limiters; diagnostics, not a roofline"}
        try:
            if "HT_red_lanes_per_sample" in cnt:
                red_scat = oat.oat_measure_red_rate(local)
                ach = cnt["HT_red_lanes_per_sample"] * n_samples / (k_t * 1e-3) if k_t > 0 else None
                diag["H^T"] = {"unit": "RED.128 lanes/s into L2", "achieved": ach, "probe_scattered_sectors": red_scat,
                               "probe_packed_sectors": oat.oat_measure_red_rate_ex(local, 1),
                               "achieved_over_scattered_probe": ach / red_scat if (ach and red_scat > 0) else None}
            if "H_sectors_per_sample" in cnt:
                gat = oat.oat_measure_gather_rate(local)
                ach = cnt["H_sectors_per_sample"] * n_samples / (k_h * 1e-3) if k_h > 0 else None
                diag["H"] = {"unit": "scattered 32 B sector loads/s (L1 misses served by L2)", "achieved": ach, "probe": gat,
                             "achieved_over_probe": ach / gat if (ach and gat > 0) else None}
        except Exception as ex:
            diag["error"] = str(ex)
        roofline["limiter_diagnostics"] = diag

        next1 = next2 = next3 = None
        if sph_sharded is not None:
            next3 = {"sharded": sph_sharded}
        if not args.no_next and world == 1:
            # ---- row NEXT-1 (EIR convolution, penalty stencil): the steps either side of the path, timed at this config's sizes
            try:
                taps = 128
                tt = np.arange(taps) * w.dt
                oat.oat_eir_set(g, (w.dt * np.exp(-tt / (0.15 * taps * w.dt)) * np.sin(2 * np.pi * 2.5 * tt)).astype(np.float32))
                u = torch.empty_like(y); lx = torch.empty_like(x)
                ms_e = timed(torch, stream, lambda: oat.oat_eir_apply(g, ynoise, u))
                ms_ea = timed(torch, stream, lambda: oat.oat_eir_apply(g, ynoise, u, adjoint=True))
                ms_p = timed(torch, stream, lambda: oat.oat_penalty_apply(g, xb, lx))
                by, bx = 2.0 * y.numel() * 4, 2.0 * x.numel() * 4          # read + write once
                fma = float(taps) * y.numel()                               # one FMA per tap and output
                next1 = {"eir_taps": taps, "ms_eir": ms_e, "ms_eir_adjoint": ms_ea, "ms_penalty": ms_p,
                         "roofline_eir": {"bound": "alu", "unit": "fp32 lane-operations/s", "achieved": fma / (ms_e * 1e-3), "peak": peak_alu,
                                          "frac": fma / (ms_e * 1e-3) / peak_alu, "frac_hbm": by / (ms_e * 1e-3) / 1e9 / hbm_gbs,
                                          "algorithmic": "128 FMAs per output against 148 SM x 128 fp32 lanes (frac: at 128 taps the FMA floor, 0.065 ms, is above the "
                                                         "HBM floor of reading + writing the Q x K vector once, 0.023 ms: frac_hbm)"},
                         "roofline_penalty": {"bound": "hbm", "achieved": bx / (ms_p * 1e-3) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                                              "frac": bx / (ms_p * 1e-3) / 1e9 / hbm_gbs, "algorithmic": "read + write of the volume once"},
                         "share_of_pls_iteration": (ms_e + ms_ea + ms_p) / (ms_step + ms_e + ms_ea + ms_p),
                         "note": "outside the timed step"}
                oat.oat_eir_set(g, np.zeros(0, dtype=np.float32))
            except Exception as ex:
                next1 = {"error": str(ex)}
            # ---- row NEXT-2 (FBP, Eq. 27): one image from the data of this config, voxel driven
            try:
                areas = wl.patch_areas_arc(64, 144, 65.0) if (args.config == 3 and not args.subset and world == 1) else wl.patch_areas_equal(w.trans_xyz, w.centre)
                wq = torch.from_numpy(oat.oat_fbp_weights(g, areas)).cuda()
                ms_f = timed(torch, stream, lambda: oat.oat_fbp(g, ynoise, wq, xb), reps=2)
                pairs = float(x.numel()) * w.n_trans
                peak_fp64 = N_SM * 64 * clk
                next2 = {"ms_fbp": ms_f, "voxel_transducer_pairs": pairs, "pairs_per_s": pairs / (ms_f * 1e-3),
                         "roofline": {"bound": "alu", "unit": "fp64 lane-operations/s", "achieved": 25.0 * pairs / (ms_f * 1e-3), "peak": peak_fp64,
                                      "frac": 25.0 * pairs / (ms_f * 1e-3) / peak_fp64,
                                      "algorithmic": "25 fp64 operations per pair (3 differences, 3 FMA, sqrt ~ 12, scale, floor, 2 conversions; reading G26 fixes fp64); "
                                                     "peak = 148 SM x 64 fp64 lanes x max SM clock"},
                         "note": "outside the timed step; fp64 distance + interval decision, fp32 brackets and sum (DESIGN.md section 5.6)"}
            except Exception as ex:
                next2 = {"error": str(ex)}
            # ---- row NEXT-3 (spherical-voxel model, frequency domain): this config's grid, 256 seeded transducers, 64 frequencies
            try:
                _, ws3 = w.seeded_subset(256)
                g3 = oat.oat_geometry_create(ws3, local)
                nf3 = 64
                oat.oat_sph_set(g3, nf3, 0.0, 0.078125)          # 0 .. 4.9 MHz
                u3 = torch.empty((ws3.n_trans, nf3), dtype=torch.complex64, device="cuda")
                xdense = torch.from_numpy(np.random.default_rng(33).standard_normal(tuple(x.shape)).astype(np.float32)).cuda()
                ms_sp = timed(torch, stream, lambda: oat.oat_sph_project(g3, x, u3), reps=2)
                ms_spd = timed(torch, stream, lambda: oat.oat_sph_project(g3, xdense, u3), reps=1)
                ms_sb = timed(torch, stream, lambda: oat.oat_sph_backproject(g3, u3, xb), reps=2)
                terms = float(x.numel()) * ws3.n_trans * nf3
                nnz = float(torch.count_nonzero(x).item())
                next3 = {"n_trans": ws3.n_trans, "n_freq": nf3, "ms_project_sparse_phantom": ms_sp, "ms_project_dense_volume": ms_spd, "ms_backproject": ms_sb,
                         "voxel_transducer_frequency_terms": terms, "nonzero_voxel_fraction_of_phantom": nnz / x.numel(),
                         "roofline_project_dense": {"bound": "alu", "unit": "fp32 lane-operations/s", "achieved": 8.0 * terms / (ms_spd * 1e-3), "peak": peak_alu,
                                                    "frac": 8.0 * terms / (ms_spd * 1e-3) / peak_alu},
                         "roofline_backproject": {"bound": "alu", "unit": "fp32 lane-operations/s", "achieved": 8.0 * terms / (ms_sb * 1e-3), "peak": peak_alu,
                                                  "frac": 8.0 * terms / (ms_sb * 1e-3) / peak_alu},
                         "algorithmic": "8 fp32 lane-operations per (voxel, transducer, frequency) term: 4 for the phasor recurrence, 4 for the complex multiply-accumulate",
                         "note": "outside the timed step; the projection skips all-zero voxels, so it is also timed on a dense N(0,1) volume"}
                g3.close()
            except Exception as ex:
                next3 = {"error": str(ex)}
        # ---- row C1 (config 4 only): the CG loop of the paper's experiments, 20 iterations (L326), timed as a whole
        cgls = None
        if args.config == 4:
            try:
                oat.oat_project(g, x, y)                      # y = H x_true (noise-free data are enough for a timing)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                _, res, _ = oat.oat_cgls(g, y, 20)
                torch.cuda.synchronize()
                dt_cg = (time.perf_counter() - t0) * 1e3
                cgls = {"iterations": 20, "ms_total": dt_cg, "ms_per_iteration": dt_cg / 20.0, "residual_first_last": [float(res[0]), float(res[-1])]}
            except Exception as ex:
                cgls = {"error": str(ex)}
        # ---- measured alternative (SURVEY 8(a) candidate V2, north_star (1)): the tile-stationary projection kernel -- bricks of the
        # volume staged in shared memory by TMA box loads -- on the same workload and input, after the timed region
        tile = None
        if not args.no_next and world == 1:
            try:
                y_ref = oat.oat_project(g, x).clone()
                oat.oat_set_variant(g, "project", 5)
                y5 = torch.empty_like(y)
                oat.oat_project(g, x, y5); torch.cuda.synchronize()
                ms5 = float(oat.oat_last_kernel_ms(g))
                oat.oat_set_variant(g, "project", 4)
                d = (y5.double() - y_ref.double()).norm() / y_ref.double().norm()
                tile = {"kernel": "oat_tile_kernel (project variant 5, not the default)", "ms_H_tile": ms5, "ms_H_default": k_h,
                        "rel_l2_vs_default": float(d.item()),
                        "note_HT": "the round-2 tile-stationary H^T (fixed-point shared-memory accumulators) missed the 1e-4 tolerance and was removed from the library; measurement: profiles/r2_tile_bwd.md",
                        "note": "16^3-cell cores + 3-cell margin per block, 3-D TMA box loads with zero fill, chunk ownership; DESIGN.md section 5.8"}
            except Exception as ex:
                tile = {"error": str(ex)}
        cpu = None
        if not args.no_cpu_baseline and world == 1:       # rank 0 at N=1 only
            try:
                from oracle import oat_oracle as orc
                threads = orc.max_threads()
                x64 = w.phantom().astype(np.float64)
                sq = oracle_sample_size(args.cpu_sample, w.n_trans, threads)
                a, b, nq = oracle_step(w, x64, sq)
                sc = w.n_trans / nq
                a1, b1, n1 = oracle_step(w, x64, 1, n_threads=1)           # the 1-thread figure of SURVEY 8(d)
                cpu = {"value": (a + b) * 1e3 * sc, "unit": "ms", "cores": min(threads, nq), "kind": "oracle",
                       "sample": f"H + H^T on {nq} of {w.n_trans} transducers (seeded subset), {a + b:.1f} s of CPU wall time scaled by {sc:.0f}x",
                       "ms_H": a * 1e3 * sc, "ms_HT": b * 1e3 * sc,
                       "one_thread": {"value": (a1 + b1) * 1e3 * w.n_trans, "unit": "ms", "cores": 1,
                                      "sample": f"H + H^T on 1 of {w.n_trans} transducers, {a1 + b1:.1f} s scaled by {w.n_trans}x"}}
            except Exception as ex:                          # the baseline must never sink the bench line
                cpu = {"value": None, "unit": "ms", "cores": None, "kind": "oracle", "sample": f"failed: {ex}"}
        metric = METRIC if (args.config == 3 and not args.subset) else f"ms per H and per H^T on {w_all.name} (value = ms per H + H^T pair)"
        line = {"metric": metric, "value": ms_step, "unit": "ms", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_step, "higher_is_better": False, "scaling": args.scaling, "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": config_object(w, args, note, world),
                "data_note": "x = seeded vessel phantom, H^T input = dense seeded N(0,1) (no band of samples is all zero, so the kernel skips nothing)",
                "ms_H": ms_h, "ms_HT": ms_t,
                "samples_per_operator": int(n_samples), "samples_per_s": 2.0 * float(tot_samples.item()) / (ms_step * 1e-3),
                "samples_per_s_H": float(tot_samples.item()) / (ms_h * 1e-3), "samples_per_s_HT": float(tot_samples.item()) / (ms_t * 1e-3),
                "gpu_launches": launches, "clocks": clocks, "e2e": e2e, "roofline": roofline, "next1": next1, "next2": next2, "next3": next3, "tile_variant": tile, "cgls": cgls, "cpu_baseline": cpu,
                "paper_context": "PAPER.md Table I: PLS-Int 20-137 min/iteration on a Tesla C2050 for 1,440-11,520 transducers on 210x210x440 voxels (another workload and machine)"}
        print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number (1-5); 3 is the metric's")
    ap.add_argument("--subset", type=int, default=0, help="debug only: use a seeded subset of transducers")
    ap.add_argument("--kband", type=int, default=0,
                    help="measurement aid: time samples sharing one angular rule (default: the config's B = 32); 1 = the paper's per-sample Eq. 37")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank a rotated copy of the array (per-GPU work fixed), strong = rows of H partitioned")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-sample", type=int, default=64, help="transducers in the oracle's timed sample (SURVEY 8(d): 64)")
    ap.add_argument("--ref-sample", type=int, default=0,
                    help="transducers per step of --impl reference; 0 = one per host thread of the oracle (all cores busy)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--project-variant", type=int, default=4, choices=[0, 4, 5],
                    help="measurement aid: 4 = default kernels, 5 = tile-stationary projection kernel, 0 = generic patch kernel")
    ap.add_argument("--backproject-variant", type=int, default=4, choices=[0, 4],
                    help="measurement aid: 4 = default kernels, 0 = generic patch kernel")
    ap.add_argument("--no-next", action="store_true", help="skip the NEXT-row legs after the timed region")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
