#!/usr/bin/env python
"""bench.py -- one H and one H^T (the whole hot path) per step on the
configuration BASELINE.json's metric is quoted on: config 3, 240^3 voxels x 9,216 transducers x
2,048 time samples (arc-array geometry), synthetic seeded phantom.

    python bench.py --gpus N --steps K --warmup W            (our arm, CUDA)
    python bench.py --impl reference --steps K --warmup W    (the fp64 oracle on host cores)

Prints ONE JSON line (see DESIGN.md §7 for every field).  Timing: CUDA events on the launching
stream, barrier + synchronize on both sides, max over ranks; L2 is flushed between steps.
"""
from __future__ import annotations

import argparse
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
# Algorithmic fp32 work per interpolation sample: position 3 FMA, 3 floor, 3 frac,
# 7 lerps (sub + FMA) or 8 weight products + 8 accumulates, 1 quadrature FMA  ->  36 flop (FMA = 2).
FLOP_PER_SAMPLE = 36.0
# Vector reductions per interpolation sample of the face-carrying H^T: ncu counts 1.562e10
# predicated-on RED.128 lanes for 2.478e10 in-box samples on the config-3 subset profiled in profiles/.
RED_PER_SAMPLE = 0.63
# 32-byte cell records requested from L2 per interpolation sample of the marching H: ncu counts
# 1.079e10 global-load sectors (L1 hit rate 5 %) for 2.478e10 in-box samples on the same subset.
SECTORS_PER_SAMPLE = 0.435
# B200 fp32 peak derived from unit counts and clocks (guide: 148 SMs x 128 fp32 lanes x 2 flop x max SM clock)
N_SM, FP32_LANES = 148, 128
# DRAM bytes (read + write) per in-box sample of the dominant kernel (H^T) from the ncu --set full capture summarised in
# profiles/r1k_final.md: (1.825 + 1.335) GB for 2.478e10 samples on the 512-transducer subset of config 3.
DRAM_BYTES_PER_SAMPLE_HT = (1.824808e9 + 1.335234e9) / 2.4784424365e10


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    sm_mhz, src = 1965.0, "fallback clocks.max.sm of B200_PROFILING.md"
    if os.path.exists(path):
        try:
            mp = json.load(open(path))
            sm_mhz = float(mp.get("sm_max_mhz", sm_mhz))
            src = "MEASURED_PEAKS.json sm_max_mhz"
        except Exception:
            pass
    return N_SM * FP32_LANES * 2.0 * sm_mhz * 1e6 / 1e12, src      # TFLOP/s


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
    return w, note


def oracle_step(w, x64, sample_q):
    """One H + one H^T of the oracle on `sample_q` seeded transducers; returns (s_H, s_HT)."""
    from oracle import oat_oracle as orc
    _, ws = w.seeded_subset(sample_q)
    t0 = time.perf_counter()
    y = orc.project(ws, x64)
    t1 = time.perf_counter()
    orc.backproject(ws, y)
    t2 = time.perf_counter()
    return t1 - t0, t2 - t1, ws.n_trans


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oat_oracle as orc
    w, note = workload(args)
    x64 = w.phantom().astype(np.float64)
    sq = max(1, min(args.ref_sample, w.n_trans))
    for _ in range(args.warmup):
        oracle_step(w, x64, 1)
    th = tt = 0.0
    for _ in range(args.steps):
        a, b, nq = oracle_step(w, x64, sq)
        th += a; tt += b
    scale = w.n_trans / sq
    ms_h, ms_t = th / args.steps * 1e3 * scale, tt / args.steps * 1e3 * scale
    cores = orc.max_threads()
    sample = f"{sq} of {w.n_trans} transducers per step (seeded subset), times scaled by {scale:.0f}x"
    line = {"impl": "reference", "metric": METRIC, "value": ms_h + ms_t, "unit": "ms", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_h + ms_t, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "n_trans": w.n_trans, "nt": w.nt, "note": note},
            "ms_H": ms_h, "ms_HT": ms_t,
            "cpu_baseline": {"value": ms_h + ms_t, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": ms_h + ms_t, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1304_2017_b200 import binding as oat, build, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()

    w, note = workload(args)
    if world > 1:                                           # weak scaling: N-times denser view sampling
        from dataclasses import replace
        w = replace(w, trans_xyz=shard.weak_replica_transducers(w.trans_xyz, rank, world, 144))
    g = oat.oat_geometry_create(w, local)
    if args.project_variant >= 0:
        oat.oat_set_variant(g, "project", args.project_variant)
    if args.backproject_variant >= 0:
        oat.oat_set_variant(g, "backproject", args.backproject_variant)
    x = torch.from_numpy(w.phantom()).cuda()
    y = torch.empty((w.n_trans, w.nt), dtype=torch.float32, device="cuda")
    xb = torch.empty_like(x)
    n_samples = oat.oat_num_surface_samples(g)              # per operator, this rank
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step(rec=None):
        flush.fill_(1)                                      # L2 flush between timed iterations
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)] if rec is not None else None
        if e: e[0].record(stream)
        oat.oat_project(g, x, y)
        kh = oat.oat_last_kernel_ms(g) if rec is not None else 0.0
        nl = oat.oat_last_launch_count(g)
        if e: e[1].record(stream)
        oat.oat_backproject(g, y, xb)
        kt = oat.oat_last_kernel_ms(g) if rec is not None else 0.0
        nl += oat.oat_last_launch_count(g)
        if world > 1:
            shard.allreduce_volume(xb)                      # the path's one exchange step (H^T only)
        if e:
            e[2].record(stream)
            rec.append((e, kh, kt, nl))

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
    k_h = float(np.mean([r[1] for r in rec])); k_t = float(np.mean([r[2] for r in rec]))
    launches = int(sum(r[3] for r in rec)) + args.steps      # + the L2-flush fill per step
    vals = torch.tensor([total_ms, ms_h, ms_t], dtype=torch.float64, device="cuda")
    tot_samples = torch.tensor([float(n_samples)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot_samples, op=dist.ReduceOp.SUM)
    total_ms, ms_h, ms_t = [float(v) for v in vals.tolist()]
    ms_step = total_ms / args.steps

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region)
    e2e = None
    if args.e2e_steps > 0:
        hx = torch.from_numpy(w.phantom()).pin_memory()
        hy = torch.empty((w.n_trans, w.nt), dtype=torch.float32).pin_memory()
        hxb = torch.empty_like(hx).pin_memory()
        n_e2e = max(1, min(args.steps, args.e2e_steps))
        oat.oat_project_host(g, hx, hy); oat.oat_backproject_host(g, hy, hxb)     # warm-up
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            oat.oat_project_host(g, hx, hy)
            oat.oat_backproject_host(g, hy, hxb)
        dt_e2e = (time.perf_counter() - t0) / n_e2e * 1e3
        v = torch.tensor([dt_e2e], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(v, op=dist.ReduceOp.MAX)
        bx, by = x.numel() * 4, y.numel() * 4
        e2e = {"value": float(v.item()), "unit": "ms", "h2d_bytes_per_step": bx + by, "d2h_bytes_per_step": by + bx,
               "steps": n_e2e, "api": "oat_project_host + oat_backproject_host (pinned host buffers)"}

    if rank == 0:
        peak, peak_src = peaks()
        dom = "backproject" if k_t >= k_h else "project"
        k_ms = max(k_t, k_h)
        achieved = n_samples * FLOP_PER_SAMPLE / (k_ms * 1e-3) / 1e12 if k_ms > 0 else 0.0
        roofline = {"bound": "alu", "kernel": f"oat_march_kernel<{1 if dom == 'backproject' else 0}> ({dom})",
                    "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak if peak else None,
                    "traffic": (DRAM_BYTES_PER_SAMPLE_HT * n_samples) if dom == "backproject" else None,
                    "traffic_note": "dram__bytes_read+write of oat_march_kernel<1> per launch, ncu --set full on the 512-transducer subset "
                                    "(profiles/r1k_final.md) scaled by samples; unit B; algorithmic unique bytes = size(x)+size(y)",
                    "kernel_ms": k_ms, "kernel_share_of_step": k_ms / ms_step if ms_step else None,
                    "peak_source": f"148 SM x 128 fp32 lanes x 2 flop x {peak_src}",
                    "algorithmic": f"{FLOP_PER_SAMPLE:.0f} fp32 flop per interpolation sample x {n_samples:.4g} samples per launch",
                    "other_kernel": {"kernel_ms": min(k_t, k_h),
                                     "frac": (n_samples * FLOP_PER_SAMPLE / (min(k_t, k_h) * 1e-3) / 1e12 / peak) if min(k_t, k_h) > 0 else None}}
        # What ncu and the micro-benchmarks name as the binding unit of each kernel: H^T retires
        # vector reductions (RED.128) at the rate the L2 atomic path sustains; the peak is measured live.
        try:
            red_scat = oat.oat_measure_red_rate(local)                 # every lane its own 32-byte sector
            red_pack = oat.oat_measure_red_rate_ex(local, 1)           # 32 lanes fill 16 sectors: the best case
            red_lanes = RED_PER_SAMPLE * n_samples
            ach = red_lanes / (k_t * 1e-3) if k_t > 0 else None
            roofline["limiter"] = {"kernel": "oat_march_kernel<1> (backproject)", "unit": "L2 vector reductions (RED.128 lanes/s)",
                                   "achieved": ach, "peak": red_pack, "frac": (ach / red_pack) if (ach and red_pack > 0) else None,
                                   "scattered_rate": red_scat, "frac_of_scattered_rate": (ach / red_scat) if (ach and red_scat > 0) else None,
                                   "algorithmic": f"{RED_PER_SAMPLE} reductions per sample (cell crossings of the marched rays, ncu inst count) x {n_samples:.4g} samples",
                                   "peak_source": "oat_measure_red_rate_ex(pattern 1): red.global.add.v4.f32, the 32 lanes of a warp filling 16 sectors of an L2-resident "
                                                  "64 MB buffer (the cost of a reduction is per distinct sector); scattered_rate = oat_measure_red_rate(): every lane its own sector; same run"}
        except Exception as ex:
            roofline["limiter"] = {"error": str(ex)}
        # H requests one 32-byte cell record from L2 per cell run of a ray; the peak is the measured scattered-sector rate
        try:
            gat_peak = oat.oat_measure_gather_rate(local)
            sec = SECTORS_PER_SAMPLE * n_samples
            roofline["limiter_H"] = {"kernel": "oat_march_kernel<0> (project)", "unit": "L1-miss sector loads from L2 (32 B sectors/s)",
                                     "achieved": sec / (k_h * 1e-3) if k_h > 0 else None, "peak": gat_peak,
                                     "frac": (sec / (k_h * 1e-3) / gat_peak) if (k_h > 0 and gat_peak > 0) else None,
                                     "algorithmic": f"{SECTORS_PER_SAMPLE} cell records per sample (one per cell run of a marched ray, ncu sector count) x {n_samples:.4g} samples",
                                     "peak_source": "oat_measure_gather_rate(): scattered ld.global.nc.v8.f32, one sector per lane, L2-resident 64 MB buffer, same run"}
        except Exception as ex:
            roofline["limiter_H"] = {"error": str(ex)}
        # ---- row NEXT-1 (EIR convolution, penalty stencil): the steps either side of the path, timed at this config's sizes
        next1 = None
        try:
            hbm = None
            try:
                hbm = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs"))
            except Exception:
                pass
            taps = 128
            tt = np.arange(taps) * w.dt
            oat.oat_eir_set(g, (w.dt * np.exp(-tt / (0.15 * taps * w.dt)) * np.sin(2 * np.pi * 2.5 * tt)).astype(np.float32))
            u = torch.empty_like(y); lx = torch.empty_like(x)

            def timed(fn, reps=5):
                fn(); torch.cuda.synchronize()
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for _ in range(reps):
                    fn()
                b.record(stream); torch.cuda.synchronize()
                return a.elapsed_time(b) / reps
            ms_e = timed(lambda: oat.oat_eir_apply(g, y, u))
            ms_ea = timed(lambda: oat.oat_eir_apply(g, y, u, adjoint=True))
            ms_p = timed(lambda: oat.oat_penalty_apply(g, xb, lx))
            by, bx = 2.0 * y.numel() * 4, 2.0 * x.numel() * 4          # read + write once
            next1 = {"eir_taps": taps, "ms_eir": ms_e, "ms_eir_adjoint": ms_ea, "ms_penalty": ms_p,
                     "eir_GBps": by / (ms_e * 1e-3) / 1e9, "penalty_GBps": bx / (ms_p * 1e-3) / 1e9,
                     "hbm_peak_GBps": hbm, "penalty_frac_of_hbm": (bx / (ms_p * 1e-3) / 1e9 / hbm) if hbm else None,
                     "eir_frac_of_hbm": (by / (ms_e * 1e-3) / 1e9 / hbm) if hbm else None,
                     "share_of_pls_iteration": (ms_e + ms_ea + ms_p) / (ms_step + ms_e + ms_ea + ms_p),
                     "note": "outside the timed step; algorithmic bytes = read + write of the vector once; the EIR is a 128-tap FIR from shared memory (LDS-bound, not HBM-bound)"}
            oat.oat_eir_set(g, np.zeros(0, dtype=np.float32))
        except Exception as ex:
            next1 = {"error": str(ex)}
        # ---- row NEXT-2 (FBP, Eq. 27): one image from the data of this config, voxel driven
        next2 = None
        try:
            from paper_1304_2017_b200 import workloads as wl2
            wb2, _ = workload(args)
            areas = wl2.patch_areas_arc(64, 144, 65.0) if (args.config == 3 and not args.subset) else wl2.patch_areas_equal(wb2.trans_xyz, wb2.centre)
            wq = torch.from_numpy(oat.oat_fbp_weights(g, areas)).cuda()
            oat.oat_fbp(g, y, wq, xb); torch.cuda.synchronize()
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record(stream); oat.oat_fbp(g, y, wq, xb); b.record(stream); torch.cuda.synchronize()
            ms_f = a.elapsed_time(b)
            pairs = float(x.numel()) * w.n_trans
            next2 = {"ms_fbp": ms_f, "voxel_transducer_pairs": pairs, "pairs_per_s": pairs / (ms_f * 1e-3),
                     "note": "outside the timed step; fp64 distance + interval decision, fp32 brackets and sum (DESIGN.md section 5.6)"}
        except Exception as ex:
            next2 = {"error": str(ex)}
        # ---- row NEXT-3 (spherical-voxel model, frequency domain): this config's grid, 256 seeded transducers, 64 frequencies
        next3 = None
        try:
            wb3, _ = workload(args)
            _, ws3 = wb3.seeded_subset(256)
            g3 = oat.oat_geometry_create(ws3, local)
            nf3 = 64
            oat.oat_sph_set(g3, nf3, 0.0, 0.078125)          # 0 .. 4.9 MHz
            u3 = torch.empty((ws3.n_trans, nf3), dtype=torch.complex64, device="cuda")
            oat.oat_sph_project(g3, x, u3); oat.oat_sph_backproject(g3, u3, xb); torch.cuda.synchronize()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            ev[0].record(stream); oat.oat_sph_project(g3, x, u3); ev[1].record(stream); oat.oat_sph_backproject(g3, u3, xb); ev[2].record(stream)
            torch.cuda.synchronize()
            terms = float(x.numel()) * ws3.n_trans * nf3
            nnz = float(torch.count_nonzero(x).item())
            next3 = {"n_trans": ws3.n_trans, "n_freq": nf3, "ms_project": ev[0].elapsed_time(ev[1]), "ms_backproject": ev[1].elapsed_time(ev[2]),
                     "voxel_transducer_frequency_terms": terms, "terms_per_s_backproject": terms / (ev[1].elapsed_time(ev[2]) * 1e-3),
                     "nonzero_voxel_fraction": nnz / x.numel(),
                     "note": "outside the timed step; the projection skips all-zero voxels (sparse vessel phantom), the backprojection visits every term"}
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
        cpu = None
        if not args.no_cpu_baseline and world == 1:       # rank 0 at N=1 only
            try:
                from oracle import oat_oracle as orc
                from paper_1304_2017_b200 import workloads as wl
                wb, _ = workload(args)
                sq = max(1, min(args.cpu_sample, wb.n_trans))
                a, b, nq = oracle_step(wb, wb.phantom().astype(np.float64), sq)
                sc = wb.n_trans / nq
                cpu = {"value": (a + b) * 1e3 * sc, "unit": "ms", "cores": orc.max_threads(), "kind": "oracle",
                       "sample": f"H + H^T on {nq} of {wb.n_trans} transducers (seeded subset), {a + b:.1f} s of CPU wall time scaled by {sc:.0f}x",
                       "ms_H": a * 1e3 * sc, "ms_HT": b * 1e3 * sc}
            except Exception as ex:                          # the baseline must never sink the bench line
                cpu = {"value": None, "unit": "ms", "cores": None, "kind": "oracle", "sample": f"failed: {ex}"}
        metric = METRIC if (args.config == 3 and not args.subset) else f"ms per H and per H^T on {w.name} (value = ms per H + H^T pair)"
        line = {"metric": metric, "value": ms_step, "unit": "ms", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"{w.name}: {w.nx}x{w.ny}x{w.nz} voxels @ {w.spacing} mm, {w.n_trans} transducers/GPU, nt={w.nt}, h={w.surf_step}, B={w.kband}",
                           "step": "one H (x -> y) followed by one H^T (y -> x), inputs resident in HBM",
                           "l2": "flushed between steps (256 MB fill)", "note": note,
                           "parallelism": "1 GPU" if world == 1 else f"{world} GPUs, transducers sharded (weak: {world}x denser views), H^T partial volumes all-reduced over NCCL"},
                "ms_H": ms_h, "ms_HT": ms_t,
                "samples_per_operator": int(n_samples), "samples_per_s": 2.0 * float(tot_samples.item()) / (ms_step * 1e-3),
                "samples_per_s_H": float(tot_samples.item()) / (ms_h * 1e-3), "samples_per_s_HT": float(tot_samples.item()) / (ms_t * 1e-3),
                "gpu_launches": launches, "clocks": clocks, "e2e": e2e, "roofline": roofline, "next1": next1, "next2": next2, "next3": next3, "cgls": cgls, "cpu_baseline": cpu,
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
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sample", type=int, default=8, help="transducers in the oracle's timed sample")
    ap.add_argument("--ref-sample", type=int, default=8, help="transducers per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--project-variant", type=int, default=-1, help="kernel variant (DESIGN.md §5); -1 = library default")
    ap.add_argument("--backproject-variant", type=int, default=-1)
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
