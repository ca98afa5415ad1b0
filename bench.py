#!/usr/bin/env python
"""bench.py -- FDAS matched-filter hot path on B200: (z,r) points/s and fraction of the roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one fdas_convolve over one batch of synthetic spectra: segment load, forward FFT,
then for every z multiply / inverse FFT / trim / power / write (DESIGN.md rows a1-a6).  The default
workload is BASELINE.json configs[2] (the config its metric is quoted on): N_f = 2^22 bins, 201
z-trials, m = 512, L = 4096.  Prints ONE JSON line (rank 0).  For N > 1 (torchrun) every rank runs
the same workload on its own seeded spectra -- the path shards by spectrum with no exchange step --
and `value` is all ranks' points over the slowest rank's device time ("scaling": "weak").

`--impl reference`: there is no reference implementation for this paper; this arm times the
double-precision oracle (oracle/, the plain statement of eq.(2)) on the host cores, on a bounded
sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fdas_conv_zr_points_per_s"
UNIT = "points/s"
FP32_LANES_PER_SM = 128  # B200: 4 SMSPs x 32 FP32 lanes, 2 flops per FMA
N_SM = 148

TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")


def ncu_traffic(workload_name, kernel_version):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the hot kernel from the committed
    `ncu --set full` capture of THIS kernel version (profiles/traffic.json: either a pointer to the tracked
    raw export of the capture, read here, or for older generations numbers transcribed from it).  None when the library's kernel version has no capture: a stale figure is
    worse than none."""
    try:
        with open(TRAFFIC_JSON) as f:
            table = json.load(f)
    except (OSError, ValueError):
        return None, None
    e = table.get(kernel_version, {}).get(workload_name)
    if not e:
        return None, None
    if "raw_csv" in e:  # the tracked raw export of the capture: header row, unit row, one row per profiled launch
        try:
            import csv
            with open(os.path.join(os.path.dirname(TRAFFIC_JSON), os.path.basename(e["raw_csv"]))) as f:
                rows = list(csv.reader(f))
            col = {name: i for i, name in enumerate(rows[0])}
            unit = rows[1]
            rd, wr = col["dram__bytes_read.sum"], col["dram__bytes_write.sum"]
            if unit[rd] != "byte" or unit[wr] != "byte":
                return None, None
            return int(float(rows[2][rd])) + int(float(rows[2][wr])), e["raw_csv"]
        except (OSError, KeyError, IndexError, ValueError):
            return None, None
    return int(e["dram_bytes_read"]) + int(e["dram_bytes_write"]), e.get("source")


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number 1..5 (4 = sweep pair --pair)")
    ap.add_argument("--pair", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-rows", type=int, default=0, help="rows of the plane the oracle is timed on (0 = auto)")
    ap.add_argument("--mode", default="convolve", choices=["convolve", "fft", "peak", "general", "spectrum"],
                    help="convolve: the FDAS hot path (BASELINE.json metric); fft: the stand-alone FFT protocol of Table 1")
    ap.add_argument("--fft-n", type=int, default=1024)
    ap.add_argument("--no-detect", action="store_true", help="skip the fused block-maximum (detection) timings")
    ap.add_argument("--dry-run", action="store_true",
                    help="no GPU: exercise the launcher, the gloo rendezvous and the cross-rank timing reduction only")
    return ap.parse_args(argv)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def algorithmic_work(wl, S, n_seg):
    """Per launch: HBM bytes and nominal FFT flops."""
    L = wl.seg_len
    out_b = 4 * wl.n_batch * wl.n_z * wl.n_f
    in_b = 8 * wl.n_batch * n_seg * L          # every segment loads L bins (overlap re-read included)
    tpl_b = 8 * wl.n_z * L                     # template bank once (L2 resident afterwards)
    fft = 5.0 * L * np.log2(L)
    flops = wl.n_batch * n_seg * (1 + wl.n_z) * fft
    return out_b + in_b + tpl_b, flops


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50", "-i", str(self.index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [l.split(", ") for (ts, l) in self.lines if t0 - 0.05 <= ts <= t1 + 0.15]
        if not rows:
            rows = [l.split(", ") for (_, l) in self.lines]
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.strip().lower() == "active":
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w": float(np.median(pw)) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(value, world, device=None):
    """MAX over ranks of a per-rank scalar (device time in ms); no data-path collective exists on this
    path, this is the timing reduction only.  Works on NCCL (GPU tensor) and gloo (CPU tensor)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(points_per_rank, world, steps, total_ms_max):
    """(z,r) points all ranks processed over the slowest rank's device time (weak scaling)."""
    return world * points_per_rank * steps / (total_ms_max * 1e-3)


def make_workload(args, rank):
    from paper_1711_10855_b200 import workload
    c = args.config
    wl = workload.make_config(c, pair=args.pair if c == 4 else 0)
    if rank:  # other ranks: same shape, own noise (weak scaling over independent spectra)
        wl.spectrum = workload.noise_spectrum(wl.n_f, workload.SEED_BASE + 1000 * c + 7919 * rank, wl.n_batch)
    return wl


def workload_string(wl):
    """config.workload: the same text from both arms (the driver compares the two lines' configs)."""
    return f"{wl.name}: N_f={wl.n_f} n_z={wl.n_z} m={wl.m} L={wl.seg_len} batch={wl.n_batch} per GPU"


def cpu_baseline_ols(wl, r0, rows):
    """The oracle's double-precision overlap-and-save on the same rows: the algorithmically fair CPU figure
    (O(L log L) per segment like the GPU path, where the direct sum is O(m) per point)."""
    import oracle
    H = wl.templates.astype(np.complex128)
    t0 = time.perf_counter()
    oracle.ols(wl.spectrum[0], H, wl.seg_len, rows=(r0, r0 + rows))
    dt = time.perf_counter() - t0
    return {"value": rows * wl.n_f / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle_ols",
            "sample": f"rows {r0}..{r0 + rows - 1} of {wl.n_z} x all {wl.n_f} columns of spectrum 0 "
                      f"(double overlap-and-save, L={wl.seg_len}, step L-m+1, in {dt:.2f} s)"}


def cpu_baseline(wl, rows=0, target_s=15.0):
    """The oracle's direct sum (eq.(2)) timed on the host cores on `rows` full rows of the plane."""
    import oracle
    H = wl.templates.astype(np.complex128)
    A = wl.spectrum[0]
    nthr = oracle.num_threads()
    mid = wl.n_z // 2
    t0 = time.perf_counter()
    oracle.direct(A, H, rows=(mid, mid + 1))
    t1 = time.perf_counter() - t0
    if rows <= 0:
        rows = int(max(1, min(wl.n_z, round(target_s / max(t1, 1e-4)))))
    r0 = max(0, min(wl.n_z - rows, mid - rows // 2))
    t0 = time.perf_counter()
    oracle.direct(A, H, rows=(r0, r0 + rows))
    dt = time.perf_counter() - t0
    pts = rows * wl.n_f
    return {"value": pts / dt, "unit": UNIT, "cores": nthr, "kind": "oracle",
            "sample": f"rows {r0}..{r0 + rows - 1} of {wl.n_z} x all {wl.n_f} columns of spectrum 0 "
                      f"(double direct sum of eq.(2), {rows * wl.n_f * wl.m:.3g} complex MACs in {dt:.2f} s)",
            "seconds": dt, "rows": [r0, rows]}, pts, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = make_workload(args, 0)
    S = wl.seg_len - wl.m
    # bounded sample per step: calibrate rows so the whole run ends within a few minutes
    base, _, _ = cpu_baseline(wl, rows=1)
    per_row = base["seconds"]
    budget = 120.0 / max(1, args.steps + args.warmup)
    rows = int(max(1, min(wl.n_z, budget / max(per_row, 1e-4))))
    for _ in range(args.warmup):
        cpu_baseline(wl, rows=rows)
    tot_pts, tot_t, last = 0, 0.0, None
    for _ in range(args.steps):
        last, pts, dt = cpu_baseline(wl, rows=rows)
        tot_pts += pts
        tot_t += dt
    value = tot_pts / tot_t
    last["value"] = value
    last.pop("rows", None)
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_string(wl), "segments": int((wl.n_f + S - 1) // S), "step_S": int(S),
                      "parallelism": "1 x independent spectra (no collective)"},
           "note": "no reference implementation exists; this is the CPU oracle (double direct sum) on a bounded sample",
           "cpu_baseline": last, "gpu_launches": 0,
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1711_10855_b200 import binding

    binding.lib()  # fail loudly if the CUDA extension is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = make_workload(args, rank)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len, n_batch=wl.n_batch)
    plan.set_templates(wl.templates)
    S, n_seg = plan.step, plan.n_seg
    bytes_alg, flops_alg = algorithmic_work(wl, S, n_seg)
    points = wl.points

    # inputs resident in HBM; rotate over enough distinct spectra to exceed the 126 MB L2
    from paper_1711_10855_b200 import workload
    spec_bytes = wl.spectrum.nbytes
    n_rot = max(1, min(8, int(np.ceil(200e6 / spec_bytes))))
    d_specs = [torch.from_numpy(wl.spectrum).cuda()]
    for i in range(1, n_rot):
        d_specs.append(torch.from_numpy(
            workload.noise_spectrum(wl.n_f, workload.SEED_BASE + 31 * i + 7919 * rank, wl.n_batch)).cuda())
    d_pow = torch.empty((wl.n_batch, wl.n_z, wl.n_f), dtype=torch.float32, device="cuda")
    stream = torch.cuda.Stream()

    with torch.cuda.stream(stream):
        for i in range(max(3, args.warmup)):
            plan.convolve(d_specs[i % n_rot], d_pow, stream=stream)
    barrier()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    t_wall0 = time.time()
    launches = 0
    ev[0].record(stream)
    for i in range(args.steps):
        plan.convolve(d_specs[i % n_rot], d_pow, stream=stream)
        launches += plan.last_launch_count
        ev[i + 1].record(stream)
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    total_ms = ev[0].elapsed_time(ev[-1])
    per_launch_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms_max = max_over_ranks(total_ms, world, "cuda")
    ms_per_step = total_ms_max / args.steps
    value = whole_job_value(points, world, args.steps, total_ms_max)

    # e2e: host buffers through the C ABI, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        h_spec = torch.from_numpy(wl.spectrum).pin_memory()
        h_pow = torch.empty((wl.n_batch, wl.n_z, wl.n_f), dtype=torch.float32).pin_memory()
        e2e_steps = max(1, min(args.steps, 5))
        plan.convolve_host(h_spec, h_pow, stream=stream)  # warm-up: allocates the plan's staging buffers
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(e2e_steps):
            plan.convolve_host(h_spec, h_pow, stream=stream)
        e1.record(stream)
        barrier()
        te = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
        e2e = {"value": whole_job_value(points, world, e2e_steps, te), "unit": UNIT,
               "h2d_bytes_per_step": int(h_spec.numel() * 8), "d2h_bytes_per_step": int(h_pow.numel() * 4),
               "steps": e2e_steps, "ms_per_step": te / e2e_steps}
        del h_pow

    # the same path fused with block-maximum detection: the plane is never written
    detect = None
    if not args.no_detect:
        shape = (wl.n_batch, wl.n_z, int(n_seg))
        d_max = torch.empty(shape, dtype=torch.float32, device="cuda")
        d_arg = torch.empty(shape, dtype=torch.int32, device="cuda")
        for i in range(3):
            plan.detect_blockmax(d_specs[i % n_rot], d_max, d_arg, stream=stream)
        barrier()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(stream)
        for i in range(args.steps):
            plan.detect_blockmax(d_specs[i % n_rot], d_max, d_arg, stream=stream)
        d1.record(stream)
        barrier()
        td = max_over_ranks(d0.elapsed_time(d1), world, "cuda")
        h_spec = torch.from_numpy(wl.spectrum).pin_memory()
        h_max = torch.empty(shape, dtype=torch.float32).pin_memory()
        h_arg = torch.empty(shape, dtype=torch.int32).pin_memory()
        det_steps = max(1, min(args.steps, 20))
        plan.detect_blockmax_host(h_spec, h_max, h_arg, stream=stream)
        barrier()
        d0.record(stream)
        for _ in range(det_steps):
            plan.detect_blockmax_host(h_spec, h_max, h_arg, stream=stream)
        d1.record(stream)
        barrier()
        te = max_over_ranks(d0.elapsed_time(d1), world, "cuda")
        # down to the candidate list (reading 20): threshold at power 30 (templates of unit norm on unit-variance noise:
        # mean power 2, so 30 is a 1e-6.5 tail per sample), capacity 4096 -> 64 KB come back instead of the 1.9 MB of maxima
        cand_cap, cand_thr = 4096, 30.0
        h_cand = torch.empty((cand_cap, 4), dtype=torch.int32).pin_memory()
        h_cnt = torch.zeros((2,), dtype=torch.int32).pin_memory()
        plan.detect_candidates_host(h_spec, cand_thr, cand_cap, h_cand, h_cnt, stream=stream)
        barrier()
        d0.record(stream)
        for _ in range(det_steps):
            plan.detect_candidates_host(h_spec, cand_thr, cand_cap, h_cand, h_cnt, stream=stream)
        d1.record(stream)
        barrier()
        tc = max_over_ranks(d0.elapsed_time(d1), world, "cuda")
        cand = {"what": "fdas_detect_candidates_host: block maxima >= threshold as an ordered (item, row, column, power) list",
                "threshold": cand_thr, "capacity": cand_cap, "found": int(h_cnt[0]), "written": int(h_cnt[1]),
                "e2e": {"value": whole_job_value(points, world, det_steps, tc), "unit": UNIT, "ms_per_step": tc / det_steps,
                        "h2d_bytes_per_step": int(h_spec.numel() * 8), "d2h_bytes_per_step": 16 * cand_cap + 8, "steps": det_steps}}
        det_bytes = 8 * wl.n_batch * int(n_seg) * wl.seg_len + 8 * wl.n_z * wl.seg_len + 8 * wl.n_batch * wl.n_z * int(n_seg)
        detect = {"what": "fdas_detect_blockmax: same (z,r) points, per (row, segment) max + argmax instead of the plane",
                  "value": whole_job_value(points, world, args.steps, td), "unit": UNIT, "ms_per_step": td / args.steps,
                  "bytes_per_launch": det_bytes, "alu_frac": None,
                  "e2e": {"value": whole_job_value(points, world, det_steps, te), "unit": UNIT, "ms_per_step": te / det_steps,
                          "h2d_bytes_per_step": int(h_spec.numel() * 8), "d2h_bytes_per_step": int(h_max.numel() * 8),
                          "steps": det_steps},
                  "candidates": cand}

    if rank == 0:
        pk = peaks()
        kern_ms = float(np.mean(per_launch_ms))
        fp32_peak = N_SM * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12  # TFLOP/s at max clock
        ach_tf = flops_alg / (kern_ms * 1e-3) / 1e12
        ach_gb = bytes_alg / (kern_ms * 1e-3) / 1e9
        t_alu = flops_alg / (fp32_peak * 1e12)
        t_hbm = bytes_alg / (pk["hbm_gbs"] * 1e9)
        alu_binds = t_alu >= t_hbm
        traffic = ncu_traffic(wl.name, binding.version())
        roofline = {
            "bound": "alu" if alu_binds else "hbm",
            "achieved": ach_tf if alu_binds else ach_gb,
            "peak": fp32_peak if alu_binds else pk["hbm_gbs"],
            "unit": "TFLOP/s" if alu_binds else "GB/s",
            "frac": (ach_tf / fp32_peak) if alu_binds else (ach_gb / pk["hbm_gbs"]),
            "traffic": traffic[0], "traffic_source": traffic[1],
            "kernel": f"fdas::fdas_convolve_kernel<{wl.seg_len}, OUT_POWER, false>", "kernel_ms": kern_ms, "kernel_ms_median": float(np.median(per_launch_ms)), "kernel_ms_min": float(np.min(per_launch_ms)),
            "flops_per_launch": flops_alg, "bytes_per_launch": bytes_alg,
            "alu": {"achieved": ach_tf, "peak": fp32_peak, "unit": "TFLOP/s", "frac": ach_tf / fp32_peak,
                    "peak_def": f"{N_SM} SMs x {FP32_LANES_PER_SM} lanes x 2 x {pk['sm_max_mhz']:.0f} MHz (nominal; flops = 5 L log2 L per transform)"},
            "hbm": {"achieved": ach_gb, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": ach_gb / pk["hbm_gbs"],
                    "peak_def": f"MEASURED_PEAKS.json hbm_gbs ({pk['source']})"},
        }
        if clocks and clocks.get("sm_mhz"):
            at_clock = N_SM * FP32_LANES_PER_SM * 2 * clocks["sm_mhz"] * 1e6 / 1e12
            roofline["alu"]["frac_at_measured_clock"] = ach_tf / at_clock
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
               "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f32", "data": "synthetic",
               "config": {"workload": workload_string(wl),
                          "segments": int(n_seg), "step_S": int(S),
                          "l2": f"output plane {d_pow.numel() * 4 / 1e9:.2f} GB >> 126 MB L2; inputs rotate over {n_rot} spectra "
                                f"({n_rot * spec_bytes / 1e6:.0f} MB) so no flush is needed",
                          "parallelism": f"{world} x independent spectra (no collective)"},
               "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline}
        if detect:
            detect["alu_frac"] = flops_alg / (detect["ms_per_step"] * 1e-3) / 1e12 / fp32_peak
            out["detect"] = detect
        out["config"]["grid"] = plan.grid
        out["kernel_version"] = binding.version()
        if not args.no_cpu_baseline and world == 1:  # rank 0 at N = 1 only
            cb, _, _ = cpu_baseline(wl, rows=args.cpu_rows)
            cb.pop("seconds", None)
            r0, rows = cb.pop("rows")
            out["cpu_baseline"] = cb
            out["cpu_baseline_ols"] = cpu_baseline_ols(wl, r0, rows)
        print(json.dumps(out))
    plan.destroy()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_fft(args):
    """--mode fft: the stand-alone FFT protocol of the paper (Table 1): N = 1024, "100 FFTs per kernel
    launch, while launching 1000 of these kernels", for each elements-per-thread variant; plus the same 100 000
    transforms in ONE launch, which is what the HBM roofline (8 bytes in + 8 bytes out per point) applies to.
    Context from the paper (other hardware, not a target): 1.80 ms on a P100 for its best variant."""
    import torch
    from paper_1711_10855_b200 import binding
    binding.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    n = args.fft_n
    n_total, per_launch = 100000, 100
    variants = [e for e in (8, 16) if (e == 8 and n <= 1024) or (e == 16 and n >= 1024)]
    rng = torch.Generator(device="cuda").manual_seed(171110855)
    x = torch.randn((n_total, n, 2), device="cuda", generator=rng)          # 0.8 GB at n = 1024: > L2
    y = torch.empty_like(x)
    stream = torch.cuda.Stream()
    pk = peaks()
    rows, launches = [], 0
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.25)
    t0 = time.time()
    for e in variants:
        plan = binding.FftPlan(n, e)
        for _ in range(max(3, args.warmup)):
            plan.exec(n_total, x, y, stream=stream)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            plan.exec(n_total, x, y, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        one_ms = e0.elapsed_time(e1) / args.steps
        launches += args.steps
        plan.exec_many(1000, per_launch, x, y, stream=stream)                  # warm-up of the protocol
        torch.cuda.synchronize()
        e0.record(stream)
        reps = max(1, min(args.steps, 5))
        for _ in range(reps):
            plan.exec_many(n_total // per_launch, per_launch, x, y, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        proto_ms = e0.elapsed_time(e1) / reps
        launches += reps * (n_total // per_launch)
        gbs = n_total * n * 16 / (one_ms * 1e-3) / 1e9
        rows.append({"elems_per_thread": e, "grid": plan.grid, "one_launch_ms": one_ms, "protocol_1000x100_ms": proto_ms,
                     "points_per_s": n_total * n / (one_ms * 1e-3), "hbm_gbs": gbs, "hbm_frac": gbs / pk["hbm_gbs"]})
        plan.destroy()
    clocks = sampler.stop(t0, time.time())
    best = min(rows, key=lambda r: r["one_launch_ms"])
    out = {"metric": "standalone_fft_points_per_s", "value": best["points_per_s"], "unit": "points/s", "n_gpus": 1,
           "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": best["one_launch_ms"], "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"100000 complex64 FFTs of N={n} (P:46 / Table 1), natural order in and out",
                      "l2": f"input and output {n_total * n * 8 / 1e9:.2f} GB each >> 126 MB L2"},
           "variants": rows, "clocks": clocks, "gpu_launches": launches,
           "paper_context": "Table 1 (P:56-60): 1.80 ms on P100, 2.21 ms on TITAN X (Pascal) for 100 000 FFTs, N = 1024; other hardware, not a target",
           "protocol_note": "protocol_1000x100_ms: fdas_fft_exec_many = 1000 launches of 100 transforms each over 100 000 distinct sequences, recorded once as a four-chain CUDA graph and launched per repetition",
           "roofline": {"bound": "hbm", "achieved": best["hbm_gbs"], "peak": pk["hbm_gbs"], "unit": "GB/s",
                        "frac": best["hbm_frac"], "traffic": ncu_traffic(f"fft{n}e{best['elems_per_thread']}", binding.version())[0],
                        "kernel": "fdas::fdas_fft_batch_kernel",
                        "bytes_per_launch": n_total * n * 16}}
    print(json.dumps(out))
    return 0


def run_general(args):
    """--mode general: the shape of the paper's Table 2 on the complex-output convolution
    (fdas_convolve_complex): filter lengths 64, 128, 256, 384, 512 on segments of 2048 points, the largest the paper's
    FFT supports.  The table's entries are speed-ups over the authors' cuFFT-based and older codes on
    P100 / TITAN X, none of which exists here: times and throughputs only."""
    import torch
    from paper_1711_10855_b200 import binding, workload
    binding.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    n_f, z_max, z_step, L = 1 << 21, 84, 2, 2048           # the C4 sweep's spectrum and template grid
    spec = [torch.from_numpy(workload.noise_spectrum(n_f, workload.SEED_BASE + 4000 + i, 1)).cuda() for i in range(8)]
    n_z = 2 * z_max // z_step + 1
    d_amp = torch.empty((1, n_z, n_f), dtype=torch.complex64, device="cuda")      # 1.43 GB >> L2
    stream = torch.cuda.Stream()
    pk = peaks()
    fp32_peak = N_SM * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    rows, launches = [], 0
    for m in (64, 128, 256, 384, 512):
        plan = binding.Plan(n_f, z_max, z_step, m, L)
        plan.set_templates(workload.templates(z_max, z_step, m).astype(np.complex64))
        for i in range(max(3, args.warmup)):
            plan.convolve_complex(spec[i % 8], d_amp, stream=stream)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(args.steps):
            plan.convolve_complex(spec[i % 8], d_amp, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        launches += args.steps
        n_seg = plan.n_seg
        flops = n_seg * (1 + n_z) * 5.0 * L * np.log2(L)
        byt = 8 * n_z * n_f + 8 * n_seg * L + 8 * n_z * L
        rows.append({"filter_length": m, "segments": int(n_seg), "ms": ms, "points_per_s": n_z * n_f / (ms * 1e-3),
                     "alu_frac": flops / (ms * 1e-3) / 1e12 / fp32_peak, "hbm_frac": byt / (ms * 1e-3) / 1e9 / pk["hbm_gbs"]})
        plan.destroy()
    print(json.dumps({"metric": "general_convolution_points_per_s", "value": rows[-1]["points_per_s"], "unit": "points/s",
                      "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "higher_is_better": True,
                      "dtype": "f32", "data": "synthetic", "gpu_launches": launches,
                      "config": {"workload": f"complex64 output, N_f={n_f}, {n_z} filters, L={L}, filter lengths 64..512 (Table 2, P:62-70)"},
                      "rows": rows,
                      "paper_context": "Table 2 lists speed-ups over cuFFT-based convolution (2.45-3.89 on P100): comparison codes absent, not reproducible"}))
    return 0


def run_spectrum(args):
    """--mode spectrum: the step before the correlation (fdas_spectrum_exec, reading 18) on the 2^23-sample
    series behind BASELINE.json config 3: real series -> 2^22 whitened bins.  HBM-bound by construction: the algorithmic
    traffic is 4 bytes per sample in and 8 bytes per bin out; every extra pass over the data shows in the fraction."""
    import torch
    from paper_1711_10855_b200 import binding
    binding.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    n_t, blk = 1 << 23, 4096
    g = torch.Generator(device="cuda").manual_seed(171110855)
    n_rot = 8                                                     # 8 x 33.5 MB of input > L2
    xs = [torch.randn(n_t, device="cuda", generator=g) for _ in range(n_rot)]
    out = torch.empty(n_t // 2, dtype=torch.complex64, device="cuda")
    plan = binding.SpectrumPlan(n_t, blk)
    stream = torch.cuda.Stream()
    pk = peaks()
    for i in range(max(3, args.warmup)):
        plan.exec(xs[i % n_rot], out, stream=stream)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.25)
    t0 = time.time()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    for i in range(args.steps):
        plan.exec(xs[i % n_rot], out, stream=stream)
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop(t0, time.time())
    per = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    ms = ev[0].elapsed_time(ev[-1]) / args.steps
    byt = 4 * n_t + 8 * (n_t // 2)
    gbs = byt / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "spectrum_bins_per_s", "value": (n_t // 2) / (ms * 1e-3), "unit": "bins/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms, "ms_median": float(np.median(per)),
                      "ms_min": float(np.min(per)), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f32", "data": "synthetic", "gpu_launches": 6 * args.steps,
                      "config": {"workload": f"real series of {n_t} float32 samples -> {n_t // 2} whitened complex64 bins (whiten_block {blk})",
                                 "l2": f"inputs rotate over {n_rot} series ({n_rot * 4 * n_t / 1e6:.0f} MB) > 126 MB L2"},
                      "clocks": clocks,
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": gbs / pk["hbm_gbs"],
                                   "traffic": None, "bytes_per_launch": byt,
                                   "note": "bytes_per_launch is per fdas_spectrum_exec (six kernel launches): samples in + bins out"},
                      "kernel_version": binding.version()}))
    plan.destroy()
    return 0


def run_peak(args):
    """--mode peak: the FP32 FMA rate of this GPU on register-only chains (fdas_debug_alu_peak) next to the nominal
    figure the "alu" roofline uses, with the clocks seen meanwhile."""
    import torch
    from paper_1711_10855_b200 import binding
    binding.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    pk = peaks()
    nominal = N_SM * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.25)
    t0 = time.time()
    rows = []
    for _ in range(max(1, min(args.steps, 10))):
        for packed in (False, True):
            tf, ms = binding.debug_alu_peak(packed)
            rows.append({"form": "FFMA2 (packed)" if packed else "FFMA (scalar)", "tflops": tf, "ms": ms,
                         "frac_of_nominal": tf / nominal, "lanes_per_clk_per_sm": tf * 1e12 / 2 / N_SM / (pk["sm_max_mhz"] * 1e6)})
    clocks = sampler.stop(t0, time.time())
    best = max(r["tflops"] for r in rows)
    print(json.dumps({"metric": "fp32_fma_peak_tflops", "value": best, "unit": "TFLOP/s", "n_gpus": 1, "nominal_tflops": nominal,
                      "nominal_def": f"{N_SM} SMs x {FP32_LANES_PER_SM} lanes x 2 x {pk['sm_max_mhz']:.0f} MHz",
                      "best_scalar": max(r["tflops"] for r in rows if "scalar" in r["form"]),
                      "best_packed": max(r["tflops"] for r in rows if "packed" in r["form"]),
                      "runs": rows, "clocks": clocks, "higher_is_better": True, "data": "synthetic"}))
    return 0


def run_dry(args):
    """--dry-run: everything of the N-rank path that needs no GPU (gloo): rendezvous, per-rank seeded
    workload shape, MAX-over-ranks of a per-rank time, whole-job value.  Prints the JSON line with
    "dry_run": true; its `value` is meaningless."""
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    from paper_1711_10855_b200 import workload
    shape = workload.config_shape(args.config, pair=args.pair if args.config == 4 else 0)
    points = shape["n_batch"] * shape["n_z"] * shape["n_f"]
    t_ms = max_over_ranks(1.0 + rank, world)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": whole_job_value(points, world, args.steps, t_ms * args.steps),
                          "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "dry_run": True,
                          "ms_per_step": t_ms, "higher_is_better": True, "scaling": "weak", "data": "synthetic",
                          "config": {"workload": shape["name"], "parallelism": f"{world} x independent spectra (no collective)"}}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves, one per GPU, exactly as
    the driver does (torch.distributed.run, one node, rendezvous on 127.0.0.1)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "VERSION")  # one line per job: the NCCL version, visible in stderr
    return subprocess.call(cmd, env=env)


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return relaunch_under_torchrun(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.dry_run:
        return run_dry(args)
    if args.mode == "fft":
        return run_fft(args)
    if args.mode == "peak":
        return run_peak(args)
    if args.mode == "general":
        return run_general(args)
    if args.mode == "spectrum":
        return run_spectrum(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
