#!/usr/bin/env python
"""bench.py -- whole-hot-path throughput of the split-step phase-screen library on B200.

One "step" = one frame of the temporal workload (BASELINE.json configs[2], 1024^2): evolve every
screen by one AR step (K1-K3), propagate the field batch through the stack (K4-K6), reduce the
beam statistics (K8) and run the adjoint propagation (K7).  Metric: split-step screen-steps/s,
counting forward and adjoint screen-steps; the AR evolution and the statistics are overhead
inside the timed region.  See DESIGN.md section 7.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--batch B]
Under torchrun each rank runs its own batch on its own GPU (weak scaling, no data-path collective).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "split-step screen-steps/sec (complex64 N^2 field)"
UNIT = "screen-steps/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config id (1-5)")
    ap.add_argument("--batch", type=int, default=0, help="override realisations per GPU")
    ap.add_argument("--h-kind", default="fresnel", choices=["fresnel", "angular"],
                    help="transfer function: north_star's Fresnel form (default) or the paper's angular spectrum")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cufft-compare", action="store_true")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel_class, N):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full`
    capture (profiles/ncu_traffic.csv: class,N,bytes,source), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as fh:
            for line in fh:
                p = [x.strip() for x in line.split(",")]
                if len(p) >= 3 and p[0] == kernel_class and p[1] == str(N):
                    return float(p[2])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms; started before the warm-up so that the
    tool is already running when the timed region starts, samples outside [t0, t1] are dropped."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self, t0=None, t1=None):
        import datetime
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
        sm, reasons, mx = [], set(), None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(parts[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
            except ValueError:
                continue
            parts = parts[1:]
            if t0 is not None and not (t0 - 0.05 <= ts <= t1 + 0.05):
                continue
            try:
                sm.append(float(parts[0]))
                mx = float(parts[1])
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=mx, reasons=sorted(reasons), samples=len(sm))
        return out


# ---------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): oracle/ as it stands, on the host cores
# ---------------------------------------------------------------------------------------------
def oracle_frame(wl, S_s, seed=0, reps=1):
    """Time `reps` frames of the same path on ONE realisation and S_s screens with the CPU oracle.
    Returns (seconds per frame, screen-steps per frame)."""
    import numpy as np
    from oracle import orc
    from paper_2604_07248_b200 import synth
    N = wl.N
    psd = orc.Psd(**wl.psd_dict())
    cn2, dz = wl.cn2_list[:S_s], wl.dz[:S_s]
    frames = synth.noise(wl.cid, seed, 0, S_s, N, wl.n_sh, frames=reps + 1)
    hi0, sh0 = frames[0]
    _, spec, shc = orc.make_screens(N, wl.dx, psd, wl.lam, cn2, dz, wl.n_sh, hi0[None], sh0[None])
    u0 = synth.input_field(wl, 1)
    a = wl.ar_a if wl.ar_a > 0 else 0.99
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    t0 = time.perf_counter()
    for r in range(reps):
        hi, sh = frames[r + 1]
        scr = orc.evolve_screens(N, wl.dx, psd, wl.lam, cn2, dz, wl.n_sh, a, 0.0, 0.0, 0.0, hi[None], sh[None], spec, shc)
        out = orc.propagate(N, wl.dx, wl.lam, dz, u0, scr, **kw)
        orc.beam_stats(N, wl.dx, out)
        orc.propagate_adjoint(N, wl.dx, wl.lam, dz, out, scr, **kw)
    dt = (time.perf_counter() - t0) / reps
    return dt, 2 * S_s


def oracle_all_cores(wl, S_s, B, timeout=240.0):
    """min(B, cores) realisations of the same sample side by side, one single-threaded oracle process each
    (the oracle is plain single-threaded C): n copies of `python bench.py --oracle-worker cid S_s seed`, each printing
    its seconds per frame.  Returns (screen-steps/s = all workers' units / the slowest worker's frame time,
    workers used, that time)."""
    n = max(1, min(B, os.cpu_count() or 1))
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="1", OPENBLAS_NUM_THREADS="1", MKL_NUM_THREADS="1")
    procs = [subprocess.Popen([sys.executable, os.path.abspath(__file__), "--oracle-worker", str(wl.cid), str(S_s),
                               str(1000 + i)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, env=env, text=True)
             for i in range(n)]
    dts, units = [], 0
    t_end = time.time() + timeout
    try:
        for p in procs:
            out, _ = p.communicate(timeout=max(1.0, t_end - time.time()))
            if p.returncode != 0:
                raise RuntimeError(f"oracle worker exited with {p.returncode}")
            dt, u = out.split()[-2:]
            dts.append(float(dt))
            units += int(u)
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    slow = max(dts)
    return units / slow, n, slow


def run_reference(args):
    """--impl reference: the oracle timed on the host cores on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2604_07248_b200 import synth
    wl = synth.CONFIGS[args.config]
    n_frames = args.steps + args.warmup
    probe, _ = oracle_frame(wl, 1)                       # one screen: sizes the sample
    budget = 150.0                                       # seconds for the whole run
    S_s = int(max(1, min(wl.S, budget / max(probe * n_frames, 1e-9))))
    for _ in range(args.warmup):
        oracle_frame(wl, S_s)
    ts = []
    for _ in range(args.steps):
        dt, units = oracle_frame(wl, S_s)
        ts.append(dt)
    ms = 1e3 * sum(ts) / len(ts)
    value = units / (ms * 1e-3)
    sample = f"1 realisation x {S_s} of {wl.S} screens per step (evolve + propagate + stats + adjoint)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "N": wl.N, "B": 1, "S": S_s, "n_sh": wl.n_sh, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# the product arm
# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2604_07248_b200 import api, synth
    from paper_2604_07248_b200 import build as b

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    if rank == 0:
        b.build()
    if world > 1:
        dist.barrier()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; the product has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")

    wl = synth.CONFIGS[args.config]
    N, S, n_sh = wl.N, wl.S, wl.n_sh
    B = args.batch if args.batch > 0 else wl.B           # realisations per GPU (weak scaling)
    px = N * N
    ctx = api.Context(local)
    psd = api.PsdParams(**wl.psd_dict())
    cn2, dz = list(wl.cn2_list), list(wl.dz)
    a = wl.ar_a if wl.ar_a > 0 else 0.99
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac,
              h_kind=api.H_ANGULAR_SPECTRUM if args.h_kind == "angular" else api.H_FRESNEL)

    # ---- synthetic inputs resident in HBM (seeded): two full frames of white
    # noise used alternately as the fresh noise of successive AR steps
    gen = torch.Generator(device=dev)
    gen.manual_seed(1234 + rank)
    def cnoise(*shape):
        return torch.view_as_complex(torch.randn(*shape, 2, device=dev, generator=gen, dtype=torch.float32))
    noise = [cnoise(B, S, N, N) for _ in range(2)]
    noise_sh = [cnoise(B, S, max(n_sh, 1), 3, 3) for _ in range(2)]
    spectrum = torch.empty((B, S, N, N), dtype=torch.complex64, device=dev)
    sh_coef = torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device=dev)
    screens = torch.empty((B, S, N, N), dtype=torch.float32, device=dev)
    u0 = torch.from_numpy(synth.input_field(wl, B)).to(dev)
    out = torch.empty_like(u0)
    gin = torch.empty_like(u0)
    stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device=dev)
    ws = ctx.workspace(N, wl.dx, B, S)
    ctx.make_screens(N, wl.dx, psd, wl.lam, cn2, dz, n_sh, noise[0], noise_sh[0] if n_sh else None,
                     spectrum=spectrum, sh_coef=sh_coef if n_sh else None, screens=screens, ws=ws)

    # The frame's fresh grid noise: drawn inside the generator's column kernel from (seed, frame) where that form exists
    # (ssp_evolve_screens_seeded; N = 512 / 1024, where it is the faster form: the paper's pipeline draws its noise on the GPU every frame),
    # read from one of the two resident noise frames elsewhere.  `resident_noise` times the second form on every grid.
    seeded = N in (512, 1024)                               # measured: 2048 / 4096 no faster than reading resident noise

    def frame(i, resident=not seeded):
        if resident:
            ctx.evolve_screens(N, wl.dx, psd, wl.lam, cn2, dz, n_sh, a, 0.0, 0.0, 0.0, noise[i & 1],
                               noise_sh[i & 1] if n_sh else None, spectrum, sh_coef if n_sh else None,
                               screens=screens, ws=ws)
        else:
            ctx.evolve_screens_seeded(N, wl.dx, psd, wl.lam, cn2, dz, n_sh, a, 0.0, 0.0, 0.0, 1234 + rank, 2 * i, 0,
                                      noise_sh[i & 1] if n_sh else None, spectrum, sh_coef if n_sh else None,
                                      screens=screens, ws=ws)
        ctx.propagate(N, wl.dx, wl.lam, dz, u0, screens, out=out, stats=stats, **kw)
        ctx.propagate_adjoint(N, wl.dx, wl.lam, dz, out, screens, out=gin, **kw)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    clk = ClockSampler(local) if rank == 0 else None
    for i in range(args.warmup):
        frame(i)
    sync_all()

    # ---- timed region: exactly K steps, CUDA events on the launching stream, the library's per-launch events OFF
    wall0 = time.time()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(args.steps):
        frame(args.warmup + i)
    e1.record()
    sync_all()
    wall1 = time.time()
    ms_total = e0.elapsed_time(e1)
    launches = ctx.launch_count() - l0
    clocks = clk.stop(wall0, wall1) if clk else None
    t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_step = ms_total / args.steps
    units_step = 2 * B * S * world                        # forward + adjoint screen-steps, all ranks
    value = units_step / (ms_step * 1e-3)

    # ---- second, profiled pass of the same steps: CUDA events recorded by the library around every launch
    # (kernels / roofline / split_step come from here; `value` above carries none of this overhead)
    n_prof = max(1, min(args.steps, 10))
    ctx.profile_enable(True)
    frame(args.warmup + args.steps)                       # creates the event pool outside the measured pass
    ctx.profile_report()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for i in range(n_prof):
        frame(args.warmup + args.steps + 1 + i)
    p1.record()
    sync_all()
    prof = ctx.profile_report()
    ctx.profile_enable(False)
    ms_prof_total = p0.elapsed_time(p1)

    # ---- the same step with the fresh noise read from a resident array instead of drawn in the kernel (reference figure)
    resident_noise = None
    if seeded:
        n_res = args.steps                                 # as many steps as the timed region: the same sustained clocks
        for i in range(args.warmup):
            frame(i, resident=True)
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        for i in range(n_res):
            frame(args.warmup + i, resident=True)
        r1.record()
        sync_all()
        t_res = torch.tensor([r0.elapsed_time(r1)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_res, op=dist.ReduceOp.MAX)
        ms_res = float(t_res.item()) / n_res
        resident_noise = {"what": "the step with ssp_evolve_screens reading the frame's fresh noise from a resident array "
                                  "(8 B/px more traffic, no draws)", "ms_per_step": ms_res,
                          "value": units_step / (ms_res * 1e-3), "steps": n_res}

    # ---- roofline of the dominant kernel class (by device time inside the timed region)
    peak, peak_src = peaks()
    NOMINAL = 8000.0                                      # GB/s, the HBM3e figure north_star names
    dom = max(prof.items(), key=lambda kv: kv[1]["ms"]) if prof else (None, None)
    roof = None
    if dom[0]:
        d = dom[1]
        achieved = d["bytes"] / (d["ms"] * 1e-3) / 1e9
        traffic = ncu_traffic(dom[0], N)
        roof = {"bound": "hbm", "kernel": dom[0], "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                "peak_nominal": NOMINAL, "frac_nominal": achieved / NOMINAL,
                "us_per_launch": 1e3 * d["ms"] / d["launches"], "bytes_per_launch": d["bytes"] / d["launches"],
                "share_of_step": d["ms"] / ms_prof_total,
                "timed": f"library CUDA events around each launch, separate profiled pass of {n_prof} steps after the timed region"}
    kernels = {k: {"launches": v["launches"], "ms": round(v["ms"], 4),
                   "GBps": round(v["bytes"] / (v["ms"] * 1e-3) / 1e9, 1)} for k, v in prof.items()}
    # split-step alone: col + row kernels of propagate and adjoint, 36 B/px per screen-step
    ss_ms = sum(v["ms"] for k, v in prof.items() if k.startswith(("col_fft", "row_", "small_")))
    ss_bytes = sum(v["bytes"] for k, v in prof.items() if k.startswith(("col_fft", "row_", "small_")))
    ss_gbps = ss_bytes / (ss_ms * 1e-3) / 1e9 if ss_ms else None
    split_step = {"screen_steps_per_s": 2 * B * S * n_prof / (ss_ms * 1e-3) if ss_ms else None,
                  "GBps": ss_gbps, "frac_of_peak": ss_gbps / peak if ss_ms else None,
                  "frac_of_nominal": ss_gbps / NOMINAL if ss_ms else None}

    # ---- forward-only temporal frame (the screens are used once): ssp_evolve_screens + ssp_propagate against
    # ssp_evolve_propagate, which synthesises each screen row inside the split step's row kernel (N = 1024)
    fwd_frame = None
    if N == 1024 and args.h_kind == "fresnel":
        ycol = torch.empty((B, S, N, N), dtype=torch.complex64, device=dev)
        def frame_unfused(i):
            ctx.evolve_screens(N, wl.dx, psd, wl.lam, cn2, dz, n_sh, a, 0.0, 0.0, 0.0, noise[i & 1],
                               noise_sh[i & 1] if n_sh else None, spectrum, sh_coef if n_sh else None, screens=screens, ws=ws)
            ctx.propagate(N, wl.dx, wl.lam, dz, u0, screens, out=out, stats=stats, **kw)
        def frame_fused(i):
            ctx.evolve_propagate(N, wl.dx, psd, wl.lam, cn2, dz, n_sh, a, 0.0, 0.0, 0.0, noise[i & 1],
                                 noise_sh[i & 1] if n_sh else None, spectrum, sh_coef if n_sh else None, u0, ycol,
                                 win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac, out=out, stats=stats, ws=ws)
        def time_frames(fn, n):
            fn(0); fn(1)
            sync_all()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record()
            for i in range(n):
                fn(i)
            f1.record()
            sync_all()
            return f0.elapsed_time(f1) / n
        n_ff = max(2, min(args.steps, 10))
        ms_u, ms_f = time_frames(frame_unfused, n_ff), time_frames(frame_fused, n_ff)
        fwd_frame = {"what": "forward-only frame, device resident: evolve_screens + propagate + stats (unfused) against "
                             "ssp_evolve_propagate (screen row pass fused into the split step's row kernel)",
                     "unfused_ms": ms_u, "fused_ms": ms_f, "fused_screen_steps_per_s": B * S * world / (ms_f * 1e-3),
                     "unfused_screen_steps_per_s": B * S * world / (ms_u * 1e-3), "speedup": ms_u / ms_f}
        del ycol

    # ---- e2e: through ssp_frame_host with pinned HOST buffers.  Per step: the input fields go host -> device, the
    # screen stacks are evolved ON the device from (seed, stream) noise draws (the paper's pipeline draws its noise on
    # the GPU too), the fields propagate, output fields and statistics come back; chunks of the batch overlap.
    # "host_screens" is the variant in which the host also supplies every screen (PCIe-bound: 4 B/px per screen-step).
    e2e = None
    if not args.no_e2e:
        h_in = torch.from_numpy(synth.input_field(wl, B)).pin_memory()
        h_out = torch.empty_like(h_in).pin_memory()
        h_st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8).pin_memory()
        d_field = torch.empty_like(u0)
        n_e2e = max(1, min(args.steps, 5))
        step_no = [0]
        Bc = api.frame_chunk(B)
        d_noise = noise[0][:Bc]                                # chunk-sized scratch for the device-side draws
        h_adj = torch.empty_like(h_in).pin_memory()
        def e2e_step(adjoint=True):
            i = step_no[0] = step_no[0] + 1
            ctx.frame_host(N, wl.dx, psd, wl.lam, cn2, dz, n_sh, a, 0.0, 0.0, 0.0, 1234 + rank, i, h_in, h_out, h_st, 0.5,
                           d_field, spectrum, sh_coef, screens, d_noise, noise_sh[0], stats, ws,
                           win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac, h_kind=kw["h_kind"],
                           h_adjoint_out=h_adj if adjoint else None, d_adjoint=gin if adjoint else None)
        def timed(fn, n):
            fn()
            sync_all()
            t0 = time.perf_counter()
            for _ in range(n):
                fn()                                          # synchronises the stream itself
            dt = (time.perf_counter() - t0) / n
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        dt = timed(e2e_step, n_e2e)
        dt_fwd = timed(lambda: e2e_step(False), n_e2e)
        e2e = {"value": 2 * B * S * world / dt, "unit": UNIT,
               "what": "the step `value` times, through ssp_frame_host with pinned HOST buffers: fields host -> device, "
                       "device-side noise draws + AR screen evolution + forward propagate + stats + adjoint propagate, "
                       "received fields, statistics and adjoint fields device -> host (forward + adjoint screen-steps counted)",
               "h2d_bytes_per_step": int(h_in.numel() * 8),
               "d2h_bytes_per_step": int(h_out.numel() * 8 + h_adj.numel() * 8 + h_st.numel()),
               "ms_per_step": dt * 1e3,
               "forward_only": {"value": B * S * world / dt_fwd, "ms_per_step": dt_fwd * 1e3,
                                "what": "the same call without the adjoint leg (forward screen-steps only)",
                                "h2d_bytes_per_step": int(h_in.numel() * 8),
                                "d2h_bytes_per_step": int(h_out.numel() * 8 + h_st.numel())}}
        del noise[1:], noise_sh[1:]                          # make room for the pinned copy of the screens
        h_scr = screens.cpu().pin_memory()
        def e2e_host_screens():
            ctx.propagate_host(N, wl.dx, wl.lam, dz, h_in, h_out, h_scr, False, S, wl.win_order,
                               wl.win_sigma_frac, h_st, 0.5, d_field, screens, stats, h_kind=kw["h_kind"])
        dt2 = timed(e2e_host_screens, max(1, min(args.steps, 3)))
        e2e["host_screens"] = {"what": "forward only, the host also supplies every screen (ssp_propagate_host)",
                               "value": B * S * world / dt2, "ms_per_step": dt2 * 1e3,
                               "h2d_bytes_per_step": int(h_in.numel() * 8 + h_scr.numel() * 4),
                               "d2h_bytes_per_step": int(h_out.numel() * 8 + h_st.numel())}

    # ---- comparison only: the same forward split steps with cuFFT through torch.fft plus
    # elementwise torch kernels -- the paper's own design -- never on the product path
    cufft = None
    if rank == 0 and world == 1 and not args.no_cufft_compare:
        import math
        fx = torch.fft.fftfreq(N, d=wl.dx, device=dev, dtype=torch.float64)
        H = torch.exp(-1j * math.pi * wl.lam * dz[0] * (fx[None, :] ** 2 + fx[:, None] ** 2)).to(torch.complex64)
        xc = (torch.arange(N, device=dev, dtype=torch.float64) - N // 2) * wl.dx
        sig = wl.win_sigma_frac * N * wl.dx
        W = torch.exp(-(((xc[None, :] ** 2 + xc[:, None] ** 2) / sig ** 2) ** (wl.win_order / 2))).to(torch.float32)
        def torch_forward():
            u = u0
            for j in range(S):
                u = torch.fft.ifft2(torch.fft.fft2(u) * H)
                u = u * torch.polar(W.expand(B, N, N), screens[:, j])
            return u
        torch_forward()
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_rep = 3
        c0.record()
        for _ in range(n_rep):
            torch_forward()
        c1.record()
        torch.cuda.synchronize()
        ms = c0.elapsed_time(c1) / n_rep
        ours_fwd = sum(v["ms"] for k, v in prof.items() if k.startswith(("col_fft", "row_", "small_"))) / n_prof / 2
        cufft = {"what": "forward split steps with torch.fft (cuFFT) + elementwise torch kernels, same batch; comparison only",
                 "screen_steps_per_s": B * S / (ms * 1e-3), "ms_per_forward": ms,
                 "ours_ms_per_forward": ours_fwd, "speedup": ms / ours_fwd if ours_fwd else None}

    # ---- the oracle on the host cores, bounded sample (rank 0, N=1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        probe, _ = oracle_frame(wl, 1)                    # one screen: sizes a sample of about 15 s
        S_s = int(max(1, min(S, 15.0 / max(probe, 1e-9))))
        dt, units = oracle_frame(wl, S_s)
        sample = f"1 realisation x {S_s} of {S} screens, one frame (evolve + propagate + stats + adjoint), {dt:.1f} s"
        cpu = {"value": units / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample}
        try:                                              # min(B, cores) realisations side by side, one process each
            v_all, n_all, slow = oracle_all_cores(wl, S_s, B)
            cpu = {"value": v_all, "unit": UNIT, "cores": n_all, "kind": "oracle",
                   "sample": f"{n_all} realisations side by side (one single-threaded oracle process each; host has "
                             f"{os.cpu_count()} cores), each {S_s} of {S} screens, one frame (evolve + propagate + stats + "
                             f"adjoint), slowest {slow:.1f} s",
                   "single_core": {"value": units / dt, "cores": 1, "sample": sample}}
        except Exception as exc:                          # keep the single-core figure
            cpu["all_cores_error"] = repr(exc)[:200]

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl.name, "N": N, "B_per_gpu": B, "S": S, "n_sh": n_sh, "ar_a": a, "h_kind": args.h_kind,
                       "step": ("evolve_screens_seeded (fresh noise drawn in the generator)" if seeded else "evolve_screens")
                               + " + propagate + beam_stats + propagate_adjoint",
                       "timing": "CUDA events around the K steps, library profiling off; kernels / roofline / split_step from a separate profiled pass",
                       "units_per_step": units_step,
                       "l2": "inputs larger than L2 (no flush): each step streams > 10 GB"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches) * world, "roofline": roof,
            "cpu_baseline": cpu, "kernels": kernels, "split_step": split_step, "resident_noise": resident_noise,
            "forward_frame": fwd_frame, "cufft_comparison": cufft,
        }
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    if len(sys.argv) == 5 and sys.argv[1] == "--oracle-worker":   # one realisation of the all-cores oracle leg
        from paper_2604_07248_b200 import synth
        from oracle import orc
        orc.lib()
        dt, units = oracle_frame(synth.CONFIGS[int(sys.argv[2])], int(sys.argv[3]), seed=int(sys.argv[4]))
        print(dt, units)
        return
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
