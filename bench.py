#!/usr/bin/env python
"""bench.py — throughput of the RK3 hot path on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--path 55|19] [--impl ours|reference]

A "step" is one full RK3 step (3 substeps: halo fill + fused 55-point kernel, or the 19-point kernel pair) of
the whole grid.  Workload at N = 1: config C4 of BASELINE.json (512^3 fp32, seeded band-limited fields,
|k| <= 32, rms Mach 0.3, nu = 1e-3), the configuration the metric is quoted on; the 2.1 GB state and the
8.6 GB each substep streams are far larger than the 126 MB L2, so no L2 flush is needed between steps.
N > 1: independent replicas (the north_star path is single-GPU; no collective is
invented), value = cells of all ranks x K / max-over-ranks device time.

value        device-resident: K steps in one fd_rk3_step(dt, K) call, CUDA events on the launching stream; the call is
             repeated --reps times (default 5) back to back from the same state and `value` is the MEDIAN repetition
             (value_min / value_max / values beside it; the clock sampler runs across all repetitions).
value_sustained  the same call sized to run >= 1.2 s (the board's power cap engages after ~0.1 s of this kernel): the
             figure that answers "sustains"; details under "sustained".
e2e          the same job through the C ABI with HOST (pinned) buffers: fd_load(host) + fd_rk3_step(dt, K) +
             fd_store(host), copies inside the timed region; bytes per step = job bytes / K.  The variant
             with a load and a store around EVERY step is reported as e2e.every_step_io.
roofline     fused 55-point kernel: algorithmic bytes (16 words/cell/substep) / mean launch
             duration from the library's per-launch CUDA events (fd_set_profiling) over the timed region.
cpu_baseline the CPU oracle as it stands, timed on the host cores on a bounded sample (rank 0, N = 1).
--impl reference   times the oracle only (there is no reference implementation; the oracle is the arm).
"""
import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Mcell-updates/s per full RK3 step"
UNIT = "Mcell-updates/s"
WORDS_PER_CELL_SUBSTEP = {"55": 16, "19": 30}  # the contract figure
# what a step really moves: w is not read on substep 1 and not written on substep 3 (alpha_1 = 0)
WORDS_PER_CELL_STEP_ACTUAL = {"55": 12 + 16 + 12, "19": 3 * 30 - 8}
DOMINANT_WORDS_ACTUAL_MEAN = {"55": (12 + 16 + 12) / 3.0, "19": (13 + 17 + 13) / 3.0}  # dominant kernel, mean over substeps
NOMINAL_HBM_GBS = 8000.0  # B200 data sheet, the figure BASELINE.md's 70 % target is stated against


def load_ncu_table():
    """profiles/ncu_traffic.json: per (config, kernel, variant) the DRAM bytes and unit utilisations ncu measured for
    the launch that reads and writes w, each with the profile file it comes from (never a literal in this file)."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f)["entries"]
    except Exception:
        return []


def ncu_entry(config, kernel, variant):
    for e in load_ncu_table():
        if e.get("config") == config and e.get("kernel") == kernel and e.get("variant") == variant:
            return e
    return None


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.01):
        self.index, self.period = index, period
        self.samples, self.power, self.reasons, self.max_mhz = [], [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                except Exception:
                    pass
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_mhz_min": (s[0] if s else None), "sm_max_mhz": self.max_mhz,
                "power_w_max": (round(max(self.power), 1) if self.power else None),
                "reasons": sorted(self.reasons), "samples": len(s)}


def load_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# --------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference): the ONLY place bench.py touches oracle/.
# --------------------------------------------------------------------------------------------------
def oracle_sample(cfg, path_name, budget_s, n_sample=None):
    """Time the oracle, as it stands, in the config's dtype on a bounded sample of the workload: the config's
    own recipe on an n_sample^3 periodic grid (same spectrum, dx, dt, nu), 1 step + as many more as fit."""
    import numpy as np
    from oracle import oracle as O
    from paper_1707_08900_b200 import inputs

    n = n_sample or min(cfg.n, 128)
    F = inputs.make_state(cfg, device="cpu", n_override=n)
    F = F if isinstance(F, np.ndarray) else F.numpy()
    dt_np = cfg.np_dtype
    path = O.PATH_55 if path_name == "55" else O.PATH_19
    dx = 2 * math.pi / n
    dt = 0.1 * dx / cfg.cs
    O.rk3_step(F[:, :16, :16, :16], dx, cfg.nu, cfg.cs, dt, 1, path, dtype=dt_np)  # builds/loads the library
    t0 = time.perf_counter()
    G = O.rk3_step(F, dx, cfg.nu, cfg.cs, dt, 1, path, dtype=dt_np)
    t1 = time.perf_counter() - t0
    more = int(max(0, min(50, math.floor((budget_s - t1) / max(t1, 1e-3)))))
    total_steps, total_t = 1, t1
    if more > 0:
        t0 = time.perf_counter()
        O.rk3_step(G, dx, cfg.nu, cfg.cs, dt, more, path, dtype=dt_np)
        total_t += time.perf_counter() - t0
        total_steps += more
    value = n ** 3 * total_steps / total_t / 1e6
    return {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"{cfg.name} recipe on a {n}^3 periodic grid, {cfg.dtype}, {path_name}-point path, "
                      f"{total_steps} full RK3 steps in {total_t:.1f} s (oracle/fd_oracle.cpp, OpenMP over k-planes)"}, total_t, total_steps, n


def run_reference(args, cfg):
    rank = _env_int("RANK", 0)
    if rank != 0:
        return 0
    steps, warm = max(1, args.steps), max(0, args.warmup)
    # each "step" of this arm = one oracle RK3 step on a bounded sample, sized so the whole run ends in minutes
    import numpy as np
    from oracle import oracle as O
    from paper_1707_08900_b200 import inputs
    n = 128
    F = inputs.make_state(cfg, device="cpu", n_override=n)
    F = F if isinstance(F, np.ndarray) else F.numpy()
    path = O.PATH_55 if args.path == "55" else O.PATH_19
    dx = 2 * math.pi / n
    dt = 0.1 * dx / cfg.cs
    for _ in range(min(warm, 3)):
        O.rk3_step(F, dx, cfg.nu, cfg.cs, dt, 1, path, dtype=cfg.np_dtype)
    t0 = time.perf_counter()
    done = 0
    for _ in range(steps):
        F = O.rk3_step(F, dx, cfg.nu, cfg.cs, dt, 1, path, dtype=cfg.np_dtype)
        done += 1
        if time.perf_counter() - t0 > 150.0:
            break
    el = time.perf_counter() - t0
    value = n ** 3 * done / el / 1e6
    sample = (f"{cfg.name} recipe on a {n}^3 periodic grid, {cfg.dtype}, {args.path}-point path, one oracle RK3 step "
              f"per bench step ({done} timed)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": done,
            "warmup": min(warm, 3), "ms_per_step": el / done * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {cfg.n}^3 periodic {cfg.dtype}, sampled at {n}^3 for the CPU oracle",
                       "path": args.path},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--path", default="55", choices=["55", "19"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", type=int, default=0, help="0 auto, 1 direct, 2 tiled, 3 paired")
    ap.add_argument("--tile-shape", type=int, default=-1, help="-1 automatic, 0 wide (12 warps), 1 tall (8 warps x 2 values)")
    ap.add_argument("--tile-overlap", type=int, default=0,
                    help="measurement aid (include/fd6_testing.h): tiles overlap by this many values, same results, the redundant "
                         "halo-ring work of temporal blocking (DESIGN.md section 7)")
    ap.add_argument("--forcing", action="store_true",
                    help="switch the forcing term of Eq. 2 on (Eq. 24-25; off in the paper's performance runs, PAPER.md:369)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sustained", action="store_true", help="skip the >= 1 s sustained measurement")
    ap.add_argument("--sustained-seconds", type=float, default=1.2)
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--reps", type=int, default=5, help="repetitions of the timed K-step call; value = their median")
    ap.add_argument("--forcing-every-step", action="store_true",
                    help="extra measurement: fd_set_forcing with a new wavevector before every single step (PAPER.md:460), "
                         "the case in which a step is never captured into a CUDA graph")
    args = ap.parse_args()

    from paper_1707_08900_b200 import inputs
    cfg = inputs.CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist
    from paper_1707_08900_b200 import fd6  # raises if libfd6.so is missing: no CPU fallback
    from paper_1707_08900_b200 import replicas

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (the product path has no CPU fallback)"
    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K, W = max(1, args.steps), max(3, args.warmup)
    n, N = cfg.n, cfg.n ** 3
    esize = 4 if cfg.dtype == "f32" else 8

    def barrier():
        replicas.barrier("cuda")

    def max_ms(ms_):
        return replicas.max_over_ranks(ms_, "cuda")

    # seeded synthetic state, generated on the device (harness only) then handed to fd_load
    F0 = inputs.make_state(cfg, device="cuda")
    if not isinstance(F0, torch.Tensor):
        F0 = torch.from_numpy(F0).cuda()
    ctx = fd6.Fd(n, n, n, cfg.dx, cfg.nu, cfg.cs, fd6.FD_F32 if cfg.dtype == "f32" else fd6.FD_F64)
    ctx.fd_set_path(fd6.FD_PATH_55 if args.path == "55" else fd6.FD_PATH_19)
    if args.variant:
        ctx.fd_set_variant(args.variant)
    if args.tile_shape >= 0:
        ctx.fd_set_tile_shape(args.tile_shape)
    if args.tile_overlap:
        from paper_1707_08900_b200 import fd6_testing
        fd6_testing.fd_debug_set_tile_overlap(ctx, args.tile_overlap)
    info = ctx.fd_get_info()  # what the context really launches (variant, prepared tile shape, work items)
    tile = None
    if info.variant in (2, 3):
        tile = (f"{'automatic' if args.tile_shape < 0 else 'forced'}: {('wide', 'tall')[info.tile_shape]} "
                f"{info.tile_x}x{info.tile_y} values, {info.work_items} work items")
        if info.variant == 2 and cfg.dtype == "f32":
            tile += " (y pairs)"
    forcing = dict(k=(3.0, 2.0, -4.0), e=(0.36, -0.48, 0.8), phi=0.7, f0=0.05) if args.forcing else None
    if forcing:
        ctx.fd_set_forcing(forcing["k"], forcing["e"], forcing["phi"], forcing["f0"], cfg.dt)
    ctx.load_state(F0)
    ctx.fd_rk3_step(cfg.dt, W)  # warm-up
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed_steps(nsteps, profiling, reps=1):
        """`reps` times: nsteps steps from the config's state in ONE fd_rk3_step call, CUDA events on the launching stream.
        Returns the per-repetition device times (ms), the launches of one repetition, the clock record, the profile."""
        ctx.fd_set_profiling(profiling)
        times, n_launch = [], 0
        with ClockSampler(local) as clk_:
            for _ in range(reps):
                ctx.load_state(F0)
                if profiling:
                    ctx.fd_reset_profile()
                barrier()
                n0 = ctx.fd_kernel_launches()
                e0.record(stream)
                ctx.fd_rk3_step(cfg.dt, nsteps)
                e1.record(stream)
                barrier()
                times.append(e0.elapsed_time(e1))
                n_launch = ctx.fd_kernel_launches() - n0
        prof_ = {fd6.KERNEL_NAMES[k]: ctx.fd_get_profile(k) for k in range(fd6.FD_K_COUNT)} if profiling else None
        ctx.fd_set_profiling(False)
        return times, n_launch, clk_, prof_

    # pass 1: `value` - right after the W warm-up steps, profiling off, each step one CUDA graph launch; the median of
    # `reps` back-to-back repetitions (>= 5 repetitions, report median and min)
    reps = max(1, args.reps)
    rep_ms, launches, clk, _ = timed_steps(K, False, reps)
    graph_state = ctx.fd_get_info().graph_state
    rep_ms = sorted(max_ms(t) for t in rep_ms)
    ms_max = rep_ms[len(rep_ms) // 2] if len(rep_ms) % 2 else 0.5 * (rep_ms[len(rep_ms) // 2 - 1] + rep_ms[len(rep_ms) // 2])
    # pass 2: the per-kernel profile (two event records around every launch: kept out of `value`)
    prof_ms, _, _, prof = timed_steps(K, True)
    prof_ms = max_ms(prof_ms[0])
    chk = torch.empty_like(F0)
    ctx.store_state(chk)
    ctx.fd_sync()
    finite = bool(torch.isfinite(chk).all().item())
    del chk
    value = replicas.whole_job_value(N, K, ms_max, world)
    rep_values = [replicas.whole_job_value(N, K, t, world) for t in rep_ms]  # descending

    # pass 3: the same measurement sustained over >= 1 s (the 1 kW power cap engages after ~0.1 s of this kernel)
    sustained = None
    if not args.no_sustained:
        Ks = max(K, int(math.ceil(args.sustained_seconds * 1e3 / (ms_max / K))))
        s_ms, _, s_clk, _ = timed_steps(Ks, False)
        s_ms = max_ms(s_ms[0])
        sustained = {"value": replicas.whole_job_value(N, Ks, s_ms, world), "unit": UNIT, "steps": Ks, "seconds": s_ms * 1e-3,
                     "ms_per_step": s_ms / Ks, "clocks": s_clk.summary()}
        sustained["vs_burst"] = sustained["value"] / value

    # optional: a new forcing wavevector before EVERY step: fd_set_forcing + fd_rk3_step(dt, 1), K times
    forcing_each = None
    if args.forcing_every_step:
        kf0 = 2 * math.pi / (n * cfg.dx)

        def forced_steps(count):
            for s_ in range(count):
                ctx.fd_set_forcing((kf0 * (2 + s_ % 3), kf0 * (1 + s_ % 2), -kf0 * 3), (0.36, -0.48, 0.8), 0.1 * s_, 0.05, cfg.dt)
                ctx.fd_rk3_step(cfg.dt, 1)

        ctx.load_state(F0)
        forced_steps(3)
        fe = []
        for _ in range(reps):
            ctx.load_state(F0)
            barrier()
            e0.record(stream)
            forced_steps(K)
            e1.record(stream)
            barrier()
            fe.append(max_ms(e0.elapsed_time(e1)))
        fe.sort()
        forcing_each = {"value": replicas.whole_job_value(N, K, fe[len(fe) // 2], world), "unit": UNIT,
                        "ms_per_step": fe[len(fe) // 2] / K, "graph_state_after": int(ctx.fd_get_info().graph_state),
                        "note": "fd_set_forcing (host tables, one H2D copy, a stream synchronise) + fd_rk3_step(dt, 1) per step; "
                                "graph_state 1 = FD_GRAPH_WAITING: plain launches, nothing captured"}
        ctx.fd_set_forcing(None, None, 0.0, 0.0, cfg.dt)
        if forcing:
            ctx.fd_set_forcing(forcing["k"], forcing["e"], forcing["phi"], forcing["f0"], cfg.dt)

    state_mb = 4 * N * esize / 1e6
    l2_note = (f"inputs larger than L2 ({state_mb / 1e3:.1f} GB state, {16 * esize * N / 1e9:.1f} GB streamed per substep); no flush needed"
               if state_mb > 3 * 126 else
               f"state of {state_mb:.0f} MB fits the 126 MB L2 and stays there from step to step, as in any run of this "
               "size (a time stepper has no cold-cache step after the first); no flush - throughput of consecutive steps")

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region
    host_in = torch.empty(F0.shape, dtype=F0.dtype, pin_memory=True)
    host_in.copy_(F0)
    host_out = torch.empty(F0.shape, dtype=F0.dtype, pin_memory=True)
    state_bytes = 4 * N * esize

    def e2e_job(nsteps):
        ctx.load_state(host_in)       # fd_load(FD_HOST): H2D + pack + halo fill
        ctx.fd_rk3_step(cfg.dt, nsteps)
        ctx.store_state(host_out)     # fd_store(FD_HOST): unpack + D2H, synchronises

    e2e_job(1)
    barrier()
    e0.record(stream)
    e2e_job(K)
    e1.record(stream)
    barrier()
    e2e_ms = max_ms(e0.elapsed_time(e1))
    e2e_value = replicas.whole_job_value(N, K, e2e_ms, world)
    io_reps = 3
    barrier()
    e0.record(stream)
    for _ in range(io_reps):
        e2e_job(1)
    e1.record(stream)
    barrier()
    e2e_each = replicas.whole_job_value(N, io_reps, max_ms(e0.elapsed_time(e1)), world)
    finite = finite and bool(torch.isfinite(host_out).all().item())

    # ---- roofline of the dominant kernel
    peak, peak_src = load_peak()
    dom = "fused55" if args.path == "55" else "pass1_19"
    words = 16 if args.path == "55" else 17
    dom_ms, dom_n = prof[dom]
    alg_bytes = words * esize * N
    avg_launch_s = dom_ms / dom_n * 1e-3 if dom_n else None
    achieved = alg_bytes / avg_launch_s / 1e9 if dom_n else None
    actual = DOMINANT_WORDS_ACTUAL_MEAN[args.path] * esize * N / avg_launch_s / 1e9 if dom_n else None
    kern_share = {k: round(v[0] / prof_ms, 4) for k, v in prof.items() if v[1]}
    variant_name = {1: "direct", 2: "tiled", 3: "paired"}.get(info.variant, str(info.variant))
    ncu = (ncu_entry(args.config, dom, variant_name) or {}) if args.tile_shape < 0 and not args.tile_overlap else {}
    step_gbs = WORDS_PER_CELL_SUBSTEP[args.path] * esize * 3 * N * K / (ms_max * 1e-3) / 1e9
    step_gbs_actual = WORDS_PER_CELL_STEP_ACTUAL[args.path] * esize * N * K / (ms_max * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": (achieved / peak if achieved else None),
                "frac_is": (f"contract figure: {words} words per cell and launch (SURVEY 8(d)); averaged over the three substeps a "
                            f"launch moves {DOMINANT_WORDS_ACTUAL_MEAN[args.path]:.1f} (w skipped on substeps 1 and 3): frac_actual_bytes"),
                "frac_nominal": (achieved / NOMINAL_HBM_GBS if achieved else None),
                # the same launches counted with the bytes they really move (w skipped on substeps 1 and 3)
                "achieved_actual_bytes": actual, "frac_actual_bytes": (actual / peak if actual else None),
                "traffic": ncu.get("dram_bytes"), "traffic_source": ncu.get("source"),
                "dram_pct_ncu": ncu.get("dram_pct"), "l1tex_pct_ncu": ncu.get("l1tex_pct"),
                "algorithmic_bytes_per_launch": alg_bytes, "avg_launch_ms": (dom_ms / dom_n if dom_n else None),
                "peak_source": peak_src, "nominal_peak": NOMINAL_HBM_GBS, "kernel_share_of_step": kern_share,
                "step_frac": step_gbs / peak, "step_frac_nominal": step_gbs / NOMINAL_HBM_GBS,
                "step_frac_actual_bytes": step_gbs_actual / peak,
                "timing": "per-launch CUDA events recorded by the library on its stream in a separate profiled pass "
                          f"({K} steps, {prof_ms / K:.3f} ms/step); value/ms_per_step come from the unprofiled pass"}
    if sustained is not None:
        roofline["step_frac_sustained"] = step_gbs / peak * sustained["vs_burst"]

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline = oracle_sample(cfg, args.path, args.cpu_budget)[0]

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": cfg.dtype, "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {n}^3 periodic {cfg.dtype}, band-limited |k|<={cfg.kmax} rms Mach {cfg.amp}, "
                                   f"nu={cfg.nu}, dt=0.1 dx/cs", "path": f"{args.path}-point",
                       "variant": variant_name, "tile_shape": tile, "tile_overlap": args.tile_overlap,
                       "l2": l2_note,
                       "launch": {0: "plain launches (graphs off)", 1: "plain launches (graph not captured)",
                                  2: "one CUDA graph per RK3 step (fd_get_info: FD_GRAPH_CAPTURED)",
                                  3: "plain launches (graph capture failed: " + info.graph_note.decode() + ")"}[int(graph_state)],
                       "parallelism": "replicas only" if world > 1 else "single GPU", "finite": finite,
                       "forcing": (f"on: k={forcing['k']}, f0={forcing['f0']}" if forcing else "off (PAPER.md:369)")},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes / K,
                    "d2h_bytes_per_step": state_bytes / K,
                    "job": f"fd_load(host pinned) + fd_rk3_step(dt,{K}) + fd_store(host pinned)", "ms": e2e_ms,
                    "every_step_io": {"value": e2e_each, "h2d_bytes_per_step": state_bytes,
                                      "d2h_bytes_per_step": state_bytes}},
            "gpu_launches": int(launches), "clocks": clk.summary(), "roofline": roofline,
        }
        line["value_min"], line["value_max"] = rep_values[-1], rep_values[0]
        line["values"] = [round(v, 1) for v in rep_values]
        line["reps"] = reps
        line["value_is"] = f"median of {reps} back-to-back repetitions of fd_rk3_step(dt, {K})"
        if sustained is not None:
            line["value_sustained"] = sustained["value"]
            line["sustained"] = sustained
        if forcing_each is not None:
            line["forcing_every_step"] = forcing_each
        if cpu_baseline is not None:
            line["cpu_baseline"] = cpu_baseline
        print(json.dumps(line), flush=True)
    ctx.fd_destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0 if finite else 1


if __name__ == "__main__":
    sys.exit(main())
