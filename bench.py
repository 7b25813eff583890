#!/usr/bin/env python
"""bench.py -- Wilson-loop point-evals/s on the paper-scale ensemble (BASELINE.json config 3).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 3]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
           --master-port P bench.py --gpus N --steps K --warmup W

One "step" = one pass of the whole hot path over one ensemble:
wl_eval (k_wilson + k_group_reduce + k_mean) -> [N > 1: all-gather of the group sums] ->
wl_jackknife_finalize.  metric = N_l * N_ppl * N_T * N_rho / time (loop-point evaluations per second).

  value     : loops resident in HBM, timed on the device with CUDA events, max over ranks.
  e2e       : the same step through the C-ABI call on HOST buffers (wl_eval_host: pinned host loops
              -> device, kernels, results -> host inside the timed region).
  roofline  : the dominant kernel (k_wilson) against the FP32 non-tensor issue roofline (DESIGN.md
              section 5): achieved = 36 algorithmic lane-ops per point-eval x point-evals / kernel time.
  cpu_baseline : the FP64 oracle (oracle/wl_oracle.c, as it stands) on a bounded sample, host cores.
  --impl reference : times the oracle alone (this tier's reference arm); needs no GPU.

Multi-GPU (weak scaling): every rank holds its own 16384 loops of one N x 16384-loop ensemble
(whole jackknife groups per rank, paper_1407_7486_b200/shard.py); the only exchange is one all-gather
of the group sums per step.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "wilson_loop_point_evals_per_s"
UNIT = "point-evals/s"

# algorithmic work per point-eval of the sech^2 profile in FP32
# (SURVEY.md section 8(d)): 29 plain FP32 lane-ops + 7 special-function lane-ops at the midpoint rule; every
# further Gauss-Legendre node of eq. (24) adds, in the easiest case (far from the axis, where the logarithm is a
# degree-1 polynomial and the reciprocal is shared): radius 2, u' 1, 1+E 1, denominator product and its share of the
# inverse 2, bracket 2, 1/w' 1, g 1, weighted sum 1 = 11 plain, and rsqrt + 2^x = 2 special-function lane-ops.
# (The survey gives a count for the midpoint rule only; counting the easiest case keeps `frac` a lower bound.)
ALG_PLAIN_OPS = 29
ALG_SFU_OPS = 7
ALG_NODE_PLAIN_OPS = 11
ALG_NODE_SFU_OPS = 2
ALG_OPS_UNIFORM = 4
ALG_OPS_FLUXTUBE = 16             # 14 plain + 2 reciprocals
# FP64 has no special-function unit: the seven elementary functions are counted as their shortest double-precision
# sequences (2 x sqrt/rsqrt: 9, 2 x 2^x: 13, 2 x reciprocal: 4, log2(1+E): 3 -- the degree the polynomial needs far from
# the axis, the easiest case; near it the same accuracy takes degree 20) + the 29 plain ops: 84.  Counting the easiest
# case keeps `frac` a lower bound whatever mix of near and far blocks a workload has.
ALG_F64_OPS_SECH2 = 84
KERNEL_F64_OPS_SECH2 = 73         # FP64-pipe instructions k_wilson<Sech2LeanF64> issues per point-eval in its farthest tier (97 in tier 0)
SM_COUNT = 148
ISSUE_LANES_PER_CLK_SM = 128      # 4 sub-partitions x 1 warp instruction (32 lanes) per clock
FP64_LANES_PER_CLK_SM = 64        # measured 63.8 (profiles/r01_pipe_rates.md)
SFU_LANES_PER_CLK_SM = 16         # measured 15.9
KERNEL_SFU_OPS = 4                # MUFU per point-eval in k_wilson<Sech2PackedF32> at Q = 1 (sqrt, rsqrt, 2 x ex2); + 2 per extra node.
                                  # The one reciprocal per staged point and thread runs on the FMA pipe (256-thread kernels
                                  # without phi_cm) or is a MUFU shared by the P = 2 grid points of a thread (grids <= 256 points)

def affinity_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    def __init__(self, index, period=0.02):
        super().__init__(daemon=True)
        self.period = period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def nvml_index_for(device_index):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[device_index])
        except (ValueError, IndexError):
            pass
    return device_index


def oracle_sample_loops(cfg, cores, per_four_cores):
    """Whole-loop sample size for the oracle legs: `per_four_cores` loops per 4 host cores."""
    n = per_four_cores * max(1, cores // 4)
    return max(1, min(cfg.n_loops, n))


def time_oracle(cfg, loops_host, T, rho, phi):
    from oracle import wl_oracle as oracle
    n = loops_host.shape[0]
    G = 1
    t0 = time.perf_counter()
    oracle.evaluate(cfg.profile, cfg.params, loops_host, T, rho, phi, n_groups=G)
    dt = time.perf_counter() - t0
    evals = n * cfg.n_ppl * len(T) * len(rho)
    return evals / dt, dt, oracle.num_threads()


def base_line(args, cfg, n_gpus):
    return {
        "metric": METRIC, "unit": UNIT, "n_gpus": n_gpus, "steps": args.steps, "warmup": args.warmup,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "data": "synthetic",
    }


def workload_config(cfg, n_gpus):
    return {
        "workload": cfg.name,
        "n_loops_per_gpu": cfg.n_loops, "n_loops_total": cfg.n_loops * n_gpus, "n_ppl": cfg.n_ppl,
        "n_T": cfg.n_T, "n_rho": cfg.n_rho, "n_groups_total": cfg.n_groups * n_gpus,
        "field": {"profile": "sech2" if cfg.profile == 1 else "uniform", "params": list(cfg.params)},
        "loop_storage": cfg.loop_dtype, "seed": cfg.seed,
        "parallelism": "dp%d (whole jackknife groups per rank)" % n_gpus,
        "cache": "inputs larger than L2 (%.0f MB of loop coordinates per step vs 126 MB L2)"
                 % (cfg.n_loops * cfg.n_ppl * 2 * (4 if cfg.loop_dtype == "f32" else 8) / 1e6),
    }


def kernel_sfu_ops(n_grid, has_phi, Q, scalar=False):
    """MUFU instructions per point-eval of k_wilson<Sech2PackedF32>, from the predicates the dispatcher uses
    (wl_wilson_sech2_f32.cu, wl_terms_packed_f32.cuh): sqrt, rsqrt and two ex2 at the midpoint rule (the scalar-only
    variant, which has no spin sum, issues 2), + 2 per further Gauss-Legendre node; the one reciprocal
    per staged point and thread is shared by the P grid points of the thread and is a MUFU unless kFmaRcp
    (= fermion loops, no phi_cm, 256-thread tiles) puts it on the FMA pipe."""
    threads = 128 if n_grid <= 256 else 256
    P = 4 if (n_grid >= 1024 and Q == 1) else 2
    fma_rcp = (not scalar) and (not has_phi) and threads >= 256
    base = 2 if scalar else KERNEL_SFU_OPS
    return base + 2 * (Q - 1) + (0.0 if fma_rcp else 1.0 / P)


def kernel_roofline(cfg, compute, Q, has_phi, sm_max_mhz):
    """(algorithmic lane-ops per point-eval, how counted, peak lane-ops/s, how derived, pipe_frac or None) of the
    k_wilson instantiation that serves (cfg, compute, Q): DESIGN.md section 5."""
    pipe_frac = None          # the binding pipe's utilisation by the instructions the kernel really issues
    if compute == "f32":
        if cfg.profile == 1:
            ops = ALG_PLAIN_OPS + ALG_SFU_OPS + (Q - 1) * (ALG_NODE_PLAIN_OPS + ALG_NODE_SFU_OPS)
            ops_how = ("%d algorithmic FP32 lane-ops per point-eval (29 plain + 7 special-function, SURVEY.md 8(d)%s)"
                       % (ops, "" if Q == 1 else "; + 11 + 2 per extra Gauss-Legendre node"))
            pipe_frac = {"pipe": "xu", "ops_per_point_eval": kernel_sfu_ops(cfg.n_T * cfg.n_rho, has_phi, Q),
                         "peak_lanes_per_clk_sm": SFU_LANES_PER_CLK_SM}
        else:
            ops = ALG_OPS_UNIFORM
            ops_how = "%d algorithmic FP32 lane-ops per point-eval (uniform field: the bare cross product)" % ops
        peak = SM_COUNT * ISSUE_LANES_PER_CLK_SM * sm_max_mhz * 1e6
        peak_how = ("derived: 148 SMs x 4 sub-partitions x 32 lanes x %d MHz (FP32 non-tensor issue roofline, the "
                    "north_star denominator; FFMA micro-benchmark measured 123-127 of 128 lanes/clk/SM, "
                    "profiles/r01_pipe_rates.md). Packed FFMA2 does not raise the FMA-pipe rate; XU and ALU-pipe work "
                    "can overlap it, so the binding pipe's own utilisation is given in pipe_frac" % sm_max_mhz)
    else:
        if cfg.profile == 1:
            ops = ALG_F64_OPS_SECH2
            ops_how = ("%d FP64 lane-ops per point-eval counted from the mathematics (29 plain + 55 for the seven "
                       "elementary functions as shortest double-precision sequences, the logarithm at the degree it needs "
                       "far from the axis; DESIGN.md section 5)" % ops)
            if Q == 1:
                pipe_frac = {"pipe": "fp64", "ops_per_point_eval": KERNEL_F64_OPS_SECH2,
                             "peak_lanes_per_clk_sm": FP64_LANES_PER_CLK_SM}
        else:
            ops = ALG_OPS_UNIFORM
            ops_how = "%d algorithmic FP64 lane-ops per point-eval (uniform field)" % ops
        peak = SM_COUNT * FP64_LANES_PER_CLK_SM * sm_max_mhz * 1e6
        peak_how = "derived: 148 SMs x 64 FP64 lanes x %d MHz (DFMA micro-benchmark measured 62-63.8 of 64)" % sm_max_mhz
    return ops, ops_how, peak, peak_how, pipe_frac


def finish_pipe_frac(pipe_frac, evals, k_ms, sm_max_mhz):
    if pipe_frac is None:
        return
    pipe_frac["frac"] = (pipe_frac["ops_per_point_eval"] * evals / (k_ms * 1e-3)) / (
        SM_COUNT * pipe_frac["peak_lanes_per_clk_sm"] * sm_max_mhz * 1e6)
    pipe_frac["note"] = ("instructions the kernel issues on its binding pipe (not an algorithmic count)"
                         + ("; the count of the farthest tier, tier 0 issues 97: a lower bound of the utilisation"
                            if pipe_frac["pipe"] == "fp64" else ""))


def measure_pipe_peaks(api):
    """The three pipe rates the rooflines rest on, measured now on this GPU: wl_pipe_probe (csrc/wl_pipe_probe.cu)
    issues nothing but scalar FFMA / MUFU.EX2 / DFMA; each is timed with CUDA events on the launching stream (2 warm-up,
    5 timed launches of ~17 ms, the median taken) while NVML samples the SM clock."""
    import torch
    sink = torch.zeros(4, dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()
    out = {}
    sampler = ClockSampler(nvml_index_for(torch.cuda.current_device()))
    sampler.start()
    raw = {}
    for pipe, name, iters in ((0, "ffma", 32768), (1, "xu_ex2", 4096), (2, "dfma", 16384)):
        for _ in range(2):
            lane_ops, sms = api.wl_pipe_probe(pipe, iters, sink)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        torch.cuda.synchronize()
        for a, b in ev:
            a.record(stream)
            api.wl_pipe_probe(pipe, iters, sink)
            b.record(stream)
        torch.cuda.synchronize()
        ms = sorted(a.elapsed_time(b) for a, b in ev)[2]
        raw[name] = (lane_ops, sms, ms)
    clocks = sampler.stop()
    mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965
    for name, (lane_ops, sms, ms) in raw.items():
        out[name + "_lanes_per_clk_sm"] = lane_ops / (ms * 1e-3) / (mhz * 1e6) / sms
        out[name + "_Tlane_ops_per_s"] = lane_ops / (ms * 1e-3) / 1e12
    out["sm_mhz"] = mhz
    out["clocks"] = clocks
    out["how"] = ("wl_pipe_probe: 4 CTAs x 256 threads per SM, 16 independent chains x 8 per loop iteration of scalar FFMA / "
                  "MUFU.EX2 / DFMA only; CUDA events, median of 5 launches; lanes per clock and SM at the NVML-sampled SM clock. "
                  "Nominal: 128 / 16 / 64. The roofline denominators stay the derived ones (nominal lanes x max clock), "
                  "which are the larger, i.e. `frac` is not flattered by a low measurement")
    return out


def time_secondary(api, cfg, compute, steps, warmup, sm_max_mhz):
    """One of the other BASELINE.json configs under the same clock as the headline: device-resident loops, wl_eval +
    wl_jackknife_finalize per step, CUDA events on the launching stream around the steps and around k_wilson."""
    import torch
    T, rho, phi = cfg.grids()
    dev = lambda a: torch.tensor(a, dtype=torch.float64, device="cuda") if a is not None else None
    Td, rd, pd = dev(T), dev(rho), dev(phi)
    field = api.wl_field_create(cfg.profile, cfg.params)
    tdt = torch.float32 if cfg.loop_dtype == "f32" else torch.float64
    loops = api.wl_loops_generate(cfg.n_loops, cfg.n_ppl, cfg.seed, tdt)
    ws = api.wl_eval_workspace_bytes(cfg.n_loops, cfg.n_ppl, cfg.n_T, cfg.n_rho, cfg.n_groups, compute)
    workspace = torch.empty(max(ws, 8), dtype=torch.uint8, device="cuda")
    W_mean = torch.empty((cfg.n_T, cfg.n_rho), dtype=torch.float64, device="cuda")
    gs = torch.empty((cfg.n_groups, cfg.n_T, cfg.n_rho), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()

    def step(events=None):
        api.wl_eval(field, loops, Td, rd, pd, n_groups=cfg.n_groups, compute=compute, W_mean=W_mean, group_sums=gs,
                    workspace=workspace, wilson_events=events)
        return api.wl_jackknife_finalize(gs, cfg.n_loops)

    for _ in range(warmup):
        step()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        a.record(stream)
        b.record(stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(nvml_index_for(torch.cuda.current_device()))
    torch.cuda.synchronize()
    sampler.start()
    e0.record(stream)
    for k in range(steps):
        mean, _ = step(ev[k])
    e1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / steps
    k_ms = sum(a.elapsed_time(b) for a, b in ev) / steps
    checksum = float(mean.sum().item())
    ops, _, peak, _, pipe_frac = kernel_roofline(cfg, compute, 1, phi is not None, sm_max_mhz)
    finish_pipe_frac(pipe_frac, cfg.point_evals, k_ms, sm_max_mhz)
    return {"workload": cfg.name, "dtype": compute, "steps": steps, "warmup": warmup,
            "value": cfg.point_evals / (ms * 1e-3), "ms_per_step": ms, "kernel_ms": k_ms,
            "frac": ops * cfg.point_evals / (k_ms * 1e-3) / peak,
            "pipe_frac": ({"pipe": pipe_frac["pipe"], "frac": pipe_frac["frac"]} if pipe_frac else None),
            "clocks": clocks, "checksum_sum_W_mean": checksum,
            "cache": "%.0f MB of loop coordinates per step%s" % (
                loops.numel() * loops.element_size() / 1e6,
                "" if loops.numel() * loops.element_size() > 126e6 else " (smaller than the 126 MB L2: L2-resident between steps)")}


def run_secondary(api, headline_workload, sm_max_mhz):
    """The other configs of BASELINE.json, 2 timed steps each after 1 warm-up step (the FP64 leg of config 4 takes
    ~8 s per step), so that every configuration north_star names is timed by the same run as the headline."""
    import torch
    from paper_1407_7486_b200 import inputs
    out = []
    for number in (4, 5, 2, 1):
        cfg = inputs.config(number)
        for compute in ("f32", "f64"):
            if compute not in cfg.compute and not (number == 1 and compute == "f32"):
                continue
            if number == headline_workload:
                continue
            steps, warmup = (2, 1) if number in (4, 5) else (5, 3)
            try:
                out.append(time_secondary(api, cfg, compute, steps, warmup, sm_max_mhz))
            except Exception as exc:                      # the headline line must still be printed
                out.append({"workload": cfg.name, "dtype": compute, "error": "%s: %s" % (type(exc).__name__, exc)})
            torch.cuda.empty_cache()
    return out


def run_reference(args, cfg):
    """This tier's reference arm: the oracle, as it stands, on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    import numpy as np
    from oracle import wl_oracle as oracle
    cores = affinity_cores()
    n = oracle_sample_loops(cfg, cores, 64)
    T, rho, phi = cfg.grids()
    loops = oracle.generate_loops(cfg.seed, n, cfg.n_ppl)
    if cfg.loop_dtype == "f32":
        loops = loops.astype(np.float32).astype(np.float64)       # the stored coordinates, promoted exactly
    for _ in range(args.warmup):
        time_oracle(cfg, loops, T, rho, phi)
    total_t, total_e, threads = 0.0, 0, 1
    for _ in range(args.steps):
        rate, dt, threads = time_oracle(cfg, loops, T, rho, phi)
        total_t += dt
        total_e += n * cfg.n_ppl * cfg.n_T * cfg.n_rho
    value = total_e / total_t
    sample = "%d whole loops x full %dx%d grid per step (of %d loops)" % (n, cfg.n_T, cfg.n_rho, cfg.n_loops)
    line = base_line(args, cfg, args.gpus)
    line.update({
        "impl": "reference", "value": value, "ms_per_step": 1e3 * total_t / args.steps, "dtype": "f64",
        "config": workload_config(cfg, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "scaling": "weak",
    })
    print(json.dumps(line), flush=True)
    return 0


def run_ours(args, cfg):
    import numpy as np
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    from paper_1407_7486_b200 import api, shard        # raises if libwl.so is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("bench.py --gpus %d must be launched with torch.distributed.run (one rank per GPU)"
                             % args.gpus)
        raise SystemExit("WORLD_SIZE %d != --gpus %d" % (world, args.gpus))
    torch.cuda.set_device(local_rank)
    # under torch.distributed.run the process group is set up even for one rank, so that the collective path
    # (all-gather of the group sums, barriers, MAX over ranks) is the one that runs
    use_dist = world > 1 or "TORCHELASTIC_RUN_ID" in os.environ
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    compute = args.compute or ("f32" if "f32" in cfg.compute else "f64")
    T, rho, phi = cfg.grids()
    dev = lambda a: torch.tensor(a, dtype=torch.float64, device="cuda") if a is not None else None
    Td, rd, pd = dev(T), dev(rho), dev(phi)
    field = api.wl_field_create(cfg.profile, cfg.params)
    sh = shard.shard_groups(cfg.n_loops * world, cfg.n_groups * world, world, rank)
    tdt = torch.float32 if cfg.loop_dtype == "f32" else torch.float64
    seeded = args.loops == "seeded"
    loops = None if seeded else api.wl_loops_generate(sh.n_loops, cfg.n_ppl, cfg.seed, tdt, loop_begin=sh.loop_begin)
    loop_bytes = sh.n_loops * cfg.n_ppl * 2 * (4 if cfg.loop_dtype == "f32" else 8)

    def options():
        if args.quadrature == 1 and not args.shuffle and args.staging == "default" and not seeded and world == 1:
            return None
        return api.wl_eval_options(quadrature_order=args.quadrature, shuffle_seed=(cfg.seed + 1000 if args.shuffle else None),
                                   staging=(1 if args.staging == "bulk" else 0),
                                   seed=(cfg.seed if seeded else None), loop_begin=sh.loop_begin,
                                   ensemble_loops=(sh.n_loops * world if world > 1 else 0))
    ws_bytes = api.wl_eval_opt_workspace_bytes(sh.n_loops, cfg.n_ppl, cfg.n_T, cfg.n_rho, sh.n_groups, compute, options())
    workspace = torch.empty(max(ws_bytes, 8), dtype=torch.uint8, device="cuda")
    W_mean = torch.empty((cfg.n_T, cfg.n_rho), dtype=torch.float64, device="cuda")
    gs_local = torch.empty((sh.n_groups, cfg.n_T, cfg.n_rho), dtype=torch.float64, device="cuda")
    n_loops_total = sh.n_loops * world
    stream = torch.cuda.current_stream()

    def step(events=None):
        if seeded:
            opt = options()
            if events is not None:
                opt.event_wilson_begin, opt.event_wilson_end = (api._event_handle(ev, None) for ev in events)
            api.wl_eval_seeded(field, cfg.seed, sh.n_loops, cfg.n_ppl, Td, rd, pd, n_groups=sh.n_groups, compute=compute,
                               storage=tdt, loop_begin=sh.loop_begin, W_mean=W_mean, group_sums=gs_local,
                               workspace=workspace, options=opt)
        else:
            api.wl_eval(field, loops, Td, rd, pd, n_groups=sh.n_groups, compute=compute, W_mean=W_mean,
                        group_sums=gs_local, workspace=workspace, wilson_events=events, options=options())
        gs = shard.all_gather_group_sums(gs_local, world) if use_dist else gs_local
        return api.wl_jackknife_finalize(gs, n_loops_total)

    def fence():
        torch.cuda.synchronize()
        if use_dist:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    fence()
    k_events = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                for _ in range(args.steps)]
    for a, b in k_events:            # create the cudaEvent_t handles outside the timed region
        a.record(stream)
        b.record(stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(nvml_index_for(local_rank))
    fence()
    sampler.start()
    e0.record(stream)
    for k in range(args.steps):
        mean, err = step(k_events[k])
    e1.record(stream)
    fence()
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)
    wilson_ms = [a.elapsed_time(b) for a, b in k_events]
    if use_dist:
        t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_per_step = ms_total / args.steps
    evals_per_gpu = cfg.point_evals
    value = evals_per_gpu * world / (ms_per_step * 1e-3)
    result_checksum = float(mean.sum().item())
    if not np.isfinite(result_checksum):
        raise SystemExit("bench.py: non-finite <W>")

    # ---- e2e: the C-ABI call on HOST buffers (wl_eval_host), copies inside the timed region ----
    e2e = None
    plain = args.quadrature == 1 and not args.shuffle and args.staging == "default" and not seeded
    if not args.no_e2e and plain:
        host_loops = torch.empty(loops.shape, dtype=loops.dtype, pin_memory=True)
        host_loops.copy_(loops)
        torch.cuda.synchronize()
        hl = host_loops.numpy()
        G_e2e = sh.n_groups
        for _ in range(min(args.warmup, 2)):
            api.wl_eval_host(field, hl, T, rho, phi, n_groups=G_e2e, compute=compute)
        fence()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            hm, he, hg = api.wl_eval_host(field, hl, T, rho, phi, n_groups=G_e2e, compute=compute)
        dt = time.perf_counter() - t0
        if use_dist:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        h2d = hl.nbytes + T.nbytes + rho.nbytes + (phi.nbytes if phi is not None else 0)
        d2h = hm.nbytes + he.nbytes + hg.nbytes
        e2e = {"value": evals_per_gpu * world * args.steps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * dt / args.steps,
               "call": "wl_eval_host (per rank: its own loops; pinned host memory; wall clock, max over ranks)"}
        # one rank: the same units of loops, hence the same bits; several ranks: the device step is cut like the
        # whole ensemble (wl_eval_options.ensemble_loops), the host call like its own loops: equal to rounding
        dm = W_mean.cpu().numpy()
        if not (np.array_equal(hm, dm) if world == 1 else np.allclose(hm, dm, rtol=1e-12, atol=0)):
            raise SystemExit("bench.py: wl_eval_host and wl_eval disagree")
        del host_loops

    if rank != 0:
        if use_dist:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (k_wilson), DESIGN.md section 5 ----
    sm_max_mhz = clocks.get("sm_max_mhz") or 1965
    k_ms = sum(wilson_ms) / len(wilson_ms)
    Q = args.quadrature
    ops, ops_how, peak, peak_how, pipe_frac = kernel_roofline(cfg, compute, Q, phi is not None, sm_max_mhz)
    achieved = ops * evals_per_gpu / (k_ms * 1e-3)
    finish_pipe_frac(pipe_frac, evals_per_gpu, k_ms, sm_max_mhz)
    traffic, traffic_note = ncu_traffic(cfg.name, compute, args)
    roofline = {
        "bound": "alu", "kernel": "k_wilson", "achieved": achieved / 1e12, "peak": peak / 1e12,
        "unit": "Tlane-op/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_note,
        "kernel_ms": k_ms, "kernel_share_of_step": k_ms / ms_per_step,
        "algorithmic_ops": ops_how, "peak_source": peak_how, "pipe_frac": pipe_frac,
        "xu_pipe_frac": pipe_frac["frac"] if (pipe_frac and pipe_frac["pipe"] == "xu") else None,
        "fp64_pipe_frac": pipe_frac["frac"] if (pipe_frac and pipe_frac["pipe"] == "fp64") else None,
        "frac_meaning": ("algorithmic lane-ops per point-eval (a count from the mathematics, not of issued instructions) "
                         "x point-evals/s over the issue peak; the utilisation figure is pipe_frac (instructions the "
                         "kernel issues on its binding pipe over that pipe's rate)"),
        # what the method needs: the ensemble read once + <W> and the group sums written once; the
        # per-unit partial sums (written by k_wilson, read by k_group_reduce) are this design's workspace, stated apart
        "algorithmic_bytes": (0 if seeded else loop_bytes) + 8 * cfg.n_T * cfg.n_rho * (1 + sh.n_groups),
        "workspace_bytes": ws_bytes,
        "traffic_over_algorithmic": (traffic / ((0 if seeded else loop_bytes) + 8 * cfg.n_T * cfg.n_rho * (1 + sh.n_groups))
                                     if traffic else None),
        "hbm_GBps_algorithmic": (0 if seeded else loop_bytes) / (k_ms * 1e-3) / 1e9,
    }

    # ---- cpu_baseline: the oracle as it stands, bounded sample, this box's host cores ----
    cpu_baseline = None
    if not args.no_cpu_baseline:
        cores = affinity_cores()
        n = oracle_sample_loops(cfg, cores, 256)
        sample_loops = (loops[:n] if loops is not None else
                        api.wl_loops_generate(n, cfg.n_ppl, cfg.seed, tdt, loop_begin=sh.loop_begin)).cpu().numpy()
        rate, dt, threads = time_oracle(cfg, sample_loops, T, rho, phi)
        cpu_baseline = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
                        "sample": "first %d whole loops x full %dx%d grid (%.1f s)" % (n, cfg.n_T, cfg.n_rho, dt)}

    launches_per_step = (api.wl_eval_launch_count(sh.n_loops, cfg.n_ppl, cfg.n_T, cfg.n_rho, sh.n_groups, compute) + 1
                         + (1 if args.shuffle else 0))      # + k_jackknife_finalize (+ k_group_permutation)
    if not args.no_pipe_peaks:
        try:
            roofline["peak_measured"] = measure_pipe_peaks(api)
        except Exception as exc:                          # the headline line must still be printed
            roofline["peak_measured"] = {"error": "%s: %s" % (type(exc).__name__, exc)}
    secondary = None
    if plain and world == 1 and not args.no_secondary and args.workload == 3 and cfg.name == "cfg3_paper_scale":
        del loops, workspace
        torch.cuda.empty_cache()
        secondary = run_secondary(api, args.workload, sm_max_mhz)
    line = base_line(args, cfg, world)
    line.update({
        "value": value, "ms_per_step": ms_per_step, "dtype": compute,
        "config": workload_config(cfg, world),
        "options": {"loops": args.loops, "quadrature_order": args.quadrature, "shuffled_groups": bool(args.shuffle),
                    "staging": args.staging},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
        "roofline": roofline, "cpu_baseline": cpu_baseline,
        "checksum_sum_W_mean": result_checksum,
    })
    if secondary is not None:
        line["secondary"] = secondary
    print(json.dumps(line), flush=True)
    if use_dist:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def _code_only(text):
    """C/C++ source without comments and with white space collapsed (string literals in the kernels hold no comment marks)."""
    import re
    text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
    text = re.sub(r"//[^\n]*", " ", text)
    return " ".join(text.split())


def source_sha16():
    """sha256 (first 16 hex digits) of the kernel sources, comments and white space left out: ties an ncu capture to the
    CODE that was profiled (editing a comment does not orphan a capture)."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1407_7486_b200", "csrc")
    files = sorted(f for f in os.listdir(csrc) if f.endswith((".cu", ".cuh"))) if os.path.isdir(csrc) else []
    for f in files:
        with open(os.path.join(csrc, f), "r", encoding="utf-8", errors="replace") as fh:
            h.update(f.encode() + b"\0" + _code_only(fh.read()).encode())
    return h.hexdigest()[:16]


def ncu_traffic(workload, compute, args):
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_wilson launch, from profiles/ncu_traffic.json
    (written by `python bench.py --ncu-summary REPORT --key ...` from an `ncu --set full` capture).  null unless the
    capture was taken on exactly these kernel sources and this (workload, compute, options)."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    try:
        with open(path) as fh:
            tab = json.load(fh)
    except (OSError, ValueError):
        return None, "no profiles/ncu_traffic.json"
    key = "%s/%s" % (workload, compute)
    if args.loops != "stored" or args.quadrature != 1 or args.shuffle or args.staging != "default":
        key += "/loops=%s,Q=%d,shuffle=%d,staging=%s" % (args.loops, args.quadrature, int(args.shuffle), args.staging)
    e = tab.get("entries", {}).get(key)
    if e is None:
        return None, "no ncu capture of %s" % key
    if e.get("source_sha16") != source_sha16():
        return None, "ncu capture of %s is from other kernel sources (%s)" % (key, e.get("source_sha16"))
    return int(e["dram_bytes_read"]) + int(e["dram_bytes_write"]), "profiles/ncu_traffic.json: %s (%s)" % (key, e.get("report"))


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", type=int, default=3, help="BASELINE.json config number (1-5); 3 = paper scale")
    ap.add_argument("--compute", choices=("f32", "f64"), default=None)
    ap.add_argument("--loops", choices=("stored", "seeded"), default="stored",
                    help="seeded: no ensemble buffer, loops regenerated inside k_wilson (wl_eval_seeded)")
    ap.add_argument("--quadrature", type=int, choices=(1, 2, 3), default=1, help="Gauss-Legendre points of eq. (24)")
    ap.add_argument("--shuffle", action="store_true", help="shuffled group assignment per proper time")
    ap.add_argument("--staging", choices=("default", "bulk"), default="default")
    ap.add_argument("--n-loops", type=int, default=None, help="override the workload's loops per GPU (a multiple of its groups)")
    ap.add_argument("--loop-dtype", choices=("f32", "f64"), default=None, help="override the loop storage precision")
    ap.add_argument("--source-sha", action="store_true", help="print the hash of the kernel sources and exit")
    ap.add_argument("--ncu-summary", metavar="REPORT", default=None,
                    help="no benchmark: summarise an `ncu --set full` report of k_wilson as a markdown table and, with --key, "
                         "record its DRAM bytes in profiles/ncu_traffic.json (bench_ncu_summary.py; no GPU needed)")
    ap.add_argument("--key", default=None, help="with --ncu-summary: entry of profiles/ncu_traffic.json, e.g. cfg3_paper_scale/f32")
    ap.add_argument("--sha", default=None, help="with --ncu-summary: source hash at capture time (--source-sha on the GPU box)")
    ap.add_argument("--md", default=None, help="with --ncu-summary: also append the table to this file")
    ap.add_argument("--kernel", default="k_wilson", help="with --ncu-summary: kernel name filter")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--pipe-peaks", action="store_true",
                    help="no benchmark: measure the FFMA / MUFU / DFMA pipe rates with wl_pipe_probe and print them as one JSON line")
    ap.add_argument("--no-pipe-peaks", action="store_true", help="leave roofline.peak_measured out of the line")
    ap.add_argument("--no-secondary", action="store_true",
                    help="skip the `secondary` block (configs 4, 5, 2, 1 timed after the config-3 headline)")
    args = ap.parse_args()
    if args.source_sha:
        print(source_sha16())
        return 0
    if args.ncu_summary:
        import bench_ncu_summary
        argv = [args.ncu_summary, "--kernel", args.kernel]
        for flag, val in (("--key", args.key), ("--sha", args.sha), ("--md", args.md)):
            if val:
                argv += [flag, val]
        return bench_ncu_summary.main(argv)
    if args.pipe_peaks:
        import torch
        if not torch.cuda.is_available():
            raise SystemExit("bench.py --pipe-peaks: no CUDA device")
        from paper_1407_7486_b200 import api
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        print(json.dumps({"pipe_peaks": measure_pipe_peaks(api)}), flush=True)
        return 0
    if args.steps < 1 or args.warmup < 0:
        raise SystemExit("--steps >= 1, --warmup >= 0")
    from paper_1407_7486_b200 import inputs
    cfg = inputs.config(args.workload)
    if args.n_loops is not None or args.loop_dtype is not None:
        import dataclasses
        cfg = dataclasses.replace(cfg, name=cfg.name + "_variant", n_loops=args.n_loops or cfg.n_loops,
                                  loop_dtype=args.loop_dtype or cfg.loop_dtype)
        if cfg.n_loops % cfg.n_groups != 0:
            raise SystemExit("--n-loops must be a multiple of the workload's %d groups" % cfg.n_groups)
    if args.impl == "reference":
        return run_reference(args, cfg)
    return run_ours(args, cfg)


if __name__ == "__main__":
    sys.exit(main())
