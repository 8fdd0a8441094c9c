#!/usr/bin/env python
"""bench.py -- Triad-ATRG coarse-grain steps/s (FP64) on B200, the metric of BASELINE.json.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c3] [--impl reference]

One "step" = one pass of the whole hot path (canonical form, RSVD bond
swap, RSVD isometries, triad tensors, squeezers, O(r^2 chi^7) contraction, normalisation) on the
steady-state tensor (all legs and the bond = chi) of the named config.  Inputs are synthetic by
construction: the 4D Ising tensor generated from (beta, h) and host-generated seeded Gaussian
sketches.

Printed JSON line (rank 0): value = whole-job steps/s with the step's sketches already resident in
HBM; e2e = the same through the C-ABI with HOST sketch buffers (pinned; H2D inside coarse_grain)
plus the ln Z/V read-back (device reduction + scalar D2H) every step; roofline = the tensor-GEMM
kernel (FP64 DMMA) timed per launch with CUDA events on the library's stream inside the timed
region; cpu_baseline = the CPU oracle on this box's host cores on a bounded sample.

N > 1: the path does not shard (BASELINE.json north_star: one GPU, no collectives) -> N
independent replicas, value = N*K / max-over-ranks time.
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

METRIC = "Triad-ATRG coarse-grain steps/s (FP64)"
UNIT = "steps/s"

# BASELINE.json configs; seed = 20241214 + config index
CONFIGS = {
    "c1": dict(T=6.0, h=0.0, chi=6, r=2, q=2, seed=20241214, ramp=4),
    "c2": dict(T=6.65, h=0.0, chi=16, r=2, q=2, seed=20241215, ramp=8),
    "c3": dict(T=6.65, h=0.0, chi=32, r=2, q=2, seed=20241216, ramp=8),
    "c4": dict(T=6.65, h=0.0, chi=24, r=2, q=2, seed=20241217, ramp=8, atrg=True),   # plain ATRG, O(chi^9)
    "c5": dict(T=6.5, h=0.01, chi=64, r=2, q=3, seed=20241218, ramp=8),
}
# DRAM traffic of one launch of the dominant kernel, from the committed `ncu --set full` capture
# (profiles/r2_gemm_persistent_full.md: dram__bytes_read.sum + dram__bytes_write.sum), next to the
# algorithmic bytes of that launch (each operand read once, the output written once)
NCU_TRAFFIC = {"launch": "a6(ii) P = EM.F at c3: M=65536 N=2048 K=1024", "dram_bytes": 0.724769792e9 + 1.035347e9,
               "algorithmic_bytes": 8.0 * (65536 * 1024 + 1024 * 2048 + 65536 * 2048),
               "source": "profiles/r2_gemm_persistent_full.md"}
# nominal dense peaks of /opt/skills/guides (B200): FP64 tensor 45 TFLOP/s, bf16 2250 TFLOP/s
FP64_OVER_BF16_NOMINAL = 45.0 / 2250.0


def workload_name(name, c):
    return ("%s: 4D Ising T=%.2f h=%g, %s chi=%d r=%d q=%d, steady-state coarse-grain steps "
            "(all legs = chi), directions cycling 1..4" % (name, c["T"], c["h"],
                                                            "plain ATRG (O(chi^9) contraction)" if c.get("atrg") else "Triad-ATRG",
                                                            c["chi"], c["r"], c["q"]))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


# ------------------------------------------------------------------------------ clocks
class ClockSampler:
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return None
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw = [], [], []
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            with open(self.path) as f:
                for line in f:
                    p = [x.strip() for x in line.split(",")]
                    if len(p) < 8:
                        continue
                    try:
                        sm.append(float(p[1]))
                        mx.append(float(p[2]))
                        pw.append(float(p[3]))
                    except ValueError:
                        continue
                    for n, v in zip(names, p[4:8]):
                        if v.lower().startswith("active"):
                            reasons.add(n)
            os.unlink(self.path)
        except Exception:
            return None
        if not sm:
            return None
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------ inputs
def pinned_sketches(tt, cfg, step_index, direction, reuse=None):
    """Host (pinned) seeded Gaussian sketches of one step: {which: torch tensor}; shapes asked from
    the library for the current state (rows, cols per DESIGN.md 'Input recipe').  reuse: buffers of a
    previous call to fill again (large configs)."""
    import torch
    import seeded_inputs as si
    out = {}
    for which in range(0, 5):
        rows, cols = tt.sketch_shape(which, direction, cfg["chi"], cfg["r"])
        if rows * cols == 0:
            continue
        if reuse is not None and which in reuse and reuse[which].numel() == rows * cols:
            t = reuse[which]
        else:
            t = torch.empty(rows * cols, dtype=torch.float64, pin_memory=True)
        si.gauss(si.subseed(cfg["seed"], step_index, which), rows * cols, out=t.numpy())
        out[which] = t
    return out


_REF_CACHE = {}


def gauge_refs(tt, cfg, direction):
    """Step-independent gauge reference matrices (reading G12), device resident.  They depend on
    (seed, which, shape) only, so directions with equal shapes share one tensor."""
    import torch
    import seeded_inputs as si
    out = {}
    for which in range(5, 9):
        rows, cols = tt.sketch_shape(which, direction, cfg["chi"], cfg["r"])
        if rows * cols == 0:
            continue
        key = (cfg["seed"], which, rows, cols)
        if key not in _REF_CACHE:
            _REF_CACHE[key] = torch.from_numpy(si.gauss(si.subseed(cfg["seed"], 0, which), rows * cols)).cuda()
        out[which] = _REF_CACHE[key]
    return out


# ------------------------------------------------------------------------------ reference arm
def oracle_sample(cfg):
    """State of the CPU oracle just before the sample step, and the sample step's arguments.
    Sample = step 4 of the config's schedule (direction 4): legs (chi/2.., chi) -> the first tensor
    with all legs = chi.  A true steady-state oracle step at chi=32 takes ~2 min on 8 cores."""
    from oracle import driver
    from oracle import tatrg_oracle as orc
    st = orc.init_ising_tensor(1.0 / cfg["T"], cfg["h"])
    for m in range(3):
        orc.coarse_grain(st, m + 1, cfg["chi"], cfg["r"], cfg["q"], driver.seeded_inputs_for(cfg["seed"], m),
                         mode="atrg" if cfg.get("atrg") else "triad")
    return st


def oracle_time_one(cfg, st0):
    import copy
    from oracle import driver
    from oracle import tatrg_oracle as orc
    st = copy.deepcopy(st0)
    t0 = time.perf_counter()
    orc.coarse_grain(st, 4, cfg["chi"], cfg["r"], cfg["q"], driver.seeded_inputs_for(cfg["seed"], 3),
                     mode="atrg" if cfg.get("atrg") else "triad")
    dt = time.perf_counter() - t0
    return dt, st


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count()


SAMPLE_TEXT = ("1 oracle coarse_grain call = step 4 of the schedule (direction 4, input legs "
               "(chi/2, chi/2, chi/2, chi) -> first tensor with all legs = chi) after 3 untimed ramp-up steps; "
               "cheaper than a steady-state step (116 s on 8 cores at chi=32), so an upper bound on the "
               "oracle's steady-state steps/s")


def run_reference(args, cfg, name):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy  # noqa: F401  (BLAS threads = all cores)
    st0 = oracle_sample(cfg)
    budget_s = 240.0
    times = []
    t, _ = oracle_time_one(cfg, st0)          # first warm-up doubles as the cost estimate
    warm = 1
    steps = args.steps
    while warm < args.warmup and (warm + 1 + steps) * t < budget_s:
        oracle_time_one(cfg, st0)
        warm += 1
    steps = max(1, min(steps, int(budget_s / t) - warm))
    for _ in range(steps):
        dt, _ = oracle_time_one(cfg, st0)
        times.append(dt)
    total = sum(times)
    val = steps / total
    cores = blas_threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "steps_requested": args.steps, "warmup": warm, "ms_per_step": 1e3 * total / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_name(name, cfg), "sample": SAMPLE_TEXT},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": SAMPLE_TEXT},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------ our arm
def reduce_over_ranks(max_values, sum_values, dist, device):
    """Replicas only: the job's time is the slowest replica's (MAX over ranks),
    counters add up.  dist = torch.distributed or None for a single process."""
    if dist is None:
        return list(max_values), list(sum_values)
    import torch
    t = torch.tensor(list(max_values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([float(v) for v in sum_values], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return [float(x) for x in t], [float(x) for x in u]


def job_value(world, steps, ms):
    """Whole-job steps/s of `world` independent replicas that each did `steps` steps in (max) `ms`."""
    return world * steps / (ms * 1e-3)


SCHEDULE_STEPS = 40   # BASELINE.json: every config is a 40-step schedule (8 for c1), directions cycling 1..4


def timed_segments(ramp, W, K, sched=SCHEDULE_STEPS):
    """The timed steps stay inside the config's schedule (BASELINE.json c3: 'steps 9...40'): after `ramp`
    untimed ramp-up steps and W warm-up steps at most sched - ramp - W steps are timed in one go; a larger
    K is split into segments, each from a fresh init + ramp-up + warm-up.  Returns lists of 0-based step
    indices."""
    room = sched - ramp - W
    if room < 1:
        raise ValueError("warm-up of %d steps leaves no timed step inside the %d-step schedule" % (W, sched))
    segs, left = [], K
    while left > 0:
        n = min(left, room)
        segs.append(list(range(ramp + W, ramp + W + n)))
        left -= n
    return segs


def run_ours(args, cfg, name):
    import torch
    import paper_2412_14104_b200 as tt

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libtatrg has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    chi, r, q, seed = cfg["chi"], cfg["r"], cfg["q"], cfg["seed"]
    K, W, ramp = args.steps, max(args.warmup, 0), cfg["ramp"]
    segs = timed_segments(ramp, W, K, 8 if name == "c1" else SCHEDULE_STEPS)
    tt.set_workspace(chi=chi, r=r, device="cuda:%d" % local, atrg=bool(cfg.get("atrg")))
    step_fn = tt.coarse_grain_atrg if cfg.get("atrg") else tt.coarse_grain
    stream = torch.cuda.Stream()
    tt.set_stream(stream)

    def start():
        """init + untimed ramp-up to the steady state (inputs generated by the library from the seed)."""
        tt.init_ising_tensor(1.0 / cfg["T"], cfg["h"])
        for m in range(ramp):
            step_fn(m % 4 + 1, chi, r, q, seed)
        return tt.get_dims()

    dims = start()
    steady = all(d == chi for d in dims[:5])
    refs = {d: gauge_refs(tt, cfg, d) for d in (1, 2, 3, 4)}

    def set_inputs(sk, d):
        for which, t in sk.items():          # CUDA tensor -> device pointer; pinned CPU tensor -> host pointer
            tt.set_sketch(which, t)
        for which, t in refs[d].items():
            tt.set_sketch(which, t)

    # Host-generated (north star) seeded sketches of every step the two passes run, page-locked.  Large
    # configs (chi = 64: 17 GB of sketch per step): one buffer set, refilled between steps outside the
    # per-step event pairs.
    per_step_bytes = sum(a * b * 8 for a, b in (tt.sketch_shape(w, 1, chi, r) for w in range(5)))
    span = W + max(len(sg) for sg in segs)
    streamed = per_step_bytes * span > (20 << 30)
    hosts = {}
    if streamed:
        host1 = pinned_sketches(tt, cfg, ramp, ramp % 4 + 1)
    else:
        for mm in range(ramp, ramp + span):
            hosts[mm] = pinned_sketches(tt, cfg, mm, mm % 4 + 1)

    # ---- pass 1: the step's sketches resident in HBM before the timed region
    if streamed:
        dev1 = {w: torch.empty_like(t, device="cuda") for w, t in host1.items()}

        def resident(mm):
            pinned_sketches(tt, cfg, mm, mm % 4 + 1, reuse=host1)
            for w, t in host1.items():
                dev1[w].copy_(t)
            torch.cuda.synchronize()
            return dev1
    else:
        dev = {mm: {w: t.cuda() for w, t in sk.items()} for mm, sk in hosts.items()}
        torch.cuda.synchronize()

        def resident(mm):
            return dev[mm]
    vis = os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",")
    sampler = ClockSampler(vis[local] if local < len(vis) and vis[local].strip().isdigit() else local)
    stages = {}
    gprof = {}
    pairs = []
    launches = 0
    flops = 0.0
    first = True
    for sg in segs:
        if not first:
            start()
        for mm in range(ramp, ramp + W):
            set_inputs(resident(mm), mm % 4 + 1)
            step_fn(mm % 4 + 1, chi, r, q, seed)
        tt.set_profile(1)
        tt.launch_count(reset=True)
        tt.gemm_flops(reset=True)
        barrier()
        if first:
            sampler.start()
        if not streamed:
            pairs.append((torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)))
            pairs[-1][0].record(stream)
        for mm in sg:
            d = mm % 4 + 1
            sk = resident(mm)
            if streamed:
                pairs.append((torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)))
                pairs[-1][0].record(stream)
            set_inputs(sk, d)
            step_fn(d, chi, r, q, seed)
            if streamed:
                pairs[-1][1].record(stream)
            for k, v in tt.stage_ms().items():
                stages[k] = stages.get(k, 0.0) + v / K
            for k, v in tt.gemm_profile().items():
                g = gprof.setdefault(k, {"ms": [0.0, 0.0], "flops": [0.0, 0.0], "launches": [0, 0]})
                for j in range(2):
                    g["ms"][j] += v["ms"][j]
                    g["flops"][j] += v["flops"][j]
                    g["launches"][j] += v["launches"][j]
        if not streamed:
            pairs[-1][1].record(stream)
        barrier()
        launches += tt.launch_count(reset=True)
        flops += tt.gemm_flops(reset=True)
        tt.set_profile(False)
        first = False
    clocks = sampler.stop()
    ms = sum(a.elapsed_time(b) for a, b in pairs)
    lnz = tt.log_Z_per_site()
    if streamed:
        del dev1
    else:
        del dev
    torch.cuda.empty_cache()

    # ---- pass 2: the SAME steps end to end through the C-ABI: host (page-locked) sketch buffers, copied
    # host -> device inside coarse_grain on the library's copy stream, + the ln Z/V read-back every step
    h2d = 0
    h2d_ms = 0.0
    pairs2 = []
    for sg in segs:
        start()
        for mm in range(ramp, ramp + W):
            sk = pinned_sketches(tt, cfg, mm, mm % 4 + 1, reuse=host1) if streamed else hosts[mm]
            set_inputs(sk, mm % 4 + 1)
            step_fn(mm % 4 + 1, chi, r, q, seed)
        barrier()
        if not streamed:
            pairs2.append((torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)))
            pairs2[-1][0].record(stream)
        for mm in sg:
            d = mm % 4 + 1
            if streamed:
                sk = pinned_sketches(tt, cfg, mm, d, reuse=host1)
                pairs2.append((torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)))
                pairs2[-1][0].record(stream)
            else:
                sk = hosts[mm]
            set_inputs(sk, d)                             # host pointers: copied inside coarse_grain
            step_fn(d, chi, r, q, seed)
            lnz2 = tt.log_Z_per_site()                    # device dot product + scalar D2H
            if streamed:
                pairs2[-1][1].record(stream)
            t_ms, t_b = tt.h2d()
            h2d += t_b
            h2d_ms += t_ms
        if not streamed:
            pairs2[-1][1].record(stream)
        barrier()
    ms_e2e = sum(a.elapsed_time(b) for a, b in pairs2)
    lnz_match = abs(lnz2 - lnz) <= 1e-12 * abs(lnz)       # both passes ran the same steps on the same inputs

    # ---- max over ranks
    (ms, ms_e2e), (launches,) = reduce_over_ranks([ms, ms_e2e], [launches], dist, "cuda")
    launches = int(launches)

    # ---- roofline of the dominant kernel (tensor-GEMM, 128x128 DMMA tile)
    peaks, how = measured_peaks()
    g_ms = sum(v["ms"][1] for v in gprof.values())
    g_fl = sum(v["flops"][1] for v in gprof.values())
    g_n = sum(v["launches"][1] for v in gprof.values())
    s_ms = sum(v["ms"][0] for v in gprof.values())
    s_fl = sum(v["flops"][0] for v in gprof.values())
    peak_bf16_ratio = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]) * FP64_OVER_BF16_NOMINAL
    achieved = g_fl / (g_ms * 1e-3) / 1e12 if g_ms > 0 else 0.0
    probe = tt.probe_fp64_peak(0, 1 << 14)
    probe_dfma = tt.probe_fp64_peak(1, 1 << 14)
    per_stage = {k: {"gemm_ms_per_step": (v["ms"][0] + v["ms"][1]) / K,
                     "gemm_tflops": ((v["flops"][0] + v["flops"][1]) / ((v["ms"][0] + v["ms"][1]) * 1e-3) / 1e12
                                     if v["ms"][0] + v["ms"][1] > 0 else 0.0),
                     "gemm_launches_per_step": (v["launches"][0] + v["launches"][1]) / K}
                 for k, v in gprof.items()}
    roofline = {"bound": "tensor",
                "kernel": "tgemm_p_kernel<A_KF,B_KF,VEC> (persistent 128x128 CTA tile, FP64 DMMA.8x8x4, gemm_p.cu)",
                "achieved": achieved, "peak": probe, "unit": "TFLOP/s", "frac": achieved / probe if probe > 0 else None,
                "traffic": NCU_TRAFFIC["dram_bytes"],
                "traffic_of": NCU_TRAFFIC,
                "peak_source": ("FP64 tensor-pipe peak measured live on this GPU: register-resident DMMA.8x8x4 loop "
                                "(tatrg_probe_fp64_peak); MEASURED_PEAKS.json has no FP64 figure; nominal 148 SM x 64 FMA/clk x "
                                "2 x 1.965 GHz = 37.2"),
                "peak_from_bf16_ratio": peak_bf16_ratio,
                "peak_from_bf16_ratio_note": ("%s bf16_tflops_sustained x nominal FP64/bf16 ratio 45/2250: the bf16 figure is "
                                              "power-throttled (~1.3 GHz) while FP64 runs at 1965 MHz, so this denominator is "
                                              "below what the FP64 pipe delivers; not used for frac" % how),
                "peak_probe_dfma_tflops": probe_dfma,
                "flops_per_launch": g_fl / g_n if g_n else 0.0, "avg_launch_ms": g_ms / g_n if g_n else 0.0,
                "launches": g_n, "share_of_step_time": g_ms / ms if ms > 0 else None,
                "small_tile_kernel": {"tflops": s_fl / (s_ms * 1e-3) / 1e12 if s_ms > 0 else 0.0,
                                      "share_of_step_time": s_ms / ms if ms > 0 else None},
                "whole_step_gemm_tflops": flops / (ms * 1e-3) / 1e12,
                "note": ("achieved = flop-weighted over ALL launches of the kernel inside the timed steps, as they run there: "
                         "steps (i), (ii) of the contraction and the grouped-leg Gram chains run on 140 of the 148 SMs beside the "
                         "squeezer chains (DESIGN.md section 4), and a third of the launches are one-wave shapes; the same kernel "
                         "alone on the machine: 34.0-35.0 TFLOP/s on the hot shapes (profiles/r2_gemm_persistent_full.md)")}

    line = None
    if rank == 0:
        timed = ", ".join("%d..%d" % (sg[0] + 1, sg[-1] + 1) for sg in segs)
        line = {"metric": METRIC, "value": job_value(world, K, ms), "unit": UNIT, "n_gpus": world, "steps": K,
                "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload_name(name, cfg), "chi": chi, "r": r, "q": q,
                           "steady_state": steady, "dims": list(dims[:5]),
                           "timed_steps": "steps %s of the config's schedule (1-based), after %d ramp-up + %d warm-up "
                                          "steps; both passes time the same steps" % (timed, ramp, W),
                           "l2": "inputs larger than L2 (Phi, Psi, A, D, X, Y are %.0f MB each)" % (8e-6 * chi ** 5),
                           "timed_region": ("per-step event pairs summed, sketch refilled between steps"
                                            if streamed else "one event pair around the timed steps of a segment"),
                           "parallelism": "replicas only" if world > 1 else "1 GPU"},
                "e2e": {"value": job_value(world, K, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": h2d // K,
                        "d2h_bytes_per_step": 8, "steps": K, "ms_per_step": ms_e2e / K,
                        "h2d_ms_per_step": h2d_ms / K,
                        "h2d_note": "copy-stream time of the step's uploads; they run beside the canonical form and the "
                                    "basis factorisations of the bond swap",
                        "ln_Z_equal_to_resident_pass": bool(lnz_match)},
                "gpu_launches": launches, "clocks": clocks, "roofline": roofline,
                "stages_ms_per_step": stages, "stages_gemm": per_stage, "ln_Z_per_site": lnz}
    return line


# ------------------------------------------------------------------------------ kernel micro-benchmark
GEMM_SHAPES = {   # the c3 (chi=32, r=2) contraction shapes of SURVEY.md 8(a), plain row-major operands
    "a6_i_EM=E.M4": (65536, 1024, 32),
    "a6_ii_P=EM.F": (65536, 2048, 1024),
    "a6_iv_Phi=P.Q": (32768, 1024, 4096),
    "a2_G1_Z=D.w": (1024, 2048, 32768),
    "a2_G2_Y=A.Z": (32768, 2048, 1024),
    # the isometry operator S = K K_w^T applied to a 64-column block (a3; the 128 x 64 CTA tile of gemm_big.cu)
    "a3_iso_t=K.w": (32768, 64, 1024),
    "a3_iso_y=Kt.t": (1024, 64, 32768),
    # Q1 = T L^-T of the bond swap's Cholesky-QR (a2): B upper triangular, the k tiles of zeros skipped (tri_b)
    "a2_Q1=T.LinvT_tri": (32768, 1024, 1024),
}


def run_gemm_micro(args):
    """Stand-alone timing of the tensor-GEMM kernel on the named shapes (CUDA events on the library's
    stream, operands larger than L2 in total, 3 warm-up + 10 timed launches each)."""
    import torch
    import paper_2412_14104_b200 as tt
    torch.cuda.set_device(0)
    tt.set_workspace(nbytes=1 << 30)
    stream = torch.cuda.Stream()
    tt.set_stream(stream)
    if args.tma:
        tt.set_routes(tt.ROUTE_TMA_PRODUCER)
    out = {"producer": "tma" if args.tma else "cp.async"}
    for name, (M, N, K) in GEMM_SHAPES.items():
        if args.gemm != "all" and args.gemm != name:
            continue
        with torch.cuda.stream(stream):
            A = torch.randn(M, K, dtype=torch.float64, device="cuda")
            B = torch.randn(K, N, dtype=torch.float64, device="cuda")
            C = torch.empty(M, N, dtype=torch.float64, device="cuda")
            tri = name.endswith("_tri")
            if tri:
                B = torch.triu(B).contiguous()
        maps = dict(am=[(M, K)], ak=[(K, 1)], bk=[(K, N)], bn=[(N, 1)], cm=[(M, N)], cn=[(N, 1)])
        for _ in range(3):
            tt.tensor_gemm(A, B, C, M, N, K, maps, tri_b=tri)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 10
        e0.record(stream)
        for _ in range(reps):
            tt.tensor_gemm(A, B, C, M, N, K, maps, tri_b=tri)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        flops = 2.0 * M * (N * (N + 1) // 2 if tri else N * K)   # tri (K = N): the non-zero part of B only
        out[name] = {"M": M, "N": N, "K": K, "ms": ms, "tflops": flops / (ms * 1e-3) / 1e12}
        del A, B, C
    out["probe_dmma_tflops"] = tt.probe_fp64_peak(0, 1 << 14)
    print(json.dumps({"gemm_micro": out}), flush=True)


def run_split_two_gpus(args, cfg, name):
    """--split under torchrun with exactly two processes: the real thing, one GPU each, the halves exchanged over
    NCCL every step (enable_phi_psi_split).  One step of the pair = one coarse-graining step, so the value is
    steps/s of the PAIR (strong scaling of one lattice, not replicas).  Not run in this project's environment
    (one GPU per box): the single-process emulation below is what was measured."""
    import torch
    import torch.distributed as dist
    import paper_2412_14104_b200 as tt
    rank, local = int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))
    if int(os.environ["WORLD_SIZE"]) != 2:
        raise RuntimeError("--split needs exactly two processes (torchrun --nproc-per-node 2)")
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    chi, r, q, seed = cfg["chi"], cfg["r"], cfg["q"], cfg["seed"]
    K, W, ramp = args.steps, max(args.warmup, 0), cfg["ramp"]
    tt.set_workspace(chi=chi, r=r, device="cuda:%d" % local, atrg=bool(cfg.get("atrg")))
    step_fn = tt.coarse_grain_atrg if cfg.get("atrg") else tt.coarse_grain
    stream = torch.cuda.Stream()
    tt.set_stream(stream)
    tt.enable_phi_psi_split()
    try:
        tt.init_ising_tensor(1.0 / cfg["T"], cfg["h"])
        with torch.cuda.stream(stream):
            for m in range(ramp + W):
                step_fn(m % 4 + 1, chi, r, q, seed)
            dist.barrier()
            torch.cuda.synchronize()
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record(stream)
            for m in range(ramp + W, ramp + W + K):
                step_fn(m % 4 + 1, chi, r, q, seed)
            t1.record(stream)
            dist.barrier()
            torch.cuda.synchronize()
        (ms,), _ = reduce_over_ranks([t0.elapsed_time(t1)], [0], dist, "cuda")
        lnz = tt.log_Z_per_site()
    finally:
        tt.disable_phi_psi_split()
    if rank == 0:
        print(json.dumps({"mode": "Phi / Psi split over two GPUs (NCCL exchange every step)", "metric": METRIC,
                          "value": K / (ms * 1e-3), "unit": UNIT, "n_gpus": 2, "steps": K, "warmup": W,
                          "ms_per_step": ms / K, "scaling": "strong", "dtype": "f64", "data": "synthetic",
                          "config": {"workload": workload_name(name, cfg)}, "ln_Z_per_site": lnz}), flush=True)
    dist.destroy_process_group()


def run_split_emulation(args, cfg, name):
    """--split: what each of the two processes of the Phi / Psi split (tatrg_set_side_split; PAPER.md:167 'two GPUs
    are used') does per step, timed on ONE GPU by playing them one after the other: the whole
    step, then rank 1 (Psi only), then rank 0 (Phi only), the same steady-state steps each; the exchange is a device
    copy of the other half (same bytes as the NVLink transfer it stands for, which is NOT measured here).  Not the
    headline metric: prints a line of its own."""
    import torch
    import paper_2412_14104_b200 as tt
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libtatrg has no CPU fallback")
    chi, r, q, seed = cfg["chi"], cfg["r"], cfg["q"], cfg["seed"]
    K, W, ramp = args.steps, max(args.warmup, 0), cfg["ramp"]
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        return run_split_two_gpus(args, cfg, name)
    tt.set_workspace(chi=chi, r=r, atrg=bool(cfg.get("atrg")))
    step_fn = tt.coarse_grain_atrg if cfg.get("atrg") else tt.coarse_grain
    stream = torch.cuda.Stream()
    tt.set_stream(stream)
    at = {"m": 0}

    def one_pass(sides, exchange):
        tt.set_side_split(sides, exchange)
        try:
            tt.init_ising_tensor(1.0 / cfg["T"], cfg["h"])
            pairs, lnz = [], []
            for m in range(ramp + W + K):
                at["m"] = m
                ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                ev[0].record(stream)
                step_fn(m % 4 + 1, chi, r, q, seed)
                ev[1].record(stream)
                if m >= ramp + W:
                    pairs.append(ev)
                lnz.append(tt.log_Z_per_site())
            torch.cuda.synchronize()
            return sum(a.elapsed_time(b) for a, b in pairs) / K, lnz
        finally:
            tt.set_side_split(3)

    whole_phi, sent = [], []
    ms_whole, lnz_whole = one_pass(3, lambda phi, psi: whole_phi.append(phi.clone()))

    def exchange_rank1(phi, psi):
        sent.append(psi.clone())
        phi.copy_(whole_phi[at["m"]])

    ms_r1, _ = one_pass(2, exchange_rank1)
    ms_r0, lnz_r0 = one_pass(1, lambda phi, psi: psi.copy_(sent[at["m"]]))
    half_bytes = int(whole_phi[-1].numel()) * 8
    print(json.dumps({"mode": "Phi / Psi split over two GPUs, the two processes played one after the other on one GPU",
                      "config": {"workload": workload_name(name, cfg), "steps": K, "warmup": W, "ramp": ramp},
                      "whole_ms_per_step": ms_whole, "rank0_ms_per_step": ms_r0, "rank1_ms_per_step": ms_r1,
                      "split_ms_per_step_without_link": max(ms_r0, ms_r1),
                      "exchange": "device copy of the other half inside the step; over NVLink each process sends and "
                                  "receives %d bytes per step (not measured: one GPU)" % half_bytes,
                      "ln_Z_rank0_vs_whole_max_rel": max(abs(a / b - 1) for a, b in zip(lnz_r0, lnz_whole))}),
          flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c3", choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--gemm", default=None, help="kernel micro-benchmark: 'all' or one of " + ", ".join(GEMM_SHAPES))
    ap.add_argument("--tma", action="store_true", help="with --gemm: feed the persistent tile from TMA instead of cp.async")
    ap.add_argument("--chi", type=int, default=None, help="override the bond dimension of the chosen config (scaling study)")
    ap.add_argument("--r", type=int, default=None, help="override the oversampling parameter r (the paper's figures use r = 7)")
    ap.add_argument("--split", action="store_true", help="time the two halves of the two-GPU Phi / Psi split one after the other on one GPU")
    args = ap.parse_args()
    if args.gemm:
        run_gemm_micro(args)
        return
    cfg = dict(CONFIGS[args.config])
    if args.chi:
        cfg["chi"] = args.chi
    if args.r:
        cfg["r"] = args.r
    if args.impl == "reference":
        run_reference(args, cfg, args.config)
        return
    if args.split:
        run_split_emulation(args, cfg, args.config)
        return
    line = run_ours(args, cfg, args.config)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            st0 = oracle_sample(cfg)
            dt, _ = oracle_time_one(cfg, st0)
            line["cpu_baseline"] = {"value": 1.0 / dt, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                                    "sample": SAMPLE_TEXT, "seconds": dt}
        else:
            line["cpu_baseline"] = None
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
