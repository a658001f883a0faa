#!/usr/bin/env python
"""bench.py -- throughput of the deflection-map hot path on synthetic cluster catalogues.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--mode fp64|fp32|mixed] [--impl reference]

A "step" is one pass of the whole hot path over one batch: one lt_gradient_grid call (per-lens precompute kernel +
gradient kernel [+ patch / flag / compaction kernels + fp64 recompute for mixed]) on BASELINE.json config 1
(1024 x 1024 pixels over [-100,100]", 1 cluster-scale + 99 galaxy-scale dPIE halos, seed 1001; recipe in DESIGN.md
section 4).  The headline `value` is the fp64 mode (the paper's DP run, Table 2); the same line carries
the fp32 and mixed numbers on the same workload under "modes".

Timing: CUDA events on the launching stream around every step, W >= 3 warm-up steps, L2 flushed (a 256 MiB buffer
is overwritten) between timed steps outside the event pairs, barrier + torch.cuda.synchronize() on both sides of the
timed region, max over ranks.  `value` has the catalogue already resident in HBM; `e2e` goes through
lt_gradient_grid_host with pinned HOST buffers (H2D of the catalogue and D2H of the whole map inside the timed region).

N > 1 (torchrun, one rank per GPU): the path shards with no exchange (pixels and MCMC samples are independent,
P:98): every rank computes the full map of its OWN catalogue (seed + rank) -- weak scaling, no collective
on the data path; NCCL is used only for the barrier and the max over ranks.

--model sie: the same path with the paper's own lens body (Algorithm 1) on a synthetic stand-in for the paper's benchmark
(6730 x 6730 pixels at 0.03", 2 cluster-scale + 700 galaxy-scale SIE halos); `vs_baseline` is then the ratio to
the paper's V100 throughput derived from Table 2 -- another machine's number, context only.

--impl reference: times the CPU oracle (oracle/lt_oracle.cpp, `double` instantiation, as it stands) on the host cores,
each step a bounded row sample of the same workload; rank 0 only.
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

METRIC = "lens_pixel_gradient_evals_per_s"
UNIT = "lens*pixel/s"
MODES = {"fp64": 0, "fp32": 1, "mixed": 2}
DTYPE = {"fp64": "f64", "fp32": "f32", "mixed": "f32+f64"}

# FLOP-count convention per lens-pixel interaction (DESIGN.md section 8 / SURVEY 8(d)): textbook evaluation with
# per-lens constants precomputed, add/sub/mul = 1, FMA = 2: 61 flops + 8 specials (2 sqrt, 2 div, 2 ln, 2 atan2).
F_NOM = 69.0
# SIE (Algorithm 1) under the same convention: translate 2 + rotate 6 + R^2 5 + g 4 (with (1 -+ eps) b0
# precomputed: 2 mul, 2 div by R counted as mul by 1/R) + rotate back 6 + accumulate 2 = 25 flops + 1 rsqrt.
F_NOM_SIE = 26.0
# NFW (eq. 16-20 + the circular formula, same convention): translate 2 + rotate 6 + R^2 5 + x 1 + ln(x/2) 1 + F 4 + bracket
# and scale 3 + eq. 20 8 + rotate back 6 + accumulate 2 = 38 flops + 8 specials (2 sqrt, 3 div, ln, arccosh/arccos, 1/x).
F_NOM_NFW = 46.0
# the paper's own numbers for the SIE benchmark workload (Table 2 P:364-373 -> BASELINE.md, derived throughput on V100)
PAPER_V100_SIE = {"fp64": 6.9e10, "mixed": 8.2e10}
# lanes per SM behind the "alu" peaks (paper's Table 1 convention: 2 ops/cycle x clock x lanes)
LANES = {"fp64": 64, "fp32": 128, "mixed": 64}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel at config 1, from the ncu --set full
# capture summarised in profiles/r01e_ncu_full_summary.md (dPIE kernels at config 1; reads only: the map stays in L2).
NCU_TRAFFIC_BYTES = {"fp64": 30976, "fp32": 35328, "mixed": 3483648}
KERNEL_NAME = {"fp64": "lt_grad_f64_kernel", "fp32": "lt_grad_f32_kernel", "mixed": "lt_grad_list_f64_kernel"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (default 1 = the metric's)")
    ap.add_argument("--mode", default="fp64", choices=list(MODES))
    ap.add_argument("--paper-regime", action="store_true", help="light galaxy halos (DESIGN.md section 4)")
    ap.add_argument("--m-max", type=float, default=0.0,
                    help="mixed mode with a calibrated rule (paper_1902_03252_b200.calibrate): this M_max, "
                         "c28 = (1 - 1/M_max)/2, minimal centre patches; 0 = the paper's constants")
    ap.add_argument("--model", default="dpie", choices=["dpie", "sie", "nfw"],
                    help="dpie: BASELINE.json configs (headline); sie: the paper's Algorithm 1 on its benchmark "
                         "workload, 6730^2 pixels x 702 halos (SURVEY 8(f) NEXT-1); nfw: 2048^2 pixels x 64 "
                         "pseudo-elliptical NFW halos (NEXT-4)")
    ap.add_argument("--no-extras", action="store_true", help="skip the other modes, cpu_baseline and peak probes")
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="target CPU work of the oracle sample")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------ helpers
class ClockSampler:
    """Samples SM clock and clock-event reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.02):
        self.samples, self.reasons, self.power = [], set(), []
        self.period, self.ok, self._stop = period, False, threading.Event()
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv, self.h = nv, nv.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # noqa: BLE001 -- NVML missing is reported, not fatal
            self.err = repr(e)
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksEventReasonHwPowerBrakeSlowdown: "hw_power_brake",
                 nv.nvmlClocksEventReasonApplicationsClocksSetting: "applications_clocks_setting"}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.ok:
            self.t.start()

    def stop(self):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"]}
        self._stop.set()
        self.t.join()
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_min_mhz": s[0] if s else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(s),
                "power_w_max": max(self.power) if self.power else None}


def physical_index(local):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except (ValueError, IndexError):
            return local
    return local


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:  # noqa: BLE001
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ------------------------------------------------------------------------------------------------ reference arm
def oracle_sample(W, cpu_seconds, ns_per_interaction=100.0):
    """Row stride so that the `double` oracle does about `cpu_seconds` of CPU work on this workload."""
    if W.lenses.shape[1] == 5:
        ns_per_interaction = 15.0                 # SIE: one sqrt, two divisions
    if W.lenses.shape[1] == 6:
        ns_per_interaction = 60.0                 # NFW: log, acosh / acos, two sqrt
    total = W.nx * W.ny * len(W.lenses) * ns_per_interaction * 1e-9
    stride = max(1, int(round(total / cpu_seconds)))
    rows = (W.ny + stride - 1) // stride
    return stride, rows


def oracle_module(W):
    if W.lenses.shape[1] == 6:
        from oracle import lt_oracle_nfw as O
    elif W.lenses.shape[1] == 5:
        from oracle import lt_oracle_sie as O
    else:
        from oracle import lt_oracle as O
    return O


def host_cores():
    """Host cores this process may run on.  torch.distributed.run exports OMP_NUM_THREADS=1 to every rank unless the
    caller has set it, which would time the oracle on one core at N > 1 and on all of them at N = 1: the thread count
    is therefore passed to the oracle explicitly."""
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def time_oracle(W, stride, threads=0):
    O = oracle_module(W)
    O.lib()
    threads = threads or host_cores()
    t0 = time.perf_counter()
    O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, precision=O.DOUBLE, n_threads=threads,
                    row_stride=stride)
    dt = time.perf_counter() - t0
    rows = (W.ny + stride - 1) // stride
    return rows * W.nx * len(W.lenses) / dt, dt


def run_reference(args, W):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = host_cores()
    # every step = one bounded sample; the whole run (warmup + steps) is sized to stay within ~2 minutes of wall time
    budget = 100.0 * cores / max(1, args.steps + args.warmup)
    stride, rows = oracle_sample(W, min(args.cpu_seconds, budget))
    for _ in range(args.warmup):
        time_oracle(W, stride)
    t = []
    for _ in range(args.steps):
        v, dt = time_oracle(W, stride)
        t.append(dt)
    ms = 1e3 * sum(t) / len(t)
    units = rows * W.nx * len(W.lenses)
    value = units / (ms * 1e-3)
    sample = "rows 0,%d,2*%d,... (%d of %d rows) of %s, all pixels of each row, `double` instantiation" % (
        stride, stride, rows, W.ny, W.name)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": W.name, "n_lens": int(len(W.lenses)), "nx": W.nx, "ny": W.ny, "seed": W.seed,
                       "mode": "fp64", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ our arm
class Runner:
    """Holds the device buffers of one workload/mode and issues steps through the C ABI (python = marshalling)."""

    def __init__(self, torch, lt, W, mode):
        self.torch, self.lt, self.W, self.mode = torch, lt, W, mode
        self.code = MODES[mode]
        n = len(W.lenses)
        self.sie = W.lenses.shape[1] == 5
        self.nfw = W.lenses.shape[1] == 6
        self.grid = {5: lt.lt_gradient_grid_sie, 6: lt.lt_gradient_grid_nfw}.get(W.lenses.shape[1], lt.lt_gradient_grid)
        self.grid_host = {5: lt.lt_gradient_grid_sie_host, 6: lt.lt_gradient_grid_nfw_host}.get(W.lenses.shape[1],
                                                                                                lt.lt_gradient_grid_host)
        # SIE: the paper's rule at its own pixel size; cluster-scale = b0 >= 1" (its cluster halos: 28.8", 14.1")
        self.mixed = (3.26, 0.0104 / 0.03, 6.0, 0.3, 1.0) if self.sie else None
        if M_MAX > 0:
            self.mixed = (M_MAX, 0.5 * (1.0 - 1.0 / M_MAX), 0.0, 0.0, 1e300)
        self.d_lenses = torch.from_numpy(W.lenses).cuda()
        dt = torch.float32 if mode == "fp32" else torch.float64
        self.out = torch.empty((W.ny, W.nx, 2), dtype=dt, device="cuda")
        self.ws = lt.alloc_workspace(n, W.nx, W.ny, self.code)
        self.h_lenses = torch.from_numpy(W.lenses).pin_memory()
        self.h_out = torch.empty((W.ny, W.nx, 2), dtype=dt).pin_memory()
        self.ws_host = lt.alloc_workspace(n, W.nx, W.ny, self.code, host=True)
        self.units = W.nx * W.ny * n
        self.h2d = self.h_lenses.numel() * 8
        self.f_nom = F_NOM_SIE if self.sie else (F_NOM_NFW if self.nfw else F_NOM)
        self.d2h = self.h_out.numel() * self.h_out.element_size()

    def step(self):
        W = self.W
        self.grid(self.d_lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, self.code, mixed=self.mixed, out=self.out,
                  workspace=self.ws)
        self.launches = self.lt.lt_last_launch_count()      # kernels of ours this step enqueued (memsets not counted)

    def step_host(self):
        W = self.W
        self.grid_host(self.h_lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, self.code, self.h_out, self.ws_host,
                       mixed=self.mixed)


def timed(torch, lt, fn, steps, warmup, flush, barrier):
    """W warm-up steps, then K steps each bracketed by CUDA events on the current stream; L2 flushed between steps
    (outside the event pairs).  A second event pair per step, recorded by the library itself around the dominant
    kernel's launch (lt_set_kernel_events), gives that kernel's duration inside the same timed region.
    Returns (mean step time [ms], mean dominant-kernel time [ms])."""
    for _ in range(warmup):
        fn()
        flush.fill_(1)

    def pairs():
        out = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in out:          # force the lazy cudaEventCreate before the timed region
            a.record()
            b.record()
        return out
    ev, kev = pairs(), pairs()
    torch.cuda.synchronize()
    barrier()
    torch.cuda.synchronize()
    for (a, b), (ka, kb) in zip(ev, kev):
        lt.lt_set_kernel_events(ka, kb)
        a.record()
        fn()
        b.record()
        flush.fill_(1)
    torch.cuda.synchronize()
    barrier()
    torch.cuda.synchronize()
    lt.lt_set_kernel_events(None, None)
    per_step = sorted(a.elapsed_time(b) for a, b in ev)
    timed.last_spread = {"median": per_step[len(per_step) // 2], "best": per_step[0], "worst": per_step[-1]}
    return sum(per_step) / steps, sum(a.elapsed_time(b) for a, b in kev) / steps


def run_ours(args, W):
    import torch
    from paper_1902_03252_b200 import lt
    lt.lib()                                          # raises if the CUDA library is missing: no fallback
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        from paper_1902_03252_b200 import workloads
        W = make_workload(args, seed_offset=rank)                                           # own catalogue per rank

    def barrier():
        if dist is not None:
            dist.barrier()

    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    peaks, peak_src = measured_peaks()
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    sampler = ClockSampler(physical_index(local))

    def measure(mode, steps, warmup, host=False):
        r = Runner(torch, lt, W, mode)
        fn = r.step_host if host else r.step
        ms, ms_kernel = timed(torch, lt, fn, steps, warmup, flush, barrier)
        rc, bad = lt.lt_last_status(r.ws_host if host else r.ws)
        if rc != 0:
            raise RuntimeError("lens parameter domain error at lens %d" % bad)
        r.ms_kernel = ms_kernel
        if dist is not None:
            t = torch.tensor([ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        extra = {}
        if mode == "mixed":
            st = lt.lt_mixed_last_stats(r.ws_host if host else r.ws)
            extra = {"flagged_fraction": st["n_flagged"] / (W.nx * W.ny), "patch_fraction": st["n_patch"] / (W.nx * W.ny),
                     "eq25_fraction": st["n_eq25"] / (W.nx * W.ny), "eq28_fraction": st["n_eq28"] / (W.nx * W.ny)}
        return r, ms, extra

    # ---- headline: the requested mode, device-resident inputs
    sampler.start()
    r, ms, extra = measure(args.mode, args.steps, args.warmup)
    spread = dict(timed.last_spread)             # this rank's timed steps (median and best beside the mean)
    value = world * r.units / (ms * 1e-3)
    # ---- e2e: same metric through the host-buffer entry point
    e2e_steps = max(3, min(args.steps, 50))
    _, ms_e2e, _ = measure(args.mode, e2e_steps, max(3, min(args.warmup, 5)), host=True)
    clocks = sampler.stop()

    ms_kernel_main = r.ms_kernel        # dominant kernel, events recorded by the library inside the timed steps
    sm_max = float(clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0)
    sm_run = float(clocks.get("sm_mhz") or sm_max)        # median SM clock sampled during the timed region

    def traffic(mode):
        # per launch of the dominant kernel, from the ncu --set full captures under profiles/ (None where not captured)
        if args.model == "nfw":
            return None
        if args.model == "sie":
            return 2343424 + 665636608 if mode == "fp64" else None
        return NCU_TRAFFIC_BYTES[mode] if (args.config == 1 and not args.paper_regime) else None

    def executed(mode, ms_k, units):
        """The same launch against the instruction floor of the pipe that bounds it: instructions per interaction counted
        in the SASS of the 4-pixel inner loop (profiles/r01e_ncu_full_summary.md).  fp64 / mixed: FP64-pipe instructions,
        each holding an SMSP's 16-lane FP64 pipe for 2 cycles; fp32: all instructions, one issue slot each."""
        per = {("dpie", "fp64"): 61.75, ("dpie", "mixed"): 61.75, ("dpie", "fp32"): 62.75,
               ("sie", "fp64"): 12.75, ("sie", "mixed"): 12.75, ("sie", "fp32"): None}.get((args.model, mode))
        if per is None:
            return None
        cycles = per * (2.0 if mode != "fp32" else 1.0)
        floor = sms * 4 * sm_max * 1e6 * 32 / cycles                   # interactions per second at 100 % of the pipe
        return {"instructions_per_interaction": per, "pipe": "fp64 (2 cycles per warp instruction)" if mode != "fp32"
                else "issue slots (1 per warp instruction)", "floor_interactions_per_s": floor,
                "frac_of_floor": units / (ms_k * 1e-3) / floor}

    def roofline(mode, ms_k, units, flagged=1.0):
        # mixed: the dominant kernel is the fp64 recompute, which processes the flagged pixels only
        units = units * flagged
        peak = 2.0 * sms * LANES[mode] * sm_max * 1e6 / 1e12
        ach = r.f_nom * units / (ms_k * 1e-3) / 1e12
        return {"bound": "alu", "kernel": KERNEL_NAME[mode], "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                "frac": ach / peak, "frac_at_sampled_clock": ach / (peak * sm_run / sm_max), "traffic": traffic(mode),
                "peak_source": "derived: 2 x %d SMs x %d lanes x %.0f MHz (DESIGN.md section 8); no FP%s vector peak in "
                               "MEASURED_PEAKS.json (%s)" % (sms, LANES[mode], sm_max, "64" if LANES[mode] == 64 else "32",
                                                             peak_src),
                "flops_per_interaction_nominal": r.f_nom, "duration_ms": ms_k,
                "duration_covers": ("fp64 recompute kernel" if mode == "mixed" else
                                    "precompute kernel + grid kernels (programmatic dependent launch: an event between "
                                    "them would serialise them)"),
                "interactions_per_launch": units, "executed": executed(mode, ms_k, units),
                "algorithmic_bytes_per_launch": r.out.numel() * r.out.element_size()}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "ms_per_step_median": spread["median"],
            "ms_per_step_best": spread["best"], "ms_per_step_worst": spread["worst"],
            "higher_is_better": True, "scaling": "weak",
            "vs_baseline": (value / PAPER_V100_SIE[args.mode] if (args.model == "sie" and world == 1 and
                                                                  args.mode in PAPER_V100_SIE) else None),
            "dtype": DTYPE[args.mode], "data": "synthetic",
            "config": {"workload": W.name, "n_lens": int(len(W.lenses)), "nx": W.nx, "ny": W.ny, "seed": W.seed,
                       "mode": args.mode, "mixed_rule": ("paper constants" if M_MAX <= 0 else "calibrated, M_max = %g" % M_MAX),
                       "parallelism": "dp%d (independent catalogues, no exchange)" % world,
                       "l2": "256 MiB buffer overwritten between timed steps", "inputs": "resident in HBM"},
            "clocks": clocks,
            "e2e": {"value": world * r.units / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e,
                    "h2d_bytes_per_step": r.h2d, "d2h_bytes_per_step": r.d2h,
                    "api": "lt_gradient_grid_host: pinned host catalogue read over PCIe by the precompute kernel, map stored into "
                           "pinned host memory over PCIe by the gradient kernels while they compute (no staging copy)"},
            "gpu_launches": r.launches * args.steps, "gpu_launches_per_step": r.launches,
            "roofline": roofline(args.mode, ms_kernel_main, r.units, extra.get("flagged_fraction", 1.0))}
    line.update(extra)

    if not args.no_extras:
        modes = {args.mode: {"value": value, "ms_per_step": ms, **extra}}
        for m in MODES:
            if m == args.mode:
                continue
            rm, ms_m, ex = measure(m, max(3, min(args.steps, 50)), max(3, min(args.warmup, 5)))
            modes[m] = {"value": world * rm.units / (ms_m * 1e-3), "ms_per_step": ms_m, **ex,
                        "kernel_ms": rm.ms_kernel,
                        "roofline_frac_nominal": roofline(m, rm.ms_kernel, rm.units,
                                                          ex.get("flagged_fraction", 1.0))["frac"]}
        line["modes"] = modes
        if rank == 0:
            # the same step replayed from a CUDA graph (what an MCMC loop would do): launch gaps removed
            gs = torch.cuda.Stream()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.stream(gs):
                with torch.cuda.graph(graph, stream=gs):
                    r.grid(r.d_lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, r.code, mixed=r.mixed, out=r.out,
                           workspace=r.ws, stream=gs)
            ts = []
            for it in range(13):
                flush.fill_(1)
                a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                graph.replay()
                b_.record()
                torch.cuda.synchronize()
                if it >= 3:
                    ts.append(a.elapsed_time(b_))
            line["cuda_graph_replay"] = {"ms_per_step": sum(ts) / len(ts), "value": r.units / (sum(ts) / len(ts) * 1e-3)}
        if rank == 0 and args.mode == "fp64":
            # the consumer of the map (section 2.2.2): triangle search for 64 synthetic source points on the
            # fp64 map just computed; memory-bound when the sources are few: 16 B per node read once
            import numpy as np
            rng = np.random.default_rng(W.seed + 77)
            src_all = torch.from_numpy(rng.normal(0.0, 8.0, (64, 2)) + W.lenses[0, :2]).cuda()
            hits = torch.empty((1 << 16, 32), dtype=torch.uint8, device="cuda")
            n_hits = torch.empty(1, dtype=torch.int32, device="cuda")
            line["find_images"] = {}
            for n_src in (4, 64):                 # few sources: bound by reading the map; many: by the source loop
                src = src_all[:n_src].contiguous()
                ts = []
                for it in range(8):
                    flush.fill_(1)
                    a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    lt.lt_find_images(r.out, W.x_min, W.y_min, W.dx, 1.0, src, hits=hits, n_hits=n_hits)
                    b_.record()
                    torch.cuda.synchronize()
                    if it >= 3:
                        ts.append(a.elapsed_time(b_))
                ms_fi = sum(ts) / len(ts)
                gbs = W.nx * W.ny * 16 / (ms_fi * 1e-3) / 1e9
                line["find_images"]["%d_sources" % n_src] = {
                    "ms": ms_fi, "images_found": int(n_hits.item()),
                    "cells_per_s": (W.nx - 1) * (W.ny - 1) / (ms_fi * 1e-3),
                    "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                                 "frac": gbs / peaks.get("hbm_gbs", 6650.0),
                                 "algorithmic_bytes": W.nx * W.ny * 16, "peak_source": peak_src}}
        if rank == 0 and args.mode == "fp64":
            # the other call of the chi^2 algorithm (step 1): the deflection at a short list of observed image
            # positions against the whole catalogue -- one warp per point, precompute kernel included
            import numpy as np
            pts_fn = {5: lt.lt_gradient_points_sie, 6: lt.lt_gradient_points_nfw}.get(W.lenses.shape[1], lt.lt_gradient_points)
            rng = np.random.default_rng(W.seed + 78)
            Ld = torch.from_numpy(W.lenses).cuda()
            line["points"] = {}
            for n_pts in (128, 4096):
                pts = torch.from_numpy(np.stack([rng.uniform(W.x_min, W.x_min + W.dx * (W.nx - 1), n_pts),
                                                 rng.uniform(W.y_min, W.y_min + W.dx * (W.ny - 1), n_pts)], axis=1)).cuda()
                po = torch.empty((n_pts, 2), dtype=torch.float64, device="cuda")
                wsp = lt.alloc_workspace(len(W.lenses), 1, 1, lt.LT_FP64)
                ts = []
                for it in range(13):
                    a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    for _ in range(20):           # back to back: per-call time of a stream of calls
                        pts_fn(Ld, pts, out=po, workspace=wsp)
                    b_.record()
                    torch.cuda.synchronize()
                    if it >= 3:
                        ts.append(a.elapsed_time(b_) / 20)
                us = sum(ts) / len(ts) * 1e3
                line["points"]["%d_points" % n_pts] = {"us": us, "n_lenses": len(W.lenses),
                                                       "value": n_pts * len(W.lenses) / (us * 1e-6), "unit": UNIT}
        if rank == 0 and args.mode == "fp64":
            # one whole chi^2 evaluation (eq. 11) as a user composes it from the library's calls, on one stream
            # with no host round trip.  The "observed" catalogue is synthetic: the images the model itself predicts for 16
            # source points (so chi^2 must come out at the interpolation error of the triangles, ~0).
            src16 = src_all[:16].contiguous()
            h0, n0 = lt.lt_find_images(r.out, W.x_min, W.y_min, W.dx, 1.0, src16)
            rec, _ = lt.hits_to_numpy(h0, n0)
            obs_np = np.stack([rec["x"], rec["y"]], axis=1)
            # keep the images the exact deflection lenses back onto their source (drops the spurious "central images" the
            # triangles around a singular or unresolved lens centre produce)
            back = obs_np - pts_fn(Ld, torch.from_numpy(obs_np).cuda()).cpu().numpy()
            keep = np.hypot(*(back - src16.cpu().numpy()[rec["source"]]).T) < 0.05 * W.dx
            rec, obs_np = rec[keep], obs_np[keep]
            off_np = np.searchsorted(rec["source"], np.arange(17)).astype(np.int32)
            d_obs, d_off = torch.from_numpy(obs_np).cuda(), torch.from_numpy(off_np).cuda()
            d_sig = torch.full((len(obs_np),), 0.5, dtype=torch.float64, device="cuda")
            grid_fn = r.grid
            ws_p = lt.alloc_workspace(len(W.lenses), 1, 1, lt.LT_FP64)

            ws_mixed = lt.alloc_workspace(len(W.lenses), W.nx, W.ny, lt.LT_MIXED)

            def chi2_once(map_mode, ws_map):
                al = pts_fn(Ld, d_obs, workspace=ws_p)
                bary = lt.lt_source_barycentres(d_obs, al, d_off, 1.0)
                gmap = grid_fn(Ld, W.x_min, W.y_min, W.dx, W.nx, W.ny, map_mode, out=r.out, workspace=ws_map)
                lt.lt_find_images(gmap, W.x_min, W.y_min, W.dx, 1.0, bary, hits=hits, n_hits=n_hits)
                return lt.lt_chi2(d_obs, d_sig, d_off, hits, n_hits)

            def chi2_timed(map_mode, ws_map):
                ts = []
                for it in range(8):
                    flush.fill_(1)
                    a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    res, terms = chi2_once(map_mode, ws_map)
                    b_.record()
                    torch.cuda.synchronize()
                    if it >= 3:
                        ts.append(a.elapsed_time(b_))
                return sum(ts) / len(ts), lt.chi2_to_python(res), terms.cpu().numpy()
            # the same evaluation on the mixed-precision map (the paper's proposal: P:330), paper constants
            ms_mx, (c2_mx, n_m_mx, n_u_mx), terms_mx = chi2_timed(lt.LT_MIXED, ws_mixed)
            ms_c2, (c2, n_m, n_u), terms_64 = chi2_timed(lt.LT_FP64, r.ws)
            # sigma * sqrt(term) is the distance between an observed image and its predicted counterpart
            shift = 0.5 * np.nanmax(np.abs(np.sqrt(terms_mx) - np.sqrt(terms_64))) if len(terms_64) else 0.0
            line["chi2_chain"] = {"ms_per_evaluation": ms_c2, "n_systems": 16, "n_images": int(len(obs_np)),
                                  "chi2": c2, "n_matched": n_m, "n_unmatched": n_u, "sigma_arcsec": 0.5,
                                  "mixed_map": {"ms_per_evaluation": ms_mx, "chi2": c2_mx, "n_matched": n_m_mx,
                                                "n_unmatched": n_u_mx,
                                                "max_change_of_image_distance_arcsec": float(shift)},
                                  "calls": "lt_gradient_points -> lt_source_barycentres -> lt_gradient_grid -> "
                                           "lt_find_images -> lt_chi2",
                                  "catalogue": "synthetic: the model's own predicted images of 16 source points that the exact "
                                               "deflection lenses back to within 0.05 pixel of their source"}
        if rank == 0:
            p64, p32 = lt.lt_peak_probe(0, 1 << 15), lt.lt_peak_probe(1, 1 << 16)
            line["peak_probe"] = {"fp64_tflops": p64 / 1e12, "fp32_tflops": p32 / 1e12,
                                  "how": "dependent-free FMA chains, full grid, same process"}
            line["roofline"]["frac_of_probe"] = line["roofline"]["achieved"] / (
                (p64 if LANES[args.mode] == 64 else p32) / 1e12)
        if rank == 0 and world == 1:
            # the cpu_baseline leg: with run_reference the one place bench.py runs the oracle (inside time_oracle)
            stride, rows = oracle_sample(W, args.cpu_seconds)
            v, dt = time_oracle(W, stride)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": host_cores(), "kind": "oracle",
                                    "seconds": dt,
                                    "sample": "rows 0,%d,... (%d of %d rows) of %s, `double` instantiation, "
                                              "OpenMP over rows" % (stride, rows, W.ny, W.name)}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def make_workload(args, seed_offset=0):
    from paper_1902_03252_b200 import workloads
    if args.model == "sie":
        return workloads.make_sie("paper", seed_offset=seed_offset)
    if args.model == "nfw":
        return workloads.make_nfw(n_override=2048, seed_offset=seed_offset)
    return workloads.make(args.config, paper_regime=args.paper_regime, seed_offset=seed_offset)


M_MAX = 0.0


def main():
    global M_MAX
    args = parse_args()
    M_MAX = args.m_max
    if args.warmup < 3:
        args.warmup = 3
    from paper_1902_03252_b200 import workloads
    W = make_workload(args)
    if args.impl == "reference":
        run_reference(args, W)
    else:
        run_ours(args, W)


if __name__ == "__main__":
    main()
