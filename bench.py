#!/usr/bin/env python
"""bench.py -- throughput of the CSPH-TVD step (BASELINE.json metric) on N B200s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cspt|reference]
                    [--workload turbulence|sedov|well|disk|sod] [--n SIZE] [--dtype f64|f32]

A "step" is one pass of the whole hot path over the grid: CFL time step (device
resident), ghost fill, Lagrangian predictor/corrector, Eulerian flux + update
(`cspt_step_cfl`).  The default workload is BASELINE.json configs[3], the 512^3 fp64
smooth periodic field the north_star target is quoted on.  Prints ONE JSON line
(rank 0).  N > 1: the path does not shard (north_star: one GPU, no collectives;
DESIGN.md section 8) so N independent replicas run, one per GPU ("replicas only").

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of
the same workload on the host cores; it is the only leg besides `cpu_baseline` that
executes oracle/.
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

METRIC = "Mcell-updates/s per CSPH-TVD step"
UNIT = "Mcell-updates/s"
# SURVEY.md 8(d) / DESIGN.md section 7: minimum HBM traffic of one cell-update = read
# 5 conserved fields + psi, write 5 conserved fields = 11 words.
MIN_WORDS_PER_CELL = 11

# Algorithmic words per cell of each kernel of the step ("kernels"):
# the fields a kernel must read once and write once, nothing for stencil re-reads.
KERNEL_WORDS = {
    "predictor": 5 + 3 + 8,        # fused primitives + predictor: U^n, f -> star group (phi*, u*, eta*, E*)
    "corrector": 8 + 5 + 3 + 7,    # star group, U^n, f -> U~, xi
    "euler": 5 + 4 + 3 + 5,        # U^n, U~, xi -> U^{n+1}
    "speed_max": 5,
}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cspt", choices=["cspt", "reference"])
    ap.add_argument("--workload", default="turbulence")
    ap.add_argument("--n", type=int, default=None, help="grid size override (default: the config's)")
    ap.add_argument("--dtype", default=None, choices=["f64", "f32"])
    ap.add_argument("--limiter", default="minmod", choices=["minmod", "vanleer"],
                    help="TVD slope limiter of the Euler stage (default: the reading the metric is quoted on)")
    ap.add_argument("--kernel", default="cubic", choices=["cubic", "poly5"],
                    help="smoothing kernel W of Eq. (7) (default: the reading the metric is quoted on)")
    ap.add_argument("--riemann", default="hll", choices=["hll", "lf", "hllc"],
                    help="Riemann solver of the Euler stage (default: the reading the metric is quoted on)")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default; north_star has no domain decomposition) or ONE grid cut "
                         "into z slabs over the ranks (SURVEY 8(f) NEXT-2, strong scaling)")
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--no-tile-skip", action="store_true",
                    help="fp32 gas-vacuum workloads: switch the CTA-level vacuum shortcut off (cspt_debug_tile_skip(0)), for A/B runs")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config throughput table")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def peaks():
    """Measured roofline denominators (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


# ---------------------------------------------------------------------------------------
# clocks: NVML samples DURING the timed region
# ---------------------------------------------------------------------------------------
_REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
            0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}


class ClockSampler:
    def __init__(self, device_index):
        self.samples, self.mask, self.ok = [], 0, False
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            h = None
            try:
                uuid = str(torch.cuda.get_device_properties(device_index).uuid)
                if not uuid.startswith("GPU-"):
                    uuid = "GPU-" + uuid
                h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if hasattr(uuid, "encode") else uuid)
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES")
                idx = device_index
                if vis:
                    try:
                        idx = int(vis.split(",")[device_index])
                    except Exception:
                        idx = device_index
                h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.h = h
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # no NVML: report that, never fake a clock
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    self.mask |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        if self.ok:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "samples": len(s),
                "reasons": [name for bit, name in sorted(_REASONS.items()) if self.mask & bit]}


# ---------------------------------------------------------------------------------------
# workload
# ---------------------------------------------------------------------------------------
def make_workload(args):
    from paper_1912_04855_b200 import workloads as wl
    w = wl.by_name(args.workload, n=args.n, dtype=args.dtype)
    return w


def config_of(w, world):
    esz = 8 if w.dtype == "f64" else 4
    name = "%s %dx%dx%d %s" % (w.name, w.nx, w.ny, w.nz, w.dtype)
    if w.name == "turbulence" and w.nx == 512:
        name += " (BASELINE.json configs[3])"
    big = 5 * w.cells * esz > 4 * 126e6
    return {"workload": name, "cfl": w.cfl, "gamma": w.gamma, "bc": list(w.bc),
            "parallelism": "replicas only" if world > 1 else "1 gpu",
            "l2": ("state (%.1f GiB) larger than L2, no flush needed" % (5 * w.cells * esz / 2 ** 30)) if big
            else "state fits L2: measures launch latency / L2, not HBM"}


def host_fields(w, pin):
    """The six input fields as (pinned) host tensors, generated slab by slab on a few threads."""
    import numpy as np
    import torch
    from concurrent.futures import ThreadPoolExecutor
    tdt = torch.float64 if w.dtype == "f64" else torch.float32
    out = [torch.empty((w.nz, w.ny, w.nx), dtype=tdt) for _ in range(6)]
    if pin:
        out = [t.pin_memory() for t in out]
    views = [t.numpy() for t in out]
    slab = max(1, min(w.nz, (1 << 22) // max(1, w.nx * w.ny)))

    def fill(k0):
        k1 = min(w.nz, k0 + slab)
        f = w.fields_slab(k0, k1)
        for v, a in zip(views, f):
            v[k0:k1] = a

    with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
        list(ex.map(fill, range(0, w.nz, slab)))
    return out


# ---------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline and --impl reference)
# ---------------------------------------------------------------------------------------
def oracle_sample(args, w_full, steps, warmup, n_sample):
    """Times `steps` oracle steps (compute_dt + step) on an n_sample^3 instance of the
    workload, all host cores (bit-identical for any thread count).  Returns per-step seconds."""
    from oracle import csph_oracle as orc
    from paper_1912_04855_b200 import workloads as wl
    cores = os.cpu_count() or 1
    try:
        cores = len(os.sched_getaffinity(0))
    except Exception:
        pass
    orc.build()
    orc.set_threads(cores)
    w = wl.by_name(args.workload, n=n_sample, dtype=w_full.dtype)
    o = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, orc.F64 if w.dtype == "f64" else orc.F32)
    o.set_state(*w.fields())
    for _ in range(warmup):
        o.step(o.compute_dt(w.cfl))
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        o.step(o.compute_dt(w.cfl))
        times.append(time.perf_counter() - t0)
    o.close()
    return w, times, cores


def cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w_full = make_workload(args)
    # bounded sample: a 96^3 instance (64^3 for long runs) so the whole run ends within minutes
    n_s = min(96 if (args.steps + args.warmup) <= 60 else 64, max(w_full.nx, w_full.ny, w_full.nz))
    if args.workload == "sod":
        n_s = None
    w, times, cores = oracle_sample(args, w_full, args.steps, args.warmup, n_s)
    tot = sum(times)
    val = w.cells * len(times) / tot / 1e6
    sample = ("each step = one oracle step (compute_dt + step) on a %dx%dx%d instance of the workload (%s), %d threads"
              % (w.nx, w.ny, w.nz, w.dtype, cores))
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": w.dtype, "data": "synthetic",
        "config": dict(config_of(w, max(1, args.gpus)), sample_of=config_of(w_full, 1)["workload"],
                       note="the oracle is timed on this bounded instance of the workload named in sample_of"),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------
# N > 1: "replicas only" -- no data-path collective, only the timing reduction
# ---------------------------------------------------------------------------------------
def max_over_ranks(ms, world, device):
    """Device time of the slowest rank (all ranks get it)."""
    if world == 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(cells_per_rank, steps, world, tmax_ms):
    """Whole-job Mcell-updates/s: the cells all ranks advanced, over the slowest rank's time."""
    return world * cells_per_rank * steps / (tmax_ms * 1e-3) / 1e6


# ---------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------
def sources_sha():
    """Hash of the CUDA sources: a stored ncu traffic figure is only quoted for the build it was captured on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1912_04855_b200", "csrc")
    for fn in sorted(os.listdir(d)):
        if fn.endswith((".cu", ".cuh")):
            with open(os.path.join(d, fn), "rb") as fh:
                h.update(fh.read())
    return h.hexdigest()[:16]


def stored_traffic(w, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture of THIS build, else None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            d = json.load(fh)
        e = d.get("%s %dx%dx%d %s" % (w.name, w.nx, w.ny, w.nz, w.dtype))
        if e and e.get("sources_sha") == sources_sha():
            return e.get(kernel), e.get("source"), (e.get("ncu") or {}).get(kernel)
    except Exception:
        pass
    return None, None, None


def device_fields(w, device):
    """The six input fields as device tensors, generated slab by slab (no full-size host copy)."""
    import numpy as np
    import torch
    from concurrent.futures import ThreadPoolExecutor
    tdt = torch.float64 if w.dtype == "f64" else torch.float32
    out = [torch.empty((w.nz, w.ny, w.nx), dtype=tdt, device=device) for _ in range(6)]
    slab = max(1, min(w.nz, (1 << 23) // max(1, w.nx * w.ny)))
    starts = list(range(0, w.nz, slab))
    with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
        for k0, f in zip(starts, ex.map(lambda k0: w.fields_slab(k0, min(w.nz, k0 + slab)), starts)):
            for t, a in zip(out, f):
                t[k0:k0 + a.shape[0]].copy_(torch.from_numpy(np.array(a)))
    return out


def time_steps(s, cfl, steps, graph=True):
    """Device milliseconds of `steps` CFL-limited steps (events on the solver's stream)."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(s.stream)
    if graph:
        s.run_cfl(cfl, steps)
    else:
        for _ in range(steps):
            s.step_cfl(cfl)
    e1.record(s.stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


# the five BASELINE.json configs (and cfg4 in fp32): (workload name, dtype override, timed steps)
CONFIG_RUNS = [("sod", None, 400), ("sedov", None, 100), ("well", None, 10), ("turbulence", "f32", 10), ("disk", None, 5)]


def run_configs(cspt, peak, headline):
    """Throughput on every BASELINE.json config at full size (north_star: "reported at 1 GPU"), a few steps each,
    inputs generated on the device slab by slab.  The headline workload's own entry is the timed region's."""
    import torch
    from paper_1912_04855_b200 import workloads as wl
    dev = torch.device("cuda", torch.cuda.current_device())
    out = [headline]
    for name, dt, steps in CONFIG_RUNS:
        w = wl.by_name(name, dtype=dt)
        esz = 8 if w.dtype == "f64" else 4
        entry = {"workload": "%s %dx%dx%d %s" % (w.name, w.nx, w.ny, w.nz, w.dtype), "steps": steps}
        try:
            torch.cuda.empty_cache()
            need = cspt.lib().cspt_workspace_bytes(w.nx, w.ny, w.nz, cspt.F64 if w.dtype == "f64" else cspt.F32) + 6 * w.cells * esz
            free, _ = torch.cuda.mem_get_info()
            if need > 0.97 * free:
                entry["skipped"] = "needs %.0f GiB of device memory, %.0f free" % (need / 2 ** 30, free / 2 ** 30)
                out.append(entry)
                continue
            s = cspt.Solver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, cspt.F64 if w.dtype == "f64" else cspt.F32)
            f = device_fields(w, dev)
            s.set_state(*f)
            del f
            torch.cuda.empty_cache()
            for _ in range(3):
                s.step_cfl(w.cfl)
            ms = time_steps(s, w.cfl, steps, graph=True) / steps
            entry.update({"ms_per_step": ms, "value": w.cells / (ms * 1e-3) / 1e6, "unit": UNIT,
                          "frac_of_measured_hbm": MIN_WORDS_PER_CELL * esz * w.cells / (ms * 1e-3) / 1e9 / peak,
                          "api": "cspt_run_cfl (CUDA graph of two steps)"})
            if w.cells < 4e6:            # launch-bound sizes: the same steps launched one by one, for comparison
                entry["ms_per_step_step_cfl_loop"] = time_steps(s, w.cfl, steps, graph=False) / steps
                entry["note"] = "state fits L2: measures launch latency / L2, not HBM"
            rho = s.get_conserved()[0]
            entry["finite"] = bool(torch.isfinite(rho).all())
            del rho
            s.close()
        except Exception as e:       # one config failing must not lose the headline line
            entry["error"] = repr(e)[:200]
        out.append(entry)
    return out


# algorithmic work of the corrector's neighbour sum, per neighbour [3 sub, 3 FMA for r^2, 1 rsqrt,
# 5 for the spline, 1 mul, 3 FMA, 3 add, 3 FMA, 1 FMA] = 23 FP instructions (FMA counted once), 26 neighbours,
# + about 40 for Eq. (6); in flops (FMA = 2): 3 + 6 + 1 + 5 + 1 + 6 + 3 + 6 + 2 = 33 per neighbour, + 60.  The implementation evaluates pairs once and
# executes FEWER instructions than this list; the roofline fraction is quoted on the list, not on what was executed.
ALGO_INSTR = {"corrector": 26 * 23 + 40}
ALGO_FLOPS = {"corrector": 26 * 33 + 60}


def run_cspt(args):
    import torch
    import torch.distributed as dist
    from paper_1912_04855_b200 import build, cspt

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CSPH-TVD path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    cspt.lib()

    w = make_workload(args)
    esz = 8 if w.dtype == "f64" else 4
    dtype = cspt.F64 if w.dtype == "f64" else cspt.F32
    fields = host_fields(w, pin=True)
    s = cspt.Solver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, dtype)
    if args.kernel == "poly5":
        s.set_kernel(cspt.KERNEL_POLY5)
    if args.no_tile_skip:
        s.debug_tile_skip(0)
    s.set_state_host(*fields)
    s.set_limiter(cspt.LIMITER_VANLEER if args.limiter == "vanleer" else cspt.LIMITER_MINMOD)
    s.set_riemann({"hll": cspt.RIEMANN_HLL, "lf": cspt.RIEMANN_LF, "hllc": cspt.RIEMANN_HLLC}[args.riemann])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        s.step_cfl(w.cfl)
    s.run_cfl(w.cfl, 2)                  # graph capture outside the timed region
    barrier()
    # FMA probe of the plain FP pipe, run for >= 80 ms with the SM clock sampled DURING it, so that its rate can be
    # quoted per clock and SM; it is a CHECK beside the architectural peak the roofline is quoted on, not the peak
    sm_count = s.sm_count()
    probe_sampler = ClockSampler(local)
    probe_sampler.start()
    try:
        fma_rate = s.probe_fma_rate(0, min_ms=80.0)
        probe_err = None
    except cspt.CsptError as e:          # never lose the bench line to the probe
        fma_rate, probe_err = None, repr(e)
    probe_clocks = probe_sampler.stop()
    issue_probe, fma_rate3 = {}, None
    if fma_rate:
        issue_probe = {str(k): s.probe_fma_rate(k, min_ms=10.0) for k in (1, 2, 4, 8)}
        fma_rate3 = s.probe_fma_rate(-1, min_ms=10.0)   # FMAs with three distinct register operands (register-file bound in fp64)
    barrier()

    # ---- timed region: exactly K steps (cspt_run_cfl), device time from CUDA events on the launching stream,
    # no per-kernel event pairs inside
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.launch_count()
    sampler.start()
    e0.record(s.stream)
    s.run_cfl(w.cfl, args.steps)
    e1.record(s.stream)
    barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    launches = s.launch_count() - l0
    tmax = max_over_ranks(ms, world, "cuda")
    value = job_value(w.cells, args.steps, world, tmax)

    # ---- the same K steps once more with an event pair around every launch: per-kernel times for the roofline
    prof_sampler = ClockSampler(local)
    prof_sampler.start()
    s.profile_enable(True)
    for _ in range(args.steps):
        s.step_cfl(w.cfl)
    prof = s.profile_read()
    s.profile_enable(False)
    barrier()
    prof_clocks = prof_sampler.stop()

    # the state must still be sane (a blown-up run would time NaN arithmetic)
    rho = s.get_conserved()[0]
    assert bool(torch.isfinite(rho).all()), "state is not finite after the timed steps"
    del rho

    # ---- end to end through the C ABI with HOST buffers: H2D of the 6 inputs, one step, D2H of U
    out = [torch.empty((w.nz, w.ny, w.nx), dtype=fields[0].dtype).pin_memory() for _ in range(5)]
    n_e2e = max(1, args.e2e_steps)
    s.set_state_host(*fields)
    s.step_cfl(w.cfl)
    s.get_conserved_host(out)           # warm-up of the host path
    barrier()
    # asynchronous host entry points: the result of one step leaves on one copy stream while the input of the next
    # arrives on another (both directions of the host link); every step still copies its own inputs and its own result
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(s.stream)
    for _ in range(n_e2e):
        s.set_state_host_async(*fields)
        s.step_cfl(w.cfl)
        s.get_conserved_host_async(out)
    s.sync()                            # the ctx's stream and both copy streams
    f1.record(s.stream)
    barrier()
    ems = f0.elapsed_time(f1)
    ems = max_over_ranks(ems, world, "cuda")
    e2e = {"value": job_value(w.cells, n_e2e, world, ems), "unit": UNIT,
           "h2d_bytes_per_step": 6 * w.cells * esz, "d2h_bytes_per_step": 5 * w.cells * esz, "steps": n_e2e,
           "what": "cspt_set_state_host_async + cspt_step_cfl + cspt_get_conserved_host_async per step, one cspt_sync at the "
                   "end, pinned host buffers (the copy out of step k overlaps the copy in of step k+1)"}
    s.close()
    del s, out, fields
    torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel, from the event pairs of the profiled pass
    peak, peak_src = peaks()
    step_ms = tmax / args.steps
    # the library records a bounded number of event pairs (8192): with very many steps the profiled pass covers only
    # the first ones, so every per-step figure is taken over the steps that WERE recorded (the Euler stage runs once
    # per step and is the last launch of a step)
    prof_steps = min(args.steps, int(prof.get("euler", (0, args.steps))[1])) or args.steps
    kern = {}
    for k, v in prof.items():
        kern[k] = {"ms_per_step": v[0] / prof_steps, "launches_per_step": v[1] / prof_steps}
    dom = max(prof.items(), key=lambda kv: kv[1][0])[0]
    dom_ms = prof[dom][0] / prof[dom][1]
    prof_step_ms = sum(v[0] for v in prof.values()) / prof_steps
    words = KERNEL_WORDS.get(dom, MIN_WORDS_PER_CELL)
    dom_bytes = words * esz * w.cells
    ach = dom_bytes / (dom_ms * 1e-3) / 1e9
    traffic, traffic_src, ncu_stored = stored_traffic(w, dom)
    hbm = {"achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "peak_source": peak_src,
           "algorithmic_bytes_per_launch": dom_bytes}
    share = (prof[dom][0] / prof_steps) / prof_step_ms
    if dom in ALGO_FLOPS and args.kernel == "cubic":
        # The corrector is bound by the plain FP64 / FP32 pipe.  Roofline as SURVEY 8(d) states it:
        # the survey's instruction list per cell (FMA counted once) over the ARCHITECTURAL rate of that pipe,
        # lanes x SMs x the maximum SM clock (64 FP64 / 128 FP32 lanes per SM, B200_PROFILING.md); an FP instruction
        # of any kind holds a lane for one slot.  Beside it: the same over the clock NVML sampled while the kernel
        # times were taken, the flop version (FMA = 2), and the in-run FMA probe with ITS sampled clock as a check.
        lanes = 64 if w.dtype == "f64" else 128
        max_mhz = clocks.get("sm_max_mhz") or 1965
        peak_i = lanes * sm_count * max_mhz * 1e6 / 1e12                 # T FP instructions / s
        ach_i = ALGO_INSTR[dom] * w.cells / (dom_ms * 1e-3) / 1e12
        ach_f = ALGO_FLOPS[dom] * w.cells / (dom_ms * 1e-3) / 1e12
        run_mhz = prof_clocks.get("sm_mhz") or clocks.get("sm_mhz")
        probe = None
        if fma_rate:
            pm = probe_clocks.get("sm_mhz")
            probe = {"fma_per_second": fma_rate, "sm_mhz_during_probe": pm, "probe_clocks": probe_clocks,
                     "fma_per_clock_per_sm": fma_rate / sm_count / (pm * 1e6) if pm else None,
                     "lanes_per_sm": lanes, "instr_frac_of_probe": ach_i * 1e12 / fma_rate,
                     "fma_per_second_three_register_operands": fma_rate3,
                     "fma_per_second_with_other_instructions": issue_probe,
                     "issue_note": "FMA rate with 1 / 2 / 4 / 8 independent integer instructions behind every FMA: cycles "
                                   "per FMA and SMSP ~ max(pipe, 1.1 * (1 + others)), pipe = 2 in fp64 and 1 in fp32 "
                                   "(DESIGN.md section 7, profiles/r2_issue_model.md)"}
        roofline = {"bound": "alu", "kernel": dom, "achieved": ach_i, "peak": peak_i, "unit": "T FP instr/s",
                    "frac": ach_i / peak_i,
                    "frac_is": "SURVEY 8(d) instruction list of the corrector (%d FP instructions per cell, FMA counted once) "
                               "x cells / kernel time, over %d lanes x %d SMs x %d MHz (maximum SM clock)"
                               % (ALGO_INSTR[dom], lanes, sm_count, max_mhz),
                    "peak_source": "architectural: lanes x SMs x sm_max_mhz (B200_PROFILING.md unit counts; NVML max clock)",
                    "frac_at_sampled_clock": ach_i / (lanes * sm_count * run_mhz * 1e6 / 1e12) if run_mhz else None,
                    "sampled_clock_mhz": run_mhz, "clocks_during_kernel_timing": prof_clocks,
                    "flops": {"achieved": ach_f, "peak": 2.0 * peak_i, "unit": "TFLOP/s", "frac": ach_f / (2.0 * peak_i),
                              "per_cell": ALGO_FLOPS[dom],
                              "note": "33 flop per neighbour (the survey's list, FMA = 2) x 26 + 60 for Eq. (6)"},
                    "traffic": traffic, "traffic_source": traffic_src, "ncu": ncu_stored,
                    "probe": probe, "probe_error": probe_err,
                    "algorithmic_instr_per_cell": ALGO_INSTR[dom], "kernel_ms": dom_ms, "share_of_step": share,
                    "hbm": hbm}
        if w.name == "disk":
            roofline["note"] = ("gas-vacuum workload: the instruction list is counted over ALL cells, while CTAs whose "
                                "inputs are exactly 0 return early (DESIGN.md section 7): not a pipe utilisation here")
    else:
        roofline = dict(hbm, bound="hbm", kernel=dom, traffic=traffic, traffic_source=traffic_src, ncu=ncu_stored, kernel_ms=dom_ms,
                        share_of_step=share)
    step_ach = MIN_WORDS_PER_CELL * esz * w.cells / (step_ms * 1e-3) / 1e9
    step_hbm = {"bytes_per_cell_update": MIN_WORDS_PER_CELL * esz, "achieved_gbs": step_ach, "frac_of_measured": step_ach / peak,
                "frac_of_nominal_8TBs": step_ach / 8000.0}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": step_ms, "kernels": kern, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": w.dtype, "data": "synthetic",
        "config": dict(config_of(w, world), limiter=args.limiter, kernel=args.kernel, riemann=args.riemann,
                       api="cspt_run_cfl", tile_skip=not args.no_tile_skip),
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "kernels_note": "per-kernel times from a second pass of the same K steps with an event pair around every launch "
                        "(%.3f ms per step in that pass, %d steps recorded)" % (prof_step_ms, prof_steps),
        "roofline": roofline, "step_hbm": step_hbm,
    }

    if world == 1 and not args.no_configs:
        headline = {"workload": "%s %dx%dx%d %s" % (w.name, w.nx, w.ny, w.nz, w.dtype), "steps": args.steps,
                    "ms_per_step": step_ms, "value": value, "unit": UNIT, "frac_of_measured_hbm": step_ach / peak,
                    "api": "cspt_run_cfl (CUDA graph of two steps)", "finite": True}
        line["configs"] = run_configs(cspt, peak, headline)

    if not args.no_cpu_baseline and world == 1:
        n_s = min(384, max(w.nx, w.ny, w.nz)) if args.workload != "sod" else None
        ws, times, cores = oracle_sample(args, w, 3, 0, n_s)
        tot = sum(times)
        line["cpu_baseline"] = {"value": ws.cells * len(times) / tot / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "cpu_model": cpu_model(),
                                "sample": "%s instance %dx%dx%d (%s), 3 steps (compute_dt + step), %d threads; %.1f s"
                                % (ws.name, ws.nx, ws.ny, ws.nz, ws.dtype, cores, tot)}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_slab(args):
    """ONE grid cut into z slabs over the ranks (paper_1912_04855_b200/slab.py): per step one halo exchange of 3 planes
    x 5 fields per face over NCCL and one scalar min all-reduce.  Strong scaling: value = the grid's cells x steps / time."""
    import torch
    import torch.distributed as dist
    from paper_1912_04855_b200 import build, cspt, slab

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CSPH-TVD path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    cspt.lib()
    w = make_workload(args)
    dtype = cspt.F64 if w.dtype == "f64" else cspt.F32
    s = slab.SlabSolver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, dtype, rank, world)
    f = w.fields_slab(s.z0, s.z1)
    s.set_state(*[torch.from_numpy(a.astype(w.np_dtype)).cuda() for a in f])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        s.step_cfl(w.cfl, want_dt=False)       # enqueue only: the time step is reduced on the device
    barrier()
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.solver.launch_count()
    sampler.start()
    e0.record(s.solver.stream)
    for _ in range(args.steps):
        s.step_cfl(w.cfl, want_dt=False)       # enqueue only: the time step is reduced on the device
    e1.record(s.solver.stream)
    barrier()
    clocks = sampler.stop()
    tmax = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
    launches = s.solver.launch_count() - l0
    rho = s.get_conserved()[0]
    assert bool(torch.isfinite(rho).all()), "state is not finite after the timed steps"
    halo = 2 * s.solver.halo_elems(cspt.HALO_U) * (8 if w.dtype == "f64" else 4)
    s.close()
    if rank == 0:
        peak, _ = peaks()
        esz = 8 if w.dtype == "f64" else 4
        value = w.cells * args.steps / (tmax * 1e-3) / 1e6
        ach = MIN_WORDS_PER_CELL * esz * w.cells / (tmax / args.steps * 1e-3) / 1e9
        cfg = config_of(w, world)
        cfg["parallelism"] = "z slabs over %d gpu(s): %d planes each, %d halo bytes per rank and step, one min all-reduce" % (
            world, w.nz // world, halo)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": tmax / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": w.dtype, "data": "synthetic", "config": dict(cfg, api="slab.SlabSolver.step_cfl"),
            "clocks": clocks, "gpu_launches": launches,
            "step_hbm": {"bytes_per_cell_update": MIN_WORDS_PER_CELL * esz, "achieved_gbs": ach,
                         "frac_of_measured_all_gpus": ach / (peak * world)}}))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    elif args.decomp == "slab":
        run_slab(args)
    else:
        run_cspt(args)


if __name__ == "__main__":
    main()
