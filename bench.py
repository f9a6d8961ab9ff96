#!/usr/bin/env python
"""bench.py — cell-updates/s per full timestep (fp64) of the GPUPEGAS hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--n 512] [--poisson periodic|isolated] [--od]

A "step" is one pass of the whole hot path over the synthetic workload: gp_max_dt (device-resident
dt) + gp_solve_poisson + gp_step.  Default workload = BASELINE.json config 5 (two-galaxy collision,
512^3, gas + collisionless component + periodic FFT gravity).  Prints ONE JSON line on rank 0.

  value      device-resident throughput: K steps bracketed by CUDA events on the library's stream, no per-kernel
             instrumentation inside; three such repeats, the median is reported (max over ranks)
  e2e        same metric through the C ABI with pinned HOST buffers: every step copies the 15
             state fields host->device, runs the full timestep, and copies them back
  roofline   dominant own kernel: algorithmic bytes per launch / its mean CUDA-event duration, measured live in a
             separate pass of K steps with per-kernel event brackets (gp_timing_*), against MEASURED_PEAKS.json
  cpu_baseline  the CPU oracle as it stands, timed on the host cores on a bounded sample

--impl reference times the CPU oracle (this tier's reference arm) on a bounded sample of the
same workload; it is the only other place this file executes oracle/.
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

METRIC = "cell-updates/s per full timestep (fp64)"
UNIT = "cell-updates/s"
W = 8  # bytes per fp64 word

# Algorithmic bytes per cell of each own kernel: every array the stage
# must read or write crosses HBM once (SURVEY.md 8(a) in->out column, 8(d) for the fused forms).
ALGO_BYTES_PER_CELL = {
    "hydro_gas_fused": (5 + 1 + 5) * W,     # 8(d): R5 + RPhi + W5
    "hydro_bme_fused": (10 + 1 + 10) * W,   # 8(d): R10 + RPhi + W10
    "cfl": 15 * W,                          # a-6
    "poisson_source": 3 * W,
    "poisson_green": 2 * W,                 # half spectrum, complex: read + write (nx/2+1)/nx * 16 B each
    "poisson_zpass_green": 2 * W,           # fused z transform + Green + inverse: the half spectrum once each way
}
# minimum bytes per cell per FULL step for the headline roofline fraction
STEP_BYTES_PER_CELL = {("gas",): 80, ("gas", "isolated"): 304, ("gas", "stars", "periodic"): 336,
                       ("gas", "stars", "isolated"): 472}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def stored_traffic(kernel, workload_key):
    """DRAM bytes per launch of `kernel` from the committed ncu --set full capture, or None."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if not os.path.exists(path):
        return None
    try:
        d = json.load(open(path))
        return d.get(workload_key, {}).get(kernel)
    except Exception:
        return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    def __init__(self, uuid, period=0.02):
        super().__init__(daemon=True)
        self.uuid, self.period = uuid, period
        self.sm, self.reasons, self.sm_max, self.power = [], set(), None, []
        self._stop_evt = threading.Event()
        self.error = None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            try:
                h = nv.nvmlDeviceGetHandleByUUID(self.uuid.encode())
            except Exception:
                h = nv.nvmlDeviceGetHandleByUUID(self.uuid)
            self.sm_max = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            }
            get = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
            while not self._stop_evt.is_set():
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                except Exception:
                    pass
                r = get(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(self.period)
        except Exception as e:  # NVML missing: report it, do not fake a clock
            self.error = repr(e)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        out = {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons), "samples": len(self.sm)}
        if self.sm:
            s = sorted(self.sm)
            out["sm_mhz"] = s[len(s) // 2]
        if self.power:
            out["power_w_max"] = max(self.power)
        if self.error:
            out["error"] = self.error
        return out


CONFIG_NOTES = {1: "Sod tube 128x4x4, gas, no gravity", 2: "smooth gas 256^3, periodic, no gravity",
                3: "cold collapse 256^3, gas + isolated FFT gravity", 4: "one disk 256^3, gas + collisionless + {p} FFT gravity",
                5: "gas + collisionless + {p} FFT gravity"}


def make_workload(args, sample_n=None):
    """The BASELINE.json config args.config at full size, or (sample_n) the same recipe on a smaller grid."""
    from paper_1311_0861_b200 import workloads as wl
    poisson = wl.POISSON_PERIODIC if args.poisson == "periodic" else wl.POISSON_ISOLATED
    c = args.config
    if c == 5:
        w = wl.two_disks(n=sample_n or args.n, poisson=poisson)
    elif c == 4:
        w = wl.disk(n=sample_n or 256, poisson=poisson)
    elif c == 3:
        w = wl.collapse(n=min(sample_n, 64) if sample_n else 256)
    elif c == 2:
        w = wl.smooth_gas(n=sample_n or 256)
    else:
        w = wl.sod()
    return w, workload_name(args)


def workload_name(args):
    note = CONFIG_NOTES[args.config].format(p=args.poisson)
    if args.config == 5:
        return f"two_disks_{args.n}^3 (BASELINE.json config 5: {note})"
    return f"{['', 'sod', 'smooth_gas', 'collapse', 'disk'][args.config]} (BASELINE.json config {args.config}: {note})"


def step_bytes_key(w):
    from paper_1311_0861_b200 import workloads as wl
    key = (("gas",) if w.components & wl.GAS else ()) + (("stars",) if w.components & wl.STARS else ())
    if w.poisson != wl.POISSON_NONE:
        key += ("periodic" if w.poisson == wl.POISSON_PERIODIC else "isolated",)
    return key


def oracle_leg(args, max_steps, budget_s):
    """Time the CPU oracle, as it stands, on a bounded sample of the workload (same recipe on an
    args.ref_n^3 grid, same cells per disk scale).  Returns (cells/s, threads, description, ms/step)."""
    import oracle
    from paper_1311_0861_b200 import workloads as wl
    w, _ = make_workload(args, sample_n=args.ref_n)
    poisson = args.poisson if w.poisson != wl.POISSON_NONE else "no"
    o = oracle.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    o.set_state(w.state())
    threads = oracle.get_threads()

    def step():
        if w.poisson != wl.POISSON_NONE:
            o.solve_poisson()
        o.step(o.max_dt(w.cfl))

    step()  # warm-up (page faults, kernel spectrum)
    t0 = time.perf_counter()
    n = 0
    while n < max_steps and (n == 0 or time.perf_counter() - t0 < budget_s):
        step()
        n += 1
    dt = time.perf_counter() - t0
    desc = (f"{n} full steps (max_dt + {poisson} Poisson + step) of the {w.name} recipe on {w.nx}x{w.ny}x{w.nz} "
            f"({w.cells} cells), OpenMP on outer loops, {threads} threads")
    return w.cells * n / dt, threads, desc, 1e3 * dt / n


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wname = workload_name(args)
    # each "step" is a bounded sample: one full oracle step of the same recipe on the args.ref_n grid
    import oracle
    from paper_1311_0861_b200 import workloads as wl
    w, _ = make_workload(args, sample_n=args.ref_n)
    o = oracle.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    o.set_state(w.state())

    def step():
        if w.poisson != wl.POISSON_NONE:
            o.solve_poisson()
        o.step(o.max_dt(w.cfl))

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = w.cells * args.steps / dt
    threads = oracle.get_threads()
    sample = (f"each step = one full oracle step of the same recipe on {w.nx}x{w.ny}x{w.nz} ({w.cells} cells); "
              f"{args.steps} steps timed with perf_counter")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wname, "reference": "CPU oracle (oracle/, plain C++17) on host cores", "sample_grid": [w.nx, w.ny, w.nz]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_gpu(args):
    import numpy as np
    import torch
    import paper_1311_0861_b200 as pkg
    from paper_1311_0861_b200 import distrib

    rank, local_rank, world = distrib.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    distrib.init("nccl", dev)
    pkg.lib()

    w, wname = make_workload(args)
    names = w.field_names
    cells = w.cells
    t_setup = time.perf_counter()
    # inputs: generated on the host (seeded, synthetic) into pinned buffers, handed over through the C ABI
    host = {k: torch.empty((w.nz, w.ny, w.nx), dtype=torch.float64, pin_memory=True) for k in names}
    w.fill({k: v.numpy() for k, v in host.items()})
    if args.od:
        # the same workload carrying the overdetermined system: rho*eps and Pi_ij ride in the fused
        # kernels, kappa and the energy balance in their epilogues; not the headline (BASELINE.json names the base step)
        sim = pkg.Simulation(w.nx, w.ny, w.nz, w.h, w.components | pkg.binding.GP_OD, w.poisson, w.G, w.gamma, w.bc)
    else:
        sim = pkg.Simulation.from_workload(w)
    for k in names:
        sim.set(k, host[k].numpy())
    if args.od:
        sim.od_derive()
    sim.synchronize()
    t_setup = time.perf_counter() - t_setup

    from paper_1311_0861_b200 import workloads as wl
    gravity = w.poisson != wl.POISSON_NONE

    def full_step():
        sim.max_dt(w.cfl, to_host=False)
        if gravity:
            sim.solve_poisson()
        sim.step(0.0)

    for _ in range(args.warmup):
        full_step()
    sim.synchronize()
    own0, fft0 = sim.launch_counts()

    uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid).replace("GPU-", "")
    sampler = ClockSampler(uuid)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream = torch.cuda.current_stream(dev)        # the library was handed this stream (binding.Simulation)

    # ---- headline: exactly K steps per repeat, nothing but the step's own launches in the timed region ----
    repeats_ms = []
    sampler.start()
    for _ in range(args.repeats):
        distrib.barrier()
        torch.cuda.synchronize()
        ev0.record(stream)
        for _ in range(args.steps):
            full_step()
        ev1.record(stream)
        torch.cuda.synchronize()
        distrib.barrier()
        repeats_ms.append(distrib.max_over_ranks(ev0.elapsed_time(ev1), dev))
    clocks = sampler.stop()
    own1, fft1 = sim.launch_counts()
    ms_max = sorted(repeats_ms)[len(repeats_ms) // 2]
    value = distrib.aggregate_throughput(cells, args.steps, ms_max, world)

    # ---- per-kernel split: a separate pass of K steps with an event pair round every launch ----
    sim.timing(True)
    for _ in range(args.steps):
        full_step()
    kernels = sim.timing_read()
    sim.timing(False)

    # the state must still be physical after the timed steps (no work skipped, no blow-up)
    dt_end = sim.max_dt(w.cfl)

    # ---- end to end through the C ABI with host buffers --------------------------------------
    e2e_steps = max(1, min(args.e2e_steps, args.steps))
    out = {k: torch.empty((w.nz, w.ny, w.nx), dtype=torch.float64, pin_memory=True) for k in names}

    def e2e_step():
        for k in names:
            sim.set(k, host[k].numpy())            # H2D inside the timed region
        if args.od:
            sim.od_derive()
        sim.max_dt(w.cfl)                          # dt comes back to the host
        if gravity:
            sim.solve_poisson()
        sim.step(0.0)
        for k in names:
            sim.get(k, out=out[k].numpy())         # D2H of the step's result

    e2e_step()
    distrib.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_ms_max = distrib.max_over_ranks(1e3 * e2e_s, dev)
    e2e_value = distrib.aggregate_throughput(cells, e2e_steps, e2e_ms_max, world)
    bytes_dir = len(names) * cells * W

    if rank != 0:
        distrib.shutdown()
        return

    # ---- roofline of the dominant own kernel ---------------------------------------------------
    peak, peak_src = measured_peak()
    own = {k: v for k, v in kernels.items() if not k.startswith("cufft")}
    top = max(own, key=lambda k: own[k][0])
    top_ms = own[top][0] / own[top][1]
    algo = ALGO_BYTES_PER_CELL.get(top, 0) * cells
    if args.od and top.startswith("hydro_"):   # one / six more fields each way
        algo += 2 * W * cells * (1 if top == "hydro_gas_fused" else 6)
    if not gravity and top.startswith("hydro_"):
        algo -= W * cells                      # no Phi to read without gravity
    achieved = algo / (top_ms * 1e-3) / 1e9
    wkey = f"{w.name}_{w.nx}_{args.poisson if gravity else 'nogravity'}" + ("_od" if args.od else "")
    roofline = {"bound": "hbm", "kernel": top, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": stored_traffic(top, wkey), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": algo, "ms_per_launch": top_ms}
    # the same kernel against the fp64 pipe: executed fp64 instructions of the committed
    # ncu capture / the live duration, peak = 148 SMs x 64 lanes x max SM clock
    roofline_alu = None
    fp64_inst = (stored_traffic("fp64_warp_inst", wkey) or {}).get(top)
    if fp64_inst:
        peak_alu = 148 * 64 * (clocks.get("sm_max_mhz") or 1965) * 1e6 / 1e12
        ach = fp64_inst * 32 / (top_ms * 1e-3) / 1e12
        rate, _ = pkg.fp64_rate_selftest()         # DFMA chains on every SM (csrc/selftest.cu)
        roofline_alu = {"bound": "alu", "kernel": top, "achieved": ach, "peak": peak_alu,
                        "unit": "T fp64 thread-instructions/s", "frac": ach / peak_alu,
                        "peak_source": "148 SMs x 64 fp64 lanes (ncu pipe peak, DESIGN.md 8) x max SM clock",
                        "peak_selftest": rate / 1e12}
    step_bytes = STEP_BYTES_PER_CELL[step_bytes_key(w)]
    if args.od:
        step_bytes += 2 * W * ((1 if w.components & wl.GAS else 0) + (6 if w.components & wl.STARS else 0))
    per_gpu = value / world
    step_roofline = {"bytes_per_cell_step": step_bytes,
                     "frac_of_8TBs": per_gpu * step_bytes / 8.0e12,
                     "frac_of_measured": per_gpu * step_bytes / (peak * 1e9)}
    breakdown = {k: {"ms_per_step": v[0] / args.steps, "launches_per_step": v[1] / args.steps} for k, v in kernels.items()}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, threads, desc, _ = oracle_leg(args, max_steps=20, budget_s=12.0)
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": wname, "grid": [w.nx, w.ny, w.nz], "components": "+".join(k for k in step_bytes_key(w) if k in ("gas", "stars")), "poisson": args.poisson if gravity else "none",
                   "overdetermined": bool(args.od), "cfl": w.cfl, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                   "cache": (f"inputs larger than L2: {len(names) * cells * W / 1e9:.1f} GB of state per step vs 126 MB L2 (no flush)"
                             if len(names) * cells * W > 4 * 126e6 else "state fits in L2 (latency-bound case, not a bandwidth measurement)"),
                   "timing": f"median of {args.repeats} repeats of {args.steps} steps, CUDA events on the library's stream, no per-kernel events inside",
                   "repeats_ms_per_step": [round(m / args.steps, 4) for m in repeats_ms],
                   "dt_after_run": dt_end, "setup_s": round(t_setup, 1)},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": bytes_dir, "d2h_bytes_per_step": bytes_dir,
                "steps": e2e_steps, "ms_per_step": e2e_ms_max / e2e_steps},
        "gpu_launches": int(own1 - own0) // args.repeats, "cufft_execs": int(fft1 - fft0) // args.repeats,
        "roofline": roofline, "roofline_alu": roofline_alu, "step_roofline": step_roofline, "kernels": breakdown,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    distrib.shutdown()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config (default 5, the headline); the others are parity cases timed for BASELINE.md")
    ap.add_argument("--n", type=int, default=512, help="grid size of the two-disk workload (BASELINE config 5: 512)")
    ap.add_argument("--poisson", default="periodic", choices=["periodic", "isolated"])
    ap.add_argument("--ref-n", type=int, default=128, help="grid size of the bounded sample the CPU oracle is timed on")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--repeats", type=int, default=3, help="repeats of the K timed steps; the median is reported")
    ap.add_argument("--selftest-peak", action="store_true",
                    help="run the DFMA self test that backs the fp64 peak of roofline_alu, print it and exit")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--od", action="store_true",
                    help="carry the overdetermined system (GP_OD context: rho*eps, Pi_ij, kappa, energy balance); the CPU legs stay the base scheme")
    args = ap.parse_args()
    if args.config == 3:
        args.poisson = "isolated"
    if args.warmup < 3:
        args.warmup = 3          # timing hygiene: at least three warm-up steps
    if args.selftest_peak:
        import paper_1311_0861_b200 as pkg
        rate, ms = pkg.fp64_rate_selftest()
        print(json.dumps({"fp64_thread_inst_per_s": rate, "kernel_ms": ms,
                          "nominal": "148 SMs x 64 lanes x 1.965 GHz = 18.61e12"}), flush=True)
        return
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: --gpus N starts the N replica ranks itself (rank 0 prints the line with n_gpus = N)
        from paper_1311_0861_b200 import distrib
        sys.exit(distrib.launch_replicas(args.gpus, [sys.executable, os.path.abspath(__file__)] + sys.argv[1:]))
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
