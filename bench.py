#!/usr/bin/env python
"""bench.py -- TCUPS of the FDTD hot path on BASELINE.json configs[1] (256^3 heterogeneous dielectric, six per-cell
coefficient arrays, z-dipole Gaussian-pulse source, PEC walls, 1000 steps, fp32), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--tsteps S] [--kernel systolic|naive] [--impl reference]

A bench "step" is one fdtd_step(S) call: S = 100 FDTD time steps of the whole grid (all rows of SURVEY.md 8(a):
E half-step, source, H half-step, walls, and for the systolic kernel tile residency, shell load/store, flags,
slide, launch ramp), so the default K = 10 is exactly the configuration's 1000 steps.  `value` is timed with the
fields resident in HBM (CUDA events on the stream the kernels run on); `e2e` goes through the same C-ABI calls
with HOST buffers: pinned host -> device copy of the six field arrays, S steps, device -> host copy, every step.
N > 1: the path does not shard ("replicas only"): every rank runs the same workload on its own GPU and
`value` sums them over the max-over-ranks time.
"""
import argparse
import json
import os
import sys
import threading
import time
from dataclasses import replace

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "TCUPS (6-component Yee cell updates/s, fp32) vs grid size; HBM GB/s"
TMA_SMEM = (229632, 147456)     # dynamic shared memory of systolic_tma.cu with / without coefficient arrays


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--tsteps", type=int, default=100, help="FDTD time steps per bench step")
    ap.add_argument("--kernel", default="systolic", choices=["systolic", "naive"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (0-based)")
    ap.add_argument("--size", type=int, default=0, help="cube size for the configs[3] sweep")
    ap.add_argument("--tile", default="", help="NXxNYxNZ systolic tile (default: library choice)")
    ap.add_argument("--T", type=int, default=0, help="temporal depth (default: library choice)")
    ap.add_argument("--variant", default="fma", choices=["fma", "nofma", "prof"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def workload_of(args, total_tsteps):
    from paper_2502_20610_b200 import workloads
    w = workloads.config(args.config, args.size or None)
    return replace(w, steps=max(total_tsteps, w.steps))


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else 0x8,
                 "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4, "hw_power_brake": 0x80}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.05)

    def result(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def algorithmic_bytes_per_cell_update(kernel, info, has_coef):
    """SURVEY.md 8(d) / DESIGN.md: global-memory bytes the schedule must move per 6-component cell update."""
    if kernel == "naive":
        return 96.0 if has_coef else 72.0
    Nx, Ny, Nz = info["tile"]
    T = info["T"]
    V = Nx * Ny * Nz
    B = (Nx + 1) * (Ny + 1) * (Nz + 1)
    X = B - V                                   # minus shell of the box
    D = V - (Nx - 1) * (Ny - 1) * (Nz - 1)      # plus shell of the tile
    nc = 6 if has_coef else 0
    loads = (3 + nc) * B + 3 * V + (T - 1) * (6 + nc) * X    # step 0: box of H(+coef), E on the tile; then shells
    stores = (T - 1) * 6 * D + 6 * V                        # shells; the whole tile at the last step
    return 4.0 * (loads + stores) / (V * T)


def max_over_ranks(dist, value, device):
    """Replicas only: the one cross-rank step of the bench is the MAX of a per-rank time.
    dist is torch.distributed (already initialised) or None for a single process."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_tcups(world, cell_updates_per_rank, seconds):
    """Whole-job throughput of `world` independent replicas that each advanced cell_updates_per_rank in `seconds`
    (the max over ranks): weak scaling, no data-path collective."""
    return world * cell_updates_per_rank / seconds / 1e12


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, same config / metric / unit."""
    import numpy as np
    from oracle.yee import YeeOracle
    from paper_2502_20610_b200 import workloads
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    ref_tsteps = 2                               # bounded sample: each bench step advances the full grid 2 time steps
    w = workload_of(args, (args.steps + args.warmup) * ref_tsteps)
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        orc.set_source(src.comp, src.box, src.amp, src.wave)
    for _ in range(args.warmup):
        orc.step(ref_tsteps)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.step(ref_tsteps)
    dt = time.perf_counter() - t0
    tcups = w.cells * ref_tsteps * args.steps / dt / 1e12
    sample = f"full {w.n[0]}x{w.n[1]}x{w.n[2]} grid, {ref_tsteps} time steps per bench step (of the config's 1000)"
    line = {"impl": "reference", "metric": METRIC, "value": tcups, "unit": "TCUPS", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "grid": list(w.n), "time_steps_per_bench_step": ref_tsteps},
            "cpu_baseline": {"value": tcups, "unit": "TCUPS", "cores": orc.nthreads, "kind": "oracle", "sample": sample},
            "e2e": {"value": tcups, "unit": "TCUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(w, config_steps):
    """The oracle timed beside the GPU run on a bounded sample (about 10-20 s of CPU work)."""
    from oracle.yee import YeeOracle
    from paper_2502_20610_b200 import workloads
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        orc.set_source(src.comp, src.box, src.amp, src.wave)
    t0 = time.perf_counter()
    orc.step(2)
    per_step = (time.perf_counter() - t0) / 2
    n = int(min(200, max(2, 12.0 / max(per_step, 1e-6))))
    t0 = time.perf_counter()
    orc.step(n)
    dt = time.perf_counter() - t0
    return {"value": w.cells * n / dt / 1e12, "unit": "TCUPS", "cores": orc.nthreads, "kind": "oracle",
            "sample": f"full {w.n[0]}x{w.n[1]}x{w.n[2]} grid, {n} of the config's {config_steps} time steps (after 2 warm-up steps)"}


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    import numpy as np
    import torch
    from paper_2502_20610_b200 import binding, build, workloads

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    if not os.path.exists(binding.lib_path(args.variant)):
        build.build(which=(args.variant,))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    S, K, W = args.tsteps, args.steps, max(args.warmup, 0)
    w = workload_of(args, (K + W) * S * 2)
    kernel = binding.KERNEL_SYSTOLIC if args.kernel == "systolic" else binding.KERNEL_NAIVE
    tile = tuple(int(x) for x in args.tile.split("x")) if args.tile else None

    E, H = workloads.make_fields(w, device=dev)
    ca, cb = workloads.make_coeffs(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant=args.variant)
    sim.set_fields(E, H)
    if ca is not None:
        sim.set_coeffs(ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(kernel, tile, args.T)
    info = sim.get_kernel()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing -------------------------------------------------------------------------------
    for _ in range(W):
        sim.step(S)
    sim.sync()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    c0 = sim.counters()
    kernel_ms = 0.0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(K):
        sim.step(S)
    ev1.record()
    barrier()
    sim.sync()
    total_ms = ev0.elapsed_time(ev1)
    kernel_ms = total_ms          # the region holds nothing but the enqueued kernels (and a 4-byte memset per launch)
    c1 = sim.counters()
    sampler.stop_flag = True
    sampler.join()
    launches = c1["launches"] - c0["launches"]
    total_ms = max_over_ranks(dist, total_ms, dev)
    cell_updates = w.cells * S * K
    value = job_tcups(world, cell_updates, total_ms * 1e-3)

    # ---- end to end through the C ABI with host buffers ----------------------------------------------------
    e2e = None
    if not args.no_e2e:
        Eh, Hh = workloads.make_fields(w)
        pin = lambda a: torch.from_numpy(a).pin_memory()
        Ein, Hin = [pin(a) for a in Eh], [pin(a) for a in Hh]
        Eout = [torch.empty_like(t).pin_memory() for t in Ein]
        Hout = [torch.empty_like(t).pin_memory() for t in Hin]
        ke = max(2, min(K, 5))
        sim.set_time(0)

        def one():
            sim.load_fields(Ein, Hin)
            sim.step(S)
            sim.get_fields(Eout, Hout)
        one()
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            sim.set_time(0)
            one()
        barrier()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dist, dt, dev)
        nbytes = 6 * w.cells * 4
        e2e = {"value": job_tcups(world, w.cells * S * ke, dt), "unit": "TCUPS", "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": ke,
               "note": "six field arrays pinned host->device, S time steps, six arrays device->host, per bench step; "
                       "the six coefficient arrays are problem constants bound once"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel -------------------------------------------------------------------
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    bpc = algorithmic_bytes_per_cell_update(args.kernel, info, ca is not None)
    achieved = bpc * cell_updates / (kernel_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (measured copy)" if "hbm_gbs" in peaks else "fallback 6.65 TB/s",
                "algorithmic_bytes_per_cell_update": bpc,
                "kernel": ("systolic_tma_kernel" if info["smem"] in TMA_SMEM else "systolic_reg_kernel") if args.kernel == "systolic" else "e_half_naive+h_half_naive",
                "launches_in_region": launches, "avg_launch_ms": kernel_ms / max(launches, 1),
                "roof_tcups": peak * 1e9 / bpc / 1e12,
                # explanatory ceilings of the systolic kernel: arithmetic-only issue floor (33 FMA-contracted
                # instructions per cell), the kernel's own instruction mix at 100 % issue, the shared-memory pipe
                "fp32_roof_tcups": 148 * 128 * 1.965e9 / 33 / 1e12,
                "issue_roof_tcups": 148 * 128 * 1.965e9 / 118 / 1e12,
                "smem_roof_tcups": 148 * 1.965e9 * 3255 / 2300 / 1e12}
    prof = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(prof):
        try:
            tr = json.load(open(prof))
            key = f"{args.kernel}:{w.name}"
            if key in tr:
                roofline["traffic"] = tr[key]["dram_bytes_per_launch"]
                roofline["traffic_source"] = tr[key].get("source")
        except Exception:
            pass

    line = {"metric": METRIC, "value": value, "unit": "TCUPS", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "grid": list(w.n), "time_steps_per_bench_step": S, "kernel": args.kernel,
                       "tile": list(info["tile"]), "T": info["T"], "tiles_per_launch": info["tiles"], "ctas": info["ctas"],
                       "smem_per_cta": info["smem"], "variant": args.variant, "parallelism": "replicas" if world > 1 else "single",
                       "l2": "inputs exceed L2 (%.0f MB of fields+coefficients vs 126 MB)" % ((6 + (6 if ca is not None else 0)) * w.cells * 4 / 1e6)
                             if (6 + (6 if ca is not None else 0)) * w.cells * 4 > 200e6 else "inputs fit L2 (no flush): below-L2 point of the size sweep"},
            "clocks": sampler.result(), "gpu_launches": int(launches), "roofline": roofline}
    if e2e is not None:
        line["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        from paper_2502_20610_b200 import workloads as _wl
        line["cpu_baseline"] = cpu_baseline(w, _wl.config(args.config, args.size or None).steps)
    print(json.dumps(line), flush=True)
    sim.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
