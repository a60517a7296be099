#!/usr/bin/env python
"""bench.py -- TCUPS of the FDTD hot path, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--tsteps S] [--kernel systolic|naive] [--impl reference]
                    [--config I] [--size n] [--no-sweep] [--no-e2e] [--no-cpu-baseline]

Headline workload: BASELINE.json configs[4] (1536x1536x768 lossy heterogeneous grid, six per-cell coefficient arrays,
anisotropic cells, point source, 81 GiB resident) -- the largest single-GPU configuration, far above L2, and the one
closest to the paper's own "bare-bones" benchmark (permittivity and conductivity fields).  A bench "step"
is one fdtd_step(S) call: S = 100 FDTD time steps of the whole grid (all rows of SURVEY.md 8(a): E half-step, source,
H half-step, walls, tile residency, shell load/store, flags, slide, launch ramp).  `value` is timed with the fields
resident in HBM (CUDA events on the stream the kernels run on); `e2e` goes through the same C-ABI calls with HOST
buffers: pinned host -> device copy of the six field arrays, S steps, device -> host copy, every step.
`sweep` (same JSON line, N = 1 only) is the metric "TCUPS vs grid size": naive and systolic kernels on configs 1, 2, 3,
the configs[3] cubes 64^3 .. 1024^3 and config 5, each timed in this run, with the fraction of its own roofline.
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

# the CPU oracle's OpenMP team: one thread per core, pinned, set before libgomp is loaded (stable cpu_baseline numbers)
os.environ.setdefault("OMP_PROC_BIND", "close")
os.environ.setdefault("OMP_PLACES", "cores")

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "TCUPS (6-component Yee cell updates/s, fp32) vs grid size; HBM GB/s"
HEADLINE_CONFIG = 4
SM_COUNT, SM_HZ_NOMINAL = 148, 1.965e9


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--tsteps", type=int, default=100, help="FDTD time steps per bench step")
    ap.add_argument("--kernel", default="systolic", choices=["systolic", "naive"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=HEADLINE_CONFIG, help="BASELINE.json configs index (0-based)")
    ap.add_argument("--size", type=int, default=0, help="cube size for the configs[3] sweep")
    ap.add_argument("--tile", default="", help="NXxNYxNZ systolic tile (default: library choice)")
    ap.add_argument("--T", type=int, default=0, help="temporal depth (default: library choice)")
    ap.add_argument("--variant", default="nofma", choices=["nofma", "fma", "prof"],
                    help="nofma = the product library (bit-exact); fma = optional contracted build")
    ap.add_argument("--storage", default="f32", choices=["f32", "f16"],
                    help="f16 = binary16 field storage with f32 arithmetic (row f1, PAPER.md:104); the headline is f32")
    ap.add_argument("--coeffs", default="arrays", choices=["arrays", "lut"],
                    help="lut = material-index coefficients (row f2, PAPER.md:103); configs 2 and 3 only; the headline uses arrays")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sweep", action="store_true")
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
        names = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4,
                 "hw_power_brake": 0x80}
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


def algorithmic_bytes_per_cell_update(kernel, tile, T, has_coef, fbytes=4, cbytes=24):
    """SURVEY.md 8(d) / DESIGN.md 6.5: global-memory bytes the schedule must move per 6-component cell update.
    T is the depth of the launch that was actually timed (min(library depth, steps per call)); fbytes = bytes per stored
    field value (4, or 2 with binary16 field storage); cbytes = coefficient bytes per cell (24: six float arrays; 3: three
    material-index bytes)."""
    if kernel == "naive":
        return 18.0 * fbytes + (float(cbytes) if has_coef else 0.0)
    Nx, Ny, Nz = tile
    V = Nx * Ny * Nz
    B = (Nx + 1) * (Ny + 1) * (Nz + 1)
    X = B - V                                   # minus shell of the box
    D = V - (Nx - 1) * (Ny - 1) * (Nz - 1)      # plus shell of the tile
    f_loads = 3 * B + 3 * V + (T - 1) * 6 * X              # step 0: box of H, E on the tile; then the minus shells
    c_cells = (B + (T - 1) * X) if has_coef else 0         # coefficients of the box, then of the entering shells
    stores = (T - 1) * 6 * D + 6 * V                       # plus shells; the whole tile at the last step
    return (fbytes * (f_loads + stores) + float(cbytes) * c_cells) / (V * T)


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


# ---- the CPU oracle beside the GPU run ----------------------------------------------------------------------------
def oracle_sample(w):
    """A bounded sample of workload w for the CPU oracle: the whole grid up to 64 M cells, else the same recipe on a grid
    a quarter as long per axis (config 5: 384x384x192, 28 M cells; the full grid would need 87 GB of host arrays)."""
    if w.cells <= (1 << 26):
        return w, f"full {w.n[0]}x{w.n[1]}x{w.n[2]} grid"
    n = tuple(max(32, x // 4) for x in w.n)
    return w.scaled(n, steps=w.steps, name=w.name), f"{n[0]}x{n[1]}x{n[2]} grid of the same recipe (1/64 of the cells of {w.name})"


def make_oracle(w):
    from oracle.yee import YeeOracle
    from paper_2502_20610_b200 import workloads
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        orc.set_source(src.comp, src.box, src.amp, src.wave)
    return orc


def cpu_baseline(w_full, config_steps, budget_s=12.0):
    """The oracle as it stands, timed on the host cores on a bounded sample (about 10-20 s of CPU work).  Runs before any
    CUDA or pinned-memory allocation of this process, with the OpenMP team pinned (see the top of this file)."""
    w, what = oracle_sample(w_full)
    orc = make_oracle(w)
    orc.step(2)                                   # warm-up: page faults, thread team
    t0 = time.perf_counter()
    orc.step(2)
    per_step = (time.perf_counter() - t0) / 2
    n = int(min(400, max(4, budget_s / max(per_step, 1e-6))))
    t0 = time.perf_counter()
    orc.step(n)
    dt = time.perf_counter() - t0
    out = {"value": w.cells * n / dt / 1e12, "unit": "TCUPS", "cores": orc.nthreads, "kind": "oracle",
           "sample": f"{what}, {n} of the config's {config_steps} time steps (after 4 warm-up steps)",
           # the CPU number belongs to sample_grid; any ratio against the GPU's full-grid value extrapolates it
           "sample_grid": list(w.n), "full_grid": list(w_full.n), "extrapolated": tuple(w.n) != tuple(w_full.n)}
    if w.fields == "zero":
        # The config starts from zero fields: as the pulse spreads, its front is a shell of subnormal values, which the
        # host cores handle slowly.  The same sample with seeded random fields (every value normal) times the oracle's
        # arithmetic without that effect.
        del orc
        orc = make_oracle(replace(w, fields="uniform"))
        orc.step(2)
        n2 = max(2, n // 2)
        t0 = time.perf_counter()
        orc.step(n2)
        out["value_random_fields"] = w.cells * n2 / (time.perf_counter() - t0) / 1e12
    return out


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, same config / metric / unit; each bench step is a
    bounded sample (2 time steps of oracle_sample(config))."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    ref_tsteps = 2
    from paper_2502_20610_b200 import workloads
    w_full = workload_of(args, (args.steps + args.warmup) * ref_tsteps)
    w, what = oracle_sample(w_full)
    orc = make_oracle(w)
    for _ in range(max(args.warmup, 1)):
        orc.step(ref_tsteps)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.step(ref_tsteps)
    dt = time.perf_counter() - t0
    tcups = w.cells * ref_tsteps * args.steps / dt / 1e12
    sample = f"{what}, {ref_tsteps} time steps per bench step (of the config's {workloads.config(args.config, args.size or None).steps})"
    line = {"impl": "reference", "metric": METRIC, "value": tcups, "unit": "TCUPS", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w_full.name, "grid": list(w_full.n), "sample_grid": list(w.n), "time_steps_per_bench_step": ref_tsteps},
            "cpu_baseline": {"value": tcups, "unit": "TCUPS", "cores": orc.nthreads, "kind": "oracle", "sample": sample},
            "e2e": {"value": tcups, "unit": "TCUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---- one timed case on the device --------------------------------------------------------------------------------
def bind_context(w, kernel, variant, E, H, coef, tile=None, T=0, stream=None):
    """A context on `stream` bound to the field arrays E, H and to the coefficient objects `coef` (shared, read-only)."""
    from paper_2502_20610_b200 import binding, workloads
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, stream=stream, variant=variant)
    sim.set_fields(E, H)
    if coef is not None and coef[0] == "lut":
        sim.set_coeff_lut(coef[1], coef[2], coef[3])
    elif coef is not None:
        sim.set_coeffs(coef[1], coef[2], None)
    src = workloads.make_source(w)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(binding.KERNEL_SYSTOLIC if kernel == "systolic" else binding.KERNEL_NAIVE, tile, T)
    return sim


def setup_case(w, kernel, variant, dev, tile=None, T=0, storage="f32", coeffs="arrays"):
    """Seeded inputs of workload w on the device, a context bound to them.  Returns (sim, (E, H, coef)) with coef = None |
    ("arrays", ca, cb) | ("lut", index arrays, ca table, cb table)."""
    import torch
    from paper_2502_20610_b200 import workloads
    E, H = workloads.make_fields(w, device=dev)
    if storage == "f16":
        E, H = [a.to(torch.float16) for a in E], [a.to(torch.float16) for a in H]
    coef = None
    if coeffs == "lut":
        coef = ("lut",) + tuple(workloads.make_coeff_lut(w, device=dev))
    else:
        ca, cb = workloads.make_coeffs(w, device=dev)
        if ca is not None:
            coef = ("arrays", ca, cb)
    sim = bind_context(w, kernel, variant, E, H, coef, tile, T)
    return sim, (E, H, coef)


def load_counters():
    """Measured per-cell-update counters of the systolic kernel (ncu captures, profiles/traffic.json)."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    except Exception:
        return {}


def roofline_of(kernel, w, info, has_coef, S, tcups, peak_gbs, counters, storage="f32", coeffs="arrays"):
    """HBM roofline of one case: algorithmic bytes per cell update of the launch that was timed x achieved rate / peak."""
    T = min(info["T"], S) if kernel == "systolic" else 0
    bpc = algorithmic_bytes_per_cell_update(kernel, info["tile"], max(T, 1), has_coef, 2 if storage == "f16" else 4, 3 if coeffs == "lut" else 24)
    achieved = bpc * tcups * 1e12 / 1e9
    out = {"bytes_per_cell_update": bpc, "T_launched": T, "achieved_gbs": achieved, "frac": achieved / peak_gbs,
           "roof_tcups": peak_gbs * 1e9 / bpc / 1e12}
    key = "systolic:coef" if has_coef else "systolic:uniform"
    if kernel == "systolic" and key in counters:
        c = counters[key]
        # explanatory on-chip ceilings from MEASURED counters: every warp instruction takes one of 4 issue slots per SM and
        # clock; every shared-memory wavefront one cycle of the SM's 128-byte data path
        hz = SM_HZ_NOMINAL
        out["issue_roof_tcups"] = SM_COUNT * 4 * hz / c["warp_inst_per_cell_update"] / 1e12
        out["smem_roof_tcups"] = SM_COUNT * hz / c["smem_wavefronts_per_cell_update"] / 1e12
    return out


def time_case(sim, S, K, W, barrier=None):
    """W untimed + K timed fdtd_step(S) calls; CUDA events on the stream the kernels run on.  Returns (ms, launches)."""
    import torch
    for _ in range(W):
        sim.step(S)
    sim.sync()
    if barrier is not None:
        barrier()
    c0 = sim.counters()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(K):
        sim.step(S)
    ev1.record()
    if barrier is not None:
        barrier()
    sim.sync()
    return ev0.elapsed_time(ev1), sim.counters()["launches"] - c0["launches"]


SWEEP = [("C1", 0, None, "f32"), ("C4-64", 3, 64, "f32"), ("C4-128", 3, 128, "f32"), ("C4-256", 3, 256, "f32"), ("C2", 1, None, "f32"),
         ("C4-512", 3, 512, "f32"), ("C3", 2, None, "f32"), ("C4-768", 3, 768, "f32"), ("C4-1024", 3, 1024, "f32"), ("C5", 4, None, "f32"),
         # row f1: binary16 field storage, f32 arithmetic (the paper's own configuration)
         ("C2", 1, None, "f16"), ("C4-1024", 3, 1024, "f16"), ("C5", 4, None, "f16"),
         # row f2: material-index coefficients (three bytes per cell instead of six floats)
         ("C2", 1, None, "lut"), ("C3", 2, None, "lut")]


def run_sweep(variant, dev, peak_gbs, counters, headline, skip_name):
    """TCUPS vs grid size (the metric; Fig. 1): both kernels on every config, a few launches each."""
    import torch
    from paper_2502_20610_b200 import workloads
    rows = []
    for name, idx, size, storage in SWEEP:
        coeffs = "lut" if storage == "lut" else "arrays"
        storage = "f32" if storage == "lut" else storage
        w0 = workloads.config(idx, size)
        if w0.name == skip_name and storage == "f32":            # the headline workload was just timed: reuse its numbers
            rows.append(headline)
            continue
        # S time steps per call, K calls: the config's own step count where that is a few launches, never less than 2 calls
        S = min(w0.steps, 100 if w0.cells > (1 << 24) else 200)
        fb = 2 if storage == "f16" else 4
        cbytes = 3 if coeffs == "lut" else 24
        row = {"workload": w0.name, "grid": list(w0.n), "field_storage": storage, "coefficients": coeffs if w0.has_coeff_arrays else "uniform",
               "working_set_mb": (6 * fb + (cbytes if w0.has_coeff_arrays else 0)) * w0.cells / 1e6, "time_steps_per_call": S}
        for kernel in ("naive", "systolic"):
            K, W = (2, 1) if w0.cells > (1 << 27) else (3, 2)
            Sk = S if kernel == "systolic" else max(10, min(S, int(2e10 / w0.cells)))       # the naive rate does not depend on S
            w = replace(w0, steps=max(w0.steps, (K + W) * Sk + 1))
            sim, keep = setup_case(w, kernel, variant, dev, storage=storage, coeffs=coeffs)
            info = sim.get_kernel()
            ms, launches = time_case(sim, Sk, K, W)
            tc = w.cells * Sk * K / (ms * 1e-3) / 1e12
            r = roofline_of(kernel, w, info, w.has_coeff_arrays, Sk, tc, peak_gbs, counters, storage, coeffs)
            row[kernel + "_tcups"] = tc
            row[kernel + "_frac"] = r["frac"]
            row[kernel + "_bytes_per_cell_update"] = r["bytes_per_cell_update"]
            if kernel == "systolic":
                row["T"] = r["T_launched"]
                row["tiles_per_launch"] = info["tiles"]
            sim.close()
            del sim, keep
            torch.cuda.empty_cache()
        row["systolic_over_naive"] = row["systolic_tcups"] / row["naive_tcups"]
        rows.append(row)
    return rows


def feature_rows(variant, dev, peak_gbs):
    """Rows f3 and f4 of SURVEY.md 8(f) measured (performance "does indeed depend on ... the output volume"):
    the absorber-coefficient generator against its 36 B/cell HBM roof (three permittivity arrays read, six coefficient
    arrays written), and config 2 with one running-DFT monitor plane switched on, as overhead against the plain run."""
    import numpy as np
    import torch
    from paper_2502_20610_b200 import binding, workloads
    rows = []
    # f3: fdtd_absorber_coeffs on 512^3, 12-cell layers on all six faces
    n = (512, 512, 512)
    shape = (n[2], n[1], n[0])
    eps = [torch.full(shape, 2.1, dtype=torch.float32, device=dev) for _ in range(3)]
    ca = [torch.empty(shape, dtype=torch.float32, device=dev) for _ in range(3)]
    cb = [torch.empty(shape, dtype=torch.float32, device=dev) for _ in range(3)]
    call = lambda: binding.absorber_coeffs(n, 0.25, eps, (12,) * 6, (0.4,) * 6, 3, ca, cb, variant=variant)
    for _ in range(3):
        call()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(10):
        call()
    ev1.record()
    torch.cuda.synchronize()
    gbs = 36.0 * n[0] * n[1] * n[2] * 10 / (ev0.elapsed_time(ev1) * 1e-3) / 1e9
    rows.append({"feature": "f3 fdtd_absorber_coeffs", "grid": list(n), "bytes_per_cell": 36.0, "achieved_gbs": gbs, "peak_gbs": peak_gbs,
                 "frac": gbs / peak_gbs, "launches": 10})
    del eps, ca, cb
    torch.cuda.empty_cache()
    # f4: config 2, systolic kernel, one z-plane monitor with 4 frequencies
    w0 = workloads.config(1)
    S, K, W = 200, 3, 2
    w = replace(w0, steps=(K + W) * S + 1)
    tc = {}
    for mon in (None, 2, 1, 0):                        # plain, then one monitor plane normal to z, y, x
        sim, keep = setup_case(w, "systolic", variant, dev)
        if mon is not None:
            F, nt = 4, (K + W) * S
            tt = np.arange(nt)[:, None]
            om = 2 * np.pi * (0.02 + 0.01 * np.arange(F))[None, :]
            wE = np.stack([np.cos(om * (tt + 1) * w.dt), -np.sin(om * (tt + 1) * w.dt)], axis=2).astype(np.float32)
            wH = np.stack([np.cos(om * (tt + 1.5) * w.dt), -np.sin(om * (tt + 1.5) * w.dt)], axis=2).astype(np.float32)
            acc = torch.zeros((6, F, 2, w.cells // w.n[mon]), dtype=torch.float32, device=dev)
            sim.set_monitor(mon, w.n[mon] // 2, wE, wH, acc)
        ms, _ = time_case(sim, S, K, W)
        tc["plain" if mon is None else mon] = w.cells * S * K / (ms * 1e-3) / 1e12       # (False and 0 would be one key)
        if mon is not None:
            assert float(acc.abs().max()) > 0.0
        sim.close()
        del sim, keep
        torch.cuda.empty_cache()
    # the cost follows the tile width along the plane's normal (7, 15, 31 cells: that share of the tile steps takes the
    # accumulate path) and how many threads share the plane's cells inside a tile (all, one warp, one lane per warp)
    for axis, name in ((2, "z"), (1, "y"), (0, "x")):
        rows.append({"feature": f"f4 running-DFT monitor, one {name} plane, 4 frequencies", "workload": w0.name, "grid": list(w0.n),
                     "plain_tcups": tc["plain"], "monitor_tcups": tc[axis], "overhead_pct": 100.0 * (tc["plain"] / tc[axis] - 1.0)})
    return rows


def e2e_leg(args, w, sim, keep, tile, S, K, dev, dist, world, barrier):
    """The same metric end to end through the C ABI with HOST buffers (copies inside the timed region).  A function of its
    own so that its device and pinned buffers die with it."""
    import torch
    from paper_2502_20610_b200 import workloads
    shape = (w.n[2], w.n[1], w.n[0])
    fdtype = torch.float16 if args.storage == "f16" else torch.float32
    nbytes = 6 * w.cells * (2 if args.storage == "f16" else 4)
    ke = 2 if nbytes > (8 << 30) else max(2, min(K, 5))
    if w.fields == "zero":
        Ein = [torch.zeros(shape, dtype=fdtype).pin_memory() for _ in range(3)]
        Hin = [torch.zeros(shape, dtype=fdtype).pin_memory() for _ in range(3)]
    else:
        Eh, Hh = workloads.make_fields(w)
        Ein, Hin = [torch.from_numpy(a).to(fdtype).pin_memory() for a in Eh], [torch.from_numpy(a).to(fdtype).pin_memory() for a in Hh]
        del Eh, Hh
    Eout = [torch.empty(shape, dtype=fdtype).pin_memory() for _ in range(3)]
    Hout = [torch.empty(shape, dtype=fdtype).pin_memory() for _ in range(3)]

    # Two independent jobs in flight, each with its own device copy of the six field arrays, its own context and stream (the
    # coefficient arrays are shared, read-only): while one job computes, the other's results go device -> host and its next
    # inputs host -> device.  Every job still does the whole path: pinned host -> device, S time steps, device -> pinned host.
    jobs = []
    try:
        for j in range(2):
            st = torch.cuda.Stream(device=dev)
            Ej, Hj = (keep[0], keep[1]) if j == 0 else ([torch.empty_like(a) for a in keep[0]], [torch.empty_like(a) for a in keep[1]])
            jobs.append((bind_context(w, args.kernel, args.variant, Ej, Hj, keep[2], tile, args.T, stream=st.cuda_stream), st, Ej, Hj))
    except torch.cuda.OutOfMemoryError:
        pass                                  # one job in flight if a second copy of the fields does not fit
    sim.sync()

    def submit(job):
        job[0].set_time(0)
        job[0].load_fields(Ein, Hin)
        job[0].step(S)

    def collect(job):
        # fdtd_get_fields waits for the job's steps, enqueues the six copies out and returns only when they have landed, so
        # the copies of two jobs into the shared pinned Eout / Hout never overlap in time (each collect overwrites the last)
        job[0].get_fields(Eout, Hout)

    def run(n):
        nj = len(jobs)
        for i in range(min(nj, n)):
            submit(jobs[i])                              # fill the pipeline
        for i in range(n):
            collect(jobs[i % nj])                        # job i's steps are done: its results start to leave
            if i + nj < n:
                submit(jobs[i % nj])                     # its next inputs follow on the same stream
        for job in jobs:
            job[0].sync()
    ke1 = ke
    ke = 2 * ke if len(jobs) > 1 else ke
    run(2)
    barrier()
    t0 = time.perf_counter()
    run(ke)
    barrier()
    dt = max_over_ranks(dist, time.perf_counter() - t0, dev)
    # one simulation at a time (what a single caller sees): copy in, S steps, copy out, strictly one after the other
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke1):
        submit(jobs[0])
        collect(jobs[0])
    barrier()
    dt1 = max_over_ranks(dist, time.perf_counter() - t0, dev)
    # The host path is checked once: the arrays job 0 just delivered to the host against a device-resident run of the same
    # S steps from the same initial state (generated on the device, never through the host), bit for bit.
    ref = jobs[-1]
    if w.fields == "zero":
        for a in ref[2] + ref[3]:
            a.zero_()
    else:
        Ed, Hd = workloads.make_fields(w, device=dev)
        for dst, src in zip(ref[2] + ref[3], Ed + Hd):
            dst.copy_(src.to(fdtype))
        del Ed, Hd
    if len(jobs) == 1:
        host = [t.clone() for t in Eout + Hout]          # job 0's arrays are about to be reused
    else:
        host = Eout + Hout
    torch.cuda.synchronize()
    ref[0].set_time(0)
    ref[0].step(S)
    ref[0].sync()
    verified = True
    for hst, d in zip(host, ref[2] + ref[3]):
        verified = verified and bool(torch.equal(hst.to(dev), d))
    if not verified:
        raise SystemExit("bench.py: the end-to-end leg's host output differs from the device-resident run")
    del host
    e2e = {"value": job_tcups(world, w.cells * S * ke, dt), "unit": "TCUPS", "h2d_bytes_per_step": nbytes,
           "d2h_bytes_per_step": nbytes, "steps": ke, "jobs_in_flight": len(jobs), "ranks": world,
           "single_job": {"value": job_tcups(world, w.cells * S * ke1, dt1), "unit": "TCUPS", "steps": ke1},
           "verified": "host output of one job == device-resident run of the same steps, bit for bit",
           "note": "per bench step: six field arrays pinned host->device, S time steps, six arrays device->pinned host, all "
                   "through the C ABI; two independent jobs in flight on two streams (copies of one overlap the steps of the "
                   "other); the coefficient arrays are problem constants bound once"}
    for job in jobs:
        job[0].close()
    del jobs
    del Ein, Hin, Eout, Hout
    return e2e


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    S, K, W = args.tsteps, args.steps, max(args.warmup, 0)
    w = workload_of(args, (K + W) * S * 2)

    # ---- the CPU oracle first: before CUDA initialisation and before any pinned allocation of this process --------
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        from paper_2502_20610_b200 import workloads as _wl
        cpu = cpu_baseline(w, _wl.config(args.config, args.size or None).steps)

    import torch
    from paper_2502_20610_b200 import binding, build, workloads
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

    tile = tuple(int(x) for x in args.tile.split("x")) if args.tile else None
    sim, keep = setup_case(w, args.kernel, args.variant, dev, tile, args.T, args.storage, args.coeffs)
    info = sim.get_kernel()
    has_coef = keep[2] is not None

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
    total_ms, launches = time_case(sim, S, K, 0, barrier)
    sampler.stop_flag = True
    sampler.join()
    total_ms = max_over_ranks(dist, total_ms, dev)
    cell_updates = w.cells * S * K
    value = job_tcups(world, cell_updates, total_ms * 1e-3)

    # ---- end to end through the C ABI with host buffers ----------------------------------------------------
    e2e = None
    if not args.no_e2e:
        # every rank pins two host copies of the six field arrays (config 5: 87 GB); N replicas do that N times.  Where
        # the host cannot hold it, rank 0 alone runs the leg (one replica's end-to-end rate, "ranks": 1).
        import psutil
        pinned = 2 * 6 * w.cells * (2 if args.storage == "f16" else 4)
        if world > 1 and world * pinned > 0.6 * psutil.virtual_memory().total:
            if rank == 0:
                e2e = e2e_leg(args, w, sim, keep, tile, S, K, dev, None, 1, torch.cuda.synchronize)
                e2e["ranks"] = 1
                e2e["note"] += "; measured on rank 0 only: %d replicas would pin %.0f GB of host memory" % (world, world * pinned / 1e9)
            barrier()
        else:
            e2e = e2e_leg(args, w, sim, keep, tile, S, K, dev, dist, world, barrier)
        torch.cuda.empty_cache()

    if rank != 0:
        sim.close()
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
    counters = load_counters()
    r = roofline_of(args.kernel, w, info, has_coef, S, value / world, peak, counters, args.storage, args.coeffs)
    tma = info["smem"] in (229632, 147456)
    roofline = {"bound": "hbm", "achieved": r["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": r["frac"], "traffic": None,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (measured copy)" if "hbm_gbs" in peaks else "fallback 6.65 TB/s",
                "algorithmic_bytes_per_cell_update": r["bytes_per_cell_update"], "T_launched": r["T_launched"],
                "kernel": ("systolic_tma_kernel" if tma else "systolic_reg_kernel") if args.kernel == "systolic" else "e_half_naive+h_half_naive",
                "launches_in_region": launches, "avg_launch_ms": total_ms / max(launches, 1), "roof_tcups": r["roof_tcups"],
                # arithmetic-only ceiling: 45 separately rounded fp32 operations per cell update, 128 lanes per SM and clock
                "fp32_roof_tcups": SM_COUNT * 128 * SM_HZ_NOMINAL / 45 / 1e12}
    for k in ("issue_roof_tcups", "smem_roof_tcups"):
        if k in r:
            roofline[k] = r[k]
            roofline["on_chip_counters_source"] = counters.get("source")
    key = f"{args.kernel}:{w.name}"
    if key in counters:
        roofline["traffic"] = counters[key]["dram_bytes_per_launch"]
        roofline["traffic_source"] = counters[key].get("source")

    ws = (6 * (2 if args.storage == "f16" else 4) + (24 if has_coef else 0)) * w.cells
    line = {"metric": METRIC, "value": value, "unit": "TCUPS", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "field_storage": args.storage, "coefficients": (args.coeffs if has_coef else "uniform"), "grid": list(w.n), "time_steps_per_bench_step": S, "kernel": args.kernel,
                       "tile": list(info["tile"]), "T": r["T_launched"] if args.kernel == "systolic" else 0, "T_library": info["T"], "tiles_per_launch": info["tiles"], "ctas": info["ctas"],
                       "smem_per_cta": info["smem"], "variant": args.variant, "parallelism": "replicas" if world > 1 else "single",
                       "l2": "inputs exceed L2 (%.0f MB of fields+coefficients vs 126 MB)" % (ws / 1e6) if ws > 200e6
                             else "inputs fit L2 (no flush): below-L2 point of the size sweep"},
            "clocks": sampler.result(), "gpu_launches": int(launches), "roofline": roofline}
    if e2e is not None:
        line["e2e"] = e2e
    if cpu is not None:
        line["cpu_baseline"] = cpu
    sim.close()
    headline_row = {"workload": w.name, "grid": list(w.n), "field_storage": args.storage,
                    "coefficients": (args.coeffs if has_coef else "uniform"), "working_set_mb": ws / 1e6, "time_steps_per_call": S,
                    args.kernel + "_tcups": value / world, args.kernel + "_frac": r["frac"],
                    args.kernel + "_bytes_per_cell_update": r["bytes_per_cell_update"], "T": r["T_launched"],
                    "tiles_per_launch": info["tiles"]}
    if world == 1 and not args.no_sweep and args.kernel == "systolic" and not args.tile and not args.T and args.storage == "f32" and args.coeffs == "arrays":
        # the headline row still needs its naive leg
        other = replace(w, steps=max(w.steps, 64))
        Sn = max(10, min(S, int(2e10 / w.cells)))
        del keep
        torch.cuda.empty_cache()
        nsim, nkeep = setup_case(other, "naive", args.variant, dev, storage=args.storage)
        ninfo = nsim.get_kernel()
        ms, _ = time_case(nsim, Sn, 2, 1)
        ntc = w.cells * Sn * 2 / (ms * 1e-3) / 1e12
        nr = roofline_of("naive", w, ninfo, has_coef, Sn, ntc, peak, counters, args.storage)
        headline_row.update({"naive_tcups": ntc, "naive_frac": nr["frac"], "naive_bytes_per_cell_update": nr["bytes_per_cell_update"],
                             "systolic_over_naive": headline_row["systolic_tcups"] / ntc})
        nsim.close()
        del nsim, nkeep
        torch.cuda.empty_cache()
        line["sweep"] = run_sweep(args.variant, dev, peak, counters, headline_row, w.name)
        line["features"] = feature_rows(args.variant, dev, peak)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
