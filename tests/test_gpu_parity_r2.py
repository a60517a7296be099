"""GPU parity, second set ("close the parity holes"): inputs the first suite never fed the kernels.

  (a) non-default db = (0.9, 0.6, 0.3) dt with anisotropic cells                       -> a2 on every kernel
  (b) NON-ZERO frozen tangential E on the low walls + a box source that covers index-0 cells (reading #6:
      "applied on frozen cells too"), with and without coefficient arrays                -> a3 + a4
  (c) "after the full run" (north_star): C1, C2 256^3 x 1000, C4 64..512 x 200 with the library defaults, BOTH builds
  (d) C3 at its full 512x512x256 on the kernel the library picks for it
  (e) C5 and 1024^3 window oracles with the default temporal depth and more steps than one launch holds
  (f) the hand-off watchdog fires (FDTD_ETIMEOUT) instead of hanging when a flag is withheld  (dbg build)
  (g) checkpoint / resume: get_fields -> new ctx -> set_fields + set_time == the straight run

All through the C ABI; bit-exact (np.array_equal) for the product library (variant "nofma", -fmad=false), which therefore
meets north_star's max|GPU-oracle| <= 1e-5 max|field| on every run length; the optional FMA-contracted variant is held to
1e-5 as well except on the 1000-step config 2 run, where its measured drift (3e-5) is asserted against 1e-4 and is the
reason it is not the product.  The inputs of (a), (b) are built here (not in workloads.make_fields,
which zeroes the frozen cells)."""
import numpy as np
import pytest

from oracle.yee import YeeOracle
from paper_2502_20610_b200 import binding, workloads
from paper_2502_20610_b200.workloads import PEC, PERIODIC

pytestmark = pytest.mark.gpu
TOL = 1e-5
KERNELS = {"naive": binding.KERNEL_NAIVE, "systolic": binding.KERNEL_SYSTOLIC, "reg": binding.KERNEL_SYSTOLIC_REG}


def _rand(seed, aid, shape):
    idx = np.arange(int(np.prod(shape)), dtype=np.int64).reshape(shape)
    return (workloads.hash24(seed, aid, idx).astype(np.float32) * np.float32(2.0 ** -23) - np.float32(1.0)).astype(np.float32)


def _to_dev(arrs, grouped=True):
    import torch
    ts = [torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0") for a in arrs]
    return workloads._grouped(ts) if grouped else ts


def _compare(E, H, Eo, Ho, exact, tol=TOL):
    scale = max(float(np.abs(x).max()) for x in Eo + Ho)
    worst = 0.0
    for g, o in zip(list(E) + list(H), Eo + Ho):
        g = g.cpu().numpy() if hasattr(g, "cpu") else g
        assert np.all(np.isfinite(g))
        if exact:
            assert np.array_equal(g, o), f"not bit-exact: max diff {np.abs(g - o).max():.3e} at {np.unravel_index(np.abs(g - o).argmax(), g.shape)}"
        worst = max(worst, float(np.abs(g.astype(np.float64) - o.astype(np.float64)).max()))
    assert worst <= tol * max(scale, 1e-30), f"max|GPU-oracle| = {worst:.3e} > {tol} * {scale:.3e}"
    return worst / max(scale, 1e-30)


def _run_gpu(n, d, dt, boundary, E0, H0, ca, cb, db, src, steps, kernel, tile, T, variant, grouped=True):
    E, H = _to_dev(E0, grouped), _to_dev(H0, grouped)
    sim = binding.Fdtd(n, d, dt, boundary, variant=variant)
    sim.set_fields(E, H)
    cad = cbd = None
    if ca is not None:
        g = _to_dev(list(ca) + list(cb), grouped)
        cad, cbd = g[:3], g[3:]
    if ca is not None or db is not None:
        sim.set_coeffs(cad, cbd, db)
    if src is not None:
        sim.set_source(*src)
    sim.set_kernel(kernel, tile, T)
    sim.step(steps)
    sim.sync()
    info = sim.get_kernel()
    sim.close()
    return E, H, info


def _run_oracle(n, d, dt, boundary, E0, H0, ca, cb, db, src, steps):
    E, H = [a.copy() for a in E0], [a.copy() for a in H0]
    orc = YeeOracle(n, d, dt, boundary, E, H, ca, cb, db)
    if src is not None:
        orc.set_source(*src)
    orc.step(steps)
    return E, H


# ---- (a) non-default db, anisotropic cells ---------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["nofma", "fma"])
@pytest.mark.parametrize("kname,tile,T", [("naive", None, 0), ("systolic", (31, 15, 7), 16), ("systolic", (31, 15, 7), 60),
                                          ("reg", (31, 15, 7), 9), ("systolic", (15, 7, 7), 12)])
@pytest.mark.parametrize("coeffs", ["none", "lossy"])
def test_nondefault_db_and_anisotropic_cells(cuda_device, kname, tile, T, variant, coeffs):
    n, d = (72, 44, 30), (1.0, 0.7, 1.6)
    w = workloads.Workload("db", n, d, (PEC,) * 3, 60, "uniform", coeffs, "dipole", seed=77)
    dt = w.dt
    db = (0.9 * dt, 0.6 * dt, 0.3 * dt)
    E0, H0 = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    s = workloads.make_source(w)
    src = (s.comp, s.box, s.amp, s.wave)
    Eo, Ho = _run_oracle(n, d, dt, w.boundary, E0, H0, ca, cb, db, src, 60)
    E, H, _ = _run_gpu(n, d, dt, w.boundary, E0, H0, ca, cb, db, src, 60, KERNELS[kname], tile, T, variant)
    _compare(E, H, Eo, Ho, exact=(variant == "nofma"))


# ---- (b) non-zero frozen wall values, source on frozen cells ---------------------------------------------------
@pytest.mark.parametrize("variant", ["nofma", "fma"])
@pytest.mark.parametrize("kname,tile,T", [("naive", None, 0), ("systolic", (31, 15, 7), 8), ("systolic", (31, 15, 7), 50),
                                          ("reg", (31, 15, 7), 11)])
@pytest.mark.parametrize("coeffs", ["none", "lossy"])
def test_nonzero_frozen_walls_and_source_on_them(cuda_device, kname, tile, T, variant, coeffs):
    n, d = (68, 40, 26), (1.0, 1.0, 0.5)
    shape = (n[2], n[1], n[0])
    w = workloads.Workload("frozen", n, d, (PEC,) * 3, 50, "uniform", coeffs, "none", seed=5)
    dt = w.dt
    E0 = [_rand(91, a, shape) for a in range(3)]              # frozen low-wall cells keep NON-ZERO random values
    H0 = [_rand(91, 3 + a, shape) for a in range(3)]
    assert all(float(np.abs(E0[a][0]).max()) > 0 for a in range(2))
    ca, cb = workloads.make_coeffs(w)
    # box source on E_y over [0,5) x [0,4) x [0,6): covers the frozen planes i = 0 and k = 0 (E_y is tangential to both)
    box = (0, 0, 0, 5, 4, 6)
    amp = 0.5 + _rand(92, 0, (box[5], box[4], box[3]))
    t = np.arange(50, dtype=np.float64)
    wave = (np.exp(-((t - 20.0) / 8.0) ** 2) * np.cos(0.4 * t)).astype(np.float32)
    src = (1, box, amp, wave)
    Eo, Ho = _run_oracle(n, d, dt, w.boundary, E0, H0, ca, cb, None, src, 50)
    assert not np.array_equal(Eo[1][0, 0, :5], E0[1][0, 0, :5])     # the source did land on frozen cells
    E, H, _ = _run_gpu(n, d, dt, w.boundary, E0, H0, ca, cb, None, src, 50, KERNELS[kname], tile, T, variant)
    _compare(E, H, Eo, Ho, exact=(variant == "nofma"))


def test_tma_kernel_per_array_maps_separate_allocations(cuda_device):
    """Component arrays that are NOT at one stride (three separate allocations of different padding) take the per-array
    3-D tensor maps: the real trigger, no debug switch."""
    import torch
    for coeffs in ("none", "lossy"):
        w = workloads.Workload("sep", (72, 60, 52), (1, 1, 1), (PEC,) * 3, 40, "uniform", coeffs, "dipole", seed=3)
        E0, H0 = workloads.make_fields(w)
        ca, cb = workloads.make_coeffs(w)
        s = workloads.make_source(w)
        Eo, Ho = _run_oracle(w.n, w.d, w.dt, w.boundary, E0, H0, ca, cb, None, (s.comp, s.box, s.amp, s.wave), 40)
        keep = []

        def sep(arrs):
            # views of one block at deliberately UNEQUAL, 256-byte aligned offsets: 0, cells + 64, 2 cells + 256 floats
            cells = arrs[0].size
            block = torch.empty(len(arrs) * cells + 1024, dtype=torch.float32, device="cuda:0")
            keep.append(block)
            out, off = [], 0
            for q, a in enumerate(arrs):
                off = (off + 63) // 64 * 64
                v = block[off:off + cells].view(a.shape)
                v.copy_(torch.from_numpy(a))
                out.append(v)
                off += cells + 64 * (q + 1)
            return out
        E, H = sep(E0), sep(H0)
        strides = {E[1].data_ptr() - E[0].data_ptr(), E[2].data_ptr() - E[1].data_ptr()}
        assert len(strides) == 2
        sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
        sim.set_fields(E, H)
        if ca is not None:
            sim.set_coeffs(sep(ca), sep(cb), None)
        sim.set_source(s.comp, s.box, s.amp, s.wave)
        sim.set_kernel(binding.KERNEL_SYSTOLIC, (31, 15, 7), 16)
        sim.step(40)
        sim.sync()
        sim.close()
        _compare(E, H, Eo, Ho, exact=True)


# ---- periodic axes and odd nx through the product kernel (padded working copy) --------------------------
PADDED = {
    "per-x": ((64, 56, 40), (1, 1, 1), (PERIODIC, PEC, PEC), "waveguide", "sheet"),
    "per-y-odd-nx": ((37, 29, 23), (1, 0.8, 1.3), (PEC, PERIODIC, PEC), "lossy", "dipole"),
    "per-xyz": ((24, 20, 12), (1, 1, 1), (PERIODIC,) * 3, "blocks", "sheet"),
    "per-z-vac": ((40, 33, 50), (1, 1, 0.5), (PEC, PEC, PERIODIC), "none", "dipole"),
    "odd-nx-pec": ((45, 31, 19), (1, 1, 1), (PEC,) * 3, "lossy", "dipole"),
}


@pytest.mark.parametrize("variant", ["nofma", "fma"])
@pytest.mark.parametrize("T", [0, 3, 8, 20])
@pytest.mark.parametrize("name", list(PADDED))
def test_padded_working_copy_matches_oracle(cuda_device, name, T, variant):
    """Grids with a periodic axis (ghost zones refilled between launches, source images in the ghosts) or nx % 4 != 0
    (row pitch padded) run the TMA kernel on the library's padded copy; 70 steps in pieces, several launches each."""
    n, d, bnd, coeffs, source = PADDED[name]
    w = workloads.Workload(name, n, d, bnd, 70, "uniform", coeffs, source, seed=21)
    E0, H0 = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    s = workloads.make_source(w)
    src = (s.comp, s.box, s.amp, s.wave)
    Eo, Ho = _run_oracle(w.n, w.d, w.dt, w.boundary, E0, H0, ca, cb, None, src, 70)
    E, H = _to_dev(E0), _to_dev(H0)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant=variant)
    sim.set_fields(E, H)
    if ca is not None:
        g = _to_dev(list(ca) + list(cb))
        sim.set_coeffs(g[:3], g[3:], None)
    sim.set_source(*src)
    sim.set_kernel(binding.KERNEL_SYSTOLIC, (31, 15, 7) if T else None, T)
    info = sim.get_kernel()
    assert info["which"] == binding.KERNEL_SYSTOLIC and info["smem"] in (229632, 147456)
    for part in (1, 29, 40):
        sim.step(part)
    sim.sync()
    sim.close()
    _compare(E, H, Eo, Ho, exact=(variant == "nofma"))


# ---- (c) "after the full run", library defaults, both builds -----------------------------------------------------
FULL = [("C1", 0, None), ("C4-64", 3, 64), ("C4-128", 3, 128), ("C4-256", 3, 256), ("C2", 1, None), ("C4-512", 3, 512)]


@pytest.fixture(scope="module")
def full_oracle():
    cache = {}

    def get(name, idx, size):
        if name not in cache:
            w = workloads.config(idx, size)
            E, H = workloads.make_fields(w)
            ca, cb = workloads.make_coeffs(w)
            orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
            s = workloads.make_source(w)
            if s is not None:
                orc.set_source(s.comp, s.box, s.amp, s.wave)
            orc.step(w.steps)
            cache.clear()                       # one full-size result at a time (512^3 is 3.2 GB)
            cache[name] = (E, H)
        return cache[name]
    return get


@pytest.mark.parametrize("name,idx,size", FULL)
def test_full_run_parity_library_defaults(cuda_device, full_oracle, name, idx, size):
    """Every step of the configuration, default tile and temporal depth (several launches), both builds, plus the naive
    kernel of the bit-exact build."""
    w = workloads.config(idx, size)
    Eo, Ho = full_oracle(name, idx, size)
    for variant, kernel in (("nofma", binding.KERNEL_SYSTOLIC), ("fma", binding.KERNEL_SYSTOLIC), ("nofma", binding.KERNEL_NAIVE)):
        E, H, sim = binding.run_workload(w, kernel=kernel, variant=variant)
        info = sim.get_kernel()
        assert sim.time == w.steps
        sim.close()
        if kernel == binding.KERNEL_SYSTOLIC:
            assert info["which"] == binding.KERNEL_SYSTOLIC
        # the contracted variant drifts 3e-5 max|field| from the oracle over the 1000 steps of config 2 (fields decay by 100x
        # after the pulse while the rounding differences made near the source persist): outside north_star's bar, so it is
        # not the product; asserted here against 1e-4 so that a real defect still fails
        rel = _compare(E, H, Eo, Ho, exact=(variant == "nofma"), tol=1e-4 if (variant == "fma" and w.steps >= 1000) else TOL)
        print(f"full run {name} {variant} kernel={kernel}: max|GPU-oracle|/max|field| = {rel:.2e}")
        del E, H


# ---- (d) C3 at full size -----------------------------------------------------------------------------------------
def test_full_size_config3_default_kernel(cuda_device):
    """BASELINE configs[2] at its full 512x512x256 (periodic x) on the kernel the library chooses for it, 160 steps
    (more than one launch of the default depth), both builds, against the oracle run on the whole grid."""
    w = workloads.config(2)
    steps = 160
    E0, H0 = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    s = workloads.make_source(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E0, H0, ca, cb, None)
    orc.set_source(s.comp, s.box, s.amp, s.wave)
    orc.step(steps)
    assert max(float(np.abs(x).max()) for x in E0) > 0
    for variant in ("nofma", "fma"):
        E, H, sim = binding.run_workload(w, steps=steps, variant=variant)       # kernel: library default for this grid
        info = sim.get_kernel()
        sim.close()
        assert info["which"] != binding.KERNEL_NAIVE, "config 3 must run a systolic kernel by default"
        _compare(E, H, E0, H0, exact=(variant == "nofma"))
        del E, H


# ---- (e) windows at the default temporal depth, more steps than one launch ------------------------------------------
def _window_check(w, steps, win, origins, need_free, nonzero=False):
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()           # earlier tests leave tens of GB in torch's caching allocator
    free, total = torch.cuda.mem_get_info()
    if free < need_free:
        assert total < 170e9, f"only {free / 1e9:.0f} GB free of {total / 1e9:.0f} GB: something holds device memory"
        pytest.skip(f"needs {need_free / 1e9:.0f} GB of free device memory (device has {total / 1e9:.0f} GB)")
    E, H, sim = binding.run_workload(w, steps=steps, variant="nofma")
    info = sim.get_kernel()
    assert info["which"] == binding.KERNEL_SYSTOLIC and steps > info["T"] >= 64       # default depth, at least two launches
    src = workloads.make_source(w)
    nx, ny, nz = w.n
    s = steps
    for (i0, j0, k0) in origins:
        lo = [max(0, i0 - s), max(0, j0 - s), max(0, k0 - s)]
        hi = [min(nx, i0 + win + s), min(ny, j0 + win + s), min(nz, k0 + win + s)]
        box = (lo[0], lo[1], lo[2], hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2])
        Eo, Ho = workloads.make_fields(w, window=box)
        cao, cbo = workloads.make_coeffs(w, window=box)
        orc = YeeOracle(box[3:], w.d, w.dt, w.boundary, Eo, Ho, cao, cbo, None)
        if src is not None:
            sb = src.box
            if all(lo[a] <= sb[a] and sb[a] + sb[3 + a] <= hi[a] for a in range(3)):
                orc.set_source(src.comp, (sb[0] - lo[0], sb[1] - lo[1], sb[2] - lo[2], sb[3], sb[4], sb[5]), src.amp, src.wave)
        orc.step(s)
        sl_o = (slice(k0 - lo[2], k0 - lo[2] + win), slice(j0 - lo[1], j0 - lo[1] + win), slice(i0 - lo[0], i0 - lo[0] + win))
        sl_g = (slice(k0, k0 + win), slice(j0, j0 + win), slice(i0, i0 + win))
        for g, o in zip(E + H, Eo + Ho):
            got = g[sl_g].cpu().numpy()
            if nonzero:
                assert float(np.abs(o[sl_o]).max()) > 0.0, f"window at {(i0, j0, k0)} compares zero with zero"
            assert np.array_equal(got, o[sl_o]), f"window at {(i0, j0, k0)}: max diff {np.abs(got - o[sl_o]).max():.3e}"
    sim.close()
    del E, H
    gc.collect()
    torch.cuda.empty_cache()


def test_config5_random_fields_windows_default_depth(cuda_device):
    """BASELINE configs[4] starts from zero fields, so after 160 steps only windows within 160 cells of the source hold
    data.  The same recipe (lossy coefficients, anisotropic cells, point source, 81 GiB) with seeded random initial fields
    puts data under every window: low corner, high corner, a high wall face, a point where tile seams of all three axes
    meet -- frozen low walls, high-wall clipping and offsets beyond 2^32 bytes are checked on non-zero values, at the
    library's default depth with more steps than one launch holds (the launch configuration bench.py times)."""
    from dataclasses import replace
    w = replace(workloads.config(4), fields="uniform", name="C5-lossy-random-fields")
    nx, ny, nz = w.n
    win = 24
    origins = [(0, 0, 0), (nx - win, ny - win, nz - win), (nx - win, ny // 2 - 7, nz // 3), (31 * 20 - win // 2, 15 * 40 - win // 2, 7 * 50 - win // 2)]
    _window_check(w, 160, win, origins, 100e9, nonzero=True)


def test_config5_windows_default_depth(cuda_device):
    w = workloads.config(4)
    nx, ny, nz = w.n
    win = 24
    _window_check(w, 160, win, [(0, 0, 0), (nx - win, ny - win, nz - win), (nx // 2 - 12, ny // 2 - 12, nz // 2 - 12)], 100e9)


def test_config4_1024_windows_default_depth(cuda_device):
    w = workloads.config(3, 1024)
    win = 24
    _window_check(w, 160, win, [(0, 0, 0), (1024 - win, 1024 - win, 1024 - win), (31 * 16 - 10, 15 * 34 - 10, 7 * 73 - 10)], 40e9)


# ---- (f) watchdog --------------------------------------------------------------------------------------------
def test_watchdog_turns_a_withheld_flag_into_etimeout(cuda_device, monkeypatch):
    """dbg build: tile 0 never raises its flags; its downwind tiles spin past the (tiny) budget and the library reports
    FDTD_ETIMEOUT at the next sync instead of hanging.  A fresh context afterwards works."""
    monkeypatch.setenv("FDTD_SPIN_BUDGET_MS", "20")
    monkeypatch.setenv("FDTD_DEBUG_WITHHOLD", "0")
    w = workloads.config(0)
    E, H = workloads.make_fields(w, device="cuda:0")
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="dbg")
    sim.set_fields(E, H)
    sim.set_kernel(binding.KERNEL_SYSTOLIC, (31, 15, 7), 8)
    sim.step(8)
    with pytest.raises(binding.FdtdError) as e:
        sim.sync()
    assert e.value.code == binding.ETIMEOUT
    sim.close()
    monkeypatch.delenv("FDTD_DEBUG_WITHHOLD")
    E, H, sim = binding.run_workload(w, steps=8, variant="dbg")
    sim.close()
    assert all(bool(np.isfinite(x.cpu().numpy()).all()) for x in E + H)


# ---- section 5: time-level shadow arrays (race detector of the hand-off protocol) -------------------------------------
def test_level_shadow_arrays_find_no_violation_and_do_find_a_broken_protocol(cuda_device, monkeypatch):
    """dbg build with FDTD_DEBUG_LEVELS=1: every value a tile takes from global memory carries the time level the schedule
    promises -- on wall grids, on the padded periodic copy, under pseudo-random delays.  With the upwind waits switched
    off (FDTD_DEBUG_SKIP=1) and the same delays the detector must report violations: it is not vacuous."""
    monkeypatch.setenv("FDTD_DEBUG_LEVELS", "1")
    cases = [workloads.config(1).scaled((72, 60, 52), steps=60), workloads.config(2).scaled((64, 56, 40), steps=60),
             workloads.config(3, 128).scaled((100, 96, 90), steps=40)]
    for seed in ("0", "777"):
        monkeypatch.setenv("FDTD_DEBUG_DELAY", seed)
        for w in cases:
            for T in (7, 0):
                E, H, sim = binding.run_workload(w, tile=(31, 15, 7) if T else None, T=T, steps=w.steps, variant="dbg")
                errs = sim.debug_level_errors()
                sim.close()
                assert errs[0] == 0, f"{w.name} T={T} delay={seed}: level violations {errs}"
    monkeypatch.setenv("FDTD_DEBUG_SKIP", "1")
    monkeypatch.setenv("FDTD_DEBUG_DELAY", "777")
    w = cases[0]
    E, H, sim = binding.run_workload(w, tile=(31, 15, 7), T=30, steps=60, variant="dbg")
    errs = sim.debug_level_errors()
    sim.close()
    assert errs[0] > 0, "the detector did not notice tiles running without their upwind waits"
    # the product library has no such arrays
    sim = binding.Fdtd((8, 8, 8), (1, 1, 1), 0.1, (0, 0, 0))
    with pytest.raises(binding.FdtdError) as e:
        sim.debug_level_errors()
    assert e.value.code == binding.ESTATE
    sim.close()


# ---- (g) checkpoint / resume ---------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", [binding.KERNEL_SYSTOLIC, binding.KERNEL_NAIVE])
def test_checkpoint_resume_equals_straight_run(cuda_device, kernel):
    """State = six arrays + step counter: stop at t = 37 (inside the source pulse), read the fields
    to the host, destroy the context, create a new one, set_fields + set_time(37), finish; equals one straight run."""
    import torch
    w = workloads.config(4).scaled((72, 60, 52), steps=90)
    Es, Hs, sim = binding.run_workload(w, kernel=kernel, steps=90, variant="nofma")
    sim.close()
    E, H = workloads.make_fields(w, device="cuda:0")
    ca, cb = workloads.make_coeffs(w, device="cuda:0")
    s = workloads.make_source(w)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E, H)
    sim.set_coeffs(ca, cb)
    sim.set_source(s.comp, s.box, s.amp, s.wave)
    sim.set_kernel(kernel, None, 0)
    sim.step(37)
    Eh = [np.empty((w.n[2], w.n[1], w.n[0]), np.float32) for _ in range(3)]
    Hh = [np.empty((w.n[2], w.n[1], w.n[0]), np.float32) for _ in range(3)]
    sim.get_fields(Eh, Hh)
    assert sim.time == 37
    sim.close()
    del E, H
    E2 = [torch.from_numpy(a).to("cuda:0") for a in Eh]
    H2 = [torch.from_numpy(a).to("cuda:0") for a in Hh]
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E2, H2)
    sim.set_coeffs(ca, cb)
    sim.set_source(s.comp, s.box, s.amp, s.wave)
    sim.set_kernel(kernel, None, 0)
    sim.set_time(37)
    sim.step(53)
    sim.sync()
    assert sim.time == 90
    sim.close()
    for a, b in zip(E2 + H2, Es + Hs):
        assert torch.equal(a, b)


# ---- advisor: a rejected fdtd_set_kernel leaves the context as it was ---------------------------------------------
def test_rejected_set_kernel_keeps_the_previous_choice(cuda_device):
    w = workloads.Workload("rej", (40, 36, 20), (1, 1, 1), (PEC, PERIODIC, PEC), 12, "uniform", "none", "none")
    E0, H0 = workloads.make_fields(w)
    Eo, Ho = _run_oracle(w.n, w.d, w.dt, w.boundary, E0, H0, None, None, None, None, 12)
    E, H = _to_dev(E0), _to_dev(H0)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E, H)
    before = sim.get_kernel()
    with pytest.raises(binding.FdtdError):
        sim.set_kernel(binding.KERNEL_SYSTOLIC, (5, 5, 5), 4)
    after = sim.get_kernel()
    assert after == before
    sim.step(12)
    sim.sync()
    assert sim.get_kernel()["which"] == before["which"]
    sim.close()
    _compare(E, H, Eo, Ho, exact=True)


def test_switch_from_other_systolic_kernels_to_tma_on_one_context(cuda_device):
    """The TMA kernel's tile-claim counters form a ring that its own launches maintain (launch L zeroes the slot of launch
    L + 32).  Launches of the cross-check kernels on the same context must not consume or dirty ring slots: 70 of them,
    then the TMA kernel, and the result is still the oracle's bit for bit (before the fix the first TMA launches found
    counters >= ntiles and advanced nothing)."""
    w = workloads.Workload("ring", (36, 20, 12), (1.0, 0.7, 1.2), (PEC,) * 3, 0, "uniform", "lossy", "none")
    E0, H0 = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    E, H = _to_dev(E0), _to_dev(H0)
    g = _to_dev(list(ca) + list(cb))
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E, H)
    sim.set_coeffs(g[:3], g[3:], None)
    sim.set_kernel(binding.KERNEL_SYSTOLIC_REG, (31, 15, 7), 1)
    sim.step(70)                                               # 70 launches of one step each
    sim.set_kernel(binding.KERNEL_SYSTOLIC_SMEM, (31, 15, 7), 1)
    sim.step(3)
    sim.set_kernel(binding.KERNEL_SYSTOLIC, (31, 15, 7), 2)
    sim.step(80)                                               # 40 TMA launches: past the 32 that used to start on stale slots
    sim.sync()
    assert sim.counters()["launches"] == 70 + 3 + 40
    sim.close()
    Eo, Ho = _run_oracle(w.n, w.d, w.dt, w.boundary, E0, H0, ca, cb, None, None, 153)
    _compare(E, H, Eo, Ho, exact=True)
