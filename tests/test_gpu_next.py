"""GPU parity of the SURVEY.md 8(f) rows and of the two-CTAs-per-SM build of the systolic kernel, through the C ABI,
against the CPU oracles (oracle/yee.py, oracle/absorber.py, oracle/monitor.py), element by element on the same
seeded inputs.  The product library is the -fmad=false build: every comparison here is BIT-EXACT."""
import numpy as np
import pytest

from oracle.absorber import absorber_coeffs
from oracle.yee import YeeOracle
from paper_2502_20610_b200 import binding, workloads
from paper_2502_20610_b200.workloads import PEC, PERIODIC
from tests.test_gpu_parity import CASES, compare, gpu_run, oracle_run

pytestmark = pytest.mark.gpu


# ---- tile 31x7x7 (systolic_tma_by8.cu: the TMA-staged kernel with a 32x8x8 box, two CTAs per SM) ---------------------
BY8_RUNS = [("C1", 8), ("C1", 33), ("C1", 100), ("C2s", 5), ("C2s", 32), ("C3s", 16), ("C4s", 40), ("C4s", 3), ("C5s", 32),
            ("C5s", 1), ("ragged", 6), ("allper", 5)]


@pytest.fixture(scope="module")
def oracle_cache():
    cache = {}

    def get(name):
        if name not in cache:
            w, steps = CASES[name]
            cache[name] = oracle_run(w, steps)
        return cache[name]
    return get


@pytest.mark.parametrize("variant", ["nofma", "fma"])
@pytest.mark.parametrize("name,T", BY8_RUNS)
def test_tile_31x7x7_matches_oracle(cuda_device, oracle_cache, name, T, variant):
    w, steps = CASES[name]
    E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 7, 7), T=T, variant=variant)
    assert info["which"] == binding.KERNEL_SYSTOLIC and info["tile"] == (31, 7, 7) and info["T"] == T
    compare((E, H), oracle_cache(name), exact=(variant == "nofma"))


# ---- f3: adiabatic-absorber coefficient generator -------------------------------------------------------------------
ABSORBER_CASES = [
    # n, dt, with eps, thickness, sigma_max, order
    ((40, 36, 28), 0.2886751, True, (8, 6, 5, 7, 4, 9), (0.11, 0.07, 0.2, 0.05, 0.3, 0.09), 2),
    ((37, 29, 23), 0.25, False, (10, 0, 0, 12, 23, 0), (0.4, 0.0, 0.0, 0.15, 0.02, 0.0), 3),
    ((64, 8, 8), 0.31, True, (32, 32, 0, 0, 0, 0), (0.25, 0.3, 0, 0, 0, 0), 1),       # the two layers of an axis meet
    ((16, 16, 16), 0.1, True, (3, 3, 3, 3, 3, 3), (0.5,) * 6, 0),                    # order 0: uniform inside the layer
    ((130, 70, 33), 0.2, True, (20, 20, 10, 10, 8, 8), (0.05,) * 6, 4),
    ((48, 20, 12), 0.27, False, (5, 6, 7, 4, 3, 2), (0.3, 0.2, 0.1, 0.25, 0.15, 0.35), 2),   # four-cells-per-thread kernel without eps arrays
    ((256, 96, 40), 0.22, True, (12, 12, 12, 12, 12, 12), (0.4,) * 6, 3),                     # many groups per row, several blocks per thread
]


@pytest.mark.parametrize("n,dt,with_eps,thickness,smax,order", ABSORBER_CASES)
def test_absorber_generator_bit_exact(cuda_device, n, dt, with_eps, thickness, smax, order):
    import torch
    shape = (n[2], n[1], n[0])
    rng = np.random.default_rng(n[0] * 1000 + order)
    eps = [rng.uniform(1.0, 12.1, shape).astype(np.float32) for _ in range(3)] if with_eps else None
    want_ca, want_cb = absorber_coeffs(n, np.float32(dt), eps, thickness, smax, order, np.float32)
    dev = torch.device("cuda:0")
    eps_d = None if eps is None else [torch.from_numpy(e).to(dev) for e in eps]
    ca = [torch.full(shape, -7.0, dtype=torch.float32, device=dev) for _ in range(3)]
    cb = [torch.full(shape, -7.0, dtype=torch.float32, device=dev) for _ in range(3)]
    binding.absorber_coeffs(n, dt, eps_d, thickness, smax, order, ca, cb)
    torch.cuda.synchronize()
    for a in range(3):
        assert np.array_equal(ca[a].cpu().numpy(), want_ca[a]), f"ca[{a}] differs"
        assert np.array_equal(cb[a].cpu().numpy(), want_cb[a]), f"cb[{a}] differs"


def test_absorber_generator_unaligned_arrays_take_the_one_cell_kernel(cuda_device):
    """nx % 4 == 0 but the output arrays start 4 bytes off a 16-byte boundary: the vector kernel does not apply, the
    result is the same."""
    import torch
    n, dt, thickness, smax, order = (32, 12, 10), 0.3, (4, 5, 3, 2, 4, 3), (0.2, 0.3, 0.1, 0.4, 0.25, 0.15), 2
    shape = (n[2], n[1], n[0])
    cells = n[0] * n[1] * n[2]
    eps = [np.random.default_rng(5 + a).uniform(1.0, 12.1, shape).astype(np.float32) for a in range(3)]
    want_ca, want_cb = absorber_coeffs(n, np.float32(dt), eps, thickness, smax, order, np.float32)
    dev = torch.device("cuda:0")
    eps_d = [torch.from_numpy(e).to(dev) for e in eps]
    block = torch.full((6 * (cells + 4),), -7.0, dtype=torch.float32, device=dev)
    outs = [block[q * (cells + 4) + 1: q * (cells + 4) + 1 + cells].view(shape) for q in range(6)]
    assert all(t.data_ptr() % 16 == 4 for t in outs)
    binding.absorber_coeffs(n, dt, eps_d, thickness, smax, order, outs[:3], outs[3:])
    torch.cuda.synchronize()
    for a in range(3):
        assert np.array_equal(outs[a].cpu().numpy(), want_ca[a]) and np.array_equal(outs[3 + a].cpu().numpy(), want_cb[a])
    guard = block.view(6, cells + 4)
    assert bool((guard[:, 0] == -7.0).all()) and bool((guard[:, cells + 1:] == -7.0).all())     # nothing written outside the arrays


def test_absorber_rejects_bad_arguments(cuda_device):
    import torch
    dev = torch.device("cuda:0")
    n = (8, 8, 8)
    out = [torch.empty((8, 8, 8), dtype=torch.float32, device=dev) for _ in range(6)]
    for th, sm, order in (((9, 0, 0, 0, 0, 0), (0.1,) * 6, 2), ((1, 0, 0, 0, 0, 0), (-0.1, 0, 0, 0, 0, 0), 2), ((1,) * 6, (0.1,) * 6, 9),
                          ((-1, 0, 0, 0, 0, 0), (0.1,) * 6, 2)):
        with pytest.raises(binding.FdtdError) as e:
            binding.absorber_coeffs(n, 0.1, None, th, sm, order, out[:3], out[3:])
        assert e.value.code == binding.EINVAL


def test_absorber_run_end_to_end_matches_oracle(cuda_device):
    """Generator output fed to the systolic kernel: a pulse hits graded layers on all six faces; the fields after the run
    equal the oracle's run on the oracle generator's coefficients, bit for bit."""
    import torch
    w = workloads.config(1).scaled((72, 60, 52), steps=120)
    n, dt = w.n, w.dt
    th, sm = (10, 10, 8, 8, 9, 7), (0.08, 0.08, 0.1, 0.1, 0.09, 0.12)
    eps_h = [np.ascontiguousarray(e, dtype=np.float32) for e in workloads.make_eps(w)]
    ca_h, cb_h = absorber_coeffs(n, np.float32(dt), eps_h, th, sm, 2, np.float32)
    E, H = workloads.make_fields(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca_h, cb_h, None)
    src = workloads.make_source(w)
    orc.set_source(src.comp, src.box, src.amp, src.wave)
    orc.step(120)
    dev = torch.device("cuda:0")
    Ed, Hd = workloads.make_fields(w, device=dev)
    eps_d = [torch.from_numpy(np.ascontiguousarray(e)).to(dev) for e in eps_h]
    ca = [torch.empty_like(Ed[0]) for _ in range(3)]
    cb = [torch.empty_like(Ed[0]) for _ in range(3)]
    binding.absorber_coeffs(n, dt, eps_d, th, sm, 2, ca, cb)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(Ed, Hd)
    sim.set_coeffs(ca, cb, None)
    sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.step(120)
    sim.sync()
    sim.close()
    compare(([x.cpu().numpy() for x in Ed], [x.cpu().numpy() for x in Hd]), (E, H), exact=True)
    assert float(np.abs(E[2]).max()) > 0


# ---- f4: running-DFT monitors ---------------------------------------------------------------------------------------
def _weights(nt, F, seed):
    """Complex weights of a windowed DFT: exp(-i w_f (t+1) dt') * hann(t), as float32 (re, im) tables for E and H."""
    t = np.arange(nt, dtype=np.float64)
    win = 0.5 - 0.5 * np.cos(2 * np.pi * (t + 0.5) / nt)
    om = 0.05 + 0.11 * np.arange(F) + 0.003 * seed
    wE = np.zeros((nt, F, 2))
    wH = np.zeros((nt, F, 2))
    for f in range(F):
        wE[:, f, 0], wE[:, f, 1] = win * np.cos(om[f] * (t + 1)), -win * np.sin(om[f] * (t + 1))
        wH[:, f, 0], wH[:, f, 1] = win * np.cos(om[f] * (t + 1.5)), -win * np.sin(om[f] * (t + 1.5))
    return wE.astype(np.float32), wH.astype(np.float32)


MONITOR_RUNS = [
    # case, steps, nt (weights table length), axis, index, F, kernel, tile, T
    ("C2s", 90, 90, 2, 26, 2, "naive", None, 0),
    ("C2s", 90, 90, 2, 26, 2, "systolic", (31, 15, 7), 32),
    ("C2s", 90, 70, 0, 36, 3, "systolic", (31, 15, 7), 128),      # table shorter than the run
    ("C2s", 90, 90, 1, 0, 1, "systolic", (31, 7, 7), 17),          # the frozen low wall plane
    ("C2s", 90, 90, 1, 59, 1, "systolic", (31, 15, 7), 7),         # the last plane
    ("C3s", 60, 60, 0, 5, 2, "naive", None, 0),
    ("C3s", 60, 60, 0, 5, 2, "systolic", (31, 15, 7), 8),          # periodic x on the padded copy: plane has ghost images
    ("C3s", 60, 60, 2, 20, 2, "systolic", (31, 15, 7), 8),
    ("ragged", 50, 50, 1, 11, 2, "systolic", (31, 15, 7), 6),      # odd nx, periodic y
    ("ragged", 50, 50, 0, 36, 2, "systolic", (31, 7, 7), 50),
    ("C5s", 90, 90, 2, 18, 4, "systolic", (31, 15, 7), 32),
]


@pytest.mark.parametrize("name,steps,nt,axis,index,F,kernel,tile,T", MONITOR_RUNS)
def test_monitor_matches_oracle_bit_exact(cuda_device, name, steps, nt, axis, index, F, kernel, tile, T):
    import torch
    from oracle.monitor import MonitorOracle
    w, _ = CASES[name]
    wE, wH = _weights(nt, F, axis + index)
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        orc.set_source(src.comp, src.box, src.amp, src.wave)
    mon = MonitorOracle(orc, axis, index, wE, wH)
    mon.step(steps)
    want = mon.acc.reshape(6, F, 2, -1)

    dev = torch.device("cuda:0")
    Ed, Hd = workloads.make_fields(w, device=dev)
    cad, cbd = workloads.make_coeffs(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(Ed, Hd)
    if cad is not None:
        sim.set_coeffs(cad, cbd, None)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(binding.KERNEL_NAIVE if kernel == "naive" else binding.KERNEL_SYSTOLIC, tile, T)
    acc = torch.zeros((6, F, 2, want.shape[3]), dtype=torch.float32, device=dev)
    sim.set_monitor(axis, index, wE, wH, acc)
    # two calls: the second one continues the accumulation
    sim.step(steps // 3)
    sim.step(steps - steps // 3)
    sim.sync()
    sim.close()
    got = acc.cpu().numpy()
    assert float(np.abs(want).max()) > 0
    assert np.array_equal(got, want), f"monitor differs: max {np.abs(got - want).max():.3e}"
    compare(([x.cpu().numpy() for x in Ed], [x.cpu().numpy() for x in Hd]), (E, H), exact=True)   # and the fields are untouched by it


def test_monitor_rejected_by_other_schedules_and_bad_arguments(cuda_device):
    import torch
    w, _ = CASES["C1"]
    dev = torch.device("cuda:0")
    Ed, Hd = workloads.make_fields(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(Ed, Hd)
    wE, wH = _weights(10, 1, 0)
    acc = torch.zeros((6, 1, 2, 64 * 64), dtype=torch.float32, device=dev)
    for axis, index in ((3, 0), (0, 64), (1, -1)):
        with pytest.raises(binding.FdtdError) as e:
            sim._check(sim._lib.fdtd_set_monitor(sim._h, axis, index, 1, 10, wE.ctypes.data_as(binding.C.POINTER(binding.C.c_float)),
                                                 wH.ctypes.data_as(binding.C.POINTER(binding.C.c_float)), binding.C.c_void_p(acc.data_ptr())))
        assert e.value.code == binding.EINVAL
    sim.set_monitor(0, 3, wE, wH, acc)
    sim.set_kernel(binding.KERNEL_SYSTOLIC_REG, (31, 15, 7), 8)
    with pytest.raises(binding.FdtdError) as e:
        sim.step(2)
    assert e.value.code == binding.EINVAL
    sim.set_monitor(0, 0, None, None, None)     # removed: the schedule runs again
    sim.step(2)
    sim.sync()
    sim.close()


# ---- f1: binary16 field storage, f32 arithmetic ---------------------------------------------------------------------
def _h16_oracle(w, steps):
    r16 = lambda a: a.astype(np.float16).astype(np.float32)
    E, H = workloads.make_fields(w)
    E, H = [r16(a) for a in E], [r16(a) for a in H]
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None, storage="f16")
    src = workloads.make_source(w)
    if src is not None:
        orc.set_source(src.comp, src.box, src.amp, src.wave)
    orc.step(steps)
    return E, H


def _h16_gpu(w, steps, kernel, tile, T, variant="nofma", calls=1):
    import torch
    dev = torch.device("cuda:0")
    E, H = workloads.make_fields(w, device=dev)
    E, H = [a.to(torch.float16) for a in E], [a.to(torch.float16) for a in H]      # round-to-nearest-even, as the oracle's inputs
    ca, cb = workloads.make_coeffs(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant=variant)
    sim.set_fields(E, H)
    if ca is not None:
        sim.set_coeffs(ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(kernel, tile, T)
    for c in range(calls):
        sim.step(steps // calls if c < calls - 1 else steps - (calls - 1) * (steps // calls))
    sim.sync()
    info = sim.get_kernel()
    sim.close()
    return [a.float().cpu().numpy() for a in E], [a.float().cpu().numpy() for a in H], info


@pytest.fixture(scope="module")
def h16_cache():
    cache = {}

    def get(name):
        if name not in cache:
            w, steps = CASES[name]
            cache[name] = _h16_oracle(w, steps)
        return cache[name]
    return get


H16_RUNS = [("C1", "naive", None, 0), ("C2s", "naive", None, 0), ("C3s", "naive", None, 0), ("ragged", "naive", None, 0),
            ("C1", "systolic", (31, 15, 7), 33), ("C1", "systolic", (31, 15, 7), 128), ("C2s", "systolic", (31, 15, 7), 32),
            ("C2s", "systolic", (31, 15, 7), 5), ("C3s", "systolic", (31, 15, 7), 16), ("C4s", "systolic", (31, 15, 7), 40),
            ("C5s", "systolic", (31, 15, 7), 32), ("C5s", "systolic", (31, 15, 7), 1), ("ragged", "systolic", (31, 15, 7), 6),
            ("allper", "systolic", (31, 15, 7), 5)]


@pytest.mark.parametrize("name,kernel,tile,T", H16_RUNS)
def test_f16_storage_matches_oracle_bit_exact(cuda_device, h16_cache, name, kernel, tile, T):
    w, steps = CASES[name]
    E, H, info = _h16_gpu(w, steps, binding.KERNEL_NAIVE if kernel == "naive" else binding.KERNEL_SYSTOLIC, tile, T, calls=2)
    want = h16_cache(name)
    assert max(float(np.abs(a).max()) for a in want[0] + want[1]) > 0
    compare((E, H), want, exact=True)


def test_f16_storage_fma_build_within_tolerance_and_other_schedules_rejected(cuda_device, h16_cache):
    w, steps = CASES["C5s"]
    E, H, _ = _h16_gpu(w, steps, binding.KERNEL_SYSTOLIC, (31, 15, 7), 32, variant="fma")
    want = h16_cache("C5s")
    scale = max(float(np.abs(a).max()) for a in want[0] + want[1])
    worst = max(float(np.abs(g - o).max()) for g, o in zip(E + H, want[0] + want[1]))
    assert worst <= 2.0 ** -10 * scale          # contraction moves a result across a binary16 rounding boundary now and then
    for kernel, tile in ((binding.KERNEL_SYSTOLIC_REG, (31, 15, 7)), (binding.KERNEL_SYSTOLIC, (31, 7, 7)), (binding.KERNEL_SYSTOLIC_SMEM, (15, 7, 7))):
        with pytest.raises(binding.FdtdError) as e:
            _h16_gpu(w, 4, kernel, tile, 4)
        assert e.value.code == binding.EINVAL


# ---- f2: launch-to-launch overlap (consecutive launches of one tile grid run concurrently, gated by per-tile flags) ----
OVERLAP_T = [2, 3, 7, 8, 15, 16, 31, 32, 33]


@pytest.mark.parametrize("name", ["C2s", "C5s", "C1"])
def test_overlapping_launches_bit_exact_for_every_depth(cuda_device, oracle_cache, name):
    """Many short launches back to back: each may start while the previous one drains.  Depths around the tile widths
    (7, 15, 31) exercise every shape of the predecessor set."""
    w, steps = CASES[name]
    for T in OVERLAP_T:
        E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 15, 7), T=T)
        compare((E, H), oracle_cache(name), exact=True)
    E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 7, 7), T=9)
    compare((E, H), oracle_cache(name), exact=True)


def test_overlapping_launches_under_perturbed_cta_order(cuda_device, oracle_cache, monkeypatch):
    """The same with pseudo-random sleeps between phases (developer build), which stretch the drain of a launch far into
    the next one; and with the overlap switched off (FDTD_NO_OVERLAP) the result is the same."""
    w, steps = CASES["C2s"]
    for seed, T in ((7, 4), (99, 9), (1234, 17), (5, 33)):
        monkeypatch.setenv("FDTD_DEBUG_DELAY", str(seed))
        E, H, _ = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 15, 7), T=T, variant="dbg")
        compare((E, H), oracle_cache("C2s"), exact=True)
    monkeypatch.delenv("FDTD_DEBUG_DELAY")
    monkeypatch.setenv("FDTD_NO_OVERLAP", "1")
    E, H, _ = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 15, 7), T=9)
    compare((E, H), oracle_cache("C2s"), exact=True)


def test_timing_is_opt_in(cuda_device):
    w, _ = CASES["C1"]
    E, H, sim = binding.run_workload(w, kernel=binding.KERNEL_SYSTOLIC, steps=3)
    with pytest.raises(binding.FdtdError) as e:
        sim.last_step_ms()
    assert e.value.code == binding.ESTATE
    sim.set_timing(True)
    sim.step(5)
    assert sim.last_step_ms() > 0
    sim.close()


# ---- f2: material-index coefficients (fdtd_set_coeff_lut) ------------------------------------------------------------
def test_lut_recipe_expands_to_the_coefficient_arrays():
    """(no GPU needed, but it guards the GPU cases below) the index form of a workload is its array form, bit for bit."""
    for name in ("C2s", "C3s", "allper"):
        w, _ = CASES[name]
        ca, cb = workloads.make_coeffs(w)
        idx, ca_lut, cb_lut = workloads.make_coeff_lut(w)
        for a in range(3):
            assert idx[a].dtype == np.uint8 and int(idx[a].max()) < ca_lut.shape[1]
            assert np.array_equal(ca_lut[a][idx[a]], ca[a]) and np.array_equal(cb_lut[a][idx[a]], cb[a])


LUT_RUNS = [("C2s", "naive", 0), ("C3s", "naive", 0), ("allper", "naive", 0),
            ("C2s", "systolic", 32), ("C2s", "systolic", 5), ("C2s", "systolic", 128), ("C3s", "systolic", 16), ("C3s", "systolic", 7),
            ("allper", "systolic", 5)]


@pytest.mark.parametrize("name,kernel,T", LUT_RUNS)
def test_lut_coefficients_match_oracle_bit_exact(cuda_device, oracle_cache, name, kernel, T):
    """The oracle runs on the expanded arrays (the definition of the table form); the CUDA path reads bytes and a table."""
    import torch
    w, steps = CASES[name]
    dev = torch.device("cuda:0")
    E, H = workloads.make_fields(w, device=dev)
    idx, ca_lut, cb_lut = workloads.make_coeff_lut(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(E, H)
    sim.set_coeff_lut(idx, ca_lut, cb_lut)
    src = workloads.make_source(w)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(binding.KERNEL_NAIVE if kernel == "naive" else binding.KERNEL_SYSTOLIC, (31, 15, 7) if kernel == "systolic" else None, T)
    sim.step(steps // 2)
    sim.step(steps - steps // 2)
    sim.sync()
    sim.close()
    compare(([x.cpu().numpy() for x in E], [x.cpu().numpy() for x in H]), oracle_cache(name), exact=True)


def test_lut_per_component_tables_and_rebinding(cuda_device):
    """Three different index arrays and three different tables (lossy materials), then back to arrays on the same context."""
    import torch
    w = workloads.config(4).scaled((64, 40, 36), steps=60)
    rng = np.random.default_rng(17)
    shape = (w.n[2], w.n[1], w.n[0])
    nmat = 7
    idx_h = [rng.integers(0, nmat, shape).astype(np.uint8) for _ in range(3)]
    ca_lut = rng.uniform(0.97, 1.0, (3, nmat)).astype(np.float32)
    cb_lut = rng.uniform(0.02, 0.25, (3, nmat)).astype(np.float32)
    ca_h = [np.ascontiguousarray(ca_lut[a][idx_h[a]]) for a in range(3)]
    cb_h = [np.ascontiguousarray(cb_lut[a][idx_h[a]]) for a in range(3)]
    E, H = workloads.make_fields(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca_h, cb_h, None)
    src = workloads.make_source(w)
    orc.set_source(src.comp, src.box, src.amp, src.wave)
    orc.step(60)
    dev = torch.device("cuda:0")
    for mode in ("lut", "arrays", "lut-naive"):
        Ed, Hd = workloads.make_fields(w, device=dev)
        sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
        sim.set_fields(Ed, Hd)
        if mode == "arrays":           # bind the table first, then replace it by arrays
            sim.set_coeff_lut([torch.from_numpy(a).to(dev) for a in idx_h], ca_lut, cb_lut)
            sim.set_coeffs([torch.from_numpy(a).to(dev) for a in ca_h], [torch.from_numpy(a).to(dev) for a in cb_h], None)
        else:
            sim.set_coeff_lut([torch.from_numpy(a).to(dev) for a in idx_h], ca_lut, cb_lut)
        sim.set_source(src.comp, src.box, src.amp, src.wave)
        sim.set_kernel(binding.KERNEL_NAIVE if mode == "lut-naive" else binding.KERNEL_SYSTOLIC, None, 0 if mode == "lut-naive" else 16)
        sim.step(60)
        sim.sync()
        sim.close()
        compare(([x.cpu().numpy() for x in Ed], [x.cpu().numpy() for x in Hd]), (E, H), exact=True)


# ---- combinations of the 8(f) rows ------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel,T", [("naive", 0), ("systolic", 16)])
def test_monitor_with_f16_storage(cuda_device, kernel, T):
    """Running DFT of binary16-stored fields: the monitor sees the rounded values, as the oracle's f16-storage build does."""
    import torch
    from oracle.monitor import MonitorOracle
    w, steps = CASES["C2s"]
    wE, wH = _weights(steps, 2, 3)
    r16 = lambda a: a.astype(np.float16).astype(np.float32)
    E, H = workloads.make_fields(w)
    E, H = [r16(a) for a in E], [r16(a) for a in H]
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None, storage="f16")
    src = workloads.make_source(w)
    orc.set_source(src.comp, src.box, src.amp, src.wave)
    mon = MonitorOracle(orc, 1, 30, wE, wH)
    mon.step(steps)
    want = mon.acc.reshape(6, 2, 2, -1)
    dev = torch.device("cuda:0")
    Ed, Hd = workloads.make_fields(w, device=dev)
    Ed, Hd = [a.to(torch.float16) for a in Ed], [a.to(torch.float16) for a in Hd]
    cad, cbd = workloads.make_coeffs(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(Ed, Hd)
    sim.set_coeffs(cad, cbd, None)
    sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(binding.KERNEL_NAIVE if kernel == "naive" else binding.KERNEL_SYSTOLIC, (31, 15, 7) if kernel == "systolic" else None, T)
    acc = torch.zeros((6, 2, 2, want.shape[3]), dtype=torch.float32, device=dev)
    sim.set_monitor(1, 30, wE, wH, acc)
    sim.step(steps)
    sim.sync()
    sim.close()
    assert float(np.abs(want).max()) > 0
    assert np.array_equal(acc.cpu().numpy(), want)
    compare(([x.float().cpu().numpy() for x in Ed], [x.float().cpu().numpy() for x in Hd]), (E, H), exact=True)


def test_monitor_with_lut_and_lut_with_f16(cuda_device, oracle_cache):
    """Monitor on a material-index run (systolic); material indices with binary16 fields: naive runs it, the systolic
    schedule says FDTD_EINVAL."""
    import torch
    from oracle.monitor import MonitorOracle
    w, steps = CASES["C3s"]
    wE, wH = _weights(steps, 1, 5)
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
    src = workloads.make_source(w)
    orc.set_source(src.comp, src.box, src.amp, src.wave)
    mon = MonitorOracle(orc, 2, 19, wE, wH)
    mon.step(steps)
    want = mon.acc.reshape(6, 1, 2, -1)
    dev = torch.device("cuda:0")
    Ed, Hd = workloads.make_fields(w, device=dev)
    idx, ca_lut, cb_lut = workloads.make_coeff_lut(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(Ed, Hd)
    sim.set_coeff_lut(idx, ca_lut, cb_lut)
    sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(binding.KERNEL_SYSTOLIC, (31, 15, 7), 8)
    acc = torch.zeros((6, 1, 2, want.shape[3]), dtype=torch.float32, device=dev)
    sim.set_monitor(2, 19, wE, wH, acc)
    sim.step(steps)
    sim.sync()
    sim.close()
    assert np.array_equal(acc.cpu().numpy(), want)
    compare(([x.cpu().numpy() for x in Ed], [x.cpu().numpy() for x in Hd]), (E, H), exact=True)
    # binary16 fields + material indices
    r16 = lambda a: a.astype(np.float16).astype(np.float32)
    E2, H2 = workloads.make_fields(w)
    E2, H2 = [r16(a) for a in E2], [r16(a) for a in H2]
    orc2 = YeeOracle(w.n, w.d, w.dt, w.boundary, E2, H2, ca, cb, None, storage="f16")
    orc2.set_source(src.comp, src.box, src.amp, src.wave)
    orc2.step(steps)
    for kernel in (binding.KERNEL_NAIVE, binding.KERNEL_SYSTOLIC):
        Ed, Hd = workloads.make_fields(w, device=dev)
        Ed, Hd = [a.to(torch.float16) for a in Ed], [a.to(torch.float16) for a in Hd]
        sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
        sim.set_fields(Ed, Hd)
        sim.set_coeff_lut(idx, ca_lut, cb_lut)
        sim.set_source(src.comp, src.box, src.amp, src.wave)
        if kernel == binding.KERNEL_NAIVE:
            sim.set_kernel(kernel, None, 0)
            sim.step(steps)
            sim.sync()
            compare(([x.float().cpu().numpy() for x in Ed], [x.float().cpu().numpy() for x in Hd]), (E2, H2), exact=True)
        else:
            with pytest.raises(binding.FdtdError) as e:      # rejected when the schedule is chosen, or at the latest by fdtd_step
                sim.set_kernel(kernel, (31, 15, 7), 8)
                sim.step(steps)
            assert e.value.code == binding.EINVAL
        sim.close()
