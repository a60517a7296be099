"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Bar (BASELINE.json north_star): max|GPU - oracle| <= 1e-5 * max|field| for the default build, and
BIT-EXACT for the -fmad=false build ("the systolic order does not change per-cell arithmetic").
Floats are compared with == (so -0 == +0; reading #13)."""
import os

import numpy as np
import pytest

from oracle.yee import YeeOracle
from paper_2502_20610_b200 import binding, workloads
from paper_2502_20610_b200.workloads import PEC, PERIODIC

pytestmark = pytest.mark.gpu
TOL = 1e-5


def oracle_run(w, steps):
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        orc.set_source(src.comp, src.box, src.amp, src.wave)
    orc.step(steps)
    return E, H


def gpu_run(w, steps, kernel, tile=None, T=0, variant="nofma"):
    E, H, sim = binding.run_workload(w, kernel=kernel, tile=tile, T=T, steps=steps, variant=variant)
    info = sim.get_kernel()
    sim.close()
    return [x.cpu().numpy() for x in E], [x.cpu().numpy() for x in H], info


def compare(got, want, exact):
    scale = max(float(np.abs(x).max()) for x in want[0] + want[1])
    worst = 0.0
    for g3, w3 in zip(got, want):
        for g, w in zip(g3, w3):
            assert np.all(np.isfinite(g))
            if exact:
                assert np.array_equal(g, w), f"not bit-exact: max diff {np.abs(g - w).max():.3e} at {np.unravel_index(np.abs(g - w).argmax(), g.shape)}"
            worst = max(worst, float(np.abs(g.astype(np.float64) - w.astype(np.float64)).max()))
    assert worst <= TOL * max(scale, 1e-30), f"max|GPU-oracle| = {worst:.3e} > {TOL} * {scale:.3e}"
    return worst / max(scale, 1e-30)


# reduced-size versions of every BASELINE config (same recipe, several tiles per axis, ragged tails)
CASES = {
    "C1": (workloads.config(0), 100),
    "C2s": (workloads.config(1).scaled((72, 60, 52), steps=150), 150),
    "C3s": (workloads.config(2).scaled((64, 56, 40), steps=120), 120),
    "C4s": (workloads.config(3, 128).scaled((100, 96, 90), steps=40), 40),
    "C5s": (workloads.config(4).scaled((48, 40, 36), steps=90), 90),
    "ragged": (workloads.Workload("ragged", (37, 29, 23), (1, 0.8, 1.3), (PEC, PERIODIC, PEC), 50, "uniform", "lossy", "dipole"), 50),
    "allper": (workloads.Workload("allper", (24, 20, 12), (1, 1, 1), (PERIODIC,) * 3, 30, "uniform", "blocks", "sheet"), 30),
}


@pytest.fixture(scope="module")
def oracle_results():
    cache = {}

    def get(name):
        if name not in cache:
            w, steps = CASES[name]
            cache[name] = oracle_run(w, steps)
        return cache[name]
    return get


@pytest.mark.parametrize("variant", ["nofma", "fma"])
@pytest.mark.parametrize("name", list(CASES))
def test_naive_matches_oracle(cuda_device, oracle_results, name, variant):
    w, steps = CASES[name]
    E, H, _ = gpu_run(w, steps, binding.KERNEL_NAIVE, variant=variant)
    compare((E, H), oracle_results(name), exact=(variant == "nofma"))


SYS_RUNS = [
    # name, tile, T
    ("C1", (31, 15, 15), 8), ("C1", (15, 15, 15), 25), ("C1", (7, 7, 7), 16),
    ("C2s", (31, 15, 7), 32), ("C2s", (15, 15, 15), 9), ("C2s", (7, 7, 7), 20),
    ("C3s", (31, 15, 7), 16), ("C3s", (15, 7, 7), 11),
    ("C4s", (31, 15, 15), 13), ("C4s", (31, 15, 7), 40),
    ("C5s", (31, 15, 7), 32), ("C5s", (15, 7, 7), 7),
    ("ragged", (15, 7, 7), 6), ("ragged", (7, 7, 7), 50),
    ("allper", (7, 7, 7), 5),
]


@pytest.mark.parametrize("variant", ["nofma", "fma"])
@pytest.mark.parametrize("name,tile,T", SYS_RUNS)
def test_systolic_matches_oracle(cuda_device, oracle_results, name, tile, T, variant):
    w, steps = CASES[name]
    E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=tile, T=T, variant=variant)
    assert info["which"] == binding.KERNEL_SYSTOLIC and info["tile"] == tile and info["T"] == T
    compare((E, H), oracle_results(name), exact=(variant == "nofma"))


# the register-resident kernel (tile 31x15x7) on every reduced config, several temporal depths, incl. T > tile width
REG_RUNS = [("C1", 8), ("C1", 33), ("C2s", 5), ("C2s", 32), ("C3s", 16), ("C3s", 7), ("C4s", 40), ("C4s", 3),
            ("C5s", 32), ("C5s", 1), ("ragged", 6), ("ragged", 50), ("allper", 5)]


@pytest.mark.parametrize("name,T", REG_RUNS)
def test_register_kernel_matches_oracle(cuda_device, oracle_results, name, T):
    """FDTD_KERNEL_SYSTOLIC_REG: the cp.async-staged register kernel (any wall type, any nx)."""
    w, steps = CASES[name]
    E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC_REG, tile=(31, 15, 7), T=T, variant="nofma")
    assert info["smem"] < 200 * 1024 and info["T"] == T
    compare((E, H), oracle_results(name), exact=True)


# the TMA-staged kernel (what FDTD_KERNEL_SYSTOLIC runs on PEC grids with nx % 4 == 0): every PEC config, several
# temporal depths incl. T = 1, T > tile width and T > grid size; both builds
TMA_RUNS = [("C1", 8), ("C1", 33), ("C1", 100), ("C2s", 5), ("C2s", 32), ("C2s", 1), ("C4s", 40), ("C4s", 3), ("C5s", 32), ("C5s", 2),
            ("C5s", 90)]


@pytest.mark.parametrize("variant", ["nofma", "fma"])
@pytest.mark.parametrize("name,T", TMA_RUNS)
def test_tma_kernel_matches_oracle(cuda_device, oracle_results, name, T, variant):
    w, steps = CASES[name]
    assert all(b == PEC for b in w.boundary) and w.n[0] % 4 == 0
    E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 15, 7), T=T, variant=variant)
    assert info["smem"] in (229632, 147456) and info["T"] == T     # the TMA kernel, not the cp.async kernel
    compare((E, H), oracle_results(name), exact=(variant == "nofma"))


@pytest.mark.parametrize("name,T", [("C2s", 32), ("C3s", 16), ("C1", 8)])
def test_shared_memory_kernel_same_tile(cuda_device, oracle_results, name, T):
    """FDTD_KERNEL_SYSTOLIC_SMEM: the first implementation (whole subdomain in shared memory), same schedule."""
    w, steps = CASES[name]
    E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC_SMEM, tile=(31, 15, 7), T=T, variant="nofma")
    assert info["which"] == binding.KERNEL_SYSTOLIC_SMEM
    compare((E, H), oracle_results(name), exact=True)


def test_systolic_default_configuration(cuda_device, oracle_results):
    # whatever tile / depth the library picks by itself
    for name in ("C1", "C2s"):
        w, steps = CASES[name]
        E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, variant="nofma")
        assert info["tiles"] > 1
        compare((E, H), oracle_results(name), exact=True)


def test_systolic_under_perturbed_cta_order(cuda_device, oracle_results, monkeypatch):
    """Pseudo-random sleeps between phases reorder the CTAs; the flag protocol must keep the result bit-exact.
    (Fault injection lives in the developer build only: variant "dbg" = -fmad=false -DFDTD_DEBUG.)"""
    w, steps = CASES["C2s"]
    for seed in (11, 12345):
        monkeypatch.setenv("FDTD_DEBUG_DELAY", str(seed))
        E, H, _ = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(7, 7, 7), T=10, variant="dbg")
        compare((E, H), oracle_results("C2s"), exact=True)
        E, H, _ = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 15, 7), T=12, variant="dbg")
        compare((E, H), oracle_results("C2s"), exact=True)


def test_step_splitting_and_time(cuda_device, oracle_results):
    """fdtd_step(a); fdtd_step(b) == fdtd_step(a+b): launch boundaries leave every cell at the same time level (a11)."""
    import torch
    w, steps = CASES["C2s"]
    dev = torch.device("cuda:0")
    E, H = workloads.make_fields(w, device=dev)
    ca, cb = workloads.make_coeffs(w, device=dev)
    src = workloads.make_source(w)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E, H)
    sim.set_coeffs(ca, cb)
    sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(binding.KERNEL_SYSTOLIC, (15, 15, 15), 16)
    for part in (1, 37, 0, 16, steps - 54):
        sim.step(part)
    sim.sync()
    assert sim.time == steps and sim.counters()["steps"] == steps
    compare(([x.cpu().numpy() for x in E], [x.cpu().numpy() for x in H]), oracle_results("C2s"), exact=True)
    sim.close()


def test_host_buffer_round_trip(cuda_device, oracle_results):
    """The end-to-end entry: host arrays in (fdtd_load_fields), host arrays out (fdtd_get_fields)."""
    import torch
    w, steps = CASES["C1"]
    dev = torch.device("cuda:0")
    Eh, Hh = workloads.make_fields(w)
    E = [torch.empty(x.shape, dtype=torch.float32, device=dev) for x in Eh]
    H = [torch.empty(x.shape, dtype=torch.float32, device=dev) for x in Hh]
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E, H)
    sim.load_fields(Eh, Hh)
    sim.step(steps)
    Eo = [np.empty_like(x) for x in Eh]
    Ho = [np.empty_like(x) for x in Hh]
    sim.get_fields(Eo, Ho)
    compare((Eo, Ho), oracle_results("C1"), exact=True)
    sim.close()


def test_api_errors(cuda_device):
    import torch
    with pytest.raises(binding.FdtdError) as e:
        binding.Fdtd((0, 8, 8), (1, 1, 1), 0.1, (0, 0, 0))
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.FdtdError):
        binding.Fdtd((8, 8, 8), (1, -1, 1), 0.1, (0, 0, 0))
    sim = binding.Fdtd((8, 8, 8), (1, 1, 1), 0.1, (0, 0, 0))
    with pytest.raises(binding.FdtdError) as e:
        sim.step(1)
    assert e.value.code == binding.ESTATE
    with pytest.raises(binding.FdtdError) as e:
        sim.set_kernel(binding.KERNEL_SYSTOLIC, (5, 5, 5), 4)     # not a built tile shape
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.FdtdError) as e:
        sim.set_source(2, (7, 7, 7, 2, 1, 1), np.ones(2, np.float32), np.ones(3, np.float32))   # box leaves the grid
    assert e.value.code == binding.EINVAL
    t = [torch.zeros((8, 8, 8), dtype=torch.float32, device="cuda:0") for _ in range(6)]
    sim.set_fields(t[:3], t[3:])
    sim.step(0)
    sim.sync()
    assert all(float(x.abs().max()) == 0.0 for x in t)              # zero stays zero (P11)
    sim.step(3)
    sim.sync()
    assert all(float(x.abs().max()) == 0.0 for x in t)
    sim.close()
    # a periodic ring that cannot be resident at once is refused, not deadlocked
    big = binding.Fdtd((4096, 64, 8), (1, 1, 1), 0.1, (0, 1, 0))
    with pytest.raises(binding.FdtdError) as e:
        big.set_kernel(binding.KERNEL_SYSTOLIC, (7, 7, 7), 4)
    assert e.value.code == binding.EINVAL
    big.close()


@pytest.mark.parametrize("variant", ["nofma"])
def test_full_size_config2_systolic_vs_oracle_and_naive(cuda_device, variant):
    """BASELINE configs[1] at its full 256^3 size in the launch configuration bench.py times (library defaults),
    shortened to 96 steps (the oracle needs ~10 s for them): bit-exact against the oracle."""
    w = workloads.config(1)
    steps = 96
    want = oracle_run(w, steps)
    E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, variant=variant)
    assert info["tiles"] > 148
    compare((E, H), want, exact=True)
    E2, H2, _ = gpu_run(w, steps, binding.KERNEL_NAIVE, variant=variant)
    compare((E2, H2), want, exact=True)


def _window_oracle_check(w, s, win, origins, need_free):
    """Parity at sizes the host cannot hold: after s steps a win^3 window depends only on inputs within
    s cells, so the oracle runs on a regenerated (win+2s)^3 sub-box (true walls where the box meets them, any wall
    elsewhere) and the inner window must match the device result bit for bit."""
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()           # earlier tests leave tens of GB in torch's caching allocator
    free, total = torch.cuda.mem_get_info()
    if free < need_free:
        assert total < 170e9, f"only {free / 1e9:.0f} GB free of {total / 1e9:.0f} GB: something holds device memory"
        pytest.skip(f"needs {need_free / 1e9:.0f} GB of free device memory (device has {total / 1e9:.0f} GB)")
    dev = torch.device("cuda:0")
    E, H = workloads.make_fields(w, device=dev)
    ca, cb = workloads.make_coeffs(w, device=dev)
    src = workloads.make_source(w)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E, H)
    if ca is not None:
        sim.set_coeffs(ca, cb)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(binding.KERNEL_SYSTOLIC, None, s)
    info = sim.get_kernel()
    assert info["smem"] in (229632, 147456) and info["tiles"] > 100000
    sim.step(s)
    sim.sync()
    nx, ny, nz = w.n
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
            assert np.array_equal(got, o[sl_o]), f"window at {(i0, j0, k0)}: max diff {np.abs(got - o[sl_o]).max():.3e}"
    return E, H, sim


def test_full_size_config5_window_oracle(cuda_device):
    """BASELINE configs[4] at its full 1536x1536x768 (81 GiB resident, 64-bit offsets, 662k tiles per launch).  Windows:
    low corner, high corner, the source, and a point where tile seams of all three axes meet."""
    w = workloads.config(4)
    nx, ny, nz = w.n
    win = 24
    origins = [(0, 0, 0), (nx - win, ny - win, nz - win), (nx // 2 - win // 2, ny // 2 - win // 2, nz // 2 - win // 2),
               (31 * 20 - win // 2, 15 * 40 - win // 2, 7 * 50 - win // 2)]
    E, H, sim = _window_oracle_check(w, 32, win, origins, 100e9)
    # the pulse has reached the source window (the comparison above is not 0 == 0 there)
    assert float(E[2][nz // 2 - 2:nz // 2 + 2, ny // 2 - 2:ny // 2 + 2, nx // 2 - 2:nx // 2 + 2].abs().max()) > 0
    sim.close()


def test_full_size_config4_1024_window_oracle(cuda_device):
    """The largest cube of the BASELINE configs[3] sweep (1024^3 random fields, uniform coefficients, 26 GB): windows at
    the low corner, at the high walls and across tile seams in the middle, 32 steps in one launch."""
    w = workloads.config(3, 1024)
    win = 24
    origins = [(0, 0, 0), (1024 - win, 1024 - win, 1024 - win), (31 * 16 - 10, 15 * 34 - 10, 7 * 73 - 10)]
    _, _, sim = _window_oracle_check(w, 32, win, origins, 40e9)
    sim.close()


# degenerate grids through the TMA kernel: smaller than one tile, one cell thick, exactly one box, ragged beyond a box
TINY = [(4, 4, 4), (8, 1, 1), (4, 1, 9), (32, 16, 8), (36, 3, 2), (64, 17, 5), (128, 2, 31)]


@pytest.mark.parametrize("n", TINY)
@pytest.mark.parametrize("coeffs", ["none", "lossy"])
def test_tma_kernel_degenerate_grids(cuda_device, n, coeffs):
    w = workloads.Workload(f"tiny{n}", n, (1.0, 0.7, 1.2), (PEC,) * 3, 23, "uniform", coeffs, "dipole")
    steps = 23
    want = oracle_run(w, steps)
    for T in (1, 4, 23):
        E, H, info = gpu_run(w, steps, binding.KERNEL_SYSTOLIC, tile=(31, 15, 7), T=T, variant="nofma")
        assert info["smem"] in (229632, 147456)
        compare((E, H), want, exact=True)
    E, H, _ = gpu_run(w, steps, binding.KERNEL_NAIVE, variant="nofma")
    compare((E, H), want, exact=True)


def test_zero_steps_and_repeated_short_calls(cuda_device, oracle_results):
    """fdtd_step(0) is a no-op; many one-step calls (one launch each, T = 1) equal one long call."""
    import torch
    w, steps = CASES["C5s"]
    dev = torch.device("cuda:0")
    E, H = workloads.make_fields(w, device=dev)
    ca, cb = workloads.make_coeffs(w, device=dev)
    src = workloads.make_source(w)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary, variant="nofma")
    sim.set_fields(E, H)
    sim.set_coeffs(ca, cb)
    sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.step(0)
    for _ in range(steps):
        sim.step(1)
    sim.sync()
    assert sim.time == steps
    compare(([x.cpu().numpy() for x in E], [x.cpu().numpy() for x in H]), oracle_results("C5s"), exact=True)
    sim.close()
