"""GPU parity, third set: the 8(f) rows at the FULL sizes bench.py times them on.

The feature suites of test_gpu_next.py stop at 100x96x90 cells.  bench.py's sweep times binary16 storage on config 2,
1024^3 and config 5 and material-index coefficients on configs 2 and 3, all at full size and at the library's default
launch depth; their narrower TMA boxes (40-wide f16 rows, 48-wide index rows) and the padded copy with byte arrays had
never met large coordinates.  Here:

  * binary16 storage on config 2 (256^3 x 200 steps), whole grid, against the oracle's f16-storage build;
  * binary16 storage on 1024^3 and on config 5's grid (random fields so that every window holds data): windows against the
    same oracle on regenerated sub-boxes (a win^3 window after s steps depends on inputs within s cells only);
  * material indices on config 2 (256^3 x 200) and on config 3 (512x512x256 x 160, periodic x: the padded working copy
    with one-byte arrays), whole grid, against the f32 oracle on the expanded arrays;
  * one running-DFT monitor plane on config 2 at 256^3.

All through the C ABI with the library's own choice of tile and depth, product build, bit-exact."""
import gc
from dataclasses import replace

import numpy as np
import pytest

from oracle.yee import YeeOracle
from paper_2502_20610_b200 import binding, workloads
from tests.test_gpu_next import _h16_gpu, _h16_oracle, _weights
from tests.test_gpu_parity import compare, oracle_run

pytestmark = pytest.mark.gpu


def _free_device_memory(need, what):
    import torch
    gc.collect()
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info()
    if free < need:
        assert total < 170e9, f"only {free / 1e9:.0f} GB free of {total / 1e9:.0f} GB: something holds device memory"
        pytest.skip(f"{what} needs {need / 1e9:.0f} GB of free device memory (device has {total / 1e9:.0f} GB)")


def test_f16_storage_config2_full_size(cuda_device):
    w = workloads.config(1)
    steps = 200
    want = _h16_oracle(w, steps)
    assert max(float(np.abs(a).max()) for a in want[0] + want[1]) > 0
    E, H, info = _h16_gpu(w, steps, binding.KERNEL_SYSTOLIC, None, 0)
    assert info["which"] == binding.KERNEL_SYSTOLIC and info["T"] >= 64 and steps > info["T"]
    compare((E, H), want, exact=True)


def _f16_windows(w, steps, win, origins, need_free):
    """binary16 run of workload w on the device (library defaults), then the f16-storage oracle on (win + 2 steps)^3
    sub-boxes regenerated from the seed; the inner windows must agree bit for bit and must hold data."""
    import torch
    _free_device_memory(need_free, w.name)
    dev = torch.device("cuda:0")
    E, H = workloads.make_fields(w, device=dev)
    E, H = [a.to(torch.float16) for a in E], [a.to(torch.float16) for a in H]
    torch.cuda.empty_cache()
    ca, cb = workloads.make_coeffs(w, device=dev)
    src = workloads.make_source(w)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(E, H)
    if ca is not None:
        sim.set_coeffs(ca, cb, None)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    info = sim.get_kernel()
    assert info["which"] == binding.KERNEL_SYSTOLIC and steps > info["T"] >= 64
    sim.step(steps)
    sim.sync()
    nx, ny, nz = w.n
    s = steps
    r16 = lambda a: a.astype(np.float16).astype(np.float32)
    for (i0, j0, k0) in origins:
        lo = [max(0, i0 - s), max(0, j0 - s), max(0, k0 - s)]
        hi = [min(nx, i0 + win + s), min(ny, j0 + win + s), min(nz, k0 + win + s)]
        box = (lo[0], lo[1], lo[2], hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2])
        Eo, Ho = workloads.make_fields(w, window=box)
        Eo, Ho = [r16(a) for a in Eo], [r16(a) for a in Ho]
        cao, cbo = workloads.make_coeffs(w, window=box)
        orc = YeeOracle(box[3:], w.d, w.dt, w.boundary, Eo, Ho, cao, cbo, None, storage="f16")
        if src is not None:
            sb = src.box
            if all(lo[a] <= sb[a] and sb[a] + sb[3 + a] <= hi[a] for a in range(3)):
                orc.set_source(src.comp, (sb[0] - lo[0], sb[1] - lo[1], sb[2] - lo[2], sb[3], sb[4], sb[5]), src.amp, src.wave)
        orc.step(s)
        sl_o = (slice(k0 - lo[2], k0 - lo[2] + win), slice(j0 - lo[1], j0 - lo[1] + win), slice(i0 - lo[0], i0 - lo[0] + win))
        sl_g = (slice(k0, k0 + win), slice(j0, j0 + win), slice(i0, i0 + win))
        for g, o in zip(E + H, Eo + Ho):
            got = g[sl_g].float().cpu().numpy()
            assert float(np.abs(o[sl_o]).max()) > 0.0, f"window at {(i0, j0, k0)} compares zero with zero"
            assert np.array_equal(got, o[sl_o]), f"window at {(i0, j0, k0)}: max diff {np.abs(got - o[sl_o]).max():.3e}"
    sim.close()
    del E, H, ca, cb
    gc.collect()
    torch.cuda.empty_cache()


def test_f16_storage_1024_windows(cuda_device):
    w = workloads.config(3, 1024)
    win = 24
    _f16_windows(w, 160, win, [(0, 0, 0), (1024 - win, 1024 - win, 1024 - win), (31 * 16 - 10, 15 * 34 - 10, 7 * 73 - 10)], 60e9)


def test_f16_storage_config5_grid_windows(cuda_device):
    """Config 5's grid, coefficients and source with seeded random initial fields (the config's own zero fields would leave
    every window but the source's empty after 160 steps)."""
    w = replace(workloads.config(4), fields="uniform", name="C5-lossy-random-fields-f16")
    nx, ny, nz = w.n
    win = 24
    _f16_windows(w, 160, win, [(0, 0, 0), (nx - win, ny - win, nz - win), (31 * 20 - 12, 15 * 40 - 12, 7 * 50 - 12)], 125e9)


def _lut_gpu(w, steps):
    import torch
    dev = torch.device("cuda:0")
    E, H = workloads.make_fields(w, device=dev)
    idx, ca_lut, cb_lut = workloads.make_coeff_lut(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(E, H)
    sim.set_coeff_lut(idx, ca_lut, cb_lut)
    src = workloads.make_source(w)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    info = sim.get_kernel()
    assert info["which"] == binding.KERNEL_SYSTOLIC
    sim.step(steps)
    sim.sync()
    sim.close()
    return [x.cpu().numpy() for x in E], [x.cpu().numpy() for x in H], info


def test_material_indices_config2_full_size(cuda_device):
    w = workloads.config(1)
    steps = 200
    want = oracle_run(w, steps)
    assert max(float(np.abs(a).max()) for a in want[0] + want[1]) > 0
    E, H, info = _lut_gpu(w, steps)
    assert steps > info["T"] >= 64
    compare((E, H), want, exact=True)


def test_material_indices_config3_full_size_padded_copy(cuda_device):
    w = workloads.config(2)
    steps = 160
    want = oracle_run(w, steps)
    assert max(float(np.abs(a).max()) for a in want[0] + want[1]) > 0
    E, H, info = _lut_gpu(w, steps)
    assert steps > info["T"]                       # several launches: the ghost zones are refilled in between
    compare((E, H), want, exact=True)


def test_monitor_plane_config2_full_size(cuda_device):
    import torch
    from oracle.monitor import MonitorOracle
    w = workloads.config(1)
    steps, F, axis, index = 200, 2, 2, w.n[2] // 2 + 3
    wE, wH = _weights(steps, F, 1)
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None)
    src = workloads.make_source(w)
    orc.set_source(src.comp, src.box, src.amp, src.wave)
    mon = MonitorOracle(orc, axis, index, wE, wH)
    mon.step(steps)
    want = mon.acc.reshape(6, F, 2, -1)
    assert float(np.abs(want).max()) > 0

    dev = torch.device("cuda:0")
    Ed, Hd = workloads.make_fields(w, device=dev)
    cad, cbd = workloads.make_coeffs(w, device=dev)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(Ed, Hd)
    sim.set_coeffs(cad, cbd, None)
    sim.set_source(src.comp, src.box, src.amp, src.wave)
    acc = torch.zeros((6, F, 2, want.shape[3]), dtype=torch.float32, device=dev)
    sim.set_monitor(axis, index, wE, wH, acc)
    info = sim.get_kernel()
    assert info["which"] == binding.KERNEL_SYSTOLIC and steps > info["T"] >= 64
    sim.step(steps)
    sim.sync()
    sim.close()
    got = acc.cpu().numpy()
    assert np.array_equal(got, want), f"monitor differs: max {np.abs(got - want).max():.3e}"
    compare(([x.cpu().numpy() for x in Ed], [x.cpu().numpy() for x in Hd]), (E, H), exact=True)
