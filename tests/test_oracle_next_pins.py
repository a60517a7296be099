"""Pins for the oracles of the SURVEY.md 8(f) rows: oracle/absorber.py (f3) and oracle/monitor.py (f4).

Everything here is fixed by physics / mathematics or by a library routine applied to independently recorded data,
never by the oracle functions themselves or by the CUDA path.  Runs without a GPU.
"""
import math

import numpy as np
import pytest

from oracle.absorber import absorber_coeffs, absorber_sigma_max
from oracle.monitor import MonitorOracle, plane_slice
from oracle.yee import PEC, PERIODIC, YeeOracle


def zeros(n, dtype=np.float64):
    return [np.zeros((n[2], n[1], n[0]), dtype) for _ in range(3)]


# ------------------------------------------------------------------------------------------------
# A1  uniform conductivity (order 0, layer = whole domain): a periodic plane wave loses energy at the analytic rate
#     exp(-sigma t / eps) of a weakly conducting medium (textbook: Im w = -sigma / (2 eps) for sigma << w eps).
#     Catches a wrong sign, eps vs 2 eps, or dt missing in (ca, cb).
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("epsr", [1.0, 2.25])
def test_a1_uniform_loss_rate(epsr):
    n, d = (1, 1, 64), (1.0, 1.0, 1.0)
    dt = 0.5
    sigma = 0.004
    shape = (n[2], n[1], n[0])
    eps = [np.full(shape, epsr)] * 3
    # one low layer per axis covering the whole axis would triple sigma: use the z axis only
    ca, cb = absorber_coeffs(n, dt, eps, (0, 0, 0, 0, n[2], 0), (0, 0, 0, 0, sigma, 0), 0, np.float64)
    k = np.arange(n[2], dtype=np.float64)
    kz = 2 * math.pi * 4 / n[2]
    E, H = zeros(n), zeros(n)
    E[0][:, 0, 0] = np.cos(kz * k)                      # E_x(z), standing + travelling mix: energy decay is what is measured
    y = YeeOracle(n, d, dt, (PERIODIC,) * 3, E, H, ca=ca, cb=cb)

    def energy():
        return epsr * float((E[0] ** 2).sum()) + float((H[1] ** 2).sum())
    # average over whole periods to remove the E/H staggering ripple
    w = 2 / dt * math.asin(dt / math.sqrt(epsr) * math.sin(kz / 2))
    per = int(round(2 * math.pi / w / dt))
    y.step(per)
    e0 = np.mean([(y.step(1), energy())[1] for _ in range(per)])
    y.step(10 * per - per)
    e1 = np.mean([(y.step(1), energy())[1] for _ in range(per)])
    rate = -math.log(e1 / e0) / (10 * per * dt)
    assert rate == pytest.approx(sigma / epsr, rel=2e-3)


# ------------------------------------------------------------------------------------------------
# A2  graded layer: round-trip power reflection of a long quadratic layer = the R0 it was designed for
#     (adiabatic limit, Oskooi et al. 2008 [5] PAPER.md:130): pins sigma_max's formula, the (p+1) of the profile
#     integral and where the layer sits.  Without the layer the wall reflects everything.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("order,R0", [(2, 1e-3), (3, 1e-2)])
def test_a2_round_trip_reflection(order, R0):
    nz, L = 700, 160
    n, d = (1, 1, nz), (1.0, 1.0, 1.0)
    dt = 0.5
    smax = absorber_sigma_max(R0, order, 1.0, L, 1.0)
    ca, cb = absorber_coeffs(n, dt, None, (0, 0, 0, 0, 0, L), (0, 0, 0, 0, 0, smax), order, np.float64)
    k = np.arange(nz, dtype=np.float64)
    lam, z0, wid = 24.0, 250.0, 45.0
    kz = 2 * math.pi / lam
    w = 2 / dt * math.asin(dt * math.sin(kz / 2))
    E, H = zeros(n), zeros(n)
    # +z travelling packet: E_x = f(z) at t = 0, H_y = f(z + 1/2 - vp dt/2) (leapfrog staggering), vp = w/kz
    f = lambda z: np.exp(-((z - z0) / wid) ** 2) * np.cos(kz * (z - z0))
    E[0][:, 0, 0] = f(k)
    H[1][:, 0, 0] = f(k + 0.5 - (w / kz) * dt / 2)
    y = YeeOracle(n, d, dt, (PERIODIC, PERIODIC, PEC), E, H, ca=ca, cb=cb)

    def energy(lo, hi):
        return float((E[0][lo:hi] ** 2).sum() + (H[1][lo:hi] ** 2).sum())
    e_in = energy(0, nz - L)
    vg = math.cos(kz / 2) / math.cos(w * dt / 2)
    # to the wall and back to the middle of the clear region
    steps = int(((nz - z0) + (nz - 270.0)) / vg / dt)
    y.step(steps)
    e_back = energy(0, nz - L)
    R = e_back / e_in
    assert R == pytest.approx(R0, rel=0.15)
    # and with sigma_max = 0 the PEC wall returns everything
    E2, H2 = zeros(n), zeros(n)
    E2[0][:, 0, 0] = f(k)
    H2[1][:, 0, 0] = f(k + 0.5 - (w / kz) * dt / 2)
    ca0, cb0 = absorber_coeffs(n, dt, None, (0, 0, 0, 0, 0, L), (0,) * 6, order, np.float64)
    y2 = YeeOracle(n, d, dt, (PERIODIC, PERIODIC, PEC), E2, H2, ca=ca0, cb=cb0)
    y2.step(steps)
    assert float((E2[0][: nz - L] ** 2).sum() + (H2[1][: nz - L] ** 2).sum()) / e_in > 0.95


# ------------------------------------------------------------------------------------------------
# A3  staggering: mirroring the domain maps the low layer on the high layer.  A component staggered along the axis
#     (E_a along a) sits at g + 1/2 and mirrors to index n-1-g; the others sit at g and mirror to n-g.
# ------------------------------------------------------------------------------------------------
def test_a3_mirror_symmetry_of_the_half_cell_offsets():
    n, dt = (20, 14, 12), 0.3
    L, smax = 5, 0.07
    for q in range(3):
        th_lo, th_hi, s_lo, s_hi = [0] * 6, [0] * 6, [0.0] * 6, [0.0] * 6
        th_lo[2 * q], s_lo[2 * q] = L, smax
        th_hi[2 * q + 1], s_hi[2 * q + 1] = L, smax
        ca_lo, cb_lo = absorber_coeffs(n, dt, None, th_lo, s_lo, 2, np.float64)
        ca_hi, cb_hi = absorber_coeffs(n, dt, None, th_hi, s_hi, 2, np.float64)
        ax = 2 - q
        for a in range(3):
            lo = np.moveaxis(ca_lo[a], ax, 0)
            hi = np.moveaxis(ca_hi[a], ax, 0)
            if a == q:
                assert np.array_equal(lo, hi[::-1])
            else:
                assert np.array_equal(lo[1:], hi[:0:-1])
                assert np.all(hi[0] == 1.0)            # coordinate 0 is a full domain away from the high layer
            assert lo.min() < 1.0 and np.all(lo[L + 1:] == 1.0)
            cbl = np.moveaxis(cb_lo[a], ax, 0)
            assert np.all(cbl[L + 1:] == dt)           # vacuum outside the layer: cb = dt, ca = 1


# ------------------------------------------------------------------------------------------------
# A4  hand values on one line, exact rationals (not the generator's own expressions): L = 4, p = 2, smax = 1/2,
#     dt = 1/4, eps = 2:  u = (4 - s)/4, sigma = u^2 / 2, ca = (4 - sigma/4)/(4 + sigma/4), cb = (1/2)/(4 + sigma/4)
# ------------------------------------------------------------------------------------------------
def test_a4_hand_values_and_corner_sum():
    from fractions import Fraction as Fr
    n = (8, 8, 8)
    eps = [np.full((8, 8, 8), 2.0)] * 3
    ca, cb = absorber_coeffs(n, 0.25, eps, (4, 0, 0, 0, 0, 0), (0.5, 0, 0, 0, 0, 0), 2, np.float64)
    for i in range(8):
        for a, s in ((0, Fr(2 * i + 1, 2)), (1, Fr(i))):
            u = max(Fr(0), (4 - s) / 4) if s < 4 else Fr(0)
            sig = u * u / 2
            assert ca[a][3, 2, i] == pytest.approx(float((4 - sig / 4) / (4 + sig / 4)), abs=1e-15)
            assert cb[a][3, 2, i] == pytest.approx(float(Fr(1, 2) / (4 + sig / 4)), abs=1e-15)
    # corner: layers on x-low and y-low add their conductivities
    cax, _ = absorber_coeffs(n, 0.25, eps, (4, 0, 0, 0, 0, 0), (0.5, 0, 0, 0, 0, 0), 2, np.float64)
    cay, _ = absorber_coeffs(n, 0.25, eps, (0, 0, 4, 0, 0, 0), (0, 0, 0.5, 0, 0, 0), 2, np.float64)
    cxy, _ = absorber_coeffs(n, 0.25, eps, (4, 0, 4, 0, 0, 0), (0.5, 0, 0.5, 0, 0, 0), 2, np.float64)
    sig = lambda c: 16.0 * (1 - c) / (1 + c)          # invert ca = (4 - s/4)/(4 + s/4)
    assert np.allclose(sig(cxy[2]), sig(cax[2]) + sig(cay[2]), atol=1e-13)


def test_a5_float32_rounds_like_float64_within_an_ulp():
    n = (12, 10, 9)
    rng = np.random.default_rng(3)
    eps = [rng.uniform(1, 12, (9, 10, 12)).astype(np.float32) for _ in range(3)]
    th, sm = (3, 2, 0, 4, 2, 2), (0.3, 0.2, 0.0, 0.25, 0.1, 0.15)
    c32 = absorber_coeffs(n, 0.2, eps, th, sm, 3, np.float32)
    c64 = absorber_coeffs(n, 0.2, [e.astype(np.float64) for e in eps], th, sm, 3, np.float64)
    for x, y in zip(c32[0] + c32[1], c64[0] + c64[1]):
        assert x.dtype == np.float32
        assert np.abs(x - y).max() < 1e-6


# ------------------------------------------------------------------------------------------------
# M1  the running DFT equals numpy.fft of an independently recorded time series (library routine on recorded data)
# ------------------------------------------------------------------------------------------------
def _random_run(n, boundary, seed, dtype=np.float64):
    rng = np.random.default_rng(seed)
    shape = (n[2], n[1], n[0])
    E = [rng.uniform(-1, 1, shape).astype(dtype) for _ in range(3)]
    H = [rng.uniform(-1, 1, shape).astype(dtype) for _ in range(3)]
    return E, H


@pytest.mark.parametrize("axis,index", [(0, 3), (1, 0), (2, 5)])
def test_m1_running_dft_equals_fft_of_recorded_series(axis, index):
    n, d, dt = (8, 7, 6), (1, 1, 1), 0.4
    nt = 32
    bins = [1, 5, 9]
    tt = np.arange(nt)
    w = np.zeros((nt, len(bins), 2))
    for f, b in enumerate(bins):
        w[:, f, 0] = np.cos(2 * np.pi * b * tt / nt)
        w[:, f, 1] = -np.sin(2 * np.pi * b * tt / nt)
    E, H = _random_run(n, (PERIODIC,) * 3, 5)
    E2, H2 = [a.copy() for a in E], [a.copy() for a in H]
    mon = MonitorOracle(YeeOracle(n, d, dt, (PERIODIC,) * 3, E, H), axis, index, w, w)
    mon.step(nt)
    # independent recording
    y = YeeOracle(n, d, dt, (PERIODIC,) * 3, E2, H2)
    sl = plane_slice(axis, index)
    rec = []
    for _ in range(nt):
        y.step(1)
        rec.append([a[sl].copy() for a in E2 + H2])
    rec = np.array(rec)                                  # (nt, 6, plane)
    F = np.fft.fft(rec, axis=0)
    for f, b in enumerate(bins):
        for c in range(6):
            assert np.allclose(mon.acc[c, f, 0], F[b, c].real, atol=1e-12)
            assert np.allclose(mon.acc[c, f, 1], F[b, c].imag, atol=1e-12)


def test_m1b_e_components_take_wE_and_h_components_take_wH():
    """M1 again with DIFFERENT tables (wE on bins 1, 5, 9; wH on bins 2, 6, 11 and scaled by 3): the E accumulators must
    be the fft bins of wE's frequencies and the H accumulators those of wH's, so a swap of the two tables inside the
    oracle -- which passes every pin that feeds the same table twice -- fails here."""
    n, d, dt = (8, 7, 6), (1, 1, 1), 0.4
    nt = 32
    binsE, binsH, scaleH = [1, 5, 9], [2, 6, 11], 3.0
    tt = np.arange(nt)
    wE, wH = np.zeros((nt, 3, 2)), np.zeros((nt, 3, 2))
    for f in range(3):
        wE[:, f, 0] = np.cos(2 * np.pi * binsE[f] * tt / nt)
        wE[:, f, 1] = -np.sin(2 * np.pi * binsE[f] * tt / nt)
        wH[:, f, 0] = scaleH * np.cos(2 * np.pi * binsH[f] * tt / nt)
        wH[:, f, 1] = -scaleH * np.sin(2 * np.pi * binsH[f] * tt / nt)
    E, H = _random_run(n, (PERIODIC,) * 3, 11)
    E2, H2 = [a.copy() for a in E], [a.copy() for a in H]
    mon = MonitorOracle(YeeOracle(n, d, dt, (PERIODIC,) * 3, E, H), 1, 2, wE, wH)
    mon.step(nt)
    y = YeeOracle(n, d, dt, (PERIODIC,) * 3, E2, H2)
    sl = plane_slice(1, 2)
    rec = []
    for _ in range(nt):
        y.step(1)
        rec.append([a[sl].copy() for a in E2 + H2])
    F = np.fft.fft(np.array(rec), axis=0)
    for f in range(3):
        for c in range(6):
            want = F[binsE[f], c] if c < 3 else scaleH * F[binsH[f], c]
            assert np.allclose(mon.acc[c, f, 0], want.real, atol=1e-11)
            assert np.allclose(mon.acc[c, f, 1], want.imag, atol=1e-11)
            other = scaleH * F[binsH[f], c] if c < 3 else F[binsE[f], c]          # what a swapped oracle would give
            assert not np.allclose(mon.acc[c, f, 0], other.real, atol=1e-3)


# ------------------------------------------------------------------------------------------------
# M2  closed form: a single cavity mode E_z(t) = A cos(w t) -> sum_t cos(w (t+1) dt) e^{-i W (t+1) dt} (geometric sums)
# ------------------------------------------------------------------------------------------------
def test_m2_cavity_mode_geometric_sum():
    n, d = (16, 12, 4), (1.0, 1.0, 1.0)
    dt = 0.5 / math.sqrt(3)
    k, j, i = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    E, H = zeros(n), zeros(n)
    mode = np.sin(np.pi * i / n[0]) * np.sin(np.pi * j / n[1])
    lam = (2 * math.sin(math.pi / (2 * n[0]))) ** 2 + (2 * math.sin(math.pi / (2 * n[1]))) ** 2
    w = math.acos(1 - dt * dt * lam / 2) / dt
    # run from (E^0, H^{1/2}) = (mode, 0): the amplitude is A cos(w t) + B sin(w t) by the three-term recurrence of P1
    E[2][:] = mode
    nt = 50
    W = 0.21
    tt = np.arange(nt)
    wt = np.zeros((nt, 1, 2))
    wt[:, 0, 0] = np.cos(W * (tt + 1) * dt)
    wt[:, 0, 1] = -np.sin(W * (tt + 1) * dt)
    y = YeeOracle(n, d, dt, (PEC, PEC, PERIODIC), E, H)
    mon = MonitorOracle(y, 2, 1, wt, wt)
    mon.step(nt)
    # the mode amplitude a(t) obeys a(t+1) + a(t-1) = 2 cos(w dt) a(t) with a(0) = a(1) = 1 (H^{1/2} = 0, so the first
    # E half-step changes nothing)  =>  a(t) = A cos(w t dt) + B sin(w t dt)
    a1 = 1.0
    A = 1.0
    B = (a1 - math.cos(w * dt)) / math.sin(w * dt)
    z = np.exp(-1j * W * dt)
    p, q = np.exp(1j * w * dt), np.exp(-1j * w * dt)
    geo = lambda r: r * z * (1 - (r * z) ** nt) / (1 - r * z)             # sum_{t=1..nt} (r z)^t
    expect = (A / 2) * (geo(p) + geo(q)) + (B / 2j) * (geo(p) - geo(q))
    got = mon.acc[2, 0, 0] + 1j * mon.acc[2, 0, 1]
    assert np.allclose(got, expect * mode[1], atol=1e-12)


def test_m3_weights_outside_the_table_are_skipped_and_float32_is_separately_rounded():
    n, d, dt = (6, 5, 4), (1, 1, 1), 0.4
    E, H = _random_run(n, (PEC,) * 3, 9, np.float32)
    w = np.random.default_rng(1).uniform(-1, 1, (5, 2, 2)).astype(np.float32)
    y = YeeOracle(n, d, dt, (PEC,) * 3, E, H)
    mon = MonitorOracle(y, 0, 2, w, w)
    mon.step(5)
    snap = mon.acc.copy()
    mon.step(3)                                           # t >= nt: nothing accumulates
    assert np.array_equal(snap, mon.acc)
    assert mon.acc.dtype == np.float32


# ------------------------------------------------------------------------------------------------
# f1: f16 field storage with f32 arithmetic (oracle build "_h16")
# ------------------------------------------------------------------------------------------------
def _h16_inputs(n, seed, boundary, coef):
    rng = np.random.default_rng(seed)
    shape = (n[2], n[1], n[0])
    r16 = lambda a: a.astype(np.float16).astype(np.float32)
    E = [r16(rng.uniform(-1, 1, shape)) for _ in range(3)]
    H = [r16(rng.uniform(-1, 1, shape)) for _ in range(3)]
    ca = [rng.uniform(0.9, 1.0, shape).astype(np.float32) for _ in range(3)] if coef else None
    cb = [rng.uniform(0.05, 0.3, shape).astype(np.float32) for _ in range(3)] if coef else None
    return E, H, ca, cb


@pytest.mark.parametrize("boundary", [(PEC, PEC, PEC), (PERIODIC, PEC, PERIODIC)])
@pytest.mark.parametrize("coef", [False, True])
def test_h1_each_half_step_is_the_f32_half_step_rounded_by_numpy(boundary, coef):
    """One half-step of the f16-storage build = the (pinned) f32 half-step followed by numpy's own binary16 rounding."""
    n, d, dt = (9, 7, 6), (1.0, 0.8, 1.3), 0.3
    E, H, ca, cb = _h16_inputs(n, 11, boundary, coef)
    E2, H2 = [a.copy() for a in E], [a.copy() for a in H]
    y16 = YeeOracle(n, d, dt, boundary, E, H, ca, cb, db=(0.3, 0.25, 0.2), storage="f16")
    y32 = YeeOracle(n, d, dt, boundary, E2, H2, ca, cb, db=(0.3, 0.25, 0.2))
    y16.e_half()
    y32.e_half()
    for a, b in zip(E, E2):
        assert np.array_equal(a, b.astype(np.float16).astype(np.float32))
    assert any(not np.array_equal(a, b) for a, b in zip(E, E2))          # the rounding does something
    for a, b in zip(E, E2):                                                # continue from the rounded state on both sides
        b[:] = a
    y16.h_half()
    y32.h_half()
    for a, b in zip(H, H2):
        assert np.array_equal(a, b.astype(np.float16).astype(np.float32))


def test_h2_exactly_representable_run_equals_the_f32_run():
    """Small dyadic data, d = 1, dt = 1/2: every intermediate value of a few steps is a binary16 number, so storage
    rounding is the identity and the two builds agree bit for bit (and the f32 build is pinned by P9's exact rationals)."""
    n, d, dt = (6, 5, 4), (1.0, 1.0, 1.0), 0.5
    rng = np.random.default_rng(2)
    shape = (n[2], n[1], n[0])
    E = [rng.integers(-4, 5, shape).astype(np.float32) / 4 for _ in range(3)]
    H = [rng.integers(-4, 5, shape).astype(np.float32) / 4 for _ in range(3)]
    E2, H2 = [a.copy() for a in E], [a.copy() for a in H]
    amp = np.ones((1, 1, 1), np.float32)
    wave = np.array([0.5, 0.25, -0.5], np.float32)
    y16 = YeeOracle(n, d, dt, (PEC, PERIODIC, PEC), E, H, storage="f16")
    y32 = YeeOracle(n, d, dt, (PEC, PERIODIC, PEC), E2, H2)
    for y in (y16, y32):
        y.set_source(2, (2, 2, 1, 1, 1, 1), amp, wave)
        y.step(3)          # values stay multiples of 2^-8 below 2^4: 11 significant bits suffice
    for a, b in zip(E + H, E2 + H2):
        assert np.array_equal(a, b)


def test_h3_source_add_is_rounded_and_error_stays_at_the_binary16_level():
    n, d = (12, 10, 8), (1.0, 1.0, 1.0)
    dt = 0.5 / math.sqrt(3)
    E, H, _, _ = _h16_inputs(n, 5, (PEC,) * 3, False)
    E64, H64 = [a.astype(np.float64) for a in E], [a.astype(np.float64) for a in H]
    amp = np.full((1, 1, 1), 0.3337, np.float32)
    wave = np.array([0.7771], np.float32)
    y16 = YeeOracle(n, d, dt, (PEC,) * 3, E, H, storage="f16")
    y16.set_source(0, (5, 5, 4, 1, 1, 1), amp, wave)
    before = [a.copy() for a in E]
    Hb = [a.copy() for a in H]
    y16.step(1)
    # re-derive E_x at the source cell: f32 update rounded, then f32 add of the rounded product, rounded again
    ye = YeeOracle(n, d, dt, (PEC,) * 3, before, Hb)
    ye.e_half()
    e1 = np.float32(np.float16(before[0][4, 5, 5]))
    inj = np.float32(amp[0, 0, 0] * wave[0])
    assert E[0][4, 5, 5] == np.float32(np.float16(e1 + inj))
    for a in E + H:
        assert np.array_equal(a, a.astype(np.float16).astype(np.float32))
    # 40 steps against f64: relative error of a few binary16 ulps per step, nothing worse
    y64 = YeeOracle(n, d, dt, (PEC,) * 3, E64, H64)
    y64.set_source(0, (5, 5, 4, 1, 1, 1), amp.astype(np.float64), wave.astype(np.float64))
    y64.step(1)
    y16.step(40)
    y64.step(40)
    scale = max(float(np.abs(a).max()) for a in E64 + H64)
    err = max(float(np.abs(a - b).max()) for a, b in zip(E + H, E64 + H64))
    assert 1e-5 * scale < err < 40 * 2.0 ** -10 * scale
