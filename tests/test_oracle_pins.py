"""Pins for the CPU oracle (oracle/yee_oracle.c): everything here is fixed by the paper or by
mathematics, never by the oracle itself or by the CUDA path.  Runs without a GPU.

Pin numbering follows SURVEY.md 8(c): P1 cavity eigenfrequency, P2 plane-wave dispersion,
P3 div H, P4 div D, P5 leapfrog energy, P6 lossy recurrence, P7 magic time step,
P8 cyclic-permutation symmetry, P9 hand-expanded 4^3, P11 zero/static, plus source pins.
"""
import math
import os
from fractions import Fraction as Fr

import numpy as np
import pytest

from oracle.yee import PEC, PERIODIC, YeeOracle
from tests.bruteforce import BruteYee, to_arrays

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "yee_4x4x4_worked_example.txt")


def zeros(n, dtype=np.float64):
    return [np.zeros((n[2], n[1], n[0]), dtype) for _ in range(3)]


def grids(n):
    k, j, i = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    return i.astype(np.float64), j.astype(np.float64), k.astype(np.float64)


def rand_fields(n, seed, dtype, boundary=(PEC,) * 3, zero_tan=True):
    rng = np.random.default_rng(seed)
    i, j, k = grids(n)
    c = (i, j, k)
    E = [rng.uniform(-1, 1, i.shape).astype(dtype) for _ in range(3)]
    H = [rng.uniform(-1, 1, i.shape).astype(dtype) for _ in range(3)]
    if zero_tan:
        for a in range(3):
            for b in range(3):
                if b != a and boundary[b] == PEC:
                    E[a][c[b] == 0] = 0
    return E, H


def three_term_ratio(trace):
    t = np.asarray(trace)
    return (t[2:] + t[:-2]) / (2 * t[1:-1])


# ------------------------------------------------------------------------------------------------
# P1  PEC-cavity eigenmode: E[s+1] + E[s-1] = 2 cos(w dt) E[s],  cos(w dt) = 1 - 2 dt^2 sum sin^2(k_a d_a/2)/d_a^2
#     (discrete dispersion relation of the Yee scheme; closed form)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,d,mode,printed", [
    ((16, 12, 10), (1, 1, 1), (1, 1, 0), 0.995559258891025),
    ((16, 12, 10), (1, 1, 0.5), (2, 1, 0), 0.995408556616681),
    ((64, 64, 64), (1, 1, 1), (1, 1, 0), 0.999799242700862),
])
def test_p1_cavity_eigenfrequency(n, d, mode, printed):
    dt = 0.5 / math.sqrt(sum(1 / x ** 2 for x in d))
    i, j, k = grids(n)
    E, H = zeros(n), zeros(n)
    E[2][:] = np.sin(mode[0] * np.pi * i / n[0]) * np.sin(mode[1] * np.pi * j / n[1])
    y = YeeOracle(n, d, dt, (PEC,) * 3, E, H)
    p = (n[2] // 2, n[1] // 3, n[0] // 3)
    trace = [E[2][p]]
    for _ in range(30):
        y.step()
        trace.append(E[2][p])
    closed = 1 - 2 * dt ** 2 * sum(math.sin(mode[a] * math.pi / (2 * n[a])) ** 2 / d[a] ** 2 for a in range(3))
    assert abs(closed - printed) < 5e-15                      # value printed in SURVEY.md 8(c) P1
    r = three_term_ratio(trace)
    assert np.max(np.abs(r - closed)) < 5e-13
    # the mode shape is an exact eigenvector: the other E components stay identically zero
    assert np.all(E[0] == 0) and np.all(E[1] == 0)


# ------------------------------------------------------------------------------------------------
# P2  oblique plane wave in a fully periodic, anisotropic box: cos(w dt) = 1 - dt^2 |K|^2 / 2, K_a=(2/d_a) sin(k_a d_a/2)
# ------------------------------------------------------------------------------------------------
def test_p2_plane_wave_dispersion_periodic():
    n, d, m = (16, 12, 8), (1, 1, 0.5), (1, 2, 1)
    dt = 0.5 / math.sqrt(6)
    kv = [2 * np.pi * m[a] / (n[a] * d[a]) for a in range(3)]
    K = [2 * np.sin(kv[a] * d[a] / 2) / d[a] for a in range(3)]
    pol = np.cross(K, [0.3, -0.5, 0.8])                        # p perpendicular to K  =>  discrete div E = 0
    idx = grids(n)
    E, H = zeros(n), zeros(n)
    for a in range(3):
        pos = [(idx[b] + (0.5 if b == a else 0.0)) * d[b] for b in range(3)]     # Yee position of E_a
        E[a][:] = pol[a] * np.cos(sum(kv[b] * pos[b] for b in range(3)))
    y = YeeOracle(n, d, dt, (PERIODIC,) * 3, E, H)
    pt = (5, 4, 3)
    trace = [E[0][pt]]
    for _ in range(40):
        y.step()
        trace.append(E[0][pt])
    closed = 1 - dt * dt * sum(x * x for x in K) / 2
    assert abs(closed - 0.927179444052395) < 5e-15            # printed in SURVEY.md 8(c) P2
    assert np.max(np.abs(three_term_ratio(trace) - closed)) < 1e-12


# ------------------------------------------------------------------------------------------------
# P3 / P4  discrete divergences are constants of the motion
# ------------------------------------------------------------------------------------------------
def div_h(H, d):
    out = 0
    for a, ax in ((0, 2), (1, 1), (2, 0)):                     # component a differs along numpy axis ax
        out = out + (np.roll(H[a], -1, ax) - H[a]) / d[a]
    return out[:-1, :-1, :-1]                                  # cells not touching a high PEC wall


def div_d(E, w, d):
    out = 0
    for a, ax in ((0, 2), (1, 1), (2, 0)):
        D = E[a] * w[a]
        out = out + (D - np.roll(D, 1, ax)) / d[a]
    return out[1:, 1:, 1:]                                     # nodes with all indices >= 1


@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-13), (np.float32, 3e-5)])
def test_p3_div_h_preserved(dtype, tol):
    n, d = (12, 10, 8), (1, 1, 0.5)
    dt = 0.5 / math.sqrt(6)
    E, H = rand_fields(n, 1, dtype)
    d0 = div_h([h.astype(np.float64) for h in H], d)
    y = YeeOracle(n, d, dt, (PEC,) * 3, E, H)
    y.step(200)
    d1 = div_h([h.astype(np.float64) for h in H], d)
    assert np.abs(d0).max() > 1.0
    assert np.abs(d1 - d0).max() < tol


def test_p4_div_d_preserved_heterogeneous():
    n, d = (12, 10, 8), (1, 1, 1)
    dt = 0.5 / math.sqrt(3)
    rng = np.random.default_rng(5)
    eps = [rng.uniform(1, 12.1, (n[2], n[1], n[0])) for _ in range(3)]
    E, H = rand_fields(n, 2, np.float64)
    d0 = div_d(E, eps, d)
    y = YeeOracle(n, d, dt, (PEC,) * 3, E, H, cb=[dt / e for e in eps])
    y.step(300)
    assert np.abs(d0).max() > 1.0
    assert np.abs(div_d(E, eps, d) - d0).max() < 2e-12


# ------------------------------------------------------------------------------------------------
# P5  leapfrog energy  W = sum eps |E^{n+1}|^2 + sum H^{n+3/2} . H^{n+1/2}  is EXACTLY conserved (ca = 1)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("hetero", [False, True])
def test_p5_leapfrog_energy_conserved(hetero):
    n, d = (12, 10, 8), (1, 1, 0.5)
    dt = 0.5 / math.sqrt(6)
    rng = np.random.default_rng(7)
    shape = (n[2], n[1], n[0])
    eps = [rng.uniform(1, 12.1, shape) if hetero else np.ones(shape) for _ in range(3)]
    E, H = rand_fields(n, 3, np.float64)
    y = YeeOracle(n, d, dt, (PEC,) * 3, E, H, cb=[dt / e for e in eps] if hetero else None)
    W, naive = [], []
    for _ in range(200):
        y.e_half()
        Hprev = [h.copy() for h in H]
        y.h_half()
        W.append(sum((eps[a] * E[a] ** 2).sum() + (H[a] * Hprev[a]).sum() for a in range(3)))
        naive.append(sum((eps[a] * E[a] ** 2).sum() + (H[a] ** 2).sum() for a in range(3)))
    W, naive = np.array(W), np.array(naive)
    assert np.ptp(W) / np.mean(W) < 5e-14
    assert np.ptp(naive) / np.mean(naive) > 1e-3               # the naive sum is NOT conserved: the pin is sharp
    assert np.ptp(naive) / np.mean(naive) < 0.5                # ... but bounded


# ------------------------------------------------------------------------------------------------
# P6  lossy uniform medium:  E[s+1] = (1 + ca - cb db lam) E[s] - ca E[s-1]
# ------------------------------------------------------------------------------------------------
def test_p6_lossy_recurrence():
    n, d = (16, 12, 10), (1, 1, 1)
    dt = 0.5 / math.sqrt(3)
    ca, epsr = 0.98, 2.1
    cb = dt * (1 + ca) / (2 * epsr)
    shape = (n[2], n[1], n[0])
    i, j, k = grids(n)
    E, H = zeros(n), zeros(n)
    E[2][:] = np.sin(np.pi * i / n[0]) * np.sin(2 * np.pi * j / n[1])
    y = YeeOracle(n, d, dt, (PEC,) * 3, E, H, ca=[np.full(shape, ca)] * 3, cb=[np.full(shape, cb)] * 3)
    p = (3, 4, 5)
    tr = [E[2][p]]
    for _ in range(60):
        y.step()
        tr.append(E[2][p])
    tr = np.array(tr)
    lam = (2 * math.sin(math.pi / (2 * n[0]))) ** 2 + (2 * math.sin(2 * math.pi / (2 * n[1]))) ** 2
    pred = (1 + ca - cb * dt * lam) * tr[1:-1] - ca * tr[:-2]
    assert np.abs(pred - tr[2:]).max() < 1e-14
    assert abs(tr[60]) < abs(tr[0])                            # it decays


# ------------------------------------------------------------------------------------------------
# P7  magic time step (dx = dt = 1, fields uniform in y, z, fully periodic): exact shift by one cell per step
# ------------------------------------------------------------------------------------------------
def test_p7_magic_time_step_exact_shift():
    n = (16, 4, 4)
    prof = np.zeros(16, np.float32)
    prof[3:7] = [1, 3, -2, 5]
    E, H = zeros(n, np.float32), zeros(n, np.float32)
    E[2][:] = prof[None, None, :]
    H[1][:] = -prof[None, None, :]                             # +x travelling: Hy^{1/2}(i+1/2) = -f(i)
    y = YeeOracle(n, (1, 1, 1), 1.0, (PERIODIC,) * 3, E, H)
    y.step(5)
    assert np.array_equal(E[2][0, 0, :], np.roll(prof, 5))
    assert np.array_equal(E[2], np.broadcast_to(np.roll(prof, 5)[None, None, :], E[2].shape))


# ------------------------------------------------------------------------------------------------
# P8  cyclic permutation (x->y->z->x) of grid, spacings and components is a symmetry, bit for bit in fp32
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("boundary", [(PEC, PEC, PEC), (PERIODIC, PEC, PEC), (PEC, PERIODIC, PERIODIC)])
def test_p8_cyclic_permutation_bit_exact(boundary):
    n, d, dt = (7, 6, 5), (1.0, 0.7, 0.5), 0.2
    rng = np.random.default_rng(3)
    shape = (n[2], n[1], n[0])
    E, H = rand_fields(n, 3, np.float32, zero_tan=False)
    ca = [rng.uniform(0.9, 1, shape).astype(np.float32) for _ in range(3)]
    cb = [rng.uniform(0.05, 0.2, shape).astype(np.float32) for _ in range(3)]
    db = [0.2, 0.15, 0.1]
    # new axes (x', y', z') = (y, z, x); component a' of the rotated problem = component (a'+1)%3 of the original.
    # numpy shape (nz, ny, nx) -> (nz', ny', nx') = (nx, nz, ny): transpose axes (2, 0, 1)
    rot = lambda A: np.ascontiguousarray(np.transpose(A, (2, 0, 1)))
    n2, d2, b2 = (n[1], n[2], n[0]), (d[1], d[2], d[0]), (boundary[1], boundary[2], boundary[0])
    E2 = [rot(E[(a + 1) % 3]) for a in range(3)]
    H2 = [rot(H[(a + 1) % 3]) for a in range(3)]
    ca2 = [rot(ca[(a + 1) % 3]) for a in range(3)]
    cb2 = [rot(cb[(a + 1) % 3]) for a in range(3)]
    db2 = [db[(a + 1) % 3] for a in range(3)]
    YeeOracle(n, d, dt, boundary, E, H, ca=ca, cb=cb, db=db).step(20)
    YeeOracle(n2, d2, dt, b2, E2, H2, ca=ca2, cb=cb2, db=db2).step(20)
    for a in range(3):
        assert np.array_equal(E2[a], rot(E[(a + 1) % 3]))
        assert np.array_equal(H2[a], rot(H[(a + 1) % 3]))


# ------------------------------------------------------------------------------------------------
# P9  hand-expanded 4^3 grids
# ------------------------------------------------------------------------------------------------
def worked_example_fields():
    E = [dict() for _ in range(3)]
    H = [dict() for _ in range(3)]
    for i in range(4):
        for j in range(4):
            for k in range(4):
                c = (i, j, k)
                E[0][c], E[1][c], E[2][c] = Fr(i + 2 * j + 3 * k), Fr(2 * i - j + k), Fr(-i + 3 * j + 2 * k)
                H[0][c], H[1][c], H[2][c] = Fr(j - k + 1), Fr(3 * i + k - 2), Fr(i * j - k)
    return E, H


def read_golden():
    rows, sums = [], []
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        f = line.split()
        if f[0] == "sum":
            sums.append((f[1], int(f[2]), [float(x) for x in f[3:9]]))
        else:
            rows.append((f[0], int(f[1]), tuple(int(x) for x in f[2:5]), [float(x) for x in f[5:11]]))
    return rows, sums


def test_p9_hand_derivation_of_cell_111():
    """Eq. (1) by hand at cell (1,1,1), step 1, dt/dy = dt/dz = 0.5:
       Ex = 6 + 0.5*[(Hz(1,1,1)-Hz(1,0,1)) - (Hy(1,1,1)-Hy(1,1,0))] = 6 + 0.5*[(0-(-1)) - (2-1)] = 6
       Ey = 2 + 0.5*[(Hx(1,1,1)-Hx(1,1,0)) - (Hz(1,1,1)-Hz(0,1,1))] = 2 + 0.5*[(1-2) - (0-(-1))] = 1
       Ez = 4 + 0.5*[(Hy(1,1,1)-Hy(0,1,1)) - (Hx(1,1,1)-Hx(1,0,1))] = 4 + 0.5*[(2-(-1)) - (1-0)] = 5"""
    E, H = worked_example_fields()
    n = (4, 4, 4)
    Ea, Ha = to_arrays(E, n, np.float32), to_arrays(H, n, np.float32)
    YeeOracle(n, (1, 1, 1), 0.5, (PEC,) * 3, Ea, Ha).e_half()
    assert (Ea[0][1, 1, 1], Ea[1][1, 1, 1], Ea[2][1, 1, 1]) == (6.0, 1.0, 5.0)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_p9_worked_example_golden_table(dtype):
    rows, sums = read_golden()
    n = (4, 4, 4)
    for tag, bnd in (("pec", (PEC,) * 3), ("perx", (PERIODIC, PEC, PEC))):
        for steps in (0, 1, 2):
            E, H = worked_example_fields()
            brute = BruteYee(n, (1, 1, 1), bnd, E, H, dt=Fr(1, 2))
            brute.step(steps)
            Ea, Ha = to_arrays(E, n, dtype), to_arrays(H, n, dtype)
            YeeOracle(n, (1, 1, 1), 0.5, bnd, Ea, Ha).step(steps)
            # oracle == exact rational brute force on every cell
            for a in range(3):
                assert np.array_equal(Ea[a], to_arrays([brute.E[a]], n, dtype)[0])
                assert np.array_equal(Ha[a], to_arrays([brute.H[a]], n, dtype)[0])
            # both == the stored table
            for t, s, (i, j, k), vals in rows:
                if t == tag and s == steps:
                    got = [Ea[a][k, j, i] for a in range(3)] + [Ha[a][k, j, i] for a in range(3)]
                    assert got == vals, (tag, steps, (i, j, k))
            for t, s, vals in sums:
                if t == tag and s == steps:
                    assert [float(x.sum()) for x in Ea + Ha] == vals


@pytest.mark.parametrize("bnd", [(PEC, PEC, PEC), (PERIODIC, PEC, PEC), (PEC, PERIODIC, PEC), (PERIODIC, PERIODIC, PERIODIC)])
def test_p9_bruteforce_random_dyadic_with_coeffs_and_source(bnd):
    """Random small dyadic inputs (fields, ca, cb, db, anisotropic power-of-two spacings, a box source):
    every intermediate is exactly representable in fp64, so the fp64 oracle must equal the exact
    rational brute force bit for bit after two steps.  Non-cubic grid catches transposed strides."""
    n, d = (4, 3, 5), (1, 2, 0.5)
    rng = np.random.default_rng(11)
    q = lambda lo, hi, den: Fr(int(rng.integers(lo * den, hi * den + 1)), den)
    cells = [(i, j, k) for i in range(n[0]) for j in range(n[1]) for k in range(n[2])]
    E = [{c: q(-2, 2, 8) for c in cells} for _ in range(3)]
    H = [{c: q(-2, 2, 8) for c in cells} for _ in range(3)]
    ca = [{c: q(0, 1, 4) for c in cells} for _ in range(3)]
    cb = [{c: q(0, 1, 4) for c in cells} for _ in range(3)]
    db = [Fr(1, 2), Fr(1, 4), Fr(3, 4)]
    box = (1, 0, 2, 2, 2, 3)
    amp = {(ii, jj, kk): q(-1, 1, 4) for ii in range(2) for jj in range(2) for kk in range(3)}
    wave = [Fr(1, 2), Fr(-3, 4), Fr(1, 4)]
    brute = BruteYee(n, d, bnd, E, H, ca=ca, cb=cb, db=db, dt=Fr(1, 2))
    brute.src = (1, box, amp, wave)
    Ea, Ha = to_arrays(E, n, np.float64), to_arrays(H, n, np.float64)
    y = YeeOracle(n, d, 0.5, bnd, Ea, Ha, ca=to_arrays(ca, n, np.float64), cb=to_arrays(cb, n, np.float64),
                  db=[float(x) for x in db])
    amp_arr = np.zeros((3, 2, 2))
    for (ii, jj, kk), v in amp.items():
        amp_arr[kk, jj, ii] = float(v)
    y.set_source(1, box, amp_arr, np.array([float(x) for x in wave]))
    for s in range(1, 4):                                      # step 4 would index past wave[]: source off
        brute.step(1)
        y.step(1)
        for a in range(3):
            assert np.array_equal(Ea[a], to_arrays([brute.E[a]], n, np.float64)[0]), (s, "E", a)
            assert np.array_equal(Ha[a], to_arrays([brute.H[a]], n, np.float64)[0]), (s, "H", a)
    brute.step(1)
    y.step(1)                                                  # t = 3 >= nwave: no injection on either side
    assert np.array_equal(Ea[1], to_arrays([brute.E[1]], n, np.float64)[0])


# ------------------------------------------------------------------------------------------------
# P11 and source pins
# ------------------------------------------------------------------------------------------------
def test_p11_zero_stays_zero_and_static_field():
    n = (6, 5, 4)
    E, H = zeros(n, np.float32), zeros(n, np.float32)
    YeeOracle(n, (1, 1, 1), 0.3, (PEC,) * 3, E, H).step(10)
    assert all(np.all(a == 0) for a in E + H)
    # uniform H has zero curl away from the frozen wall cells; uniform E in a periodic box is static
    E, H = zeros(n, np.float32), zeros(n, np.float32)
    for a in range(3):
        E[a][:] = 0.25 * (a + 1)
        H[a][:] = -0.5 * (a + 1)
    YeeOracle(n, (1, 1, 1), 0.3, (PERIODIC,) * 3, E, H).step(10)
    for a in range(3):
        assert np.all(E[a] == np.float32(0.25 * (a + 1))) and np.all(H[a] == np.float32(-0.5 * (a + 1)))


def test_source_first_step_closed_form_and_linearity():
    n, d, dt = (8, 7, 6), (1, 1, 0.5), 0.25
    E, H = zeros(n), zeros(n)
    y = YeeOracle(n, d, dt, (PEC,) * 3, E, H)
    wave = np.array([0.5, -1.0, 0.25])
    y.set_source(2, (4, 3, 2, 1, 1, 1), np.array([[[2.0]]]), wave)
    y.step(1)
    # after one step: Ez(4,3,2) = amp*wave[0] = 1;  Hx -= db*(dEz/dy): Hx(4,3,2) = +dt*1/dy, Hx(4,2,2) = -dt/dy
    assert E[2][2, 3, 4] == 1.0 and np.count_nonzero(E[2]) == 1
    assert H[0][2, 3, 4] == dt * 1.0 and H[0][2, 2, 4] == -dt * 1.0
    # Hy += db*(dEz/dx): Hy(4,3,2) = -dt, Hy(3,3,2) = +dt ; Hz untouched
    assert H[1][2, 3, 4] == -dt and H[1][2, 3, 3] == dt and np.count_nonzero(H[2]) == 0
    # linearity in fp64: run(A + source) - run(A) - run(source) ~ 0
    EA, HA = rand_fields(n, 4, np.float64)
    EB, HB = [e.copy() for e in EA], [h.copy() for h in HA]
    ya = YeeOracle(n, d, dt, (PEC,) * 3, EA, HA)
    yb = YeeOracle(n, d, dt, (PEC,) * 3, EB, HB)
    yb.set_source(2, (4, 3, 2, 1, 1, 1), np.array([[[2.0]]]), wave)
    ya.step(5)
    yb.step(5)
    y.step(4)
    for a in range(3):
        assert np.abs(EB[a] - EA[a] - E[a]).max() < 1e-14
        assert np.abs(HB[a] - HA[a] - H[a]).max() < 1e-14


def test_thread_count_does_not_change_bits():
    n = (9, 8, 7)
    E1, H1 = rand_fields(n, 9, np.float32)
    E2, H2 = [e.copy() for e in E1], [h.copy() for h in H1]
    YeeOracle(n, (1, 1, 0.5), 0.2, (PEC, PERIODIC, PEC), E1, H1, nthreads=1).step(7)
    YeeOracle(n, (1, 1, 0.5), 0.2, (PEC, PERIODIC, PEC), E2, H2, nthreads=5).step(7)
    assert all(np.array_equal(a, b) for a, b in zip(E1 + H1, E2 + H2))
