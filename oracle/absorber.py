"""CPU oracle of the adiabatic-absorber coefficient generator.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it never touches the CUDA
path and shares no code with it.

What the paper says (section 4): the engine "does not use PMLs, but instead relies on the imaginary part of
the permittivity to allow for the formation of adiabatic absorbers [5]" -- Oskooi et al. 2008: a conductivity that rises
smoothly (polynomially) from zero over a layer in front of the wall.  The paper gives no formula; reading #14
fixes the one below.  Pins: tests/test_oracle_next_pins.py (uniform lossy medium against the analytic decay rate,
round-trip reflection of a graded layer against exp(-2 sigma_max L d / ((p+1) n)), mirror symmetry of the half-cell
staggering, sum rule at corners).

    Domain along axis q: coordinates [0, n_q] in cells; the low wall at 0, the high wall (ghost) at n_q.
    Component E_a of cell (i,j,k) sits at coordinate  s_q = g_q + 1/2 if q == a else g_q        (Yee staggering, include/fdtd.h)
    Low layer of L cells :  u = (L - s_q) / L          where s_q < L
    High layer of L cells:  u = (s_q - (n_q - L)) / L  where s_q > n_q - L
    sigma_q   = sigma_max[face] * u^p                  (p = integer order >= 0; p = 0: uniform sigma_max inside the layer)
    sigma     = (sigma_x + sigma_y) + sigma_z          (layers of different axes add, in this order)
    ca_a      = (2 eps_a - sigma dt) / (2 eps_a + sigma dt)
    cb_a      = (2 dt) / (2 eps_a + sigma dt)          (semi-implicit conductivity term; include/fdtd.h "Generator side")

Every statement is one rounded operation in `dtype` (float32 to compare bit for bit with the CUDA generator, float64 for
the physical pins).
"""
import math

import numpy as np


def absorber_sigma_max(R0, order, n_index, L, d):
    """sigma_max of a layer of L cells of size d in a medium of refractive index n_index whose round-trip POWER
    reflection is R0 when the transition is adiabatic: a plane wave exp(i(kx - wt)) in a medium (eps, sigma) has
    Im k = sigma / (2 n) to first order in sigma/(w eps) (eps0 = mu0 = 1), so the round trip through
    sigma(u) = sigma_max u^p multiplies the amplitude by exp(-2 * sigma_max L d / (2 n (p+1))) and the power by its
    square:  R0 = exp(-2 sigma_max L d / ((p+1) n))."""
    return -(order + 1) * n_index * math.log(R0) / (2.0 * L * d)


def layer_profile(nq, own_axis, L_lo, L_hi, smax_lo, smax_hi, order, dtype):
    """sigma_q along one axis for a component that is (own_axis=True) or is not staggered along it: array of nq values."""
    f = np.dtype(dtype).type
    out = np.zeros(nq, dtype)
    for g in range(nq):
        s = f(g) + (f(0.5) if own_axis else f(0.0))
        sig = f(0.0)
        for L, smax, low in ((L_lo, smax_lo, True), (L_hi, smax_hi, False)):
            if L <= 0:
                continue
            if low:
                if not (s < f(L)):
                    continue
                num = f(L) - s
            else:
                edge = f(nq - L)
                if not (s > edge):
                    continue
                num = s - edge
            u = f(num / f(L))
            w = f(1.0)
            for _ in range(order):
                w = f(w * u)
            sig = f(sig + f(f(smax) * w))      # a cell can sit in both layers of one axis only if they overlap: they add
        out[g] = sig
    return out


def absorber_coeffs(n, dt, eps, thickness, sigma_max, order, dtype=np.float32):
    """ca[3], cb[3] of shape (nz, ny, nx).  eps: None (vacuum) or three arrays; thickness = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi)
    in cells; sigma_max: six values, same order."""
    f = np.dtype(dtype).type
    nx, ny, nz = n
    ca, cb = [], []
    for a in range(3):
        prof = [layer_profile(n[q], q == a, thickness[2 * q], thickness[2 * q + 1], sigma_max[2 * q], sigma_max[2 * q + 1], order, dtype)
                for q in range(3)]
        sig = (prof[0][None, None, :] + prof[1][None, :, None]).astype(dtype)
        sig = (sig + prof[2][:, None, None]).astype(dtype)
        e = np.ones((nz, ny, nx), dtype) if eps is None else np.asarray(eps[a], dtype)
        e2 = (f(2.0) * e).astype(dtype)
        sd = (sig * f(dt)).astype(dtype)
        den = (e2 + sd).astype(dtype)
        num = (e2 - sd).astype(dtype)
        ca.append((num / den).astype(dtype))
        cb.append((f(f(2.0) * f(dt)) / den).astype(dtype))
    return ca, cb
