"""Hand-expanded Yee update in exact rational arithmetic on tiny grids -- a pin for the oracle.

This is NOT the oracle retyped: it works on dictionaries keyed by (i, j, k), fetches every
neighbour by coordinate with the wall rule written as a lookup default, uses Fractions (no
rounding at all), and writes each of the six component updates as the formula printed in
eq. (1) of the paper or its cyclic/Faraday counterpart (SURVEY.md 8(c) "Written out").
With dyadic inputs the fp64 oracle must reproduce it EXACTLY, so a dropped term, a wrong sign
or index, a transposed operand or a mishandled wall in oracle/yee_oracle_impl.h fails here.
"""
from fractions import Fraction as Fr
from itertools import product

PEC, PERIODIC = 0, 1


class BruteYee:
    def __init__(self, n, d, bnd, E, H, ca=None, cb=None, db=None, dt=None):
        """E, H: three dicts {(i,j,k): Fraction}; ca/cb: three dicts or None; db: three Fractions."""
        self.n, self.bnd = n, bnd
        self.inv = [1 / Fr(x) for x in d]
        self.E = [dict(e) for e in E]
        self.H = [dict(h) for h in H]
        self.ca = ca
        self.cb = cb
        self.dt = Fr(dt)
        self.db = [Fr(x) for x in db] if db is not None else [Fr(dt)] * 3
        self.src = None
        self.t = 0

    def cells(self):
        return product(range(self.n[0]), range(self.n[1]), range(self.n[2]))

    # value one cell back; on a PEC axis there is none at index 0 (caller never needs it there)
    def back(self, F, c, ax):
        q = list(c)
        q[ax] -= 1
        if q[ax] < 0:
            if self.bnd[ax] == PERIODIC:
                q[ax] = self.n[ax] - 1
            else:
                return None
        return F[tuple(q)]

    # value one cell forward; beyond a high PEC wall the tangential E ghost is zero
    def fwd(self, F, c, ax):
        q = list(c)
        q[ax] += 1
        if q[ax] == self.n[ax]:
            if self.bnd[ax] == PERIODIC:
                q[ax] = 0
            else:
                return Fr(0)
        return F[tuple(q)]

    def on_low_wall(self, c, ax):
        return self.bnd[ax] == PEC and c[ax] == 0

    def e_half(self):
        Ex, Ey, Ez = self.E
        Hx, Hy, Hz = self.H
        ix, iy, iz = self.inv
        nEx, nEy, nEz = {}, {}, {}
        for c in self.cells():
            cax, cay, caz = [(self.ca[a][c] if self.ca else Fr(1)) for a in range(3)]
            cbx, cby, cbz = [(self.cb[a][c] if self.cb else self.dt) for a in range(3)]
            # E_x(i+1/2,j,k) is tangential to the y- and z-walls
            if not (self.on_low_wall(c, 1) or self.on_low_wall(c, 2)):
                nEx[c] = cax * Ex[c] + cbx * ((Hz[c] - self.back(Hz, c, 1)) * iy - (Hy[c] - self.back(Hy, c, 2)) * iz)
            if not (self.on_low_wall(c, 2) or self.on_low_wall(c, 0)):
                nEy[c] = cay * Ey[c] + cby * ((Hx[c] - self.back(Hx, c, 2)) * iz - (Hz[c] - self.back(Hz, c, 0)) * ix)
            if not (self.on_low_wall(c, 0) or self.on_low_wall(c, 1)):
                nEz[c] = caz * Ez[c] + cbz * ((Hy[c] - self.back(Hy, c, 0)) * ix - (Hx[c] - self.back(Hx, c, 1)) * iy)
        Ex.update(nEx), Ey.update(nEy), Ez.update(nEz)

    def source(self):
        if self.src is None:
            return
        comp, box, amp, wave = self.src
        if not (0 <= self.t < len(wave)):
            return
        for kk, jj, ii in product(range(box[5]), range(box[4]), range(box[3])):
            c = (box[0] + ii, box[1] + jj, box[2] + kk)
            self.E[comp][c] += amp[(ii, jj, kk)] * wave[self.t]

    def h_half(self):
        Ex, Ey, Ez = self.E
        Hx, Hy, Hz = self.H
        ix, iy, iz = self.inv
        nHx, nHy, nHz = {}, {}, {}
        for c in self.cells():
            nHx[c] = Hx[c] - self.db[0] * ((self.fwd(Ez, c, 1) - Ez[c]) * iy - (self.fwd(Ey, c, 2) - Ey[c]) * iz)
            nHy[c] = Hy[c] - self.db[1] * ((self.fwd(Ex, c, 2) - Ex[c]) * iz - (self.fwd(Ez, c, 0) - Ez[c]) * ix)
            nHz[c] = Hz[c] - self.db[2] * ((self.fwd(Ey, c, 0) - Ey[c]) * ix - (self.fwd(Ex, c, 1) - Ex[c]) * iy)
        Hx.update(nHx), Hy.update(nHy), Hz.update(nHz)

    def step(self, nsteps=1):
        for _ in range(nsteps):
            self.e_half()
            self.source()
            self.h_half()
            self.t += 1


def to_arrays(dicts, n, dtype):
    import numpy as np
    out = []
    for dct in dicts:
        a = np.zeros((n[2], n[1], n[0]), dtype)
        for (i, j, k), v in dct.items():
            a[k, j, i] = float(v)
        out.append(a)
    return out
