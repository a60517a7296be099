"""CPU oracle of the running-DFT output monitors.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it never touches the CUDA
path and shares no code with it.

The paper excludes outputs from its benchmark but names them as what real runs carry ("the output volume and format",
PAPER.md:106).  DESIGN.md reading #15 fixes the definition: a monitor is a plane (axis q, index m) of the grid, a list of
F frequencies and two caller-supplied tables of complex weights, one per time step and frequency; during step t (t = the
context's step counter, 0-based)

    after the E half-step and the source:   AE_a[f] += E_a[plane] * wE[t][f]        a = x, y, z
    after the H half-step:                  AH_a[f] += H_a[plane] * wH[t][f]

with complex weights (re, im) and real fields: re += v*w_re, im += v*w_im, each product rounded, then the add.  The
weights are inputs (the caller builds exp(-i w_f (t+1) dt) for E and exp(-i w_f (t+3/2) dt) for H, or a window): the
monitor itself holds no trigonometry, so the CUDA path and this oracle agree bit for bit with -fmad=false.

This file follows that definition literally: one oracle step, then the two accumulations (the H half-step does not touch
E, so accumulating E after the whole step is the same as after its half-step).
Pins: tests/test_oracle_next_pins.py (numpy.fft of an independently recorded time series; closed-form geometric sum
for a single cavity mode).
"""
import numpy as np


def plane_slice(axis, index):
    """Index tuple of the plane `axis` = index for arrays of shape (nz, ny, nx)."""
    sl = [slice(None)] * 3
    sl[2 - axis] = index
    return tuple(sl)


class MonitorOracle:
    """Running DFT of the six components on one plane, driven by a YeeOracle."""

    def __init__(self, yee, axis, index, wE, wH):
        """wE, wH: arrays (nt, F, 2) of (re, im) weights, dtype of the fields."""
        self.yee, self.sl = yee, plane_slice(axis, index)
        self.dtype = yee.dtype
        self.wE = np.asarray(wE, self.dtype)
        self.wH = np.asarray(wH, self.dtype)
        assert self.wE.shape == self.wH.shape and self.wE.ndim == 3 and self.wE.shape[2] == 2
        self.F = self.wE.shape[1]
        pshape = yee.E[0][self.sl].shape
        # acc[field 0..5 = Ex Ey Ez Hx Hy Hz][f][re/im][plane]
        self.acc = np.zeros((6, self.F, 2) + pshape, self.dtype)

    def step(self, nsteps=1):
        for _ in range(nsteps):
            t = self.yee.t
            self.yee.step(1)
            if t < 0 or t >= self.wE.shape[0]:
                continue
            for c in range(6):
                v = (self.yee.E[c] if c < 3 else self.yee.H[c - 3])[self.sl]
                w = self.wE[t] if c < 3 else self.wH[t]
                for f in range(self.F):
                    for p in range(2):
                        prod = (v * w[f, p]).astype(self.dtype)
                        self.acc[c, f, p] = (self.acc[c, f, p] + prod).astype(self.dtype)
