"""ctypes front end of the CPU oracle (oracle/yee_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never touches the CUDA path.

Arrays are numpy, C-contiguous, shape (nz, ny, nx) so that x is fastest:
idx = i + nx*(j + ny*k)  (SURVEY.md 8(b) layout contract).
"""
import ctypes as C
import os

import numpy as np

from . import build_oracle

PEC, PERIODIC = 0, 1
_lib = None


def _grid_struct(ctype):
    P = C.POINTER(ctype)

    class Grid(C.Structure):
        _fields_ = [
            ("n", C.c_int * 3), ("bnd", C.c_int * 3), ("rd", ctype * 3),
            ("E", P * 3), ("H", P * 3), ("ca", P * 3), ("cb", P * 3),
            ("cb_scalar", ctype), ("db", ctype * 3),
            ("src_comp", C.c_int), ("src_box", C.c_int * 6),
            ("src_amp", P), ("src_wave", P), ("src_nwave", C.c_int), ("nthreads", C.c_int),
        ]
    return Grid


_GRID = {np.dtype(np.float32): _grid_struct(C.c_float), np.dtype(np.float64): _grid_struct(C.c_double)}
_CT = {np.dtype(np.float32): C.c_float, np.dtype(np.float64): C.c_double}
_SUF = {np.dtype(np.float32): "f32", np.dtype(np.float64): "f64"}


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle.build())
        for suf in ("f32", "f64", "h16"):
            getattr(_lib, "yee_oracle_run_" + suf).restype = C.c_int
            getattr(_lib, "yee_oracle_e_half_" + suf).restype = C.c_int
            getattr(_lib, "yee_oracle_h_half_" + suf).restype = C.c_int
    return _lib


class YeeOracle:
    """Plain leapfrog on caller-owned numpy arrays, updated in place.

    n = (nx, ny, nz); d = (dx, dy, dz); boundary = per-axis PEC|PERIODIC.
    E, H: lists of three arrays of shape (nz, ny, nx), dtype float32 or float64.
    ca, cb: None or lists of three per-cell arrays (entries may be None individually);
    cb None -> dt; db None -> (dt, dt, dt)  (SURVEY.md 8(b) fdtd_set_coeffs contract).
    """

    def __init__(self, n, d, dt, boundary, E, H, ca=None, cb=None, db=None, nthreads=None, storage=None):
        """storage="f16" (float32 arrays only): every stored field value is rounded to IEEE binary16 (row f1);
        the arrays must hold binary16-representable values on entry."""
        self.dtype = np.dtype(E[0].dtype)
        assert self.dtype in _GRID
        self.suffix = _SUF[self.dtype]
        if storage == "f16":
            assert self.dtype == np.dtype(np.float32)
            for a in list(E) + list(H):
                assert np.array_equal(a, a.astype(np.float16).astype(np.float32)), "f16 storage: inputs must be binary16 values"
            self.suffix = "h16"
        else:
            assert storage is None
        self.n = tuple(int(x) for x in n)
        shape = (self.n[2], self.n[1], self.n[0])
        self.E, self.H = list(E), list(H)
        for a in self.E + self.H:
            assert a.dtype == self.dtype and a.shape == shape and a.flags.c_contiguous
        ct = _CT[self.dtype]
        self._keep = []
        g = _GRID[self.dtype]()
        for a in range(3):
            g.n[a] = self.n[a]
            g.bnd[a] = int(boundary[a])
            g.rd[a] = self.dtype.type(1.0 / float(d[a]))
            g.E[a] = self.E[a].ctypes.data_as(C.POINTER(ct))
            g.H[a] = self.H[a].ctypes.data_as(C.POINTER(ct))
            for name, arrs in (("ca", ca), ("cb", cb)):
                arr = None if arrs is None else arrs[a]
                if arr is not None:
                    arr = np.ascontiguousarray(arr, dtype=self.dtype)
                    assert arr.shape == shape
                    self._keep.append(arr)
                    getattr(g, name)[a] = arr.ctypes.data_as(C.POINTER(ct))
            g.db[a] = self.dtype.type(dt if db is None else db[a])
        g.cb_scalar = self.dtype.type(dt)
        g.nthreads = int(nthreads or os.cpu_count() or 1)
        self.nthreads = g.nthreads
        self.g = g
        self.t = 0

    def set_source(self, comp, box, amp, wave):
        """box = (i0, j0, k0, ni, nj, nk); amp shape (nk, nj, ni) (x fastest); wave 1-D."""
        amp = np.ascontiguousarray(amp, dtype=self.dtype).reshape(-1)
        wave = np.ascontiguousarray(wave, dtype=self.dtype).reshape(-1)
        assert amp.size == box[3] * box[4] * box[5]
        self._keep += [amp, wave]
        ct = _CT[self.dtype]
        self.g.src_comp = int(comp)
        for q in range(6):
            self.g.src_box[q] = int(box[q])
        self.g.src_amp = amp.ctypes.data_as(C.POINTER(ct))
        self.g.src_wave = wave.ctypes.data_as(C.POINTER(ct))
        self.g.src_nwave = int(wave.size)

    def step(self, nsteps=1):
        rc = getattr(lib(), "yee_oracle_run_" + self.suffix)(C.byref(self.g), C.c_longlong(self.t), C.c_int(nsteps))
        if rc != 0:
            raise ValueError("yee_oracle_run rejected its arguments")
        self.t += nsteps

    def e_half(self):
        getattr(lib(), "yee_oracle_e_half_" + self.suffix)(C.byref(self.g))

    def h_half(self):
        getattr(lib(), "yee_oracle_h_half_" + self.suffix)(C.byref(self.g))
