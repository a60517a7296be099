"""ctypes front end of tests/emu/systolic_emu.cpp (CPU-side schedule harness; test code only)."""
import ctypes as C
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "..", "..", "paper_2502_20610_b200", "csrc")
LIB = os.path.join(HERE, "libsystolic_emu.so")
_FP = C.POINTER(C.c_float)


class GridParams(C.Structure):   # mirrors csrc/fdtd_types.h
    _fields_ = [("E", _FP * 3), ("H", _FP * 3), ("ca", _FP * 3), ("cb", _FP * 3),
                ("cidx", C.c_void_p * 3), ("lut", _FP), ("nmat", C.c_int), ("fld16", C.c_int),
                ("n", C.c_int * 3), ("per", C.c_int * 3), ("rd", C.c_float * 3), ("cb_scalar", C.c_float),
                ("db", C.c_float * 3), ("src_comp", C.c_int), ("src_box", C.c_int * 6),
                ("src_amp", _FP), ("src_wave", _FP), ("src_nwave", C.c_int)]


def build():
    srcs = [os.path.join(HERE, "systolic_emu.cpp")] + [os.path.join(CSRC, f) for f in ("systolic_tile.cuh", "fdtd_types.h", "yee_update.h")]
    if not os.path.exists(LIB) or any(os.path.getmtime(s) > os.path.getmtime(LIB) for s in srcs):
        subprocess.run(["g++", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c++17", "-shared", "-fPIC", "-Wall",
                        "-o", LIB + ".tmp", srcs[0]], check=True, cwd=HERE)
        os.replace(LIB + ".tmp", LIB)
    lib = C.CDLL(LIB)
    lib.systolic_emu_run.restype = C.c_int
    assert lib.systolic_emu_sizeof_grid() == C.sizeof(GridParams), "harness.GridParams is out of step with csrc/fdtd_types.h"
    return lib


def run(n, d, dt, boundary, E, H, ca, cb, db, source, box, T, nsteps, ctas=8, policy=1, seed=1, t0=0):
    """Advance float32 numpy arrays in place with the tile stages under the given scheduler policy."""
    lib = build()
    g = GridParams()
    keep = []
    for a in range(3):
        g.n[a] = n[a]
        g.per[a] = int(boundary[a])
        g.rd[a] = np.float32(1.0 / float(d[a]))
        g.db[a] = np.float32(dt if db is None else db[a])
        g.E[a] = E[a].ctypes.data_as(_FP)
        g.H[a] = H[a].ctypes.data_as(_FP)
        if ca is not None:
            g.ca[a] = ca[a].ctypes.data_as(_FP)
            g.cb[a] = cb[a].ctypes.data_as(_FP)
    g.cb_scalar = np.float32(dt)
    g.src_comp = -1
    if source is not None:
        comp, sbox, amp, wave = source
        amp = np.ascontiguousarray(amp, np.float32).reshape(-1)
        wave = np.ascontiguousarray(wave, np.float32).reshape(-1)
        keep += [amp, wave]
        g.src_comp = comp
        for q in range(6):
            g.src_box[q] = sbox[q]
        g.src_amp = amp.ctypes.data_as(_FP)
        g.src_wave = wave.ctypes.data_as(_FP)
        g.src_nwave = wave.size
    stages = C.c_longlong(0)
    rc = lib.systolic_emu_run(C.byref(g), (C.c_int * 3)(*box), int(T), int(nsteps), C.c_longlong(t0), int(ctas), int(policy),
                              C.c_ulonglong(seed), C.byref(stages))
    return rc, stages.value
