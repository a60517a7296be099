"""Thin ctypes binding of libfdtd_b200 (include/fdtd.h): argument marshalling only -- every step of the path
runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream, nothing else.

There is NO CPU fallback: if the shared library is missing `load()` raises, and on a box without a B200
`Fdtd(...)` raises FdtdError(FDTD_ECUDA).
"""
from __future__ import annotations

import ctypes as C
import os

PEC, PERIODIC = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE, ETIMEOUT = range(6)
KERNEL_NAIVE, KERNEL_SYSTOLIC, KERNEL_SYSTOLIC_SMEM, KERNEL_SYSTOLIC_REG = 0, 1, 2, 3
_ERRNAME = {1: "FDTD_EINVAL", 2: "FDTD_ENOMEM", 3: "FDTD_ECUDA", 4: "FDTD_ESTATE", 5: "FDTD_ETIMEOUT"}

HERE = os.path.dirname(os.path.abspath(__file__))
_LIBFILES = {"nofma": "libfdtd_b200.so", "fma": "libfdtd_b200_fma.so", "dbg": "libfdtd_b200_dbg.so", "prof": "libfdtd_b200_prof.so"}
_libs = {}

_F3 = C.c_void_p * 3
_PROTOS = {
    "fdtd_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, C.c_float,
                              C.POINTER(C.c_int), C.c_void_p]),
    "fdtd_set_fields": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "fdtd_set_fields_f16": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "fdtd_load_fields": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "fdtd_set_coeffs": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_float)]),
    "fdtd_set_coeff_lut": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float), C.POINTER(C.c_float)]),
    "fdtd_set_source": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                  C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_int]),
    "fdtd_set_monitor": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_void_p]),
    "fdtd_step": (C.c_int, [C.c_void_p, C.c_int]),
    "fdtd_get_fields": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "fdtd_sync": (C.c_int, [C.c_void_p]),
    "fdtd_set_time": (C.c_int, [C.c_void_p, C.c_longlong]),
    "fdtd_get_time": (C.c_longlong, [C.c_void_p]),
    "fdtd_set_kernel": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]),
    "fdtd_get_kernel": (C.c_int, [C.c_void_p, C.POINTER(C.c_int)]),
    "fdtd_get_counters": (C.c_int, [C.c_void_p, C.POINTER(C.c_longlong)]),
    "fdtd_set_timing": (C.c_int, [C.c_void_p, C.c_int]),
    "fdtd_last_step_ms": (C.c_int, [C.c_void_p, C.POINTER(C.c_float)]),
    "fdtd_plan_tiles": (C.c_int, [C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_int, C.POINTER(C.c_int)]),
    "fdtd_plan_owner": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "fdtd_debug_level_errors": (C.c_int, [C.c_void_p, C.POINTER(C.c_longlong)]),
    "fdtd_absorber_coeffs": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_float, C.POINTER(C.c_void_p), C.POINTER(C.c_int), C.POINTER(C.c_float),
                                       C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_void_p]),
    "fdtd_step_noalloc": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, C.c_float, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                    C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_float), C.c_int, C.c_int, C.c_void_p, C.c_char_p, C.c_int]),
    "fdtd_last_error": (C.c_char_p, [C.c_void_p]),
    "fdtd_build_info": (C.c_char_p, []),
    "fdtd_destroy": (None, [C.c_void_p]),
}
EXPORTS = tuple(_PROTOS)


class FdtdError(RuntimeError):
    def __init__(self, code, msg=""):
        self.code = code
        super().__init__(f"{_ERRNAME.get(code, code)}: {msg}" if msg else str(_ERRNAME.get(code, code)))


def lib_path(variant="nofma"):
    return os.path.join(HERE, _LIBFILES[variant])


def load(variant="nofma"):
    """dlopen the in-tree library; raises if it has not been built (python -m paper_2502_20610_b200.build)."""
    if variant not in _libs:
        path = lib_path(variant)
        if not os.path.exists(path):
            raise FileNotFoundError(f"{path} is missing: build it with `python -m paper_2502_20610_b200.build` "
                                    "(there is no CPU fallback)")
        lib = C.CDLL(path)
        for name, (res, args) in _PROTOS.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _libs[variant] = lib
    return _libs[variant]


def _ptr3(tensors):
    if tensors is None:
        return None
    arr = _F3()
    for a in range(3):
        t = tensors[a]
        arr[a] = None if t is None else (t.data_ptr() if hasattr(t, "data_ptr") else t.ctypes.data)
    return C.cast(arr, C.POINTER(C.c_void_p))


def plan_tiles(n, boundary, N, T, variant="nofma"):
    out = (C.c_int * 3)()
    rc = load(variant).fdtd_plan_tiles((C.c_int * 3)(*n), (C.c_int * 3)(*boundary), (C.c_int * 3)(*N), int(T), out)
    if rc != OK:
        raise FdtdError(rc)
    return tuple(out)


def plan_owner(n, boundary, N, T, g, s, variant="nofma"):
    tile, off = C.c_int(), C.c_int()
    rc = load(variant).fdtd_plan_owner(int(n), int(boundary), int(N), int(T), int(g), int(s), C.byref(tile), C.byref(off))
    if rc != OK:
        raise FdtdError(rc)
    return tile.value, off.value


def absorber_coeffs(n, dt, eps, thickness, sigma_max, order, ca, cb, stream=None, variant="nofma"):
    """fdtd_absorber_coeffs: fill the CUDA tensors ca[3], cb[3] (shape (nz, ny, nx)) with the graded-conductivity update
    coefficients; eps: None or three CUDA tensors.  Enqueued on the current torch stream."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    rc = load(variant).fdtd_absorber_coeffs(int(n[0]), int(n[1]), int(n[2]), float(dt), _ptr3(eps), (C.c_int * 6)(*[int(x) for x in thickness]),
                                            (C.c_float * 6)(*[float(x) for x in sigma_max]), int(order), _ptr3(ca), _ptr3(cb),
                                            C.c_void_p(int(stream) or None))
    if rc != OK:
        raise FdtdError(rc, "fdtd_absorber_coeffs")


NOALLOC_MAX_TILES = 131072


def step_noalloc(n, d, dt, E, H, ca=None, cb=None, db=None, nsteps=1, T=0, stream=None, variant="nofma"):
    """fdtd_step_noalloc: advance the six float32 CUDA tensors E[3], H[3] (shape (nz, ny, nx)) in place by `nsteps` steps
    with the systolic kernel, without any device allocation inside the library (its flags, counters and claim order sit in
    a fixed array inside the .so).  For hosts that own all device memory themselves or cannot stall on cudaMalloc.  PEC
    walls, nx % 4 == 0, no source; blocks until the GPU work is done.  Raises FdtdError with the library's message."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
    err = C.create_string_buffer(512)
    dbp = None if db is None else (C.c_float * 3)(*[float(x) for x in db])
    rc = load(variant).fdtd_step_noalloc(int(n[0]), int(n[1]), int(n[2]), float(d[0]), float(d[1]), float(d[2]), float(dt), _ptr3(E), _ptr3(H),
                                         _ptr3(ca), _ptr3(cb), dbp, int(nsteps), int(T), C.c_void_p(int(stream) or None), err, len(err))
    if rc != OK:
        raise FdtdError(rc, err.value.decode())


class Fdtd:
    """One simulation context.  E, H (and ca, cb) are lists of three float32 CUDA tensors of shape (nz, ny, nx),
    contiguous, which the library borrows and updates in place."""

    def __init__(self, n, d, dt, boundary, stream=None, variant="nofma"):
        import torch
        self._lib = load(variant)
        self.variant = variant
        self.n = tuple(int(x) for x in n)
        self._h = C.c_void_p()
        self._keep = []
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
        rc = self._lib.fdtd_create(C.byref(self._h), *self.n, *[float(x) for x in d], float(dt),
                                   (C.c_int * 3)(*[int(b) for b in boundary]), C.c_void_p(int(stream) or None))
        if rc != OK:
            self._h = C.c_void_p()
            raise FdtdError(rc, "fdtd_create failed (no B200 / bad arguments)")

    def _check(self, rc):
        if rc != OK:
            raise FdtdError(rc, self._lib.fdtd_last_error(self._h).decode())

    def _check_tensors(self, ts, dtype=None):
        import torch
        shape = (self.n[2], self.n[1], self.n[0])
        for t in ts:
            assert t.is_cuda and t.dtype == (dtype or torch.float32) and t.is_contiguous() and tuple(t.shape) == shape, "bad field tensor"

    def set_fields(self, E, H):
        """Six float32 CUDA tensors, or six float16 CUDA tensors (binary16 field storage, fdtd_set_fields_f16)."""
        import torch
        half = E[0].dtype == torch.float16
        self._check_tensors(list(E) + list(H), torch.float16 if half else torch.float32)
        self._keep = [list(E), list(H)] + self._keep[2:]
        fn = self._lib.fdtd_set_fields_f16 if half else self._lib.fdtd_set_fields
        self._check(fn(self._h, _ptr3(E), _ptr3(H)))

    def load_fields(self, E, H):
        """Copy initial data from host (pinned numpy / CPU tensors) or device arrays into the bound buffers."""
        self._check(self._lib.fdtd_load_fields(self._h, _ptr3(E), _ptr3(H)))

    def set_coeffs(self, ca=None, cb=None, db=None):
        if ca is not None:
            self._check_tensors(ca)
        if cb is not None:
            self._check_tensors(cb)
        self._keep.append((ca, cb))
        dbp = None if db is None else (C.c_float * 3)(*[float(x) for x in db])
        self._check(self._lib.fdtd_set_coeffs(self._h, _ptr3(ca), _ptr3(cb), dbp))

    def set_coeff_lut(self, idx, ca_lut, cb_lut, db=None):
        """Material-index coefficients: idx = three uint8 CUDA tensors (nz, ny, nx); ca_lut, cb_lut: numpy (3, nmat)."""
        import numpy as np
        import torch
        shape = (self.n[2], self.n[1], self.n[0])
        for t in idx:
            assert t.is_cuda and t.dtype == torch.uint8 and t.is_contiguous() and tuple(t.shape) == shape, "bad index tensor"
        ca_lut = np.ascontiguousarray(ca_lut, dtype=np.float32)
        cb_lut = np.ascontiguousarray(cb_lut, dtype=np.float32)
        assert ca_lut.shape == cb_lut.shape and ca_lut.ndim == 2 and ca_lut.shape[0] == 3
        self._keep.append(list(idx))
        fp = C.POINTER(C.c_float)
        dbp = None if db is None else (C.c_float * 3)(*[float(x) for x in db])
        self._check(self._lib.fdtd_set_coeff_lut(self._h, _ptr3(idx), int(ca_lut.shape[1]), ca_lut.ctypes.data_as(fp), cb_lut.ctypes.data_as(fp), dbp))

    def set_source(self, comp, box, amp, wave):
        import numpy as np
        if amp is None:
            self._check(self._lib.fdtd_set_source(self._h, 0, 0, 0, 0, 0, 0, 0, None, None, 0))
            return
        amp = np.ascontiguousarray(amp, dtype=np.float32).reshape(-1)
        wave = np.ascontiguousarray(wave, dtype=np.float32).reshape(-1)
        fp = C.POINTER(C.c_float)
        self._check(self._lib.fdtd_set_source(self._h, int(comp), *[int(x) for x in box], amp.ctypes.data_as(fp),
                                              wave.ctypes.data_as(fp), int(wave.size)))

    def set_monitor(self, axis, index, wE, wH, acc):
        """Running DFT on the plane axis = index.  wE, wH: numpy (nt, F, 2); acc: float32 CUDA tensor (6, F, 2, cells),
        borrowed and accumulated into (the caller zeroes it).  acc=None removes the monitor."""
        import numpy as np
        if acc is None:
            self._check(self._lib.fdtd_set_monitor(self._h, 0, 0, 0, 0, None, None, None))
            return
        wE = np.ascontiguousarray(wE, dtype=np.float32)
        wH = np.ascontiguousarray(wH, dtype=np.float32)
        assert wE.shape == wH.shape and wE.ndim == 3 and wE.shape[2] == 2
        nt, F = wE.shape[0], wE.shape[1]
        assert acc.is_cuda and acc.is_contiguous() and acc.numel() == 6 * F * 2 * (self.n[0] * self.n[1] * self.n[2] // self.n[axis])
        self._keep.append(acc)
        fp = C.POINTER(C.c_float)
        self._check(self._lib.fdtd_set_monitor(self._h, int(axis), int(index), F, nt, wE.ctypes.data_as(fp), wH.ctypes.data_as(fp),
                                               C.c_void_p(acc.data_ptr())))

    def set_kernel(self, which, tile=None, T=0):
        tx, ty, tz = tile if tile is not None else (0, 0, 0)
        self._check(self._lib.fdtd_set_kernel(self._h, int(which), int(tx), int(ty), int(tz), int(T)))

    def get_kernel(self):
        out = (C.c_int * 8)()
        self._check(self._lib.fdtd_get_kernel(self._h, out))
        return {"which": out[0], "tile": (out[1], out[2], out[3]), "T": out[4], "tiles": out[5], "ctas": out[6], "smem": out[7]}

    def step(self, n):
        self._check(self._lib.fdtd_step(self._h, int(n)))

    def sync(self):
        self._check(self._lib.fdtd_sync(self._h))

    def get_fields(self, E=None, H=None):
        self._check(self._lib.fdtd_get_fields(self._h, _ptr3(E), _ptr3(H)))

    def set_time(self, t):
        self._check(self._lib.fdtd_set_time(self._h, int(t)))

    @property
    def time(self):
        return int(self._lib.fdtd_get_time(self._h))

    def counters(self):
        out = (C.c_longlong * 4)()
        self._check(self._lib.fdtd_get_counters(self._h, out))
        return {"launches": out[0], "steps": out[1], "chunks": out[2], "tiles": out[3]}

    def debug_level_errors(self):
        """Developer build + FDTD_DEBUG_LEVELS=1: (violations, kind, cell offset, level found, level expected)."""
        out = (C.c_longlong * 5)()
        self._check(self._lib.fdtd_debug_level_errors(self._h, out))
        return tuple(out)

    def set_timing(self, on=True):
        self._check(self._lib.fdtd_set_timing(self._h, int(bool(on))))

    def last_step_ms(self):
        ms = C.c_float()
        self._check(self._lib.fdtd_last_step_ms(self._h, C.byref(ms)))
        return ms.value

    def close(self):
        if self._h:
            self._lib.fdtd_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def run_workload(w, kernel=KERNEL_SYSTOLIC, tile=None, T=0, steps=None, variant="nofma", device="cuda:0"):
    """Build the seeded inputs of workload `w` on the device, run `steps` steps, return (E, H) CUDA tensors and the
    context (still open).  Convenience used by tests, smoke() and bench.py."""
    import torch
    from . import workloads
    dev = torch.device(device)
    E, H = workloads.make_fields(w, device=dev)
    ca, cb = workloads.make_coeffs(w, device=dev)
    sim = Fdtd(w.n, w.d, w.dt, w.boundary, variant=variant)
    sim.set_fields(E, H)
    if ca is not None:
        sim.set_coeffs(ca, cb, None)
    src = workloads.make_source(w)
    if src is not None:
        sim.set_source(src.comp, src.box, src.amp, src.wave)
    sim.set_kernel(kernel, tile, T)
    sim.step(w.steps if steps is None else steps)
    sim.sync()
    return E, H, sim
