"""Seeded synthetic inputs for the FDTD hot path -- the ONLY module shared by the CUDA-path tests,
the oracle tests and bench.py.  It holds none of the method's arithmetic (no curl, no update):
just grid shapes, material/coefficient recipes, source tables and a counter-based RNG.

The paper's own benchmark is a synthetic "bare-bones" grid with permittivity and conductivity
fields and no sources (section 4); no public dataset is involved.  The five workloads
below are BASELINE.json's `configs` made concrete (recipe: SURVEY.md 8(d), restated in DESIGN.md).

Every random array is a pure function of (seed, array id, linear cell index):
    z = idx + GOLD*(seed*1024 + array_id + 1);  z = splitmix64_finalise(z);  m = z >> 40 (24 bits)
so any sub-window can be regenerated on the host bit-identically to a full array generated on the
GPU (needed for the window-oracle parity route at 81 GiB).  `idx = i + nx*(j + ny*k)`.

Array layout everywhere: shape (nz, ny, nx), C-contiguous, x fastest.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import numpy as np

PEC, PERIODIC = 0, 1
_GOLD = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB
_MASK64 = (1 << 64) - 1

# array ids
AID_E, AID_H = (0, 1, 2), (3, 4, 5)
AID_EPS, AID_CA = (8, 9, 10), (11, 12, 13)
AID_BLOCK = 16


def _signed(c: int) -> int:
    c &= _MASK64
    return c - (1 << 64) if c >= (1 << 63) else c


def hash24(seed: int, array_id: int, idx):
    """24-bit counter hash.  idx: numpy uint64/int64 array or torch int64 tensor -> same type, values in [0, 2^24)."""
    off = (_GOLD * (int(seed) * 1024 + int(array_id) + 1)) & _MASK64
    if isinstance(idx, np.ndarray):
        with np.errstate(over="ignore"):
            z = idx.astype(np.uint64) + np.uint64(off)
            z = (z ^ (z >> np.uint64(30))) * np.uint64(_M1)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(_M2)
            z = z ^ (z >> np.uint64(31))
            return (z >> np.uint64(40)).astype(np.int64)
    # torch int64: multiplication wraps like uint64; logical shift = arithmetic shift + mask
    z = idx + _signed(off)
    z = (z ^ ((z >> 30) & ((1 << 34) - 1))) * _signed(_M1)
    z = (z ^ ((z >> 27) & ((1 << 37) - 1))) * _signed(_M2)
    z = z ^ ((z >> 31) & ((1 << 33) - 1))
    return (z >> 40) & ((1 << 24) - 1)


def _lin_index(n, window=None, like=None):
    """Linear cell indices of `window` = (i0, j0, k0, ni, nj, nk) (default: whole grid), shape (nk, nj, ni)."""
    nx, ny, nz = n
    i0, j0, k0, ni, nj, nk = window if window is not None else (0, 0, 0, nx, ny, nz)
    if like is None:
        i = np.arange(i0, i0 + ni, dtype=np.int64)[None, None, :]
        j = np.arange(j0, j0 + nj, dtype=np.int64)[None, :, None]
        k = np.arange(k0, k0 + nk, dtype=np.int64)[:, None, None]
    else:
        import torch
        i = torch.arange(i0, i0 + ni, dtype=torch.int64, device=like)[None, None, :]
        j = torch.arange(j0, j0 + nj, dtype=torch.int64, device=like)[None, :, None]
        k = torch.arange(k0, k0 + nk, dtype=torch.int64, device=like)[:, None, None]
    return i, j, k, i + nx * (j + ny * k)


def _to_f32(x):
    if isinstance(x, np.ndarray):
        return np.ascontiguousarray(x.astype(np.float32))
    import torch
    return x.to(torch.float32).contiguous()


def _to_f64(x):
    if isinstance(x, np.ndarray):
        return x.astype(np.float64)
    import torch
    return x.to(torch.float64)


@dataclass(frozen=True)
class Source:
    comp: int                       # 0..2 = Ex, Ey, Ez
    box: Tuple[int, int, int, int, int, int]   # i0, j0, k0, ni, nj, nk
    amp: np.ndarray = field(repr=False, compare=False)    # (nk, nj, ni) float32
    wave: np.ndarray = field(repr=False, compare=False)   # (nwave,) float32


@dataclass(frozen=True)
class Workload:
    name: str
    n: Tuple[int, int, int]
    d: Tuple[float, float, float]
    boundary: Tuple[int, int, int]
    steps: int
    fields: str          # "uniform" (U[-1,1), low-wall tangential E zeroed) | "zero"
    coeffs: str          # "none" | "blocks" | "waveguide" | "lossy"
    source: str          # "none" | "dipole" | "sheet"
    seed: int = 1234
    courant: float = 0.5

    @property
    def dt(self) -> float:
        """Courant number 0.5 everywhere: dt = 0.5/sqrt(sum 1/d_a^2) (SURVEY.md 8(c) reading #12)."""
        return self.courant / math.sqrt(sum(1.0 / (x * x) for x in self.d))

    @property
    def cells(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]

    @property
    def has_coeff_arrays(self) -> bool:
        return self.coeffs != "none"

    def scaled(self, n, steps=None, name=None) -> "Workload":
        """Same recipe on another grid (parity tests run reduced sizes of every config)."""
        return replace(self, n=tuple(n), steps=self.steps if steps is None else steps,
                       name=name or f"{self.name}@{n[0]}x{n[1]}x{n[2]}")


def config(idx: int, size: Optional[int] = None) -> Workload:
    """BASELINE.json configs[idx] (0-based).  configs[3] is a size sweep: pass `size`."""
    if idx == 0:
        return Workload("C1-vacuum64", (64, 64, 64), (1, 1, 1), (PEC,) * 3, 100, "uniform", "none", "none")
    if idx == 1:
        return Workload("C2-blocks256", (256, 256, 256), (1, 1, 1), (PEC,) * 3, 1000, "zero", "blocks", "dipole")
    if idx == 2:
        return Workload("C3-waveguide", (512, 512, 256), (1, 1, 1), (PERIODIC, PEC, PEC), 2000, "zero", "waveguide", "sheet")
    if idx == 3:
        s = int(size or 256)
        return Workload(f"C4-vacuum{s}", (s, s, s), (1, 1, 1), (PEC,) * 3, 200, "uniform", "none", "none")
    if idx == 4:
        return Workload("C5-lossy", (1536, 1536, 768), (1, 1, 0.5), (PEC,) * 3, 500, "zero", "lossy", "dipole")
    raise IndexError(idx)


C4_SIZES = (64, 128, 256, 512, 768, 1024)


# ----------------------------------------------------------------------------------------------
# fields
# ----------------------------------------------------------------------------------------------
def _grouped(ts):
    """Device tensors only: the same values as views into ONE block, at a uniform 256-byte aligned stride.  The C ABI still
    receives one pointer per component; at a uniform stride between them the library fetches all components of
    a shell piece with a single 4-D TMA box (include/fdtd.h, fdtd_set_fields / fdtd_set_coeffs)."""
    import torch
    shape, cells = tuple(ts[0].shape), ts[0].numel()
    stride = (cells + 63) // 64 * 64              # every component stays 256-byte aligned
    block = torch.empty(len(ts) * stride, dtype=ts[0].dtype, device=ts[0].device)
    out = []
    for q in range(len(ts)):
        v = block[q * stride:q * stride + cells].view(shape)
        v.copy_(ts[q])
        ts[q] = None
        out.append(v)
    return out


_SLAB_CELLS = 1 << 26      # device arrays larger than this are generated slab by slab (the generators' int64 temporaries
                           # are several times the size of a component: 81 GiB config 5 would not fit beside them)


def _slabwise(gen, w, device, ncomp):
    """Run `gen(w, window, device)` (-> list of ncomp tensors for the window) over z slabs of the whole grid and return
    ncomp views of one block at a uniform 256-byte aligned stride (see _grouped); None entries pass through."""
    import torch
    nx, ny, nz = w.n
    cells = nx * ny * nz
    stride = (cells + 63) // 64 * 64
    block = torch.empty(ncomp * stride, dtype=torch.float32, device=device)
    out = [block[q * stride:q * stride + cells].view(nz, ny, nx) for q in range(ncomp)]
    nk = max(1, _SLAB_CELLS // (nx * ny))
    for k0 in range(0, nz, nk):
        kk = min(nk, nz - k0)
        part = gen(w, (0, 0, k0, nx, ny, kk), device)
        for q in range(ncomp):
            out[q][k0:k0 + kk].copy_(part[q])
        del part
    return out


def make_fields(w: Workload, window=None, device=None):
    """-> (E, H): two lists of three float32 arrays of shape (nk, nj, ni) for `window` (default whole grid).
    device=None: numpy; else torch tensors on that device (bit-identical values)."""
    if device is not None and window is None and w.cells > _SLAB_CELLS:
        g = _slabwise(lambda ww, win, dev: sum(make_fields(ww, win, dev), []), w, device, 6)
        return g[:3], g[3:]
    i, j, k, idx = _lin_index(w.n, window, like=device)
    shape = tuple(idx.shape)
    if w.fields == "zero":
        if device is None:
            return ([np.zeros(shape, np.float32) for _ in range(3)], [np.zeros(shape, np.float32) for _ in range(3)])
        import torch
        return (_grouped([torch.zeros(shape, dtype=torch.float32, device=device) for _ in range(3)]),
                _grouped([torch.zeros(shape, dtype=torch.float32, device=device) for _ in range(3)]))
    assert w.fields == "uniform"
    coords = (i, j, k)
    E, H = [], []
    for a in range(3):
        m = hash24(w.seed, AID_E[a], idx)
        v = _to_f32(m) * np.float32(2.0 ** -23) - np.float32(1.0)          # exact in fp32: U[-1,1) on a 2^-23 lattice
        # tangential E on the low PEC walls is frozen by the method; the generator zeroes it (reading #5)
        for b in range(3):
            if b != a and w.boundary[b] == PEC:
                v = v * _to_f32(coords[b] != 0)
        E.append(_to_f32(v))
        m = hash24(w.seed, AID_H[a], idx)
        H.append(_to_f32(_to_f32(m) * np.float32(2.0 ** -23) - np.float32(1.0)))
    if device is not None:
        E, H = _grouped(E), _grouped(H)
    return E, H


# ----------------------------------------------------------------------------------------------
# coefficients:  E_a <- ca_a E_a + cb_a curl_a H ;   generator side  ca=(2eps-sigma dt)/(2eps+sigma dt),
# cb = 2dt/(2eps+sigma dt)  <=>  cb = dt(1+ca)/(2eps)   (SURVEY.md 8(c) reading #2)
# ----------------------------------------------------------------------------------------------
def waveguide_rect(n):
    """Core rectangle (j0, j1, k0, k1) of the strip waveguide: 50 wide x 22 tall at 512x512x256, scaled."""
    nx, ny, nz = n
    wy = max(2, round(ny * 50 / 512))
    wz = max(2, round(nz * 22 / 256))
    j0 = (ny - wy) // 2
    k0 = (nz - wz) // 2
    return j0, j0 + wy, k0, k0 + wz


def make_eps(w: Workload, window=None, device=None):
    """Relative permittivity per component, float64 arrays (three of them), or None for vacuum."""
    if w.coeffs == "none":
        return None
    i, j, k, idx = _lin_index(w.n, window, like=device)
    shape = tuple(idx.shape)
    if w.coeffs == "blocks":                       # C2: random 8^3-voxel blocks, eps in {1.0, 2.1, 12.1}
        nbx, nby = (w.n[0] + 7) // 8, (w.n[1] + 7) // 8
        bid = (i >> 3) + nbx * ((j >> 3) + nby * (k >> 3))
        sel = hash24(w.seed, AID_BLOCK, bid) % 3
        eps = _to_f64(sel == 0) * 1.0 + _to_f64(sel == 1) * 2.1 + _to_f64(sel == 2) * 12.1
        eps = eps + 0.0 * _to_f64(idx)
        return [eps, eps, eps]
    if w.coeffs == "waveguide":                    # C3: eps=12.1 core in eps=2.1 cladding, uniform along x
        j0, j1, k0, k1 = waveguide_rect(w.n)
        core = (j >= j0) & (j < j1) & (k >= k0) & (k < k1)
        eps = _to_f64(core) * 12.1 + _to_f64(~core) * 2.1 + 0.0 * _to_f64(idx)
        return [eps, eps, eps]
    if w.coeffs == "lossy":                        # C5: independent eps per cell per component, U[1, 12.1)
        return [1.0 + 11.1 * (_to_f64(hash24(w.seed, AID_EPS[a], idx)) * 2.0 ** -24) for a in range(3)]
    raise ValueError(w.coeffs)


def make_coeffs(w: Workload, window=None, device=None):
    """-> (ca, cb): lists of three float32 per-cell arrays, or (None, None) when the workload has uniform
    coefficients (ca = 1, cb = dt).  All six arrays are materialised and read even where ca == 1."""
    if device is not None and window is None and w.cells > _SLAB_CELLS and w.has_coeff_arrays:
        g = _slabwise(lambda ww, win, dev: sum(make_coeffs(ww, win, dev), []), w, device, 6)
        return g[:3], g[3:]
    eps = make_eps(w, window, device)
    if eps is None:
        return None, None
    dt = w.dt
    ca, cb = [], []
    for a in range(3):
        if w.coeffs == "lossy":
            _, _, _, idx = _lin_index(w.n, window, like=device)
            ca64 = 0.98 + 0.02 * (_to_f64(hash24(w.seed, AID_CA[a], idx)) * 2.0 ** -24)
        else:
            ca64 = eps[a] * 0.0 + 1.0
        cb64 = dt * (1.0 + ca64) / (2.0 * eps[a])
        ca.append(_to_f32(ca64))
        cb.append(_to_f32(cb64))
    if device is not None:
        g = _grouped(ca + cb)
        ca, cb = g[:3], g[3:]
    return ca, cb


def make_coeff_lut(w: Workload, window=None, device=None):
    """Material-index form of make_coeffs for the few-material workloads (C2 "blocks": eps in {1.0, 2.1, 12.1}; C3
    "waveguide": cladding 2.1 / core 12.1): -> (idx, ca_lut, cb_lut) with idx = three uint8 per-cell arrays and
    ca_lut, cb_lut float32 arrays of shape (3, nmat), such that ca_lut[a][idx[a]] == make_coeffs(w)[0][a] bit for bit
    (the same double expression, rounded once).  None for the other workloads."""
    if w.coeffs not in ("blocks", "waveguide"):
        return None
    i, j, k, idx = _lin_index(w.n, window, like=device)
    if w.coeffs == "blocks":
        nbx, nby = (w.n[0] + 7) // 8, (w.n[1] + 7) // 8
        bid = (i >> 3) + nbx * ((j >> 3) + nby * (k >> 3))
        sel = hash24(w.seed, AID_BLOCK, bid) % 3 + 0 * idx
        eps_of = [1.0, 2.1, 12.1]
    else:
        j0, j1, k0, k1 = waveguide_rect(w.n)
        core = (j >= j0) & (j < j1) & (k >= k0) & (k < k1)
        sel = core * 1 + 0 * idx
        eps_of = [2.1, 12.1]
    if isinstance(sel, np.ndarray):
        m = np.ascontiguousarray(sel.astype(np.uint8))
        mats = [m, m.copy(), m.copy()]
    else:
        import torch
        m = sel.to(torch.uint8).contiguous()
        mats = [m, m.clone(), m.clone()]
    ca_lut = np.ones((3, len(eps_of)), np.float32)
    cb_lut = np.array([[np.float32(w.dt * (1.0 + 1.0) / (2.0 * e)) for e in eps_of]] * 3, np.float32)
    return mats, ca_lut, cb_lut


# ----------------------------------------------------------------------------------------------
# sources (host tables, computed in double then rounded: oracle and GPU consume identical bits)
# ----------------------------------------------------------------------------------------------
def make_source(w: Workload) -> Optional[Source]:
    if w.source == "none":
        return None
    nx, ny, nz = w.n
    dt = w.dt
    t = np.arange(w.steps, dtype=np.float64)
    if w.source == "dipole":                       # C2 / C5: z-dipole Gaussian pulse at the centre, lambda0 = 40 cells
        t0, tau, lam0 = 120.0, 40.0, 40.0
        if w.steps < 240:                          # reduced runs: compress the pulse so it still fires
            t0, tau = w.steps / 3.0, max(2.0, w.steps / 9.0)
        wave = np.exp(-((t - t0) / tau) ** 2) * np.sin(2 * np.pi * dt * (t - t0) / lam0)
        amp = np.ones((1, 1, 1), np.float32)
        return Source(2, (nx // 2, ny // 2, nz // 2, 1, 1, 1), amp, wave.astype(np.float32))
    if w.source == "sheet":                        # C3: mode-like Gaussian sheet, E_y on the plane x = 16
        t0, tau, lam0 = 600.0, 200.0, 155.0
        if w.steps < 1200:
            t0, tau = w.steps / 3.0, max(2.0, w.steps / 9.0)
        wave = np.exp(-((t - t0) / tau) ** 2) * np.sin(2 * np.pi * dt * (t - t0) / lam0)
        j0, j1, k0, k1 = waveguide_rect(w.n)
        cy, cz = 0.5 * (j0 + j1 - 1), 0.5 * (k0 + k1 - 1)
        sy, sz = 0.5 * (j1 - j0), 0.5 * (k1 - k0)
        jj = np.arange(ny, dtype=np.float64)[None, :, None]
        kk = np.arange(nz, dtype=np.float64)[:, None, None]
        amp = np.exp(-((jj - cy) / sy) ** 2 - ((kk - cz) / sz) ** 2)      # (nz, ny, 1)
        if w.boundary[2] == PEC:
            amp[0, :, :] = 0.0                     # E_y at k = 0 is tangential to the low z wall: never driven
        return Source(1, (min(16, nx // 4), 0, 0, 1, ny, nz), amp.astype(np.float32), wave.astype(np.float32))
    raise ValueError(w.source)
