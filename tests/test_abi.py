"""The C-ABI library loads and exports every symbol include/fdtd.h declares; host-only entry points work.
No compute call is made here (no GPU in the CPU suite)."""
import os
import re

import pytest

from paper_2502_20610_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libs():
    build.build()
    return {v: binding.load(v) for v in ("fma", "nofma")}


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "fdtd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fdtd_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(libs):
    names = declared_symbols()
    assert len(names) >= 19
    for lib in libs.values():
        for name in names:
            assert hasattr(lib, name), name
    assert set(names) == set(binding.EXPORTS)


def test_build_info_names_the_variant(libs):
    assert b"fmad=true" in libs["fma"].fdtd_build_info()
    assert b"fmad=false" in libs["nofma"].fdtd_build_info()


def test_plan_tiles_counts():
    # PEC: ceil((n+T)/N) tiles (launch ramp, a11); periodic: ceil(n/N) (ring)
    assert binding.plan_tiles((256, 256, 256), (0, 0, 0), (31, 15, 15), 32) == (10, 20, 20)
    assert binding.plan_tiles((512, 512, 256), (1, 0, 0), (31, 15, 7), 32) == (17, 37, 42)
    assert binding.plan_tiles((5, 4, 3), (0, 1, 0), (7, 7, 7), 6) == (2, 1, 2)
    with pytest.raises(binding.FdtdError):
        binding.plan_tiles((0, 4, 3), (0, 0, 0), (7, 7, 7), 6)


@pytest.mark.parametrize("n,bnd,N,T", [(37, 0, 7, 9), (16, 1, 7, 6), (6, 1, 3, 11), (5, 0, 15, 4), (23, 1, 7, 5)])
def test_plan_owner_partitions_space_time(n, bnd, N, T):
    """Every (cell, step) has exactly one owner, offsets stay inside the tile, and the owner of a cell moves
    downwind by at most one tile per step (regions slide one cell per step along the diagonal)."""
    nb = binding.plan_tiles((n, 1, 1), (bnd, 0, 0), (N, 1, 1), T)[0]
    for s in range(T):
        seen = {}
        for g in range(n):
            tile, off = binding.plan_owner(n, bnd, N, T, g, s)
            assert 0 <= tile < nb and 0 <= off < N
            seen.setdefault(tile, []).append(off)
            if s > 0:
                prev, _ = binding.plan_owner(n, bnd, N, T, g, s - 1)
                step = (tile - prev) % nb if bnd else tile - prev
                assert step in (0, 1)
        for offs in seen.values():          # a tile's cells are contiguous: offsets are distinct
            assert len(set(offs)) == len(offs)
    if not bnd:                              # PEC: cell g at step s sits at position g+s of the moving frame
        assert binding.plan_owner(n, bnd, N, T, n - 1, T - 1) == ((n + T - 2) // N, (n + T - 2) % N)


def test_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    with pytest.raises(binding.FdtdError) as e:
        binding.Fdtd((8, 8, 8), (1, 1, 1), 0.25, (0, 0, 0))
    assert e.value.code == binding.ECUDA


def test_missing_library_raises(monkeypatch):
    monkeypatch.setitem(binding._LIBFILES, "ghost", "libdoes_not_exist.so")
    with pytest.raises(FileNotFoundError):
        binding.load("ghost")
