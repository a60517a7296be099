"""Build the shared libraries in-tree with nvcc for sm_100a (nvcc cross-compiles without a GPU).

Product library:
    libfdtd_b200.so        -fmad=false (variant "nofma", the default everywhere): every operation of the update rounded
                           separately, BIT-EXACT against the fp32 oracle on every configuration and run length
Optional variant (not the product: its drift from the oracle exceeds 1e-5 max|field| on 1000-step runs):
    libfdtd_b200_fma.so    ptxas may contract mul+add into FMA (variant "fma", ~2 % faster)
Developer libraries (-DFDTD_DEBUG: timing probes, fault injection, time-level shadow arrays; never the product path):
    libfdtd_b200_dbg.so    -fmad=false -DFDTD_DEBUG   (perturbed-order, watchdog and level-shadow tests)
    libfdtd_b200_prof.so   -DFDTD_DEBUG -DFDTD_PROFILE (clock64 section timers, dumped to stderr by fdtd_destroy)

    python -m paper_2502_20610_b200.build [--force] [--verbose] [--all]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["absorber_kernels.cu", "fdtd_api.cu", "fdtd_noalloc.cu", "naive_kernels.cu", "pad_kernels.cu", "systolic_kernel.cu", "systolic_reg.cu", "systolic_tma.cu", "systolic_tma_by8.cu", "systolic_tma_h16.cu", "systolic_tma_lut.cu"]
HEADERS = ["fdtd_internal.h", "fdtd_types.h", "yee_update.h", "systolic_tile.cuh", os.path.join("..", "..", "include", "fdtd.h")]
LIBS = {
    "nofma": (os.path.join(HERE, "libfdtd_b200.so"), ["-fmad=false", "-DFDTD_NOFMA"]),
    "fma": (os.path.join(HERE, "libfdtd_b200_fma.so"), []),
    "dbg": (os.path.join(HERE, "libfdtd_b200_dbg.so"), ["-fmad=false", "-DFDTD_NOFMA", "-DFDTD_DEBUG"]),
    "prof": (os.path.join(HERE, "libfdtd_b200_prof.so"), ["-DFDTD_DEBUG", "-DFDTD_PROFILE"]),
}
DEFAULT = ("nofma", "fma", "dbg")
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "--ftz=false", "--prec-div=true", "--prec-sqrt=true",
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(lib):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, which=DEFAULT):
    """Compile what is stale (the variants side by side, nvcc --threads inside each); returns {variant: path}."""
    out, jobs = {}, []
    for key in which:
        lib, extra = LIBS[key]
        if force or _stale(lib):
            cmd = [_nvcc(), *NVCC_FLAGS, "--threads", "0", *extra, *(["-Xptxas", "-v"] if verbose else []),
                   "-o", lib + ".tmp", *[os.path.join(CSRC, s) for s in SOURCES]]
            jobs.append((key, lib, cmd, subprocess.Popen(cmd, cwd=CSRC, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        out[key] = lib
    failed = []
    for key, lib, cmd, proc in jobs:
        log, _ = proc.communicate()
        if verbose or proc.returncode != 0:
            sys.stderr.write(f"---- {key}\n{log}")
        if proc.returncode != 0:
            failed.append(" ".join(cmd))
        else:
            os.replace(lib + ".tmp", lib)
    if failed:
        raise RuntimeError("nvcc failed: " + failed[0])
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, which=tuple(LIBS) if "--all" in sys.argv else DEFAULT))
