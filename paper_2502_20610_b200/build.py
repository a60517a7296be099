"""Build libfdtd_b200.so (default, FMA contraction allowed) and libfdtd_b200_nofma.so (-fmad=false: bit-exact
against the fp32 oracle) in-tree with nvcc for sm_100a.  nvcc cross-compiles without a GPU.

    python -m paper_2502_20610_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["fdtd_api.cu", "naive_kernels.cu", "systolic_kernel.cu", "systolic_reg.cu", "systolic_tma.cu"]
HEADERS = ["fdtd_internal.h", "fdtd_types.h", "yee_update.h", "systolic_tile.cuh", os.path.join("..", "..", "include", "fdtd.h")]
LIBS = {
    "fma": (os.path.join(HERE, "libfdtd_b200.so"), []),
    "nofma": (os.path.join(HERE, "libfdtd_b200_nofma.so"), ["-fmad=false", "-DFDTD_NOFMA"]),
    # developer build: clock64 section timers inside the systolic kernel, dumped to stderr by fdtd_destroy
    "prof": (os.path.join(HERE, "libfdtd_b200_prof.so"), ["-DFDTD_PROFILE"]),
}
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


def build(force=False, verbose=False, which=("fma", "nofma")):
    """Compile what is stale; returns {variant: path}."""
    out = {}
    for key in which:
        lib, extra = LIBS[key]
        if force or _stale(lib):
            cmd = [_nvcc(), *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []),
                   "-o", lib + ".tmp", *[os.path.join(CSRC, s) for s in SOURCES]]
            res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
            if verbose or res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
            if res.returncode != 0:
                raise RuntimeError("nvcc failed: " + " ".join(cmd))
            os.replace(lib + ".tmp", lib)
        out[key] = lib
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
