"""fdtd_step_noalloc: the systolic kernel for hosts that cannot let the library allocate device memory.

Some users of this library own every byte of HBM themselves (an application that hands the whole device to its own memory
pool before it loads us) or step inside a loop that must never hit the device-wide stall of a cudaMalloc / cudaFree.  They
cannot use fdtd_create / fdtd_step, which allocate the schedule's bookkeeping (hand-off flags, claim counters, claim order,
watchdog word).  fdtd_step_noalloc runs the same kernel on a fixed array compiled into the library.  What has to hold, and
is checked here:

  * same result as the context path, bit for bit (the product build's bar everywhere in tests/), on two calls in a row:
    the second call finds the array full of the first call's flags and claim order and must not be fooled by them (the
    calls use different launch shapes, so a stale table or an uncleared flag would show);
  * jobs beyond the fixed array's capacity, and grids that would need the padded working copy, are refused with a message
    that says why, before anything touches the GPU.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a problem in this side entrance should not
hide the parity suites.  It passes alone in a fresh process and after the other files (it shares nothing with them but the
library, and the entry point clears what it needs on every call)."""
import numpy as np
import pytest

from paper_2502_20610_b200 import binding, workloads
from paper_2502_20610_b200.workloads import PEC, Workload

T = 16                     # temporal depth of both paths: 40 steps = launches of 16, 16, 8; 24 steps = 16, 8
STEPS = (40, 24)           # the two consecutive calls

CASES = {
    # C5's recipe (lossy heterogeneous coefficients, anisotropic cells) on a grid of 4 x 4 x 8 tiles with ragged tails,
    # random fields so that every cell carries data
    "lossy-arrays": Workload("noalloc-lossy", (100, 45, 38), (1, 1, 0.5), (PEC,) * 3, 0, "uniform", "lossy", "none"),
    # C1's recipe: vacuum, no coefficient arrays (the kernel's other instantiation)
    "vacuum-uniform": Workload("noalloc-vacuum", (64, 64, 64), (1, 1, 1), (PEC,) * 3, 0, "uniform", "none", "none"),
}


def _clone_all(ts, grouped):
    """Copies of three tensors: as views of one block (the library then fetches them with one 4-D box) or as three
    separate allocations (one 3-D box each)."""
    if ts is None:
        return None
    return workloads._grouped([t.clone() for t in ts]) if grouped else [t.clone() for t in ts]


@pytest.mark.gpu
@pytest.mark.parametrize("grouped", [True, False], ids=["one-block", "separate-arrays"])
@pytest.mark.parametrize("case", sorted(CASES))
def test_two_calls_in_a_row_match_the_context_path(cuda_device, case, grouped):
    import torch
    w = CASES[case]
    E0, H0 = workloads.make_fields(w, device=cuda_device)
    ca, cb = workloads.make_coeffs(w, device=cuda_device)

    # the existing path: a context, the same kernel and depth, state read after 40 and after 40 + 24 steps
    Er, Hr = _clone_all(E0, True), _clone_all(H0, True)
    sim = binding.Fdtd(w.n, w.d, w.dt, w.boundary)
    sim.set_fields(Er, Hr)
    if ca is not None:
        sim.set_coeffs(ca, cb, None)
    sim.set_kernel(binding.KERNEL_SYSTOLIC, None, T)
    want = []
    for n in STEPS:
        sim.step(n)
        sim.sync()
        want.append([t.clone() for t in Er + Hr])
    sim.close()

    # the entry point that allocates nothing, on its own copies of the inputs
    E, H = _clone_all(E0, grouped), _clone_all(H0, grouped)
    can, cbn = (_clone_all(ca, grouped), _clone_all(cb, grouped)) if ca is not None else (None, None)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for call, n in enumerate(STEPS):
        binding.step_noalloc(w.n, w.d, w.dt, E, H, can, cbn, None, nsteps=n, T=T)
        for got, ref, name in zip(E + H, want[call], ("Ex", "Ey", "Ez", "Hx", "Hy", "Hz")):
            assert torch.isfinite(got).all()
            assert float(ref.abs().max()) > 0.0                       # the comparison is not zero against zero
            assert torch.equal(got, ref), f"call {call + 1}, {name}: max diff {(got - ref).abs().max().item():.3e}"
    assert torch.cuda.memory_allocated() == before                     # torch's own view: nothing of ours came from its pool


@pytest.mark.gpu
def test_first_call_matches_the_oracle(cuda_device):
    """The context path is itself held to the oracle elsewhere; one direct check so that this file stands alone."""
    from oracle.yee import YeeOracle
    w = CASES["lossy-arrays"]
    E, H = workloads.make_fields(w, device=cuda_device)
    ca, cb = workloads.make_coeffs(w, device=cuda_device)
    Eo, Ho = workloads.make_fields(w)
    cao, cbo = workloads.make_coeffs(w)
    binding.step_noalloc(w.n, w.d, w.dt, E, H, ca, cb, None, nsteps=STEPS[0], T=T)
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, Eo, Ho, cao, cbo, None)
    orc.step(STEPS[0])
    for got, ref in zip(E + H, Eo + Ho):
        assert np.array_equal(got.cpu().numpy(), ref)


def _host_arrays(n=4 * 4 * 4):
    return [np.zeros(n, np.float32) for _ in range(3)]


def test_job_beyond_the_static_array_is_refused_with_a_reason():
    """2048^3 at depth 128 is 71 x 146 x 311 tiles, far beyond FDTD_NOALLOC_MAX_TILES: refused on the host, the pointers
    are never looked at (they are small host arrays here) and no GPU is needed."""
    tiles = binding.plan_tiles((2048, 2048, 2048), (0, 0, 0), (31, 15, 7), 128)
    assert tiles[0] * tiles[1] * tiles[2] > binding.NOALLOC_MAX_TILES
    with pytest.raises(binding.FdtdError) as e:
        binding.step_noalloc((2048, 2048, 2048), (1, 1, 1), 0.25, _host_arrays(), _host_arrays(), nsteps=500, T=128, stream=0)
    assert e.value.code == binding.EINVAL
    assert "FDTD_NOALLOC_MAX_TILES" in str(e.value) and "smaller T" in str(e.value)
    # the same grid in shallow launches fits the limit as far as the size check goes (then fails later for lack of a GPU
    # or of real device pointers -- not tried here); the limit itself is what fdtd_plan_tiles says
    t8 = binding.plan_tiles((512, 512, 512), (0, 0, 0), (31, 15, 7), 128)
    assert t8[0] * t8[1] * t8[2] == 83076 <= binding.NOALLOC_MAX_TILES


def test_grid_that_needs_a_padded_copy_is_refused():
    with pytest.raises(binding.FdtdError) as e:
        binding.step_noalloc((30, 8, 8), (1, 1, 1), 0.25, _host_arrays(), _host_arrays(), nsteps=4, stream=0)
    assert e.value.code == binding.EINVAL and "multiple of 4" in str(e.value)
    with pytest.raises(binding.FdtdError) as e:      # ca without cb
        binding.step_noalloc((32, 8, 8), (1, 1, 1), 0.25, _host_arrays(), _host_arrays(), ca=_host_arrays(), nsteps=4, stream=0)
    assert e.value.code == binding.EINVAL


def test_without_a_gpu_it_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    with pytest.raises(binding.FdtdError) as e:
        binding.step_noalloc((32, 8, 8), (1, 1, 1), 0.25, _host_arrays(32 * 8 * 8), _host_arrays(32 * 8 * 8), nsteps=4, stream=0)
    assert e.value.code == binding.ECUDA
