"""CPU-side checks of the systolic schedule: the tile stage functions of csrc/systolic_tile.cuh (the code the
CUDA kernel runs) are driven by tests/emu under adversarial schedulers and must reproduce the oracle BIT-EXACTLY
(schedule invariance, SURVEY.md 8(c) pin P10: "the exact same update equations").  No GPU needed."""
import numpy as np
import pytest

from oracle.yee import PEC, PERIODIC, YeeOracle
from paper_2502_20610_b200 import workloads
from tests.emu import harness


def make_case(n, boundary, coeffs, source, seed, steps, d=(1, 1, 1)):
    w = workloads.Workload("t", tuple(n), tuple(d), tuple(boundary), steps, "uniform", coeffs, source, seed=seed)
    E, H = workloads.make_fields(w)
    ca, cb = workloads.make_coeffs(w)
    src = workloads.make_source(w)
    return w, E, H, ca, cb, src


def run_both(n, boundary, coeffs, source, box, T, steps, policy, ctas, seed=7, d=(1, 1, 1)):
    w, E, H, ca, cb, src = make_case(n, boundary, coeffs, source, seed, steps, d)
    Eo, Ho = [x.copy() for x in E], [x.copy() for x in H]
    orc = YeeOracle(w.n, w.d, w.dt, w.boundary, Eo, Ho, ca, cb, None, nthreads=2)
    if src is not None:
        orc.set_source(src.comp, src.box, src.amp, src.wave)
    orc.step(steps)
    rc, stages = harness.run(w.n, w.d, w.dt, w.boundary, E, H, ca, cb, None,
                             None if src is None else (src.comp, src.box, src.amp, src.wave),
                             box, T, steps, ctas=ctas, policy=policy, seed=seed)
    assert rc == 0, f"emulated launch failed rc={rc} (2 = deadlock)"
    for a in range(3):
        assert np.all(np.isfinite(E[a])) and np.all(np.isfinite(H[a]))
        assert np.array_equal(E[a], Eo[a]), f"E[{a}] differs: max {np.abs(E[a] - Eo[a]).max()}"
        assert np.array_equal(H[a], Ho[a]), f"H[{a}] differs: max {np.abs(H[a] - Ho[a]).max()}"
    return stages


@pytest.mark.parametrize("policy", [0, 1, 2, 3, 4])
def test_pec_vacuum_all_policies(policy):
    run_both((13, 11, 9), (PEC,) * 3, "none", "none", (4, 4, 4), T=5, steps=12, policy=policy, ctas=6)


@pytest.mark.parametrize("policy", [0, 1, 3])
def test_pec_coeffs_source_anisotropic(policy):
    run_both((20, 14, 10), (PEC,) * 3, "lossy", "dipole", (8, 8, 8), T=7, steps=15, policy=policy, ctas=5, d=(1, 1, 0.5))


@pytest.mark.parametrize("policy", [1, 2, 3, 4])
def test_periodic_x_ring_with_sheet_source(policy):
    # config-3 style: ring in x, PEC in y and z, sheet source, waveguide coefficients
    run_both((16, 12, 10), (PERIODIC, PEC, PEC), "waveguide", "sheet", (8, 4, 4), T=6, steps=13, policy=policy, ctas=9)


@pytest.mark.parametrize("boundary", [(PERIODIC,) * 3, (PEC, PERIODIC, PEC), (PEC, PEC, PERIODIC), (PERIODIC, PERIODIC, PEC)])
def test_other_periodic_combinations(boundary):
    run_both((9, 7, 6), boundary, "blocks", "dipole", (4, 4, 4), T=4, steps=9, policy=1, ctas=64)


def test_ring_shorter_than_depth_and_single_tile_ring():
    # T larger than the ring, and a ring made of a single tile that is its own upwind neighbour
    run_both((6, 9, 5), (PERIODIC, PEC, PEC), "none", "none", (4, 4, 4), T=11, steps=11, policy=1, ctas=8)
    run_both((3, 8, 6), (PERIODIC, PEC, PEC), "none", "none", (4, 4, 4), T=5, steps=10, policy=3, ctas=8)


def test_tile_larger_than_domain_and_thin_domain():
    run_both((5, 4, 3), (PEC,) * 3, "lossy", "dipole", (8, 8, 8), T=6, steps=8, policy=1, ctas=4)
    run_both((17, 1, 6), (PEC,) * 3, "none", "none", (8, 4, 4), T=4, steps=8, policy=2, ctas=4)


def test_production_box_shapes():
    # the boxes the GPU kernel is built with, several tiles per axis and a ragged tail
    run_both((40, 22, 20), (PEC,) * 3, "none", "none", (32, 16, 16), T=6, steps=6, policy=1, ctas=4)
    run_both((40, 22, 12), (PEC,) * 3, "blocks", "dipole", (32, 16, 8), T=5, steps=7, policy=4, ctas=4)
    run_both((20, 20, 20), (PERIODIC, PEC, PEC), "waveguide", "sheet", (16, 16, 16), T=5, steps=5, policy=3, ctas=4)


def test_few_ctas_still_progress():
    # one virtual CTA: tiles strictly one after another (every upwind tile has finished all its steps)
    run_both((11, 9, 8), (PEC,) * 3, "none", "none", (4, 4, 4), T=5, steps=10, policy=1, ctas=1)
