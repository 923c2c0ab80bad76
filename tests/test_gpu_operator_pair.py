"""GPU check of the two-application operator kernel (csrc/operator_mf.cu op_mf_rc2_kernel, option op_pair = 1, the default inside the
s-step Arnoldi block; op_mf_rc2g_kernel on grids with Dirichlet or outflow sides): out1 = A M^-1 v - theta1 v and out2 = A M^-1 out1 - theta2 out1 from
ONE pass over the coefficient planes, against the same two results from two passes of the single-application kernel (itself checked
against apply_operator(apply_preconditioner(v)) in test_gpu_operator_recompute.py and through it against the oracle) and against the
two-step reference built from the un-preconditioned operator and the stored inverse blocks.

Bar: 1e-12 of max|result| per element (the kernels differ in the rounding of M^-1: here the inverse is formed explicitly)."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_gpu, small_random_state

pytestmark = pytest.mark.gpu

TOL = 1e-12
PER = (0, 0, 0, 0)


def _reference(w, dt, V, t1, t2, opts):
    g = make_gpu(w, dict(opts, op_recompute=0))
    o1 = g.apply_operator(dt, g.apply_preconditioner(dt, V)) - t1 * V
    o2 = g.apply_operator(dt, g.apply_preconditioner(dt, o1)) - t2 * o1
    return o1, o2


def _check(w, opts=None, K=20.0, thetas=((0.0, 1.0), (1.0, 1.0), (0.25, 0.0)), expect_fused=True):
    rng = np.random.default_rng(13)
    V = rng.standard_normal((3, w["ny"], w["nx"]))
    dt = K * 0.4 * min(w["dx"], w["dy"]) / w["c"]
    opts = dict(opts or {})
    for t1, t2 in thetas:
        r1, r2 = _reference(w, dt, V, t1, t2, opts)
        a1, a2, fused = make_gpu(w, opts).apply_operator_pair(dt, V, t1, t2)
        b1, b2, fused0 = make_gpu(w, dict(opts, op_pair=0)).apply_operator_pair(dt, V, t1, t2)
        assert fused == expect_fused and not fused0
        for got, ref, name in ((a1, r1, "out1"), (a2, r2, "out2"), (b1, r1, "out1 (two passes)"), (b2, r2, "out2 (two passes)")):
            err = np.max(np.abs(got - ref)) / np.max(np.abs(ref))
            assert err <= TOL, f"{name}, theta = ({t1}, {t2}): scaled max-abs {err:.2e}"


@pytest.mark.parametrize("shape", [(4, 4), (5, 7), (28, 8), (29, 9), (56, 64), (57, 65), (200, 70), (61, 130), (300, 200)])
def test_pair_kernel_periodic_grids(shape):
    # one strip, a ragged second strip (28 columns per strip), exactly one / two 64-row blocks and one row more, rows and columns that wrap
    nx, ny = shape
    _check(small_random_state(nx, ny, seed=5 + nx, bc=PER, sig_range=(-1.0, 1.0), dx=0.011, dy=0.017, c=1.3))


@pytest.mark.parametrize("opts", [dict(well_balanced=0), dict(ap_mode=0), dict(eig_mode=1), dict(closure=1), dict(linearisation=1)])
def test_scheme_switches_take_two_passes(opts):
    # J is rebuilt from the reduced flux for the default scheme only (op_recompute = 2 falls back to 1 otherwise): no pair kernel
    _check(small_random_state(97, 45, seed=29, bc=PER, sig_range=(-1.0, 1.0)), opts, expect_fused=False, thetas=((0.0, 1.0),))


def test_pair_kernel_with_matter_coupling_and_large_dt():
    w = small_random_state(123, 80, seed=31, bc=PER, sig_range=(-1.0, 2.0))
    rng = np.random.default_rng(2)
    w["T"] = rng.uniform(0.5, 1.5, (w["ny"], w["nx"]))
    w["rho_cv"] = rng.uniform(0.5, 2.0, (w["ny"], w["nx"]))
    _check(w, K=200.0)


def test_pair_kernel_with_clamped_and_nonpositive_cells():
    # |F| > cE in many cells (their J is the clamped closure's, taken from the stored planes), E <= 0 in a few, f = 1 exactly in a row
    w = small_random_state(157, 90, seed=41, fmax=1.7, bc=PER, c=1.3)
    rng = np.random.default_rng(8)
    bad = rng.integers(0, w["nx"] * w["ny"], size=40)
    w["E"].reshape(-1)[bad] = -w["E"].reshape(-1)[bad]
    w["E"][7, :] = 2.0 ** rng.integers(-2, 3, w["nx"])
    w["F"][0, 7, :] = 0.0
    w["F"][1, 7, :] = w["c"] * w["E"][7, :]
    _check(w, K=5.0)


@pytest.mark.parametrize("bc", [(1, 1, 0, 0), (0, 0, 2, 2), (0, 0, 1, 1), (2, 2, 0, 0), (1, 2, 2, 1), (2, 1, 1, 2), (2, 2, 1, 1), (1, 1, 1, 1), (2, 2, 2, 2)])
@pytest.mark.parametrize("shape", [(200, 70), (61, 130), (30, 5), (29, 66), (91, 200), (4, 4)])
def test_pair_kernel_dirichlet_and_outflow_sides(bc, shape):
    # ghost lanes and ghost rows of BOTH applications, folded boundary columns / top row (outflow), the boundary faces of mf.xlo / mf.ylo;
    # one to four 64-row blocks (first, interior, last), ragged strips, grids narrower than one strip
    nx, ny = shape
    _check(small_random_state(nx, ny, seed=3 + nx + ny, bc=bc, sig_range=(-1.0, 1.0), dx=0.011, dy=0.017, c=1.3), thetas=((0.0, 1.0), (1.0, 0.5)))


def test_pair_kernel_boundaries_with_clamped_cells_and_large_dt():
    w = small_random_state(157, 90, seed=41, fmax=1.7, bc=(1, 2, 2, 1), c=1.3)
    rng = np.random.default_rng(8)
    w["E"][7, :] = 2.0 ** rng.integers(-2, 3, w["nx"])
    w["F"][0, 7, :] = 0.0
    w["F"][1, 7, :] = w["c"] * w["E"][7, :]
    _check(w, K=5.0)
    _check(small_random_state(123, 80, seed=31, bc=(2, 1, 2, 2), sig_range=(-1.0, 2.0)), K=200.0)


@pytest.mark.parametrize("shape", [(2, 2), (3, 40), (40, 3)])
@pytest.mark.parametrize("bc", [PER, (1, 2, 2, 1)])
def test_tiny_grids_take_two_passes(shape, bc):
    nx, ny = shape
    _check(small_random_state(nx, ny, seed=19, bc=bc), expect_fused=False, thetas=((1.0, 1.0),))


@pytest.mark.parametrize("recompute", [0, 1])
def test_pair_needs_the_rebuilt_operator(recompute):
    _check(small_random_state(64, 40, seed=23, bc=PER), dict(op_recompute=recompute), expect_fused=False, thetas=((0.0, 1.0),))


def test_solver_is_the_same_with_and_without_the_pair_kernel():
    # the bench medium, small: same iteration count, same residual history, states equal to rounding
    w = wl.random_medium(256, seed=5)
    dt = 20 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    out = []
    for pair in (1, 0):
        g = make_gpu(w, dict(op_pair=pair))
        its, res = g.step_implicit(dt, 1e-10, 30, 2000)
        out.append((its, res, g.get_state(), np.array(g.history())))
    (i1, r1, s1, h1), (i0, r0, s0, h0) = out
    assert r1 <= 1e-10 and r0 <= 1e-10 and i1 == i0
    k = min(len(h1), len(h0), 40)
    assert np.max(np.abs(np.log10(h1[1:k] / h0[1:k]))) <= 1e-3
    E1, F1 = s1; E0, F0 = s0
    assert np.linalg.norm(E1 - E0) <= 1e-10 * np.linalg.norm(E0) and np.linalg.norm(F1 - F0) <= 1e-10 * np.linalg.norm(F0)


@pytest.mark.parametrize("bc", [(1, 2, 2, 1), (0, 0, 2, 2), (2, 2, 0, 0)])
def test_pair_kernel_boundaries_on_a_grid_of_several_waves(bc):
    # 37 strips x 13 block rows: interior blocks (periodic code) and boundary blocks (general code) side by side in one grid
    w = wl.random_medium(1030, seed=77, ny=777)
    w["bc"] = bc
    _check(w, K=10.0, thetas=((1.0, 1.0),))
