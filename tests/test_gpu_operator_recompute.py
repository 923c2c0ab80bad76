"""GPU check of the matrix-free operator that rebuilds the diagonal block in the kernel (option op_recompute = 1, the default;
csrc/operator_mf.cu op_mf_rc_kernel): A M^-1 v from the solver's preconditioned kernel against the two-step reference
apply_operator(apply_preconditioner(v)) — the un-preconditioned flux-form operator (parity with the oracle: test_gpu_implicit.py)
applied to M^-1 v from the stored inverse blocks — and against the kernel that loads M^-1 (op_recompute = 0).

Bar: 1e-12 of max|result| per element (the two differ in the rounding of M^-1 only: one is stored rounded, one rebuilt)."""
import numpy as np
import pytest

from helpers import make_gpu, small_random_state

pytestmark = pytest.mark.gpu

TOL = 1e-12


def _check(w, opts=None, K=20.0):
    rng = np.random.default_rng(11)
    V = rng.standard_normal((3, w["ny"], w["nx"]))
    dt = K * 0.4 * min(w["dx"], w["dy"]) / w["c"]
    base = dict(opts or {})
    ref_solver = make_gpu(w, dict(base, op_recompute=0))
    ref = ref_solver.apply_operator(dt, ref_solver.apply_preconditioner(dt, V))
    scale = np.max(np.abs(ref))
    for rc in (0, 1, 2):
        g = make_gpu(w, dict(base, op_recompute=rc, apply_operator_precond=1))
        got = g.apply_operator(dt, V)
        err = np.max(np.abs(got - ref)) / scale
        assert err <= TOL, f"op_recompute={rc}: scaled max-abs {err:.2e}"


@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 1, 0, 0), (0, 0, 2, 2), (1, 2, 2, 1), (2, 2, 1, 1), (2, 1, 0, 0), (1, 1, 1, 1), (2, 2, 2, 2)])
@pytest.mark.parametrize("shape", [(200, 70), (61, 47), (30, 5), (31, 66), (91, 130)])
def test_recomputed_block_all_boundaries(bc, shape):
    # several 30-column strips with a ragged last strip, one- and two-strip grids, more rows than one 64-row block
    nx, ny = shape
    _check(small_random_state(nx, ny, seed=3 + nx, bc=bc, sig_range=(-1.0, 1.0), dx=0.011, dy=0.017, c=1.3))


@pytest.mark.parametrize("shape", [(1, 40), (40, 1), (2, 2), (2, 37), (37, 2), (3, 3)])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (2, 2, 2, 2), (1, 1, 1, 1)])
def test_recomputed_block_degenerate_grids(bc, shape):
    nx, ny = shape
    _check(small_random_state(nx, ny, seed=17 + nx + ny, bc=bc))


@pytest.mark.parametrize("opts", [dict(well_balanced=0), dict(ap_mode=0), dict(eig_mode=1), dict(closure=1), dict(linearisation=1)])
def test_recomputed_block_scheme_switches(opts):
    # well_balanced = 0 carries the cell-centred source plane dF (Eq. 16)
    _check(small_random_state(97, 45, seed=29, bc=(1, 2, 0, 0), sig_range=(-1.0, 1.0)), opts)


def test_recomputed_block_with_matter_coupling_and_large_dt():
    w = small_random_state(123, 80, seed=31, bc=(0, 0, 2, 1), sig_range=(-1.0, 2.0))
    rng = np.random.default_rng(2)
    w["T"] = rng.uniform(0.5, 1.5, (w["ny"], w["nx"]))
    w["rho_cv"] = rng.uniform(0.5, 2.0, (w["ny"], w["nx"]))
    _check(w, K=200.0)


def test_recomputed_jacobian_with_clamped_and_nonpositive_cells():
    # |F| > cE in many cells (their J is the clamped closure's, taken from the stored planes), E <= 0 in a few, f = 1 exactly in a row
    w = small_random_state(157, 90, seed=41, fmax=1.7, bc=(0, 0, 2, 1), c=1.3)
    rng = np.random.default_rng(8)
    bad = rng.integers(0, w["nx"] * w["ny"], size=40)
    w["E"].reshape(-1)[bad] = -w["E"].reshape(-1)[bad]
    w["E"][7, :] = 2.0 ** rng.integers(-2, 3, w["nx"])
    w["F"][0, 7, :] = 0.0
    w["F"][1, 7, :] = w["c"] * w["E"][7, :]
    _check(w, K=5.0)


def test_solver_iteration_counts_do_not_depend_on_the_variant():
    import m1_workloads as wl
    w = wl.random_medium(256, seed=5)
    dt = 20 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    res = []
    for rc in (0, 1, 2):
        g = make_gpu(w, dict(op_recompute=rc))
        its, r = g.step_implicit(dt, 1e-10, 30, 2000)
        res.append((its, g.get_state()))
        assert r <= 1e-10
    for k in (1, 2):
        assert abs(res[0][0] - res[k][0]) <= 1
        for a, b in zip(res[0][1], res[k][1]):
            assert np.max(np.abs(a - b)) <= 1e-9 * np.max(np.abs(b))
