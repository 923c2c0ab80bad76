"""GPU parity for the Newton-Raphson iteration on the implicit step."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, make_gpu, small_random_state, rel_l2, state_rel_l2

pytestmark = pytest.mark.gpu


def _dt(w, k):
    return k * wl.explicit_dt(w["dx"], w["dy"], w["c"])


@pytest.mark.parametrize("op", [0, 1])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 2, 0, 0), (2, 2, 1, 1)])
def test_newton_matches_oracle(bc, op):
    w = small_random_state(33, 26, seed=61, bc=bc, sig_range=(-1.0, 1.5))
    o, g = make_oracle(w), make_gpu(w, dict(operator=op))
    dt = _dt(w, 20.0)
    io, no, ro, uo = o.step_implicit_newton(dt, 1e-11, 30, 4000, 1e-9, 30)
    ig, ng, rg, ug = g.step_implicit_newton(dt, 1e-11, 30, 4000, 1e-9, 30)
    assert ng == no and ug <= 1e-9 and rg <= 1e-11
    assert abs(ig - io) <= max(3, 0.03 * io)
    assert state_rel_l2(g.get_state(), o.get_state()) <= 1e-8


def test_newton_converges_to_the_nonlinear_backward_euler_solution_on_the_gpu():
    # the CUDA path's converged iterate against the CUDA path's own non-linear residual: U - U^n + dt R(U) = 0
    w = small_random_state(64, 48, seed=62, sig_range=(-1.0, 1.5))
    g = make_gpu(w)
    dt = _dt(w, 30.0)
    its, nn, res, upd = g.step_implicit_newton(dt, 1e-12, 30, 4000, 1e-11, 40)
    assert 2 <= nn < 40 and upd <= 1e-11
    E, F = g.get_state()
    RE, RF = g.residual()
    U, R = np.concatenate((E[None], F)), np.concatenate((RE[None], RF))
    U0 = np.concatenate((w["E"][None], w["F"]))
    assert np.linalg.norm(U - U0 + dt * R) <= 1e-10 * np.linalg.norm(U)


def test_one_newton_iteration_is_the_linearised_step():
    w = small_random_state(40, 30, seed=63)
    g1, g2 = make_gpu(w), make_gpu(w)
    dt = _dt(w, 25.0)
    i1, r1 = g1.step_implicit(dt, 1e-10, 30, 4000)
    i2, nn, r2, upd = g2.step_implicit_newton(dt, 1e-10, 30, 4000, 0.0, 1)
    assert nn == 1 and i1 == i2
    assert all(np.array_equal(a, b) for a, b in zip(g1.get_state(), g2.get_state()))   # deterministic reductions: bit-equal


def test_newton_with_temperature_matches_oracle():
    w = small_random_state(29, 23, seed=64, sig_range=(-1.0, 1.0))
    rng = np.random.default_rng(5)
    w["T"] = np.exp(0.2 * rng.standard_normal((23, 29)))
    w["rho_cv"] = 10.0 ** rng.uniform(-0.5, 1.0, (23, 29))
    o, g = make_oracle(w), make_gpu(w)
    dt = _dt(w, 15.0)
    io, no, ro, uo = o.step_implicit_newton(dt, 1e-11, 30, 4000, 1e-9, 30)
    ig, ng, rg, ug = g.step_implicit_newton(dt, 1e-11, 30, 4000, 1e-9, 30)
    assert ng == no
    assert state_rel_l2(g.get_state(with_T=True), o.get_state(with_T=True)) <= 1e-8
