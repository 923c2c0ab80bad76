"""GPU parity for the semi-implicit step: explicit hyperbolic part, implicit sources."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, make_gpu, small_random_state, rel_l2, state_rel_l2

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("op", [0, 1])
@pytest.mark.parametrize("wb", [1, 0])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 2, 2, 1), (2, 2, 1, 1)])
def test_semi_implicit_matches_oracle(bc, wb, op):
    w = small_random_state(45, 31, seed=91, bc=bc, sig_range=(0.0, 3.0))       # c sigma dt up to ~10: stiff sources
    o, g = make_oracle(w, dict(well_balanced=wb)), make_gpu(w, dict(well_balanced=wb, operator=op))
    dt = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    for _ in range(3):
        io, ro = o.step_semi_implicit(dt, 1e-12, 30, 2000)
        ig, rg = g.step_semi_implicit(dt, 1e-12, 30, 2000)
        assert rg <= 1e-12
    assert state_rel_l2(g.get_state(), o.get_state()) <= 1e-10


def test_semi_implicit_equals_explicit_without_opacity_and_closed_form():
    w = wl.beam(64)                                     # sigma = 0: the paper's beam test runs semi-implicitly
    dt = wl.explicit_dt(w["dx"], w["dy"])
    g1, g2 = make_gpu(w), make_gpu(w)
    for _ in range(20):
        g1.step_explicit(dt)
        its, res = g2.step_semi_implicit(dt)
        assert its == 0
    assert state_rel_l2(g2.get_state(), g1.get_state()) <= 1e-13
    n = 12
    wu = dict(nx=n, ny=n, dx=1.0 / n, dy=1.0 / n, c=1.3, bc=(0, 0, 0, 0), E=np.full((n, n), 2.0),
              F=np.stack((np.full((n, n), 0.4), np.full((n, n), -0.3))), sigma_a=np.full((n, n), 5.0), sigma_s=np.full((n, n), 70.0))
    g = make_gpu(wu)
    g.step_semi_implicit(3.0, 1e-13, 30, 500)
    E, F = g.get_state()
    assert np.allclose(E, 2.0 / (1.0 + 1.3 * 3.0 * 5.0), rtol=1e-11) and np.allclose(F[0], 0.4 / (1.0 + 1.3 * 3.0 * 75.0), rtol=1e-10)


def test_semi_implicit_with_temperature_and_bicgstab():
    w = small_random_state(29, 23, seed=92, sig_range=(0.0, 2.0))
    rng = np.random.default_rng(6)
    w["T"] = np.exp(0.2 * rng.standard_normal((23, 29)))
    w["rho_cv"] = 10.0 ** rng.uniform(-0.5, 1.0, (23, 29))
    o, g = make_oracle(w, dict(krylov=1)), make_gpu(w, dict(krylov=1))
    dt = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    for _ in range(2):
        o.step_semi_implicit(dt, 1e-12, 30, 2000)
        g.step_semi_implicit(dt, 1e-12, 30, 2000)
    assert state_rel_l2(g.get_state(with_T=True), o.get_state(with_T=True)) <= 1e-10
