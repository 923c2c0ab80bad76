"""GPU parity for BiCGStab (the paper's Krylov method), option krylov = 1."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, make_gpu, small_random_state, rel_l2, state_rel_l2, bicgstab_count_ok

pytestmark = pytest.mark.gpu
BCS = [(0, 0, 0, 0), (1, 1, 0, 0), (1, 2, 2, 1), (2, 2, 1, 1)]


def _dt(w, k):
    return k * wl.explicit_dt(w["dx"], w["dy"], w["c"])


@pytest.mark.parametrize("op", [0, 1])
@pytest.mark.parametrize("bc", BCS)
def test_bicgstab_matches_oracle(bc, op):
    w = small_random_state(37, 29, seed=71, bc=bc, sig_range=(-1.0, 2.0))
    o, g = make_oracle(w, dict(krylov=1)), make_gpu(w, dict(krylov=1, operator=op))
    dt = _dt(w, 50.0)
    io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
    ig, rg = g.step_implicit(dt, 1e-10, 30, 4000)
    assert ro <= 1e-10 and rg <= 1e-10
    assert state_rel_l2(g.get_state(), o.get_state()) <= 1e-8
    assert bicgstab_count_ok(ig, io)


def test_bicgstab_matches_dense_direct_solve():
    w = small_random_state(9, 8, seed=77, bc=(1, 2, 0, 0))
    o, g = make_oracle(w), make_gpu(w, dict(krylov=1))
    dt = _dt(w, 100.0)
    M, b = o.dense_matrix(dt)
    x = np.linalg.solve(M, b).reshape(3, w["ny"], w["nx"])
    its, res = g.step_implicit(dt, 1e-12, 30, 2000)
    E, F = g.get_state()
    assert res <= 1e-12 and 0 < its < 2000
    assert rel_l2(np.concatenate((E[None], F)), x) <= 1e-9


def test_bicgstab_config3_window_and_gmres_agree():
    w = wl.random_medium(256, seed=1234)
    dt = _dt(w, 100.0)
    gb, gg = make_gpu(w, dict(krylov=1)), make_gpu(w)
    ib, rb = gb.step_implicit(dt, 1e-10, 30, 4000)
    ig, rg = gg.step_implicit(dt, 1e-10, 30, 4000)
    assert rb <= 1e-10 and rg <= 1e-10 and ib < ig
    assert state_rel_l2(gb.get_state(), gg.get_state()) <= 1e-8
    o = make_oracle(w, dict(krylov=1))
    io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
    assert state_rel_l2(gb.get_state(), o.get_state()) <= 1e-8
    h = gb.history()
    assert h[-1] <= 1e-10 and len(h) >= ib + 1


def test_bicgstab_maxit_zero_iterations_and_temperature():
    w = small_random_state(40, 30, seed=44)
    g = make_gpu(w, dict(krylov=1))
    its, res = g.step_implicit(_dt(w, 200.0), 1e-14, 30, 7)
    assert its == 7 and res > 1e-14
    w2 = small_random_state(16, 16, seed=45)
    w2["F"][:] = 0.0; w2["E"][:] = 2.0; w2["sigma_a"][:] = 0.0
    g2 = make_gpu(w2, dict(krylov=1))
    assert g2.step_implicit(_dt(w2, 10.0), 1e-10, 30, 100)[0] == 0
    w3 = small_random_state(29, 23, seed=64, sig_range=(-1.0, 1.0))
    rng = np.random.default_rng(5)
    w3["T"] = np.exp(0.2 * rng.standard_normal((23, 29)))
    w3["rho_cv"] = 10.0 ** rng.uniform(-0.5, 1.0, (23, 29))
    o3, g3 = make_oracle(w3, dict(krylov=1)), make_gpu(w3, dict(krylov=1))
    o3.step_implicit(_dt(w3, 30.0), 1e-11, 30, 4000)
    g3.step_implicit(_dt(w3, 30.0), 1e-11, 30, 4000)
    assert state_rel_l2(g3.get_state(with_T=True), o3.get_state(with_T=True)) <= 1e-8
