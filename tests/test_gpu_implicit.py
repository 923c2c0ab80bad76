"""GPU parity, rows a5-a7: assembly + block-stencil operator + GMRES(m)/block-Jacobi against the oracle.

Bars (north_star): implicit state relative L2 <= 1e-8 with the GMRES residual converged to 1e-10; the assembled
operator itself is compared to round-off."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, make_gpu, small_random_state, rel_l2, state_rel_l2

pytestmark = pytest.mark.gpu

TOL_IMPLICIT = 1e-8
BCS = [(0, 0, 0, 0), (1, 1, 0, 0), (0, 0, 2, 2), (1, 2, 2, 1), (2, 2, 1, 1)]


def _dt(w, k=1.0):
    return k * wl.explicit_dt(w["dx"], w["dy"], w["c"])


OPS = [0, 1]   # 0: pre-multiplied block stencil, 1: matrix-free coefficient planes


@pytest.mark.parametrize("op", OPS)
@pytest.mark.parametrize("bc", BCS)
@pytest.mark.parametrize("wb", [1, 0])
def test_operator_and_rhs_match_oracle(bc, wb, op):
    # A V (assembly kernel + scaled block-stencil + diagonal multiply) vs the oracle's flux-form operator
    w = small_random_state(41, 23, seed=31, dx=0.013, dy=0.021, c=1.3, bc=bc)
    o, g = make_oracle(w, dict(well_balanced=wb)), make_gpu(w, dict(well_balanced=wb, operator=op))
    dt = _dt(w, 30.0)
    rng = np.random.default_rng(5)
    V = rng.standard_normal((3, w["ny"], w["nx"]))
    want = o.apply_linear(dt, V, mode=0)
    got, b = g.apply_operator(dt, V, with_b=True)
    assert rel_l2(got, want) <= 1e-13
    U = np.concatenate((w["E"][None], w["F"]))
    want_b = U - o.apply_linear(dt, np.zeros_like(U), mode=1)
    assert rel_l2(b, want_b) <= 1e-13


@pytest.mark.parametrize("op", OPS)
def test_operator_with_clamped_cells_and_tiny_grids(op):
    for (nx, ny, fmax) in [(6, 5, 1.6), (1, 7, 0.9), (7, 1, 0.9), (2, 2, 0.9), (1, 1, 0.5), (300, 3, 0.9), (127, 70, 0.9)]:
        w = small_random_state(nx, ny, seed=22 + nx, fmax=fmax)
        o, g = make_oracle(w), make_gpu(w, dict(operator=op))
        V = np.random.default_rng(1).standard_normal((3, ny, nx))
        assert rel_l2(g.apply_operator(0.3, V), o.apply_linear(0.3, V)) <= 1e-13


@pytest.mark.parametrize("op", OPS)
@pytest.mark.parametrize("bc", BCS)
def test_implicit_step_small_all_boundaries(bc, op):
    w = small_random_state(37, 29, seed=41, bc=bc, sig_range=(-1.0, 2.0))
    o, g = make_oracle(w), make_gpu(w, dict(operator=op))
    dt = _dt(w, 50.0)
    io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
    ig, rg = g.step_implicit(dt, 1e-10, 30, 4000)
    assert ro <= 1e-10 and rg <= 1e-10
    assert state_rel_l2(g.get_state(), o.get_state()) <= TOL_IMPLICIT
    assert abs(ig - io) <= max(2, 0.02 * io)


def test_gmres_solution_matches_dense_direct_solve():
    # P10 on the GPU side: tiny grid, dense LU of the ORACLE's assembled matrix
    w = small_random_state(9, 8, seed=77, bc=(1, 2, 0, 0))
    o, g = make_oracle(w), make_gpu(w)
    dt = _dt(w, 100.0)
    M, b = o.dense_matrix(dt)
    x = np.linalg.solve(M, b).reshape(3, w["ny"], w["nx"])
    its, res = g.step_implicit(dt, 1e-12, 30, 2000)
    E, F = g.get_state()
    assert res <= 1e-12
    assert rel_l2(np.concatenate((E[None], F)), x) <= 1e-9


@pytest.mark.parametrize("ortho", [1, 2])
@pytest.mark.parametrize("restart", [5, 17, 30, 40])
def test_restart_lengths_and_orthogonalisation(restart, ortho):
    # restart > 16 (vectors_per_pass) exercises the two-pass multi-vector kernels
    w = small_random_state(50, 34, seed=43)
    o, g = make_oracle(w), make_gpu(w, dict(orthogonalisation=ortho))
    dt = _dt(w, 40.0)
    io, ro = o.step_implicit(dt, 1e-10, restart, 4000)
    ig, rg = g.step_implicit(dt, 1e-10, restart, 4000)
    assert rg <= 1e-10
    assert state_rel_l2(g.get_state(), o.get_state()) <= TOL_IMPLICIT
    assert abs(ig - io) <= max(3, 0.05 * io)
    h = g.history()
    assert len(h) >= ig + 1 and h[-1] <= 1e-10


def test_maxit_is_respected_and_not_an_error():
    w = small_random_state(40, 30, seed=44)
    g = make_gpu(w)
    its, res = g.step_implicit(_dt(w, 200.0), 1e-14, 10, 7)
    assert its == 7 and res > 1e-14


def test_steady_state_returns_zero_iterations():
    w = small_random_state(16, 16, seed=45)
    w["F"][:] = 0.0
    w["E"][:] = 2.0
    w["sigma_a"][:] = 0.0
    g = make_gpu(w)
    its, res = g.step_implicit(_dt(w, 10.0), 1e-10, 30, 100)
    assert its == 0 and res <= 1e-10


@pytest.mark.parametrize("op", OPS)
def test_config1_gaussian_diffusion_20_steps(op):
    # BASELINE.json configs[0]: 64^2, sigma_s = 1e3, 20 implicit steps at 10x the explicit dt
    w = wl.gaussian_diffusion(64)
    o, g = make_oracle(w), make_gpu(w, dict(operator=op))
    dt = _dt(w, 10.0)
    for _ in range(20):
        io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
        ig, rg = g.step_implicit(dt, 1e-10, 30, 4000)
        assert rg <= 1e-10 and abs(ig - io) <= 2
    Eg, Fg = g.get_state()
    Eo, Fo = o.get_state()
    assert rel_l2(Eg, Eo) <= TOL_IMPLICIT
    assert np.linalg.norm(Fg - Fo) <= TOL_IMPLICIT * max(np.linalg.norm(Fo), np.linalg.norm(Eo))
    # and the CUDA result itself against the analytic diffusion solution (pin P3), D = c/(3 sigma)
    t = 20 * dt
    s2 = w["s0"] ** 2 + 2.0 * t / (3.0 * 1e3)
    x, y, _, _ = wl.cell_centres(64, 64)
    X, Y = np.meshgrid(x, y)
    exact = (w["s0"] ** 2 / s2) * np.exp(-((X - 0.5) ** 2 + (Y - 0.5) ** 2) / (2 * s2)) + w["floor"]
    assert rel_l2(Eg, exact) <= 0.03
    assert g.count_unrealizable() == (0, 0)


def test_config2_opacity_jump_implicit_steady_and_restoring():
    from oracle.steady_profile import steady_profile_1d
    w = wl.opacity_jump(256)
    prof = steady_profile_1d(w["sigma_line"], w["dx"], c=1.0, F0=w["F0"], E_out=w["E_out"], sigma_ghost=w["sigma_ghost"])
    n = w["nx"]
    w["E"] = np.tile(prof["E"], (n, 1))
    w["F"] = np.stack((np.tile(prof["Fx"], (n, 1)), np.zeros((n, n))))
    one = np.ones(n)
    w["ghosts"] = {0: (prof["ghost_lo"][0] * one, np.stack((prof["ghost_lo"][1] * one, 0 * one)), 0 * one, w["sigma_ghost"][0] * one),
                   1: (prof["ghost_hi"][0] * one, np.stack((prof["ghost_hi"][1] * one, 0 * one)), 0 * one, w["sigma_ghost"][1] * one)}
    dt = _dt(w, 100.0)
    # (a) steady: the 50 implicit steps BASELINE.json configs[1] states keep the state to round-off
    g = make_gpu(w)
    for _ in range(50):
        g.step_implicit(dt, 1e-10, 30, 4000)
    Eg, Fg = g.get_state()
    assert np.max(np.abs(Eg - w["E"])) / np.max(w["E"]) < 1e-9
    assert np.max(np.abs(Fg[0] - w["F"][0])) / w["F0"] < 1e-6
    # (b) perturbed by 1e-6: the Krylov loop really runs; parity with the oracle
    rng = np.random.default_rng(8)
    w2 = dict(w)
    w2["E"] = w["E"] * (1.0 + 1e-6 * rng.standard_normal(w["E"].shape))
    o, g = make_oracle(w2), make_gpu(w2)
    for _ in range(3):
        io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
        ig, rg = g.step_implicit(dt, 1e-10, 30, 4000)
        assert rg <= 1e-10
    assert io > 0 and ig > 0
    assert state_rel_l2(g.get_state(), o.get_state()) <= TOL_IMPLICIT


@pytest.mark.parametrize("op", OPS)
@pytest.mark.parametrize("k", [50.0, 100.0])
def test_config3_random_medium_256_window(k, op):
    # the config-3 generator on a 256^2 grid (the oracle finishes in seconds), dt = 50x and 100x
    w = wl.random_medium(256, seed=1234)
    o, g = make_oracle(w), make_gpu(w, dict(operator=op))
    dt = _dt(w, k)
    io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
    ig, rg = g.step_implicit(dt, 1e-10, 30, 4000)
    assert ro <= 1e-10 and rg <= 1e-10
    assert state_rel_l2(g.get_state(), o.get_state()) <= TOL_IMPLICIT
    assert abs(ig - io) <= max(2, 0.02 * io)
    assert o.count_unrealizable() == g.count_unrealizable()


def test_nonfinite_state_is_reported():
    w = small_random_state(12, 12, seed=46)
    w["E"][3, 3] = np.nan
    g = make_gpu(w)
    with pytest.raises(RuntimeError, match="non-finite"):
        g.step_implicit(_dt(w, 10.0), 1e-10, 30, 100)


def test_huge_maxit_and_option_switching_on_one_handle():
    # history capacity is capped (2^20 entries); operator / Krylov method / restart can change between solves of one handle
    w = small_random_state(24, 20, seed=47)
    g = make_gpu(w)
    o = make_oracle(w)
    dt = _dt(w, 30.0)
    o.step_implicit(dt, 1e-11, 30, 4000)
    want = o.get_state()
    for opts in (dict(operator=1, krylov=0), dict(operator=0, krylov=0), dict(operator=0, krylov=1), dict(operator=1, krylov=1)):
        g.set_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
        for k, v in opts.items():
            g.set_option(k, v)
        its, res = g.step_implicit(dt, 1e-11, 7 if opts["operator"] else 30, 3_000_000)
        assert res <= 1e-11 and its > 0
        assert state_rel_l2(g.get_state(), want) <= TOL_IMPLICIT
        assert len(g.history()) >= 2
