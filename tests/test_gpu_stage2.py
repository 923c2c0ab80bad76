"""GPU parity, row a8 (stage 2): matter coupling (Eq. 4), point source, explicit velocity sources (Eq. 6,
PAPER.md:101, 253) against the oracle on the same seeded inputs."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, make_gpu, small_random_state, rel_l2, state_rel_l2

pytestmark = pytest.mark.gpu


def _coupled_state(nx, ny, seed, bc=(0, 0, 0, 0)):
    w = small_random_state(nx, ny, seed=seed, bc=bc, sig_range=(-1.0, 1.5))
    rng = np.random.default_rng(seed + 1000)
    w["T"] = np.exp(0.2 * rng.standard_normal((ny, nx)))
    w["rho_cv"] = 10.0 ** rng.uniform(-0.5, 1.0, (ny, nx))
    w["source_E"] = np.zeros((ny, nx))
    w["source_E"][ny // 2, nx // 2] = 50.0
    w["ux"] = 1e-2 * rng.standard_normal((ny, nx))
    w["uy"] = 1e-2 * rng.standard_normal((ny, nx))
    return w


def _dt(w, k=1.0):
    return k * wl.explicit_dt(w["dx"], w["dy"], w["c"])


@pytest.mark.parametrize("kernel", [0, 1, 3])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 2, 2, 1)])
def test_explicit_step_with_temperature(bc, kernel):
    # kernel 0: one thread per cell; kernels 1 and 3 (default): the marching kernels with the stage-2 terms (emission, source_E, Eq. 4)
    w = _coupled_state(141, 37, seed=3, bc=bc)
    o, g = make_oracle(w, dict(a_r=0.7)), make_gpu(w, dict(a_r=0.7, explicit_kernel=kernel))
    dt = 0.2 * _dt(w)
    for _ in range(3):
        o.step_explicit(dt)
        g.step_explicit(dt)
    assert state_rel_l2(g.get_state(with_T=True), o.get_state(with_T=True)) <= 1e-11


@pytest.mark.parametrize("op", [0, 1])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 1, 0, 0), (2, 2, 1, 1)])
def test_implicit_step_with_temperature(bc, op):
    w = _coupled_state(37, 29, seed=5, bc=bc)
    o, g = make_oracle(w, dict(a_r=0.7)), make_gpu(w, dict(a_r=0.7, operator=op))
    dt = _dt(w, 40.0)
    for _ in range(2):
        io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
        ig, rg = g.step_implicit(dt, 1e-10, 30, 4000)
        assert rg <= 1e-10 and abs(ig - io) <= max(2, 0.02 * io)
    assert state_rel_l2(g.get_state(with_T=True), o.get_state(with_T=True)) <= 1e-8


def test_total_energy_conserved_by_the_coupled_implicit_step():
    # Eq. 12 rows 1 + 3 summed: sum(E + rho c_v T) is conserved (periodic, no source) to solver tolerance
    w = _coupled_state(48, 40, seed=7)
    w["source_E"] = None
    g = make_gpu(w, dict(a_r=1.0))
    tot0 = np.sum(w["E"] + w["rho_cv"] * w["T"])
    for _ in range(3):
        g.step_implicit(_dt(w, 50.0), 1e-12, 30, 4000)
    E, F, T = g.get_state(with_T=True)
    assert abs(np.sum(E + w["rho_cv"] * T) - tot0) <= 1e-9 * tot0


def test_zero_dimensional_relaxation_worked_value():
    # SURVEY.md O10 worked value (0-D, c = a_r = 1, sigma_a = 50, rho c_v = 1.5, dt = 0.3, E = 0.2, T = 1.3):
    # first linearised step gives E = 0.583533885252, T = 1.044310743165 and E + rho c_v T = 2.15 exactly
    n = 4
    w = dict(nx=n, ny=n, dx=1.0, dy=1.0, c=1.0, bc=(0, 0, 0, 0), E=np.full((n, n), 0.2), F=np.zeros((2, n, n)),
             sigma_a=np.full((n, n), 50.0), sigma_s=np.zeros((n, n)), T=np.full((n, n), 1.3), rho_cv=np.full((n, n), 1.5))
    g = make_gpu(w)
    g.step_implicit(0.3, 1e-13, 30, 100)
    E, F, T = g.get_state(with_T=True)
    assert np.allclose(E, 0.583533885252, rtol=0, atol=2e-12)
    assert np.allclose(T, 1.044310743165, rtol=0, atol=2e-12)
    assert np.allclose(E + 1.5 * T, 2.15, rtol=0, atol=1e-12)


def test_velocity_sources():
    w = _coupled_state(33, 21, seed=9)
    o, g = make_oracle(w), make_gpu(w)
    o.add_velocity_sources(0.01)
    g.add_velocity_sources(0.01)
    assert state_rel_l2(g.get_state(), o.get_state()) <= 1e-13


def test_config5_stratified_coupled_window():
    # BASELINE.json configs[4] generator on a 192^2 grid: one implicit step at 100x the explicit dt, then the velocity sources
    w = wl.stratified_coupled(192, seed=4321)
    o, g = make_oracle(w), make_gpu(w)
    dt = _dt(w, 100.0)
    io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
    ig, rg = g.step_implicit(dt, 1e-10, 30, 4000)
    assert ro <= 1e-10 and rg <= 1e-10 and abs(ig - io) <= max(2, 0.02 * io)
    o.add_velocity_sources(dt)
    g.add_velocity_sources(dt)
    assert state_rel_l2(g.get_state(with_T=True), o.get_state(with_T=True)) <= 1e-8


def test_marshak_wave_on_the_gpu():
    # the CUDA path itself against the independent discretisation of Eq. 11 (1.1 % bound of the paper) and
    # against the oracle; 400 x 1 grid, Dirichlet source on the left, outflow on the right, matter coupling, BiCGStab.
    from helpers import marshak_diffusion_reference
    w = wl.marshak(400)
    nsteps, dt = 300, 10.0
    Tref = marshak_diffusion_reference(w, dt, nsteps)
    o, g = make_oracle(w, dict(krylov=1)), make_gpu(w, dict(krylov=1))
    for _ in range(nsteps):
        o.step_implicit(dt, 1e-11, 30, 20000)
        its, res = g.step_implicit(dt, 1e-11, 30, 20000)
        assert res <= 1e-10
    Eg, Fg, Tg = g.get_state(with_T=True)
    assert rel_l2(Tg[0], Tref) <= 0.011
    Eo, Fo, To = o.get_state(with_T=True)
    assert rel_l2(Tg, To) <= 1e-7 and rel_l2(Eg, Eo) <= 1e-7
    g0 = make_gpu(w, dict(krylov=1, ap_mode=0))
    for _ in range(nsteps):
        g0.step_implicit(dt, 1e-10, 30, 20000)
    assert rel_l2(g0.get_state(with_T=True)[2][0], Tref) >= 0.5
