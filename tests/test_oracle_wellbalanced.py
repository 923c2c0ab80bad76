"""BASELINE configs[1]: constant-flux steady state across an opacity jump (Sect. 3.1.2, 5.2; R8)."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle
from oracle.oracle_m1 import XLO, XHI
from oracle.steady_profile import steady_profile_1d


def jump_workload(n, ny=None, options=None):
    """Config-2 input state: generator (opacity, boundary data) + the oracle's discrete steady profile."""
    cfg = wl.opacity_jump(n)
    ny = ny or n
    prof = steady_profile_1d(cfg["sigma_line"], cfg["dx"], cfg["c"], cfg["F0"], cfg["E_out"], cfg["sigma_ghost"], options)
    one = np.ones(ny)
    w = dict(nx=n, ny=ny, dx=cfg["dx"], dy=cfg["dx"], c=cfg["c"], bc=cfg["bc"],
             E=np.tile(prof["E"], (ny, 1)), F=np.stack((np.tile(prof["Fx"], (ny, 1)), np.zeros((ny, n)))),
             sigma_a=np.zeros((ny, n)), sigma_s=np.tile(cfg["sigma_line"], (ny, 1)))
    w["ghosts"] = {
        XLO: (prof["ghost_lo"][0] * one, np.stack((prof["ghost_lo"][1] * one, 0 * one)), 0 * one, cfg["sigma_ghost"][0] * one),
        XHI: (prof["ghost_hi"][0] * one, np.stack((prof["ghost_hi"][1] * one, 0 * one)), 0 * one, cfg["sigma_ghost"][1] * one),
    }
    return w, prof, cfg


@pytest.fixture(scope="module")
def jump64():
    # nx = 256 as in configs[1]: the explicit step needs c sigma dt = 1e3 * 0.4/nx < 2 (forward Euler on the source)
    return jump_workload(256, ny=4)


def test_profile_is_discrete_steady_state(jump64):
    w, prof, cfg = jump64
    assert prof["residual_inf"] < 1e-12 * prof["scale"]
    RE, RF = make_oracle(w).residual()
    assert max(np.max(np.abs(RE)), np.max(np.abs(RF))) < 1e-12 * prof["scale"]
    # WB evidence: the flux stays flat across the jump ...
    assert np.max(np.abs(prof["Fx"] - cfg["F0"])) / cfg["F0"] < 5e-3
    assert np.all(np.diff(prof["E"]) < 0)       # E decreases monotonically towards the outflow


def test_non_wb_profile_has_flux_spike():
    # ... whereas the steady state of the cell-centred source (Eq. 16) has an O(1) flux error at the jump
    cfg = wl.opacity_jump(64)
    prof = steady_profile_1d(cfg["sigma_line"], cfg["dx"], cfg["c"], cfg["F0"], cfg["E_out"], cfg["sigma_ghost"],
                             dict(well_balanced=0))
    assert prof["residual_inf"] < 1e-11 * prof["scale"]
    err = np.abs(prof["Fx"] - cfg["F0"]) / cfg["F0"]
    assert err.max() > 0.3 and np.argmax(err) in (31, 32, 33)


def test_steady_to_roundoff_explicit_and_implicit(jump64):
    # BASELINE configs[1]: 50 explicit + 50 implicit steps, "the state must stay steady to round-off"
    w, prof, cfg = jump64
    o = make_oracle(w)
    U0 = np.concatenate((w["E"][None], w["F"]))
    dt = wl.explicit_dt(w["dx"], w["dy"])
    for _ in range(50):
        o.step_explicit(dt)
    tot = 0
    for _ in range(50):
        its, res = o.step_implicit(100 * dt, tol=1e-10)
        tot += its
    E, F = o.get_state()
    U1 = np.concatenate((E[None], F))
    assert np.max(np.abs(U1 - U0)) / np.max(np.abs(U0)) < 1e-12
    assert np.max(np.abs(F[1])) < 1e-13
    assert tot == 0           # ||b - A U*|| <= tol ||b||: the Krylov loop is never entered on the exact steady state


def test_perturbed_steady_state_is_pulled_back(jump64):
    # exercises the Krylov loop on config 2: a 1e-6 relative perturbation decays under implicit steps
    w, prof, cfg = jump64
    rng = np.random.default_rng(2)
    wp = dict(w, E=w["E"] * (1 + 1e-6 * rng.standard_normal(w["E"].shape)))
    o = make_oracle(wp)
    d0 = np.max(np.abs(wp["E"] - w["E"]))
    tot = 0
    for _ in range(10):
        its, res = o.step_implicit(100 * wl.explicit_dt(w["dx"], w["dy"]), tol=1e-12)
        assert res <= 1e-12
        tot += its
    E, F = o.get_state()
    assert tot > 0
    assert np.max(np.abs(E - w["E"])) < 0.5 * d0


@pytest.mark.slow
def test_config2_full_size_profile():
    # the full 256-cell profile of configs[1] (1-D Newton polish only; the 2-D run is the GPU parity test)
    cfg = wl.opacity_jump(256)
    prof = steady_profile_1d(cfg["sigma_line"], cfg["dx"], cfg["c"], cfg["F0"], cfg["E_out"], cfg["sigma_ghost"])
    assert prof["residual_inf"] < 1e-12 * prof["scale"]
    assert np.max(np.abs(prof["Fx"] - cfg["F0"])) / cfg["F0"] < 1e-3
