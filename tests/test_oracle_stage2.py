"""Pins for the oracle's stage-2 pieces: the velocity sources of Eq. 6, the explicit matter terms
(emission, Eq. 4, point source) and the point source on the implicit right-hand side.

Every expected value below is written out from the paper's formulas in numpy (Eq. 3a, Eq. 4, Eq. 5d-5e, Eq. 6 and the
Eddington tensor of PAPER.md:79 in the paper's own form D = (1-chi)/2 I + (3 chi-1)/2 n(x)n); nothing calls the oracle
to produce its own expectation.
"""
import numpy as np
import pytest

from helpers import make_oracle, small_random_state


# ---------------------------------------------------------------------------------------------------------------------
# Eq. 6 and step 3 of the splitting (Eq. 5d: dE/dt = S_E, Eq. 5e: dF/dt = c S_F)
# ---------------------------------------------------------------------------------------------------------------------

def _pressure_paper_form(E, Fx, Fy, c):
    """P = D E with D = (1-chi)/2 I + (3chi-1)/2 n(x)n, chi = (3+4f^2)/(5+2 sqrt(4-3f^2)), f = |F|/(cE)."""
    Fn = np.hypot(Fx, Fy)
    f = Fn / (c * E)
    assert np.all(f < 1.0)
    chi = (3 + 4 * f ** 2) / (5 + 2 * np.sqrt(4 - 3 * f ** 2))
    with np.errstate(invalid="ignore", divide="ignore"):
        nx = np.where(Fn > 0, Fx / Fn, 0.0)
        ny = np.where(Fn > 0, Fy / Fn, 0.0)
    iso, ani = 0.5 * (1 - chi), 0.5 * (3 * chi - 1)
    return E * (iso + ani * nx * nx), E * ani * nx * ny, E * (iso + ani * ny * ny)


def _eq6(E, Fx, Fy, sig, ux, uy, aT4, c):
    Pxx, Pxy, Pyy = _pressure_paper_form(E, Fx, Fy, c)
    uPx, uPy = ux * Pxx + uy * Pxy, ux * Pxy + uy * Pyy            # u . P (P symmetric)
    uF = ux * Fx + uy * Fy
    SE = sig / c * uF + sig / c * E * (ux * ux + uy * uy) + sig / c * (ux * uPx + uy * uPy)
    SFx = sig * uPx + sig * aT4 * ux + sig / c ** 2 * ux * uF
    SFy = sig * uPy + sig * aT4 * uy + sig / c ** 2 * uy * uF
    return SE, SFx, SFy


def _velocity_workload(seed, c, with_T=True, sigma_s_zero=False):
    w = small_random_state(7, 6, seed=seed, c=c, dx=0.13, dy=0.09)
    rng = np.random.default_rng(seed + 1000)
    shp = w["E"].shape
    if sigma_s_zero:
        w["sigma_s"] = np.zeros(shp)
    if with_T:
        w["T"] = np.exp(0.3 * rng.standard_normal(shp))
        w["rho_cv"] = rng.uniform(0.5, 2.0, shp)
    w["ux"] = 0.05 * c * rng.standard_normal(shp)
    w["uy"] = 0.05 * c * rng.standard_normal(shp)
    return w


@pytest.mark.parametrize("c", [1.0, 1.7, 0.6])
def test_velocity_sources_equal_eq6_on_a_rough_state(c):
    # c != 1 exercises every power of c in Eq. 6 and the factor c of Eq. 5e; a_r != 1 the emission-like term.
    a_r, dt = 0.8, 0.037
    w = _velocity_workload(31, c)
    o = make_oracle(w, options={"a_r": a_r})
    o.add_velocity_sources(dt)
    E1, F1, T1 = o.get_state(with_T=True)
    sig = w["sigma_a"] + w["sigma_s"]                               # reading R14: Eq. 6's grey sigma is sigma_t
    SE, SFx, SFy = _eq6(w["E"], w["F"][0], w["F"][1], sig, w["ux"], w["uy"], a_r * w["T"] ** 4, c)
    for got, want in ((E1, w["E"] + dt * SE), (F1[0], w["F"][0] + dt * c * SFx), (F1[1], w["F"][1] + dt * c * SFy)):
        assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))
    assert np.array_equal(T1, w["T"])                               # step 3 does not touch the gas temperature
    # the increments are not small: a dropped term would be seen
    assert np.max(np.abs(dt * SE)) > 1e-5 * np.max(w["E"]) and np.max(np.abs(dt * c * SFx)) > 1e-5 * np.max(np.abs(w["F"]))


def test_velocity_sources_each_term_isolated():
    c, a_r, dt, sig = 1.9, 0.7, 0.01, 3.0
    n = 3
    base = dict(nx=n, ny=n, dx=1 / n, dy=1 / n, c=c, bc=(0, 0, 0, 0), sigma_a=np.full((n, n), 1.0), sigma_s=np.full((n, n), sig - 1.0))

    def run(E, Fx, Fy, ux, uy, T=None):
        w = dict(base, E=np.full((n, n), E), F=np.stack((np.full((n, n), Fx), np.full((n, n), Fy))),
                 ux=np.full((n, n), ux), uy=np.full((n, n), uy))
        if T is not None:
            w["T"] = np.full((n, n), T)
        o = make_oracle(w, options={"a_r": a_r})
        o.add_velocity_sources(dt)
        E1, F1 = o.get_state()
        return (E1[1, 1] - E) / dt, (F1[0][1, 1] - Fx) / (dt * c), (F1[1][1, 1] - Fy) / (dt * c)

    # (i) f = 0 closed form: P = E/3 I  =>  S_E = (sigma/c)(4/3) E u^2,  S_F = sigma (E/3 + a_r T^4) u
    E, ux, uy, T = 2.0, 0.3, -0.2, 1.1
    SE, SFx, SFy = run(E, 0.0, 0.0, ux, uy, T)
    u2 = ux * ux + uy * uy
    assert SE == pytest.approx(sig / c * (4.0 / 3.0) * E * u2, rel=1e-11)
    assert SFx == pytest.approx(sig * (E / 3.0 + a_r * T ** 4) * ux, rel=1e-11)
    assert SFy == pytest.approx(sig * (E / 3.0 + a_r * T ** 4) * uy, rel=1e-11)
    # (ii) T absent: the a_r T^4 u term is gone
    SE, SFx, SFy = run(E, 0.0, 0.0, ux, uy, None)
    assert SFx == pytest.approx(sig * E / 3.0 * ux, rel=1e-11) and SFy == pytest.approx(sig * E / 3.0 * uy, rel=1e-11)
    # (iii) u = 0: nothing happens
    assert run(E, 0.4, 0.1, 0.0, 0.0, T) == (0.0, 0.0, 0.0)
    # (iv) u perpendicular to F (F along x, u along y): u.F = 0; P diagonal  =>
    #      S_E = (sigma/c) u^2 (E + Pyy),  S_Fx = 0,  S_Fy = sigma (Pyy + a_r T^4) u_y
    Fx = 0.5 * c * E
    f = 0.5
    chi = (3 + 4 * f * f) / (5 + 2 * np.sqrt(4 - 3 * f * f))
    Pxx, Pyy = chi * E, 0.5 * (1 - chi) * E                         # n = e_x: D_xx = chi, D_yy = (1-chi)/2
    SE, SFx, SFy = run(E, Fx, 0.0, 0.0, uy, T)
    assert SE == pytest.approx(sig / c * uy * uy * (E + Pyy), rel=1e-11)
    assert abs(SFx) <= 1e-13 * abs(SFy)
    assert SFy == pytest.approx(sig * (Pyy + a_r * T ** 4) * uy, rel=1e-11)
    # (v) u parallel to F: S_E = (sigma/c)(u F + u^2 (E + Pxx)),  S_Fx = sigma (Pxx + a_r T^4) u + (sigma/c^2) u^2 F
    SE, SFx, SFy = run(E, Fx, 0.0, ux, 0.0, T)
    assert SE == pytest.approx(sig / c * (ux * Fx + ux * ux * (E + Pxx)), rel=1e-11)
    assert SFx == pytest.approx(sig * (Pxx + a_r * T ** 4) * ux + sig / c ** 2 * ux * ux * Fx, rel=1e-11)
    assert abs(SFy) <= 1e-13 * abs(SFx)
    # (vi) the sign of u.F: reversing u flips the first term of S_E only
    SEm, _, _ = run(E, Fx, 0.0, -ux, 0.0, T)
    assert SE - SEm == pytest.approx(2 * sig / c * ux * Fx, rel=1e-11)


def test_velocity_sources_reduce_to_the_papers_grey_sigma():
    # sigma_s = 0: the build's sigma_t is the paper's single grey sigma
    c, dt = 1.3, 0.02
    w = _velocity_workload(37, c, sigma_s_zero=True)
    o = make_oracle(w)
    o.add_velocity_sources(dt)
    E1, F1 = o.get_state()
    SE, SFx, SFy = _eq6(w["E"], w["F"][0], w["F"][1], w["sigma_a"], w["ux"], w["uy"], w["T"] ** 4, c)
    assert np.max(np.abs(E1 - (w["E"] + dt * SE))) <= 1e-13 * np.max(w["E"])
    assert np.max(np.abs(F1[0] - (w["F"][0] + dt * c * SFx))) <= 1e-13 * np.max(np.abs(w["F"]))


# ---------------------------------------------------------------------------------------------------------------------
# Explicit matter terms: emission in Eq. 3a, Eq. 4 taken explicitly, point source Q
# ---------------------------------------------------------------------------------------------------------------------

def _uniform(n, c, E0, T0, sa, ss, rcv, Q=None):
    w = dict(nx=n, ny=n, dx=1 / n, dy=1 / n, c=c, bc=(0, 0, 0, 0), E=np.full((n, n), E0), F=np.zeros((2, n, n)),
             sigma_a=np.full((n, n), sa), sigma_s=np.full((n, n), ss), T=np.full((n, n), T0), rho_cv=np.full((n, n), rcv))
    if Q is not None:
        w["source_E"] = np.full((n, n), Q)
    return w


@pytest.mark.parametrize("E0,T0", [(0.2, 1.3), (3.0, 0.7)])     # emission-dominated and absorption-dominated
def test_explicit_step_with_T_uniform_state_closed_form(E0, T0):
    # uniform state, F = 0: all fluxes cancel, so the step is Eq. 3a / Eq. 4 with forward Euler:
    #   E1 = E + c dt sigma_a (a_r T^4 - E) + dt Q,   T1 = T - c dt sigma_a (a_r T^4 - E)/(rho c_v),   F1 = 0
    c, a_r, sa, ss, rcv, dt, Q = 1.4, 0.9, 2.5, 4.0, 1.5, 0.013, 0.37
    w = _uniform(5, c, E0, T0, sa, ss, rcv, Q)
    o = make_oracle(w, options={"a_r": a_r})
    o.step_explicit(dt)
    E, F, T = o.get_state(with_T=True)
    ex = c * dt * sa * (a_r * T0 ** 4 - E0)
    assert np.allclose(E, E0 + ex + dt * Q, rtol=1e-13, atol=0)
    assert np.allclose(T, T0 - ex / rcv, rtol=1e-13, atol=0)
    assert np.max(np.abs(F)) <= 1e-14
    # the residual hook carries the same terms: R_E = -(c sigma_a (a_r T^4 - E) + Q)
    o2 = make_oracle(w, options={"a_r": a_r})
    RE, RF = o2.residual()
    assert np.allclose(RE, -(c * sa * (a_r * T0 ** 4 - E0) + Q), rtol=1e-12, atol=0)
    # sigma_s must not enter the exchange term (north_star: sigma_a only)
    w2 = _uniform(5, c, E0, T0, sa, 0.0, rcv, Q)
    o3 = make_oracle(w2, options={"a_r": a_r})
    o3.step_explicit(dt)
    E3, _, T3 = o3.get_state(with_T=True)
    assert np.array_equal(E3, E) and np.array_equal(T3, T)


def test_explicit_step_with_T_conserves_total_energy_and_counts_the_source():
    # "To ensure the conservation of the total energy when the hydrodynamics is frozen": periodic grid,
    # sum(E + rho c_v T) is unchanged by an explicit step (Q = 0) and grows by dt sum(Q) otherwise.
    c, dt = 1.2, 2e-3
    w = small_random_state(11, 9, seed=41, c=c, dx=0.1, dy=0.08, sig_range=(-1.0, 1.0))
    rng = np.random.default_rng(42)
    shp = w["E"].shape
    w["T"] = np.exp(0.4 * rng.standard_normal(shp))
    w["rho_cv"] = rng.uniform(0.5, 2.0, shp)
    tot0 = np.sum(w["E"] + w["rho_cv"] * w["T"])
    o = make_oracle(w)
    for _ in range(5):
        o.step_explicit(dt)
    E, F, T = o.get_state(with_T=True)
    assert abs(np.sum(E + w["rho_cv"] * T) - tot0) <= 1e-13 * tot0
    assert np.max(np.abs(T - w["T"])) > 1e-4                        # the exchange is not negligible
    w["source_E"] = rng.uniform(0.0, 5.0, shp)
    o = make_oracle(w)
    o.step_explicit(dt)
    E, F, T = o.get_state(with_T=True)
    assert np.sum(E + w["rho_cv"] * T) - tot0 == pytest.approx(dt * np.sum(w["source_E"]), rel=1e-10)
    # without rho_cv the heat capacity defaults to 1 (binding documentation)
    del w["source_E"]
    w1 = dict(w); w1["rho_cv"] = None
    o = make_oracle(w1)
    o.step_explicit(dt)
    E, F, T = o.get_state(with_T=True)
    assert abs(np.sum(E + T) - np.sum(w["E"] + w["T"])) <= 1e-13 * tot0


def test_explicit_T_update_uses_time_n_values_cell_by_cell():
    # Eq. 4 forward Euler, rough state: T1 - T0 = -c dt sigma_a (a_r T0^4 - E0)/(rho c_v) with E at time n (not E1)
    c, a_r, dt = 0.8, 1.3, 1e-3
    w = small_random_state(8, 6, seed=43, c=c, sig_range=(-1.0, 1.0))
    rng = np.random.default_rng(44)
    w["T"] = np.exp(0.4 * rng.standard_normal(w["E"].shape))
    w["rho_cv"] = rng.uniform(0.5, 2.0, w["E"].shape)
    o = make_oracle(w, options={"a_r": a_r})
    o.step_explicit(dt)
    _, _, T = o.get_state(with_T=True)
    want = w["T"] - c * dt * w["sigma_a"] * (a_r * w["T"] ** 4 - w["E"]) / w["rho_cv"]
    assert np.max(np.abs(T - want)) <= 1e-14 * np.max(want)


# ---------------------------------------------------------------------------------------------------------------------
# Implicit side: point source on the right-hand side; affine terms of the T-coupled operator
# ---------------------------------------------------------------------------------------------------------------------

def test_implicit_0d_step_with_point_source_closed_form():
    # uniform state: (1 + c dt sigma_a eta) E1 = E0 + c dt sigma_a eta a_r T0^4 + dt Q   (reading R10 + Eq. 3a with a source)
    # and Eq. 12 rows 1+3 summed: E1 + rho c_v T1 = E0 + rho c_v T0 + dt Q
    c, a_r, sa, rcv, dt, E0, T0, Q = 1.3, 0.9, 50.0, 1.5, 0.3, 0.2, 1.3, 0.45
    w = _uniform(4, c, E0, T0, sa, 7.0, rcv, Q)
    o = make_oracle(w, options={"a_r": a_r})
    o.step_implicit(dt, tol=1e-14)
    E, F, T = o.get_state(with_T=True)
    Th = a_r * T0 ** 4
    den = rcv + 4 * a_r * c * sa * dt * T0 ** 3
    eta = rcv / den
    E1 = (E0 + c * dt * sa * eta * Th + dt * Q) / (1 + c * dt * sa * eta)
    T1 = T0 + c * sa * dt * (E1 - Th) / den
    assert E[0, 0] == pytest.approx(E1, rel=1e-12) and T[0, 0] == pytest.approx(T1, rel=1e-12)
    assert E[0, 0] + rcv * T[0, 0] == pytest.approx(E0 + rcv * T0 + dt * Q, rel=1e-13)
    # without T: E1 = (E0 + dt Q)/(1 + c dt sigma_a)  (pure absorption)
    w2 = dict(w); w2["T"] = None; w2["rho_cv"] = None
    o = make_oracle(w2)
    o.step_implicit(dt, tol=1e-14)
    E, F = o.get_state()
    assert E[0, 0] == pytest.approx((E0 + dt * Q) / (1 + c * dt * sa), rel=1e-12)


@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 2, 2, 1)])
def test_operator_consistency_with_matter_terms(bc):
    # With T present the linearised system (I + dt L_n) U = b relates to the non-linear residual R (separately pinned) by
    #   A U^n + A_ghost - b = dt R(U^n) - c dt sigma_a (1 - eta)(E - a_r T^4) e_E,
    # eta = rho c_v/(rho c_v + 4 a_r c sigma_a dt T^3): the only difference is the linearised T^4 (reading R10).
    c, a_r, dt = 1.3, 0.85, 0.4
    w = small_random_state(9, 7, seed=51, c=c, dx=0.11, dy=0.07, bc=bc, sig_range=(-1.0, 1.0))
    rng = np.random.default_rng(52)
    shp = w["E"].shape
    w["T"] = np.exp(0.4 * rng.standard_normal(shp))
    w["rho_cv"] = rng.uniform(0.5, 2.0, shp)
    w["source_E"] = rng.uniform(0.0, 2.0, shp)
    o = make_oracle(w, options={"a_r": a_r})
    RE, RF = o.residual()
    U = np.concatenate((w["E"][None], w["F"]))
    AU = o.apply_linear(dt, U, mode=0) + o.apply_linear(dt, U, mode=1)
    M, b = o.dense_matrix(dt)
    b = b.reshape(U.shape)
    Th = a_r * w["T"] ** 4
    eta = w["rho_cv"] / (w["rho_cv"] + 4 * a_r * c * w["sigma_a"] * dt * w["T"] ** 3)
    expect = dt * np.concatenate((RE[None], RF))
    expect[0] -= c * dt * w["sigma_a"] * (1 - eta) * (w["E"] - Th)
    # b holds U^n + emission + source - (Dirichlet ghost terms); apply_linear(mode 1) = + ghost terms
    lhs_flux = AU - (U + np.concatenate(((c * dt * w["sigma_a"] * eta * Th + dt * w["source_E"])[None], np.zeros_like(w["F"]))))
    assert np.max(np.abs(lhs_flux - expect)) < 1e-12 * np.max(np.abs(expect))
    lhs_mat = (M @ U.ravel()).reshape(U.shape) - b
    assert np.max(np.abs(lhs_mat - expect)) < 1e-12 * np.max(np.abs(expect))


def test_implicit_small_dt_matches_explicit_with_matter_terms():
    # both steps are consistent with Eqs. 3-4 and a source: they agree to O(dt^2), T included
    c = 1.1
    w = small_random_state(8, 6, seed=61, c=c, sig_range=(-1.0, 1.0))
    rng = np.random.default_rng(62)
    w["T"] = np.exp(0.3 * rng.standard_normal(w["E"].shape))
    w["rho_cv"] = rng.uniform(0.5, 2.0, w["E"].shape)
    w["source_E"] = rng.uniform(0.0, 2.0, w["E"].shape)
    diffs = []
    for dt in (2e-4, 1e-4):
        oe, oi = make_oracle(w), make_oracle(w)
        oe.step_explicit(dt)
        oi.step_implicit(dt, tol=1e-14)
        d = [np.max(np.abs(a - b)) for a, b in zip(oe.get_state(with_T=True), oi.get_state(with_T=True))]
        diffs.append(d)
    ratio = np.array(diffs[0]) / np.array(diffs[1])
    assert np.all(ratio > 3.3) and np.all(ratio < 4.7), ratio      # second order in dt
