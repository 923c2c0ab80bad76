"""Pins for the oracle's per-cell physics (closure, Eq. 14 eigenvalues, pressure Jacobian).

Each test ties oracle/oracle_m1.c to something other than itself: values the paper states, closed forms,
eigenvalues of a numerically differentiated flux Jacobian, finite differences, rotation covariance.
"""
import math
import os

import numpy as np
import pytest

from oracle.oracle_m1 import OracleM1

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_fixed_values.txt")


def golden():
    vals = {}
    with open(GOLDEN) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()
                vals[k] = float(v)
    return vals


@pytest.fixture(scope="module")
def o():
    return OracleM1(4, 4, 0.25, 0.25, 1.0)


def test_chi_limits_paper(o):
    g = golden()
    assert o.closure_point(2.0, 0.0, 0.0)["chi"] == pytest.approx(g["chi_at_f0"], abs=1e-15)
    assert o.closure_point(2.0, 2.0, 0.0)["chi"] == pytest.approx(g["chi_at_f1"], abs=1e-15)


def test_pressure_limits(o):
    # f = 0: isotropic P = E/3 I; f = 1: P = E n(x)n
    q = o.closure_point(3.0, 0.0, 0.0)
    assert (q["Pxx"], q["Pxy"], q["Pyy"]) == pytest.approx((1.0, 0.0, 1.0), abs=1e-15)
    th = 0.7
    q = o.closure_point(3.0, 3.0 * math.cos(th), 3.0 * math.sin(th))
    assert q["Pxx"] == pytest.approx(3.0 * math.cos(th) ** 2, abs=1e-14)
    assert q["Pxy"] == pytest.approx(3.0 * math.cos(th) * math.sin(th), abs=1e-14)
    assert q["Pyy"] == pytest.approx(3.0 * math.sin(th) ** 2, abs=1e-14)


def test_chi_closed_form_and_trace(o):
    # (3+4f^2)/(5+2 xi) == (5 - 2 xi)/3 because (5-2xi)(5+2xi) = 9 + 12 f^2; in-plane trace Dxx+Dyy = (1+chi)/2
    for f in np.linspace(0.0, 1.0, 41):
        q = o.closure_point(1.7, 1.7 * f * math.cos(0.3), 1.7 * f * math.sin(0.3))
        xi = math.sqrt(4.0 - 3.0 * f * f)
        assert q["chi"] == pytest.approx((5.0 - 2.0 * xi) / 3.0, abs=2e-15)
        assert (q["Pxx"] + q["Pyy"]) / 1.7 == pytest.approx(0.5 * (1.0 + q["chi"]), abs=1e-14)
        # monotone Eddington factor between 1/3 and 1
        assert 1.0 / 3.0 - 1e-15 <= q["chi"] <= 1.0 + 1e-15


def test_c_scaling(o):
    # f = |F|/(cE): doubling c and F leaves D unchanged
    o2 = OracleM1(4, 4, 0.25, 0.25, 2.0)
    a = o.closure_point(1.3, 0.4, -0.2)
    b = o2.closure_point(1.3, 0.8, -0.4)
    for k in ("chi", "Pxx", "Pxy", "Pyy", "f"):
        assert a[k] == pytest.approx(b[k], rel=1e-15)
    assert b["lmax_x"] == pytest.approx(2.0 * a["lmax_x"], rel=1e-15)


def test_rotation_covariance(o):
    E, f = 2.0, 0.6
    for th in (0.2, 1.1, 2.9, 4.4):
        q = o.closure_point(E, E * f * math.cos(th), E * f * math.sin(th))
        q0 = o.closure_point(E, E * f, 0.0)
        R = np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])
        P0 = np.array([[q0["Pxx"], q0["Pxy"]], [q0["Pxy"], q0["Pyy"]]])
        P = R @ P0 @ R.T
        assert [q["Pxx"], q["Pxy"], q["Pyy"]] == pytest.approx([P[0, 0], P[0, 1], P[1, 1]], abs=1e-14)


def test_clamp_f_above_one(o):
    # f = 1 imposed in the Eddington tensor where f > 1 (state itself untouched)
    th = 2.2
    a = o.closure_point(1.0, 1.7 * math.cos(th), 1.7 * math.sin(th))
    b = o.closure_point(1.0, 1.0 * math.cos(th), 1.0 * math.sin(th))
    assert a["f"] == 1.0
    for k in ("Pxx", "Pxy", "Pyy", "lmin_x", "lmax_x", "lmin_y", "lmax_y"):
        assert a[k] == pytest.approx(b[k], abs=1e-14)
    # E <= 0 is only guarded in the division
    q = o.closure_point(0.0, 0.0, 0.0)
    assert q["f"] == 0.0 and q["Pxx"] == 0.0


def test_eigenvalue_closed_forms(o):
    g = golden()
    q = o.closure_point(1.0, 0.0, 0.0)
    for k in ("lmax_x", "lmax_y"):
        assert q[k] == pytest.approx(g["lambda_p1_over_c"], abs=1e-15)
    for k in ("lmin_x", "lmin_y"):
        assert q[k] == pytest.approx(-g["lambda_p1_over_c"], abs=1e-15)
    q = o.closure_point(1.0, 1.0, 0.0)      # free streaming along the face normal: both speeds = +c
    assert (q["lmin_x"], q["lmax_x"]) == pytest.approx((1.0, 1.0), abs=1e-15)
    assert (q["lmin_y"], q["lmax_y"]) == pytest.approx((0.0, 0.0), abs=1e-15)   # tangential: 0


def _flux_jacobian_eigs(o, E, Fx, Fy, direction, c=1.0):
    """Eigenvalues of d(flux)/dU for U=(E,Fx,Fy), flux = (Fx, c^2 Pxx, c^2 Pxy) (x) or (Fy, c^2 Pxy, c^2 Pyy) (y),
    by central differences on the oracle's pressure."""
    U0 = np.array([E, Fx, Fy])

    def flux(U):
        q = o.closure_point(*U)
        if direction == 0:
            return np.array([U[1], c * c * q["Pxx"], c * c * q["Pxy"]])
        return np.array([U[2], c * c * q["Pxy"], c * c * q["Pyy"]])

    Jm = np.empty((3, 3))
    for k in range(3):
        h = 1e-6
        Up, Um = U0.copy(), U0.copy()
        Up[k] += h
        Um[k] -= h
        Jm[:, k] = (flux(Up) - flux(Um)) / (2 * h)
    ev = np.linalg.eigvals(Jm)
    assert np.max(np.abs(ev.imag)) < 1e-6        # hyperbolic
    return np.sort(ev.real)


@pytest.mark.parametrize("f,deg", [(0.5, 0), (0.5, 90), (0.5, 45), (0.9, 45), (0.9, 90), (0.3, 120), (0.05, 200), (0.97, 10)])
def test_eq14_matches_flux_jacobian_spectrum(o, f, deg):
    # lambda_max/min "are the eigenvalues of Eq. 3"
    th = math.radians(deg)
    E = 1.3
    Fx, Fy = E * f * math.cos(th), E * f * math.sin(th)
    q = o.closure_point(E, Fx, Fy)
    ex = _flux_jacobian_eigs(o, E, Fx, Fy, 0)
    ey = _flux_jacobian_eigs(o, E, Fx, Fy, 1)
    assert (q["lmin_x"], q["lmax_x"]) == pytest.approx((ex[0], ex[2]), abs=2e-8)
    assert (q["lmin_y"], q["lmax_y"]) == pytest.approx((ey[0], ey[2]), abs=2e-8)
    assert abs(q["lmax_x"]) <= 1.0 + 1e-14 and abs(q["lmin_x"]) <= 1.0 + 1e-14   # never faster than c


def test_eq14_literature_form(o):
    # Equivalent form (Gonzalez et al. 2007 style): [mu f +- sqrt(2/3 (xi^2 - xi) + 2 mu^2 (2 - f^2 - xi))]/xi
    rng = np.random.default_rng(7)
    for _ in range(50):
        f, th = rng.uniform(0, 1), rng.uniform(0, 2 * math.pi)
        q = o.closure_point(1.0, f * math.cos(th), f * math.sin(th))
        xi, mu = math.sqrt(4 - 3 * f * f), math.cos(th)
        root = math.sqrt(max(0.0, 2.0 / 3.0 * (xi * xi - xi) + 2 * mu * mu * (2 - f * f - xi)))
        assert q["lmax_x"] == pytest.approx((mu * f + root) / xi, abs=1e-13)
        assert q["lmin_x"] == pytest.approx((mu * f - root) / xi, abs=1e-13)


@pytest.mark.parametrize("c", [1.0, 1.3])
def test_pressure_jacobian_fd_and_euler(c):
    o = OracleM1(4, 4, 0.25, 0.25, c)
    rng = np.random.default_rng(11)
    for _ in range(40):
        E = math.exp(rng.standard_normal())
        f, th = rng.uniform(0.0, 0.98), rng.uniform(0, 2 * math.pi)
        U = np.array([E, c * E * f * math.cos(th), c * E * f * math.sin(th)])
        J = o.closure_point(*U)["J"]
        Jfd = np.empty((3, 3))
        for k in range(3):
            h = 1e-6 * max(abs(U[k]), 0.1)
            Up, Um = U.copy(), U.copy()
            Up[k] += h
            Um[k] -= h
            qp, qm = o.closure_point(*Up), o.closure_point(*Um)
            Jfd[:, k] = (np.array([qp["Pxx"], qp["Pxy"], qp["Pyy"]]) - np.array([qm["Pxx"], qm["Pxy"], qm["Pyy"]])) / (2 * h)
        assert np.max(np.abs(J - Jfd)) < 2e-8
        q = o.closure_point(*U)
        # Euler's identity: P is homogeneous of degree 1 in (E, F)  =>  J U = P
        assert J @ U == pytest.approx([q["Pxx"], q["Pxy"], q["Pyy"]], abs=1e-14 * max(1.0, E))


def test_pressure_jacobian_special_points(o):
    # f = 0: dP/dE = I/3, dP/dF = 0
    J = o.closure_point(2.0, 0.0, 0.0)["J"]
    assert J[:, 0] == pytest.approx([1 / 3, 0, 1 / 3], abs=1e-15)
    assert np.max(np.abs(J[:, 1:])) == 0.0
    # tiny f: no blow-up from the n-dependent terms (J -> isotropic + O(f))
    J = o.closure_point(1.0, 1e-9, -2e-9)["J"]
    assert J[:, 0] == pytest.approx([1 / 3, 0, 1 / 3], abs=1e-12)
    assert np.max(np.abs(J[:, 1:])) < 1e-8
    # clamped branch (|F| > cE): Jacobian of P = E n(x)n, checked by finite differences and Euler's identity
    U = np.array([1.0, 1.2, 0.9])
    J = o.closure_point(*U)["J"]
    q = o.closure_point(*U)
    assert J @ U == pytest.approx([q["Pxx"], q["Pxy"], q["Pyy"]], abs=1e-14)
    for k in range(3):
        h = 1e-6
        Up, Um = U.copy(), U.copy()
        Up[k] += h
        Um[k] -= h
        qp, qm = o.closure_point(*Up), o.closure_point(*Um)
        fd = (np.array([qp["Pxx"], qp["Pxy"], qp["Pyy"]]) - np.array([qm["Pxx"], qm["Pxy"], qm["Pyy"]])) / (2 * h)
        assert J[:, k] == pytest.approx(fd, abs=1e-8)


def test_p1_closure_switch():
    o = OracleM1(4, 4, 0.25, 0.25, 1.0)
    o.set_option("closure", 1)
    q = o.closure_point(3.0, 1.0, 0.5)
    assert (q["Pxx"], q["Pxy"], q["Pyy"]) == pytest.approx((1.0, 0.0, 1.0), abs=1e-15)
    assert q["lmax_x"] == pytest.approx(1 / math.sqrt(3), abs=1e-15)
