"""Pins for the 3-D oracle (oracle/oracle_m1_3d.c; "its extension to higher dimensions is straightforward").

The 2-D oracle is pinned against the paper (tests/test_oracle_*.py); the 3-D one is pinned against the 2-D one and against what
the mathematics fixes: a state that does not depend on one coordinate must evolve like the 2-D scheme in the other two (for
every choice of that coordinate, which also pins each direction's code against the others), a slab free-streams at c along z,
sums are conserved, the pressure Jacobian matches finite differences and Euler's identity, the implicit step matches a dense solve."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, small_random_state, rel_l2
from oracle.oracle_m1_3d import OracleM1_3D, closure_point
from oracle import oracle_m1_3d


@pytest.fixture(scope="module", autouse=True)
def _build():
    oracle_m1_3d.build()


def _embed(w2, axis, n3):
    """A 2-D workload as a 3-D one that does not depend on coordinate `axis` (0: x, 1: y, 2: z).  Returns constructor args, state
    and the permutation that maps the 2-D (Fx, Fy) onto the 3-D flux components."""
    ny, nx = w2["E"].shape
    def lift(a):                     # [ny, nx] -> [nz, ny, nx] with the two live coordinates placed in order
        if axis == 2: return np.broadcast_to(a[None, :, :], (n3, ny, nx)).copy()           # live (x, y) = 2-D (x, y)
        if axis == 1: return np.broadcast_to(a[:, None, :], (ny, n3, nx)).copy()           # live (x, z) = 2-D (x, y)
        return np.broadcast_to(a[:, :, None], (ny, nx, n3)).copy()                         # live (y, z) = 2-D (x, y)
    live = {2: (0, 1), 1: (0, 2), 0: (1, 2)}[axis]
    E = lift(w2["E"])
    F = np.zeros((3,) + E.shape)
    F[live[0]] = lift(w2["F"][0]); F[live[1]] = lift(w2["F"][1])
    d = [0.0, 0.0, 0.0]; d[live[0]] = w2["dx"]; d[live[1]] = w2["dy"]; d[axis] = 0.37
    n = [0, 0, 0]; n[live[0]] = nx; n[live[1]] = ny; n[axis] = n3
    bc = [0] * 6
    bc[2 * live[0]], bc[2 * live[0] + 1] = w2["bc"][0], w2["bc"][1]
    bc[2 * live[1]], bc[2 * live[1] + 1] = w2["bc"][2], w2["bc"][3]
    return n, d, bc, E, F, lift(w2["sigma_a"]), lift(w2["sigma_s"]), live, lift


@pytest.mark.parametrize("axis", [2, 1, 0])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (2, 2, 0, 0), (0, 0, 2, 2)])
def test_a_state_independent_of_one_coordinate_evolves_like_the_2d_oracle(axis, bc):
    w2 = small_random_state(7, 6, seed=401, dx=0.11, dy=0.07, c=1.3, bc=bc, sig_range=(-1.0, 1.0))
    n, d, bc3, E, F, sa, ss, live, lift = _embed(w2, axis, 3)
    o2 = make_oracle(w2)
    o3 = OracleM1_3D(n[0], n[1], n[2], d[0], d[1], d[2], w2["c"], bc3)
    o3.set_state(E, F, sa, ss)
    dt = wl.explicit_dt(w2["dx"], w2["dy"], w2["c"])
    for _ in range(3):
        o2.step_explicit(dt); o3.step_explicit(dt)
    E2, F2 = o2.get_state()
    E3, F3 = o3.get_state()
    assert np.max(np.abs(E3 - lift(E2))) <= 1e-14 * np.max(np.abs(E2))
    assert np.max(np.abs(F3[live[0]] - lift(F2[0]))) <= 1e-14 * np.max(np.abs(F2))
    assert np.max(np.abs(F3[live[1]] - lift(F2[1]))) <= 1e-14 * np.max(np.abs(F2))
    assert np.max(np.abs(F3[axis])) == 0.0
    # and one implicit step (both sides: GMRES(30) + diagonal blocks, tolerance 1e-12)
    i2, r2 = o2.step_implicit(20 * dt, 1e-12, 30, 2000)
    i3, r3 = o3.step_implicit(20 * dt, 1e-12, 30, 2000)
    E2, F2 = o2.get_state()
    E3, F3 = o3.get_state()
    assert r2 <= 1e-12 and r3 <= 1e-12 and abs(i2 - i3) <= 1
    assert rel_l2(E3, lift(E2)) <= 1e-10 and rel_l2(F3[live[0]], lift(F2[0])) <= 1e-10 and rel_l2(F3[live[1]], lift(F2[1])) <= 1e-10
    assert np.max(np.abs(F3[axis])) <= 1e-13 * np.max(np.abs(F2))


def _rough3(nx, ny, nz, seed, c=1.0, fmax=0.9):
    w = wl.random_medium_3d(nx, ny, nz, seed=seed, c=c, fmax=fmax, log_sigma=(-1.0, 1.0), smooth=False)
    return w["E"], w["F"], w["sigma_a"], w["sigma_s"]


def test_relabelling_the_axes_relabels_the_result():
    # (x, y, z) -> (z, x, y): arrays transposed, flux components permuted, spacings permuted; a genuinely 3-D rough state
    c = 1.2
    E, F, sa, ss = _rough3(5, 4, 6, seed=402, c=c)
    d = (0.1, 0.13, 0.07)
    a = OracleM1_3D(5, 4, 6, *d, c, (0, 0, 2, 2, 0, 0))
    a.set_state(E, F, sa, ss)
    perm = lambda A: np.ascontiguousarray(np.transpose(A, (1, 2, 0)))        # new [nz'=ny, ny'=nx, nx'=nz]
    Fp = np.stack((perm(F[2]), perm(F[0]), perm(F[1])))                        # new x = old z, new y = old x, new z = old y
    b = OracleM1_3D(6, 5, 4, d[2], d[0], d[1], c, (0, 0, 0, 0, 2, 2))
    b.set_state(perm(E), Fp, perm(sa), perm(ss))
    dt = 0.4 * min(d) / c
    a.step_explicit(dt); b.step_explicit(dt)
    ia, _ = a.step_implicit(10 * dt, 1e-12, 30, 3000); ib, _ = b.step_implicit(10 * dt, 1e-12, 30, 3000)
    Ea, Fa = a.get_state(); Eb, Fb = b.get_state()
    assert abs(ia - ib) <= 1
    assert rel_l2(Eb, perm(Ea)) <= 1e-10
    assert rel_l2(Fb[0], perm(Fa[2])) <= 1e-10 and rel_l2(Fb[1], perm(Fa[0])) <= 1e-10 and rel_l2(Fb[2], perm(Fa[1])) <= 1e-10


def test_closure_3d_limits_trace_and_rotation():
    q = closure_point(1.0, 2.0, [0.0, 0.0, 0.0])
    assert np.allclose(q["P"], np.eye(3) * 2.0 / 3.0, atol=1e-15)                       # f = 0: P = E/3 I
    assert np.allclose(q["lmax"], 1 / np.sqrt(3)) and np.allclose(q["lmin"], -1 / np.sqrt(3))
    nvec = np.array([2.0, -1.0, 2.0]) / 3.0
    q = closure_point(1.7, 3.0, 1.7 * 3.0 * nvec)                                       # f = 1: P = E n(x)n
    assert np.allclose(q["P"], 3.0 * np.outer(nvec, nvec), atol=1e-14)
    rng = np.random.default_rng(5)
    for _ in range(20):
        E = np.exp(rng.standard_normal()); c = rng.uniform(0.5, 2.0)
        F = rng.standard_normal(3); F *= rng.uniform(0, 0.99) * c * E / np.linalg.norm(F)
        q = closure_point(c, E, F)
        assert np.trace(q["P"]) == pytest.approx(E, rel=1e-13)                          # tr D = 1
        assert np.allclose(q["P"], q["P"].T)
        # the 2-D oracle's closure is the z-invariant special case
        Rm, _ = np.linalg.qr(rng.standard_normal((3, 3)))                               # covariance under rotations
        q2 = closure_point(c, E, Rm @ F)
        assert np.allclose(q2["P"], Rm @ q["P"] @ Rm.T, atol=1e-13 * E)
        # Eq. 14 depends on the normal component and the tangential magnitude only
        q3 = closure_point(c, E, [F[0], np.hypot(F[1], F[2]), 0.0])
        assert q3["lmax"][0] == pytest.approx(q["lmax"][0], rel=1e-12) and q3["lmin"][0] == pytest.approx(q["lmin"][0], rel=1e-12, abs=1e-14)


def test_pressure_jacobian_3d_fd_and_euler():
    rng = np.random.default_rng(6)
    for fscale in (0.3, 0.8, 1.4):            # 1.4: the clamped closure
        c = 1.3; E = 1.7
        F = rng.standard_normal(3); F *= fscale * c * E / np.linalg.norm(F)
        q = closure_point(c, E, F)
        U = np.concatenate(([E], F))
        assert np.allclose(np.einsum("abe,e->ab", q["J"], U), q["P"], atol=1e-13)       # Euler: P homogeneous of degree 1
        for e in range(4):
            h = 1e-6 * max(abs(U[e]), 1.0)
            Up, Um = U.copy(), U.copy(); Up[e] += h; Um[e] -= h
            fd = (closure_point(c, Up[0], Up[1:])["P"] - closure_point(c, Um[0], Um[1:])["P"]) / (2 * h)
            assert np.allclose(q["J"][:, :, e], fd, atol=2e-8)


def test_free_streaming_slab_moves_at_c_along_z_and_sums_are_conserved():
    nx, ny, nz = 2, 2, 64
    dz = 1.0 / nz
    z = (np.arange(nz) + 0.5) * dz
    prof = np.where(np.abs(z - 0.3) < 0.1, 1.0, 0.0) + 1e-8
    E = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
    F = np.zeros((3, nz, ny, nx)); F[2] = E                                               # f = 1 along +z, c = 1
    o = OracleM1_3D(nx, ny, nz, 0.5, 0.5, dz, 1.0)
    o.set_state(E, F, np.zeros_like(E), np.zeros_like(E))
    dt = 0.4 * dz
    nst = 40
    for _ in range(nst):
        o.step_explicit(dt)
    E1, F1 = o.get_state()
    cen = lambda p: np.angle(np.sum((p - 1e-8) * np.exp(2j * np.pi * z))) / (2 * np.pi)
    assert (cen(E1[:, 0, 0]) - cen(prof)) % 1.0 == pytest.approx(nst * dt, abs=2e-3)       # centroid moves by c t
    assert np.sum(E1) == pytest.approx(np.sum(E), rel=1e-13) and np.sum(F1[2]) == pytest.approx(np.sum(F[2]), rel=1e-13)
    assert np.max(np.abs(F1[:2])) <= 1e-14
    assert np.max(np.linalg.norm(F1, axis=0) / E1) <= 1 + 1e-12                          # realizability


def test_operator_consistency_and_dense_solve_3d():
    c = 1.1
    E, F, sa, ss = _rough3(3, 4, 3, seed=403, c=c)
    o = OracleM1_3D(3, 4, 3, 0.2, 0.17, 0.23, c, (0, 0, 2, 2, 0, 0))
    o.set_state(E, F, sa, ss)
    U = np.concatenate((E[None], F))
    dt = 0.5
    R = o.residual()
    assert np.max(np.abs(o.apply_linear(dt, U) - (U + dt * R))) <= 1e-12 * np.max(np.abs(U + dt * R))   # homogeneity: A U^n = U^n + dt R(U^n)
    n = U.size
    A = np.zeros((n, n))
    for k in range(n):
        e = np.zeros(n); e[k] = 1.0
        A[:, k] = o.apply_linear(dt, e.reshape(U.shape)).ravel()
    B = o.diag_blocks(dt)
    N = E.size
    for cell in (0, 7, N - 1):
        idx = [e * N + cell for e in range(4)]
        assert np.allclose(B[cell], A[np.ix_(idx, idx)], atol=1e-13)
    x = np.linalg.solve(A, U.ravel()).reshape(U.shape)
    its, res = o.step_implicit(dt, 1e-12, 30, 2000)
    E1, F1 = o.get_state()
    assert res <= 1e-12 and its > 0
    assert rel_l2(np.concatenate((E1[None], F1)), x) <= 1e-10
    # periodic in x and z, sigma_a > 0: energy decays; with sigma_a = 0 and all-periodic it is conserved
    o2 = OracleM1_3D(3, 4, 3, 0.2, 0.17, 0.23, c)
    o2.set_state(E, F, np.zeros_like(E), ss)
    o2.step_implicit(dt, 1e-13, 30, 2000)
    assert np.sum(o2.get_state()[0]) == pytest.approx(np.sum(E), rel=1e-11)
