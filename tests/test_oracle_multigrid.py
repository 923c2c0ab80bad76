"""Pins for the oracle's multigrid preconditioner (R15) -- CPU only.

The hierarchy and the V-cycle are checked against dense / scipy linear algebra built from the assembled fine blocks only
(`OracleM1.assemble`), never from the multigrid code itself."""
import numpy as np
import pytest
import scipy.sparse as sp

import m1_workloads as W
from helpers import make_oracle


def fine_matrix(o, dt):
    """Cell-interleaved sparse matrix (unknown 3*cell + component) from the assembled 5-point blocks."""
    A5, col, b = o.assemble(dt)
    N = A5.shape[0]
    rows, cols, vals = [], [], []
    for cell in range(N):
        for k in range(5):
            cj = col[cell, k]
            if cj < 0:
                continue
            for r in range(3):
                for s in range(3):
                    rows.append(3 * cell + r); cols.append(3 * cj + s); vals.append(A5[cell, k, r, s])
    return sp.coo_matrix((vals, (rows, cols)), shape=(3 * N, 3 * N)).tocsr().toarray(), b


def injection(nx, ny):
    """P0: piecewise-constant injection from 2x2 aggregates (1 wide at an odd end), per component."""
    cx, cy = (nx + 1) // 2, (ny + 1) // 2
    P = np.zeros((3 * nx * ny, 3 * cx * cy))
    for j in range(ny):
        for i in range(nx):
            a = (j // 2) * cx + i // 2
            for q in range(3):
                P[3 * (j * nx + i) + q, 3 * a + q] = 1.0
    return P, cx, cy


def block_diag_inverse(A):
    n = A.shape[0] // 3
    Di = np.zeros_like(A)
    for k in range(n):
        Di[3 * k:3 * k + 3, 3 * k:3 * k + 3] = np.linalg.inv(A[3 * k:3 * k + 3, 3 * k:3 * k + 3])
    return Di


def dense_vcycle(A, nx, ny, omega, coarse_sweeps):
    """M^-1 as a dense matrix, from the five steps of PAPER.md:283-287 written with matrices."""
    n = A.shape[0]
    S = omega * block_diag_inverse(A)
    I = np.eye(n)
    if nx == 1 and ny == 1:
        Z = S.copy()
        for _ in range(coarse_sweeps - 1):
            Z = Z + S @ (I - A @ Z)
        return Z
    P0, cx, cy = injection(nx, ny)
    P = block_diag_inverse(A) @ P0
    Ac = P0.T @ A @ P
    Z = S + P @ dense_vcycle(Ac, cx, cy, omega, coarse_sweeps) @ P0.T @ (I - A @ S)
    return Z + S @ (I - A @ Z)


def interleave(V):
    return np.ascontiguousarray(V.reshape(3, -1).T).reshape(-1)


def small_problem(nx, ny, bc=(0, 0, 0, 0), seed=5):
    rng = np.random.default_rng(seed)
    E = np.exp(rng.normal(size=(ny, nx)))
    u = rng.uniform(0, 0.9, (ny, nx)); th = rng.uniform(0, 2 * np.pi, (ny, nx))
    F = np.stack([u * E * np.cos(th), u * E * np.sin(th)])
    w = dict(nx=nx, ny=ny, dx=1.0 / nx, dy=1.3 / ny, c=1.0, bc=bc, E=E, F=F,
             sigma_a=rng.uniform(0, 1, (ny, nx)), sigma_s=10.0 ** rng.uniform(-1, 2, (ny, nx)))
    if any(bc):
        w['ghosts'] = {}
        for side in range(4):
            if bc[side] == 1:
                m = ny if side < 2 else nx
                w['ghosts'][side] = (np.full(m, 1.0), np.zeros((2, m)), np.zeros(m), np.ones(m))
    return w


@pytest.mark.parametrize("nx,ny,bc", [(8, 6, (0, 0, 0, 0)), (7, 5, (0, 0, 0, 0)), (6, 5, (1, 2, 0, 0)), (5, 4, (2, 1, 1, 2))])
def test_coarse_operator_is_the_galerkin_product(nx, ny, bc):
    w = small_problem(nx, ny, bc)
    o = make_oracle(w)
    dt = 40 * 0.4 * w['dx']
    A, _ = fine_matrix(o, dt)
    nlev, n1x, n1y, A1, col1 = o.mg_level(dt, 1)
    P0, cx, cy = injection(nx, ny)
    assert (n1x, n1y) == (cx, cy)
    ref = P0.T @ A @ block_diag_inverse(A) @ P0        # R A P with P = D^-1 P0
    got = np.zeros_like(ref)
    for cell in range(cx * cy):
        for k in range(5):
            if col1[cell, k] >= 0:
                got[3 * cell:3 * cell + 3, 3 * col1[cell, k]:3 * col1[cell, k] + 3] += A1[cell, k]
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    # the hierarchy ends at a single cell
    nl, lx, ly, _, _ = o.mg_level(dt, nlev - 1)
    assert (lx, ly) == (1, 1) and nl == nlev


@pytest.mark.parametrize("nx,ny,bc", [(8, 6, (0, 0, 0, 0)), (7, 5, (0, 0, 0, 0)), (6, 5, (1, 2, 0, 0))])
def test_vcycle_equals_the_dense_five_step_operator(nx, ny, bc):
    w = small_problem(nx, ny, bc, seed=9)
    o = make_oracle(w)
    dt = 60 * 0.4 * w['dx']
    A, _ = fine_matrix(o, dt)
    Minv = dense_vcycle(A, nx, ny, 0.8, 2)
    rng = np.random.default_rng(1)
    for _ in range(3):
        R = rng.normal(size=(3, ny, nx))
        z = interleave(o.mg_apply(dt, R))
        ref = Minv @ interleave(R)
        assert np.abs(z - ref).max() <= 1e-12 * np.abs(ref).max()
    # options reach the cycle
    o.set_option('mg_omega', 0.6); o.set_option('mg_coarse_sweeps', 4)
    R = rng.normal(size=(3, ny, nx))
    ref = dense_vcycle(A, nx, ny, 0.6, 4) @ interleave(R)
    assert np.abs(interleave(o.mg_apply(dt, R)) - ref).max() <= 1e-12 * np.abs(ref).max()


@pytest.mark.parametrize("krylov", [0, 1])
def test_multigrid_preconditioned_solve_equals_dense_lu(krylov):
    w = small_problem(12, 10, seed=3)
    o = make_oracle(w)
    dt = 100 * 0.4 * w['dx']
    A, b = fine_matrix(o, dt)
    x = np.linalg.solve(A, interleave(b))
    o.set_option('preconditioner', 1); o.set_option('krylov', krylov)
    its, res = o.step_implicit(dt, 1e-12, 30, 500)
    E, F = o.get_state()
    got = interleave(np.stack([E, F[0], F[1]]))
    assert res <= 1e-12 and 0 < its < 100
    assert np.linalg.norm(got - x) <= 1e-9 * np.linalg.norm(x)


def test_multigrid_cuts_the_iteration_count_and_is_grid_independent():
    # PAPER.md:327 (Fig. 1): about 10 iterations with AMG against about 250 with relaxation, constant in the number of cells
    counts = {}
    for n in (32, 64):
        w = W.random_medium(n)
        dt = 100 * 0.4 * w['dx'] / w['c']
        for pk in (0, 1):
            o = make_oracle(w); o.set_option('preconditioner', pk)
            its, res = o.step_implicit(dt, 1e-10, 30, 2000)
            assert res <= 1e-10
            counts[n, pk] = its
    assert counts[64, 1] * 5 < counts[64, 0]
    assert counts[64, 1] <= 1.35 * counts[32, 1]     # measured 30 -> 38 (-> 44 at 128^2, 47 at 256^2: saturating)


def test_vcycle_alone_converges_in_the_diffusion_regime():
    # config-1 type problem (sigma dx >> 1, dt = 100x): the stationary iteration x += M^-1 (b - A x) contracts, and faster
    # than the smoother alone (measured 0.943 against 0.971 at 16^2; unsmoothed aggregation is a preconditioner, not a solver)
    w = W.gaussian_diffusion(16)
    o = make_oracle(w)
    dt = 100 * 0.4 * w['dx'] / w['c']
    A, _ = fine_matrix(o, dt)
    I = np.eye(A.shape[0])
    rho = np.abs(np.linalg.eigvals(I - dense_vcycle(A, 16, 16, 0.8, 2) @ A)).max()
    rho_jacobi = np.abs(np.linalg.eigvals(I - 0.8 * block_diag_inverse(A) @ A)).max()
    assert rho < 1.0 and (1.0 - rho) > 1.5 * (1.0 - rho_jacobi)
