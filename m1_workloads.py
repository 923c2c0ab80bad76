"""Seeded synthetic inputs for the M1 radiative-transfer step — shared by the oracle tests and the CUDA tests/bench.

This module holds NONE of the method's arithmetic (no closure, no fluxes, no solver): it only draws the
initial fields, opacities and grids that BASELINE.json's configs describe.  Everything is host numpy, fp64,
planes of shape [ny, nx] (x fastest); F has shape [2, ny, nx] = (Fx, Fy).

The paper (arXiv 2011.13926) uses analytic set-ups, not datasets; these generators restate BASELINE.json's
five configs.  Recipes (also in DESIGN.md, "Input recipe"):

  config 1  gaussian_diffusion   : 64^2 unit box, periodic, E = exp(-r^2/(2 s0^2)) + 1e-6, s0 = 0.05, F = 0,
                                   sigma_s = 1e3, sigma_a = 0.
  config 2  opacity_jump         : 256^2 unit box, sigma_a = 0, sigma_s = 1 (x < 1/2) | 1e3 (x >= 1/2), F0 = 0.1;
                                   the discrete steady profile itself is computed by oracle/steady_profile.py.
  config 3/4 random_medium       : draw order with numpy.random.default_rng(seed):
                                   (1) log10 sigma_a ~ U[-3,3]  [ny,nx]   (2) log10 sigma_s ~ U[-3,3]  [ny,nx]
                                   (3) g ~ N(0,1) -> E = exp(g)  (4) u ~ U[0,0.9]  (5) theta ~ U[0,2pi)
                                   both log10-opacity fields are smoothed with a separable periodic 5x5 box mean
                                   (applied to the log field) and exponentiated; |F| = u c E, direction theta.
  config 5  stratified_coupled   : see the function docstring.
  3-D       random_medium_3d     : the config-3 recipe in three dimensions (planes [nz, ny, nx], F = [3, nz, ny, nx]): draw order
                                   (1) g ~ N(0,1) -> E = exp(g)  (2) u ~ U[0, fmax]  (3) a direction vector N(0,1)^3, normalised
                                   (4) log10 sigma_a ~ U[lo, hi]  (5) log10 sigma_s ~ U[lo, hi]; with smooth=True both log fields get
                                   a separable periodic 5-point box mean per direction before exponentiation.
"""
from __future__ import annotations

import numpy as np

CFL_EXPLICIT = 0.4  # explicit dt = CFL * min(dx, dy) / c  (reading R3)


def explicit_dt(dx, dy, c=1.0, cfl=CFL_EXPLICIT):
    return cfl * min(dx, dy) / c


def cell_centres(nx, ny, lx=1.0, ly=1.0):
    dx, dy = lx / nx, ly / ny
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dy
    return x, y, dx, dy


def gaussian_diffusion(n=64, sigma_s=1e3, s0=0.05, floor=1e-6):
    """BASELINE.json configs[0]."""
    x, y, dx, dy = cell_centres(n, n)
    X, Y = np.meshgrid(x, y)
    r2 = (X - 0.5) ** 2 + (Y - 0.5) ** 2
    E = np.exp(-r2 / (2.0 * s0 * s0)) + floor
    F = np.zeros((2, n, n))
    return dict(nx=n, ny=n, dx=dx, dy=dy, c=1.0, bc=(0, 0, 0, 0), E=E, F=F,
                sigma_a=np.zeros((n, n)), sigma_s=np.full((n, n), float(sigma_s)), s0=s0, floor=floor)


def opacity_jump(n=256, sig_lo=1.0, sig_hi=1e3, F0=0.1, E_out=100.0):
    """BASELINE.json configs[1]: the opacity field and the boundary data of the constant-flux steady state.
    The discrete steady profile E(x) is NOT computed here (it needs the scheme: oracle/steady_profile.py)."""
    x, y, dx, dy = cell_centres(n, n)
    sig_line = np.where(x < 0.5, sig_lo, sig_hi)
    return dict(nx=n, ny=n, dx=dx, dy=dy, c=1.0, bc=(1, 1, 0, 0), x=x,
                sigma_a=np.zeros((n, n)), sigma_s=np.tile(sig_line, (n, 1)), sigma_line=sig_line,
                sigma_ghost=(sig_lo, sig_hi), F0=F0, E_out=E_out)


def beam(n=128, angle_deg=45.0, E_beam=1.0, T_ratio=0.3):
    """Beam test of the paper (Sect. 5.3): box [-1,1]^2, n x n cells, sigma = 0, background in equilibrium at
    T0 = T_ratio * T_beam (E = T_ratio^4 E_beam, F = 0); a beam with f = 1 enters through x = -1, y in [-0.875, -0.75] at
    `angle_deg`.  Boundaries: Dirichlet on x = -1 (beam / background ghosts), outflow elsewhere.  Units c = 1."""
    dx = dy = 2.0 / n
    y = -1.0 + (np.arange(n) + 0.5) * dy
    E_bg = E_beam * T_ratio ** 4
    E = np.full((n, n), E_bg)
    F = np.zeros((2, n, n))
    inb = (y >= -0.875) & (y <= -0.75)
    th = np.deg2rad(angle_deg)
    Eg = np.where(inb, E_beam, E_bg)
    Fg = np.stack((np.where(inb, E_beam * np.cos(th), 0.0), np.where(inb, E_beam * np.sin(th), 0.0)))
    zeros = np.zeros(n)
    return dict(nx=n, ny=n, dx=dx, dy=dy, c=1.0, bc=(1, 2, 2, 2), E=E, F=F, sigma_a=np.zeros((n, n)), sigma_s=np.zeros((n, n)),
                ghosts={0: (Eg, Fg, zeros, zeros)}, inflow_cells=int(inb.sum()), E_bg=E_bg)


def marshak(nx=400, sigma=1e4, rho_cv=1.0, T0=0.3, T_left=1.0):
    """Marshak wave of the paper (Sect. 5.1) in non-dimensional units (c = a_r = 1, unit length):
    nx x 1 cells, sigma dx = 25, medium in equilibrium at T0 (E = T0^4, F = 0), a source at T_left lit at the left boundary
    (Dirichlet ghost E = T_left^4, F = 0), zero-gradient on the right, frozen hydrodynamics, constant rho c_v."""
    dx = 1.0 / nx
    one = np.ones((1, nx))
    return dict(nx=nx, ny=1, dx=dx, dy=1.0, c=1.0, bc=(1, 2, 0, 0), E=T0 ** 4 * one, F=np.zeros((2, 1, nx)), T=T0 * one,
                sigma_a=sigma * one, sigma_s=0.0 * one, rho_cv=rho_cv * one,
                ghosts={0: (np.array([T_left ** 4]), np.zeros((2, 1)), np.array([sigma]), np.array([0.0]))},
                sigma=sigma, T0=T0, T_left=T_left, a_r=1.0)


def _box5_periodic(a):
    out = np.zeros_like(a)
    for s in (-2, -1, 0, 1, 2):
        out += np.roll(a, s, axis=1)
    a = out / 5.0
    out = np.zeros_like(a)
    for s in (-2, -1, 0, 1, 2):
        out += np.roll(a, s, axis=0)
    return out / 5.0


def random_medium(n=1024, seed=1234, c=1.0, ny=None):
    """BASELINE.json configs[2] and configs[3] (same generator, n = 1024 and 4096)."""
    nx, ny = n, (n if ny is None else ny)
    rng = np.random.default_rng(seed)
    lsa = rng.uniform(-3.0, 3.0, size=(ny, nx))
    lss = rng.uniform(-3.0, 3.0, size=(ny, nx))
    g = rng.standard_normal(size=(ny, nx))
    u = rng.uniform(0.0, 0.9, size=(ny, nx))
    th = rng.uniform(0.0, 2.0 * np.pi, size=(ny, nx))
    sigma_a = 10.0 ** _box5_periodic(lsa)
    sigma_s = 10.0 ** _box5_periodic(lss)
    E = np.exp(g)
    F = np.empty((2, ny, nx))
    F[0] = u * c * E * np.cos(th)
    F[1] = u * c * E * np.sin(th)
    dx, dy = 1.0 / nx, 1.0 / ny
    return dict(nx=nx, ny=ny, dx=dx, dy=dy, c=c, bc=(0, 0, 0, 0), E=E, F=F, sigma_a=sigma_a, sigma_s=sigma_s, seed=seed)


def random_medium_3d(nx, ny=None, nz=None, seed=1234, c=1.0, fmax=0.9, log_sigma=(-3.0, 3.0), smooth=True):
    """The random medium in three dimensions (SURVEY 8(f) row 4 tail); see the module docstring for the draw order."""
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    rng = np.random.default_rng(seed)
    shp = (nz, ny, nx)
    E = np.exp(rng.standard_normal(shp))
    u = rng.uniform(0.0, fmax, shp)
    v = rng.standard_normal((3,) + shp)
    v /= np.linalg.norm(v, axis=0)
    F = u * c * E * v

    def box(a):
        for ax in range(3):
            a = sum(np.roll(a, sh, axis=ax) for sh in (-2, -1, 0, 1, 2)) / 5.0
        return a
    la, ls = rng.uniform(*log_sigma, shp), rng.uniform(*log_sigma, shp)
    if smooth:
        la, ls = box(la), box(ls)
    return dict(nx=nx, ny=ny, nz=nz, c=c, E=E, F=F, sigma_a=10.0 ** la, sigma_s=10.0 ** ls, seed=seed)


def stratified_coupled(n=2048, seed=4321, c=1.0, gamma=5.0 / 3.0, H=0.1, kappa=1e3, u_rms=1e-3, a_r=1.0):
    """BASELINE.json configs[4] (stage 2).  Draw order with default_rng(seed):
    (1) xi ~ N(0,1) [ny,nx] density perturbation  (2) g ~ N(0, 0.1^2) -> T = exp(g)  (3) psi ~ N(0,1) stream function.
    rho = exp(-y/H)(1 + 0.01 xi); rho c_v = rho/(gamma-1) (k_b/(mu m_H) = 1); sigma_a = sigma_s = kappa rho;
    E = a_r T^4, F = 0; velocity = curl of the 5x5-box-smoothed (three passes) periodic stream function by central
    differences, rescaled to rms |u| = u_rms c; source_E = Q in the 2x2 central cells, Q = 100/dt_explicit."""
    nx = ny = n
    x, y, dx, dy = cell_centres(nx, ny)
    rng = np.random.default_rng(seed)
    xi = rng.standard_normal(size=(ny, nx))
    g = 0.1 * rng.standard_normal(size=(ny, nx))
    psi = rng.standard_normal(size=(ny, nx))
    rho = np.exp(-y / H)[:, None] * (1.0 + 0.01 * xi)
    T = np.exp(g)
    for _ in range(3):
        psi = _box5_periodic(psi)
    ux = (np.roll(psi, -1, axis=0) - np.roll(psi, 1, axis=0)) / (2.0 * dy)
    uy = -(np.roll(psi, -1, axis=1) - np.roll(psi, 1, axis=1)) / (2.0 * dx)
    scale = u_rms * c / np.sqrt(np.mean(ux * ux + uy * uy))
    ux, uy = ux * scale, uy * scale
    E = a_r * T ** 4
    src = np.zeros((ny, nx))
    src[ny // 2 - 1: ny // 2 + 1, nx // 2 - 1: nx // 2 + 1] = 100.0 / explicit_dt(dx, dy, c)
    return dict(nx=nx, ny=ny, dx=dx, dy=dy, c=c, bc=(0, 0, 0, 0), E=E, F=np.zeros((2, ny, nx)), T=T,
                sigma_a=kappa * rho, sigma_s=kappa * rho, rho_cv=rho / (gamma - 1.0), ux=ux, uy=uy, source_E=src,
                a_r=a_r, seed=seed)
