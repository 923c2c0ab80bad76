"""Discrete constant-flux steady state across an opacity jump — TEST INFRASTRUCTURE (oracle tool).

BASELINE.json configs[1] asks for "the constant-flux steady state ... E(x) from the discrete steady profile".
The paper gives the face relation (Eq. 23) and imposes it at the boundary (Eq. 24)
but no closed form for the profile of the full AP-HLL scheme, so the profile is computed here from the
oracle's own residual (reading R8):

  1. recurrence from the outflow end:  P_i = P_{i+1} + sigma_{i+1/2} F0 dx / c  with F == F0 (Eq. 23), and
     P = chi(F0/(cE)) E inverted for E on the large-E branch (scalar bisection on the oracle's closure);
  2. Newton polish of the 1-D discrete equations R(U) = 0 (unknowns E_i, Fx_i; Dirichlet ghosts hold the two
     end states of the recurrence), dense finite-difference Jacobian of oracle_m1_residual on an nx x 1 grid
     that is periodic in y.

This file calls only oracle/ code and numpy.  It is used by tests and by the config-2 parity test to make the
INPUT state handed to both the oracle and the CUDA library.
"""
from __future__ import annotations

import numpy as np

from .oracle_m1 import OracleM1, BC_DIRICHLET, BC_PERIODIC, XLO, XHI


def _pressure(o: OracleM1, E: float, F0: float) -> float:
    return o.closure_point(E, F0, 0.0)["Pxx"]


def _invert_pressure(o: OracleM1, P: float, F0: float, c: float) -> float:
    """E >= F0/c with Pxx(E, F0) = P, on the branch where Pxx grows with E."""
    lo = F0 / c            # f = 1: P = E
    hi = max(4.0 * P, 2.0 * lo) + 1.0
    while _pressure(o, hi, F0) < P:
        hi *= 2.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if _pressure(o, mid, F0) < P:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def steady_profile_1d(sigma_line, dx, c=1.0, F0=0.1, E_out=100.0, sigma_ghost=None, options=None,
                      tol=2e-13, max_newton=12):
    """Returns dict(E[nx], Fx[nx], ghost_lo=(E, Fx), ghost_hi=(E, Fx), residual_inf, newton_iterations).

    sigma_line: total opacity of the nx cells (sigma_a = 0 assumed); sigma_ghost: opacities of the two ghosts
    (default: copies of the end cells); options: dict of oracle scheme switches."""
    sigma_line = np.asarray(sigma_line, dtype=np.float64)
    nx = sigma_line.size
    sg = (sigma_line[0], sigma_line[-1]) if sigma_ghost is None else sigma_ghost
    options = dict(options or {})

    o = OracleM1(nx, 1, dx, 1.0, c, bc=(BC_DIRICHLET, BC_DIRICHLET, BC_PERIODIC, BC_PERIODIC))
    for k, v in options.items():
        o.set_option(k, v)

    # 1. recurrence, from the outflow ghost (index nx) down to the inflow ghost (index -1)
    sig_ext = np.concatenate(([sg[0]], sigma_line, [sg[1]]))   # index k <-> cell k-1
    E_ext = np.empty(nx + 2)
    E_ext[-1] = E_out
    P = _pressure(o, E_out, F0)
    for k in range(nx, -1, -1):
        sig_face = 0.5 * (sig_ext[k] + sig_ext[k + 1])
        P = P + sig_face * F0 * dx / c
        E_ext[k] = _invert_pressure(o, P, F0, c)

    zeros = np.zeros(1)
    o.set_boundary(XLO, [E_ext[0]], [[F0], [0.0]], zeros, [sg[0]])
    o.set_boundary(XHI, [E_ext[-1]], [[F0], [0.0]], zeros, [sg[1]])
    sa = np.zeros((1, nx))
    ss = sigma_line.reshape(1, nx)

    def resid(E, Fx):
        F = np.zeros((2, 1, nx))
        F[0, 0] = Fx
        o.set_state(E.reshape(1, nx), F, sa, ss)
        RE, RF = o.residual()
        return np.concatenate((RE[0], RF[0, 0]))

    E = E_ext[1:-1].copy()
    Fx = np.full(nx, F0)
    scale = np.max(np.abs(E)) * c * c / dx
    r = resid(E, Fx)
    its = 0
    # 2. Newton polish with a dense central finite-difference Jacobian
    while np.max(np.abs(r)) > tol * scale and its < max_newton:
        Jm = np.empty((2 * nx, 2 * nx))
        U = np.concatenate((E, Fx))
        for k in range(2 * nx):
            hstep = 1e-6 * max(abs(U[k]), 1e-3)
            Up, Um = U.copy(), U.copy()
            Up[k] += hstep
            Um[k] -= hstep
            Jm[:, k] = (resid(Up[:nx], Up[nx:]) - resid(Um[:nx], Um[nx:])) / (2.0 * hstep)
        dU = np.linalg.solve(Jm, -r)
        E_new, Fx_new = E + dU[:nx], Fx + dU[nx:]
        r_new = resid(E_new, Fx_new)
        if np.max(np.abs(r_new)) >= np.max(np.abs(r)):   # no further gain: round-off floor reached
            break
        E, Fx, r = E_new, Fx_new, r_new
        its += 1
    return dict(E=E, Fx=Fx, ghost_lo=(E_ext[0], F0), ghost_hi=(E_ext[-1], F0),
                residual_inf=float(np.max(np.abs(r))), scale=float(scale), newton_iterations=its)
