"""GPU parity at BASELINE.json's full bench size (configs[3], 4096 x 4096), in the launch configuration bench.py times.

Explicit: the oracle still finishes one step at this size in seconds, so every element is compared.  Implicit: the
oracle's solve would take minutes; instead the CUDA solution is substituted into the ORACLE's flux-form operator (one
application) and the oracle's residual of the linear system is checked — a property that holds at any size."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, make_gpu, rel_l2, state_rel_l2, assert_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def w4096():
    return wl.random_medium(4096, seed=1234)


def test_explicit_step_4096_every_element(w4096):
    w = w4096
    dt = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    o, g = make_oracle(w), make_gpu(w)
    o.step_explicit(dt)
    g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), 1e-11)


@pytest.mark.parametrize("krylov", [0, 1])
def test_implicit_step_4096_satisfies_the_oracles_linear_system(w4096, krylov):
    w = w4096
    dt = 10.0 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    g = make_gpu(w, dict(krylov=krylov))
    its, res = g.step_implicit(dt, 1e-10, 30, 4000)
    assert res <= 1e-10 and 0 < its < 4000
    E, F = g.get_state()
    x = np.concatenate((E[None], F))
    o = make_oracle(w)                                   # holds U^n: the coefficients of the linearisation
    Ax = o.apply_linear(dt, x, mode=0)
    b = np.concatenate((w["E"][None], w["F"]))           # periodic, no T: b = U^n
    assert np.linalg.norm((b - Ax).ravel()) <= 2e-10 * np.linalg.norm(b.ravel())
    # sampled cells: the implicit update is not the identity and not the explicit update
    assert rel_l2(x, b) > 1e-3


@pytest.mark.parametrize("prec,krylov", [(64, 0), (32, 1)])
def test_multigrid_step_4096_satisfies_the_oracles_linear_system(w4096, prec, krylov):
    # the multigrid-preconditioned solve at the bench size, in the configurations bench.py times (fp32 blocks + BiCGStab on the
    # rough medium; fp64 blocks + GMRES as the reference form): the solution must satisfy the ORACLE's flux-form system
    w = w4096
    dt = 10.0 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    g = make_gpu(w, dict(preconditioner=1, mg_precision=prec, krylov=krylov))
    its, res = g.step_implicit(dt, 1e-10, 30, 400)
    assert res <= 1e-10 and 0 < its < 40
    E, F = g.get_state()
    x = np.concatenate((E[None], F))
    o = make_oracle(w)
    Ax = o.apply_linear(dt, x, mode=0)
    b = np.concatenate((w["E"][None], w["F"]))
    assert np.linalg.norm((b - Ax).ravel()) <= 2e-10 * np.linalg.norm(b.ravel())


def test_vcycle_1024_matches_oracle():
    # 11 levels, many tiles: the cycle element by element against the oracle's at config 3's size
    w = wl.random_medium(1024, seed=1234)
    dt = 100.0 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    o, g = make_oracle(w, dict(preconditioner=1)), make_gpu(w, dict(preconditioner=1))
    R = np.random.default_rng(11).standard_normal((3, 1024, 1024))
    assert rel_l2(g.apply_preconditioner(dt, R), o.mg_apply(dt, R)) <= 1e-9


def test_8192_grid_indices_beyond_32_bits():
    # 67 M cells, 201 M unknowns: plane offsets (k N, k <= 36) exceed 2^31; explicit step against the oracle on every element,
    # the implicit solution in the oracle's operator, multigrid and compressed-basis solves against it
    n = 8192
    w = wl.random_medium(n, seed=99)
    dt = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    o, g = make_oracle(w), make_gpu(w)
    o.step_explicit(dt)
    g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), 1e-11)
    E0, F0 = g.get_state()
    b = np.concatenate((E0[None], F0))
    its, res = g.step_implicit(10.0 * dt, 1e-10, 30, 1000)
    assert res <= 1e-10 and 0 < its < 200
    E, F = g.get_state()
    x = np.concatenate((E[None], F))
    g.close()
    Ax = o.apply_linear(10.0 * dt, x, mode=0)            # the oracle holds the same U^n (its own explicit step)
    assert np.linalg.norm((b - Ax).ravel()) <= 2e-10 * np.linalg.norm(b.ravel())
    del o, Ax
    for opts in (dict(preconditioner=1, mg_precision=32, krylov=1), dict(basis_precision=32)):
        g2 = make_gpu(dict(w, E=E0, F=F0), opts)
        its2, res2 = g2.step_implicit(10.0 * dt, 1e-10, 30, 1000)
        E2, F2 = g2.get_state()
        g2.close()
        assert res2 <= 1e-10
        assert rel_l2(np.concatenate((E2[None], F2)), x) <= 1e-8
