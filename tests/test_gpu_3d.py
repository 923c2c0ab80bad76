"""GPU parity of the 3-D step (csrc/m1_3d.cu) against the 3-D oracle (oracle/oracle_m1_3d.c), element by element.
Bars as in 2-D: explicit relative L2 <= 1e-11 (and every element within 1e-11 of the field's maximum), implicit <= 1e-8 with the
GMRES residual converged, iteration counts within 2 or 2 %."""
import numpy as np
import pytest

import m1_workloads as wl
import paper_2011_13926_b200 as ark
from helpers import assert_parity, state_rel_l2
from oracle.oracle_m1_3d import OracleM1_3D
from oracle import oracle_m1_3d

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _build():
    oracle_m1_3d.build()


def rough3(nx, ny, nz, seed, c=1.0, fmax=0.9, sig=(-1.0, 1.0)):
    w = wl.random_medium_3d(nx, ny, nz, seed=seed, c=c, fmax=fmax, log_sigma=sig, smooth=False)
    return w["E"], w["F"], w["sigma_a"], w["sigma_s"]


def pair(shape, d, c, bc, state):
    nx, ny, nz = shape
    o = OracleM1_3D(nx, ny, nz, *d, c, bc)
    g = ark.ArkM1_3D(nx, ny, nz, *d, c, bc)
    o.set_state(*state); g.set_state(*state)
    return o, g


BCS3 = [(0, 0, 0, 0, 0, 0), (2, 2, 0, 0, 0, 0), (0, 0, 2, 2, 2, 2), (2, 2, 2, 2, 2, 2)]


@pytest.mark.parametrize("kernel", [1, 0])
@pytest.mark.parametrize("bc", BCS3)
@pytest.mark.parametrize("shape", [(19, 13, 11), (33, 5, 7), (1, 9, 1), (130, 3, 2)])
def test_explicit_3d_parity(shape, bc, kernel):
    c, d = 1.3, (0.013, 0.021, 0.017)
    o, g = pair(shape, d, c, bc, rough3(*shape, seed=501 + shape[0], c=c))
    g.set_option("explicit_kernel", kernel)
    dt = 0.4 * min(d) / c / 1.5            # the unsplit 3-D limit is a third, not a half
    for _ in range(3):
        o.step_explicit(dt); g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), 1e-11)


@pytest.mark.parametrize("kernel", [1, 0])
def test_explicit_3d_clamped_and_nonpositive_cells(kernel):
    shape, c, d = (12, 9, 8), 1.0, (0.1, 0.1, 0.1)
    E, F, sa, ss = rough3(*shape, seed=502, fmax=1.6)          # |F| > cE in many cells: clamp
    E[2, 3, 4] = -0.5; E[1, 1, 1] = 0.0; F[:, 5, 5, 5] = 0.0      # E <= 0 guard, F = 0
    o, g = pair(shape, d, c, (0, 0, 2, 2, 0, 0), (E, F, sa, ss))
    g.set_option("explicit_kernel", kernel)
    o.step_explicit(0.02); g.step_explicit(0.02)
    assert_parity(g.get_state(), o.get_state(), 1e-11)


@pytest.mark.parametrize("bc", BCS3)
@pytest.mark.parametrize("ratio", [10.0, 60.0])
def test_implicit_3d_parity(bc, ratio):
    shape, c, d = (14, 11, 9), 1.2, (0.02, 0.025, 0.03)
    o, g = pair(shape, d, c, bc, rough3(*shape, seed=503, c=c, sig=(-1.0, 1.5)))
    dt = ratio * 0.4 * min(d) / c
    io, ro = o.step_implicit(dt, 1e-10, 30, 3000)
    ig, rg = g.step_implicit(dt, 1e-10, 30, 3000)
    assert ro <= 1e-10 and rg <= 1e-10
    assert state_rel_l2(g.get_state(), o.get_state()) <= 1e-8
    assert abs(ig - io) <= max(2, 0.02 * io), (ig, io)


def test_implicit_3d_restart_cycles_clamped_cells_and_sequence():
    shape, c, d = (10, 8, 12), 1.0, (0.05, 0.04, 0.06)
    o, g = pair(shape, d, c, (0, 0, 0, 0, 2, 2), rough3(*shape, seed=504, fmax=1.3))
    dt = 0.4 * min(d)
    o.step_explicit(dt / 2); g.step_explicit(dt / 2)
    for restart in (7, 30):
        io, ro = o.step_implicit(40 * dt, 1e-10, restart, 3000)
        ig, rg = g.step_implicit(40 * dt, 1e-10, restart, 3000)
        assert rg <= 1e-10 and abs(ig - io) <= max(2, 0.03 * io), (restart, ig, io)
        assert state_rel_l2(g.get_state(), o.get_state()) <= 1e-8
    assert g.kernel_launches() > 0


def test_3d_mid_size_many_blocks():
    # 96 x 80 x 64 = 491 520 cells: thousands of blocks, the oracle still finishes in seconds
    shape, c, d = (96, 80, 64), 1.0, (1 / 96, 1 / 80, 1 / 64)
    o, g = pair(shape, d, c, (0, 0, 0, 0, 0, 0), rough3(*shape, seed=505))
    dt = 0.4 * min(d) / 1.5
    o.step_explicit(dt); g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), 1e-11)
    io, ro = o.step_implicit(5 * dt, 1e-10, 30, 500)
    ig, rg = g.step_implicit(5 * dt, 1e-10, 30, 500)
    assert rg <= 1e-10 and abs(ig - io) <= 2
    assert state_rel_l2(g.get_state(), o.get_state()) <= 1e-8


@pytest.mark.parametrize("bc", BCS3)
def test_operator_and_preconditioner_3d_against_the_oracle(bc):
    # A V from the solver's own assembly + operator kernels against the oracle's flux form; A M^-1 V with M^-1 from the oracle's
    # 4x4 diagonal blocks (which the oracle obtains by applying its operator to unit vectors — no block formula shared)
    shape, c, d = (9, 7, 6), 1.2, (0.02, 0.025, 0.03)
    o, g = pair(shape, d, c, bc, rough3(*shape, seed=506, c=c, fmax=1.2))
    dt = 25 * 0.4 * min(d) / c
    V = np.random.default_rng(1).standard_normal((4,) + shape[::-1])
    Ao = o.apply_linear(dt, V)
    assert np.max(np.abs(g.apply_operator(dt, V) - Ao)) <= 1e-13 * np.max(np.abs(Ao))
    B = o.diag_blocks(dt)
    N = V[0].size
    Z = np.stack([np.linalg.solve(B[k], V.reshape(4, N)[:, k]) for k in range(N)], axis=1).reshape(V.shape)
    AMo = o.apply_linear(dt, Z)
    assert np.max(np.abs(g.apply_operator(dt, V, precond=True) - AMo)) <= 1e-12 * np.max(np.abs(AMo))


@pytest.mark.parametrize("restart", [30, 7])
def test_3d_block_arnoldi_reproduces_the_one_column_solver(restart):
    # arnoldi_block = 5 (default) / 3 against 1: same iteration count, same state (the s-step kernels of krylov_sstep.cu on 4N-vectors)
    shape, d, c, bc = (40, 23, 17), (0.02, 0.03, 0.025), 1.2, (0, 0, 2, 2, 0, 0)
    state = rough3(*shape, seed=21, c=c)
    dt = 20 * 0.4 * min(d) / c
    res = {}
    for blk in (1, 3, 5):
        g = ark.ArkM1_3D(*shape, *d, c, bc)
        g.set_option("arnoldi_block", blk)
        g.set_state(*state)
        its, r = g.step_implicit(dt, 1e-10, restart, 2000)
        assert r <= 1e-10
        res[blk] = (its, g.get_state())
    for blk in (3, 5):
        assert abs(res[blk][0] - res[1][0]) <= 1
        assert state_rel_l2(res[blk][1], res[1][1]) <= 1e-9
