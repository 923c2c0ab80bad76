"""GPU tests of the block forms of the Arnoldi process (option arnoldi_block: 1 = one column per pass over the basis, 2 = two columns,
3..5 = s-step blocks, 5 the default; csrc/krylov_kernels.cu, csrc/krylov_sstep.cu).  In exact arithmetic every variant produces the
iterates of GMRES(m), so the bar is the one-column solver's and the oracle's: the same iteration count (the residual estimate of
every column is the same Givens recurrence), the same residual history, the state within the implicit parity bar (1e-8; measured
1e-13 or better between variants)."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_gpu, make_oracle, small_random_state, state_rel_l2

pytestmark = pytest.mark.gpu

BLOCKS = [2, 3, 4, 5]


def _solve(w, dt, blk, restart=30, tol=1e-10, maxit=4000, opts=None):
    g = make_gpu(w, dict(opts or {}, arnoldi_block=blk))
    its, res = g.step_implicit(dt, tol, restart, maxit)
    return its, res, g.get_state(), np.array(g.history())


def _check_against_one_column(w, dt, restart=30, tol=1e-10, maxit=4000, opts=None, blocks=BLOCKS, dcount=1, converges=True, hist_tol=1e-3):
    i1, r1, s1, h1 = _solve(w, dt, 1, restart, tol, maxit, opts)
    assert (r1 <= tol) == converges
    for blk in blocks:
        ib, rb, sb, hb = _solve(w, dt, blk, restart, tol, maxit, opts)
        if converges:
            assert rb <= tol, f"arnoldi_block={blk}: residual {rb:.2e}"
        else:
            assert abs(rb - r1) <= 1e-6 * r1, f"arnoldi_block={blk}: residual {rb:.6e} against {r1:.6e} at the iteration limit"
        assert abs(ib - i1) <= dcount, f"arnoldi_block={blk}: {ib} iterations against {i1}"
        assert state_rel_l2(sb, s1) <= 1e-9
        k = min(len(h1), len(hb), 40)       # the histories agree while rounding has not had 100+ iterations to separate them
        assert np.max(np.abs(np.log10(hb[1:k] / h1[1:k]))) <= hist_tol, f"arnoldi_block={blk}: residual histories differ"
    return i1


@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 2, 2, 1), (2, 2, 1, 1)])
@pytest.mark.parametrize("shape,k", [((96, 80), 20.0), ((61, 47), 10.0), ((37, 29), 30.0)])
def test_block_variants_reproduce_the_one_column_solver(shape, k, bc):
    # odd numbers of unknowns (61 x 47, 37 x 29: the vector kernels' scalar tail), every boundary kind
    nx, ny = shape
    w = small_random_state(nx, ny, seed=500 + nx, bc=bc)
    _check_against_one_column(w, k * wl.explicit_dt(w["dx"], w["dy"], w["c"]))


@pytest.mark.parametrize("restart", [3, 5, 7, 13, 17, 31, 40, 60, 100])
def test_block_variants_with_restart_lengths_that_do_not_divide(restart):
    # blocks of 5 / 4 / 3 followed by a pair and / or a single column; more than 32 basis vectors (two launches of the dot kernel)
    w = wl.random_medium(128, seed=9)
    dt = 40 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    _check_against_one_column(w, dt, restart=restart, dcount=2)


def test_block_variants_against_the_oracle():
    w = small_random_state(72, 50, seed=77, bc=(1, 1, 0, 0))
    dt = 25 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    o = make_oracle(w)
    io, ro = o.step_implicit(dt, 1e-10, 30, 4000)
    for blk in [1] + BLOCKS:
        ib, rb, sb, _ = _solve(w, dt, blk)
        assert rb <= 1e-10 and abs(ib - io) <= max(2, 0.02 * io)
        assert state_rel_l2(sb, o.get_state()) <= 1e-8


@pytest.mark.parametrize("shape", [(2, 3), (3, 3), (4, 2), (5, 4)])
def test_krylov_space_exhausted_inside_a_block(shape):
    # 18 .. 60 unknowns with restart 30: the space is exhausted (or the tolerance met) inside a block; a truncated block must end the
    # cycle and the solve must still reach the dense solution
    nx, ny = shape
    w = small_random_state(nx, ny, seed=600 + nx * ny, bc=(0, 0, 0, 0))
    dt = 50 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    o = make_oracle(w)
    M, b = o.dense_matrix(dt)
    x = np.linalg.solve(M, b).reshape(3, ny, nx)
    for blk in [1] + BLOCKS:
        ib, rb, (E, F), _ = _solve(w, dt, blk, tol=1e-12, maxit=400)
        assert rb <= 1e-12, f"arnoldi_block={blk}: residual {rb:.2e} after {ib} iterations"
        got = np.concatenate((E[None], F))
        assert np.linalg.norm(got - x) <= 1e-9 * np.linalg.norm(x)


def test_block_variants_with_matter_coupling_and_loose_tolerance():
    w = small_random_state(80, 64, seed=91, bc=(0, 0, 2, 1), sig_range=(-1.0, 2.0))
    rng = np.random.default_rng(4)
    w["T"] = rng.uniform(0.5, 1.5, (w["ny"], w["nx"]))
    w["rho_cv"] = rng.uniform(0.5, 2.0, (w["ny"], w["nx"]))
    dt = 100 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    _check_against_one_column(w, dt, tol=1e-6)        # the stop test fires in the middle of a block
    _check_against_one_column(w, dt, tol=1e-10, maxit=23, dcount=0, converges=False)   # maxit reached inside a block: same count, same state


@pytest.mark.parametrize("k", [100.0, 200.0])
def test_ill_conditioned_blocks_are_refined(k):
    # The smooth diffusive problem at 1024^2: the residual falls tenfold per iteration, so the vectors of the first s-step block are
    # nearly dependent (pivot ratios 1, 1.6e-4, 3.5e-6, 7.9e-9, 4.0e-12 measured).  Without the second round of the in-block
    # orthogonalisation the 5-column block needed 29 iterations instead of 17 at 100x and 44 instead of 29 at 200x.
    w = wl.gaussian_diffusion(1024)
    dt = k * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    # histories: equal to 1e-5 relative down to a residual of 1e-8, within 0.3 % at 1e-10 (eleven orders below the start)
    _check_against_one_column(w, dt, dcount=1, hist_tol=1e-2)


def _stats(w, dt, blk, restart=30, tol=1e-10, maxit=4000):
    g = make_gpu(w, dict(arnoldi_block=blk))
    its, res = g.step_implicit(dt, tol, restart, maxit)
    return its, res, g.block_stats()


@pytest.mark.parametrize("blk", [3, 4, 5])
def test_well_conditioned_blocks_finish_in_the_update_pass(blk):
    # bench medium (small): the dot pass predicts the in-block solve from S - C^T C, the update pass applies it and the measured Gram
    # matrix of the result passes the orthogonality check: no block takes the separate in-block pass, and the count is that of the
    # one-column solver (checked for the same systems above).  Every full block of the solve is accounted for in the four counters.
    w = wl.random_medium(192, seed=21)
    dt = 10 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    i1, r1, s1 = _stats(w, dt, 1)
    assert s1 == dict(update_pass=0, predicted_refined=0, separate_pass=0, separate_refined=0)
    ib, rb, sb = _stats(w, dt, blk)
    assert rb <= 1e-10 and abs(ib - i1) <= 1
    assert sb["update_pass"] >= 1 and sb["separate_pass"] == 0 and sb["separate_refined"] == 0 and sb["predicted_refined"] == 0
    full_blocks_per_cycle = 30 // blk
    assert sum(sb.values()) <= -(-ib // 30) * full_blocks_per_cycle and sum(sb.values()) >= (ib // 30) * full_blocks_per_cycle


def test_ill_conditioned_blocks_do_not_use_the_prediction():
    # smooth diffusive problem (see test_ill_conditioned_blocks_are_refined): the predicted pivot ratios of the first block fall below
    # 1e-3, so the prediction is not applied and the block takes the measured factorisation with its second round
    w = wl.gaussian_diffusion(1024)
    dt = 100 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    its, res, st = _stats(w, dt, 5)
    assert res <= 1e-10 and its <= 18
    assert st["separate_refined"] >= 1 and st["update_pass"] + st["predicted_refined"] < sum(st.values())
