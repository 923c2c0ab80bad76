"""GPU parity, rows a1-a4: the CUDA explicit step (through the C ABI) against the oracle, element by element.

Bar (north_star): relative L2 <= 1e-11 per field after explicit steps on the same seeded inputs."""
import numpy as np
import pytest

import m1_workloads as wl
from helpers import make_oracle, make_gpu, small_random_state, rel_l2, state_rel_l2, assert_parity

pytestmark = pytest.mark.gpu

TOL_EXPLICIT = 1e-11

BCS = [(0, 0, 0, 0), (1, 1, 0, 0), (0, 0, 2, 2), (1, 2, 2, 1), (2, 2, 1, 1), (1, 1, 1, 1)]


def _dt(w):
    return wl.explicit_dt(w["dx"], w["dy"], w["c"])


@pytest.mark.parametrize("kernel", [0, 1, 3])
@pytest.mark.parametrize("bc", BCS)
def test_explicit_step_small_all_boundaries(bc, kernel):
    # 37 x 29: ragged in both directions, dx != dy, c != 1
    w = small_random_state(37, 29, seed=101, dx=0.013, dy=0.021, c=1.3, bc=bc, sig_range=(-1.0, 1.0))
    o, g = make_oracle(w), make_gpu(w, dict(explicit_kernel=kernel))
    dt = _dt(w)
    for _ in range(3):
        o.step_explicit(dt)
        g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), TOL_EXPLICIT)


@pytest.mark.parametrize("kernel", [0, 1, 3])
@pytest.mark.parametrize("shape", [(300, 70), (127, 5), (126, 64), (1, 40), (40, 1), (2, 2), (253, 131)])
def test_explicit_step_ragged_shapes(shape, kernel):
    # several 126-column strips plus a ragged tail; degenerate one-cell-wide grids
    nx, ny = shape
    w = small_random_state(nx, ny, seed=7 + nx + ny, sig_range=(-1.0, 1.0))
    o, g = make_oracle(w), make_gpu(w, dict(explicit_kernel=kernel))
    dt = _dt(w)
    for _ in range(2):
        o.step_explicit(dt)
        g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), TOL_EXPLICIT)


@pytest.mark.parametrize("kernel", [1, 3])
@pytest.mark.parametrize("bc", [(1, 2, 2, 1), (2, 1, 1, 2), (0, 0, 1, 1)])
def test_explicit_step_midsize_long_blocks(bc, kernel):
    # 701 x 1003: blocks of 48 rows (kernel 3: twelve trips of the four-row rotation loop, the last block with a ragged tail of
    # rows handled by the general loader), 24 strips of 30 columns with a ragged last strip, Dirichlet and outflow ghost columns
    # in the branch-free hot loop, y-ghost rows in the prologue and in the tail
    w = small_random_state(701, 1003, seed=77, dx=0.011, dy=0.009, c=1.1, bc=bc, sig_range=(-2.0, 2.0))
    o, g = make_oracle(w), make_gpu(w, dict(explicit_kernel=kernel))
    dt = _dt(w)
    for _ in range(2):
        o.step_explicit(dt)
        g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), TOL_EXPLICIT)


def test_residual_matches_oracle():
    w = small_random_state(61, 47, seed=5, bc=(1, 2, 0, 0))
    o, g = make_oracle(w), make_gpu(w)
    RE, RF = o.residual()
    GE, GF = g.residual()
    assert rel_l2(GE, RE) <= 1e-12 and rel_l2(GF, RF) <= 1e-12


def test_clamped_and_degenerate_cells():
    # |F| > cE in many cells (closure clamp), F = 0 cells, f = 1 exactly tangential to a face
    w = small_random_state(48, 33, seed=9, fmax=1.7)
    w["F"][:, 3, :] = 0.0
    # f = 1 exactly, along y: lambda+- = 0 on the x-faces between such cells (the a+- = 1/2, Lambda = 0 guard).
    # E is a power of two there so that F/(cE) is exactly 1 however the division is carried out: Eq. 14 has a
    # square-root singularity at f = 1 (d lambda/d f ~ (1-f)^-1/2), so one ulp in f would move lambda by 1e-8
    # (DESIGN.md "Conditioning at f = 1").
    w["E"][5, :] = 2.0 ** np.random.default_rng(1).integers(-2, 3, w["nx"])
    w["F"][0, 5, :] = 0.0
    w["F"][1, 5, :] = w["E"][5, :]
    o, g = make_oracle(w), make_gpu(w)
    assert o.count_unrealizable() == g.count_unrealizable()
    assert o.count_unrealizable()[1] > 0
    for kernel in (0, 1, 3):
        o, g = make_oracle(w), make_gpu(w, dict(explicit_kernel=kernel))
        o.step_explicit(1e-3)
        g.step_explicit(1e-3)
        assert_parity(g.get_state(), o.get_state(), TOL_EXPLICIT)


@pytest.mark.parametrize("opts", [dict(well_balanced=0), dict(ap_mode=0), dict(ap_mode=2), dict(eig_mode=1), dict(eig_mode=2),
                                  dict(closure=1), dict(eig_floor=0.1)])
@pytest.mark.parametrize("kernel", [0, 1, 3])
def test_scheme_switches(opts, kernel):
    w = small_random_state(45, 31, seed=13, bc=(1, 1, 0, 0), sig_range=(-1.0, 1.0))
    o, g = make_oracle(w, opts), make_gpu(w, dict(opts, explicit_kernel=kernel))
    dt = _dt(w)
    o.step_explicit(dt)
    g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), TOL_EXPLICIT)


def test_config2_opacity_jump_stays_steady():
    # BASELINE.json configs[1]: the discrete steady state must stay steady under 50 explicit steps, on both sides
    from oracle.steady_profile import steady_profile_1d
    w = wl.opacity_jump(256)
    prof = steady_profile_1d(w["sigma_line"], w["dx"], c=1.0, F0=w["F0"], E_out=w["E_out"], sigma_ghost=w["sigma_ghost"])
    n = w["nx"]
    w["E"] = np.tile(prof["E"], (n, 1))
    w["F"] = np.stack((np.tile(prof["Fx"], (n, 1)), np.zeros((n, n))))
    one = np.ones(n)
    w["ghosts"] = {0: (prof["ghost_lo"][0] * one, np.stack((prof["ghost_lo"][1] * one, 0 * one)), 0 * one, w["sigma_ghost"][0] * one),
                   1: (prof["ghost_hi"][0] * one, np.stack((prof["ghost_hi"][1] * one, 0 * one)), 0 * one, w["sigma_ghost"][1] * one)}
    o, g = make_oracle(w), make_gpu(w)
    dt = _dt(w)
    for _ in range(50):
        o.step_explicit(dt)
    g.steps_explicit(dt, 50)
    Eg, Fg = g.get_state()
    assert_parity((Eg, Fg), o.get_state(), TOL_EXPLICIT)
    drift = max(np.max(np.abs(Eg - w["E"])) / np.max(np.abs(w["E"])), np.max(np.abs(Fg[0] - w["F"][0])) / w["F0"])
    assert drift < 1e-9


def test_config3_random_medium_1024():
    # BASELINE.json configs[2]: one explicit step at 1024^2, every element compared
    w = wl.random_medium(1024, seed=1234)
    o, g = make_oracle(w), make_gpu(w)
    dt = _dt(w)
    o.step_explicit(dt)
    g.step_explicit(dt)
    assert_parity(g.get_state(), o.get_state(), TOL_EXPLICIT)


def test_conservation_periodic():
    # P6: periodic, sigma_a = 0 -> sum(E) conserved to round-off by the CUDA path itself
    w = small_random_state(130, 77, seed=3)
    w["sigma_a"][:] = 0.0
    g = make_gpu(w)
    g.steps_explicit(_dt(w), 10)
    E, _ = g.get_state()
    assert abs(E.sum() - w["E"].sum()) <= 1e-12 * abs(w["E"].sum())


def test_error_codes():
    import paper_2011_13926_b200 as ark
    with pytest.raises(ValueError):
        ark.ArkM1(0, 4, 0.1, 0.1)
    with pytest.raises(ValueError):
        ark.ArkM1(4, 4, 0.1, 0.1, bc=(0, 1, 0, 0))      # periodic must be paired
    g = ark.ArkM1(4, 4, 0.1, 0.1)
    with pytest.raises(RuntimeError):
        g.step_explicit(0.1)                            # no state yet
    w = small_random_state(4, 4, seed=1)
    g.set_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
    with pytest.raises(RuntimeError):
        g.step_explicit(-1.0)
    with pytest.raises(RuntimeError):
        g.step_implicit(0.1, tol=0.0)
    with pytest.raises(RuntimeError):
        g.set_option("no_such_option", 1)


def test_device_and_host_pointers_give_the_same_result():
    import torch
    w = small_random_state(64, 40, seed=17)
    g1 = make_gpu(w)
    import paper_2011_13926_b200 as ark
    g2 = ark.ArkM1(w["nx"], w["ny"], w["dx"], w["dy"], w["c"], bc=w["bc"])
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(w[k])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s")}
    g2.set_state(t["E"], t["F"], t["sigma_a"], t["sigma_s"])
    g1.step_explicit(1e-3)
    g2.step_explicit(1e-3)
    E2 = torch.empty_like(t["E"]); F2 = torch.empty_like(t["F"])
    g2.get_state(out=(E2, F2))
    E1, F1 = g1.get_state()
    assert np.array_equal(E1, E2.cpu().numpy()) and np.array_equal(F1, F2.cpu().numpy())


def test_nonpositive_energy_cells_do_not_poison_the_step():
    # E <= 0 (positivity is not guaranteed): E is floored in the division only, F/(cE) overflows and the
    # clamp must give the same finite result as the oracle's IEEE sequence (1/sqrt(inf) = 0), in every kernel
    w = small_random_state(40, 28, seed=19)
    w["E"][7, 9] = -0.3
    w["E"][20, 3] = 0.0
    for kernel in (0, 1, 3):
        o, g = make_oracle(w), make_gpu(w, dict(explicit_kernel=kernel))
        o.step_explicit(1e-3)
        g.step_explicit(1e-3)
        Eg, Fg = g.get_state()
        assert np.all(np.isfinite(Eg)) and np.all(np.isfinite(Fg))
        assert_parity((Eg, Fg), o.get_state(), TOL_EXPLICIT)
    o, g = make_oracle(w), make_gpu(w)
    V = np.random.default_rng(2).standard_normal((3, 28, 40))
    assert rel_l2(g.apply_operator(0.02, V), o.apply_linear(0.02, V)) <= 1e-12


def test_beam_test_of_the_paper():
    # PAPER.md:410-416 (Sect. 5.3): Dirichlet inflow + outflow boundaries, sigma = 0, both eigenvalue modes.
    # (a) parity with the oracle after 300 steps, inflow at f = 0.999 (at f = 1 exactly Eq. 14 is ill-conditioned);
    # (b) the CUDA path alone at f = 1: the beam is narrower with the eigenvalues of Eq. 14 than with +-c (paper: ~24 vs ~30).
    w = wl.beam(128)
    dt = _dt(w)
    w2 = dict(w)
    Eg, Fg, za, zs = w["ghosts"][0]
    w2["ghosts"] = {0: (Eg, 0.999 * Fg, za, zs)}
    for eig in (0, 1):
        o, g = make_oracle(w2, dict(eig_mode=eig)), make_gpu(w2, dict(eig_mode=eig))
        for _ in range(300):
            o.step_explicit(dt)
        g.steps_explicit(dt, 300)
        assert_parity(g.get_state(), o.get_state(), TOL_EXPLICIT)
    width = {}
    for eig in (0, 1):
        g = make_gpu(w, dict(eig_mode=eig))
        g.steps_explicit(dt, 1400)
        E, F = g.get_state()
        cut = E[64, :] - w["E_bg"]
        width[eig] = int((cut > 0.5 * cut.max()).sum())
        assert g.count_unrealizable() == (0, 0)
    assert width[0] < width[1] and 0.7 <= width[0] / width[1] <= 0.9


def test_side_stream_and_two_handles():
    # the handle enqueues on the stream it was given (torch side stream here); two handles are independent
    import torch
    import paper_2011_13926_b200 as ark
    w = small_random_state(96, 64, seed=23)
    ref = make_gpu(w)
    ref.steps_explicit(1e-3, 3)
    ref.step_implicit(0.05, 1e-10, 30, 500)
    want = ref.get_state()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        dev = {k: torch.from_numpy(np.ascontiguousarray(w[k])).cuda() for k in ("E", "F", "sigma_a", "sigma_s")}
        g = ark.ArkM1(w["nx"], w["ny"], w["dx"], w["dy"], w["c"], bc=w["bc"], stream=side)
        g.set_state(dev["E"], dev["F"], dev["sigma_a"], dev["sigma_s"])
        g.steps_explicit(1e-3, 3)
        g.step_implicit(0.05, 1e-10, 30, 500)
        got = g.get_state()
    assert all(np.array_equal(a, b) for a, b in zip(got, want))
    assert g.kernel_launches() == ref.kernel_launches() and g.device_bytes() == ref.device_bytes() > 0


def test_fast_reciprocal_and_rsqrt_are_accurate_to_one_ulp():
    # the hot kernels replace IEEE div/sqrt by a MUFU seed + Newton steps; measured on the device against
    # the IEEE sequences over 2^20 samples in 200 binades
    import paper_2011_13926_b200 as ark
    e_rcp, e_rsqrt, e_sqrt, e_rcp3 = ark.fastmath_errors(1 << 20)
    ulp = 2.0 ** -52
    assert e_rcp <= ulp and e_rsqrt <= 1.2 * ulp and e_sqrt <= 1.2 * ulp and e_rcp3 <= 1.2 * ulp
