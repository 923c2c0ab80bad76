"""GPU tests of the slab-decomposed step (include/ark_m1.h "Domain-decomposed step").

The decomposition is checked where it can be checked on ONE GPU: all slabs in one process (local transport: device copies and a
summing kernel, nothing waits on another rank), two processes sharing the GPU with halos staged through the host and gloo, and
the NCCL transport with a single rank.  The stitched result must equal the one-slab result — to round-off for the explicit step
(bit for bit with the generic kernel; the marching kernels evaluate a face in their prologue or in their row loop depending on
where a block starts, two instances of the same expressions in which nvcc contracts multiply-adds differently: 1 ulp), to the
solver tolerance for the implicit step — and both must match the oracle."""

ULPS = 4e-16      # a few units in the last place, relative to the largest element of a field
import os
import socket
import tempfile

import numpy as np
import pytest

import m1_workloads as wl
import paper_2011_13926_b200 as ark
from helpers import make_oracle, make_gpu, small_random_state, assert_parity, state_rel_l2

pytestmark = pytest.mark.gpu

BCS = [(0, 0, 0, 0), (1, 1, 0, 0), (0, 0, 1, 2), (1, 2, 2, 1), (2, 2, 1, 1)]


def _dt(w, k=1.0):
    return k * wl.explicit_dt(w["dx"], w["dy"], w["c"])


def _group(w, nranks, **kw):
    g = ark.ArkM1Group(w["nx"], w["ny"], w["dx"], w["dy"], w["c"], bc=w["bc"], nranks=nranks, **kw)
    g.scatter(w)
    return g


@pytest.mark.parametrize("nranks", [2, 3, 5])
@pytest.mark.parametrize("bc", BCS)
def test_explicit_steps_stitch_to_roundoff(bc, nranks):
    # 37 x 29 rows over 2, 3, 5 slabs (ragged: 29 = 9 + 10 + 10, ...), dx != dy, c != 1, every boundary set
    w = small_random_state(37, 29, seed=301, dx=0.013, dy=0.021, c=1.3, bc=bc, sig_range=(-1.0, 1.0))
    one, grp, o = make_gpu(w), _group(w, nranks), make_oracle(w)
    dt = _dt(w)
    for _ in range(3):
        one.step_explicit(dt); grp.step_explicit(dt); o.step_explicit(dt)
    Eg, Fg = grp.get_state()
    assert_parity((Eg, Fg), one.get_state(), 3 * ULPS)
    assert_parity((Eg, Fg), o.get_state(), 1e-11)
    st = grp.comm_stats()
    periodic_y = bc[2] == 0
    links = nranks if periodic_y else nranks - 1
    assert st["exchanges"] == 3 and st["halo_bytes"] == 3 * 2 * links * 5 * 37 * 8


@pytest.mark.parametrize("kernel", [0, 1, 3])
def test_explicit_every_kernel_and_one_row_slabs(kernel):
    w = small_random_state(70, 12, seed=302, bc=(0, 0, 0, 0), sig_range=(-1.0, 1.0))
    one, grp = make_gpu(w, dict(explicit_kernel=kernel)), _group(w, 12)          # twelve slabs of one row each
    grp.set_option("explicit_kernel", kernel)
    dt = _dt(w)
    for _ in range(2):
        one.step_explicit(dt); grp.step_explicit(dt)
    if kernel == 0:       # one thread per cell, one code path: the decomposition changes nothing at all
        assert all(np.array_equal(a, b) for a, b in zip(grp.get_state(), one.get_state()))
    assert_parity(grp.get_state(), one.get_state(), 2 * ULPS)


@pytest.mark.parametrize("nranks", [2, 4])
@pytest.mark.parametrize("bc", BCS)
def test_implicit_step_matches_one_slab_and_oracle(bc, nranks):
    w = small_random_state(45, 38, seed=303, dx=0.02, dy=0.017, c=1.2, bc=bc, sig_range=(-1.0, 1.5))
    one, grp, o = make_gpu(w), _group(w, nranks), make_oracle(w)
    dt = _dt(w, 20.0)
    i1, r1 = one.step_implicit(dt, 1e-11, 30, 2000)
    ig, rg = grp.step_implicit(dt, 1e-11, 30, 2000)
    io, ro = o.step_implicit(dt, 1e-11, 30, 2000)
    assert rg <= 1e-11 and r1 <= 1e-11
    assert state_rel_l2(grp.get_state(), one.get_state()) <= 1e-9
    assert state_rel_l2(grp.get_state(), o.get_state()) <= 1e-8
    assert abs(ig - i1) <= 2 and abs(ig - io) <= max(2, 0.02 * io)
    st = grp.comm_stats()
    # s-step blocks (the default): five all-reduces per block of five columns (dots, Gram matrix, norms, and the two of the refinement
    # round) instead of two per column, plus ||b|| and the residuals
    cycles = -(-ig // 30)                             # a cycle is enqueued whole: 6 blocks x 5 all-reduces, whatever column it stops at
    assert 3 * (ig // 5) <= st["allreduces"] <= 32 * cycles + 4
    grp1 = _group(w, nranks)
    grp1.set_option("arnoldi_block", 1)
    ig1, rg1 = grp1.step_implicit(dt, 1e-11, 30, 2000)
    assert rg1 <= 1e-11 and abs(ig1 - i1) <= 2
    assert grp1.comm_stats()["allreduces"] >= 2 * ig1 + 2          # one column per pass: dots and norm per iteration
    assert state_rel_l2(grp1.get_state(), grp.get_state()) <= 1e-9


def test_implicit_restart_cycles_and_long_restart():
    w = small_random_state(40, 33, seed=304, sig_range=(-1.0, 1.0))
    dt = _dt(w, 60.0)
    for restart in (5, 17, 40):
        one, grp = make_gpu(w), _group(w, 3)
        i1, r1 = one.step_implicit(dt, 1e-10, restart, 4000)
        ig, rg = grp.step_implicit(dt, 1e-10, restart, 4000)
        assert rg <= 1e-10 and abs(ig - i1) <= max(2, 0.02 * i1)
        assert state_rel_l2(grp.get_state(), one.get_state()) <= 1e-8


def test_matter_coupled_steps_decomposed():
    w = wl.stratified_coupled(48, seed=11)
    one, grp, o = make_gpu(w), _group(w, 4), make_oracle(w)
    dte = _dt(w)
    one.step_explicit(dte); grp.step_explicit(dte); o.step_explicit(dte)
    assert_parity(grp.get_state(with_T=True), one.get_state(with_T=True), ULPS)
    assert_parity(grp.get_state(with_T=True), o.get_state(with_T=True), 1e-11)
    i1, _ = one.step_implicit(50 * dte, 1e-11, 30, 3000)
    ig, rg = grp.step_implicit(50 * dte, 1e-11, 30, 3000)
    io, _ = o.step_implicit(50 * dte, 1e-11, 30, 3000)
    assert rg <= 1e-11
    assert state_rel_l2(grp.get_state(with_T=True), o.get_state(with_T=True)) <= 1e-8
    assert state_rel_l2(grp.get_state(with_T=True), one.get_state(with_T=True)) <= 1e-9


def test_mixed_explicit_implicit_sequence_on_config3_window():
    w = wl.random_medium(256, seed=1234)
    one, grp = make_gpu(w), _group(w, 8)
    dt = _dt(w)
    for _ in range(2):
        one.step_explicit(dt); grp.step_explicit(dt)
    i1, _ = one.step_implicit(10 * dt, 1e-10, 30, 4000)
    ig, rg = grp.step_implicit(10 * dt, 1e-10, 30, 4000)
    one.step_explicit(dt); grp.step_explicit(dt)
    assert rg <= 1e-10 and abs(ig - i1) <= 2
    assert state_rel_l2(grp.get_state(), one.get_state()) <= 1e-8


def test_unsupported_options_and_slab_handles_are_rejected():
    w = small_random_state(20, 16, seed=305)
    grp = _group(w, 2)
    with pytest.raises(RuntimeError, match="slab of an ark_m1_group"):
        grp.slabs[0].step_explicit(_dt(w))
    grp.set_option("krylov", 1)
    with pytest.raises(RuntimeError, match="supports GMRES"):
        grp.step_implicit(_dt(w, 10.0))
    with pytest.raises(ValueError):
        ark.ArkM1Group(20, 4, 0.1, 0.1, nranks=5)                # more slabs than rows
    with pytest.raises(ValueError):
        ark.ArkM1Group(20, 16, 0.1, 0.1, bc=(0, 0, 0, 1), nranks=2)   # periodic on one side of y only


def test_nccl_transport_single_rank():
    # one rank: no halos, but the transport is set up (dlopen, ncclCommInitRank) and every reduction goes through ncclAllReduce
    w = small_random_state(33, 27, seed=306)
    try:
        uid = ark.nccl_unique_id()
    except RuntimeError as exc:
        pytest.skip(str(exc))
    one = make_gpu(w)
    grp = ark.ArkM1Group(w["nx"], w["ny"], w["dx"], w["dy"], w["c"], bc=w["bc"], nranks=1, kind="nccl", rank=0, unique_id=uid)
    grp.scatter(w)
    dt = _dt(w)
    one.step_explicit(dt); grp.step_explicit(dt)
    i1, _ = one.step_implicit(20 * dt, 1e-10, 30, 1000)
    ig, rg = grp.step_implicit(20 * dt, 1e-10, 30, 1000)
    assert rg <= 1e-10 and abs(ig - i1) <= 1
    assert state_rel_l2(grp.get_state(), one.get_state()) <= 1e-9
    assert grp.comm_stats()["allreduces"] >= 3 * (ig // 5)         # s-step blocks: at least dots, Gram matrix and norms per block of five columns


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 1, 2, 1)])
def test_two_processes_sharing_the_gpu_with_host_staged_halos(bc):
    # the one multi-PROCESS form that can run on a one-GPU box: the ranks' kernels never wait on one another on the device (the
    # waiting happens on the host, in gloo)
    import torch.multiprocessing as mp
    w = small_random_state(41, 26, seed=307, bc=bc, sig_range=(-1.0, 1.0))
    one = make_gpu(w)
    dt = _dt(w)
    one.step_explicit(dt); one.step_explicit(dt)
    i1, r1 = one.step_implicit(15 * dt, 1e-10, 30, 2000)
    E1, F1 = one.get_state()
    with tempfile.TemporaryDirectory() as d:
        wfile = os.path.join(d, "w.npz")
        flat = {k: v for k, v in w.items() if k != "ghosts"}
        np.savez(wfile, **flat)
        gh = w.get("ghosts") or {}
        ctx = mp.get_context("spawn")
        port = _free_port()
        if gh:
            np.savez(os.path.join(d, "gh.npz"), **{f"s{side}_{k}": a for side, g4 in gh.items() for k, a in enumerate(g4)})
        procs = [ctx.Process(target=_host_rank_with_ghosts, args=(r, 2, port, wfile, d, bool(gh))) for r in range(2)]
        for p in procs:
            p.start()
        for p in procs:
            p.join(300)
        assert all(p.exitcode == 0 for p in procs), [p.exitcode for p in procs]
        parts = sorted((np.load(os.path.join(d, f"rank{r}.npz")) for r in range(2)), key=lambda z: int(z["y0"]))
        E = np.concatenate([z["E"] for z in parts], axis=0)
        F = np.concatenate([z["F"] for z in parts], axis=1)
        assert int(parts[0]["y0"]) == 0 and int(parts[1]["y1"]) == w["ny"] and int(parts[0]["y1"]) == int(parts[1]["y0"])
        assert all(float(z["res"]) <= 1e-10 for z in parts) and abs(int(parts[0]["its"]) - i1) <= 2
        assert int(parts[0]["its"]) == int(parts[1]["its"])
        assert state_rel_l2((E, F), (E1, F1)) <= 1e-8


def _host_rank_with_ghosts(rank, world, port, wfile, outdir, has_gh):
    if has_gh:
        z = np.load(os.path.join(outdir, "gh.npz"))
        sides = sorted({int(k[1]) for k in z.files})
        ghosts = {s: tuple(z[f"s{s}_{k}"] for k in range(4)) for s in sides}
        _host_rank_impl(rank, world, port, wfile, outdir, ghosts)
    else:
        _host_rank_impl(rank, world, port, wfile, outdir, None)


def _host_rank_impl(rank, world, port, wfile, outdir, ghosts):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    w = dict(np.load(wfile, allow_pickle=True))
    w = {k: (v.item() if v.ndim == 0 else v) for k, v in w.items()}
    w["bc"] = tuple(int(b) for b in w["bc"])
    if ghosts:
        w["ghosts"] = ghosts
    tr = ark.gloo_host_transport(dist, rank, world)
    g = ark.ArkM1Group(int(w["nx"]), int(w["ny"]), float(w["dx"]), float(w["dy"]), float(w["c"]), bc=w["bc"], nranks=world, kind="host",
                       rank=rank, transport=tr)
    g.scatter(w)
    dt = wl.explicit_dt(float(w["dx"]), float(w["dy"]), float(w["c"]))
    g.step_explicit(dt); g.step_explicit(dt)
    its, res = g.step_implicit(15 * dt, 1e-10, 30, 2000)
    (y0, y1, E, F), = g.gather()
    np.savez(os.path.join(outdir, f"rank{rank}.npz"), y0=y0, y1=y1, E=E, F=F, its=its, res=res)
    dist.barrier()
    g.close()
    dist.destroy_process_group()
