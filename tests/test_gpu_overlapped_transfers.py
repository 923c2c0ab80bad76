"""GPU tests of the overlapped state transfers (csrc/pipeline.cu: ark_m1_prefetch_state / commit_state / get_state_async /
wait_transfers): a loop of steps fed from host buffers through the copy stream gives, bit for bit, what the same loop gives with the
blocking ark_m1_set_state / ark_m1_get_state — the transfers compute nothing — and the blocking path is the one every parity test
against the oracle uses."""
import numpy as np
import pytest
import torch

import m1_workloads as wl
from helpers import make_gpu, small_random_state

pytestmark = pytest.mark.gpu


def _states(nx, ny, k):
    return [small_random_state(nx, ny, seed=100 + s, bc=(0, 0, 0, 0)) for s in range(k)]


def _pinned(w):
    return {key: torch.from_numpy(np.ascontiguousarray(w[key])).pin_memory() for key in ("E", "F", "sigma_a", "sigma_s")}


def test_pipelined_loop_equals_blocking_loop_bit_for_bit():
    nx, ny, K = 160, 96, 4
    ws = _states(nx, ny, K)
    dt = 5 * wl.explicit_dt(ws[0]["dx"], ws[0]["dy"], ws[0]["c"])
    # blocking reference: a new state each step
    g = make_gpu(ws[0])
    ref = []
    for w in ws:
        g.set_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
        g.step_explicit(0.1 * dt)
        its, res = g.step_implicit(dt, 1e-10, 30, 2000)
        E, F = g.get_state()
        ref.append((its, E.copy(), F.copy()))
    # pipelined: the next state goes up and the last result comes down beside the running step
    g2 = make_gpu(ws[0])
    hosts = [_pinned(w) for w in ws]
    outs = [(torch.empty((ny, nx), dtype=torch.float64).pin_memory(), torch.empty((2, ny, nx), dtype=torch.float64).pin_memory()) for _ in ws]
    g2.prefetch_state(hosts[0]["E"], hosts[0]["F"], hosts[0]["sigma_a"], hosts[0]["sigma_s"])
    its_p = []
    for k in range(K):
        g2.commit_state()
        if k + 1 < K:
            h = hosts[k + 1]
            g2.prefetch_state(h["E"], h["F"], h["sigma_a"], h["sigma_s"])
        g2.step_explicit(0.1 * dt)
        its, res = g2.step_implicit(dt, 1e-10, 30, 2000)
        its_p.append(its)
        g2.get_state_async(outs[k])
    g2.wait_transfers()
    assert g2.device_bytes() - g.device_bytes() == 8 * nx * ny * 8          # staging (5 planes) + snapshot (3 planes), nothing else
    for k in range(K):
        assert its_p[k] == ref[k][0]
        assert np.array_equal(outs[k][0].numpy(), ref[k][1]) and np.array_equal(outs[k][1].numpy(), ref[k][2])


def test_same_output_buffer_reused_and_pageable_arrays():
    # one output pair reused every step (the second download waits on the device for the first); numpy (pageable) inputs
    nx, ny = 61, 47
    ws = _states(nx, ny, 3)
    dt = 3 * wl.explicit_dt(ws[0]["dx"], ws[0]["dy"], ws[0]["c"])
    g = make_gpu(ws[0])
    E_out = np.empty((ny, nx)); F_out = np.empty((2, ny, nx))
    last = None
    for w in ws:
        g.prefetch_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
        g.commit_state()
        g.step_explicit(dt)
        g.get_state_async((E_out, F_out))
        last = w
    g.wait_transfers()
    gr = make_gpu(last)
    gr.step_explicit(dt)
    E, F = gr.get_state()
    assert np.array_equal(E_out, E) and np.array_equal(F_out, F)


def test_commit_without_prefetch_is_an_error_and_wait_without_transfers_is_not():
    w = small_random_state(32, 20, seed=5)
    g = make_gpu(w)
    g.wait_transfers()
    with pytest.raises(RuntimeError, match="no state was prefetched"):
        g.commit_state()
    g.prefetch_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
    g.commit_state()
    with pytest.raises(RuntimeError, match="no state was prefetched"):
        g.commit_state()
    E, F = g.get_state()
    assert np.array_equal(E, w["E"]) and np.array_equal(F, w["F"])


def test_transfers_follow_a_caller_stream():
    w = small_random_state(90, 70, seed=9, bc=(1, 2, 2, 1))
    dt = 4 * wl.explicit_dt(w["dx"], w["dy"], w["c"])
    ref = make_gpu(w)
    ref.step_implicit(dt, 1e-10, 30, 2000)
    E0, F0 = ref.get_state()
    import paper_2011_13926_b200 as ark
    st = torch.cuda.Stream()
    g = ark.ArkM1(w["nx"], w["ny"], w["dx"], w["dy"], w["c"], bc=w["bc"], stream=st)
    for side, gh in (w.get("ghosts") or {}).items():
        g.set_boundary(side, *gh)
    h = _pinned(w)
    out = (torch.empty((w["ny"], w["nx"]), dtype=torch.float64).pin_memory(), torch.empty((2, w["ny"], w["nx"]), dtype=torch.float64).pin_memory())
    g.prefetch_state(h["E"], h["F"], h["sigma_a"], h["sigma_s"])
    g.commit_state()
    g.step_implicit(dt, 1e-10, 30, 2000)
    g.get_state_async(out)
    g.wait_transfers()
    assert np.array_equal(out[0].numpy(), E0) and np.array_equal(out[1].numpy(), F0)
