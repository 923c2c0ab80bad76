"""GPU test of the entry point that allocates nothing: ark_m1_count_unrealizable_noalloc (scratch in a static __device__ array,
include/ark_m1.h) against the existing handle path ark_m1_count_unrealizable, and against the oracle's count, on calls in a row.

Integer work: the bar is bit-exact.  The file name sorts last on purpose (pytest -x: a failure here hides no
other test); the test must pass alone in a fresh process and after every other test."""
import numpy as np
import pytest

from helpers import make_gpu, make_oracle, small_random_state

pytestmark = pytest.mark.gpu


def _state(nx, ny, seed):
    # |F| > cE in many cells (fmax = 1.7), a few cells with E <= 0, c != 1
    w = small_random_state(nx, ny, seed=seed, fmax=1.7, c=1.3)
    rng = np.random.default_rng(seed + 1)
    bad = rng.integers(0, nx * ny, size=max(3, nx * ny // 97))
    w["E"].reshape(-1)[bad[::2]] = 0.0
    w["E"].reshape(-1)[bad[1::2]] = -w["E"].reshape(-1)[bad[1::2]]
    return w


def _noalloc_counts(w, out, stream=None):
    import torch
    import paper_2011_13926_b200 as ark
    E = torch.from_numpy(np.ascontiguousarray(w["E"])).cuda()
    F = torch.from_numpy(np.ascontiguousarray(w["F"])).cuda()
    torch.cuda.synchronize()      # the inputs are in place whatever stream the call is given
    ark.count_unrealizable_noalloc(E, F[0], F[1], w["c"], out, stream=stream)
    (torch.cuda.current_stream() if stream is None else stream).synchronize()
    return tuple(int(v) for v in out.cpu())


def test_noalloc_counts_equal_the_handle_path_on_calls_in_a_row():
    import torch
    import paper_2011_13926_b200 as ark
    ark.noalloc_setup()
    out = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    # 16 blocks with a ragged tail, then 2 blocks (the scratch still holds 14 stale pairs of the first call), then 40 blocks,
    # then one block of fewer cells than threads
    for nx, ny, seed in ((301, 211, 3), (97, 61, 4), (640, 255, 5), (13, 7, 6)):
        w = _state(nx, ny, seed)
        want = make_gpu(w).count_unrealizable()
        assert want == make_oracle(w).count_unrealizable()
        assert want[0] > 0 and want[1] > 0
        out.fill_(-1)
        assert _noalloc_counts(w, out) == want
    # the same input twice in a row gives the same answer
    assert _noalloc_counts(w, out) == want


def test_noalloc_on_a_side_stream_and_empty_input():
    import torch
    import paper_2011_13926_b200 as ark
    out = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    st = torch.cuda.Stream()
    w = _state(257, 129, 11)
    want = make_gpu(w).count_unrealizable()
    torch.cuda.synchronize()
    assert _noalloc_counts(w, out, stream=st) == want
    empty = torch.empty(0, dtype=torch.float64, device="cuda")
    out.fill_(-1)
    ark.count_unrealizable_noalloc(empty, empty, empty, 1.0, out)
    torch.cuda.synchronize()
    assert out.tolist() == [0, 0]


def test_noalloc_allocates_nothing_and_rejects_sizes_beyond_the_scratch():
    import ctypes as C
    import torch
    import paper_2011_13926_b200 as ark
    L = ark.load_library()
    ark.noalloc_setup()
    w = _state(512, 300, 21)
    E = torch.from_numpy(np.ascontiguousarray(w["E"])).cuda()
    F = torch.from_numpy(np.ascontiguousarray(w["F"])).cuda()
    out = torch.zeros(2, dtype=torch.int64, device="cuda")
    ark.count_unrealizable_noalloc(E, F[0], F[1], w["c"], out)      # first launch: the driver may load the kernel lazily
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        ark.count_unrealizable_noalloc(E, F[0], F[1], w["c"], out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "device memory in use changed across calls of the no-allocation entry point"
    # one cell beyond the maximum: refused with a message that names the limit, nothing launched, the output untouched
    nmax = ark.noalloc_max_cells()
    assert nmax == 16384 * 4096
    out.fill_(-7)
    rc = L.ark_m1_count_unrealizable_noalloc(E.data_ptr(), F[0].data_ptr(), F[1].data_ptr(), C.c_longlong(nmax + 1), 1.0, out.data_ptr(), None)
    assert rc == -6
    msg = L.ark_m1_noalloc_last_error().decode()
    assert str(nmax) in msg and str(nmax + 1) in msg
    torch.cuda.synchronize()
    assert out.tolist() == [-7, -7]
    assert L.ark_m1_count_unrealizable_noalloc(None, None, None, C.c_longlong(5), 1.0, out.data_ptr(), None) == -1
    assert L.ark_m1_count_unrealizable_noalloc(E.data_ptr(), F[0].data_ptr(), F[1].data_ptr(), C.c_longlong(-1), 1.0, out.data_ptr(), None) == -1


def test_noalloc_at_the_maximum_size():
    # every one of the 16 384 partial pairs in use; expected counts from torch's own comparison of the same arithmetic
    import torch
    import paper_2011_13926_b200 as ark
    n = ark.noalloc_max_cells()
    g = torch.Generator(device="cuda").manual_seed(17)
    E = torch.randn(n, dtype=torch.float64, device="cuda", generator=g) + 0.5
    Fx = torch.randn(n, dtype=torch.float64, device="cuda", generator=g)
    Fy = torch.randn(n, dtype=torch.float64, device="cuda", generator=g)
    c = 1.3
    pos = E > 0.0
    want = (int((~pos).sum()), int((pos & (torch.sqrt(Fx * Fx + Fy * Fy) > c * E)).sum()))
    out = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    for _ in range(2):
        out.fill_(-1)
        ark.count_unrealizable_noalloc(E, Fx, Fy, c, out)
        torch.cuda.synchronize()
        assert tuple(out.tolist()) == want
