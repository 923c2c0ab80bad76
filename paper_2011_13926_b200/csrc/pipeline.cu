// pipeline.cu — state transfers that overlap the solver (include/ark_m1.h "Overlapped transfers").
//
// A caller that steps many states from HOST buffers pays, with ark_m1_set_state / ark_m1_get_state, the upload of the next state
// and the download of the last result in series with the solve: 671 MB up and 403 MB down per 4096^2 step, 13-14 ms of a 94 ms step.
// Neither copy depends on the solve that runs beside it, so they go to a copy stream of the handle's own:
//   ark_m1_prefetch_state   host (or device) arrays -> a staging buffer [E | Fx | Fy | sigma_a | sigma_s], on the copy stream;
//   ark_m1_commit_state     the handle's stream waits for that upload and takes the staged state (device copies, 0.5 ms);
//   ark_m1_get_state_async  the handle's stream snapshots the current state (device copy, 0.3 ms), the copy stream takes the
//                           snapshot to the caller's arrays while the handle's stream goes on with the next step;
//   ark_m1_wait_transfers   the host waits until both directions are done (the caller's arrays are then its own again).
// Ordering is by events only: a new upload waits for the commit of the previous one to have read the staging buffer, a new
// snapshot waits for the previous download to have left the snapshot buffer.  Costs 8 planes of device memory, allocated at the
// first call.  Nothing here changes the arithmetic: the staged state is what ark_m1_set_state would have been given.
#include <new>
#include <string.h>

#include "ark_m1_handle.h"

struct ArkPipe {
    cudaStream_t cs;
    double* stage;           // 5N: E | Fx | Fy | sigma_a | sigma_s
    double* snap;            // 3N: E | Fx | Fy
    cudaEvent_t up, committed, snapped, down;
    bool up_pending, committed_once, down_pending;
};

void ark_pipe_free(ark_m1* h);

static int pipe_init(ark_m1* h, ArkPipe* p)
{
    const size_t B = (size_t)h->N * sizeof(double);
    int rc;
    if ((rc = ark_dmalloc(h, (void**)&p->stage, 5 * B))) return rc;
    if ((rc = ark_dmalloc(h, (void**)&p->snap, 3 * B))) return rc;
    CU(cudaStreamCreateWithFlags(&p->cs, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&p->up, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&p->committed, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&p->snapped, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&p->down, cudaEventDisableTiming));
    return 0;
}

static int pipe_of(ark_m1* h, ArkPipe** out)
{
    if (h->pipe) { *out = (ArkPipe*)h->pipe; return 0; }
    ArkPipe* p = new (std::nothrow) ArkPipe;
    if (!p) return ark_fail(h, ARK_M1_E_ALLOC, "overlapped transfers: out of host memory%s", "");
    memset(p, 0, sizeof *p);
    h->pipe = p;
    const int rc = pipe_init(h, p);
    if (rc) { ark_pipe_free(h); return rc; }      // (the message of the failed call stays in the handle)
    *out = p;
    return 0;
}

void ark_pipe_free(ark_m1* h)
{
    ArkPipe* p = (ArkPipe*)h->pipe;
    if (!p) return;
    if (p->cs) { cudaStreamSynchronize(p->cs); cudaStreamDestroy(p->cs); }
    if (p->up) cudaEventDestroy(p->up);
    if (p->committed) cudaEventDestroy(p->committed);
    if (p->snapped) cudaEventDestroy(p->snapped);
    if (p->down) cudaEventDestroy(p->down);
    ark_dfree(h, p->stage); ark_dfree(h, p->snap);
    delete p;
    h->pipe = nullptr;
}

extern "C" {

int ark_m1_prefetch_state(ark_m1* h, const double* E, const double* F, const double* sigma_a, const double* sigma_s)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    if (!E || !F || !sigma_a || !sigma_s) return ark_fail(h, ARK_M1_E_ARG, "prefetch_state: NULL array%s", "");
    if (h->in_group) return ark_fail(h, ARK_M1_E_UNSUPPORTED, "prefetch_state: this handle is a slab of an ark_m1_group%s", "");
    ArkPipe* p;
    int rc = pipe_of(h, &p);
    if (rc) return rc;
    const size_t N = (size_t)h->N, B = N * sizeof(double);
    if (p->committed_once) CU(cudaStreamWaitEvent(p->cs, p->committed, 0));      // the last commit has read the staging buffer
    CU(cudaMemcpyAsync(p->stage, E, B, cudaMemcpyDefault, p->cs));
    CU(cudaMemcpyAsync(p->stage + N, F, 2 * B, cudaMemcpyDefault, p->cs));
    CU(cudaMemcpyAsync(p->stage + 3 * N, sigma_a, B, cudaMemcpyDefault, p->cs));
    CU(cudaMemcpyAsync(p->stage + 4 * N, sigma_s, B, cudaMemcpyDefault, p->cs));
    CU(cudaEventRecord(p->up, p->cs));
    p->up_pending = true;
    return 0;
}

int ark_m1_commit_state(ark_m1* h)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    ArkPipe* p = (ArkPipe*)h->pipe;
    if (!p || !p->up_pending) return ark_fail(h, ARK_M1_E_NOTSET, "commit_state: no state was prefetched%s", "");
    const size_t N = (size_t)h->N;
    CU(cudaStreamWaitEvent(h->st, p->up, 0));
    const int rc = ark_m1_set_state(h, p->stage, p->stage + N, p->stage + 3 * N, p->stage + 4 * N, nullptr);
    if (rc) return rc;
    CU(cudaEventRecord(p->committed, h->st));
    p->committed_once = true;
    p->up_pending = false;
    return 0;
}

int ark_m1_get_state_async(ark_m1* h, double* E, double* F)
{
    if (!h || !E || !F) return ARK_M1_E_ARG;
    GUARD(h);
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "get_state_async: no state set%s", "");
    ArkPipe* p;
    int rc = pipe_of(h, &p);
    if (rc) return rc;
    const size_t N = (size_t)h->N, B = N * sizeof(double);
    if (p->down_pending) CU(cudaStreamWaitEvent(h->st, p->down, 0));              // the last download has left the snapshot buffer
    CU(cudaMemcpyAsync(p->snap, h->U[h->cur], 3 * B, cudaMemcpyDeviceToDevice, h->st));
    CU(cudaEventRecord(p->snapped, h->st));
    CU(cudaStreamWaitEvent(p->cs, p->snapped, 0));
    CU(cudaMemcpyAsync(E, p->snap, B, cudaMemcpyDefault, p->cs));
    CU(cudaMemcpyAsync(F, p->snap + N, 2 * B, cudaMemcpyDefault, p->cs));
    CU(cudaEventRecord(p->down, p->cs));
    p->down_pending = true;
    return 0;
}

int ark_m1_wait_transfers(ark_m1* h)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    ArkPipe* p = (ArkPipe*)h->pipe;
    if (!p) return 0;
    CU(cudaStreamSynchronize(p->cs));
    p->down_pending = false;
    return 0;
}

}  // extern "C"
