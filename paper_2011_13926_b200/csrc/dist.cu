// dist.cu — domain-decomposed M1 step: 1-D slabs in y, one slab per rank (the paper's parallel design restated for NVLink
// GPUs: "regular domain decomposition with ghost cells"; rows of the linear system distributed over the ranks,
// PAPER.md:315; "the preconditioners and the linear solver require several communications per iteration").
//
// What is exchanged (byte counts in DESIGN.md section 8):
//   explicit step / assembly : the boundary rows of (E, Fx, Fy, sigma_a, sigma_t) -> the neighbour's ghost lines (5 nx doubles per side)
//   operator application     : (z, c^2 J z), z = M^-1 v, of the boundary rows (6 nx doubles per side), packed by a kernel
//   Gram-Schmidt             : one all-reduce of the j+1 dot products and one of ||w||^2 per iteration (fp64, <= 17 doubles)
// Everything else (closure, fluxes, assembly, block-Jacobi, updates, combination) is local to the slab and runs in the kernels
// of the one-GPU path, unchanged: a halo side is BC_HALO in the slab's Grid (m1_device.cuh).
//
// Transports behind one interface (Group::exchange / Group::allreduce):
//   LOCAL : all slabs live in this process on one GPU and one stream; exchange = device-to-device copies, all-reduce = a
//           kernel.  No kernel ever waits for another, so this is safe on a single GPU: it is how the decomposition is
//           tested against the one-slab result on the one-GPU test box, and it is what the driver loop below is written
//           for (every phase loops over the local slabs).
//   HOST  : one slab per process; halos and sums are staged through pinned host buffers and handed to callbacks supplied
//           by the caller (tests: torch.distributed/gloo).  Works between processes that share a GPU.
//   NCCL  : one slab per process and GPU; ncclSend/ncclRecv for the halos and ncclAllReduce for the sums, enqueued on the
//           solver's stream (no host round trip per iteration).  libnccl is opened with dlopen, so the library has no link
//           dependency on it.
// Supported configuration: GMRES(m) + block-Jacobi with the matrix-free operator and the marching kernels (the defaults).
#include <dlfcn.h>
#include <string.h>
#include <new>

#include "ark_m1_handle.h"

using namespace ark;

// ---- minimal NCCL declarations (ABI of nccl.h 2.x; resolved with dlsym) ------------------------------------------------------
typedef struct ncclComm* ncclComm_t;
typedef struct { char internal[128]; } ncclUniqueId;
enum { NCCL_SUCCESS = 0, NCCL_FLOAT64 = 8, NCCL_SUM = 0 };
struct NcclApi {
    void* lib;
    int (*GetUniqueId)(ncclUniqueId*);
    int (*CommInitRank)(ncclComm_t*, int, ncclUniqueId, int);
    int (*CommDestroy)(ncclComm_t);
    int (*AllReduce)(const void*, void*, size_t, int, int, ncclComm_t, cudaStream_t);
    int (*Send)(const void*, size_t, int, int, ncclComm_t, cudaStream_t);
    int (*Recv)(void*, size_t, int, int, ncclComm_t, cudaStream_t);
    int (*GroupStart)(void);
    int (*GroupEnd)(void);
    const char* (*GetErrorString)(int);
};

static int nccl_open(NcclApi* a, char* err, size_t nerr)
{
    memset(a, 0, sizeof *a);
    // a copy already in the process (torch's bundled libnccl.so.2) is reused; otherwise the system library
    a->lib = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
    if (!a->lib) a->lib = dlopen("libnccl.so", RTLD_NOW | RTLD_GLOBAL);
    if (!a->lib) { snprintf(err, nerr, "dlopen(libnccl.so.2): %s", dlerror()); return ARK_M1_E_UNSUPPORTED; }
#define ARK_SYM(field, name) *(void**)(&a->field) = dlsym(a->lib, name); if (!a->field) { snprintf(err, nerr, "dlsym(%s) failed", name); return ARK_M1_E_UNSUPPORTED; }
    ARK_SYM(GetUniqueId, "ncclGetUniqueId") ARK_SYM(CommInitRank, "ncclCommInitRank") ARK_SYM(CommDestroy, "ncclCommDestroy")
    ARK_SYM(AllReduce, "ncclAllReduce") ARK_SYM(Send, "ncclSend") ARK_SYM(Recv, "ncclRecv")
    ARK_SYM(GroupStart, "ncclGroupStart") ARK_SYM(GroupEnd, "ncclGroupEnd") ARK_SYM(GetErrorString, "ncclGetErrorString")
#undef ARK_SYM
    return 0;
}

enum { TR_LOCAL = 0, TR_HOST = 1, TR_NCCL = 2 };
enum { HALO_STATE_LINES = 5, HALO_ZP_LINES = 6, RED_CAP = 1024 };   // RED_CAP: doubles of the all-reduce buffer (restart + 1 sums at most)

struct Slab {
    ark_m1* h;
    int rank;            // global rank of this slab
    int y0, y1;          // global rows [y0, y1)
    int lo, hi;          // neighbour ranks below / above (-1: none, the side keeps the global boundary condition)
    double* send[2];     // device, 6 nx doubles each: what goes to lo / hi
    double* red;         // device, RED_CAP doubles: this slab's partial sums / the all-reduced sums
};

struct ark_m1_group {
    int nranks, transport, nx, ny;
    std::vector<Slab>* slabs;      // slabs held by this process (all of them for TR_LOCAL, one otherwise)
    cudaStream_t st;
    int device;
    ark_m1_host_transport host;
    double* hbuf;                  // pinned: [send_lo | send_hi | recv_lo | recv_hi] of 6 nx doubles each, then MAXV + 2 for the sums
    NcclApi nccl;
    ncclComm_t comm;
    double** red_ptrs;             // device array of the local slabs' `red` pointers (TR_LOCAL all-reduce kernel)
    long long halo_bytes, reduce_calls, exchange_calls;
    char err[512];
};

// ---- kernels --------------------------------------------------------------------------------------------------------------
// boundary rows of the state and opacity planes: out_lo <- row 0, out_hi <- row ny-1, lines E, Fx, Fy, sigma_a, sigma_t
__global__ void halo_pack_state_kernel(int nx, int ny, const double* __restrict__ U, const double* __restrict__ sa, const double* __restrict__ st,
                                       double* __restrict__ out_lo, double* __restrict__ out_hi)
{
    const long long N = (long long)nx * ny;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nx; i += gridDim.x * blockDim.x) {
        for (int side = 0; side < 2; ++side) {
            double* o = side == 0 ? out_lo : out_hi;
            if (!o) continue;
            const long long id = (long long)(side == 0 ? 0 : ny - 1) * nx + i;
            o[i] = U[id]; o[nx + i] = U[N + id]; o[2 * nx + i] = U[2 * N + id]; o[3 * nx + i] = sa[id]; o[4 * nx + i] = st[id];
        }
    }
}

// TR_LOCAL all-reduce: every slab's buffer receives the sum over the slabs, added in rank order (deterministic)
__global__ void sum_slabs_kernel(double** bufs, int nslab, int n)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    double s = 0.0;
    for (int r = 0; r < nslab; ++r) s += bufs[r][k];
    for (int r = 0; r < nslab; ++r) bufs[r][k] = s;
}

// ---- host -----------------------------------------------------------------------------------------------------------------
static int gfail(ark_m1_group* G, int code, const char* msg, const char* detail)
{
    if (G) snprintf(G->err, sizeof G->err, "%s%s%s", msg, detail ? ": " : "", detail ? detail : "");
    return code;
}
#define GCU(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return gfail(G, ARK_M1_E_CUDA, #call, cudaGetErrorString(e__)); } while (0)
#define GNC(call) do { int e__ = (call); if (e__ != NCCL_SUCCESS) return gfail(G, ARK_M1_E_CUDA, #call, G->nccl.GetErrorString(e__)); } while (0)
#define GRC(call) do { int rc__ = (call); if (rc__ < 0) return gfail(G, rc__, #call, ark_m1_last_error(s.h)); } while (0)

extern "C" int ark_m1_slab_range(int ny, int nranks, int rank, int* y0, int* y1)
{
    if (ny < 1 || nranks < 1 || rank < 0 || rank >= nranks || nranks > ny || !y0 || !y1) return ARK_M1_E_ARG;
    *y0 = (int)((long long)ny * rank / nranks);
    *y1 = (int)((long long)ny * (rank + 1) / nranks);
    return 0;
}

// Send `count` doubles of every slab's send[0] to its lower neighbour (which receives them as ITS upper halo) and send[1] to
// its upper neighbour; the receive buffers are the slabs' recv_state or recv_zp lines.
static int group_exchange(ark_m1_group* G, int which /*0: state lines, 1: zp lines*/, size_t count)
{
    std::vector<Slab>& S = *G->slabs;
    G->exchange_calls++;
    if (G->transport == TR_LOCAL) {
        for (Slab& s : S) {
            if (s.lo >= 0) { double* dst = which ? S[s.lo].h->halo_zp[1] : S[s.lo].h->halo_state[1]; GCU(cudaMemcpyAsync(dst, s.send[0], count * sizeof(double), cudaMemcpyDeviceToDevice, G->st)); G->halo_bytes += count * 8; }
            if (s.hi >= 0) { double* dst = which ? S[s.hi].h->halo_zp[0] : S[s.hi].h->halo_state[0]; GCU(cudaMemcpyAsync(dst, s.send[1], count * sizeof(double), cudaMemcpyDeviceToDevice, G->st)); G->halo_bytes += count * 8; }
        }
        return 0;
    }
    Slab& s = S[0];
    double* recv_lo = which ? s.h->halo_zp[0] : s.h->halo_state[0];
    double* recv_hi = which ? s.h->halo_zp[1] : s.h->halo_state[1];
    G->halo_bytes += (long long)count * 8 * ((s.lo >= 0) + (s.hi >= 0));
    if (G->transport == TR_NCCL) {
        // order: sends (to lo, to hi), then receives (from hi, from lo) — with two ranks and a periodic direction both
        // neighbours are the same peer, and NCCL pairs the operations on one peer in order
        GNC(G->nccl.GroupStart());
        if (s.lo >= 0) GNC(G->nccl.Send(s.send[0], count, NCCL_FLOAT64, s.lo, G->comm, G->st));
        if (s.hi >= 0) GNC(G->nccl.Send(s.send[1], count, NCCL_FLOAT64, s.hi, G->comm, G->st));
        if (s.hi >= 0) GNC(G->nccl.Recv(recv_hi, count, NCCL_FLOAT64, s.hi, G->comm, G->st));
        if (s.lo >= 0) GNC(G->nccl.Recv(recv_lo, count, NCCL_FLOAT64, s.lo, G->comm, G->st));
        GNC(G->nccl.GroupEnd());
        return 0;
    }
    // TR_HOST: stage through pinned memory and hand the buffers to the caller's transport
    const size_t L = (size_t)HALO_ZP_LINES * G->nx;
    double *hs_lo = G->hbuf, *hs_hi = G->hbuf + L, *hr_lo = G->hbuf + 2 * L, *hr_hi = G->hbuf + 3 * L;
    if (s.lo >= 0) GCU(cudaMemcpyAsync(hs_lo, s.send[0], count * sizeof(double), cudaMemcpyDeviceToHost, G->st));
    if (s.hi >= 0) GCU(cudaMemcpyAsync(hs_hi, s.send[1], count * sizeof(double), cudaMemcpyDeviceToHost, G->st));
    GCU(cudaStreamSynchronize(G->st));
    if (G->host.sendrecv(G->host.ctx, s.lo, s.hi, hs_lo, hs_hi, hr_lo, hr_hi, (long long)count) != 0) return gfail(G, ARK_M1_E_CUDA, "host transport: sendrecv failed", nullptr);
    if (s.lo >= 0) GCU(cudaMemcpyAsync(recv_lo, hr_lo, count * sizeof(double), cudaMemcpyHostToDevice, G->st));
    if (s.hi >= 0) GCU(cudaMemcpyAsync(recv_hi, hr_hi, count * sizeof(double), cudaMemcpyHostToDevice, G->st));
    return 0;
}

// Sum the first n doubles of every slab's `red` buffer over all ranks; every rank ends with the same sums.
static int group_allreduce(ark_m1_group* G, int n)
{
    std::vector<Slab>& S = *G->slabs;
    G->reduce_calls++;
    if (G->transport == TR_LOCAL) {
        sum_slabs_kernel<<<(n + 63) / 64, 64, 0, G->st>>>(G->red_ptrs, (int)S.size(), n);      // one thread per sum (a single block of 64 silently left sums 64.. unreduced)
        GCU(cudaGetLastError());
        return 0;
    }
    Slab& s = S[0];
    if (G->transport == TR_NCCL) {
        GNC(G->nccl.AllReduce(s.red, s.red, (size_t)n, NCCL_FLOAT64, NCCL_SUM, G->comm, G->st));
        return 0;
    }
    double* hr = G->hbuf + 4 * (size_t)HALO_ZP_LINES * G->nx;
    GCU(cudaMemcpyAsync(hr, s.red, n * sizeof(double), cudaMemcpyDeviceToHost, G->st));
    GCU(cudaStreamSynchronize(G->st));
    if (G->host.allreduce_sum(G->host.ctx, hr, n) != 0) return gfail(G, ARK_M1_E_CUDA, "host transport: allreduce failed", nullptr);
    GCU(cudaMemcpyAsync(s.red, hr, n * sizeof(double), cudaMemcpyHostToDevice, G->st));
    return 0;
}

static void group_free(ark_m1_group* G)
{
    if (!G) return;
    if (G->slabs) {
        for (Slab& s : *G->slabs) {
            if (s.h) {
                cudaStreamSynchronize(s.h->st);
                for (int k = 0; k < 2; ++k) { cudaFree(s.h->halo_state[k]); cudaFree(s.h->halo_zp[k]); s.h->halo_state[k] = s.h->halo_zp[k] = nullptr; cudaFree(s.send[k]); }
                cudaFree(s.red);
                ark_m1_destroy(s.h);
            }
        }
        delete G->slabs;
    }
    if (G->red_ptrs) cudaFree(G->red_ptrs);
    if (G->hbuf) cudaFreeHost(G->hbuf);
    if (G->comm && G->nccl.CommDestroy) G->nccl.CommDestroy(G->comm);
    cudaGetLastError();
    delete G;
}

static ark_m1_group* group_create(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc, int transport, int rank, int nranks,
                                  const ark_m1_host_transport* ht, const void* nccl_id)
{
    if (nx < 1 || ny < 1 || nranks < 1 || nranks > ny || rank < 0 || rank >= nranks) return nullptr;
    ark_m1_bc gb = { 0, 0, 0, 0 };
    if (bc) gb = *bc;
    const int kinds[4] = { gb.xlo, gb.xhi, gb.ylo, gb.yhi };
    for (int k = 0; k < 4; ++k) if (kinds[k] < BC_PERIODIC || kinds[k] > BC_OUTFLOW) return nullptr;
    if ((gb.xlo == BC_PERIODIC) != (gb.xhi == BC_PERIODIC) || (gb.ylo == BC_PERIODIC) != (gb.yhi == BC_PERIODIC)) return nullptr;   // periodic comes in pairs
    ark_m1_group* G = new (std::nothrow) ark_m1_group;
    if (!G) return nullptr;
    memset(G, 0, sizeof *G);
    G->nranks = nranks; G->transport = transport; G->nx = nx; G->ny = ny;
    G->slabs = new std::vector<Slab>();
    if (ht) G->host = *ht;
    cudaGetDevice(&G->device);
    const bool yper = (gb.ylo == BC_PERIODIC);
    const int first = (transport == TR_LOCAL) ? 0 : rank, last = (transport == TR_LOCAL) ? nranks : rank + 1;
    bool ok = true;
    for (int r = first; r < last && ok; ++r) {
        Slab s; memset(&s, 0, sizeof s);
        s.rank = r;
        ark_m1_slab_range(ny, nranks, r, &s.y0, &s.y1);
        s.lo = (r > 0) ? r - 1 : ((yper && nranks > 1) ? nranks - 1 : -1);
        s.hi = (r < nranks - 1) ? r + 1 : ((yper && nranks > 1) ? 0 : -1);
        ark_m1_bc lb = gb;
        // a periodic direction cut into slabs is no longer periodic for the slab; pair the kinds for ark_m1_create and set the
        // halo sides afterwards
        if (nranks > 1) { lb.ylo = (s.lo >= 0 || yper) ? BC_OUTFLOW : gb.ylo; lb.yhi = (s.hi >= 0 || yper) ? BC_OUTFLOW : gb.yhi; }
        s.h = ark_m1_create(nx, s.y1 - s.y0, dx, dy, c, &lb);
        ok = (s.h != nullptr);
        if (ok) {
            if (s.lo >= 0) s.h->g.bc[YLO] = BC_HALO;
            if (s.hi >= 0) s.h->g.bc[YHI] = BC_HALO;
            s.h->in_group = 1;
            for (int k = 0; k < 2 && ok; ++k) {
                ok = cudaMalloc((void**)&s.h->halo_state[k], sizeof(double) * HALO_ZP_LINES * nx) == cudaSuccess
                  && cudaMalloc((void**)&s.h->halo_zp[k], sizeof(double) * HALO_ZP_LINES * nx) == cudaSuccess
                  && cudaMalloc((void**)&s.send[k], sizeof(double) * HALO_ZP_LINES * nx) == cudaSuccess;
                if (ok) { cudaMemset(s.h->halo_state[k], 0, sizeof(double) * HALO_ZP_LINES * nx); cudaMemset(s.h->halo_zp[k], 0, sizeof(double) * HALO_ZP_LINES * nx); }
            }
            ok = ok && cudaMalloc((void**)&s.red, sizeof(double) * RED_CAP) == cudaSuccess;
        }
        G->slabs->push_back(s);
    }
    if (ok && transport == TR_LOCAL) {
        std::vector<double*> p;
        for (Slab& s : *G->slabs) p.push_back(s.red);
        ok = cudaMalloc((void**)&G->red_ptrs, sizeof(double*) * p.size()) == cudaSuccess
          && cudaMemcpy(G->red_ptrs, p.data(), sizeof(double*) * p.size(), cudaMemcpyHostToDevice) == cudaSuccess;
    }
    if (ok && transport == TR_HOST)
        ok = ht && ht->sendrecv && ht->allreduce_sum
          && cudaMallocHost((void**)&G->hbuf, sizeof(double) * (4 * (size_t)HALO_ZP_LINES * nx + RED_CAP)) == cudaSuccess;
    if (ok && transport == TR_NCCL) {
        ok = nccl_id && nccl_open(&G->nccl, G->err, sizeof G->err) == 0;
        if (ok) {
            ncclUniqueId id; memcpy(&id, nccl_id, sizeof id);
            ok = G->nccl.CommInitRank(&G->comm, nranks, id, rank) == NCCL_SUCCESS;
        }
    }
    if (!ok) { cudaGetLastError(); group_free(G); return nullptr; }
    return G;
}

extern "C" {

ark_m1_group* ark_m1_group_create_local(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc, int nranks)
{
    return group_create(nx, ny, dx, dy, c, bc, TR_LOCAL, 0, nranks, nullptr, nullptr);
}

ark_m1_group* ark_m1_group_create_host(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc, int rank, int nranks,
                                       const ark_m1_host_transport* transport)
{
    return group_create(nx, ny, dx, dy, c, bc, TR_HOST, rank, nranks, transport, nullptr);
}

int ark_m1_nccl_unique_id(void* out128)
{
    if (!out128) return ARK_M1_E_ARG;
    NcclApi a; char err[256];
    int rc = nccl_open(&a, err, sizeof err);
    if (rc) return rc;
    ncclUniqueId id;
    if (a.GetUniqueId(&id) != NCCL_SUCCESS) return ARK_M1_E_CUDA;
    memcpy(out128, &id, sizeof id);
    return 0;
}

ark_m1_group* ark_m1_group_create_nccl(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc, int rank, int nranks,
                                       const void* unique_id128)
{
    return group_create(nx, ny, dx, dy, c, bc, TR_NCCL, rank, nranks, nullptr, unique_id128);
}

void ark_m1_group_destroy(ark_m1_group* G) { group_free(G); }

int ark_m1_group_local_slabs(const ark_m1_group* G) { return G ? (int)G->slabs->size() : 0; }

ark_m1* ark_m1_group_slab(ark_m1_group* G, int k, int* rank, int* y0, int* y1)
{
    if (!G || k < 0 || k >= (int)G->slabs->size()) return nullptr;
    const Slab& s = (*G->slabs)[k];
    if (rank) *rank = s.rank;
    if (y0) *y0 = s.y0;
    if (y1) *y1 = s.y1;
    return s.h;
}

int ark_m1_group_set_stream(ark_m1_group* G, void* cuda_stream)
{
    if (!G) return ARK_M1_E_ARG;
    G->st = (cudaStream_t)cuda_stream;
    for (Slab& s : *G->slabs) { int rc = ark_m1_set_stream(s.h, cuda_stream); if (rc) return rc; }
    return 0;
}

const char* ark_m1_group_last_error(const ark_m1_group* G) { return G ? G->err : "null group"; }

int ark_m1_group_comm_stats(const ark_m1_group* G, long long* halo_bytes, long long* exchanges, long long* allreduces)
{
    if (!G) return ARK_M1_E_ARG;
    if (halo_bytes) *halo_bytes = G->halo_bytes;
    if (exchanges) *exchanges = G->exchange_calls;
    if (allreduces) *allreduces = G->reduce_calls;
    return 0;
}

}  // extern "C"

// ghost lines of every slab <- boundary rows of the neighbours' current state and opacities
static int refresh_state_halos(ark_m1_group* G)
{
    for (Slab& s : *G->slabs) {
        ark_m1* h = s.h;
        if (!h->have_state) return gfail(G, ARK_M1_E_NOTSET, "a slab has no state", nullptr);
        const int blk = 128, grd = (G->nx + blk - 1) / blk;
        halo_pack_state_kernel<<<grd, blk, 0, G->st>>>(h->g.nx, h->g.ny, h->U[h->cur], h->sa, h->stot, s.lo >= 0 ? s.send[0] : nullptr, s.hi >= 0 ? s.send[1] : nullptr);
        GCU(cudaGetLastError());
        h->launches++;
    }
    return group_exchange(G, 0, (size_t)HALO_STATE_LINES * G->nx);
}

static int check_supported(ark_m1_group* G, bool implicit)
{
    for (Slab& s : *G->slabs) {
        ark_m1* h = s.h;
        if (h->N >= (1LL << 31)) return gfail(G, ARK_M1_E_UNSUPPORTED, "slab too large for the marching kernels", nullptr);
        if (implicit && (h->krylov != 0 || h->precond != 0 || h->op_kind != 1 || h->asm_kernel != 1 || h->ortho != 1 || h->basis_prec != 64))
            return gfail(G, ARK_M1_E_UNSUPPORTED, "the decomposed implicit step supports GMRES + block-Jacobi with the matrix-free operator, marching assembly, one-pass CGS and the fp64 basis (the defaults)", nullptr);
    }
    return 0;
}

extern "C" int ark_m1_group_step_explicit(ark_m1_group* G, double dt)
{
    if (!G) return ARK_M1_E_ARG;
    if (!(dt > 0.0)) return gfail(G, ARK_M1_E_ARG, "step_explicit: dt must be > 0", nullptr);
    DeviceGuard guard(G->device);
    int rc = check_supported(G, false);
    if (rc) return rc;
    if ((rc = refresh_state_halos(G))) return rc;
    for (Slab& s : *G->slabs) GRC(ark_explicit_once(s.h, dt));
    return 0;
}

// w_out = sgn * scale * A [M^-1] v + add on every slab, after the halo exchange of (z, c^2 J z)
static int group_operator(ark_m1_group* G, size_t v_off, bool v_is_x, size_t out_off, int scale_idx, bool add_b, double sgn,
                          bool use_stop, int precond, double theta = 0.0)
{
    for (Slab& s : *G->slabs) {
        ark_m1* h = s.h;
        const double* v = v_is_x ? h->U[h->cur] : h->V + v_off * h->stride;
        const int* stop = use_stop ? &h->W.ctl->inner_stop : nullptr;
        h->launches++;
        GCU(launch_halo_pack_zp(h->g, h->mf, h->A.Minv, v, precond, s.lo >= 0 ? s.send[0] : nullptr, s.hi >= 0 ? s.send[1] : nullptr, stop, G->st));
    }
    int rc = group_exchange(G, 1, (size_t)HALO_ZP_LINES * G->nx);
    if (rc) return rc;
    for (Slab& s : *G->slabs) {
        ark_m1* h = s.h;
        const double* v = v_is_x ? h->U[h->cur] : h->V + v_off * h->stride;
        const int* stop = use_stop ? &h->W.ctl->inner_stop : nullptr;
        ark_kmark(h, KC_SPMV, (precond ? (h->mf.rc ? (h->mf.rcj ? 136.0 : 192.0) : 264.0) : 216.0) * h->N);
        GCU(launch_op_mf(h->g, h->mf, h->A.Minv, v, h->V + out_off * h->stride, scale_idx >= 0 ? h->W.scale + scale_idx : nullptr,
                         add_b ? h->A.b : nullptr, sgn, stop, precond, h->sm_count, G->st, theta));
    }
    return 0;
}

// one all-reduce of n sums followed by the s-step epilogue `which` on every slab (krylov_sstep.cu)
static int group_sstep_epilogue(ark_m1_group* G, int n, int which, int sb, int nv, int round)
{
    int rc = group_allreduce(G, n);
    if (rc) return rc;
    for (Slab& s : *G->slabs) {
        s.h->launches++;
        GCU(launch_sstep_epilogue(s.h->W, which, sb, nv, s.red, 1.0, round, G->st));
    }
    return 0;
}

// all-reduce the first n sums of every slab and run the scalar epilogue `mode` on each slab's (replicated) solver state
static int group_reduce_epilogue(ark_m1_group* G, int n, int mode, int nv, int col0, int red_off, bool use_stop)
{
    int rc = group_allreduce(G, n);
    if (rc) return rc;
    for (Slab& s : *G->slabs) {
        ark_m1* h = s.h;
        h->launches++;
        GCU(launch_epilogue(h->W, mode, nv, col0, s.red + red_off, use_stop ? &h->W.ctl->inner_stop : nullptr, G->st));
    }
    return 0;
}

static int group_true_residual(ark_m1_group* G)
{
    int rc = group_operator(G, 0, true, 0, -1, true, -1.0, false, 0);       // V0 <- b - A x
    if (rc) return rc;
    for (Slab& s : *G->slabs) {
        ark_m1* h = s.h;
        GmresWork W = h->W; W.red_out = s.red;
        ark_kmark(h, KC_DOT, 24.0 * h->N);
        GCU(launch_multi_dot(h->V, h->V, h->stride, 1, 0, 3 * h->N, W, DOT_RNORM, h->sm_count, G->st));
    }
    return group_reduce_epilogue(G, 1, DOT_RNORM, 1, 0, 0, false);
}

static int group_fetch_ctl(ark_m1_group* G)
{
    for (Slab& s : *G->slabs) GCU(cudaMemcpyAsync(s.h->ctl_host, s.h->W.ctl, sizeof(GmresCtl), cudaMemcpyDeviceToHost, G->st));
    GCU(cudaStreamSynchronize(G->st));
    return 0;
}

extern "C" int ark_m1_group_step_implicit(ark_m1_group* G, double dt, double tol, int restart, int maxit, double* final_residual)
{
    if (!G) return ARK_M1_E_ARG;
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0) return gfail(G, ARK_M1_E_ARG, "step_implicit: need dt > 0, tol > 0, restart >= 1, maxit >= 0", nullptr);
    DeviceGuard guard(G->device);
    std::vector<Slab>& S = *G->slabs;
    int rc = check_supported(G, true);
    if (rc) return rc;
    if (restart + 1 > RED_CAP) return gfail(G, ARK_M1_E_UNSUPPORTED, "step_implicit: restart too long for the all-reduce buffer", nullptr);
    const int m = restart;
    for (Slab& s : S) { GRC(ark_ensure_implicit(s.h, m, maxit)); s.h->mf.halo[0] = s.h->halo_zp[0]; s.h->mf.halo[1] = s.h->halo_zp[1]; }
    if ((rc = refresh_state_halos(G))) return rc;
    for (Slab& s : S) { GCU(cudaEventRecord(s.h->ev[0], G->st)); GRC(ark_assemble_system(s.h, dt, nullptr)); GCU(cudaEventRecord(s.h->ev[1], G->st)); }
    // ---- GMRES(m), right-preconditioned with block-Jacobi: the loop of gmres_solve (ark_m1_api.cu) with every reduction split
    //      into local sums -> all-reduce -> epilogue, and a halo exchange in front of every operator application
    for (Slab& s : S) {
        ark_m1* h = s.h;
        ark_kmark(h, KC_SMALL, 0.0);
        GCU(launch_begin_solve(h->W, tol, m, maxit, G->st));
        GmresWork W = h->W; W.red_out = s.red;
        ark_kmark(h, KC_DOT, 24.0 * h->N);
        GCU(launch_multi_dot(h->A.b, h->A.b, 0, 1, 0, 3 * h->N, W, DOT_BNORM, h->sm_count, G->st));
    }
    if ((rc = group_reduce_epilogue(G, 1, DOT_BNORM, 1, 0, 0, false))) return rc;
    if ((rc = group_true_residual(G))) return rc;
    if ((rc = group_fetch_ctl(G))) return rc;
    const int MV = S[0].h->maxv;
    // s-step Arnoldi blocks (krylov_sstep.cu), as in the one-GPU solver: per block of SB columns SB halo exchanges (one per operator
    // application) and FIVE all-reduces (dots, Gram matrix, norms, and the two of the refinement round, whose kernels return at once
    // for a well-conditioned block) instead of 2 SB with one column per pass.  Columns a restart length leaves over use the one-column step.
    const int SB = (S[0].h->arnoldi_block >= 3 && m <= 120 && SMAX * (m + 1) <= RED_CAP) ? S[0].h->arnoldi_block : 0;
    while (!S[0].h->ctl_host->inner_stop) {
        for (int j = 0; j < m; ++j) {
            if (SB && j + SB <= m) {
                for (int k = 0; k < SB; ++k)
                    if ((rc = group_operator(G, (size_t)(j + k), false, (size_t)(j + k + 1), k == 0 ? j : -1, false, 1.0, true, 1, k == 0 ? 0.0 : 1.0))) return rc;
                const int ld = m + 1;
                for (Slab& s : S) {
                    ark_m1* h = s.h;
                    double* w = h->V + (size_t)(j + 1) * h->stride;
                    GmresWork W = h->W; W.red_out = s.red;
                    // the block's own slots are dotted like basis vectors (W^T W): the in-block solve is predicted from the reduced sums
                    const int nd = j + 1 + SB;
                    for (int c0 = 0; c0 < nd; c0 += 32) {
                        const int nv = (nd - c0) < 32 ? (nd - c0) : 32, nbasis = (j + 1 - c0) < 0 ? 0 : ((j + 1 - c0) < nv ? (j + 1 - c0) : nv);
                        ark_kmark(h, KC_DOT, 24.0 * (nbasis + SB) * h->N);
                        GCU(launch_dotS(w, h->V + (size_t)c0 * h->stride, h->stride, SB, nv, c0, 3 * h->N, W, h->sm_count, G->st, j));
                    }
                }
                if ((rc = group_sstep_epilogue(G, SB * ld, 0, SB, j + 1 + SB, 1))) return rc;
                for (Slab& s : S) {
                    ark_m1* h = s.h;
                    GmresWork W = h->W; W.red_out = s.red;
                    ark_kmark(h, KC_UPDATE, (24.0 * (j + 1) + 48.0 * SB) * h->N);
                    GCU(launch_updateS(h->V + (size_t)(j + 1) * h->stride, h->V, h->stride, SB, j + 1, 3 * h->N, W, h->sm_count, G->st));
                }
                if ((rc = group_sstep_epilogue(G, SB * (SB + 1) / 2, 1, SB, j + 1, 0))) return rc;
                for (int round = 1; round <= 2; ++round) {
                    if (round == 2) {
                        for (Slab& s : S) {
                            ark_m1* h = s.h;
                            GmresWork W = h->W; W.red_out = s.red;
                            ark_kmark(h, KC_SMALL, 0.0);
                            GCU(launch_gramS(h->V + (size_t)(j + 1) * h->stride, h->stride, SB, 3 * h->N, W, h->sm_count, G->st));
                        }
                        if ((rc = group_sstep_epilogue(G, SB * (SB + 1) / 2, 3, SB, j + 1, 2))) return rc;
                    }
                    for (Slab& s : S) {
                        ark_m1* h = s.h;
                        GmresWork W = h->W; W.red_out = s.red;
                        ark_kmark(h, KC_SMALL, 0.0);      // a pass of its own only for a block whose predicted solve was not used
                        GCU(launch_qrS(h->V + (size_t)(j + 1) * h->stride, h->stride, SB, 3 * h->N, W, 1.0, round, h->sm_count, G->st));
                    }
                    if ((rc = group_sstep_epilogue(G, SB - 1, 2, SB, j + 1, round))) return rc;
                }
                j += SB - 1;
                continue;
            }
            if ((rc = group_operator(G, (size_t)j, false, (size_t)j + 1, j, false, 1.0, true, 1))) return rc;
            const int nchunk = (j + MV) / MV, csize = (j + nchunk) / nchunk;
            for (Slab& s : S) {
                ark_m1* h = s.h;
                double* w = h->V + (size_t)(j + 1) * h->stride;
                for (int c0 = 0; c0 <= j; c0 += csize) {
                    const int nv = (j + 1 - c0) < csize ? (j + 1 - c0) : csize;
                    GmresWork W = h->W; W.red_out = s.red + c0;
                    ark_kmark(h, KC_DOT, 24.0 * (nv + 1) * h->N);
                    GCU(launch_multi_dot(w, h->V + (size_t)c0 * h->stride, h->stride, nv, c0, 3 * h->N, W, DOT_H, h->sm_count, G->st));
                }
            }
            if ((rc = group_allreduce(G, j + 1))) return rc;
            for (Slab& s : S) {
                ark_m1* h = s.h;
                double* w = h->V + (size_t)(j + 1) * h->stride;
                for (int c0 = 0; c0 <= j; c0 += csize) {
                    const int nv = (j + 1 - c0) < csize ? (j + 1 - c0) : csize;
                    h->launches++;
                    GCU(launch_epilogue(h->W, DOT_H, nv, c0, s.red + c0, &h->W.ctl->inner_stop, G->st));
                }
                for (int c0 = 0; c0 <= j; c0 += csize) {
                    const int nv = (j + 1 - c0) < csize ? (j + 1 - c0) : csize;
                    const int last = (c0 + csize > j);
                    GmresWork W = h->W; W.red_out = s.red;
                    ark_kmark(h, KC_UPDATE, 24.0 * (nv + 2) * h->N);
                    GCU(launch_update(w, h->V + (size_t)c0 * h->stride, h->stride, nv, c0, 3 * h->N, W, last, h->sm_count, G->st));
                }
            }
            if ((rc = group_reduce_epilogue(G, 1, DOT_UPD, 1, 0, 0, true))) return rc;
        }
        for (Slab& s : S) {
            ark_m1* h = s.h;
            ark_kmark(h, KC_SMALL, 0.0);
            GCU(launch_solve_y(h->W, G->st));
            ark_kmark(h, KC_COMBINE, 8.0 * (3.0 * m + 15.0) * h->N);
            GCU(launch_combine(h->g, h->V, h->stride, h->A.Minv, h->U[h->cur], h->W, h->sm_count, G->st));
        }
        if ((rc = group_true_residual(G))) return rc;
        if ((rc = group_fetch_ctl(G))) return rc;
    }
    int its = 0;
    for (Slab& s : S) {
        GCU(cudaEventRecord(s.h->ev[2], G->st));
        double res = 0.0;
        GRC(ark_finish_implicit(s.h, dt, &res));
        if (final_residual) *final_residual = res;
        its = s.h->ctl_host->its;
    }
    return its;
}
