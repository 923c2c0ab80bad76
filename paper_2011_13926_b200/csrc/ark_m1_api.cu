// ark_m1_api.cu — the C ABI of include/ark_m1.h: handle, device memory, step drivers.
// Host logic only; every arithmetic step of the path runs in the kernels of this directory.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <map>
#include <vector>

#include "ark_m1_handle.h"

using namespace ark;

// The handle lives on the device that was current at ark_m1_create.  Every entry point makes that device current for its
// duration and restores the caller's (a multi-GPU process may have switched devices in between).
DeviceGuard::DeviceGuard(int dev) : prev(-1), switched(false)
{
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
}
DeviceGuard::~DeviceGuard() { if (switched) cudaSetDevice(prev); }

namespace ark {
int current_sm_count()
{
    static int cached[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    if (cached[dev] == 0) { int n = 0; cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev); cached[dev] = n > 0 ? n : 148; }
    return cached[dev];
}
}  // namespace ark

int ark_fail(ark_m1* h, int code, const char* fmt, const char* detail)
{
    if (h) snprintf(h->err, sizeof h->err, fmt, detail ? detail : "");
    return code;
}

// Record the start of a launch of class `cls` moving `bytes` algorithmic bytes (only when kernel timing is on).
void ark_kmark(ark_m1* h, int cls, double bytes)
{
    h->launches++;
    if (!h->ktiming) return;
    if (h->kused == h->kev->size()) { cudaEvent_t e; cudaEventCreate(&e); h->kev->push_back(e); }
    cudaEventRecord((*h->kev)[h->kused++], h->st);
    h->kcls->push_back(cls); h->kbytes->push_back(bytes);
}
// Close the open series: one final event, then (after a sync) accumulate per-class elapsed times.
void ark_kflush(ark_m1* h)
{
    if (!h->ktiming || h->kcls->empty()) return;
    if (h->kused == h->kev->size()) { cudaEvent_t e; cudaEventCreate(&e); h->kev->push_back(e); }
    cudaEventRecord((*h->kev)[h->kused], h->st);
    cudaStreamSynchronize(h->st);
    for (size_t k = 0; k < h->kcls->size(); ++k) {
        float ms = 0.f; cudaEventElapsedTime(&ms, (*h->kev)[k], (*h->kev)[k + 1]);
        const int c = (*h->kcls)[k];
        h->kstat[c][0] += 1.0; h->kstat[c][1] += ms; h->kstat[c][2] += (*h->kbytes)[k];
    }
    h->kcls->clear(); h->kbytes->clear(); h->kused = 0;
}

int ark_dmalloc(ark_m1* h, void** p, size_t bytes)
{
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) { *p = nullptr; cudaGetLastError(); return ark_fail(h, ARK_M1_E_ALLOC, "cudaMalloc: %s", cudaGetErrorString(e)); }
    h->bytes += (long long)bytes;
    if (h->allocs) (*h->allocs)[*p] = bytes;
    return 0;
}

// cudaFree of a dmalloc'ed pointer with the byte count kept right (null is fine)
void ark_dfree(ark_m1* h, void* p)
{
    if (!p) return;
    cudaFree(p);
    if (!h->allocs) return;
    auto it = h->allocs->find(p);
    if (it != h->allocs->end()) { h->bytes -= (long long)it->second; h->allocs->erase(it); }
}

// the multigrid hierarchy is built from assembled blocks: it overrides the matrix-free operator
static inline int opk(const ark_m1* h) { return h->precond == 1 ? 0 : h->op_kind; }
// bytes per cell the preconditioned matrix-free operator does not move when it rebuilds the diagonal block (the nine M^-1 planes)
static inline double mf_saved(const ark_m1* h) { return h->mf.rc ? (h->mf.rcj ? 128.0 : 72.0) : 0.0; }

// compressed-basis GMRES applies to the default solver configuration only; elsewhere the option is ignored
static inline bool use_cb(const ark_m1* h) { return h->basis_prec == 32 && h->krylov == 0 && h->precond == 0 && h->op_kind == 1 && h->ortho == 1; }

Fields ark_fields_of(const ark_m1* h)
{
    Fields f;
    const double* U = h->U[h->cur];
    f.E = U; f.Fx = U + h->N; f.Fy = U + 2 * h->N; f.sa = h->sa; f.st = h->stot;
    for (int s = 0; s < 4; ++s) for (int k = 0; k < 5; ++k) f.gh[s][k] = h->gh[s][k];
    for (int s = 0; s < 2; ++s)      // halo sides of a slab: the ghost lines are the received boundary rows of the neighbour rank
        if (h->g.bc[YLO + s] == BC_HALO) for (int k = 0; k < 5; ++k) f.gh[YLO + s][k] = h->halo_state[s] + (size_t)k * h->g.nx;
    f.T = h->have_T ? h->T[h->cur] : nullptr;
    f.rho_cv = h->rho_cv; f.source_E = h->source_E;
    return f;
}

// a slab with halo sides can only be advanced through its group (the halos must be exchanged first)
static inline bool needs_group(const ark_m1* h) { return h->g.bc[YLO] == BC_HALO || h->g.bc[YHI] == BC_HALO; }
#define NO_SLAB(h, what) do { if (needs_group(h)) return ark_fail(h, ARK_M1_E_UNSUPPORTED, what ": this handle is a slab of an ark_m1_group; use the ark_m1_group_* call%s", ""); } while (0)

extern "C" {

const char* ark_m1_version(void) { return "ark_m1 0.1 (sm_100a, fp64)"; }

ark_m1* ark_m1_create(int nx, int ny, double dx, double dy, double c, const ark_m1_bc* bc)
{
    if (nx < 1 || ny < 1 || !(dx > 0) || !(dy > 0) || !(c > 0)) return nullptr;
    int b[4] = { 0, 0, 0, 0 };
    if (bc) { b[0] = bc->xlo; b[1] = bc->xhi; b[2] = bc->ylo; b[3] = bc->yhi; }
    for (int s = 0; s < 4; ++s) if (b[s] < 0 || b[s] > 2) return nullptr;
    if ((b[0] == BC_PERIODIC) != (b[1] == BC_PERIODIC) || (b[2] == BC_PERIODIC) != (b[3] == BC_PERIODIC)) return nullptr;
    if ((ny + 3) / 4 > 65535) return nullptr;      // several kernels map four rows to one gridDim.y slot (limit 65535): ny <= 262140
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    ark_m1* h = new (std::nothrow) ark_m1;
    if (!h) return nullptr;
    memset(h, 0, sizeof *h);
    h->g.nx = nx; h->g.ny = ny; h->g.dx = dx; h->g.dy = dy; h->g.c = c;
    for (int s = 0; s < 4; ++s) h->g.bc[s] = b[s];
    h->s.wb = 1; h->s.ap = 1; h->s.eig = 0; h->s.closure = 0; h->s.lin = 0; h->s.eig_floor = 0.0; h->s.a_r = 1.0; h->s.src_off = 0; h->s.hyp_off = 0;
    h->ortho = 1; h->explicit_kernel = 3; h->op_kind = 1; h->maxv = 16; h->asm_kernel = 1; h->op_recompute = 2; h->apply_precond = 0; h->arnoldi_block = 5; h->op_pair = 1;
    h->basis_prec = 64; h->precond = 0; h->mg.omega = 0.8; h->mg.coarse_sweeps = 2; h->mg.nlev = 0; h->mg.precision = 64;
    h->device = dev; h->N = (long long)nx * ny; h->st = 0;
    cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
    h->hist_host = new std::vector<double>();
    h->allocs = new std::map<void*, size_t>();
    h->kev = new std::vector<cudaEvent_t>(); h->kcls = new std::vector<int>(); h->kbytes = new std::vector<double>();
    const size_t N = (size_t)h->N;
    bool ok = true;
    for (int k = 0; k < 2 && ok; ++k) ok = ark_dmalloc(h, (void**)&h->U[k], 3 * N * sizeof(double)) == 0;
    ok = ok && ark_dmalloc(h, (void**)&h->sa, N * sizeof(double)) == 0;
    ok = ok && ark_dmalloc(h, (void**)&h->ss_tmp, N * sizeof(double)) == 0;
    ok = ok && ark_dmalloc(h, (void**)&h->stot, N * sizeof(double)) == 0;
    ok = ok && ark_dmalloc(h, (void**)&h->counts, 2 * sizeof(unsigned long long)) == 0;
    for (int s = 0; s < 4 && ok; ++s) {
        const size_t len = (s < 2) ? ny : nx;
        for (int k = 0; k < 5 && ok; ++k) {
            ok = ark_dmalloc(h, (void**)&h->gh[s][k], len * sizeof(double)) == 0;
            if (ok) cudaMemset(h->gh[s][k], 0, len * sizeof(double));
        }
    }
    ok = ok && cudaMallocHost((void**)&h->ctl_host, sizeof(GmresCtl)) == cudaSuccess;
    for (int k = 0; k < 3 && ok; ++k) ok = cudaEventCreate(&h->ev[k]) == cudaSuccess;
    if (!ok) { ark_m1_destroy(h); return nullptr; }
    return h;
}

static void free_implicit(ark_m1* h)
{
    for (int l = 0; l < h->mg.nlev; ++l) { ark_dfree(h, h->mg.lev[l].off32); h->mg.lev[l].off32 = nullptr; }
    for (int l = 1; l < h->mg.nlev; ++l) { ark_dfree(h, h->mg.lev[l].off); ark_dfree(h, h->mg.lev[l].Dinv); ark_dfree(h, h->mg.lev[l].r); ark_dfree(h, h->mg.lev[l].e); }
    h->mg.nlev = 0; ark_dfree(h, h->mgz); h->mgz = nullptr;
    ark_dfree(h, h->V32); h->V32 = nullptr; ark_dfree(h, h->wk); h->wk = nullptr; h->m32_alloc = 0; h->vslots = 0;
    ark_dfree(h, h->A.off); ark_dfree(h, h->A.C); ark_dfree(h, h->A.Minv); ark_dfree(h, h->A.b); ark_dfree(h, h->V); ark_dfree(h, h->tvec); cudaFree(h->wblock); ark_dfree(h, h->nprev); h->nprev = nullptr;
    ark_dfree(h, h->mf.J); ark_dfree(h, h->mf.fE); ark_dfree(h, h->mf.fN); ark_dfree(h, h->mf.dE); ark_dfree(h, h->mf.dF); ark_dfree(h, h->mf.fxy); ark_dfree(h, h->mf.xlo); ark_dfree(h, h->mf.ylo);
    memset(&h->mf, 0, sizeof h->mf);
    h->A.off = h->A.C = h->A.Minv = h->A.b = nullptr; h->V = h->tvec = nullptr; h->wblock = nullptr; h->m_alloc = 0; h->maxit_alloc = 0;
}

void ark_m1_destroy(ark_m1* h)
{
    if (!h) return;
    GUARD(h);
    cudaStreamSynchronize(h->st);
    ark_pipe_free(h);
    for (int k = 0; k < 2; ++k) { cudaFree(h->U[k]); cudaFree(h->T[k]); }
    cudaFree(h->sa); cudaFree(h->ss_tmp); cudaFree(h->stot); cudaFree(h->counts);
    for (int s = 0; s < 4; ++s) for (int k = 0; k < 5; ++k) cudaFree(h->gh[s][k]);
    cudaFree(h->rho_cv); cudaFree(h->ux); cudaFree(h->uy); cudaFree(h->source_E);
    free_implicit(h);
    if (h->ctl_host) cudaFreeHost(h->ctl_host);
    for (int k = 0; k < 3; ++k) if (h->ev[k]) cudaEventDestroy(h->ev[k]);
    delete h->hist_host; delete h->allocs; h->allocs = nullptr;
    if (h->kev) for (cudaEvent_t e : *h->kev) cudaEventDestroy(e);
    delete h->kev; delete h->kcls; delete h->kbytes;
    cudaGetLastError();
    delete h;
}

int ark_m1_set_stream(ark_m1* h, void* cuda_stream)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    CU(cudaStreamSynchronize(h->st));
    h->st = (cudaStream_t)cuda_stream;
    return 0;
}

int ark_m1_set_state(ark_m1* h, const double* E, const double* F, const double* sigma_a, const double* sigma_s, const double* T)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    if (!E || !F || !sigma_a || !sigma_s) return ark_fail(h, ARK_M1_E_ARG, "set_state: NULL array%s", "");
    const size_t N = (size_t)h->N, B = N * sizeof(double);
    double* U = h->U[h->cur];
    CU(cudaMemcpyAsync(U, E, B, cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(U + N, F, 2 * B, cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(h->sa, sigma_a, B, cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(h->ss_tmp, sigma_s, B, cudaMemcpyDefault, h->st));
    CU(launch_add_planes(h->stot, h->sa, h->ss_tmp, (long long)N, h->st));
    if (T) {
        for (int k = 0; k < 2; ++k) if (!h->T[k]) { int rc = ark_dmalloc(h, (void**)&h->T[k], B); if (rc) return rc; }
        CU(cudaMemcpyAsync(h->T[h->cur], T, B, cudaMemcpyDefault, h->st));
    }
    h->have_T = (T != nullptr);
    h->have_state = true;
    return 0;
}

int ark_m1_set_boundary(ark_m1* h, int side, const double* E_g, const double* F_g, const double* sa_g, const double* ss_g)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    if (side < 0 || side > 3 || !E_g || !F_g || !sa_g || !ss_g) return ark_fail(h, ARK_M1_E_ARG, "set_boundary: bad argument%s", "");
    const size_t len = (side < 2) ? h->g.ny : h->g.nx, B = len * sizeof(double);
    CU(cudaMemcpyAsync(h->gh[side][0], E_g, B, cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(h->gh[side][1], F_g, B, cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(h->gh[side][2], F_g + len, B, cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(h->gh[side][3], sa_g, B, cudaMemcpyDefault, h->st));
    // sigma_t ghost = sigma_a + sigma_s: stage sigma_s in the sigma_t line, then add in place
    CU(cudaMemcpyAsync(h->gh[side][4], ss_g, B, cudaMemcpyDefault, h->st));
    CU(launch_add_planes(h->gh[side][4], h->gh[side][3], h->gh[side][4], (long long)len, h->st));
    return 0;
}

int ark_m1_set_option(ark_m1* h, const char* key, double value)
{
    if (!h || !key) return ARK_M1_E_ARG;
    GUARD(h);
    const int iv = (int)value;
    if (!strcmp(key, "well_balanced")) h->s.wb = (value != 0.0);
    else if (!strcmp(key, "ap_mode")) { if (iv < 0 || iv > 2) return ark_fail(h, ARK_M1_E_ARG, "ap_mode must be 0, 1 or 2%s", ""); h->s.ap = iv; }
    else if (!strcmp(key, "eig_mode")) { if (iv < 0 || iv > 2) return ark_fail(h, ARK_M1_E_ARG, "eig_mode must be 0, 1 or 2%s", ""); h->s.eig = iv; }
    else if (!strcmp(key, "closure")) { if (iv < 0 || iv > 1) return ark_fail(h, ARK_M1_E_ARG, "closure must be 0 or 1%s", ""); h->s.closure = iv; }
    else if (!strcmp(key, "linearisation")) { if (iv < 0 || iv > 1) return ark_fail(h, ARK_M1_E_ARG, "linearisation must be 0 or 1%s", ""); h->s.lin = iv; }
    else if (!strcmp(key, "eig_floor")) { if (!(value >= 0.0)) return ark_fail(h, ARK_M1_E_ARG, "eig_floor must be >= 0%s", ""); h->s.eig_floor = value; }
    else if (!strcmp(key, "a_r")) h->s.a_r = value;
    else if (!strcmp(key, "orthogonalisation")) { if (iv < 1 || iv > 2) return ark_fail(h, ARK_M1_E_ARG, "orthogonalisation must be 1 or 2%s", ""); h->ortho = iv; }
    else if (!strcmp(key, "explicit_kernel")) { if (iv != 0 && iv != 1 && iv != 3) return ark_fail(h, ARK_M1_E_ARG, "explicit_kernel must be 0 (cell), 1 (128-column march) or 3 (one-warp march, default)%s", ""); h->explicit_kernel = iv; }
    else if (!strcmp(key, "assembly_kernel")) { if (iv < 0 || iv > 1) return ark_fail(h, ARK_M1_E_ARG, "assembly_kernel must be 0 (tile) or 1 (marching)%s", ""); h->asm_kernel = iv; }
    else if (!strcmp(key, "krylov")) { if (iv < 0 || iv > 1) return ark_fail(h, ARK_M1_E_ARG, "krylov must be 0 (GMRES) or 1 (BiCGStab)%s", ""); h->krylov = iv; }
    else if (!strcmp(key, "vectors_per_pass")) { if (iv < 1 || iv > MAXV) return ark_fail(h, ARK_M1_E_ARG, "vectors_per_pass must be in [1, 16]%s", ""); h->maxv = iv; }
    else if (!strcmp(key, "release_workspace")) { if (value != 0.0) { cudaStreamSynchronize(h->st); free_implicit(h); } }
    else if (!strcmp(key, "kernel_timing")) { ark_kflush(h); h->ktiming = (value != 0.0); if (h->ktiming) memset(h->kstat, 0, sizeof h->kstat); }
    else if (!strcmp(key, "operator")) { if (iv < 0 || iv > 1) return ark_fail(h, ARK_M1_E_ARG, "operator must be 0 (block stencil) or 1 (matrix-free)%s", ""); h->op_kind = iv; }
    else if (!strcmp(key, "apply_operator_precond")) h->apply_precond = (value != 0.0);
    else if (!strcmp(key, "op_pair")) h->op_pair = (value != 0.0);
    else if (!strcmp(key, "arnoldi_block")) { if (iv < 1 || iv > SMAX) return ark_fail(h, ARK_M1_E_ARG, "arnoldi_block must be 1 (one column per pass over the basis), 2 (two columns) or 3..5 (s-step block)%s", ""); h->arnoldi_block = iv; }
    else if (!strcmp(key, "op_recompute")) { if (iv < 0 || iv > 2) return ark_fail(h, ARK_M1_E_ARG, "op_recompute must be 0 (load M^-1), 1 (rebuild the diagonal block in the operator) or 2 (rebuild J as well)%s", ""); h->op_recompute = iv; }
    else if (!strcmp(key, "preconditioner")) { if (iv < 0 || iv > 1) return ark_fail(h, ARK_M1_E_ARG, "preconditioner must be 0 (block-Jacobi) or 1 (multigrid)%s", ""); h->precond = iv; }
    else if (!strcmp(key, "mg_omega")) { if (!(value > 0.0) || !(value < 2.0)) return ark_fail(h, ARK_M1_E_ARG, "mg_omega must be in (0, 2)%s", ""); h->mg.omega = value; }
    else if (!strcmp(key, "mg_coarse_sweeps")) { if (iv < 1) return ark_fail(h, ARK_M1_E_ARG, "mg_coarse_sweeps must be >= 1%s", ""); h->mg.coarse_sweeps = iv; }
    else if (!strcmp(key, "basis_precision")) { if (iv != 32 && iv != 64) return ark_fail(h, ARK_M1_E_ARG, "basis_precision must be 64 or 32%s", ""); h->basis_prec = iv; }
    else if (!strcmp(key, "mg_precision")) { if (iv != 32 && iv != 64) return ark_fail(h, ARK_M1_E_ARG, "mg_precision must be 64 or 32%s", ""); h->mg.precision = iv; }
    else return ark_fail(h, ARK_M1_E_ARG, "unknown option %s", key);
    return 0;
}

int ark_m1_set_field(ark_m1* h, const char* name, const double* plane)
{
    if (!h || !name) return ARK_M1_E_ARG;
    GUARD(h);
    double** dst = nullptr;
    if (!strcmp(name, "rho_cv")) dst = &h->rho_cv; else if (!strcmp(name, "ux")) dst = &h->ux;
    else if (!strcmp(name, "uy")) dst = &h->uy; else if (!strcmp(name, "source_E")) dst = &h->source_E;
    else return ark_fail(h, ARK_M1_E_ARG, "unknown field %s", name);
    const size_t B = (size_t)h->N * sizeof(double);
    if (!plane) { CU(cudaStreamSynchronize(h->st)); ark_dfree(h, *dst); *dst = nullptr; return 0; }
    if (!*dst) { int rc = ark_dmalloc(h, (void**)dst, B); if (rc) return rc; }
    CU(cudaMemcpyAsync(*dst, plane, B, cudaMemcpyDefault, h->st));
    return 0;
}

int ark_m1_get_state(ark_m1* h, double* E, double* F, double* T)
{
    if (!h || !E || !F) return ARK_M1_E_ARG;
    GUARD(h);
    const size_t N = (size_t)h->N, B = N * sizeof(double);
    const double* U = h->U[h->cur];
    CU(cudaMemcpyAsync(E, U, B, cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(F, U + N, 2 * B, cudaMemcpyDefault, h->st));
    if (T && h->have_T) CU(cudaMemcpyAsync(T, h->T[h->cur], B, cudaMemcpyDefault, h->st));
    CU(cudaStreamSynchronize(h->st));
    return 0;
}

}  // extern "C"

int ark_explicit_once(ark_m1* h, double dt)
{
    const Fields f = ark_fields_of(h);
    double* O = h->U[h->cur ^ 1];
    double* OT = h->have_T ? h->T[h->cur ^ 1] : nullptr;
    // algorithmic bytes per cell: 5 planes in, 3 out; the coupled step adds T in/out (16), rho c_v (8) and the source plane (8)
    const double bpc = 64.0 + (h->have_T ? 16.0 + (h->rho_cv ? 8.0 : 0.0) : 0.0) + (h->source_E ? 8.0 : 0.0);
    const bool small = h->N < (1LL << 31);          // the march kernels use 32-bit in-plane offsets (their launchers check it too)
    if (h->explicit_kernel == 3 && small)
        KL(KC_EXPLICIT, bpc * h->N, launch_explicit_march3(h->g, h->s, f, dt, O, O + h->N, O + 2 * h->N, OT, h->sm_count, h->st));
    else if (h->explicit_kernel >= 1 && small)
        KL(KC_EXPLICIT, bpc * h->N, launch_explicit_march(h->g, h->s, f, dt, O, O + h->N, O + 2 * h->N, OT, h->sm_count, h->st));
    else
        KL(KC_EXPLICIT, bpc * h->N, launch_explicit_cell(h->g, h->s, f, dt, 0, O, O + h->N, O + 2 * h->N, OT, h->st));
    h->cur ^= 1;
    return 0;
}

extern "C" {

int ark_m1_step_explicit(ark_m1* h, double dt)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "step_explicit");
    if (!(dt > 0.0)) return ark_fail(h, ARK_M1_E_ARG, "step_explicit: dt must be > 0%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "step_explicit: no state set%s", "");
    return ark_explicit_once(h, dt);
}

int ark_m1_steps_explicit(ark_m1* h, double dt, int nsteps)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "steps_explicit");
    if (!(dt > 0.0) || nsteps < 0) return ark_fail(h, ARK_M1_E_ARG, "steps_explicit: dt must be > 0 and nsteps >= 0%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "steps_explicit: no state set%s", "");
    for (int k = 0; k < nsteps; ++k) { int rc = ark_explicit_once(h, dt); if (rc) return rc; }
    return 0;
}

int ark_m1_residual(ark_m1* h, double* RE, double* RF)
{
    if (!h || !RE || !RF) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "residual");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "residual: no state set%s", "");
    const Fields f = ark_fields_of(h);
    double* O = h->U[h->cur ^ 1];
    const size_t N = (size_t)h->N;
    KL(KC_EXPLICIT, 64.0 * h->N, launch_explicit_cell(h->g, h->s, f, 0.0, 1, O, O + N, O + 2 * N, nullptr, h->st));
    CU(cudaMemcpyAsync(RE, O, N * sizeof(double), cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(RF, O + N, 2 * N * sizeof(double), cudaMemcpyDefault, h->st));
    CU(cudaStreamSynchronize(h->st));
    return 0;
}

int ark_m1_add_velocity_sources(ark_m1* h, double dt)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    if (!h->have_state || !h->ux || !h->uy) return ark_fail(h, ARK_M1_E_NOTSET, "add_velocity_sources: state, ux, uy must be set%s", "");
    const Fields f = ark_fields_of(h);
    double* U = h->U[h->cur];
    KL(KC_SMALL, 88.0 * h->N, launch_velocity_sources(h->g, h->s, f, h->ux, h->uy, dt, U, U + h->N, U + 2 * h->N, h->st));
    return 0;
}

int ark_m1_count_unrealizable(ark_m1* h, long long* nE, long long* nf)
{
    if (!h || !nE || !nf) return ARK_M1_E_ARG;
    GUARD(h);
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "count_unrealizable: no state set%s", "");
    CU(cudaMemsetAsync(h->counts, 0, 2 * sizeof(unsigned long long), h->st));
    KL(KC_SMALL, 24.0 * h->N, launch_count_unrealizable(h->g, ark_fields_of(h), h->counts, h->st));
    unsigned long long out[2];
    CU(cudaMemcpyAsync(out, h->counts, sizeof out, cudaMemcpyDeviceToHost, h->st));
    CU(cudaStreamSynchronize(h->st));
    *nE = (long long)out[0]; *nf = (long long)out[1];
    return 0;
}

long long ark_m1_device_bytes(const ark_m1* h) { return h ? h->bytes : 0; }
const char* ark_m1_last_error(const ark_m1* h) { return h ? h->err : "null handle"; }

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------
// Implicit step
// ---------------------------------------------------------------------------------------------------------
int ark_ensure_implicit(ark_m1* h, int m, int maxit)
{
    const size_t N = (size_t)h->N, n = 3 * N;
    const bool have_op = (opk(h) == 0) ? (h->A.off != nullptr) : (h->mf.J != nullptr);
    if (h->m_alloc >= m && h->maxit_alloc >= maxit && have_op && (h->precond == 0 || (h->mg.nlev > 0 && (h->mg.precision == 64 || h->mg.lev[0].off32)))
        && h->vslots >= (use_cb(h) ? 6 : ((m + 1) > 6 ? (m + 1) : 6)) && (!use_cb(h) || (h->m32_alloc >= m && h->wk))) return 0;
    CU(cudaStreamSynchronize(h->st));
    const long long before = h->bytes;
    (void)before;
    if (h->A.Minv == nullptr) {
        int rc;
        if ((rc = ark_dmalloc(h, (void**)&h->A.Minv, 9 * N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->A.b, n * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->tvec, n * sizeof(double)))) return rc;
    }
    if (opk(h) == 0 && h->A.off == nullptr) {
        int rc;
        if ((rc = ark_dmalloc(h, (void**)&h->A.off, 36 * N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->A.C, 9 * N * sizeof(double)))) return rc;
    }
    if (opk(h) == 1 && h->mf.J == nullptr) {
        int rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.J, 9 * N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.fE, 4 * N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.fN, 4 * N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.dE, N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.dF, N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.fxy, 2 * N * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.xlo, 4 * (size_t)h->g.ny * sizeof(double)))) return rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mf.ylo, 4 * (size_t)h->g.nx * sizeof(double)))) return rc;
    }
    if (h->precond == 1 && h->mg.nlev == 0) {       // levels 1.. of the multigrid hierarchy (about 1/3 of the fine storage)
        int rc;
        if ((rc = ark_dmalloc(h, (void**)&h->mgz, n * sizeof(double)))) return rc;
        MgHier& H = h->mg;
        H.lev[0].g = h->g; H.lev[0].off = nullptr; H.lev[0].off32 = nullptr; H.lev[0].Dinv = nullptr; H.lev[0].r = nullptr; H.lev[0].e = nullptr;
        int L = 1; double cells = 1.0;
        while ((H.lev[L - 1].g.nx > 1 || H.lev[L - 1].g.ny > 1) && L < MG_MAXLEV) {
            MgLevel& c = H.lev[L];
            c.g = H.lev[L - 1].g; c.g.nx = (c.g.nx + 1) / 2; c.g.ny = (c.g.ny + 1) / 2;
            const size_t Nc = (size_t)c.g.nx * c.g.ny;
            c.off = c.Dinv = c.r = c.e = nullptr; c.off32 = nullptr;
            H.nlev = L + 1;                          // so that a failure below frees what was allocated
            if ((rc = ark_dmalloc(h, (void**)&c.off, 36 * Nc * sizeof(double)))) return rc;
            if ((rc = ark_dmalloc(h, (void**)&c.Dinv, 9 * Nc * sizeof(double)))) return rc;
            if ((rc = ark_dmalloc(h, (void**)&c.r, 3 * Nc * sizeof(double)))) return rc;
            if ((rc = ark_dmalloc(h, (void**)&c.e, 3 * Nc * sizeof(double)))) return rc;
            cells += (double)Nc / (double)N;
            ++L;
        }
        if (H.lev[L - 1].g.nx > 1 || H.lev[L - 1].g.ny > 1) return ark_fail(h, ARK_M1_E_UNSUPPORTED, "multigrid: grid too large for %s levels", "24");
        H.nlev = L; h->mg_cells = cells;
    }
    if (h->precond == 1 && h->mg.precision == 32 && h->mg.lev[0].off32 == nullptr) {
        for (int l = 0; l < h->mg.nlev; ++l) {
            const size_t Nl = (size_t)h->mg.lev[l].g.nx * h->mg.lev[l].g.ny;
            int rc = ark_dmalloc(h, (void**)&h->mg.lev[l].off32, 36 * Nl * sizeof(float));
            if (rc) return rc;
        }
    }
    h->stride = (long long)((n + 31) / 32 * 32);
    {   // fp64 vector slots: the whole basis, or (compressed-basis path) the six slots BiCGStab and the staging calls use
        const int need = use_cb(h) ? 6 : ((m + 1) > 6 ? (m + 1) : 6);
        if (h->vslots < need) {
            ark_dfree(h, h->V); h->V = nullptr; h->vslots = 0;
            int rc = ark_dmalloc(h, (void**)&h->V, (size_t)need * h->stride * sizeof(double));
            if (rc) return rc;
            h->vslots = need;
        }
        if (use_cb(h)) {
            int rc;
            if (h->m32_alloc < m) {
                ark_dfree(h, h->V32); h->V32 = nullptr; h->m32_alloc = 0;
                if ((rc = ark_dmalloc(h, (void**)&h->V32, (size_t)(m + 1) * h->stride * sizeof(float)))) return rc;
                h->m32_alloc = m;
            }
            if (!h->wk && (rc = ark_dmalloc(h, (void**)&h->wk, n * sizeof(double)))) return rc;
        }
    }
    const int mm = m > h->m_alloc ? m : h->m_alloc;
    const int mi = maxit > h->maxit_alloc ? maxit : h->maxit_alloc;
    // small block: ctl | H | cs | sn | g | y | scale | coef | hist | partial
    if (h->wblock) { cudaFree(h->wblock); h->wblock = nullptr; }
    long long caph = (long long)mi + mi / (mm > 0 ? mm : 1) + 8;
    if (caph > (1LL << 20)) caph = (1LL << 20);     // the history keeps at most 2^20 entries (later ones are counted, not stored)
    const int caphist = (int)caph;
    const size_t nd = 2 * (size_t)(mm + 1) * mm + 2 * (size_t)mm + (mm + 1) + mm + 5 * (size_t)(mm + 1) + caphist
                      + 2 * (size_t)SMAX * (mm + 1) + 2 * SMAX * SMAX + (size_t)sstep_partial_doubles(h->sm_count)
                      + (size_t)(krylov_max_blocks(h->sm_count) > op_mf_blocks(h->g, h->sm_count) ? krylov_max_blocks(h->sm_count) : op_mf_blocks(h->g, h->sm_count)) * MAXV;
    const size_t ctl_bytes = (sizeof(GmresCtl) + 255) / 256 * 256;
    if (cudaMalloc(&h->wblock, ctl_bytes + nd * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return ark_fail(h, ARK_M1_E_ALLOC, "cudaMalloc (solver scalars)%s", ""); }
    CU(cudaMemset(h->wblock, 0, ctl_bytes + nd * sizeof(double)));
    GmresWork& W = h->W;
    W.ctl = (GmresCtl*)h->wblock;
    double* p = (double*)((char*)h->wblock + ctl_bytes);
    W.H = p; p += (size_t)(mm + 1) * mm;
    W.cs = p; p += mm; W.sn = p; p += mm; W.g = p; p += mm + 1; W.y = p; p += mm;
    W.scale = p; p += mm + 1; W.coef = p; p += mm + 1; W.hist = p; p += caphist;
    W.Hraw = p; p += (size_t)(mm + 1) * mm; W.c1 = p; p += mm + 1; W.c2 = p; p += mm + 1; W.coef2 = p; p += mm + 1;
    W.cS = p; p += (size_t)SMAX * (mm + 1); W.coefS = p; p += (size_t)SMAX * (mm + 1); W.Rb = p; p += SMAX * SMAX; W.tb = p; p += SMAX * SMAX;
    W.partialS = p; p += sstep_partial_doubles(h->sm_count);
    W.partial = p;
    W.caphist = caphist;
    h->m_alloc = mm; h->maxit_alloc = mi;
    return 0;
}

// V0 <- b - A x  (A x = Ahat (C x)), then its norm with the DOT_RNORM epilogue.
static int true_residual(ark_m1* h, const double* x)
{
    const long long n = 3 * h->N;
    if (opk(h) == 1) {
        KL(KC_SPMV, 216.0 * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, x, h->V, nullptr, h->A.b, -1.0, nullptr, 0, h->sm_count, h->st));
    } else {
        KL(KC_DIAGMUL, 120.0 * h->N, launch_diag_mul(h->g, h->A.C, x, h->tvec, h->st));
        KL(KC_SPMV, 360.0 * h->N, launch_spmv_hat(h->g, h->A.off, h->tvec, h->V, nullptr, h->A.b, -1.0, nullptr, h->st));
    }
    KL(KC_DOT, 24.0 * h->N, launch_multi_dot(h->V, h->V, h->stride, 1, 0, n, h->W, DOT_RNORM, h->sm_count, h->st));
    return 0;
}

int ark_fetch_ctl(ark_m1* h)
{
    CU(cudaMemcpyAsync(h->ctl_host, h->W.ctl, sizeof(GmresCtl), cudaMemcpyDeviceToHost, h->st));
    CU(cudaStreamSynchronize(h->st));
    return 0;
}

int ark_assemble_system(ark_m1* h, double dt, const double* bsrc)
{
    const Fields f = ark_fields_of(h);
    if (opk(h) == 1) {
        h->mf.rx = h->s.hyp_off ? 0.0 : dt / h->g.dx; h->mf.ry = h->s.hyp_off ? 0.0 : dt / h->g.dy;
        h->mf.rc = h->op_recompute; h->mf.has_dF = (h->s.wb == 0);
        // the reduced-flux planes are written by the marching assembly; the M1 Jacobian formula holds for the default scheme
        h->mf.rcj = (h->op_recompute == 2 && h->s.is_default() && h->asm_kernel == 1 && h->N < (1LL << 31)) ? 1 : 0;
        h->mf.rc = h->op_recompute ? 1 : 0;
        if (h->asm_kernel == 1 && h->N < (1LL << 31))
            KL(KC_ASSEMBLE, 304.0 * h->N, launch_assemble_march(h->g, h->s, f, dt, h->A, h->mf, bsrc, h->sm_count, h->st));     // 288 + the two reduced-flux planes
        else
            KL(KC_ASSEMBLE, 288.0 * h->N, launch_assemble(h->g, h->s, f, dt, h->A, h->mf, bsrc, h->st));
    } else {
        MfPlanes none; memset(&none, 0, sizeof none);
        KL(KC_ASSEMBLE, 496.0 * h->N, launch_assemble(h->g, h->s, f, dt, h->A, none, bsrc, h->st));
        float* o32 = (h->precond == 1 && h->mg.precision == 32) ? h->mg.lev[0].off32 : nullptr;
        KL(KC_SCALE, (648.0 + (o32 ? 144.0 : 0.0)) * h->N, launch_scale_offdiag(h->g, h->A, o32, h->st));
    }
    if (h->precond == 1) {       // Galerkin hierarchy: each level reads 36 doubles per finer cell, writes 45 (+ the scaling pass) per cell
        h->mg.lev[0].off = h->A.off;
        for (int l = 1; l < h->mg.nlev; ++l) {
            const MgLevel& f = h->mg.lev[l - 1]; const MgLevel& c = h->mg.lev[l];
            const double Nf = (double)f.g.nx * f.g.ny, Nc = (double)c.g.nx * c.g.ny;
            h->launches++;      // two kernels per level
            KL(KC_MGSETUP, 288.0 * Nf + (360.0 + 648.0) * Nc, launch_mg_galerkin(f.g, f.off, c.g, c.off, c.Dinv, h->mg.precision == 32 ? c.off32 : nullptr, h->st));
        }

    }
    return 0;
}

// z^ = Mhat^-1 v: one V-cycle in the hat variable (v, zhat: 3N, distinct).  Two stencil passes per level.
static int mg_apply(ark_m1* h, const double* v, double* zhat, const int* stop)
{
    int nl = 0;
    ark_kmark(h, KC_MG, (h->mg.precision == 32 ? (168.0 + 192.0) : (312.0 + 336.0)) * h->N * h->mg_cells);
    CU(launch_mg_vcycle(h->mg, v, zhat, stop, h->st, &nl));
    h->launches += nl - 1;
    return 0;
}

// Restarted GMRES(m) on the assembled system, x = U[cur] in place (initial guess on entry).  Leaves the final control
// block in h->ctl_host.
static int gmres_solve(ark_m1* h, double tol, int m, int maxit)
{
    int rc;
    const long long n = 3 * h->N, S = h->stride;
    const int sm = h->sm_count;
    double* x = h->U[h->cur];
    GmresWork W = h->W;
    const int* stop = &W.ctl->inner_stop;
    const int MV = h->maxv;            // basis vectors per pass of the multi-vector kernels
    KL(KC_SMALL, 0.0, launch_begin_solve(W, tol, m, maxit, h->st));
    KL(KC_DOT, 24.0 * h->N, launch_multi_dot(h->A.b, h->A.b, 0, 1, 0, n, W, DOT_BNORM, sm, h->st));
    if ((rc = true_residual(h, x))) return rc;
    if ((rc = ark_fetch_ctl(h))) return rc;
    // two columns per pass over the basis: GMRES + block-Jacobi + matrix-free operator + one-pass Gram-Schmidt, m within the staged epilogue
    const bool blk_ok = (h->precond == 0 && opk(h) == 1 && h->ortho == 1 && m <= 120);
    const bool pair = (h->arnoldi_block >= 2 && blk_ok && m >= 2);
    const int SB = (h->arnoldi_block >= 3 && blk_ok) ? h->arnoldi_block : 0;     // columns per s-step block (krylov_sstep.cu)
    const bool pair2 = SB && h->op_pair && op_mf2_ok(h->g, h->mf);               // two operator applications per pass inside a block
    while (!h->ctl_host->inner_stop) {
        for (int j = 0; j < m; ++j) {
            double* w = h->V + (size_t)(j + 1) * S;
            if (SB && j + SB <= m) {
                // s-step Arnoldi block (krylov_sstep.cu): W_1 = A^ v_j, W_k = (A^ - 1) W_{k-1} in the slots j+1 .. j+SB, one dot pass and one
                // update pass over the basis for all SB vectors, in-block solve, Hessenberg columns recovered on the device
                // (pairs of applications in one pass where the two-application kernel applies: operator_mf.cu, op_mf_rc2_kernel)
                for (int k = 0; k < SB; ++k) {
                    if (pair2 && k + 1 < SB) {
                        KL(KC_SPMV, 160.0 * h->N, launch_op_mf2(h->g, h->mf, h->A.Minv, h->V + (size_t)(j + k) * S, h->V + (size_t)(j + k + 1) * S, h->V + (size_t)(j + k + 2) * S,
                                                               k == 0 ? W.scale + j : nullptr, stop, sm, h->st, k == 0 ? 0.0 : 1.0, 1.0));
                        ++k;
                        continue;
                    }
                    KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, h->V + (size_t)(j + k) * S, h->V + (size_t)(j + k + 1) * S,
                                                                          k == 0 ? W.scale + j : nullptr, nullptr, 1.0, stop, 1, sm, h->st, k == 0 ? 0.0 : 1.0));
                }
                // the dot pass takes the block's own slots j+1 .. j+SB as basis vectors as well (W^T W, read from L1/L2): it predicts the
                // in-block solve, the update pass applies it and checks the result (krylov_sstep.cu: sstep_predict)
                const int nd = j + 1 + SB;
                for (int c0 = 0; c0 < nd; c0 += 32) {
                    const int nv = (nd - c0) < 32 ? (nd - c0) : 32, nbasis = (j + 1 - c0) < 0 ? 0 : ((j + 1 - c0) < nv ? (j + 1 - c0) : nv);
                    KL(KC_DOT, 24.0 * (nbasis + SB) * h->N, launch_dotS(w, h->V + (size_t)c0 * S, S, SB, nv, c0, n, W, sm, h->st, j));
                }
                KL(KC_UPDATE, (24.0 * (j + 1) + 48.0 * SB) * h->N, launch_updateS(w, h->V, S, SB, j + 1, n, W, sm, h->st, 1.0));
                // in-block solve as a pass of its own: only for a block whose prediction was not used (returns at once otherwise; its
                // 24 (2 SB - 1) B per cell are not booked)
                KL(KC_SMALL, 0.0, launch_qrS(w, S, SB, n, W, 1.0, 1, sm, h->st));
                // second round for a block flagged ill-conditioned (both kernels return at once otherwise)
                KL(KC_SMALL, 0.0, launch_gramS(w, S, SB, n, W, sm, h->st));
                KL(KC_SMALL, 0.0, launch_qrS(w, S, SB, n, W, 1.0, 2, sm, h->st));
                j += SB - 1;
                continue;
            }
            if (pair && j + 1 < m) {
                // two-column Arnoldi step: W1 = A M^-1 v_j, W2 = A M^-1 W1, both
                // orthogonalised against v_0..v_j in the same passes over the basis, then W2 against W1'
                double* w2 = h->V + (size_t)(j + 2) * S;
                if (h->op_pair && op_mf2_ok(h->g, h->mf))      // both applications in one pass (operator_mf.cu, op_mf_rc2_kernel)
                    KL(KC_SPMV, 160.0 * h->N, launch_op_mf2(h->g, h->mf, h->A.Minv, h->V + (size_t)j * S, w, w2, W.scale + j, stop, sm, h->st, 0.0, 0.0));
                else {
                    KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, h->V + (size_t)j * S, w, W.scale + j, nullptr, 1.0, stop, 1, sm, h->st));
                    KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, w, w2, nullptr, nullptr, 1.0, stop, 1, sm, h->st));
                }
                const int MV2 = krylov_pair_max_vectors();
                const int nchunk2 = (j + MV2) / MV2, csize2 = (j + nchunk2) / nchunk2;
                for (int c0 = 0; c0 <= j; c0 += csize2) {
                    const int nv = (j + 1 - c0) < csize2 ? (j + 1 - c0) : csize2;
                    KL(KC_DOT, 24.0 * (nv + 2) * h->N, launch_multi_dot2(w, w2, h->V + (size_t)c0 * S, S, nv, c0, n, W, sm, h->st));
                }
                KL(KC_UPDATE, 24.0 * (j + 1 + 4) * h->N, launch_update2_all(w, w2, h->V, S, j + 1, n, W, sm, h->st));
                KL(KC_UPDATE, 72.0 * h->N, launch_update(w2, w, S, 1, j + 1, n, W, 1, sm, h->st, UPD_B2B));
                ++j;
                continue;
            }
            if (h->precond == 1) {          // w = Ahat Mhat^-1 (scale_j v_j): the V-cycle is linear, the scale goes on last
                if ((rc = mg_apply(h, h->V + (size_t)j * S, h->mgz, stop))) return rc;
                KL(KC_SPMV, 336.0 * h->N, launch_spmv_hat(h->g, h->A.off, h->mgz, w, W.scale + j, nullptr, 1.0, stop, h->st));
            } else if (opk(h) == 1)
                KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, h->V + (size_t)j * S, w, W.scale + j, nullptr, 1.0, stop, 1, sm, h->st));
            else
                KL(KC_SPMV, 336.0 * h->N, launch_spmv_hat(h->g, h->A.off, h->V + (size_t)j * S, w, W.scale + j, nullptr, 1.0, stop, h->st));
            // the j+1 basis vectors go through the multi-vector kernels in ceil((j+1)/MV) chunks of (nearly) equal size
            const int nchunk = (j + MV) / MV, csize = (j + nchunk) / nchunk;
            for (int pass = 0; pass < h->ortho; ++pass) {
                for (int c0 = 0; c0 <= j; c0 += csize) {
                    const int nv = (j + 1 - c0) < csize ? (j + 1 - c0) : csize;
                    KL(KC_DOT, 24.0 * (nv + 1) * h->N, launch_multi_dot(w, h->V + (size_t)c0 * S, S, nv, c0, n, W, pass == 0 ? DOT_H : DOT_H2, sm, h->st));
                }
                for (int c0 = 0; c0 <= j; c0 += csize) {
                    const int nv = (j + 1 - c0) < csize ? (j + 1 - c0) : csize;
                    const int last = (c0 + csize > j) && (pass == h->ortho - 1);
                    KL(KC_UPDATE, 24.0 * (nv + 2) * h->N, launch_update(w, h->V + (size_t)c0 * S, S, nv, c0, n, W, last, sm, h->st));
                }
            }
        }
        KL(KC_SMALL, 0.0, launch_solve_y(W, h->st));
        if (h->precond == 1) {              // x += D^-1 Mhat^-1 (V y)
            KL(KC_COMBINE, 8.0 * (3.0 * m + 3.0) * h->N, launch_combine(h->g, h->V, S, nullptr, h->tvec, W, sm, h->st));
            if ((rc = mg_apply(h, h->tvec, h->mgz, nullptr))) return rc;
            KL(KC_COMBINE, 168.0 * h->N, launch_combine_y(h->g, h->A.Minv, h->mgz, x, h->st));
        } else
            KL(KC_COMBINE, 8.0 * (3.0 * m + 15.0) * h->N, launch_combine(h->g, h->V, S, h->A.Minv, x, W, sm, h->st));
        if ((rc = true_residual(h, x))) return rc;
        if ((rc = ark_fetch_ctl(h))) return rc;
    }
    return 0;
}

// Compressed-basis GMRES(m) (krylov_cb.cu; option "basis_precision" = 32): same algorithm and control flow as gmres_solve, the
// Arnoldi vectors stored in single precision (h->V32), one fp64 work vector (h->wk) carrying w = A M^-1 v_j through the
// orthogonalisation.  The true fp64 residual b - A x is recomputed at every restart, so the exit test is the same.
static int true_residual_cb(ark_m1* h, const double* x)
{
    const long long n = 3 * h->N;
    KL(KC_SPMV, 216.0 * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, x, h->wk, nullptr, h->A.b, -1.0, nullptr, 0, h->sm_count, h->st));
    KL(KC_DOT, 24.0 * h->N, launch_multi_dot(h->wk, h->wk, 0, 1, 0, n, h->W, DOT_RNORM, h->sm_count, h->st));
    KL(KC_UPDATE, 36.0 * h->N, launch_mg_to_float(h->wk, h->V32, n, h->st));          // v_0 = r, rounded once
    return 0;
}

static int gmres_solve_cb(ark_m1* h, double tol, int m, int maxit)
{
    int rc;
    const long long n = 3 * h->N, S = h->stride;
    const int sm = h->sm_count;
    double* x = h->U[h->cur];
    double* w = h->wk;
    GmresWork W = h->W;
    const int* stop = &W.ctl->inner_stop;
    const int MV = h->maxv < 16 ? h->maxv : 16;
    KL(KC_SMALL, 0.0, launch_begin_solve(W, tol, m, maxit, h->st));
    KL(KC_DOT, 24.0 * h->N, launch_multi_dot(h->A.b, h->A.b, 0, 1, 0, n, W, DOT_BNORM, sm, h->st));
    if ((rc = true_residual_cb(h, x))) return rc;
    if ((rc = ark_fetch_ctl(h))) return rc;
    while (!h->ctl_host->inner_stop) {
        for (int j = 0; j < m; ++j) {
            float* vnext = h->V32 + (size_t)(j + 1) * S;
            KL(KC_SPMV, (252.0 - mf_saved(h)) * h->N, launch_op_mf_f32(h->g, h->mf, h->A.Minv, h->V32 + (size_t)j * S, w, W.scale + j, stop, sm, h->st));
            for (int c0 = 0; c0 <= j; c0 += MV) {
                const int nv = (j + 1 - c0) < MV ? (j + 1 - c0) : MV;
                KL(KC_DOT, (24.0 + 12.0 * nv) * h->N, launch_multi_dot32(w, h->V32 + (size_t)c0 * S, S, nv, c0, n, W, DOT_H, sm, h->st));
            }
            for (int c0 = 0; c0 <= j; c0 += MV) {
                const int nv = (j + 1 - c0) < MV ? (j + 1 - c0) : MV;
                const int last = (c0 + MV > j);
                // intermediate chunks update w in place; the last one only stores the rounded result as v_{j+1} and its norm
                KL(KC_UPDATE, (24.0 + 12.0 * nv + (last ? 12.0 : 24.0)) * h->N,
                   launch_update32(w, h->V32 + (size_t)c0 * S, S, nv, c0, n, W, last, last ? 0 : 1, last ? vnext : nullptr, sm, h->st));
            }
        }
        KL(KC_SMALL, 0.0, launch_solve_y(W, h->st));
        KL(KC_COMBINE, 8.0 * (1.5 * m + 15.0) * h->N, launch_combine32(h->g, h->V32, S, h->A.Minv, x, W, sm, h->st));
        if ((rc = true_residual_cb(h, x))) return rc;
        if ((rc = ark_fetch_ctl(h))) return rc;
    }
    return 0;
}

// Right-preconditioned BiCGStab (the paper's Krylov method) on the assembled system; same conventions as
// gmres_solve.  Vector slots of h->V: 0 = r (and s), 1 = t, 2 = r^, 3 = p, 4 = v, 5 = y (x = x0 + M^-1 y).
// Iterations are enqueued in batches of 8 without host round trips; one iteration = two operator applications.
static int op_apply_hat(ark_m1* h, const double* vin, double* vout, const int* stop)
{
    if (h->precond == 1) {
        int rc = mg_apply(h, vin, h->mgz, stop);
        if (rc) return rc;
        KL(KC_SPMV, 336.0 * h->N, launch_spmv_hat(h->g, h->A.off, h->mgz, vout, nullptr, nullptr, 1.0, stop, h->st));
        return 0;
    }
    if (opk(h) == 1)
        KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, vin, vout, nullptr, nullptr, 1.0, stop, 1, h->sm_count, h->st));
    else
        KL(KC_SPMV, 336.0 * h->N, launch_spmv_hat(h->g, h->A.off, vin, vout, nullptr, nullptr, 1.0, stop, h->st));
    return 0;
}

static int bicgstab_solve(ark_m1* h, double tol, int maxit)
{
    int rc;
    const long long n = 3 * h->N, S = h->stride;
    const int sm = h->sm_count;
    double* x = h->U[h->cur];
    GmresWork W = h->W;
    const int* stop = &W.ctl->inner_stop;
    double *r = h->V, *t = h->V + S, *rh = h->V + 2 * S, *p = h->V + 3 * S, *v = h->V + 4 * S, *y = h->V + 5 * S;
    KL(KC_SMALL, 0.0, launch_begin_solve(W, tol, 1, maxit, h->st));
    KL(KC_DOT, 24.0 * h->N, launch_multi_dot(h->A.b, h->A.b, 0, 1, 0, n, W, DOT_BNORM, sm, h->st));
    CU(cudaMemsetAsync(y, 0, (size_t)n * sizeof(double), h->st));
    if ((rc = true_residual(h, x))) return rc;
    if ((rc = ark_fetch_ctl(h))) return rc;
    while (!h->ctl_host->inner_stop) {
        const int its0 = h->ctl_host->its;
        KL(KC_UPDATE, 96.0 * h->N, launch_bicg_begin(r, rh, p, v, n, W, h->st));
        for (;;) {
            for (int k = 0; k < 8; ++k) {
                KL(KC_UPDATE, 96.0 * h->N, launch_bicg_p(r, p, v, n, W, h->st));
                if (opk(h) == 1) {   // matrix-free operator with the reductions fused in
                    KL(KC_SPMV, (288.0 - mf_saved(h)) * h->N, launch_op_mf_dot(h->g, h->mf, h->A.Minv, p, v, stop, 1, rh, W, sm, h->st));
                    KL(KC_UPDATE, 72.0 * h->N, launch_bicg_s(r, v, n, W, h->st));
                    KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf_dot(h->g, h->mf, h->A.Minv, r, t, stop, 2, nullptr, W, sm, h->st));
                } else {
                    if ((rc = op_apply_hat(h, p, v, stop))) return rc;
                    KL(KC_DOT, 48.0 * h->N, launch_multi_dot(v, rh, S, 1, 0, n, W, BICG_ALPHA, sm, h->st));
                    KL(KC_UPDATE, 72.0 * h->N, launch_bicg_s(r, v, n, W, h->st));
                    if ((rc = op_apply_hat(h, r, t, stop))) return rc;
                    KL(KC_DOT, 72.0 * h->N, launch_multi_dot(t, r, S, 2, 0, n, W, BICG_OMEGA, sm, h->st));
                }
                KL(KC_UPDATE, 168.0 * h->N, launch_bicg_xr(y, p, r, t, rh, n, W, sm, h->st));
            }
            if ((rc = ark_fetch_ctl(h))) return rc;
            if (h->ctl_host->inner_stop) break;
        }
        if (h->precond == 1) {
            if ((rc = mg_apply(h, y, h->mgz, nullptr))) return rc;
            KL(KC_COMBINE, 168.0 * h->N, launch_combine_y(h->g, h->A.Minv, h->mgz, x, h->st));
            CU(cudaMemsetAsync(y, 0, (size_t)n * sizeof(double), h->st));
        } else
            KL(KC_COMBINE, 168.0 * h->N, launch_combine_y(h->g, h->A.Minv, y, x, h->st));
        if ((rc = true_residual(h, x))) return rc;      // resets inner_stop unless converged / out of iterations
        if ((rc = ark_fetch_ctl(h))) return rc;
        if (h->ctl_host->its == its0) break;            // breakdown without progress
    }
    return 0;
}

// History copy, matter update, timings, error mapping shared by the implicit entry points.
int ark_finish_implicit(ark_m1* h, double dt, double* final_residual)
{
    GmresWork W = h->W;
    const GmresCtl c = *h->ctl_host;
    const int nh = c.nhist < W.caphist ? c.nhist : W.caphist;
    h->hist_host->assign((size_t)nh, 0.0);
    if (nh > 0) CU(cudaMemcpyAsync(h->hist_host->data(), W.hist, (size_t)nh * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (h->have_T && !c.nonfinite) {
        KL(KC_SMALL, 40.0 * h->N, launch_matter_update(h->g, h->s, dt, h->sa, h->rho_cv, h->U[h->cur], h->T[h->cur], h->st));
    }
    CU(cudaStreamSynchronize(h->st));
    ark_kflush(h);
    float ms01 = 0, ms12 = 0;
    cudaEventElapsedTime(&ms01, h->ev[0], h->ev[1]); cudaEventElapsedTime(&ms12, h->ev[1], h->ev[2]);
    h->timings[0] = ms01; h->timings[1] = ms12; h->timings[2] = (double)ms01 + ms12;
    if (c.nonfinite) return ark_fail(h, ARK_M1_E_NONFINITE, "step_implicit: non-finite norm in the solver (state or opacity holds NaN/Inf?)%s", "");
    if (final_residual) *final_residual = (c.bnorm > 0.0) ? c.rnorm / c.bnorm : c.rnorm;
    return 0;
}

extern "C" int ark_m1_step_implicit(ark_m1* h, double dt, double tol, int restart, int maxit, double* final_residual)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "ark_m1_step_implicit");
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0) return ark_fail(h, ARK_M1_E_ARG, "step_implicit: need dt > 0, tol > 0, restart >= 1, maxit >= 0%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "step_implicit: no state set%s", "");
    int rc = ark_ensure_implicit(h, (h->krylov == 1 && restart < 5) ? 5 : restart, maxit);
    if (rc) return rc;
    CU(cudaEventRecord(h->ev[0], h->st));
    if ((rc = ark_assemble_system(h, dt, nullptr))) return rc;
    CU(cudaEventRecord(h->ev[1], h->st));
    if ((rc = (h->krylov == 1) ? bicgstab_solve(h, tol, maxit) : (use_cb(h) ? gmres_solve_cb(h, tol, restart, maxit) : gmres_solve(h, tol, restart, maxit)))) return rc;
    CU(cudaEventRecord(h->ev[2], h->st));
    if ((rc = ark_finish_implicit(h, dt, final_residual))) return rc;
    return h->ctl_host->its;
}

// Newton-Raphson on the implicit step.  With the Jacobian of DESIGN.md reading R4 and P homogeneous of
// degree 1 the Newton update J_k (U^{k+1} - U^k) = -(U^k - U^n + dt R(U^k)) equals (I + dt L_{U^k}) U^{k+1} = U^n + affine:
// re-assemble with the coefficients of the iterate, keep U^n on the right-hand side, start GMRES from U^k.
extern "C" int ark_m1_step_implicit_newton(ark_m1* h, double dt, double tol, int restart, int maxit, double newton_tol, int max_newton,
                                           int* newton_iterations, double* final_residual, double* final_update)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "ark_m1_step_implicit_newton");
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0 || !(newton_tol >= 0.0) || max_newton < 1)
        return ark_fail(h, ARK_M1_E_ARG, "step_implicit_newton: need dt > 0, tol > 0, restart >= 1, maxit >= 0, newton_tol >= 0, max_newton >= 1%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "step_implicit_newton: no state set%s", "");
    int rc = ark_ensure_implicit(h, (h->krylov == 1 && restart < 5) ? 5 : restart, maxit);
    if (rc) return rc;
    const size_t n = 3 * (size_t)h->N;
    if (!h->nprev && (rc = ark_dmalloc(h, (void**)&h->nprev, n * sizeof(double)))) return rc;
    double* x = h->U[h->cur];
    double* base = h->U[h->cur ^ 1];                 // U^n lives in the other state buffer during the iteration
    CU(cudaMemcpyAsync(base, x, n * sizeof(double), cudaMemcpyDeviceToDevice, h->st));
    CU(cudaEventRecord(h->ev[0], h->st));
    CU(cudaEventRecord(h->ev[1], h->st));
    int total = 0, k = 0;
    double upd = 0.0;
    for (k = 0; k < max_newton; ++k) {
        CU(cudaMemcpyAsync(h->nprev, x, n * sizeof(double), cudaMemcpyDeviceToDevice, h->st));
        if ((rc = ark_assemble_system(h, dt, base))) return rc;
        if ((rc = (h->krylov == 1) ? bicgstab_solve(h, tol, maxit) : (use_cb(h) ? gmres_solve_cb(h, tol, restart, maxit) : gmres_solve(h, tol, restart, maxit)))) return rc;
        total += h->ctl_host->its;
        if (h->ctl_host->nonfinite) break;
        KL(KC_SMALL, 72.0 * h->N, launch_sub(h->nprev, x, h->nprev, (long long)n, h->st));
        KL(KC_DOT, 24.0 * h->N, launch_multi_dot(h->nprev, h->nprev, 0, 1, 0, (long long)n, h->W, DOT_AUX0, h->sm_count, h->st));
        KL(KC_DOT, 24.0 * h->N, launch_multi_dot(x, x, 0, 1, 0, (long long)n, h->W, DOT_AUX1, h->sm_count, h->st));
        if ((rc = ark_fetch_ctl(h))) return rc;
        const double d = h->ctl_host->aux[0], nrm = h->ctl_host->aux[1];
        upd = (nrm > 0.0) ? d / nrm : d;
        if (upd <= newton_tol) { ++k; break; }
    }
    CU(cudaEventRecord(h->ev[2], h->st));
    if ((rc = ark_finish_implicit(h, dt, final_residual))) return rc;
    if (newton_iterations) *newton_iterations = k;
    if (final_update) *final_update = upd;
    return total;
}

// Semi-implicit step: explicit flux step without sources, then the source-only linear system (the assembled
// implicit system with its flux terms switched off; it depends on the opacities only).
extern "C" int ark_m1_step_semi_implicit(ark_m1* h, double dt, double tol, int restart, int maxit, double* final_residual)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "ark_m1_step_semi_implicit");
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0) return ark_fail(h, ARK_M1_E_ARG, "step_semi_implicit: need dt > 0, tol > 0, restart >= 1, maxit >= 0%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "step_semi_implicit: no state set%s", "");
    if (h->N >= (1LL << 31)) return ark_fail(h, ARK_M1_E_UNSUPPORTED, "step_semi_implicit: grid too large for the marching kernels%s", "");
    {   // U* = U^n - dt div(flux): marching kernel with the sources off (T untouched)
        h->s.src_off = 1;
        const Fields f = ark_fields_of(h);
        double* O = h->U[h->cur ^ 1];
        ark_kmark(h, KC_EXPLICIT, 64.0 * h->N);
        cudaError_t e = (h->explicit_kernel == 3)
            ? launch_explicit_march3(h->g, h->s, f, dt, O, O + h->N, O + 2 * h->N, nullptr, h->sm_count, h->st)
            : launch_explicit_march(h->g, h->s, f, dt, O, O + h->N, O + 2 * h->N, nullptr, h->sm_count, h->st);
        h->s.src_off = 0;
        if (e != cudaSuccess) return ark_fail(h, ARK_M1_E_CUDA, "launch_explicit_march: %s", cudaGetErrorString(e));
        if (h->have_T) CU(cudaMemcpyAsync(h->T[h->cur ^ 1], h->T[h->cur], (size_t)h->N * sizeof(double), cudaMemcpyDeviceToDevice, h->st));
        h->cur ^= 1;
    }
    h->s.hyp_off = 1;
    const int rc = ark_m1_step_implicit(h, dt, tol, restart, maxit, final_residual);
    h->s.hyp_off = 0;
    return rc;
}

extern "C" int ark_m1_apply_operator(ark_m1* h, double dt, const double* Vin, double* out, double* b_out)
{
    if (!h || !Vin || !out) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "ark_m1_apply_operator");
    if (!(dt > 0.0)) return ark_fail(h, ARK_M1_E_ARG, "apply_operator: dt must be > 0%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "apply_operator: no state set%s", "");
    int rc = ark_ensure_implicit(h, 1, 1);
    if (rc) return rc;
    const size_t n = 3 * (size_t)h->N;
    if ((rc = ark_assemble_system(h, dt, nullptr))) return rc;
    double* vin = h->V;                       // slot 0 as staging for the input, slot 1 for the output
    double* vout = h->V + h->stride;
    CU(cudaMemcpyAsync(vin, Vin, n * sizeof(double), cudaMemcpyDefault, h->st));
    if (opk(h) == 1) {
        if (h->apply_precond) KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, vin, vout, nullptr, nullptr, 1.0, nullptr, 1, h->sm_count, h->st));
        else KL(KC_SPMV, 192.0 * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, vin, vout, nullptr, nullptr, 1.0, nullptr, 0, h->sm_count, h->st));
    } else {
        KL(KC_DIAGMUL, 120.0 * h->N, launch_diag_mul(h->g, h->A.C, vin, h->tvec, h->st));
        KL(KC_SPMV, 336.0 * h->N, launch_spmv_hat(h->g, h->A.off, h->tvec, vout, nullptr, nullptr, 1.0, nullptr, h->st));
    }
    CU(cudaMemcpyAsync(out, vout, n * sizeof(double), cudaMemcpyDefault, h->st));
    if (b_out) CU(cudaMemcpyAsync(b_out, h->A.b, n * sizeof(double), cudaMemcpyDefault, h->st));
    CU(cudaStreamSynchronize(h->st));
    return 0;
}

// out1 = A M^-1 V - theta1 V, out2 = A M^-1 out1 - theta2 out1: the two-application kernel of the s-step block where it applies
// (matrix-free operator with J and the block rebuilt, grid of at least 4 x 4 cells, option "op_pair" 1), else two single applications.
// Returns 1 if the fused kernel ran, 0 if not.
extern "C" int ark_m1_apply_operator_pair(ark_m1* h, double dt, const double* Vin, double* out1, double* out2, double theta1, double theta2)
{
    if (!h || !Vin || !out1 || !out2) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "ark_m1_apply_operator_pair");
    if (!(dt > 0.0)) return ark_fail(h, ARK_M1_E_ARG, "apply_operator_pair: dt must be > 0%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "apply_operator_pair: no state set%s", "");
    if (opk(h) != 1) return ark_fail(h, ARK_M1_E_UNSUPPORTED, "apply_operator_pair: the matrix-free operator only (option operator = 1)%s", "");
    int rc = ark_ensure_implicit(h, 1, 2);
    if (rc) return rc;
    const size_t n = 3 * (size_t)h->N;
    if ((rc = ark_assemble_system(h, dt, nullptr))) return rc;
    double* vin = h->V;
    double* v1 = h->V + h->stride;
    double* v2 = h->V + 2 * h->stride;
    CU(cudaMemcpyAsync(vin, Vin, n * sizeof(double), cudaMemcpyDefault, h->st));
    const int fused = h->op_pair && op_mf2_ok(h->g, h->mf);
    if (fused) KL(KC_SPMV, 160.0 * h->N, launch_op_mf2(h->g, h->mf, h->A.Minv, vin, v1, v2, nullptr, nullptr, h->sm_count, h->st, theta1, theta2));
    else {
        KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, vin, v1, nullptr, nullptr, 1.0, nullptr, 1, h->sm_count, h->st, theta1));
        KL(KC_SPMV, (264.0 - mf_saved(h)) * h->N, launch_op_mf(h->g, h->mf, h->A.Minv, v1, v2, nullptr, nullptr, 1.0, nullptr, 1, h->sm_count, h->st, theta2));
    }
    CU(cudaMemcpyAsync(out1, v1, n * sizeof(double), cudaMemcpyDefault, h->st));
    CU(cudaMemcpyAsync(out2, v2, n * sizeof(double), cudaMemcpyDefault, h->st));
    CU(cudaStreamSynchronize(h->st));
    return fused;
}

// out = M^-1 V with the right preconditioner the solver would use for a step dt: the inverse 3x3 diagonal blocks
// (block-Jacobi) or D^-1 times one multigrid V-cycle ("preconditioner" = 1).
extern "C" int ark_m1_apply_preconditioner(ark_m1* h, double dt, const double* Vin, double* out)
{
    if (!h || !Vin || !out) return ARK_M1_E_ARG;
    GUARD(h);
    NO_SLAB(h, "ark_m1_apply_preconditioner");
    if (!(dt > 0.0)) return ark_fail(h, ARK_M1_E_ARG, "apply_preconditioner: dt must be > 0%s", "");
    if (!h->have_state) return ark_fail(h, ARK_M1_E_NOTSET, "apply_preconditioner: no state set%s", "");
    int rc = ark_ensure_implicit(h, 1, 1);
    if (rc) return rc;
    const size_t n = 3 * (size_t)h->N;
    if ((rc = ark_assemble_system(h, dt, nullptr))) return rc;
    double* vin = h->V;
    double* vout = h->V + h->stride;
    CU(cudaMemcpyAsync(vin, Vin, n * sizeof(double), cudaMemcpyDefault, h->st));
    CU(cudaMemsetAsync(vout, 0, n * sizeof(double), h->st));
    if (h->precond == 1) {
        if ((rc = mg_apply(h, vin, h->mgz, nullptr))) return rc;
        KL(KC_COMBINE, 168.0 * h->N, launch_combine_y(h->g, h->A.Minv, h->mgz, vout, h->st));
    } else {
        KL(KC_COMBINE, 168.0 * h->N, launch_combine_y(h->g, h->A.Minv, vin, vout, h->st));
    }
    CU(cudaMemcpyAsync(out, vout, n * sizeof(double), cudaMemcpyDefault, h->st));
    CU(cudaStreamSynchronize(h->st));
    ark_kflush(h);
    return 0;
}

extern "C" int ark_m1_get_history(ark_m1* h, double* buf, int cap)
{
    if (!h) return ARK_M1_E_ARG;
    GUARD(h);
    const int n = (int)h->hist_host->size();
    if (buf) for (int k = 0; k < n && k < cap; ++k) buf[k] = (*h->hist_host)[k];
    return n;
}

extern "C" int ark_m1_get_timings(ark_m1* h, double* out3)
{
    if (!h || !out3) return ARK_M1_E_ARG;
    GUARD(h);
    for (int k = 0; k < 3; ++k) out3[k] = h->timings[k];
    return 0;
}

// Per-kernel-class statistics since "kernel_timing" was switched on: out[3*k + 0..2] = launches, milliseconds,
// algorithmic bytes of class k (k < ark_m1_kernel_classes()).  Synchronises.
extern "C" int ark_m1_get_kernel_stats(ark_m1* h, double* out, int cap)
{
    if (!h || !out) return ARK_M1_E_ARG;
    GUARD(h);
    ark_kflush(h);
    for (int k = 0; k < KC_COUNT && 3 * k + 2 < cap; ++k) for (int q = 0; q < 3; ++q) out[3 * k + q] = h->kstat[k][q];
    return KC_COUNT;
}
extern "C" const char* ark_m1_kernel_class_name(int k) { return (k >= 0 && k < KC_COUNT) ? kc_names[k] : ""; }
extern "C" long long ark_m1_kernel_launches(const ark_m1* h) { return h ? h->launches : 0; }

extern "C" int ark_m1_block_stats(const ark_m1* h, long long* out4)
{
    if (!h || !out4) return ARK_M1_E_ARG;
    for (int k = 0; k < 4; ++k) out4[k] = h->ctl_host ? h->ctl_host->blk_stat[k] : 0;
    return ARK_M1_OK;
}

// Self-test of the fast reciprocal / reciprocal square root used by the hot kernels: max relative errors against the IEEE
// sequences over n samples in 200 binades.  No handle needed.  Returns 0 or ARK_M1_E_CUDA.
extern "C" int ark_m1_fastmath_errors(int n, double* out4)
{
    if (!out4 || n < 1) return ARK_M1_E_ARG;
    double* d = nullptr;
    if (cudaMalloc((void**)&d, 4 * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return ARK_M1_E_ALLOC; }
    cudaError_t e = cudaMemset(d, 0, 4 * sizeof(double));
    if (e == cudaSuccess) e = launch_fastmath_selftest(n, d, 0);
    if (e == cudaSuccess) e = cudaMemcpy(out4, d, 4 * sizeof(double), cudaMemcpyDeviceToHost);
    cudaFree(d);
    return e == cudaSuccess ? 0 : ARK_M1_E_CUDA;
}
