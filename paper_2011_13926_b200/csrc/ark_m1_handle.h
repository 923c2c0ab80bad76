// ark_m1_handle.h — the solver handle and the host helpers shared by ark_m1_api.cu (one GPU) and dist.cu (slab decomposition).
#pragma once
#include <cuda_runtime.h>
#include <stdio.h>
#include <map>
#include <vector>

#include "../../include/ark_m1.h"
#include "ark_m1_internal.h"

using namespace ark;

// kernel classes for the launch statistics
enum { KC_EXPLICIT = 0, KC_ASSEMBLE, KC_SCALE, KC_DIAGMUL, KC_SPMV, KC_DOT, KC_UPDATE, KC_COMBINE, KC_SMALL, KC_MG, KC_MGSETUP, KC_COUNT };
static const char* const kc_names[KC_COUNT] __attribute__((unused)) = { "explicit", "assemble", "scale_offdiag", "diag_mul", "spmv_hat", "multi_dot",
                                                 "update_norm", "combine", "small", "mg_vcycle", "mg_setup" };

struct ark_m1 {
    Grid g;
    Scheme s;
    cudaStream_t st;
    int device, sm_count;
    long long N;
    long long bytes;
    std::map<void*, size_t>* allocs;   // device allocations counted in `bytes`
    bool have_state, have_T;
    // state: two buffers of 3N doubles [E | Fx | Fy]; U[cur] is current
    double* U[2];
    int cur;
    double *sa, *ss_tmp, *stot, *T[2];
    double* gh[4][5];
    double *rho_cv, *ux, *uy, *source_E;
    unsigned long long* counts;   // 2
    // options
    int ortho, explicit_kernel, op_kind, maxv, krylov, asm_kernel;
    int arnoldi_block; // 2 (default): GMRES builds two Arnoldi columns per pass over the basis (gmres_solve); 1: one
    int op_pair;       // 1 (default): inside an s-step block two operator applications go through ONE pass where the grid allows (op_mf_rc2_kernel)
    int apply_precond; // 1: ark_m1_apply_operator returns A M^-1 V through the solver's preconditioned matrix-free kernel (matrix-free operator only)
    int op_recompute;  // 1 (default): the matrix-free operator rebuilds the diagonal block instead of loading M^-1 (MfPlanes::rc)
    int basis_prec;    // 64, or 32: compressed-basis GMRES (krylov_cb.cu); applies to GMRES + block-Jacobi + matrix-free operator
    float* V32;        // (m32_alloc + 1) basis vectors of `stride` floats
    double* wk;        // 3N: the fp64 work vector of the compressed-basis path
    int m32_alloc, vslots;
    int precond;       // 0: 3x3 block-Jacobi, 1: multigrid V-cycle (forces the assembled block-stencil operator)
    MgHier mg;         // hierarchy (levels >= 1 allocated lazily)
    double* mgz;       // 3N: V-cycle output (hat variable)
    double mg_cells;   // sum over levels of cells / N (for the byte counts)
    // implicit workspace (lazy)
    BlockMatrix A;
    MfPlanes mf;       // matrix-free coefficient planes (op_kind == 1)
    double* V;         // (m+1) vectors of `stride` doubles
    double* tvec;      // 3N
    double* nprev;     // 3N, previous Newton iterate (lazy)
    long long stride;
    int m_alloc, maxit_alloc;
    GmresWork W;
    void* wblock;      // allocation behind W
    GmresCtl* ctl_host;  // pinned
    std::vector<double>* hist_host;
    cudaEvent_t ev[3];
    double timings[3];
    // per-kernel-class timing (option "kernel_timing"): one event before every launch + one at the end
    int ktiming;
    std::vector<cudaEvent_t>* kev;
    std::vector<int>* kcls;
    std::vector<double>* kbytes;
    size_t kused;
    double kstat[KC_COUNT][3];   // launches, milliseconds, algorithmic bytes
    // slab decomposition (dist.cu): the handle is one slab of an ark_m1_group; y sides marked BC_HALO take their ghost lines from
    // halo_state (E, Fx, Fy, sigma_a, sigma_t of the neighbour's boundary row) and the operator's ghost rows from halo_zp
    int in_group;
    double* halo_state[2];       // [5][nx]: row below (0) / above (1) the slab
    double* halo_zp[2];          // [6][nx]: (z, c^2 J z) of the same rows, refreshed before every operator application
    long long launches;          // kernels launched by this handle
    void* pipe;                  // overlapped state transfers (pipeline.cu): copy stream, staging and snapshot buffers; null until first used
    char err[512];
};


// ---- host helpers defined in ark_m1_api.cu ---------------------------------------------------------------------------
struct DeviceGuard {      // makes the handle's device current for the duration of an entry point
    int prev;
    bool switched;
    explicit DeviceGuard(int dev);
    ~DeviceGuard();
};
#define GUARD(h) DeviceGuard guard__((h)->device)

int ark_fail(ark_m1* h, int code, const char* fmt, const char* detail);
#define CU(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return ark_fail(h, ARK_M1_E_CUDA, #call ": %s", cudaGetErrorString(e__)); } while (0)
void ark_kmark(ark_m1* h, int cls, double bytes);      // statistics: start of a launch of class cls moving `bytes`
void ark_kflush(ark_m1* h);
#define KL(cls, bytes, call) do { ark_kmark(h, (cls), (double)(bytes)); CU(call); } while (0)
int ark_dmalloc(ark_m1* h, void** p, size_t bytes);
void ark_dfree(ark_m1* h, void* p);
ark::Fields ark_fields_of(const ark_m1* h);
int ark_ensure_implicit(ark_m1* h, int m, int maxit);
int ark_assemble_system(ark_m1* h, double dt, const double* bsrc);
int ark_fetch_ctl(ark_m1* h);
int ark_finish_implicit(ark_m1* h, double dt, double* final_residual);
int ark_explicit_once(ark_m1* h, double dt);
void ark_pipe_free(ark_m1* h);      // pipeline.cu
