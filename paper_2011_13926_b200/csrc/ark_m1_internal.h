// ark_m1_internal.h — handle layout and kernel launchers shared by the .cu files of libark_m1.so.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "m1_device.cuh"

namespace ark {

// ---------------------------------------------------------------------------------------------------------
// Device-resident control block of one GMRES solve.  Every Krylov kernel reads it; the "last block done"
// epilogues of the reduction kernels update it, so that a whole restart cycle is enqueued without a host
// round trip.
// ---------------------------------------------------------------------------------------------------------
struct GmresCtl {
    double bnorm, target, rnorm;   // ||b||, tol*||b||, last TRUE residual norm
    double est;                    // last residual estimate |g_{j+1}|
    int m, maxit;
    int its;                       // inner iterations so far (all cycles)
    int j;                         // inner iterations in the current cycle
    int inner_stop;                // 1: skip the remaining inner kernels of this cycle
    int converged;                 // 1: true residual <= target
    int nonfinite;                 // 1: a norm was NaN/Inf
    int nhist;
    unsigned int ticket;           // "last block" counter of the reduction kernels
    int pad;
    double aux[2];                 // scratch norms (Newton update size)
    double bs[8];                  // BiCGStab scalars: rho, alpha, omega, rho_new, ||r|| (recursive), flag "restart after this iteration"
    double blk[8];                 // two-column Arnoldi step: r11 = ||W1'||, <W1', W2'>, <W1', W1'>; s-step block: [3] accepted columns, [4] refine flag,
                                   // [5] in-block solve predicted by the dot pass (applied by the update pass), [6] block finished by the update pass
    double gram[25];               // s-step block: W^T W from the dot pass (the block's own slots dotted like basis vectors)
    int blk_stat[4];               // s-step blocks of this solve: finished in the update pass / predicted, then refined / classic / classic, refined
};

struct GmresWork {                 // device pointers into one small allocation
    GmresCtl* ctl;
    double* H;      // (m+1) x m, row-major H[i*m + j]
    double* cs;     // m
    double* sn;     // m
    double* g;      // m+1
    double* y;      // m
    double* scale;  // m+1 : v_i = scale[i] * V_i (basis stored unnormalised)
    double* coef;   // m+1 : coefficients of the pending update / combination
    double* hist;   // caphist
    double* partial;// [max_blocks][MAXV] block partial sums
    int caphist;
    double* Hraw;   // (m+1) x m: the Arnoldi columns before the Givens rotations (two-column step only; may be null)
    double* c1;     // m+1 : <W1, v_i> of the two-column step
    double* c2;     // m+1 : <W2, v_i>
    double* coef2;  // m+1 : coefficients of the second vector's update
    // s-step Arnoldi block (krylov_sstep.cu), SB = 3..5 columns per pass over the basis; ld = m + 1
    double* cS;     // SMAX x ld : C_{i,k} = <W_{k+1}, v_i>
    double* coefS;  // SMAX x ld : C_{i,k} scale_i, the update coefficients
    double* Rb;     // SMAX x SMAX: T, the unit upper-triangular factor applied so far in the block (W' = Q~ T; T = T2 T1 after a refinement round)
    double* tb;     // SMAX x SMAX: t_{l,k} = R_{l,k} / R_{l,l} of the current round's Cholesky factor, the coefficients of the in-block solve
    double* partialS;// [gs blocks][SMAX * 32]: block partial sums of the s-step dot kernel
    double* red_out;// null: the reduction kernels run their scalar epilogue themselves (one GPU).  Non-null (slab decomposition):
                    // they store this rank's sums here instead; all-reduce and launch_epilogue follow
};

enum { MAXV = 16 };                // basis vectors handled per pass of the multi-vector kernels (the measured optimum: DESIGN.md section 5)

enum DotMode { DOT_BNORM = 0, DOT_RNORM = 1, DOT_H = 2, DOT_H2 = 3, DOT_UPD = 4, DOT_NONE = 5, DOT_AUX0 = 6, DOT_AUX1 = 7,
               BICG_ALPHA = 8, BICG_OMEGA = 9, BICG_RHO = 10,
               DOT_B2 = 11,      // two-column step: <W1, V_i>, <W2, V_i> of a chunk
               UPD_B2A = 12,     // ... first column finished: <W1', W1'>, <W1', W2'>
               UPD_B2B = 13 };   // ... second column finished: ||W2''||^2
enum { SMAX = 5 };                // columns per s-step Arnoldi block (Gram matrix of SMAX (SMAX + 1) / 2 <= MAXV sums)
enum { BS_RHO = 0, BS_ALPHA = 1, BS_OMEGA = 2, BS_RHO_NEW = 3, BS_RN = 4, BS_RESTART = 5 };

// number of SMs of the CURRENT device (cached per device; ark_m1_api.cu) — grid sizes are multiples of it
int current_sm_count();

// ---------------------------------------------------------------------------------------------------------
// Launchers (each enqueues on `st`, returns cudaGetLastError()).
// ---------------------------------------------------------------------------------------------------------
// explicit_kernels.cu
cudaError_t launch_explicit_cell(const Grid& g, const Scheme& s, const Fields& f, double dt, int mode,
                                 double* outE, double* outFx, double* outFy, double* outT, cudaStream_t st);
cudaError_t launch_explicit_march(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                  double* outE, double* outFx, double* outFy, double* outT, int sm_count, cudaStream_t st);
cudaError_t launch_explicit_march3(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                   double* outE, double* outFx, double* outFy, double* outT, int sm_count, cudaStream_t st);
cudaError_t launch_velocity_sources(const Grid& g, const Scheme& s, const Fields& f, const double* ux, const double* uy,
                                    double dt, double* E, double* Fx, double* Fy, cudaStream_t st);
cudaError_t launch_count_unrealizable(const Grid& g, const Fields& f, unsigned long long* counts2, cudaStream_t st);
cudaError_t launch_fastmath_selftest(int n, double* out3, cudaStream_t st);
cudaError_t launch_add_planes(double* st_out, const double* a, const double* b, long long n, cudaStream_t st);   // st_out may be b

// implicit_kernels.cu
struct BlockMatrix {      // SoA planes of N doubles each
    double* off;          // 36 planes: block k in {W,E,S,N}, entry (r,c): plane k*9 + r*3 + c   (A_k M_nbr^-1 after scaling)
    double* C;            // 9 planes: diagonal block
    double* Minv;         // 9 planes: inverse of the diagonal block
    double* b;            // 3 planes: right-hand side
};
// Matrix-free operator storage (option "operator" = 1): coefficient planes instead of assembled blocks.
struct MfPlanes {
    double* J;     // 9 planes: dP_ab/dU of the cell, rows xx, xy, yy
    double* fE;    // 4 planes: a+, Lambda, alpha, c dt sigma_f/4 of the EAST face of the cell
    double* fN;    // 4 planes: the same for the NORTH face
    double* dE;    // 1 plane : c dt sigma_a eta
    double* dF;    // 1 plane : c dt sigma_t when the source is cell-centred (Eq. 16), 0 with the WB source
    double* xlo;   // [4][ny] : west face of column 0 (non-periodic x)
    double* ylo;   // [4][nx] : south face of row 0 (non-periodic y)
    double rx, ry; // dt/dx, dt/dy of the assembled step
    const double* halo[2];   // slab decomposition (BC_HALO sides): received (z, c^2 J z) of the row below / above, [6][nx] each
    double* fxy;   // 2 planes: reduced flux (fx, fy) of the cell; fx = 4 marks a cell whose J is not the M1 closure's (clamped)
    int rc;        // 1: the preconditioned operator rebuilds the diagonal block from J and the faces instead of loading M^-1 (operator_mf.cu)
    int rcj;       // 1 (with rc): it also rebuilds J from (fx, fy) instead of loading its nine planes (default scheme, marching assembly)
    int has_dF;    // 0: dF is identically zero (WB source) and is not loaded
};
// A.off / A.C may be null when mf.J is set (then only Minv, b and the coefficient planes are written)
// bsrc: planes [E|Fx|Fy] that supply the U^n part of the right-hand side (null: the state in `f`; non-null in Newton
// iterations, where `f` is the iterate that only supplies the coefficients)
cudaError_t launch_assemble(const Grid& g, const Scheme& s, const Fields& f, double dt, BlockMatrix A, MfPlanes mf,
                            const double* bsrc, cudaStream_t st);
// same outputs for the matrix-free storage from the marching kernel (assemble_march.cu)
cudaError_t launch_assemble_march(const Grid& g, const Scheme& s, const Fields& f, double dt, BlockMatrix A, MfPlanes mf,
                                  const double* bsrc, int sm_count, cudaStream_t st);
// out = sgn * s * (A [M^-1] v) + add, flux form from the coefficient planes; precond = 1 applies M^-1 (Minv) first
// theta: the result is reduced by theta * v (shifted operator for the s-step Krylov basis; 0 = plain)
cudaError_t launch_op_mf(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, double* out,
                         const double* scale_ptr, const double* add, double sgn, const int* skip_flag, int precond,
                         int sm_count, cudaStream_t st, double theta = 0.0);
bool op_mf2_ok(const Grid& g, const MfPlanes& mf);
cudaError_t launch_op_mf2(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, double* out1, double* out2,
                          const double* scale_ptr, const int* skip_flag, int sm_count, cudaStream_t st, double th1, double th2);
// (z, c^2 J z) of the slab's first and last row for the neighbour ranks (out_lo / out_hi: [6][nx], either may be null)
cudaError_t launch_halo_pack_zp(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, int precond,
                                double* out_lo, double* out_hi, const int* skip_flag, cudaStream_t st);
cudaError_t launch_op_mf_f32(const Grid& g, const MfPlanes& mf, const double* Minv, const float* v, double* out,
                             const double* scale_ptr, const int* skip_flag, int sm_count, cudaStream_t st);
cudaError_t launch_scale_offdiag(const Grid& g, BlockMatrix A, float* off32, cudaStream_t st);   // off32: optional fp32 copy
// t = C x
cudaError_t launch_diag_mul(const Grid& g, const double* Cblk, const double* x, double* t, cudaStream_t st);
// out = sgn*(s*(v + sum_k Ahat_k v_nbr)) + (add ? add : 0);  s = *scale_ptr[scale_idx] if scale_ptr else 1
cudaError_t launch_spmv_hat(const Grid& g, const double* off, const double* v, double* out, const double* scale_ptr,
                            const double* add, double sgn, const int* skip_flag, cudaStream_t st);
int op_mf_blocks(const Grid& g, int sm_count);      // grid size of the matrix-free operator (sizes the partial-sum buffer)
cudaError_t launch_op_mf_dot(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, double* out,
                             const int* skip_flag, int dot, const double* aux, GmresWork W, int sm_count, cudaStream_t st);
cudaError_t launch_matter_update(const Grid& g, const Scheme& s, double dt, const double* sa, const double* rho_cv,
                                 const double* Enew, double* T, cudaStream_t st);

// multigrid.cu — V-cycle preconditioner in the block-Jacobi-scaled variable (option "preconditioner" = 1)
#define MG_MAXLEV 24
struct MgLevel {
    Grid g;          // nx, ny of the level; spacing unused; boundary kinds of the fine grid
    double* off;     // 36 planes: scaled neighbour blocks of the level (level 0: the fine A.off)
    float* off32;    // the same in single precision (option "mg_precision" = 32; null otherwise)
    double* Dinv;    // 9 planes: inverse diagonal block of the level's Galerkin operator (level 0: unused)
    double* r;       // 3 planes: restricted residual = right-hand side of the level (level 0: the caller's vector)
    double* e;       // 3 planes: the level's correction Dinv z^ handed to the finer level (level 0: the caller's output)
};
struct MgHier { int nlev; MgLevel lev[MG_MAXLEV]; double omega; int coarse_sweeps; int precision; };
// coarse blocks of one level from the finer one (Galerkin, 2x2 aggregates): writes coff (scaled) and cDinv
cudaError_t launch_mg_galerkin(const Grid& gf, const double* off, const Grid& gc, double* coff, double* cDinv, float* coff32, cudaStream_t st);
cudaError_t launch_mg_to_float(const double* a, float* b, long long n, cudaStream_t st);   // b = (float) a
// zhat_out = one V-cycle on r_in (level-0 vectors of 3N doubles, distinct); *nl = kernels launched
cudaError_t launch_mg_vcycle(const MgHier& H, const double* r_in, double* zhat_out, const int* skip_flag, cudaStream_t st, int* nl);

// krylov_kernels.cu
int  krylov_max_blocks(int sm_count);
// dots of w with nv vectors V0 + k*stride (k < nv) -> epilogue `mode`; col0 = index of the first vector in the basis
cudaError_t launch_multi_dot(const double* w, const double* V0, long long stride, int nv, int col0, long long n,
                             GmresWork W, int mode, int sm_count, cudaStream_t st);
// w -= sum_k coef[col0+k] V_k ; if with_norm: ||w||^2 -> epilogue DOT_UPD
cudaError_t launch_update(double* w, const double* V0, long long stride, int nv, int col0, long long n,
                          GmresWork W, int with_norm, int sm_count, cudaStream_t st, int mode = DOT_UPD);
// the pair kernels of the two-column Arnoldi step: nv <= krylov_pair_max_vectors() basis vectors per pass
int krylov_pair_max_vectors();
cudaError_t launch_multi_dot2(const double* w1, const double* w2, const double* V0, long long stride, int nv, int col0, long long n,
                              GmresWork W, int sm_count, cudaStream_t st);
cudaError_t launch_update2_all(double* w1, double* w2, const double* V0, long long stride, int nv, long long n, GmresWork W, int sm_count, cudaStream_t st);
// krylov_sstep.cu — the s-step Arnoldi block: sb = 3..SMAX vectors W_1..W_sb in consecutive slots w1, w1 + stride, ...
int sstep_partial_doubles(int sm_count);
// C_{i,k} = <W_{k+1}, V_i> scale_i for nv <= 32 basis vectors starting at index col0 (V0 = their first slot)
cudaError_t launch_dotS(const double* w1, const double* V0, long long stride, int sb, int nv, int col0, long long n, GmresWork W, int sm_count, cudaStream_t st,
                        int jpred = -1);
// W_k -= sum_i coefS_{i,k} V_i over all nv basis vectors; Gram matrix of the result -> Cholesky, first column of the block finished
cudaError_t launch_updateS(double* w1, const double* V0, long long stride, int sb, int nv, long long n, GmresWork W, int sm_count, cudaStream_t st,
                           double theta = 1.0);
// in-block triangular solve with the Cholesky coefficients, norms of the results -> columns 2..sb of the block finished (theta = shift)
// round 1 follows the update pass; round 2 (after launch_gramS) runs only when the block was flagged ill-conditioned (refinement)
cudaError_t launch_qrS(double* w1, long long stride, int sb, long long n, GmresWork W, double theta, int round, int sm_count, cudaStream_t st);
// Gram matrix of the block after round 1, second Cholesky factor (returns at once unless the block was flagged for refinement)
cudaError_t launch_gramS(const double* w1, long long stride, int sb, long long n, GmresWork W, int sm_count, cudaStream_t st);
// slab decomposition: with W.red_out set the four kernels above leave this rank's sums there (dots: [sb][m + 1] raw sums); after the
// all-reduce, the epilogue of step `which` (0 dots, 1 update pass, 2 in-block solve of `round`, 3 second-round Gram matrix) on `red`
cudaError_t launch_sstep_epilogue(GmresWork W, int which, int sb, int nv, const double* red, double theta, int round, cudaStream_t st);
// the whole inner orthogonalisation step for index j decided on the device (j = ctl->j): see krylov_kernels.cu
cudaError_t launch_solve_y(GmresWork W, cudaStream_t st);
// the scalar epilogue of reduction `mode` on nv sums d[0..nv) (device; after an all-reduce over the ranks)
cudaError_t launch_epilogue(GmresWork W, int mode, int nv, int col0, const double* d, const int* skip_flag, cudaStream_t st);
// x += Minv * (sum_{k<ctl->j} coef[k] V_k)  per cell;  Minv == nullptr: x = sum_{k<ctl->j} coef[k] V_k
cudaError_t launch_combine(const Grid& g, const double* V, long long stride, const double* Minv, double* x,
                           GmresWork W, int sm_count, cudaStream_t st);
// compressed-basis GMRES (krylov_cb.cu): basis vectors stored in single precision, fp64 arithmetic; nv <= 16
cudaError_t launch_multi_dot32(const double* w, const float* V0, long long stride, int nv, int col0, long long n,
                               GmresWork W, int mode, int sm_count, cudaStream_t st);
cudaError_t launch_update32(double* w, const float* V0, long long stride, int nv, int col0, long long n, GmresWork W,
                            int with_norm, int write_w, float* out32, int sm_count, cudaStream_t st);
cudaError_t launch_combine32(const Grid& g, const float* V, long long stride, const double* Minv, double* x,
                             GmresWork W, int sm_count, cudaStream_t st);
// BiCGStab vector kernels (krylov_kernels.cu); every one returns at once when ctl->inner_stop is set
cudaError_t launch_bicg_begin(double* r, double* rhat, double* p, double* v, long long n, GmresWork W, cudaStream_t st);
cudaError_t launch_bicg_p(const double* r, double* p, const double* v, long long n, GmresWork W, cudaStream_t st);      // p = r + beta (p - omega v)
cudaError_t launch_bicg_s(double* r, const double* v, long long n, GmresWork W, cudaStream_t st);                        // r -= alpha v
cudaError_t launch_bicg_xr(double* y, const double* p, double* r, const double* t, const double* rhat, long long n,
                           GmresWork W, int sm_count, cudaStream_t st);   // y += alpha p + omega r; r -= omega t; rho, ||r||
cudaError_t launch_combine_y(const Grid& g, const double* Minv, double* y, double* x, cudaStream_t st);                  // x += M^-1 y; y = 0
cudaError_t launch_sub(double* out, const double* a, const double* b, long long n, cudaStream_t st);   // out = a - b (out may be a or b)
cudaError_t launch_begin_solve(GmresWork W, double tol, int m, int maxit, cudaStream_t st);

}  // namespace ark
