// krylov_kernels.cu — row a6: the vector kernels of restarted GMRES(m) with right block-Jacobi preconditioning
// (Krylov solve of the linearised system, "solve A K^-1 y = b and then K x = y").
//
// Design:
//  * The Arnoldi basis is stored UNNORMALISED: v_i = scale[i] * V_i.  The operator, the dots and the updates
//    carry scale[i] as a scalar, so no pass over memory is spent on normalisation.
//  * Orthogonalisation = one-pass classical Gram-Schmidt: one multi-dot kernel (w read once against up to MAXV
//    basis vectors per pass) and one multi-axpy kernel fused with the norm of the result (CGS2 optional).
//  * Reductions are deterministic: block partial sums -> fixed-order final sum by the last block to finish
//    (ticket counter), whose thread 0 then runs the scalar epilogue (Hessenberg column, Givens rotations,
//    residual estimate, stop flag) on the device.  A whole restart cycle is enqueued without host round trips;
//    kernels of a cycle that has already met its stop criterion return immediately (ctl->inner_stop).
#include "krylov_device.cuh"

namespace ark {

int krylov_max_blocks(int sm_count) { return sm_count * 4; }

// ---------------------------------------------------------------------------------------------------------
// The two streaming kernels of the orthogonalisation.  Both are pure HBM streams (0.12 DFMA per byte), so the only thing that
// matters is how many bytes each SM keeps in flight — and that must not depend on what ptxas does with a particular NV
// (round 1: register counts between 40 and 166 over the 32 instances, loads serialised in some, 3 of the 4 blocks per SM
// resident in others: 4.7-8.4 TB/s).  Shape used here, the same for every instance:
//   * __launch_bounds__(256, 2): 2 blocks per SM always fit (<= 128 registers), grid = 2 x SMs, one wave, no tail;
//   * a trip handles U elements (double2) per thread, U chosen so that (NV + 1) U >= 16: the trip first issues ALL its
//     (NV + 1) U 16-byte loads into register arrays, then does the arithmetic -> 512 threads x >= 16 x 16 B >= 128 KB in
//     flight per SM whatever NV is;
//   * streaming loads (ld.global.cs: the basis is read once per kernel and is far larger than L2).
// ---------------------------------------------------------------------------------------------------------
// (measured at 4096^2 with 2, 3, 4 blocks per SM x 8, 12, 16, 24 loads per trip: 2.889-2.898 ms per GMRES iteration for all of
// them — once every instance keeps > 100 KB per SM in flight the streams sit at what the HBM delivers, 7.6 TB/s read-only and
// 7.0 TB/s with the write stream of the update)
static constexpr int GS_BLOCKS_PER_SM = 2;
__host__ __device__ constexpr int gs_unroll(int nv) { return (nv + 1) >= 16 ? 1 : (16 + nv) / (nv + 1); }   // ceil(16 / (nv + 1))

__device__ __forceinline__ double2 ld_stream(const double2* p) { return __ldcs(p); }

template <int NV>
__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM) multi_dot_kernel(const double* __restrict__ w, const double* __restrict__ V0,
                                                                               long long stride, long long n, GmresWork W, int mode, int col0)
{
    if ((mode == DOT_H || mode == DOT_H2 || mode == BICG_ALPHA || mode == BICG_OMEGA) && W.ctl->inner_stop) return;
    constexpr int U = gs_unroll(NV);
    double acc[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) acc[k] = 0.0;
    const long long n2 = n >> 1, T = (long long)gridDim.x * KTHREADS;
    const double2* w2 = reinterpret_cast<const double2*>(w);
    long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x;
    for (; e + (U - 1) * T < n2; e += U * T) {
        double2 a[U], b[U][NV];
#pragma unroll
        for (int u = 0; u < U; ++u) a[u] = ld_stream(w2 + e + u * T);
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k = 0; k < NV; ++k) b[u][k] = ld_stream(reinterpret_cast<const double2*>(V0 + k * stride) + e + u * T);
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k = 0; k < NV; ++k) acc[k] = fma(a[u].y, b[u][k].y, fma(a[u].x, b[u][k].x, acc[k]));
    }
    for (; e < n2; e += T) {                      // fewer than U elements left for this thread
        const double2 a = w2[e];
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const double2 b = reinterpret_cast<const double2*>(V0 + k * stride)[e];
            acc[k] = fma(a.y, b.y, fma(a.x, b.x, acc[k]));
        }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) acc[k] += w[n - 1] * V0[k * stride + n - 1];
    }
    reduce_and_finish<NV>(acc, W, mode, col0);
}

template <int NV, bool WITH_NORM>
__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM) update_kernel(double* __restrict__ w, const double* __restrict__ V0,
                                                                            long long stride, long long n, GmresWork W, int col0, int mode)
{
    if (W.ctl->inner_stop) return;
    constexpr int U = gs_unroll(NV);
    double cf[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) cf[k] = W.coef[col0 + k];
    double acc[1] = { 0.0 };
    const long long n2 = n >> 1, T = (long long)gridDim.x * KTHREADS;
    double2* w2 = reinterpret_cast<double2*>(w);
    long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x;
    for (; e + (U - 1) * T < n2; e += U * T) {
        double2 a[U], b[U][NV];
#pragma unroll
        for (int u = 0; u < U; ++u) a[u] = ld_stream(w2 + e + u * T);
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k = 0; k < NV; ++k) b[u][k] = ld_stream(reinterpret_cast<const double2*>(V0 + k * stride) + e + u * T);
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int k = 0; k < NV; ++k) { a[u].x = fma(-cf[k], b[u][k].x, a[u].x); a[u].y = fma(-cf[k], b[u][k].y, a[u].y); }
            w2[e + u * T] = a[u];
            if (WITH_NORM) acc[0] = fma(a[u].y, a[u].y, fma(a[u].x, a[u].x, acc[0]));
        }
    }
    for (; e < n2; e += T) {
        double2 a = w2[e];
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const double2 b = reinterpret_cast<const double2*>(V0 + k * stride)[e];
            a.x = fma(-cf[k], b.x, a.x); a.y = fma(-cf[k], b.y, a.y);
        }
        w2[e] = a;
        if (WITH_NORM) acc[0] = fma(a.y, a.y, fma(a.x, a.x, acc[0]));
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        double a = w[n - 1];
#pragma unroll
        for (int k = 0; k < NV; ++k) a -= cf[k] * V0[k * stride + n - 1];
        w[n - 1] = a;
        if (WITH_NORM) acc[0] += a * a;
    }
    if (WITH_NORM) reduce_and_finish<1, KTHREADS, true>(acc, W, mode, 0);
}

// ---------------------------------------------------------------------------------------------------------
// The pair kernels of the two-column Arnoldi step (ark_m1_api.cu gmres_solve):
// W1 = A v_j and W2 = A W1 are orthogonalised against the basis TOGETHER, so the basis is read once per pass for two columns.
// Same in-flight shape as the single-vector kernels: (NV + 2) U >= 16 batched 16-byte loads per trip.
// ---------------------------------------------------------------------------------------------------------
static constexpr int MAXV2 = MAXV / 2;      // basis vectors per pass of the pair kernels (2 MAXV2 sums per block)
__host__ __device__ constexpr int gs_unroll2(int nv) { return (nv + 2) >= 16 ? 1 : (15 + nv + 2) / (nv + 2); }

template <int NV>
__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM) multi_dot2_kernel(const double* __restrict__ w1, const double* __restrict__ w2,
                                                                                const double* __restrict__ V0, long long stride, long long n,
                                                                                GmresWork W, int col0)
{
    if (W.ctl->inner_stop) return;
    constexpr int U = gs_unroll2(NV);
    double acc[2 * NV];
#pragma unroll
    for (int k = 0; k < 2 * NV; ++k) acc[k] = 0.0;
    const long long n2 = n >> 1, T = (long long)gridDim.x * KTHREADS;
    const double2* p1 = reinterpret_cast<const double2*>(w1);
    const double2* p2 = reinterpret_cast<const double2*>(w2);
    long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x;
    for (; e + (U - 1) * T < n2; e += U * T) {
        double2 a1[U], a2[U], b[U][NV];
#pragma unroll
        for (int u = 0; u < U; ++u) { a1[u] = ld_stream(p1 + e + u * T); a2[u] = ld_stream(p2 + e + u * T); }
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k = 0; k < NV; ++k) b[u][k] = ld_stream(reinterpret_cast<const double2*>(V0 + k * stride) + e + u * T);
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k = 0; k < NV; ++k) {
                acc[k] = fma(a1[u].y, b[u][k].y, fma(a1[u].x, b[u][k].x, acc[k]));
                acc[NV + k] = fma(a2[u].y, b[u][k].y, fma(a2[u].x, b[u][k].x, acc[NV + k]));
            }
    }
    for (; e < n2; e += T) {
        const double2 a1 = p1[e], a2 = p2[e];
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const double2 b = reinterpret_cast<const double2*>(V0 + k * stride)[e];
            acc[k] = fma(a1.y, b.y, fma(a1.x, b.x, acc[k]));
            acc[NV + k] = fma(a2.y, b.y, fma(a2.x, b.x, acc[NV + k]));
        }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) { acc[k] += w1[n - 1] * V0[k * stride + n - 1]; acc[NV + k] += w2[n - 1] * V0[k * stride + n - 1]; }
    }
    reduce_and_finish<2 * NV>(acc, W, DOT_B2, col0);
}

// W1 -= sum coef[k] V_k, W2 -= sum coef2[k] V_k over ALL nv <= MAXALL basis vectors in one pass, with <W1', W1'> and <W1', W2'> ->
// epilogue UPD_B2A: W1 and W2 are read and written once per pair of columns (in chunks of 8 vectors the two vectors moved 96 B per
// cell per chunk, up to four times per pair: 74 -> 59 ms of update time per solve at 4096^2).  The
// 2 nv coefficients sit in shared memory as (coef, coef2) pairs (one broadcast LDS.128 per vector); the basis goes through the
// registers in batches of UB vectors x U elements, every batch's loads issued before its arithmetic.
static constexpr int MAXALL = 128;
static constexpr int UB = 8;
template <int NB, int U>
__device__ __forceinline__ void update2_batch(double2 (&a1)[U], double2 (&a2)[U], const double* __restrict__ Vb, long long stride, long long e, long long T,
                                              const double2* __restrict__ cf)
{
    double2 b[U][NB];
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
        for (int k = 0; k < NB; ++k) b[u][k] = ld_stream(reinterpret_cast<const double2*>(Vb + k * stride) + e + u * T);
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        const double2 c = cf[k];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            a1[u].x = fma(-c.x, b[u][k].x, a1[u].x); a1[u].y = fma(-c.x, b[u][k].y, a1[u].y);
            a2[u].x = fma(-c.y, b[u][k].x, a2[u].x); a2[u].y = fma(-c.y, b[u][k].y, a2[u].y);
        }
    }
}

template <int U>
__device__ __forceinline__ void update2_sweep(double2 (&a1)[U], double2 (&a2)[U], const double* __restrict__ V0, long long stride, long long e, long long T,
                                              const double2* __restrict__ cf, int nv)
{
    int k0 = 0;
    for (; k0 + UB <= nv; k0 += UB) update2_batch<UB, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0);
    switch (nv - k0) {
        case 1: update2_batch<1, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0); break;
        case 2: update2_batch<2, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0); break;
        case 3: update2_batch<3, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0); break;
        case 4: update2_batch<4, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0); break;
        case 5: update2_batch<5, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0); break;
        case 6: update2_batch<6, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0); break;
        case 7: update2_batch<7, U>(a1, a2, V0 + k0 * stride, stride, e, T, cf + k0); break;
        default: break;
    }
}

__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM) update2_all_kernel(double* __restrict__ w1, double* __restrict__ w2, const double* __restrict__ V0,
                                                                                 long long stride, long long n, GmresWork W, int nv)
{
    if (W.ctl->inner_stop) return;
    constexpr int U = 2;
    __shared__ double2 cf[MAXALL];
    for (int k = threadIdx.x; k < nv; k += KTHREADS) cf[k] = make_double2(W.coef[k], W.coef2[k]);
    __syncthreads();
    double acc[2] = { 0.0, 0.0 };
    const long long n2 = n >> 1, T = (long long)gridDim.x * KTHREADS;
    double2* p1 = reinterpret_cast<double2*>(w1);
    double2* p2 = reinterpret_cast<double2*>(w2);
    long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x;
    for (; e + (U - 1) * T < n2; e += U * T) {
        double2 a1[U], a2[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { a1[u] = ld_stream(p1 + e + u * T); a2[u] = ld_stream(p2 + e + u * T); }
        update2_sweep<U>(a1, a2, V0, stride, e, T, cf, nv);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            p1[e + u * T] = a1[u]; p2[e + u * T] = a2[u];
            acc[0] = fma(a1[u].y, a1[u].y, fma(a1[u].x, a1[u].x, acc[0]));
            acc[1] = fma(a1[u].y, a2[u].y, fma(a1[u].x, a2[u].x, acc[1]));
        }
    }
    for (; e < n2; e += T) {
        double2 a1[1] = { p1[e] }, a2[1] = { p2[e] };
        update2_sweep<1>(a1, a2, V0, stride, e, T, cf, nv);
        p1[e] = a1[0]; p2[e] = a2[0];
        acc[0] = fma(a1[0].y, a1[0].y, fma(a1[0].x, a1[0].x, acc[0]));
        acc[1] = fma(a1[0].y, a2[0].y, fma(a1[0].x, a2[0].x, acc[1]));
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        double a1 = w1[n - 1], a2 = w2[n - 1];
        for (int k = 0; k < nv; ++k) { a1 -= cf[k].x * V0[k * stride + n - 1]; a2 -= cf[k].y * V0[k * stride + n - 1]; }
        w1[n - 1] = a1; w2[n - 1] = a2;
        acc[0] += a1 * a1; acc[1] += a1 * a2;
    }
    reduce_and_finish<2, KTHREADS, true>(acc, W, UPD_B2A, 0);
}

// grid of the Gram-Schmidt streams: one wave of GS_BLOCKS_PER_SM blocks per SM (fewer on small vectors)
static int gs_grid(long long n, int sm_count)
{
    const long long need = ((n >> 1) + KTHREADS - 1) / KTHREADS;
    const long long cap = (long long)sm_count * GS_BLOCKS_PER_SM;
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

static int grid_for(long long n, int sm_count)
{
    const long long need = ((n >> 1) + KTHREADS - 1) / KTHREADS;
    const long long cap = krylov_max_blocks(sm_count);
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

template <int NV>
static void dot_launch(int grd, const double* w, const double* V0, long long stride, long long n, GmresWork W, int mode,
                       int col0, cudaStream_t st)
{
    multi_dot_kernel<NV><<<grd, KTHREADS, 0, st>>>(w, V0, stride, n, W, mode, col0);
}

cudaError_t launch_multi_dot(const double* w, const double* V0, long long stride, int nv, int col0, long long n,
                             GmresWork W, int mode, int sm_count, cudaStream_t st)
{
    const int grd = gs_grid(n, sm_count);
    switch (nv) {
#define ARK_CASE(K) case K: dot_launch<K>(grd, w, V0, stride, n, W, mode, col0, st); break;
        ARK_CASE(1) ARK_CASE(2) ARK_CASE(3) ARK_CASE(4) ARK_CASE(5) ARK_CASE(6) ARK_CASE(7) ARK_CASE(8)
        ARK_CASE(9) ARK_CASE(10) ARK_CASE(11) ARK_CASE(12) ARK_CASE(13) ARK_CASE(14) ARK_CASE(15) ARK_CASE(16)
#undef ARK_CASE
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

template <int NV>
static void upd_launch(int grd, double* w, const double* V0, long long stride, long long n, GmresWork W, int col0,
                       int with_norm, int mode, cudaStream_t st)
{
    if (with_norm) update_kernel<NV, true><<<grd, KTHREADS, 0, st>>>(w, V0, stride, n, W, col0, mode);
    else update_kernel<NV, false><<<grd, KTHREADS, 0, st>>>(w, V0, stride, n, W, col0, mode);
}

cudaError_t launch_update(double* w, const double* V0, long long stride, int nv, int col0, long long n,
                          GmresWork W, int with_norm, int sm_count, cudaStream_t st, int mode)
{
    const int grd = gs_grid(n, sm_count);
    switch (nv) {
#define ARK_CASE(K) case K: upd_launch<K>(grd, w, V0, stride, n, W, col0, with_norm, mode, st); break;
        ARK_CASE(1) ARK_CASE(2) ARK_CASE(3) ARK_CASE(4) ARK_CASE(5) ARK_CASE(6) ARK_CASE(7) ARK_CASE(8)
        ARK_CASE(9) ARK_CASE(10) ARK_CASE(11) ARK_CASE(12) ARK_CASE(13) ARK_CASE(14) ARK_CASE(15) ARK_CASE(16)
#undef ARK_CASE
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

int krylov_pair_max_vectors() { return MAXV2; }

cudaError_t launch_multi_dot2(const double* w1, const double* w2, const double* V0, long long stride, int nv, int col0, long long n,
                              GmresWork W, int sm_count, cudaStream_t st)
{
    const int grd = gs_grid(n, sm_count);
    switch (nv) {
#define ARK_CASE(K) case K: multi_dot2_kernel<K><<<grd, KTHREADS, 0, st>>>(w1, w2, V0, stride, n, W, col0); break;
        ARK_CASE(1) ARK_CASE(2) ARK_CASE(3) ARK_CASE(4) ARK_CASE(5) ARK_CASE(6) ARK_CASE(7) ARK_CASE(8)
#undef ARK_CASE
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// W1, W2 -= their projections on all nv basis vectors V0 .. V0 + (nv-1) stride, one pass; <W1', W1'>, <W1', W2'> -> epilogue UPD_B2A
cudaError_t launch_update2_all(double* w1, double* w2, const double* V0, long long stride, int nv, long long n, GmresWork W, int sm_count, cudaStream_t st)
{
    if (nv < 1 || nv > MAXALL) return cudaErrorInvalidValue;
    update2_all_kernel<<<gs_grid(n, sm_count), KTHREADS, 0, st>>>(w1, w2, V0, stride, n, W, nv);
    return cudaGetLastError();
}

// Scalar epilogue as a kernel of its own (slab decomposition: the sums were all-reduced over the ranks in between).
__global__ void __launch_bounds__(128) epilogue_kernel(GmresWork W, int mode, int nv, int col0, const double* __restrict__ d, const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    __shared__ double hcol[EPI_MAX + 1], ccs[EPI_MAX], ssn[EPI_MAX], dd[MAXV];
    if (threadIdx.x < nv) dd[threadIdx.x] = d[threadIdx.x];
    bool staged = false;
    if (mode == DOT_UPD) {
        const int j = W.ctl->j, m = W.ctl->m;
        staged = (j < EPI_MAX);
        if (staged) for (int i = threadIdx.x; i <= j; i += blockDim.x) { hcol[i] = W.H[i * m + j]; if (i < j) { ccs[i] = W.cs[i]; ssn[i] = W.sn[i]; } }
    }
    __syncthreads();
    if (threadIdx.x == 0) epilogue(W, mode, dd, nv, col0, staged ? hcol : nullptr, ccs, ssn);
}

cudaError_t launch_epilogue(GmresWork W, int mode, int nv, int col0, const double* d, const int* skip_flag, cudaStream_t st)
{
    epilogue_kernel<<<1, 128, 0, st>>>(W, mode, nv, col0, d, skip_flag);
    return cudaGetLastError();
}

// Cycle end: back substitution H y = g over the ctl->j columns built in this cycle; coef_i = y_i scale_i.
__global__ void solve_y_kernel(GmresWork W)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int jj = W.ctl->j, m = W.ctl->m;
    for (int i = jj - 1; i >= 0; --i) {
        double s = W.g[i];
        for (int k = i + 1; k < jj; ++k) s -= W.H[i * m + k] * W.y[k];
        W.y[i] = s / W.H[i * m + i];
        W.coef[i] = W.y[i] * W.scale[i];
    }
}

cudaError_t launch_solve_y(GmresWork W, cudaStream_t st)
{
    solve_y_kernel<<<1, 32, 0, st>>>(W);
    return cudaGetLastError();
}

// x += M^-1 (V y)  ("K x = y"), per cell.
__global__ void __launch_bounds__(KTHREADS) combine_kernel(long long N, const double* __restrict__ V, long long stride,
                                                           const double* __restrict__ Minv, double* __restrict__ x, GmresWork W)
{
    const int jj = W.ctl->j;
    if (jj == 0 && Minv) return;
    for (long long id = blockIdx.x * (long long)KTHREADS + threadIdx.x; id < N; id += (long long)gridDim.x * KTHREADS) {
        double u0 = 0.0, u1 = 0.0, u2 = 0.0;
#pragma unroll 4
        for (int k = 0; k < jj; ++k) {
            const double cf = W.coef[k];
            const double* v = V + k * stride;
            u0 += cf * v[id]; u1 += cf * v[N + id]; u2 += cf * v[2 * N + id];
        }
        if (!Minv) { x[id] = u0; x[N + id] = u1; x[2 * N + id] = u2; continue; }   // plain combination (multigrid path)
        x[id]         += Minv[0 * N + id] * u0 + Minv[1 * N + id] * u1 + Minv[2 * N + id] * u2;
        x[N + id]     += Minv[3 * N + id] * u0 + Minv[4 * N + id] * u1 + Minv[5 * N + id] * u2;
        x[2 * N + id] += Minv[6 * N + id] * u0 + Minv[7 * N + id] * u1 + Minv[8 * N + id] * u2;
    }
}

cudaError_t launch_combine(const Grid& g, const double* V, long long stride, const double* Minv, double* x,
                           GmresWork W, int sm_count, cudaStream_t st)
{
    const long long N = (long long)g.nx * g.ny;
    const long long need = (N + KTHREADS - 1) / KTHREADS, cap = (long long)sm_count * 8;
    combine_kernel<<<(int)(need < cap ? need : cap), KTHREADS, 0, st>>>(N, V, stride, Minv, x, W);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// BiCGStab (the paper's Krylov method), right-preconditioned on A M^-1 like the GMRES path; the
// solution is accumulated in y (x = x0 + M^-1 y at the end of a cycle).  Scalars live in ctl->bs.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(KTHREADS) bicg_begin_kernel(double* __restrict__ r, double* __restrict__ rhat, double* __restrict__ p,
                                                              double* __restrict__ v, long long n, GmresWork W)
{
    GmresCtl* c = W.ctl;
    if (c->inner_stop) return;
    for (long long k = blockIdx.x * (long long)KTHREADS + threadIdx.x; k < n; k += (long long)gridDim.x * KTHREADS) {
        rhat[k] = r[k]; p[k] = 0.0; v[k] = 0.0;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        c->bs[BS_RHO] = 1.0; c->bs[BS_ALPHA] = 1.0; c->bs[BS_OMEGA] = 1.0;
        c->bs[BS_RHO_NEW] = c->rnorm * c->rnorm;      // <r^, r> with r^ = r
        c->bs[BS_RN] = c->rnorm; c->bs[BS_RESTART] = 0.0;
    }
}

__global__ void __launch_bounds__(KTHREADS) bicg_p_kernel(const double* __restrict__ r, double* __restrict__ p, const double* __restrict__ v,
                                                          long long n, GmresWork W)
{
    const GmresCtl* c = W.ctl;
    if (c->inner_stop) return;
    const double omega = c->bs[BS_OMEGA];
    const double beta = (c->bs[BS_RHO_NEW] / c->bs[BS_RHO]) * (c->bs[BS_ALPHA] / omega);
    const long long n2 = n >> 1;
    const double2* r2 = reinterpret_cast<const double2*>(r); const double2* v2 = reinterpret_cast<const double2*>(v);
    double2* p2 = reinterpret_cast<double2*>(p);
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n2; e += (long long)gridDim.x * KTHREADS) {
        const double2 a = r2[e], b = v2[e]; double2 q = p2[e];
        q.x = fma(beta, fma(-omega, b.x, q.x), a.x); q.y = fma(beta, fma(-omega, b.y, q.y), a.y);
        p2[e] = q;
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) p[n - 1] = r[n - 1] + beta * (p[n - 1] - omega * v[n - 1]);
}

__global__ void __launch_bounds__(KTHREADS) bicg_s_kernel(double* __restrict__ r, const double* __restrict__ v, long long n, GmresWork W)
{
    const GmresCtl* c = W.ctl;
    if (c->inner_stop) return;
    const double alpha = c->bs[BS_ALPHA];
    const long long n2 = n >> 1;
    double2* r2 = reinterpret_cast<double2*>(r); const double2* v2 = reinterpret_cast<const double2*>(v);
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n2; e += (long long)gridDim.x * KTHREADS) {
        double2 a = r2[e]; const double2 b = v2[e];
        a.x = fma(-alpha, b.x, a.x); a.y = fma(-alpha, b.y, a.y);
        r2[e] = a;
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) r[n - 1] -= alpha * v[n - 1];
}

__global__ void __launch_bounds__(KTHREADS) bicg_xr_kernel(double* __restrict__ y, const double* __restrict__ p, double* __restrict__ r,
                                                           const double* __restrict__ t, const double* __restrict__ rhat, long long n, GmresWork W)
{
    const GmresCtl* c = W.ctl;
    if (c->inner_stop) return;
    const double alpha = c->bs[BS_ALPHA], omega = c->bs[BS_OMEGA];
    double acc[2] = { 0.0, 0.0 };
    const long long n2 = n >> 1;
    double2* y2 = reinterpret_cast<double2*>(y); double2* r2 = reinterpret_cast<double2*>(r);
    const double2* p2 = reinterpret_cast<const double2*>(p); const double2* t2 = reinterpret_cast<const double2*>(t);
    const double2* h2 = reinterpret_cast<const double2*>(rhat);
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n2; e += (long long)gridDim.x * KTHREADS) {
        double2 yy = y2[e], s = r2[e]; const double2 pp = p2[e], tt = t2[e], hh = h2[e];
        yy.x = fma(alpha, pp.x, fma(omega, s.x, yy.x)); yy.y = fma(alpha, pp.y, fma(omega, s.y, yy.y));
        s.x = fma(-omega, tt.x, s.x); s.y = fma(-omega, tt.y, s.y);
        y2[e] = yy; r2[e] = s;
        acc[0] += hh.x * s.x + hh.y * s.y; acc[1] += s.x * s.x + s.y * s.y;
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const long long k = n - 1;
        y[k] += alpha * p[k] + omega * r[k];
        r[k] -= omega * t[k];
        acc[0] += rhat[k] * r[k]; acc[1] += r[k] * r[k];
    }
    reduce_and_finish<2>(acc, W, BICG_RHO, 0);
}

// x += M^-1 y, y = 0 (end of a BiCGStab cycle; "K x = y")
__global__ void __launch_bounds__(KTHREADS) combine_y_kernel(long long N, const double* __restrict__ Minv, double* __restrict__ y, double* __restrict__ x)
{
    for (long long id = blockIdx.x * (long long)KTHREADS + threadIdx.x; id < N; id += (long long)gridDim.x * KTHREADS) {
        const double u0 = y[id], u1 = y[N + id], u2 = y[2 * N + id];
        x[id]         += Minv[0 * N + id] * u0 + Minv[1 * N + id] * u1 + Minv[2 * N + id] * u2;
        x[N + id]     += Minv[3 * N + id] * u0 + Minv[4 * N + id] * u1 + Minv[5 * N + id] * u2;
        x[2 * N + id] += Minv[6 * N + id] * u0 + Minv[7 * N + id] * u1 + Minv[8 * N + id] * u2;
        y[id] = 0.0; y[N + id] = 0.0; y[2 * N + id] = 0.0;
    }
}

cudaError_t launch_bicg_begin(double* r, double* rhat, double* p, double* v, long long n, GmresWork W, cudaStream_t st)
{
    bicg_begin_kernel<<<current_sm_count() * 4, KTHREADS, 0, st>>>(r, rhat, p, v, n, W);
    return cudaGetLastError();
}
cudaError_t launch_bicg_p(const double* r, double* p, const double* v, long long n, GmresWork W, cudaStream_t st)
{
    bicg_p_kernel<<<current_sm_count() * 4, KTHREADS, 0, st>>>(r, p, v, n, W);
    return cudaGetLastError();
}
cudaError_t launch_bicg_s(double* r, const double* v, long long n, GmresWork W, cudaStream_t st)
{
    bicg_s_kernel<<<current_sm_count() * 4, KTHREADS, 0, st>>>(r, v, n, W);
    return cudaGetLastError();
}
cudaError_t launch_bicg_xr(double* y, const double* p, double* r, const double* t, const double* rhat, long long n,
                           GmresWork W, int sm_count, cudaStream_t st)
{
    bicg_xr_kernel<<<grid_for(n, sm_count), KTHREADS, 0, st>>>(y, p, r, t, rhat, n, W);
    return cudaGetLastError();
}
cudaError_t launch_combine_y(const Grid& g, const double* Minv, double* y, double* x, cudaStream_t st)
{
    const long long N = (long long)g.nx * g.ny;
    const long long need = (N + KTHREADS - 1) / KTHREADS;
    combine_y_kernel<<<(int)(need < current_sm_count() * 8 ? need : current_sm_count() * 8), KTHREADS, 0, st>>>(N, Minv, y, x);
    return cudaGetLastError();
}

// o may alias a or b (the Newton loop subtracts in place): no __restrict__
__global__ void sub_kernel(double* o, const double* a, const double* b, long long n)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) o[k] = a[k] - b[k];
}

cudaError_t launch_sub(double* out, const double* a, const double* b, long long n, cudaStream_t st)
{
    const long long need = (n + 255) / 256;
    sub_kernel<<<(int)(need < current_sm_count() * 8 ? need : current_sm_count() * 8), 256, 0, st>>>(out, a, b, n);
    return cudaGetLastError();
}

__global__ void begin_solve_kernel(GmresWork W, double tol, int m, int maxit)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    GmresCtl* c = W.ctl;
    c->bnorm = 0.0; c->target = 0.0; c->rnorm = 0.0; c->est = tol;
    c->m = m; c->maxit = maxit; c->its = 0; c->j = 0; c->inner_stop = 0; c->converged = 0; c->nonfinite = 0;
    c->nhist = 0; c->ticket = 0;
    for (int k = 0; k < 8; ++k) c->blk[k] = 0.0;
    for (int k = 0; k < 4; ++k) c->blk_stat[k] = 0;
}

cudaError_t launch_begin_solve(GmresWork W, double tol, int m, int maxit, cudaStream_t st)
{
    begin_solve_kernel<<<1, 32, 0, st>>>(W, tol, m, maxit);
    return cudaGetLastError();
}

}  // namespace ark
