// krylov_cb.cu — compressed-basis variant of the GMRES vector kernels (option "basis_precision" = 32).
//
// The Krylov iteration at 4096^2 runs at the HBM roofline, and 73 % of its bytes are the Arnoldi basis
// read twice per iteration.  Here the basis vectors are STORED in single precision while everything that is computed — the
// operator, the dot products, the updates, the Hessenberg matrix, the solution — stays fp64: w = A M^-1 v_j is formed in fp64
// from the stored v_j, orthogonalised in fp64 against the stored vectors, and only then rounded once when it is stored as
// v_{j+1}.  The Arnoldi relation then holds for the stored basis up to 6e-8 per vector; the true fp64 residual is recomputed at
// every restart, so the solve still ends at the requested fp64 tolerance (it may take a few more iterations).
// Bytes per iteration at inner index j: dot 24 + 12 (j+1), update 24 + 12 (j+1) + 12, operator 252
// (mean over j < 30: 684 B/cell against 1119 for the fp64 basis).
//
// Same conventions as krylov_kernels.cu: unnormalised basis with scale[i], one-pass classical Gram-Schmidt, deterministic
// two-stage reductions with device-side epilogues.  Four elements per thread: the fp64 vector as two double2, each basis
// vector as one float4 (the same registers as the double2 of the fp64 kernels).
#include "krylov_device.cuh"

namespace ark {

template <int NV>
__global__ void __launch_bounds__(KTHREADS) multi_dot32_kernel(const double* __restrict__ w, const float* __restrict__ V0,
                                                               long long stride, long long n, GmresWork W, int mode, int col0)
{
    if ((mode == DOT_H || mode == DOT_H2) && W.ctl->inner_stop) return;
    double acc[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) acc[k] = 0.0;
    const long long n4 = n >> 2;
    const double2* w2 = reinterpret_cast<const double2*>(w);
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n4; e += (long long)gridDim.x * KTHREADS) {
        const double2 a = w2[2 * e], b = w2[2 * e + 1];
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const float4 v = reinterpret_cast<const float4*>(V0 + k * stride)[e];
            acc[k] += a.x * (double)v.x + a.y * (double)v.y + b.x * (double)v.z + b.y * (double)v.w;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (long long t = n4 << 2; t < n; ++t)
#pragma unroll
            for (int k = 0; k < NV; ++k) acc[k] += w[t] * (double)V0[k * stride + t];
    reduce_and_finish<NV>(acc, W, mode, col0);
}

// w -= sum_k coef[col0+k] V_k.  write_w: store the result back to w (fp64).  out32: store it rounded as the next basis vector.
template <int NV, bool WITH_NORM>
__global__ void __launch_bounds__(KTHREADS) update32_kernel(double* __restrict__ w, const float* __restrict__ V0, long long stride,
                                                            long long n, GmresWork W, int col0, int write_w, float* __restrict__ out32)
{
    if (W.ctl->inner_stop) return;
    double cf[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) cf[k] = W.coef[col0 + k];
    double acc[1] = { 0.0 };
    const long long n4 = n >> 2;
    double2* w2 = reinterpret_cast<double2*>(w);
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n4; e += (long long)gridDim.x * KTHREADS) {
        double2 a = w2[2 * e], b = w2[2 * e + 1];
        float4 v[NV];
#pragma unroll
        for (int k = 0; k < NV; ++k) v[k] = reinterpret_cast<const float4*>(V0 + k * stride)[e];
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            a.x = fma(-cf[k], (double)v[k].x, a.x); a.y = fma(-cf[k], (double)v[k].y, a.y);
            b.x = fma(-cf[k], (double)v[k].z, b.x); b.y = fma(-cf[k], (double)v[k].w, b.y);
        }
        if (write_w) { w2[2 * e] = a; w2[2 * e + 1] = b; }
        if (out32) reinterpret_cast<float4*>(out32)[e] = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
        if (WITH_NORM) acc[0] += a.x * a.x + a.y * a.y + b.x * b.x + b.y * b.y;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (long long t = n4 << 2; t < n; ++t) {
            double a = w[t];
#pragma unroll
            for (int k = 0; k < NV; ++k) a -= cf[k] * (double)V0[k * stride + t];
            if (write_w) w[t] = a;
            if (out32) out32[t] = (float)a;
            if (WITH_NORM) acc[0] += a * a;
        }
    if (WITH_NORM) reduce_and_finish<1, KTHREADS, true>(acc, W, DOT_UPD, 0);
}

static int grid_for4(long long n, int sm_count)
{
    const long long need = ((n >> 2) + KTHREADS - 1) / KTHREADS;
    const long long cap = krylov_max_blocks(sm_count);
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

cudaError_t launch_multi_dot32(const double* w, const float* V0, long long stride, int nv, int col0, long long n,
                               GmresWork W, int mode, int sm_count, cudaStream_t st)
{
    const int grd = grid_for4(n, sm_count);
    switch (nv) {
#define ARK_CASE(K) case K: multi_dot32_kernel<K><<<grd, KTHREADS, 0, st>>>(w, V0, stride, n, W, mode, col0); break;
        ARK_CASE(1) ARK_CASE(2) ARK_CASE(3) ARK_CASE(4) ARK_CASE(5) ARK_CASE(6) ARK_CASE(7) ARK_CASE(8)
        ARK_CASE(9) ARK_CASE(10) ARK_CASE(11) ARK_CASE(12) ARK_CASE(13) ARK_CASE(14) ARK_CASE(15) ARK_CASE(16)
#undef ARK_CASE
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_update32(double* w, const float* V0, long long stride, int nv, int col0, long long n, GmresWork W,
                            int with_norm, int write_w, float* out32, int sm_count, cudaStream_t st)
{
    const int grd = grid_for4(n, sm_count);
    switch (nv) {
#define ARK_CASE(K) case K: if (with_norm) update32_kernel<K, true><<<grd, KTHREADS, 0, st>>>(w, V0, stride, n, W, col0, write_w, out32); \
                            else update32_kernel<K, false><<<grd, KTHREADS, 0, st>>>(w, V0, stride, n, W, col0, write_w, out32); break;
        ARK_CASE(1) ARK_CASE(2) ARK_CASE(3) ARK_CASE(4) ARK_CASE(5) ARK_CASE(6) ARK_CASE(7) ARK_CASE(8)
        ARK_CASE(9) ARK_CASE(10) ARK_CASE(11) ARK_CASE(12) ARK_CASE(13) ARK_CASE(14) ARK_CASE(15) ARK_CASE(16)
#undef ARK_CASE
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// x += Minv * (sum_{k<ctl->j} coef[k] V_k) per cell, basis in single precision
__global__ void __launch_bounds__(KTHREADS) combine32_kernel(long long N, const float* __restrict__ V, long long stride,
                                                             const double* __restrict__ Minv, double* __restrict__ x, GmresWork W)
{
    const int jj = W.ctl->j;
    if (jj == 0) return;
    for (long long id = blockIdx.x * (long long)KTHREADS + threadIdx.x; id < N; id += (long long)gridDim.x * KTHREADS) {
        double u0 = 0.0, u1 = 0.0, u2 = 0.0;
#pragma unroll 4
        for (int k = 0; k < jj; ++k) {
            const double cf = W.coef[k];
            const float* v = V + k * stride;
            u0 += cf * (double)v[id]; u1 += cf * (double)v[N + id]; u2 += cf * (double)v[2 * N + id];
        }
        x[id]         += Minv[0 * N + id] * u0 + Minv[1 * N + id] * u1 + Minv[2 * N + id] * u2;
        x[N + id]     += Minv[3 * N + id] * u0 + Minv[4 * N + id] * u1 + Minv[5 * N + id] * u2;
        x[2 * N + id] += Minv[6 * N + id] * u0 + Minv[7 * N + id] * u1 + Minv[8 * N + id] * u2;
    }
}

cudaError_t launch_combine32(const Grid& g, const float* V, long long stride, const double* Minv, double* x,
                             GmresWork W, int sm_count, cudaStream_t st)
{
    const long long N = (long long)g.nx * g.ny;
    const long long need = (N + KTHREADS - 1) / KTHREADS, cap = (long long)sm_count * 8;
    combine32_kernel<<<(int)(need < cap ? need : cap), KTHREADS, 0, st>>>(N, V, stride, Minv, x, W);
    return cudaGetLastError();
}

}  // namespace ark
