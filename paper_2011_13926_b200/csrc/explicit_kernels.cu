// explicit_kernels.cu — rows a1-a4 of the hot path: closure, AP-HLL face fluxes, WB source, explicit update.
//
//   U^{n+1}_i = U^n_i - dt [ (G_{i+1/2} - G_{i-1/2})/dx + (H_{j+1/2} - H_{j-1/2})/dy - S_i ]
// with G, H the fluxes of Eq. 13 times alpha on the energy row (Eq. 12),
// S^E = -c sigma_a E (+ c sigma_a a_r T^4), S^F the well-balanced source of Eqs. 18-19
// applied dimension by dimension (reading R6).
//
// Two kernels compute the same thing:
//   explicit_cell_kernel  : one thread per cell, five closures and four faces per thread.  Handles every scheme
//                           switch, the temperature coupling and the residual output; the reference point for
//                           the optimised kernel and the path for small or unusual cases.
//   explicit_march_kernel : see explicit_march.cu (row-marching, one closure per cell, one flux per face).
#include "ark_m1_internal.h"

namespace ark {

template <bool SD>
__device__ __forceinline__ void face_flux(const Face& fc, int dir, double c2,
                                          const CellU& L, const Clo& qL, const CellU& R, const Clo& qR, double G[3])
{
    const double FnL = dir == 0 ? L.Fx : L.Fy, FnR = dir == 0 ? R.Fx : R.Fy;
    const double PnxL = dir == 0 ? qL.Pxx : qL.Pxy, PnxR = dir == 0 ? qR.Pxx : qR.Pxy;
    const double PnyL = dir == 0 ? qL.Pxy : qL.Pyy, PnyR = dir == 0 ? qR.Pxy : qR.Pyy;
    G[0] = fc.alpha * (fc.ap * FnL + fc.am * FnR + fc.Lam * (R.E - L.E));
    G[1] = c2 * (fc.ap * PnxL + fc.am * PnxR) + fc.Lam * (R.Fx - L.Fx);
    G[2] = c2 * (fc.ap * PnyL + fc.am * PnyR) + fc.Lam * (R.Fy - L.Fy);
}

// R(U) of one cell from its five-point neighbourhood.
template <bool SD>
__device__ __forceinline__ void residual_cell(const Grid& g, const Scheme& s, const Fields& f, int i, int j,
                                              CellU& uc, double R[3])
{
    CellU u[5]; Clo q[5];   // centre, west, east, south, north
    fetch_cell(f, g, i, j, u[0]);
    fetch_cell(f, g, i - 1, j, u[1]);
    fetch_cell(f, g, i + 1, j, u[2]);
    fetch_cell(f, g, i, j - 1, u[3]);
    fetch_cell(f, g, i, j + 1, u[4]);
#pragma unroll
    for (int k = 0; k < 5; ++k) closure_eval<false, SD>(s, g.c, u[k].E, u[k].Fx, u[k].Fy, q[k], nullptr);
    Face fw, fe, fs, fn;
    face_eval<SD>(s, g.c, g.dx, q[1].lmin[0], q[1].lmax[0], q[1].f, u[1].st, q[0].lmin[0], q[0].lmax[0], q[0].f, u[0].st, fw);
    face_eval<SD>(s, g.c, g.dx, q[0].lmin[0], q[0].lmax[0], q[0].f, u[0].st, q[2].lmin[0], q[2].lmax[0], q[2].f, u[2].st, fe);
    face_eval<SD>(s, g.c, g.dy, q[3].lmin[1], q[3].lmax[1], q[3].f, u[3].st, q[0].lmin[1], q[0].lmax[1], q[0].f, u[0].st, fs);
    face_eval<SD>(s, g.c, g.dy, q[0].lmin[1], q[0].lmax[1], q[0].f, u[0].st, q[4].lmin[1], q[4].lmax[1], q[4].f, u[4].st, fn);
    const double c = g.c, c2 = c * c;
    double Gw[3], Ge[3], Hs[3], Hn[3];
    face_flux<SD>(fw, 0, c2, u[1], q[1], u[0], q[0], Gw);
    face_flux<SD>(fe, 0, c2, u[0], q[0], u[2], q[2], Ge);
    face_flux<SD>(fs, 1, c2, u[3], q[3], u[0], q[0], Hs);
    face_flux<SD>(fn, 1, c2, u[0], q[0], u[4], q[4], Hn);
    double SE = -c * u[0].sa * u[0].E, SFx, SFy;
    if (f.T) { const double T = f.T[u[0].idx]; SE += c * u[0].sa * s.a_r * (T * T) * (T * T); }
    if (f.source_E) SE += f.source_E[u[0].idx];
    const bool wb = SD ? true : (s.wb != 0);
    if (wb) {   // Eqs. 18-19: {sigma F}_i = (sigma_{i+1/2} F_{i+1/2} + sigma_{i-1/2} F_{i-1/2})/2, face values = means
        SFx = -c * 0.25 * (fe.sig * (u[0].Fx + u[2].Fx) + fw.sig * (u[1].Fx + u[0].Fx));
        SFy = -c * 0.25 * (fn.sig * (u[0].Fy + u[4].Fy) + fs.sig * (u[3].Fy + u[0].Fy));
    } else {    // Eq. 16
        SFx = -c * u[0].st * u[0].Fx; SFy = -c * u[0].st * u[0].Fy;
    }
    const double idx = 1.0 / g.dx, idy = 1.0 / g.dy;
    R[0] = (Ge[0] - Gw[0]) * idx + (Hn[0] - Hs[0]) * idy - SE;
    R[1] = (Ge[1] - Gw[1]) * idx + (Hn[1] - Hs[1]) * idy - SFx;
    R[2] = (Ge[2] - Gw[2]) * idx + (Hn[2] - Hs[2]) * idy - SFy;
    uc = u[0];
}

// mode 0: out = U - dt R (and the explicit matter-energy update of Eq. 4 when T is set); mode 1: out = R.
template <bool SD>
__global__ void __launch_bounds__(128) explicit_cell_kernel(Grid g, Scheme s, Fields f, double dt, int mode,
                                                            double* __restrict__ oE, double* __restrict__ oFx,
                                                            double* __restrict__ oFy, double* __restrict__ oT)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    CellU u; double R[3];
    residual_cell<SD>(g, s, f, i, j, u, R);
    const long long id = (long long)j * g.nx + i;
    if (mode == 1) { oE[id] = R[0]; oFx[id] = R[1]; oFy[id] = R[2]; return; }
    oE[id] = u.E - dt * R[0]; oFx[id] = u.Fx - dt * R[1]; oFy[id] = u.Fy - dt * R[2];
    if (f.T && oT) {   // Eq. 4, explicit
        const double T = f.T[id], rcv = f.rho_cv ? f.rho_cv[id] : 1.0;
        oT[id] = T - dt * g.c * u.sa * (s.a_r * (T * T) * (T * T) - u.E) / rcv;
    }
}

cudaError_t launch_explicit_cell(const Grid& g, const Scheme& s, const Fields& f, double dt, int mode,
                                 double* outE, double* outFx, double* outFy, double* outT, cudaStream_t st)
{
    dim3 blk(32, 4), grd((g.nx + 31) / 32, (g.ny + 3) / 4);
    if (s.is_default()) explicit_cell_kernel<true><<<grd, blk, 0, st>>>(g, s, f, dt, mode, outE, outFx, outFy, outT);
    else explicit_cell_kernel<false><<<grd, blk, 0, st>>>(g, s, f, dt, mode, outE, outFx, outFy, outT);
    return cudaGetLastError();
}

// Step 3 of the operator splitting: explicit velocity sources of Eq. 6, cell-centred:
//   S_E = (sigma/c) u.F + (sigma/c) E u.u + (sigma/c) u.(u.P);   S_F = sigma u.P + sigma a_r T^4 u + (sigma/c^2) u (u.F)
//   E += dt S_E,  F += dt c S_F
__global__ void velocity_sources_kernel(Grid g, Scheme s, Fields f, const double* __restrict__ ux, const double* __restrict__ uy,
                                        double dt, double* __restrict__ E, double* __restrict__ Fx, double* __restrict__ Fy)
{
    const long long N = (long long)g.nx * g.ny;
    for (long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x; id < N; id += (long long)gridDim.x * blockDim.x) {
        const double e = f.E[id], fx = f.Fx[id], fy = f.Fy[id], sg = f.st[id], vx = ux[id], vy = uy[id];
        Clo q; closure_eval<false, false>(s, g.c, e, fx, fy, q, nullptr);
        const double uPx = vx * q.Pxx + vy * q.Pxy, uPy = vx * q.Pxy + vy * q.Pyy;
        const double uF = vx * fx + vy * fy, uu = vx * vx + vy * vy;
        double Th = 0.0;
        if (f.T) { const double T = f.T[id]; Th = s.a_r * (T * T) * (T * T); }
        const double c = g.c;
        const double SE = (sg / c) * (uF + e * uu + (vx * uPx + vy * uPy));
        const double SFx = sg * uPx + sg * Th * vx + (sg / (c * c)) * vx * uF;
        const double SFy = sg * uPy + sg * Th * vy + (sg / (c * c)) * vy * uF;
        E[id] = e + dt * SE; Fx[id] = fx + dt * c * SFx; Fy[id] = fy + dt * c * SFy;
    }
}

cudaError_t launch_velocity_sources(const Grid& g, const Scheme& s, const Fields& f, const double* ux, const double* uy,
                                    double dt, double* E, double* Fx, double* Fy, cudaStream_t st)
{
    const long long N = (long long)g.nx * g.ny;
    const int blk = 256; const int grd = (int)((N + blk - 1) / blk < current_sm_count() * 8 ? (N + blk - 1) / blk : current_sm_count() * 8);
    velocity_sources_kernel<<<grd, blk, 0, st>>>(g, s, f, ux, uy, dt, E, Fx, Fy);
    return cudaGetLastError();
}

// Row a7: guards of PAPER.md:245, 513.  counts[0] = cells with E <= 0, counts[1] = cells with |F| > cE (E > 0).
__global__ void count_unrealizable_kernel(Grid g, Fields f, unsigned long long* counts)
{
    const long long N = (long long)g.nx * g.ny;
    unsigned int a = 0, b = 0;
    for (long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x; id < N; id += (long long)gridDim.x * blockDim.x) {
        const double e = f.E[id], fx = f.Fx[id], fy = f.Fy[id];
        if (!(e > 0.0)) ++a;
        else if (sqrt(fx * fx + fy * fy) > g.c * e) ++b;
    }
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o); }
    if ((threadIdx.x & 31) == 0) {
        if (a) atomicAdd(&counts[0], (unsigned long long)a);
        if (b) atomicAdd(&counts[1], (unsigned long long)b);
    }
}

cudaError_t launch_count_unrealizable(const Grid& g, const Fields& f, unsigned long long* counts2, cudaStream_t st)
{
    const long long N = (long long)g.nx * g.ny;
    const int blk = 256; const int grd = (int)((N + blk - 1) / blk < current_sm_count() * 8 ? (N + blk - 1) / blk : current_sm_count() * 8);
    count_unrealizable_kernel<<<grd, blk, 0, st>>>(g, f, counts2);
    return cudaGetLastError();
}

// Self-test of the fast reciprocal / reciprocal square root (m1_device.cuh) against the IEEE sequences, on n samples spread
// over 200 binades: out[0..3] = max relative error of rcp_fast, rsqrt_fast, sqrt_fast (vs sqrt) and rcp_fast3.
__global__ void fastmath_selftest_kernel(int n, double* __restrict__ out3)
{
    double e0 = 0.0, e1 = 0.0, e2 = 0.0, e3 = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double x = exp2((double)(i % 200 - 100)) * (1.0 + (double)i / (double)n);
        e0 = fmax(e0, fabs(rcp_fast(x) - 1.0 / x) * x);
        const double rs = 1.0 / sqrt(x), sq = sqrt(x);
        e1 = fmax(e1, fabs(rsqrt_fast(x) - rs) * sq);
        e2 = fmax(e2, fabs(sqrt_fast(x) - sq) / sq);
        e3 = fmax(e3, fabs(rcp_fast3(x) - 1.0 / x) * x);
    }
    for (int o = 16; o > 0; o >>= 1) {
        e0 = fmax(e0, __shfl_down_sync(0xffffffffu, e0, o)); e1 = fmax(e1, __shfl_down_sync(0xffffffffu, e1, o)); e2 = fmax(e2, __shfl_down_sync(0xffffffffu, e2, o));
        e3 = fmax(e3, __shfl_down_sync(0xffffffffu, e3, o));
    }
    if ((threadIdx.x & 31) == 0) {      // errors are non-negative: their bit patterns order like unsigned integers
        atomicMax((unsigned long long*)&out3[0], (unsigned long long)__double_as_longlong(e0));
        atomicMax((unsigned long long*)&out3[1], (unsigned long long)__double_as_longlong(e1));
        atomicMax((unsigned long long*)&out3[2], (unsigned long long)__double_as_longlong(e2));
        atomicMax((unsigned long long*)&out3[3], (unsigned long long)__double_as_longlong(e3));
    }
}

cudaError_t launch_fastmath_selftest(int n, double* out3, cudaStream_t st)
{
    fastmath_selftest_kernel<<<current_sm_count(), 256, 0, st>>>(n, out3);
    return cudaGetLastError();
}

// o may alias a or b (set_boundary adds in place): no __restrict__
__global__ void add_planes_kernel(double* o, const double* a, const double* b, long long n)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) o[k] = a[k] + b[k];
}

cudaError_t launch_add_planes(double* o, const double* a, const double* b, long long n, cudaStream_t st)
{
    const int blk = 256; const int grd = (int)((n + blk - 1) / blk < current_sm_count() * 8 ? (n + blk - 1) / blk : current_sm_count() * 8);
    add_planes_kernel<<<grd, blk, 0, st>>>(o, a, b, n);
    return cudaGetLastError();
}

}  // namespace ark
