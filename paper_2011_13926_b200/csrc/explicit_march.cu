// explicit_march.cu — the optimised fused explicit step (rows a1-a4), pure radiation (no T, no source_E).
//
// Same arithmetic as explicit_cell_kernel, organised so that every
// closure is evaluated once per cell and every face flux once per face (the kernel sits at the fp64-ALU/HBM
// ridge):
//   * a block owns a strip of TX-2 columns (+1 halo column each side) and marches over RY rows;
//   * a thread owns one column: it keeps the closure of its cell in row j and row j+1 in registers, so the
//     y-face flux needs no neighbour thread, and the north flux of row j is reused as the south flux of row j+1;
//   * x-faces: each thread publishes the x-face data of its cell in shared memory, computes the flux through
//     its EAST face, publishes it, and reads its WEST flux from the thread to its left;
//   * the raw state of row j+2 is requested from HBM before row j is processed (software prefetch).
// HBM traffic: 5 planes read, 3 written = 64 B/cell (+ the halo columns/rows, served mostly by L2).
#include "explicit_device.cuh"

namespace ark {

// COUPLED: stage-2 terms of the cell kernel (emission c sigma_a a_r T^4, source_E, explicit matter-energy update of Eq. 4).
template <bool SD, bool COUPLED>
__global__ void __launch_bounds__(TX, 4) explicit_march_kernel(Grid g, Scheme s, Fields f, double dt, int RY,
                                                            double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy,
                                                            double* __restrict__ oT)
{
    __shared__ XPub pub[TX + 1];   // +1: the last thread reads a (unused) right neighbour
    __shared__ double flx[4][TX];
    const int t = threadIdx.x;
    const int i = blockIdx.x * (TX - 2) - 1 + t;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    const bool col_active = (i <= g.nx);                    // i in [-1, nx]
    const bool upd = (t >= 1 && t <= TX - 2 && i >= 0 && i < g.nx);
    const double c = g.c, cdt = c * dt;
    const double rdx = dt / g.dx, rdy = dt / g.dy;
    const double k3x = 1.5 * g.dx / c, k3y = 1.5 * g.dy / c;   // Eq. 25: 3 sigma_f dx (1-f^2)/c = k3 (sigma_L + sigma_R)(1-f^2)
    const double qc = 0.125 * c * dt;                            // WB source weight 1/4 (Eqs. 18-19) times dt, times the 1/2 of sigma_f
    const bool wb = SD ? true : (s.wb != 0);

    // resolve the column once
    int xmode = 0, ii = i, xside = 0;
    if (!col_active) xmode = 2;
    else if (i < 0 || i >= g.nx) {
        xside = (i < 0) ? XLO : XHI;
        const int bc = g.bc[xside];
        if (bc == BC_DIRICHLET) { xmode = 1; ii = 0; }
        else if (bc == BC_PERIODIC) ii = (i < 0) ? g.nx - 1 : 0;
        else ii = (i < 0) ? 0 : g.nx - 1;
    }

    // prologue: rows j0-1 (south) and j0 (centre); flux through the south face of row j0
    Raw uS = load_row(f, g, xmode, ii, xside, j0 - 1);
    Raw uC = load_row(f, g, xmode, ii, xside, j0);
    Raw uN = load_row(f, g, xmode, ii, xside, j0 + 1);
    CloF qS, qC;
    cell_closure<SD>(s, c, uS, qS);
    cell_closure<SD>(s, c, uC, qC);
    double Hs0, Hs1, Hs2, Ss;   // south flux and sigma_s (Fy_{j-1} + Fy_j)
    {
        FaceF fs;
        cell_face<SD>(s, c, g.dy, k3y, qS.lminy, qS.lmaxy, qS.f, uS.st, qC.lminy, qC.lmaxy, qC.f, uC.st, fs);
        // y-face: normal = y.  (G0, Gn, Gt) = (E, Fy, Fx) fluxes
        ARK_FACE_FLUX(fs, uS.E, uC.E, uS.Fy, uC.Fy, uS.Fx, uC.Fx, qS.Pyy, qC.Pyy, qS.Pxy, qC.Pxy, Hs0, Hs2, Hs1, Ss);
    }
    // 32-bit in-plane offsets (host guarantees nx*ny < 2^31)
    unsigned int row_off = (unsigned int)j0 * (unsigned int)g.nx + (unsigned int)(i < 0 ? 0 : i);

#pragma unroll 1
    for (int j = j0; j < j1; ++j) {
        // prefetch the raw state two rows ahead
        const Raw uNN = load_row(f, g, (j + 1 < j1) ? xmode : 2, ii, xside, j + 2);
        // publish the x-face data of this cell (computed one row ago)
        XPub me; me.E = uC.E; me.Fx = uC.Fx; me.Fy = uC.Fy; me.Pxx = qC.Pxx; me.Pxy = qC.Pxy;
        me.lmin = qC.lminx; me.lmax = qC.lmaxx; me.f = qC.f; me.st = uC.st;
        pub[t] = me;
        // closure of the north cell, north face (independent of the neighbours: overlaps the barrier)
        CloF qN;
        cell_closure<SD>(s, c, uN, qN);
        FaceF fn;
        cell_face<SD>(s, c, g.dy, k3y, qC.lminy, qC.lmaxy, qC.f, uC.st, qN.lminy, qN.lmaxy, qN.f, uN.st, fn);
        double Hn0, Hn1, Hn2, Sn;
        ARK_FACE_FLUX(fn, uC.E, uN.E, uC.Fy, uN.Fy, uC.Fx, uN.Fx, qC.Pyy, qN.Pyy, qC.Pxy, qN.Pxy, Hn0, Hn2, Hn1, Sn);
        __syncthreads();
        // east face from the east neighbour's published data
        double Ge0, Ge1, Ge2, Se;
        {
            const XPub R = pub[t + 1];
            FaceF fe;
            cell_face<SD>(s, c, g.dx, k3x, me.lmin, me.lmax, me.f, me.st, R.lmin, R.lmax, R.f, R.st, fe);
            ARK_FACE_FLUX(fe, me.E, R.E, me.Fx, R.Fx, me.Fy, R.Fy, me.Pxx, R.Pxx, me.Pxy, R.Pxy, Ge0, Ge1, Ge2, Se);
        }
        flx[0][t] = Ge0; flx[1][t] = Ge1; flx[2][t] = Ge2; flx[3][t] = Se;
        __syncthreads();
        {
            const int tw = (t > 0) ? t - 1 : 0;
            const double Gw0 = flx[0][tw], Gw1 = flx[1][tw], Gw2 = flx[2][tw], Sw = flx[3][tw];
            double dSFx, dSFy;   // -dt * S^F
            if (wb) { dSFx = qc * (Se + Sw); dSFy = qc * (Sn + Ss); }
            else { dSFx = dt * c * uC.st * uC.Fx; dSFy = dt * c * uC.st * uC.Fy; }
            double dSE = cdt * uC.sa * uC.E;        // -dt * S^E
            if (COUPLED && upd && !(!SD && s.src_off)) {
                if (f.T) {
                    const double T = f.T[row_off], rcv = f.rho_cv ? f.rho_cv[row_off] : 1.0;
                    const double Theta = s.a_r * (T * T) * (T * T);
                    dSE -= cdt * uC.sa * Theta;
                    if (oT) oT[row_off] = T - cdt * uC.sa * (Theta - uC.E) / rcv;      // Eq. 4, explicit
                }
                if (f.source_E) dSE -= dt * f.source_E[row_off];
            }
            if (!SD && s.src_off) { dSE = 0.0; dSFx = 0.0; dSFy = 0.0; }     // semi-implicit step: hyperbolic part only
            const double nE  = uC.E  - fma(rdx, Ge0 - Gw0, fma(rdy, Hn0 - Hs0, dSE));
            const double nFx = uC.Fx - fma(rdx, Ge1 - Gw1, fma(rdy, Hn1 - Hs1, dSFx));
            const double nFy = uC.Fy - fma(rdx, Ge2 - Gw2, fma(rdy, Hn2 - Hs2, dSFy));
            if (upd) { oE[row_off] = nE; oFx[row_off] = nFx; oFy[row_off] = nFy; }
        }
        row_off += (unsigned int)g.nx;
        // shift the window north
        uC = uN; qC = qN; uN = uNN;
        Hs0 = Hn0; Hs1 = Hn1; Hs2 = Hn2; Ss = Sn;
    }
}

cudaError_t launch_explicit_march(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                  double* outE, double* outFx, double* outFy, double* outT, int sm_count, cudaStream_t st)
{
    const int strips = (g.nx + (TX - 2) - 1) / (TX - 2);
    // rows per block: enough blocks for ~8 per SM, between 4 and MARCH_RY rows.  (A single wave of
    // SMs x resident-blocks blocks with ~240 rows each was measured 8% slower at 4096^2: uneven blocks per SM.)
    long long want = ((long long)g.ny * strips + (long long)sm_count * 8 - 1) / ((long long)sm_count * 8);
    int RY = (int)(want < 4 ? 4 : (want > MARCH_RY ? MARCH_RY : want));
    if (RY > g.ny) RY = g.ny;
    if ((long long)g.nx * g.ny >= (1LL << 31) || (g.ny + RY - 1) / RY > 65535) return cudaErrorInvalidConfiguration;   // 32-bit in-plane offsets; gridDim.y
    dim3 grd(strips, (g.ny + RY - 1) / RY);
    const bool coupled = (f.T != nullptr) || (f.source_E != nullptr);
    if (coupled) {
        if (s.is_default()) explicit_march_kernel<true, true><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, outT);
        else explicit_march_kernel<false, true><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, outT);
    } else {
        if (s.is_default()) explicit_march_kernel<true, false><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, nullptr);
        else explicit_march_kernel<false, false><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, nullptr);
    }
    return cudaGetLastError();
}

}  // namespace ark
