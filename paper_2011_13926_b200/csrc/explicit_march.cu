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
#include "ark_m1_internal.h"

namespace ark {

static constexpr int TX = 128;

struct Raw { double E, Fx, Fy, st, sa; };

// Row loader with boundary handling.  i may be -1 or nx (x ghost), j may be -1 or ny (y ghost), never both.
__device__ __forceinline__ Raw load_raw(const Fields& f, const Grid& g, int i, int j, bool col_active)
{
    Raw r; r.E = 1.0; r.Fx = 0.0; r.Fy = 0.0; r.st = 0.0; r.sa = 0.0;
    if (!col_active) return r;
    const bool xout = (i < 0 || i >= g.nx), yout = (j < 0 || j >= g.ny);
    if (xout && yout) return r;          // corner ghosts are never used by a 5-point stencil
    CellU u; fetch_cell(f, g, i, j, u);
    r.E = u.E; r.Fx = u.Fx; r.Fy = u.Fy; r.st = u.st; r.sa = u.sa;
    return r;
}

struct XPub { double E, Fx, Fy, Pxx, Pxy, lmin, lmax, f, st; };   // what the west neighbour needs for its east face

template <bool SD>
__global__ void __launch_bounds__(TX) explicit_march_kernel(Grid g, Scheme s, Fields f, double dt, int RY,
                                                            double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy)
{
    __shared__ XPub pub[TX];
    __shared__ double flx[4][TX];
    const int t = threadIdx.x;
    const int i = blockIdx.x * (TX - 2) - 1 + t;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    const bool col_active = (i <= g.nx);                    // i in [-1, nx]
    const bool upd = (t >= 1 && t <= TX - 2 && i >= 0 && i < g.nx);
    const double c = g.c, c2 = c * c;
    const double rdx = dt / g.dx, rdy = dt / g.dy;
    const bool wb = SD ? true : (s.wb != 0);

    // prologue: rows j0-1 (south) and j0 (centre); flux through the south face of row j0
    Raw uS = load_raw(f, g, i, j0 - 1, col_active);
    Raw uC = load_raw(f, g, i, j0, col_active);
    Raw uN = load_raw(f, g, i, j0 + 1, col_active && (j0 + 1 <= g.ny));
    Clo qS, qC;
    closure_eval<false, SD>(s, c, uS.E, uS.Fx, uS.Fy, qS, nullptr);
    closure_eval<false, SD>(s, c, uC.E, uC.Fx, uC.Fy, qC, nullptr);
    double Hs0, Hs1, Hs2, Ss;   // south flux and sigma_s (Fy_{j-1} + Fy_j)
    {
        Face fs;
        face_eval<SD>(s, c, g.dy, qS.lmin[1], qS.lmax[1], qS.f, uS.st, qC.lmin[1], qC.lmax[1], qC.f, uC.st, fs);
        Hs0 = fs.alpha * (fs.ap * uS.Fy + fs.am * uC.Fy + fs.Lam * (uC.E - uS.E));
        Hs1 = c2 * (fs.ap * qS.Pxy + fs.am * qC.Pxy) + fs.Lam * (uC.Fx - uS.Fx);
        Hs2 = c2 * (fs.ap * qS.Pyy + fs.am * qC.Pyy) + fs.Lam * (uC.Fy - uS.Fy);
        Ss = fs.sig * (uS.Fy + uC.Fy);
    }

    for (int j = j0; j < j1; ++j) {
        // prefetch the raw state two rows ahead
        const Raw uNN = load_raw(f, g, i, j + 2, col_active && (j + 2 <= g.ny) && (j + 1 < j1));
        // closure of the north cell, north face
        Clo qN;
        closure_eval<false, SD>(s, c, uN.E, uN.Fx, uN.Fy, qN, nullptr);
        Face fn;
        face_eval<SD>(s, c, g.dy, qC.lmin[1], qC.lmax[1], qC.f, uC.st, qN.lmin[1], qN.lmax[1], qN.f, uN.st, fn);
        const double Hn0 = fn.alpha * (fn.ap * uC.Fy + fn.am * uN.Fy + fn.Lam * (uN.E - uC.E));
        const double Hn1 = c2 * (fn.ap * qC.Pxy + fn.am * qN.Pxy) + fn.Lam * (uN.Fx - uC.Fx);
        const double Hn2 = c2 * (fn.ap * qC.Pyy + fn.am * qN.Pyy) + fn.Lam * (uN.Fy - uC.Fy);
        const double Sn = fn.sig * (uC.Fy + uN.Fy);

        // publish the x-face data of this cell, read the east neighbour's
        XPub me; me.E = uC.E; me.Fx = uC.Fx; me.Fy = uC.Fy; me.Pxx = qC.Pxx; me.Pxy = qC.Pxy;
        me.lmin = qC.lmin[0]; me.lmax = qC.lmax[0]; me.f = qC.f; me.st = uC.st;
        pub[t] = me;
        __syncthreads();
        double Ge0 = 0.0, Ge1 = 0.0, Ge2 = 0.0, Se = 0.0;
        if (t < TX - 1) {
            const XPub R = pub[t + 1];
            Face fe;
            face_eval<SD>(s, c, g.dx, me.lmin, me.lmax, me.f, me.st, R.lmin, R.lmax, R.f, R.st, fe);
            Ge0 = fe.alpha * (fe.ap * me.Fx + fe.am * R.Fx + fe.Lam * (R.E - me.E));
            Ge1 = c2 * (fe.ap * me.Pxx + fe.am * R.Pxx) + fe.Lam * (R.Fx - me.Fx);
            Ge2 = c2 * (fe.ap * me.Pxy + fe.am * R.Pxy) + fe.Lam * (R.Fy - me.Fy);
            Se = fe.sig * (me.Fx + R.Fx);
        }
        flx[0][t] = Ge0; flx[1][t] = Ge1; flx[2][t] = Ge2; flx[3][t] = Se;
        __syncthreads();
        if (upd) {
            const double Gw0 = flx[0][t - 1], Gw1 = flx[1][t - 1], Gw2 = flx[2][t - 1], Sw = flx[3][t - 1];
            double SFx, SFy;
            if (wb) { SFx = -0.25 * c * (Se + Sw); SFy = -0.25 * c * (Sn + Ss); }
            else { SFx = -c * uC.st * uC.Fx; SFy = -c * uC.st * uC.Fy; }
            const double SE = -c * uC.sa * uC.E;
            const long long id = (long long)j * g.nx + i;
            oE[id]  = uC.E  - (rdx * (Ge0 - Gw0) + rdy * (Hn0 - Hs0) - dt * SE);
            oFx[id] = uC.Fx - (rdx * (Ge1 - Gw1) + rdy * (Hn1 - Hs1) - dt * SFx);
            oFy[id] = uC.Fy - (rdx * (Ge2 - Gw2) + rdy * (Hn2 - Hs2) - dt * SFy);
        }
        // shift the window north
        uC = uN; qC = qN; uN = uNN;
        Hs0 = Hn0; Hs1 = Hn1; Hs2 = Hn2; Ss = Sn;
    }
}

cudaError_t launch_explicit_march(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                  double* outE, double* outFx, double* outFy, int sm_count, cudaStream_t st)
{
    const int strips = (g.nx + (TX - 2) - 1) / (TX - 2);
    // rows per block: enough blocks for ~8 per SM, between 4 and 64 rows
    long long want = ((long long)g.ny * strips + (long long)sm_count * 8 - 1) / ((long long)sm_count * 8);
    int RY = (int)(want < 4 ? 4 : (want > 64 ? 64 : want));
    if (RY > g.ny) RY = g.ny;
    dim3 grd(strips, (g.ny + RY - 1) / RY);
    if (s.is_default()) explicit_march_kernel<true><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    else explicit_march_kernel<false><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    return cudaGetLastError();
}

}  // namespace ark
