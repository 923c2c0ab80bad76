// explicit_march3.cu — row-marching explicit kernel with a THREE-SLOT register rotation (explicit_kernel = 3).
//
// Same arithmetic and organisation as explicit_march_kernel (column strips, rows marched, one closure per cell, one flux
// per face, x-faces through shared memory).  The difference is purely in how the marching window is held:
// explicit_march_kernel shifts (centre <- north <- prefetched) by register copies every row, which ptxas emits as ~45
// IMAD.MOV per row — and IMAD issues at half rate on B200 (measured: 16 independent IMAD = 31 cycles per warp).  Here a
// slot = {raw state, closure, north-face flux} and the three slots exchange ROLES instead of contents: the row body is a
// forceinline function instantiated three times with permuted arguments, so no copy is ever made.
//   row j   : centre = X, north = Y, prefetch target = Z   (south flux = Z.H, written one row ago when Z was the centre)
//   row j+1 : centre = Y, north = Z, prefetch target = X
//   row j+2 : centre = Z, north = X, prefetch target = Y
#include "explicit_device.cuh"

namespace ark {

struct Slot {
    Raw u;                      // raw state of the cell
    CloF q;                     // closure (c^2 P, eigenvalues, |f|)
    double H0, H1, H2, S;       // flux through the NORTH face of the cell (E, Fx, Fy rows) and sigma_n (Fy_j + Fy_j+1)
};

struct March3Ctx {
    double c, cdt, dt, rdx, rdy, k3x, k3y, qc;
    int xmode, ii, xside, t;
    bool upd, wb;
};

template <bool SD>
__device__ __forceinline__ void row_step(const Grid& g, const Scheme& s, const Fields& f, const March3Ctx& k,
                                         Slot& C, Slot& N, Slot& P, int j, int j1, unsigned int row_off,
                                         XPub* pub, double (*flx)[TX],
                                         double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy)
{
    // prefetch the raw state two rows ahead into the slot that was the centre one row ago (its flux P.H is still needed
    // below as the south flux; only the raw fields are overwritten)
    if (j + 1 < j1) P.u = load_row(f, g, k.xmode, k.ii, k.xside, j + 2);
    // publish the x-face data of the centre cell
    XPub me; me.E = C.u.E; me.Fx = C.u.Fx; me.Fy = C.u.Fy; me.Pxx = C.q.Pxx; me.Pxy = C.q.Pxy;
    me.lmin = C.q.lminx; me.lmax = C.q.lmaxx; me.f = C.q.f; me.st = C.u.st;
    pub[k.t] = me;
    // closure of the north cell, north face
    cell_closure<SD>(s, k.c, N.u, N.q);
    FaceF fn;
    cell_face<SD>(s, k.c, g.dy, k.k3y, C.q.lminy, C.q.lmaxy, C.q.f, C.u.st, N.q.lminy, N.q.lmaxy, N.q.f, N.u.st, fn);
    ARK_FACE_FLUX(fn, C.u.E, N.u.E, C.u.Fy, N.u.Fy, C.u.Fx, N.u.Fx, C.q.Pyy, N.q.Pyy, C.q.Pxy, N.q.Pxy, C.H0, C.H2, C.H1, C.S);
    __syncthreads();
    double Ge0, Ge1, Ge2, Se;
    {
        const XPub R = pub[k.t + 1];
        FaceF fe;
        cell_face<SD>(s, k.c, g.dx, k.k3x, me.lmin, me.lmax, me.f, me.st, R.lmin, R.lmax, R.f, R.st, fe);
        ARK_FACE_FLUX(fe, me.E, R.E, me.Fx, R.Fx, me.Fy, R.Fy, me.Pxx, R.Pxx, me.Pxy, R.Pxy, Ge0, Ge1, Ge2, Se);
    }
    flx[0][k.t] = Ge0; flx[1][k.t] = Ge1; flx[2][k.t] = Ge2; flx[3][k.t] = Se;
    __syncthreads();
    {
        const int tw = (k.t > 0) ? k.t - 1 : 0;
        const double Gw0 = flx[0][tw], Gw1 = flx[1][tw], Gw2 = flx[2][tw], Sw = flx[3][tw];
        double dSFx, dSFy;   // -dt * S^F
        if (k.wb) { dSFx = k.qc * (Se + Sw); dSFy = k.qc * (C.S + P.S); }
        else { dSFx = k.dt * k.c * C.u.st * C.u.Fx; dSFy = k.dt * k.c * C.u.st * C.u.Fy; }
        const double dSE = k.cdt * C.u.sa * C.u.E;
        const double nE  = C.u.E  - fma(k.rdx, Ge0 - Gw0, fma(k.rdy, C.H0 - P.H0, dSE));
        const double nFx = C.u.Fx - fma(k.rdx, Ge1 - Gw1, fma(k.rdy, C.H1 - P.H1, dSFx));
        const double nFy = C.u.Fy - fma(k.rdx, Ge2 - Gw2, fma(k.rdy, C.H2 - P.H2, dSFy));
        if (k.upd) { oE[row_off] = nE; oFx[row_off] = nFx; oFy[row_off] = nFy; }
    }
}

template <bool SD>
__global__ void __launch_bounds__(TX, ARK_MARCH_MINB) explicit_march3_kernel(Grid g, Scheme s, Fields f, double dt, int RY,
                                                            double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy)
{
    __shared__ XPub pub[TX + 1];
    __shared__ double flx[4][TX];
    March3Ctx k;
    k.t = threadIdx.x;
    const int i = blockIdx.x * (TX - 2) - 1 + k.t;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    k.upd = (k.t >= 1 && k.t <= TX - 2 && i >= 0 && i < g.nx);
    k.c = g.c; k.dt = dt; k.cdt = g.c * dt;
    k.rdx = dt / g.dx; k.rdy = dt / g.dy;
    k.k3x = 3.0 * g.dx / g.c; k.k3y = 3.0 * g.dy / g.c;
    k.qc = 0.25 * g.c * dt;
    k.wb = SD ? true : (s.wb != 0);
    k.xmode = 0; k.ii = i; k.xside = 0;
    if (i > g.nx) k.xmode = 2;
    else if (i < 0 || i >= g.nx) {
        k.xside = (i < 0) ? XLO : XHI;
        const int bc = g.bc[k.xside];
        if (bc == BC_DIRICHLET) { k.xmode = 1; k.ii = 0; }
        else if (bc == BC_PERIODIC) k.ii = (i < 0) ? g.nx - 1 : 0;
        else k.ii = (i < 0) ? 0 : g.nx - 1;
    }

    // prologue: Z = row j0-1 (its north flux = south flux of row j0), X = row j0, Y = raw of row j0+1
    Slot X, Y, Z;
    Z.u = load_row(f, g, k.xmode, k.ii, k.xside, j0 - 1);
    X.u = load_row(f, g, k.xmode, k.ii, k.xside, j0);
    Y.u = load_row(f, g, k.xmode, k.ii, k.xside, j0 + 1);
    cell_closure<SD>(s, k.c, Z.u, Z.q);
    cell_closure<SD>(s, k.c, X.u, X.q);
    {
        FaceF fs;
        cell_face<SD>(s, k.c, g.dy, k.k3y, Z.q.lminy, Z.q.lmaxy, Z.q.f, Z.u.st, X.q.lminy, X.q.lmaxy, X.q.f, X.u.st, fs);
        ARK_FACE_FLUX(fs, Z.u.E, X.u.E, Z.u.Fy, X.u.Fy, Z.u.Fx, X.u.Fx, Z.q.Pyy, X.q.Pyy, Z.q.Pxy, X.q.Pxy, Z.H0, Z.H2, Z.H1, Z.S);
    }
    unsigned int row_off = (unsigned int)j0 * (unsigned int)g.nx + (unsigned int)(i < 0 ? 0 : i);
    const unsigned int nxu = (unsigned int)g.nx;

    int j = j0;
    for (; j + 2 < j1; j += 3) {
        row_step<SD>(g, s, f, k, X, Y, Z, j, j1, row_off, pub, flx, oE, oFx, oFy);
        row_step<SD>(g, s, f, k, Y, Z, X, j + 1, j1, row_off + nxu, pub, flx, oE, oFx, oFy);
        row_step<SD>(g, s, f, k, Z, X, Y, j + 2, j1, row_off + 2 * nxu, pub, flx, oE, oFx, oFy);
        row_off += 3 * nxu;
    }
    if (j < j1) {       // one or two rows left (block-uniform)
        row_step<SD>(g, s, f, k, X, Y, Z, j, j1, row_off, pub, flx, oE, oFx, oFy);
        if (j + 1 < j1) row_step<SD>(g, s, f, k, Y, Z, X, j + 1, j1, row_off + nxu, pub, flx, oE, oFx, oFy);
    }
}

cudaError_t launch_explicit_march3(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                   double* outE, double* outFx, double* outFy, int sm_count, cudaStream_t st)
{
    const int strips = (g.nx + (TX - 2) - 1) / (TX - 2);
    long long want = ((long long)g.ny * strips + (long long)sm_count * 8 - 1) / ((long long)sm_count * 8);
    int RY = (int)(want < 3 ? 3 : (want > 33 ? 33 : want));   // multiples of three rows avoid the remainder path
    RY = (RY + 2) / 3 * 3;
    if (RY > g.ny) RY = g.ny;
    dim3 grd(strips, (g.ny + RY - 1) / RY);
    if (s.is_default()) explicit_march3_kernel<true><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    else explicit_march3_kernel<false><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    return cudaGetLastError();
}

}  // namespace ark
