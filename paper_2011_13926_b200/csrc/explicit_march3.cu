// explicit_march3.cu — row-marching explicit kernel with a FOUR-SLOT register rotation (explicit_kernel = 3, the default).
//
// Same arithmetic and organisation as explicit_march_kernel (column strips, rows marched, one closure per cell, one flux
// per face).  The differences are in how the marching window is held and in what a row step contains:
//  * a slot = {raw state, closure, north-face flux}; the four slots exchange ROLES instead of contents (the row body is a
//    forceinline function instantiated four times with permuted arguments), so no register copy is ever made
//    (explicit_march_kernel shifts its window by ~45 IMAD.MOV per row);
//      row j   : south = A (only its north flux is still alive), centre = B, north = C, closure target = D (row j+2)
//      row j+1 : south = B, centre = C, north = D, target = A      ... and so on, period 4
//  * the closure is computed one row further ahead than the faces need it, so that the closure chain of row j+2 and the
//    face -> update chain of row j are independent inside one basic block (see row_step);
//  * one warp per block: the x-face exchange is done with warp shuffles, there is no barrier at all.
#include "explicit_device.cuh"

namespace ark {

// Block = ONE warp of 32 columns (30 updated + 1 halo lane each side): no hardware barrier, no coupling between warps
// (0.272 ms at 4096^2 against 0.284 with 128 columns).  12 blocks per SM (150 registers) against 16
// (128 registers): 0.2321 against 0.2357 ms with the four-slot window — the fp64 pipe, not the warp count, is the limit.
static constexpr int TX3 = 32;          // threads = columns per block
static constexpr int MARCH3_MINB = 12;   // resident blocks per SM asked of ptxas
static constexpr int MARCH3_RY = 48;     // rows per block (cap; a multiple of 4)

struct Slot {
    Raw u;                      // raw state of the cell
    CloF q;                     // closure (c^2 P, eigenvalues, |f|)
    double H0, H1, H2, S;       // flux through the NORTH face of the cell (E, Fx, Fy rows) and sigma_n (Fy_j + Fy_j+1)
};

struct March3Ctx {
    double c, cdt, dt, rdx, rdy, k3x, k3y, qc;
    int xmode, ii, xside, t;
    bool upd, wb;
    // branch-free loader of the hot loop: value of plane p in grid row j = bp[j * stride]
    //   grid column: bp = plane + ii, stride = nx;  Dirichlet x-ghost: bp = ghost column, stride = 1;  inactive lane: cell 0, stride = 0
    const double *bE, *bFx, *bFy, *bst, *bsa;
    unsigned int stride;
};

// The raw rows travel HBM -> shared memory with cp.async (LDGSTS), three rows ahead of their use, each thread into its own
// slots of ring[row mod 4][field][thread]: the request holds no registers, so ptxas has no reason to sink it towards the
// use (with plain loads it did, and the exposed latency cost more than the copies saved).
// FAST: row j+5 is known to be a grid row (0 <= j+5 < ny): five unconditional copies from the thread's base pointers.
//
// One row step = update of row j.  The closure is taken ONE ROW FURTHER AHEAD than the faces need it: the step computes the
// closure of row j+2 (slot Q) while the north face (rows j, j+1), the east face and the update of row j use closures that
// were finished in earlier steps.  The long closure chain (4 MUFU-seeded roots in sequence) and the face -> update chain are
// then independent inside one basic block and overlap; with the closure of row j+1 computed in the same step (the three-slot
// form) the step was one serial chain closure -> north face -> update per warp (DFMA dependent-issue latency on B200: 8.4
// cycles, ark_m1_fp64_issue_rate).
template <bool SD, bool FAST, bool COUPLED>
__device__ __forceinline__ void row_step(const Grid& g, const Scheme& s, const Fields& f, const March3Ctx& k,
                                         Slot& P, Slot& C, Slot& N, Slot& Q, int j, int j1, unsigned int row_off,
                                         double (*ringQ)[TX3], double (*ringR)[TX3],
                                         double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy,
                                         double* __restrict__ oT)
{
    // COUPLED (stage 2, Eq. 4): the matter planes of the centre row are only needed by the update at the end of the row step;
    // their loads are issued here so that the closure work hides the latency
    double Tm = 0.0, rcv = 1.0, srcE = 0.0;
    const bool coupled_on = COUPLED && k.upd && !(!SD && s.src_off);
    if (coupled_on) {
        if (f.T) { Tm = f.T[row_off]; if (f.rho_cv) rcv = f.rho_cv[row_off]; }
        if (f.source_E) srcE = f.source_E[row_off];
    }
    // request row j+5 into the ring slot of row j+1 (read one step ago), then take row j+2 (fourth youngest group) out of the ring
    if (FAST) {
        const unsigned int o = (unsigned int)(j + 5) * k.stride;
        cp_async8(&ringR[0][k.t], k.bE + o); cp_async8(&ringR[1][k.t], k.bFx + o); cp_async8(&ringR[2][k.t], k.bFy + o);
        cp_async8(&ringR[3][k.t], k.bst + o); cp_async8(&ringR[4][k.t], k.bsa + o);
        cp_async_commit();
    } else load_row_async<TX3>(ringR, k.t, f, g, k.xmode, k.ii, k.xside, j + 5, j + 5 <= j1);
    cp_async_wait<3>();
    Q.u.E = ringQ[0][k.t]; Q.u.Fx = ringQ[1][k.t]; Q.u.Fy = ringQ[2][k.t]; Q.u.st = ringQ[3][k.t]; Q.u.sa = ringQ[4][k.t];
    // publish the x-face data of the centre cell
    XPub me; me.E = C.u.E; me.Fx = C.u.Fx; me.Fy = C.u.Fy; me.Pxx = C.q.Pxx; me.Pxy = C.q.Pxy;
    me.lmin = C.q.lminx; me.lmax = C.q.lmaxx; me.f = C.q.f; me.st = C.u.st;
    // ... to the west neighbour (lane t reads lane t+1) by warp shuffle: no shared memory, no synchronisation
    XPub R;
    R.E = __shfl_down_sync(0xffffffffu, me.E, 1); R.Fx = __shfl_down_sync(0xffffffffu, me.Fx, 1); R.Fy = __shfl_down_sync(0xffffffffu, me.Fy, 1);
    R.Pxx = __shfl_down_sync(0xffffffffu, me.Pxx, 1); R.Pxy = __shfl_down_sync(0xffffffffu, me.Pxy, 1);
    R.lmin = __shfl_down_sync(0xffffffffu, me.lmin, 1); R.lmax = __shfl_down_sync(0xffffffffu, me.lmax, 1);
    R.f = __shfl_down_sync(0xffffffffu, me.f, 1); R.st = __shfl_down_sync(0xffffffffu, me.st, 1);
    // closure of row j+2, north face and east face of row j: one basic block of independent chains
    cell_closure<SD>(s, k.c, Q.u, Q.q);
    FaceF fn;
    cell_face<SD>(s, k.c, g.dy, k.k3y, C.q.lminy, C.q.lmaxy, C.q.f, C.u.st, N.q.lminy, N.q.lmaxy, N.q.f, N.u.st, fn);
    ARK_FACE_FLUX(fn, C.u.E, N.u.E, C.u.Fy, N.u.Fy, C.u.Fx, N.u.Fx, C.q.Pyy, N.q.Pyy, C.q.Pxy, N.q.Pxy, C.H0, C.H2, C.H1, C.S);
    double Ge0, Ge1, Ge2, Se;
    {
        FaceF fe;
        cell_face<SD>(s, k.c, g.dx, k.k3x, me.lmin, me.lmax, me.f, me.st, R.lmin, R.lmax, R.f, R.st, fe);
        ARK_FACE_FLUX(fe, me.E, R.E, me.Fx, R.Fx, me.Fy, R.Fy, me.Pxx, R.Pxx, me.Pxy, R.Pxy, Ge0, Ge1, Ge2, Se);
    }
    {   // the west flux is the east flux of lane t-1
        const double Gw0 = __shfl_up_sync(0xffffffffu, Ge0, 1), Gw1 = __shfl_up_sync(0xffffffffu, Ge1, 1);
        const double Gw2 = __shfl_up_sync(0xffffffffu, Ge2, 1), Sw = __shfl_up_sync(0xffffffffu, Se, 1);
        double dSFx, dSFy;   // -dt * S^F
        if (k.wb) { dSFx = k.qc * (Se + Sw); dSFy = k.qc * (C.S + P.S); }
        else { dSFx = k.dt * k.c * C.u.st * C.u.Fx; dSFy = k.dt * k.c * C.u.st * C.u.Fy; }
        double dSE = k.cdt * C.u.sa * C.u.E;
        if (coupled_on) {       // emission c sigma_a a_r T^4, source_E, explicit matter-energy update of Eq. 4
            if (f.T) {
                const double Theta = s.a_r * (Tm * Tm) * (Tm * Tm);
                dSE -= k.cdt * C.u.sa * Theta;
                if (oT) oT[row_off] = Tm - k.cdt * C.u.sa * (Theta - C.u.E) / rcv;
            }
            dSE -= k.dt * srcE;
        }
        if (!SD && s.src_off) { dSE = 0.0; dSFx = 0.0; dSFy = 0.0; }     // semi-implicit step: hyperbolic part only
        const double nE  = C.u.E  - fma(k.rdx, Ge0 - Gw0, fma(k.rdy, C.H0 - P.H0, dSE));
        const double nFx = C.u.Fx - fma(k.rdx, Ge1 - Gw1, fma(k.rdy, C.H1 - P.H1, dSFx));
        const double nFy = C.u.Fy - fma(k.rdx, Ge2 - Gw2, fma(k.rdy, C.H2 - P.H2, dSFy));
        if (k.upd) { oE[row_off] = nE; oFx[row_off] = nFx; oFy[row_off] = nFy; }
    }
}

template <bool SD, bool COUPLED>
__global__ void __launch_bounds__(TX3, MARCH3_MINB) explicit_march3_kernel(Grid g, Scheme s, Fields f, double dt, int RY,
                                                            double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy,
                                                            double* __restrict__ oT)
{
    __shared__ double ring[4][5][TX3];     // raw rows in flight: row r lives in ring[r mod 4]
    March3Ctx k;
    k.t = threadIdx.x;
    const int i = blockIdx.x * (TX3 - 2) - 1 + k.t;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    k.upd = (k.t >= 1 && k.t <= TX3 - 2 && i >= 0 && i < g.nx);
    k.c = g.c; k.dt = dt; k.cdt = g.c * dt;
    k.rdx = dt / g.dx; k.rdy = dt / g.dy;
    k.k3x = 1.5 * g.dx / g.c; k.k3y = 1.5 * g.dy / g.c;     // 3 delta/(2c): FaceF.sig is sigma_L + sigma_R
    k.qc = 0.125 * g.c * dt;                                   // Eqs. 18-19: 1/4, times the 1/2 of sigma_f
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

    if (k.xmode == 0) { k.bE = f.E + k.ii; k.bFx = f.Fx + k.ii; k.bFy = f.Fy + k.ii; k.bst = f.st + k.ii; k.bsa = f.sa + k.ii; k.stride = (unsigned int)g.nx; }
    else if (k.xmode == 1) { k.bE = f.gh[k.xside][0]; k.bFx = f.gh[k.xside][1]; k.bFy = f.gh[k.xside][2]; k.bsa = f.gh[k.xside][3]; k.bst = f.gh[k.xside][4]; k.stride = 1u; }
    else { k.bE = f.E; k.bFx = f.Fx; k.bFy = f.Fy; k.bst = f.st; k.bsa = f.sa; k.stride = 0u; }

    // prologue: A = row j0-1 (only its north flux = south flux of row j0 is kept), B = row j0, C = row j0+1 with closures;
    // rows j0+2 .. j0+4 requested into the ring
    Slot A, B, C, D;
    A.u = load_row(f, g, k.xmode, k.ii, k.xside, j0 - 1);
    B.u = load_row(f, g, k.xmode, k.ii, k.xside, j0);
    C.u = load_row(f, g, k.xmode, k.ii, k.xside, j0 + 1);
    load_row_async<TX3>(ring[(j0 + 2) % 4], k.t, f, g, k.xmode, k.ii, k.xside, j0 + 2, j0 + 2 <= j1);
    load_row_async<TX3>(ring[(j0 + 3) % 4], k.t, f, g, k.xmode, k.ii, k.xside, j0 + 3, j0 + 3 <= j1);
    load_row_async<TX3>(ring[(j0 + 4) % 4], k.t, f, g, k.xmode, k.ii, k.xside, j0 + 4, j0 + 4 <= j1);
    cell_closure<SD>(s, k.c, A.u, A.q);
    cell_closure<SD>(s, k.c, B.u, B.q);
    cell_closure<SD>(s, k.c, C.u, C.q);
    {
        FaceF fs;
        cell_face<SD>(s, k.c, g.dy, k.k3y, A.q.lminy, A.q.lmaxy, A.q.f, A.u.st, B.q.lminy, B.q.lmaxy, B.q.f, B.u.st, fs);
        ARK_FACE_FLUX(fs, A.u.E, B.u.E, A.u.Fy, B.u.Fy, A.u.Fx, B.u.Fx, A.q.Pyy, B.q.Pyy, A.q.Pxy, B.q.Pxy, A.H0, A.H2, A.H1, A.S);
    }
    unsigned int row_off = (unsigned int)j0 * (unsigned int)g.nx + (unsigned int)(i < 0 ? 0 : i);
    const unsigned int nxu = (unsigned int)g.nx;

    int j = j0;
    // hot loop: four rows per trip, every requested row (j+5 .. j+8) inside the grid.  RY is a multiple of 4 (launcher), so
    // j mod 4 == 0 at every trip and the ring slots are compile-time constants; the four slots exchange roles, not contents.
    const int jfast = min(j1, g.ny - 5);
    if (j0 % 4 == 0) {
        for (; j + 3 < jfast; j += 4) {
            row_step<SD, true, COUPLED>(g, s, f, k, A, B, C, D, j,     j1, row_off,           ring[2], ring[1], oE, oFx, oFy, oT);
            row_step<SD, true, COUPLED>(g, s, f, k, B, C, D, A, j + 1, j1, row_off + nxu,     ring[3], ring[2], oE, oFx, oFy, oT);
            row_step<SD, true, COUPLED>(g, s, f, k, C, D, A, B, j + 2, j1, row_off + 2 * nxu, ring[0], ring[3], oE, oFx, oFy, oT);
            row_step<SD, true, COUPLED>(g, s, f, k, D, A, B, C, j + 3, j1, row_off + 3 * nxu, ring[1], ring[0], oE, oFx, oFy, oT);
            row_off += 4 * nxu;
        }
    }
    // remaining rows (block-uniform trip count): general loader, the window is shifted by copies
    for (; j < j1; ++j) {
        row_step<SD, false, COUPLED>(g, s, f, k, A, B, C, D, j, j1, row_off, ring[(j + 2) % 4], ring[(j + 1) % 4], oE, oFx, oFy, oT);
        const Slot T = A; A = B; B = C; C = D; D = T;
        row_off += nxu;
    }
}

cudaError_t launch_explicit_march3(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                   double* outE, double* outFx, double* outFy, double* outT, int sm_count, cudaStream_t st)
{
    const int strips = (g.nx + (TX3 - 2) - 1) / (TX3 - 2);
    long long want = ((long long)g.ny * strips + (long long)sm_count * 8 - 1) / ((long long)sm_count * 8);
    int RY = (int)(want < 4 ? 4 : (want > MARCH3_RY ? MARCH3_RY : want));   // multiples of four rows avoid the remainder path
    RY = (RY + 3) / 4 * 4;
    if (RY > g.ny) RY = g.ny;
    if ((long long)g.nx * g.ny >= (1LL << 31) || (g.ny + RY - 1) / RY > 65535) return cudaErrorInvalidConfiguration;   // 32-bit in-plane offsets; gridDim.y
    dim3 grd(strips, (g.ny + RY - 1) / RY);
    const bool coupled = (f.T != nullptr) || (f.source_E != nullptr);
    if (coupled) {
        if (s.is_default()) explicit_march3_kernel<true, true><<<grd, TX3, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, outT);
        else explicit_march3_kernel<false, true><<<grd, TX3, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, outT);
    } else {
        if (s.is_default()) explicit_march3_kernel<true, false><<<grd, TX3, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, nullptr);
        else explicit_march3_kernel<false, false><<<grd, TX3, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy, nullptr);
    }
    return cudaGetLastError();
}

}  // namespace ark
