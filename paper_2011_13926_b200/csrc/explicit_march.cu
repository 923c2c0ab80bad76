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

// tuning knobs (defaults chosen by measurement on B200)
#ifndef ARK_MARCH_TX
#define ARK_MARCH_TX 128
#endif
#ifndef ARK_MARCH_UNROLL
#define ARK_MARCH_UNROLL 1
#endif
#ifndef ARK_MARCH_MINB
#define ARK_MARCH_MINB 4
#endif
#ifndef ARK_MARCH_RY
#define ARK_MARCH_RY 32
#endif
#ifndef ARK_MARCH_ASYNC
#define ARK_MARCH_ASYNC 0   // 1: prefetch rows with cp.async into a shared-memory ring
#endif
static constexpr int TX = ARK_MARCH_TX;

struct Raw { double E, Fx, Fy, st, sa; };

// Row loader with boundary handling.  The column is resolved once per thread (xmode/ii), so that the common case
// (interior row) costs one multiply-add and five loads.
//   xmode 0: column ii of the grid (after periodic wrap / outflow clamp);  1: Dirichlet x-ghost of side xside;  2: inactive.
// j may be -1 or ny (y ghost).  Corner ghosts are never used by a 5-point stencil and return a dummy state.
#ifndef ARK_MARCH_PINLOAD
#define ARK_MARCH_PINLOAD 0     // 1: the hot-path loads are volatile asm, so that ptxas cannot sink the prefetch
#endif
__device__ __forceinline__ double ld_pinned(const double* p)
{
#if ARK_MARCH_PINLOAD
    double x;
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(x) : "l"(p) : "memory");
    return x;
#else
    return *p;
#endif
}

__device__ __forceinline__ Raw load_row(const Fields& f, const Grid& g, int xmode, int ii, int xside, int j)
{
    Raw r; r.E = 1.0; r.Fx = 0.0; r.Fy = 0.0; r.st = 0.0; r.sa = 0.0;
    if (xmode == 2) return r;
    if (j >= 0 && j < g.ny) {
        if (xmode == 0) {
            const unsigned int id = (unsigned int)j * (unsigned int)g.nx + (unsigned int)ii;
            r.E = ld_pinned(f.E + id); r.Fx = ld_pinned(f.Fx + id); r.Fy = ld_pinned(f.Fy + id); r.st = ld_pinned(f.st + id); r.sa = ld_pinned(f.sa + id);
        } else {
            r.E = f.gh[xside][0][j]; r.Fx = f.gh[xside][1][j]; r.Fy = f.gh[xside][2][j]; r.sa = f.gh[xside][3][j]; r.st = f.gh[xside][4][j];
        }
        return r;
    }
    if (xmode != 0) return r;                       // corner
    const int side = (j < 0) ? YLO : YHI;
    const int bc = g.bc[side];
    if (bc == BC_DIRICHLET) {
        r.E = f.gh[side][0][ii]; r.Fx = f.gh[side][1][ii]; r.Fy = f.gh[side][2][ii]; r.sa = f.gh[side][3][ii]; r.st = f.gh[side][4][ii];
        return r;
    }
    const int jj = (bc == BC_PERIODIC) ? ((j < 0) ? g.ny - 1 : 0) : ((j < 0) ? 0 : g.ny - 1);
    const long long id = (long long)jj * g.nx + ii;
    r.E = f.E[id]; r.Fx = f.Fx[id]; r.Fy = f.Fy[id]; r.st = f.st[id]; r.sa = f.sa[id];
    return r;
}

// Asynchronous variant of load_row (ARK_MARCH_ASYNC): the five values of one cell go straight from global to this
// thread's own slots of a shared-memory ring with cp.async (LDGSTS), so no registers are held while the request is in
// flight and the compiler cannot sink the prefetch towards its use.  A thread only ever reads back its own slots,
// hence cp.async.wait_group is the only synchronisation needed.  ring layout: [stage][field][thread].
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc)
{
    const unsigned int d = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

template <int TXN>
__device__ __forceinline__ void load_row_async(double (*ring)[TXN], int t, const Fields& f, const Grid& g,
                                               int xmode, int ii, int xside, int j, bool wanted)
{
    // ring points at [field][thread] of the target stage; order of fields: E, Fx, Fy, st, sa
    const double* p0 = nullptr; const double* p1; const double* p2; const double* p3; const double* p4;
    if (wanted && xmode != 2 && j <= g.ny) {
        if (j >= 0 && j < g.ny) {
            if (xmode == 0) {
                const unsigned int id = (unsigned int)j * (unsigned int)g.nx + (unsigned int)ii;
                p0 = f.E + id; p1 = f.Fx + id; p2 = f.Fy + id; p3 = f.st + id; p4 = f.sa + id;
            } else {
                p0 = f.gh[xside][0] + j; p1 = f.gh[xside][1] + j; p2 = f.gh[xside][2] + j; p3 = f.gh[xside][4] + j; p4 = f.gh[xside][3] + j;
            }
        } else if (xmode == 0) {
            const int side = (j < 0) ? YLO : YHI;
            const int bc = g.bc[side];
            if (bc == BC_DIRICHLET) {
                p0 = f.gh[side][0] + ii; p1 = f.gh[side][1] + ii; p2 = f.gh[side][2] + ii; p3 = f.gh[side][4] + ii; p4 = f.gh[side][3] + ii;
            } else {
                const int jj = (bc == BC_PERIODIC) ? ((j < 0) ? g.ny - 1 : 0) : ((j < 0) ? 0 : g.ny - 1);
                const unsigned int id = (unsigned int)jj * (unsigned int)g.nx + (unsigned int)ii;
                p0 = f.E + id; p1 = f.Fx + id; p2 = f.Fy + id; p3 = f.st + id; p4 = f.sa + id;
            }
        }
    }
    if (p0) {
        cp_async8(&ring[0][t], p0); cp_async8(&ring[1][t], p1); cp_async8(&ring[2][t], p2);
        cp_async8(&ring[3][t], p3); cp_async8(&ring[4][t], p4);
    } else {   // dummy state (inactive column, corner ghost, row not needed)
        ring[0][t] = 1.0; ring[1][t] = 0.0; ring[2][t] = 0.0; ring[3][t] = 0.0; ring[4][t] = 0.0;
    }
    cp_async_commit();
}

struct XPub { double E, Fx, Fy, Pxx, Pxy, lmin, lmax, f, st; };   // what the west neighbour needs for its east face

// What the march kernel keeps per cell: pressure, Eq. 14 eigenvalues for both face orientations, |f|.
struct CloF { double Pxx, Pxy, Pyy, lminx, lmaxx, lminy, lmaxy, f; };   // Pxx.. hold c^2 P (what the flux needs)

// Default-scheme closure with 2 reciprocals and 4 reciprocal square roots per cell:
//   1/(cE);  rs = 1/sqrt(4 - 3 f^2) gives xi = s rs and 1/xi = rs;  one reciprocal of (2+xi)(5+2xi) gives both
//   1/(5+2xi) (for chi) and 1/(2+xi) (for the anisotropic part and the eigenvalue prefactor);  |f| and the two
//   eigenvalue roots as x rsqrt(x).
__device__ __forceinline__ void closure_fast(double c, double E, double Fx, double Fy, CloF& q)
{
    const double Es = (E > ARK_E_FLOOR) ? E : ARK_E_FLOOR;
    const double ice = rcp_fast(c * Es);
    double fx = Fx * ice, fy = Fy * ice;
    const double f2raw = fx * fx + fy * fy;
    // |f| and the clamp of PAPER.md:513, branch-free: one rsqrt serves both (f = f2 rsqrt(f2); rescale by rsqrt(f2) if f2 > 1)
    const bool tiny = !(f2raw > 1e-290);
    const bool huge = !(f2raw <= 1e300);          // E <= 0 (floored): F/(cE) overflows; 1/sqrt(inf) = 0 like IEEE
    const double rf = rsqrt_fast((tiny || huge) ? 1.0 : f2raw);
    const bool clamp = f2raw > 1.0;
    const double sc = clamp ? (huge ? 0.0 : rf) : 1.0;
    fx *= sc; fy *= sc;
    const double f2 = clamp ? 1.0 : f2raw;
    q.f = clamp ? 1.0 : (tiny ? 0.0 : f2raw * rf);
    const double s = 4.0 - 3.0 * f2;       // >= 1
    const double rs = rsqrt_fast(s);
    const double xi = s * rs;
    const double t2 = 2.0 + xi, t5 = 5.0 + 2.0 * xi;
    const double rp = rcp_fast(t2 * t5);
    const double i2 = rp * t5, i5 = rp * t2;            // 1/(2+xi), 1/(5+2xi)
    const double chi = (3.0 + 4.0 * f2) * i5;
    const double q3 = 3.0 * i2;
    const double iso = 0.5 - 0.5 * chi;
    const double Ec = (c * c) * E;                      // c^2 folded into the stored pressure
    const double Eq = Ec * q3, Ei = Ec * iso;
    q.Pxx = fma(Eq * fx, fx, Ei); q.Pxy = Eq * fx * fy; q.Pyy = fma(Eq * fy, fy, Ei);
    // Eq. 14
    const double a = (xi - 1.0) * t2;
    const double crs = c * rs;                                // c/xi
    const double k = 0.81649658092772603273 * crs * i2;       // c sqrt(2/3)/(xi (xi+2))
    const double a2 = a + a;
    const double rx = k * sqrt_fast(a * fma(3.0 * fy, fy, a2));
    const double ry = k * sqrt_fast(a * fma(3.0 * fx, fx, a2));
    const double mx = fx * crs, my = fy * crs;
    q.lmaxx = mx + rx; q.lminx = mx - rx;
    q.lmaxy = my + ry; q.lminy = my - ry;
}

// Face coefficients with ONE reciprocal.  With D = dl - kk l+ l- (kk = 3 sigma_f delta (1 - f_f^2)/c >= 0, l+ l- <= 0):
//   1/dl = D/(dl D),  alpha = 1/(1 - kk Lambda) = dl/D = dl^2/(dl D).   a- = 1 - a+ is never formed: the fluxes use
//   a+ x_L + a- x_R = x_R + a+ (x_L - x_R).
struct FaceF { double ap, Lam, alpha, sig; };
__device__ __forceinline__ void face_fast(double k3, double lminL, double lmaxL, double fL, double stL,
                                          double lminR, double lmaxR, double fR, double stR, FaceF& fc)
{
    const double lp = fmax(0.0, fmax(lmaxL, lmaxR));
    const double lm = fmin(0.0, fmin(lminL, lminR));
    const double dl = lp - lm;
    fc.sig = 0.5 * (stL + stR);
    const double ff = 0.5 * (fL + fR);
    const double kk = k3 * fc.sig * fma(-ff, ff, 1.0);
    const bool ok = dl > 0.0;
    const double dls = ok ? dl : 1.0;
    const double D = fma(-kk * lp, lm, dls);
    const double qq = rcp_fast(dls * D);
    const double apv = lp * (qq * D);
    fc.ap = ok ? apv : 0.5;
    fc.Lam = lm * apv;                     // l+ l-/dl; 0 when dl == 0 (then l+ = l- = 0)
    fc.alpha = dls * (dls * qq);           // 1 when dl == 0
}

// Scheme dispatch: the default scheme uses the fast forms above, every other switch combination the generic ones.
template <bool SD>
__device__ __forceinline__ void cell_closure(const Scheme& s, double c, const Raw& u, CloF& q)
{
    if (SD) closure_fast(c, u.E, u.Fx, u.Fy, q);
    else {
        Clo t; closure_eval<false, false>(s, c, u.E, u.Fx, u.Fy, t, nullptr);
        const double c2 = c * c;
        q.Pxx = c2 * t.Pxx; q.Pxy = c2 * t.Pxy; q.Pyy = c2 * t.Pyy; q.f = t.f;
        q.lminx = t.lmin[0]; q.lmaxx = t.lmax[0]; q.lminy = t.lmin[1]; q.lmaxy = t.lmax[1];
    }
}
template <bool SD>
__device__ __forceinline__ void cell_face(const Scheme& s, double c, double delta, double k3,
                                          double lminL, double lmaxL, double fL, double stL,
                                          double lminR, double lmaxR, double fR, double stR, FaceF& fc)
{
    if (SD) face_fast(k3, lminL, lmaxL, fL, stL, lminR, lmaxR, fR, stR, fc);
    else {
        Face t; face_eval<false>(s, c, delta, lminL, lmaxL, fL, stL, lminR, lmaxR, fR, stR, t);
        fc.ap = t.ap; fc.Lam = t.Lam; fc.alpha = t.alpha; fc.sig = t.sig;     // a+ + a- = 1 in every scheme variant
    }
}

// Flux of Eq. 13 through one face (normal component Fn, pressures already times c^2):
//   G0 = alpha (a+ Fn_L + a- Fn_R + Lam (E_R - E_L)),  G1/G2 = a+ P_L + a- P_R + Lam (F_R - F_L),  S = sigma_f (Fn_L + Fn_R)
#define ARK_FACE_FLUX(fc, EL, ER, FnL, FnR, FtL, FtR, PnL, PnR, PtL, PtR, G0, Gn, Gt, S)              \
    do {                                                                                             \
        const double dFn_ = (FnR) - (FnL);                                                           \
        G0 = (fc).alpha * fma((fc).Lam, (ER) - (EL), fma(-(fc).ap, dFn_, (FnR)));                    \
        Gn = fma((fc).Lam, dFn_, fma((fc).ap, (PnL) - (PnR), (PnR)));                                \
        Gt = fma((fc).Lam, (FtR) - (FtL), fma((fc).ap, (PtL) - (PtR), (PtR)));                       \
        S = (fc).sig * ((FnL) + (FnR));                                                              \
    } while (0)

template <bool SD>
__global__ void __launch_bounds__(TX, ARK_MARCH_MINB) explicit_march_kernel(Grid g, Scheme s, Fields f, double dt, int RY,
                                                            double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy)
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
    const double k3x = 3.0 * g.dx / c, k3y = 3.0 * g.dy / c;   // Eq. 25: 3 sigma dx (1-f^2)/c = k3 sigma (1-f^2)
    const double qc = 0.25 * c * dt;                            // WB source weight (Eqs. 18-19) times dt
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
#if ARK_MARCH_ASYNC
    __shared__ double ring[3][5][TX];
    load_row_async<TX>(ring[0], t, f, g, xmode, ii, xside, j0 + 1, true);      // slot 0 <- row j0+1
    load_row_async<TX>(ring[1], t, f, g, xmode, ii, xside, j0 + 2, j0 + 1 < j1);
    int slot_n = 0, slot_p = 2;     // slot holding row j+1; slot receiving row j+3
#endif
    Raw uS = load_row(f, g, xmode, ii, xside, j0 - 1);
    Raw uC = load_row(f, g, xmode, ii, xside, j0);
#if !ARK_MARCH_ASYNC
    Raw uN = load_row(f, g, xmode, ii, xside, j0 + 1);
#endif
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

    constexpr int kUnroll = ARK_MARCH_UNROLL;
#pragma unroll kUnroll
    for (int j = j0; j < j1; ++j) {
#if ARK_MARCH_ASYNC
        // request row j+3, then take row j+1 out of the ring (its group is the third youngest)
        load_row_async<TX>(ring[slot_p], t, f, g, xmode, ii, xside, j + 3, j + 2 < j1);
        cp_async_wait<2>();
        Raw uN;
        uN.E = ring[slot_n][0][t]; uN.Fx = ring[slot_n][1][t]; uN.Fy = ring[slot_n][2][t]; uN.st = ring[slot_n][3][t]; uN.sa = ring[slot_n][4][t];
        slot_p = slot_n; slot_n = (slot_n == 2) ? 0 : slot_n + 1;
#else
        // prefetch the raw state two rows ahead
        const Raw uNN = load_row(f, g, (j + 1 < j1) ? xmode : 2, ii, xside, j + 2);
#endif
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
            const double dSE = cdt * uC.sa * uC.E;
            const double nE  = uC.E  - fma(rdx, Ge0 - Gw0, fma(rdy, Hn0 - Hs0, dSE));
            const double nFx = uC.Fx - fma(rdx, Ge1 - Gw1, fma(rdy, Hn1 - Hs1, dSFx));
            const double nFy = uC.Fy - fma(rdx, Ge2 - Gw2, fma(rdy, Hn2 - Hs2, dSFy));
            if (upd) { oE[row_off] = nE; oFx[row_off] = nFx; oFy[row_off] = nFy; }
        }
        row_off += (unsigned int)g.nx;
        // shift the window north
#if ARK_MARCH_ASYNC
        uC = uN; qC = qN;
#else
        uC = uN; qC = qN; uN = uNN;
#endif
        Hs0 = Hn0; Hs1 = Hn1; Hs2 = Hn2; Ss = Sn;
    }
}

// ---------------------------------------------------------------------------------------------------------
// Barrier-free variant: a WARP owns 30 columns (+1 halo lane each side) and exchanges the x-face data with
// __shfl_down/__shfl_up, so warps never wait for one another and the row body is one basic block.
// ---------------------------------------------------------------------------------------------------------
#ifndef ARK_WARP_WPB
#define ARK_WARP_WPB 4      // warps per block
#endif
#ifndef ARK_WARP_MINB
#define ARK_WARP_MINB 4
#endif
static constexpr int WPB = ARK_WARP_WPB;
static constexpr int WCOLS = 30;

__device__ __forceinline__ double shfl_dn(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_up(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }

template <bool SD>
__global__ void __launch_bounds__(32 * WPB, ARK_WARP_MINB) explicit_warp_kernel(Grid g, Scheme s, Fields f, double dt, int RY,
                                                            double* __restrict__ oE, double* __restrict__ oFx, double* __restrict__ oFy)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int i = (blockIdx.x * WPB + warp) * WCOLS - 1 + lane;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    const bool col_active = (i <= g.nx);
    const bool upd = (lane >= 1 && lane <= WCOLS && i >= 0 && i < g.nx);
    const double c = g.c, cdt = c * dt;
    const double rdx = dt / g.dx, rdy = dt / g.dy;
    const double k3x = 3.0 * g.dx / c, k3y = 3.0 * g.dy / c;
    const double qc = 0.25 * c * dt;
    const bool wb = SD ? true : (s.wb != 0);

    int xmode = 0, ii = i, xside = 0;
    if (!col_active) xmode = 2;
    else if (i < 0 || i >= g.nx) {
        xside = (i < 0) ? XLO : XHI;
        const int bc = g.bc[xside];
        if (bc == BC_DIRICHLET) { xmode = 1; ii = 0; }
        else if (bc == BC_PERIODIC) ii = (i < 0) ? g.nx - 1 : 0;
        else ii = (i < 0) ? 0 : g.nx - 1;
    }
    Raw uS = load_row(f, g, xmode, ii, xside, j0 - 1);
    Raw uC = load_row(f, g, xmode, ii, xside, j0);
    Raw uN = load_row(f, g, xmode, ii, xside, j0 + 1);
    CloF qS, qC;
    cell_closure<SD>(s, c, uS, qS);
    cell_closure<SD>(s, c, uC, qC);
    double Hs0, Hs1, Hs2, Ss;
    {
        FaceF fs;
        cell_face<SD>(s, c, g.dy, k3y, qS.lminy, qS.lmaxy, qS.f, uS.st, qC.lminy, qC.lmaxy, qC.f, uC.st, fs);
        ARK_FACE_FLUX(fs, uS.E, uC.E, uS.Fy, uC.Fy, uS.Fx, uC.Fx, qS.Pyy, qC.Pyy, qS.Pxy, qC.Pxy, Hs0, Hs2, Hs1, Ss);
    }
    unsigned int row_off = (unsigned int)j0 * (unsigned int)g.nx + (unsigned int)(i < 0 ? 0 : i);

    for (int j = j0; j < j1; ++j) {
        const Raw uNN = load_row(f, g, (j + 1 < j1) ? xmode : 2, ii, xside, j + 2);
        // east neighbour's x-face data (lane + 1)
        const double RE = shfl_dn(uC.E), RFx = shfl_dn(uC.Fx), RFy = shfl_dn(uC.Fy), RPxx = shfl_dn(qC.Pxx), RPxy = shfl_dn(qC.Pxy);
        const double Rlmin = shfl_dn(qC.lminx), Rlmax = shfl_dn(qC.lmaxx), Rf = shfl_dn(qC.f), Rst = shfl_dn(uC.st);
        // north cell closure + north face
        CloF qN;
        cell_closure<SD>(s, c, uN, qN);
        FaceF fn;
        cell_face<SD>(s, c, g.dy, k3y, qC.lminy, qC.lmaxy, qC.f, uC.st, qN.lminy, qN.lmaxy, qN.f, uN.st, fn);
        double Hn0, Hn1, Hn2, Sn;
        ARK_FACE_FLUX(fn, uC.E, uN.E, uC.Fy, uN.Fy, uC.Fx, uN.Fx, qC.Pyy, qN.Pyy, qC.Pxy, qN.Pxy, Hn0, Hn2, Hn1, Sn);
        // east face
        double Ge0, Ge1, Ge2, Se;
        {
            FaceF fe;
            cell_face<SD>(s, c, g.dx, k3x, qC.lminx, qC.lmaxx, qC.f, uC.st, Rlmin, Rlmax, Rf, Rst, fe);
            ARK_FACE_FLUX(fe, uC.E, RE, uC.Fx, RFx, uC.Fy, RFy, qC.Pxx, RPxx, qC.Pxy, RPxy, Ge0, Ge1, Ge2, Se);
        }
        // west flux = east flux of lane - 1
        const double Gw0 = shfl_up(Ge0), Gw1 = shfl_up(Ge1), Gw2 = shfl_up(Ge2), Sw = shfl_up(Se);
        double dSFx, dSFy;
        if (wb) { dSFx = qc * (Se + Sw); dSFy = qc * (Sn + Ss); }
        else { dSFx = dt * c * uC.st * uC.Fx; dSFy = dt * c * uC.st * uC.Fy; }
        const double dSE = cdt * uC.sa * uC.E;
        const double nE  = uC.E  - fma(rdx, Ge0 - Gw0, fma(rdy, Hn0 - Hs0, dSE));
        const double nFx = uC.Fx - fma(rdx, Ge1 - Gw1, fma(rdy, Hn1 - Hs1, dSFx));
        const double nFy = uC.Fy - fma(rdx, Ge2 - Gw2, fma(rdy, Hn2 - Hs2, dSFy));
        if (upd) { oE[row_off] = nE; oFx[row_off] = nFx; oFy[row_off] = nFy; }
        row_off += (unsigned int)g.nx;
        uC = uN; qC = qN; uN = uNN;
        Hs0 = Hn0; Hs1 = Hn1; Hs2 = Hn2; Ss = Sn;
    }
}

cudaError_t launch_explicit_warp(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                 double* outE, double* outFx, double* outFy, int sm_count, cudaStream_t st)
{
    const int strips = (g.nx + WCOLS * WPB - 1) / (WCOLS * WPB);
    long long want = ((long long)g.ny * strips + (long long)sm_count * 8 - 1) / ((long long)sm_count * 8);
    int RY = (int)(want < 4 ? 4 : (want > ARK_MARCH_RY ? ARK_MARCH_RY : want));
    if (RY > g.ny) RY = g.ny;
    dim3 grd(strips, (g.ny + RY - 1) / RY);
    if (s.is_default()) explicit_warp_kernel<true><<<grd, 32 * WPB, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    else explicit_warp_kernel<false><<<grd, 32 * WPB, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    return cudaGetLastError();
}

cudaError_t launch_explicit_march(const Grid& g, const Scheme& s, const Fields& f, double dt,
                                  double* outE, double* outFx, double* outFy, int sm_count, cudaStream_t st)
{
    const int strips = (g.nx + (TX - 2) - 1) / (TX - 2);
    // rows per block: enough blocks for ~8 per SM, between 4 and ARK_MARCH_RY rows.  (A single wave of
    // SMs x resident-blocks blocks with ~240 rows each was measured 8% slower at 4096^2: uneven blocks per SM.)
    long long want = ((long long)g.ny * strips + (long long)sm_count * 8 - 1) / ((long long)sm_count * 8);
    int RY = (int)(want < 4 ? 4 : (want > ARK_MARCH_RY ? ARK_MARCH_RY : want));
    if (RY > g.ny) RY = g.ny;
    dim3 grd(strips, (g.ny + RY - 1) / RY);
    if (s.is_default()) explicit_march_kernel<true><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    else explicit_march_kernel<false><<<grd, TX, 0, st>>>(g, s, f, dt, RY, outE, outFx, outFy);
    return cudaGetLastError();
}

}  // namespace ark
