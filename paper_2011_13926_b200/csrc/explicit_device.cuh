// explicit_device.cuh — device helpers shared by the optimised explicit kernels (explicit_march.cu, explicit_march3.cu):
// row loaders with boundary handling, the fast default-scheme closure and face forms, the face-flux macro.
#pragma once
#include "ark_m1_internal.h"

namespace ark {

static constexpr int TX = 128;         // columns per block of explicit_march_kernel (126 updated + 2 halo)
static constexpr int MARCH_RY = 32;    // rows per block (cap)

struct Raw { double E, Fx, Fy, st, sa; };

// Row loader with boundary handling.  The column is resolved once per thread (xmode/ii), so that the common case
// (interior row) costs one multiply-add and five loads.
//   xmode 0: column ii of the grid (after periodic wrap / outflow clamp);  1: Dirichlet x-ghost of side xside;  2: inactive.
// j may be -1 or ny (y ghost).  Corner ghosts are never used by a 5-point stencil and return a dummy state.
__device__ __forceinline__ Raw load_row_general(const Fields& f, const Grid& g, int xmode, int ii, int xside, int j);

// Hot path first (interior row of a grid column: no default values are materialised), everything else in load_row_general.
__device__ __forceinline__ Raw load_row(const Fields& f, const Grid& g, int xmode, int ii, int xside, int j)
{
    if (xmode == 0 && (unsigned int)j < (unsigned int)g.ny) {
        Raw r;
        const unsigned int id = (unsigned int)j * (unsigned int)g.nx + (unsigned int)ii;
        r.E = f.E[id]; r.Fx = f.Fx[id]; r.Fy = f.Fy[id]; r.st = f.st[id]; r.sa = f.sa[id];
        return r;
    }
    return load_row_general(f, g, xmode, ii, xside, j);
}

__device__ __forceinline__ Raw load_row_general(const Fields& f, const Grid& g, int xmode, int ii, int xside, int j)
{
    Raw r; r.E = 1.0; r.Fx = 0.0; r.Fy = 0.0; r.st = 0.0; r.sa = 0.0;
    if (xmode == 2) return r;
    if (j >= 0 && j < g.ny) {
        if (xmode == 0) {
            const unsigned int id = (unsigned int)j * (unsigned int)g.nx + (unsigned int)ii;
            r.E = f.E[id]; r.Fx = f.Fx[id]; r.Fy = f.Fy[id]; r.st = f.st[id]; r.sa = f.sa[id];
        } else {
            r.E = f.gh[xside][0][j]; r.Fx = f.gh[xside][1][j]; r.Fy = f.gh[xside][2][j]; r.sa = f.gh[xside][3][j]; r.st = f.gh[xside][4][j];
        }
        return r;
    }
    if (xmode != 0) return r;                       // corner
    const int side = (j < 0) ? YLO : YHI;
    const int bc = g.bc[side];
    if (bc == BC_DIRICHLET || bc == BC_HALO) {
        r.E = f.gh[side][0][ii]; r.Fx = f.gh[side][1][ii]; r.Fy = f.gh[side][2][ii]; r.sa = f.gh[side][3][ii]; r.st = f.gh[side][4][ii];
        return r;
    }
    const int jj = (bc == BC_PERIODIC) ? ((j < 0) ? g.ny - 1 : 0) : ((j < 0) ? 0 : g.ny - 1);
    const long long id = (long long)jj * g.nx + ii;
    r.E = f.E[id]; r.Fx = f.Fx[id]; r.Fy = f.Fy[id]; r.st = f.st[id]; r.sa = f.sa[id];
    return r;
}

// Asynchronous variant of load_row: the five values of one cell go straight from global to this
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
            if (bc == BC_DIRICHLET || bc == BC_HALO) {
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
struct CloF { double Pxx, Pxy, Pyy, lminx, lmaxx, lminy, lmaxy, f; };   // Pxx.. hold c^2 P (what the flux needs); f = |f|/2

// Default-scheme closure with 2 reciprocals and 4 reciprocal square roots per cell:
//   1/(cE);  rs = 1/sqrt(4 - 3 f^2) gives xi = s rs and 1/xi = rs;  the reciprocal of 2 + xi (anisotropic part and the
//   eigenvalue prefactor; chi itself is (5 - 2 xi)/3, no division);  |f| and the two eigenvalue roots as x rsqrt(x).
__device__ __forceinline__ void closure_fast(double c, double E, double Fx, double Fy, CloF& q)
{
    const double Es = dmax_sel(E, ARK_E_FLOOR);
    const double ice = rcp_fast3(c * Es);
    double fx = Fx * ice, fy = Fy * ice;
    // f^2 + 1e-300 (folded into the fma): the reciprocal square root below needs no guard for F = 0
    const double f2raw = fma(fx, fx, fma(fy, fy, 1e-300));
    // |f| and the clamp of PAPER.md:513, branch-free: one rsqrt serves both (f = f2 rsqrt(f2); rescale by rsqrt(f2) if f2 > 1).
    // (A warp-uniform branch around the rare clamp/overflow selects was measured: no gain, it splits the row's basic block.)
    const bool huge = !(f2raw <= 1e300);          // E <= 0 (floored): F/(cE) overflows; 1/sqrt(inf) = 0 like IEEE
    const double rf = rsqrt_fast(huge ? 1.0 : f2raw);
    const bool clamp = f2raw > 1.0;
    const double sc = clamp ? (huge ? 0.0 : rf) : 1.0;
    fx *= sc; fy *= sc;
    const double f2 = clamp ? 1.0 : f2raw;
    const double fh = clamp ? 0.5 : (0.5 * f2raw) * rf;      // |f|/2: the face needs (f_L + f_R)/2
    q.f = fh;
    const double s = 4.0 - 3.0 * f2;       // >= 1
    const double rs = rsqrt_fast(s);
    const double xi = s * rs;
    // chi = (3 + 4 f^2)/(5 + 2 xi) needs no division: xi^2 = 4 - 3 f^2 gives 3 + 4 f^2 = (25 - 4 xi^2)/3 =
    // (5 - 2 xi)(5 + 2 xi)/3, so chi = (5 - 2 xi)/3, the isotropic part (1 - chi)/2 = (xi - 1)/3 and the anisotropic
    // coefficient (3 chi - 1)/(2 f^2) = (2 - xi)/f^2 = 3/(2 + xi): one reciprocal, of 2 + xi, serves the pressure and Eq. 14
    const double t2 = 2.0 + xi, xm1 = xi - 1.0;
    const double i2 = rcp_fast3(t2);                    // 1/(2+xi)
    const double c2 = c * c;                            // uniform: hoisted out of the row loop
    const double Eq = E * ((3.0 * c2) * i2), Ei = E * ((0.33333333333333333333 * c2) * xm1);   // c^2 folded into the stored pressure
    q.Pxx = fma(Eq * fx, fx, Ei); q.Pxy = Eq * fx * fy; q.Pyy = fma(Eq * fy, fy, Ei);
    // Eq. 14
    const double a = xm1 * t2;
    const double crs = c * rs;                                // c/xi
    const double k = 1.41421356237309504880 * crs * i2;       // c sqrt(2/3)/(xi (xi+2)) times the sqrt(3) taken out of the roots
    const double a23 = 0.66666666666666666667 * a;
    // roots of Eq. 14: sqrt(a (3 f_t^2 + 2a)) = sqrt(3) sqrt(a (f_t^2 + 2a/3)).  x' = x + 1e-200 folded into the product's fma:
    // branch-free, and x = 0 (f = 1) gives ~1e-100 instead of 0 (the eigenvalues are O(c); 1e-100 is below every rounding
    // error of the path).  It also makes l+ - l- > 0 on every face (face_fast needs no zero-width guard).
    const double rx = k * sqrt_core(fma(a, fma(fy, fy, a23), 1e-200));
    const double ry = k * sqrt_core(fma(a, fma(fx, fx, a23), 1e-200));
    const double mx = fx * crs, my = fy * crs;
    q.lmaxx = mx + rx; q.lminx = mx - rx;
    q.lmaxy = my + ry; q.lminy = my - ry;
}

// Face coefficients with ONE reciprocal.  With D = dl - kk l+ l- (kk = 3 sigma_f delta (1 - f_f^2)/c >= 0, l+ l- <= 0):
//   1/dl = D/(dl D),  alpha = 1/(1 - kk Lambda) = dl/D = dl^2/(dl D).   a- = 1 - a+ is never formed: the fluxes use
//   a+ x_L + a- x_R = x_R + a+ (x_L - x_R).
struct FaceF { double ap, Lam, alpha, sig; };     // sig = sigma_L + sigma_R = TWICE the face opacity of Eq. 18 (the 1/2 sits in k3h and qc)
__device__ __forceinline__ void face_fast(double k3h, double lminL, double lmaxL, double fL, double stL,
                                          double lminR, double lmaxR, double fR, double stR, FaceF& fc)
{
    const double lp = dmax_sel(dmax_sel(lmaxL, lmaxR), 0.0);
    const double lm = dmin_sel(dmin_sel(lminL, lminR), 0.0);
    const double dl = lp - lm;
    fc.sig = stL + stR;
    const double ff = fL + fR;             // the cells store |f|/2
    const double kk = k3h * fc.sig * fma(-ff, ff, 1.0);
    // dl > 0 always: closure_fast's eigenvalue roots are >= ~1e-101 c, so (l+, l-) = (0, 0) cannot occur; on a face between
    // cells with f = 1 exactly along the face, dl ~ 1e-100 c gives a+ = 1/2, Lambda ~ -1e-101 c, alpha = 1 (the oracle's guard
    // values 1/2, 0, 1)
    const double D = fma(-kk * lp, lm, dl);
    const double qq = rcp_fast3(dl * D);
    fc.ap = lp * (qq * D);
    fc.Lam = lm * fc.ap;                   // l+ l-/dl
    fc.alpha = dl * (dl * qq);
}

// Scheme dispatch: the default scheme uses the fast forms above, every other switch combination the generic ones.
template <bool SD>
__device__ __forceinline__ void cell_closure(const Scheme& s, double c, const Raw& u, CloF& q)
{
    if (SD) closure_fast(c, u.E, u.Fx, u.Fy, q);
    else {
        Clo t; closure_eval<false, false>(s, c, u.E, u.Fx, u.Fy, t, nullptr);
        const double c2 = c * c;
        q.Pxx = c2 * t.Pxx; q.Pxy = c2 * t.Pxy; q.Pyy = c2 * t.Pyy; q.f = 0.5 * t.f;
        q.lminx = t.lmin[0]; q.lmaxx = t.lmax[0]; q.lminy = t.lmin[1]; q.lmaxy = t.lmax[1];
    }
}
// k3h = 3 delta/(2c): Eq. 25's 3 sigma_f delta (1 - f_f^2)/c = k3h (sigma_L + sigma_R)(1 - f_f^2)
template <bool SD>
__device__ __forceinline__ void cell_face(const Scheme& s, double c, double delta, double k3h,
                                          double lminL, double lmaxL, double fL, double stL,
                                          double lminR, double lmaxR, double fR, double stR, FaceF& fc)
{
    if (SD) face_fast(k3h, lminL, lmaxL, fL, stL, lminR, lmaxR, fR, stR, fc);
    else {
        Face t; face_eval<false>(s, c, delta, lminL, lmaxL, 2.0 * fL, stL, lminR, lmaxR, 2.0 * fR, stR, t);
        fc.ap = t.ap; fc.Lam = t.Lam; fc.alpha = t.alpha; fc.sig = 2.0 * t.sig;     // a+ + a- = 1 in every scheme variant
    }
}

// Flux of Eq. 13 through one face (normal component Fn, pressures already times c^2):
//   G0 = alpha (a+ Fn_L + a- Fn_R + Lam (E_R - E_L)),  G1/G2 = a+ P_L + a- P_R + Lam (F_R - F_L),  S = (sigma_L + sigma_R)(Fn_L + Fn_R) = 2 sigma_f (Fn_L + Fn_R)
#define ARK_FACE_FLUX(fc, EL, ER, FnL, FnR, FtL, FtR, PnL, PnR, PtL, PtR, G0, Gn, Gt, S)              \
    do {                                                                                             \
        const double dFn_ = (FnR) - (FnL);                                                           \
        G0 = (fc).alpha * fma((fc).Lam, (ER) - (EL), fma(-(fc).ap, dFn_, (FnR)));                    \
        Gn = fma((fc).Lam, dFn_, fma((fc).ap, (PnL) - (PnR), (PnR)));                                \
        Gt = fma((fc).Lam, (FtR) - (FtL), fma((fc).ap, (PtL) - (PtR), (PtR)));                       \
        S = (fc).sig * ((FnL) + (FnR));                                                              \
    } while (0)


}  // namespace ark
