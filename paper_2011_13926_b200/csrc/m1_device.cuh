// m1_device.cuh — per-cell and per-face device arithmetic of the AP/WB M1 scheme (arXiv 2011.13926).
//
// PAPER.md passages restated here (never the oracle's code; the two share nothing):
//   closure chi(f) = (3 + 4 f^2)/(5 + 2 sqrt(4 - 3 f^2)), P = D E                 PAPER.md:79  (Sect. 2.2)
//   f > 1: "impose f = 1 in the computation of the Eddington tensor"
//   eigenvalues lambda_max/min of the M1 flux Jacobian                             PAPER.md:170 (Eq. 14)
//   lambda+ = max(0, lambda_max), lambda- = min(0, lambda_min)
//   HLL-type fluxes F*, P*                                                         PAPER.md:162-164 (Eq. 13)
//   AP factor alpha (Eq. 25 = C.9), variant C.8
//   face opacity sigma_{i+1/2} = (sigma_i + sigma_{i+1})/2                         PAPER.md:199 (Eq. 19)
//
// Algebra used: with the reduced flux vector (fx, fy) = F/(cE), xi = sqrt(4-3f^2),
//   (3 chi - 1)/2 * n_a n_b = 3 f_a f_b/(2 + xi)          (no division by |F|, no cancellation at small f)
//   chi'(f) = 2 f/xi,   d(P_ab)/dE = D_ab + (f^2 delta_ab - 3 f_a f_b)/xi
//   d(P_ab)/dF_k = [ f_a f_b f_k (q^2/xi) - delta_ab f_k/xi + q (delta_ak f_b + delta_bk f_a) ]/c,  q = 3/(2+xi)
//                  (from (3/xi - 2q)/f^2 = q^2/xi, using 2 - xi = 3 f^2/(2 + xi))
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace ark {

// BC_HALO (internal, y sides of a slab of the domain-decomposed step, dist.cu): the ghost line holds the neighbour rank's
// boundary row, refreshed by the halo exchange.  For the closure/flux kernels it is a Dirichlet ghost (a ghost enters like an
// interior cell, R9); for the linear system it is an UNKNOWN: nothing moves to b, and the operator takes the
// neighbour's z = M^-1 v and c^2 J z from the halo buffer of MfPlanes.
enum { BC_PERIODIC = 0, BC_DIRICHLET = 1, BC_OUTFLOW = 2, BC_HALO = 3 };
enum { XLO = 0, XHI = 1, YLO = 2, YHI = 3 };

struct Scheme {
    int wb;            // 1: Eqs. 18-19, 0: Eq. 16
    int ap;            // 1: Eq. 25, 0: alpha = 1, 2: Eq. C.8
    int eig;           // 0: Eq. 14, 1: +-c, 2: +-c/sqrt(3)
    int closure;       // 0: M1, 1: P1
    int lin;           // 0: Newton (analytic pressure Jacobian), 1: frozen Eddington tensor
    double eig_floor;
    double a_r;
    int src_off;       // internal (semi-implicit step): 1 drops the source terms from the explicit update
    int hyp_off;       // internal (semi-implicit step): 1 drops the flux-divergence terms from the assembled operator
    __host__ __device__ bool is_default() const {
        return wb == 1 && ap == 1 && eig == 0 && closure == 0 && lin == 0 && eig_floor == 0.0 && src_off == 0 && hyp_off == 0;
    }
};

struct Grid {
    int nx, ny;
    double dx, dy, c;
    int bc[4];
};

// Read-only view of the state planes and the Dirichlet ghost lines.
struct Fields {
    const double* E;
    const double* Fx;
    const double* Fy;
    const double* sa;   // sigma_a
    const double* st;   // sigma_t = sigma_a + sigma_s
    const double* gh[4][5];  // per side: E, Fx, Fy, sigma_a, sigma_t lines
    const double* T;         // may be null
    const double* rho_cv;    // may be null (=> 1)
    const double* source_E;  // may be null
};

struct CellU {  // raw state of one cell as the scheme sees it
    double E, Fx, Fy, sa, st;
    long long idx;  // cell index, -1 for a Dirichlet ghost
};

// Closure results of one cell.
struct Clo {
    double f;                   // |f| after the clamp
    double Pxx, Pxy, Pyy;       // radiative pressure
    double lmin[2], lmax[2];    // Eq. 14 for an x-face ([0]) and a y-face ([1])
};
struct Jac {                    // dP_ab/d(E,Fx,Fy); rows xx, xy, yy
    double xx[3], xy[3], yy[3];
};

#define ARK_E_FLOOR 1e-300

// ---------------------------------------------------------------------------------------------------------
// Fast fp64 reciprocal / reciprocal square root for the hot kernels: MUFU seed (rcp/rsqrt.approx.ftz.f64, relative
// error 2^-20 measured on B200) + Newton steps in DFMA.  Measured against IEEE on 2^20 arguments over 200 binades:
// rcp_fast bit-identical to 1/x, rsqrt_fast <= 1 ulp, x*rsqrt_fast(x) vs sqrt(x) <= 1 ulp; cost 4.7 / 6.2 DFMA
// issue slots against 8.7 (div) / 14.5 (sqrt) for the IEEE sequences, and none of their integer slow-path checks.
// Arguments must be normal and positive (callers guard zeros).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_fast(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0); y = fma(y, e, y);     // 2^-40
    e = fma(-x, y, 1.0); y = fma(y, e, y);            // 2^-80 -> rounding
    return y;
}
// Reciprocal with ONE third-order step, y (1 + e + e^2) with e = 1 - x y: 3 DFMA instead of 4, <= 1 ulp instead of
// correctly rounded (the explicit kernel is fp64-issue bound and has four reciprocals per cell).
__device__ __forceinline__ double rcp_fast3(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);                   // 2^-60 -> rounding
}
__device__ __forceinline__ double rsqrt_fast(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);                 // e = 1 - x y^2
    const double p = fma(0.375, e, 0.5);              // y (1 + e/2 + 3 e^2/8): third order, 2^-60
    return fma(y * e, p, y);
}
// max/min of two doubles as compare + select (2 fp64-pipe + 2 ALU issue slots).  fmax()/fmin() and the `x > K ? x : K` idiom
// compile on sm_100a to DSETP.MAX + SEL + FSEL + a NaN-quieting LOP3 + register copies (~9 issue slots, one dependent chain);
// the arguments here are never NaN.
__device__ __forceinline__ double dmax_sel(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.gt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}
__device__ __forceinline__ double dmin_sel(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}

// sqrt(x) for normal x > 0, the same third-order correction applied to t = x y ~ sqrt(x): one multiply less than x * rsqrt_fast(x)
__device__ __forceinline__ double sqrt_core(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    return fma(t * e, p, t);
}
// sqrt(x) for x >= 0; exactly 0 for x below 1e-290 (the seed flushes subnormals)
__device__ __forceinline__ double sqrt_fast(double x) { return (x > 1e-290) ? sqrt_core(x) : 0.0; }

// IEEE or fast (<= 1 ulp) reciprocal / square root, selected at compile time (FAST is used by the assembly kernel).
template <bool FAST> __device__ __forceinline__ double rcp_sel(double x) { return FAST ? rcp_fast(x) : 1.0 / x; }
template <bool FAST> __device__ __forceinline__ double sqrt_sel(double x) { return FAST ? sqrt_fast(x) : sqrt(x); }
template <bool FAST> __device__ __forceinline__ double rsqrt_sel(double x) { return FAST ? rsqrt_fast(x) : 1.0 / sqrt(x); }

// PAPER.md:79, 170, 513.  SCHEME_DEFAULT folds the scheme switches at compile time.
template <bool WITH_JAC, bool SCHEME_DEFAULT, bool FAST = false>
__device__ __forceinline__ void closure_eval(const Scheme& s, double c, double E, double Fx, double Fy, Clo& q, Jac* J)
{
    const double Es = (E > ARK_E_FLOOR) ? E : ARK_E_FLOOR;
    const double ice = rcp_sel<FAST>(c * Es);
    double fx = Fx * ice, fy = Fy * ice;
    double f2 = fx * fx + fy * fy;
    const bool clamped = f2 > 1.0;
    if (clamped) {
        // f2 = inf happens when E <= 0 (floored to 1e-300): 1/sqrt(inf) = 0 like the IEEE sequence, not NaN
        const double r = (FAST && !(f2 <= 1e300)) ? 0.0 : rsqrt_sel<FAST>(f2);
        fx *= r; fy *= r; f2 = 1.0;
    }
    const bool p1 = !SCHEME_DEFAULT && s.closure == 1;
    double xi, chi, q3;  // q3 = 3/(2+xi): (3chi-1)/2 n_a n_b = q3 f_a f_b
    if (p1) { xi = 2.0; chi = 1.0 / 3.0; q3 = 0.0; }
    else {
        xi = sqrt_sel<FAST>(4.0 - 3.0 * f2);
        chi = (3.0 + 4.0 * f2) * rcp_sel<FAST>(5.0 + 2.0 * xi);
        q3 = 3.0 * rcp_sel<FAST>(2.0 + xi);
    }
    const double iso = 0.5 * (1.0 - chi);
    const double Dxx = iso + q3 * fx * fx, Dxy = q3 * fx * fy, Dyy = iso + q3 * fy * fy;
    q.Pxx = Dxx * E; q.Pxy = Dxy * E; q.Pyy = Dyy * E;
    q.f = sqrt_sel<FAST>(f2);

    const int eig = SCHEME_DEFAULT ? 0 : s.eig;
    if (eig == 1) { q.lmax[0] = q.lmax[1] = c; q.lmin[0] = q.lmin[1] = -c; }
    else if (eig == 2 || p1) {
        const double l = c * 0.57735026918962576451;
        q.lmax[0] = q.lmax[1] = l; q.lmin[0] = q.lmin[1] = -l;
    } else {  // Eq. 14: normal component f_n, tangential f_t
        const double a = (xi - 1.0) * (xi + 2.0);
        const double ixi = rcp_sel<FAST>(xi);
        const double k = 0.81649658092772603273 * ixi * rcp_sel<FAST>(xi + 2.0);  // sqrt(2/3)/(xi (xi+2))
        const double rx = k * sqrt_sel<FAST>(a * (2.0 * a + 3.0 * fy * fy));
        const double ry = k * sqrt_sel<FAST>(a * (2.0 * a + 3.0 * fx * fx));
        const double mx = fx * ixi, my = fy * ixi;
        q.lmax[0] = c * (mx + rx); q.lmin[0] = c * (mx - rx);
        q.lmax[1] = c * (my + ry); q.lmin[1] = c * (my - ry);
    }

    if (WITH_JAC) {
        const bool frozen = p1 || (!SCHEME_DEFAULT && s.lin == 1);
        if (frozen) {  // P = D^n E
            J->xx[0] = Dxx; J->xx[1] = 0.0; J->xx[2] = 0.0;
            J->xy[0] = Dxy; J->xy[1] = 0.0; J->xy[2] = 0.0;
            J->yy[0] = Dyy; J->yy[1] = 0.0; J->yy[2] = 0.0;
        } else if (clamped) {
            // clamped closure P = E n(x)n, n = F/|F|: dP_ab/dE = n_a n_b, dP_ab/dF_k = (E/|F|)(d_ak n_b + d_bk n_a - 2 n_a n_b n_k)
            const double g = E * rsqrt_sel<FAST>(Fx * Fx + Fy * Fy);
            const double nx = fx, ny = fy;  // unit vector after the clamp
            J->xx[0] = nx * nx; J->xx[1] = g * (2.0 * nx - 2.0 * nx * nx * nx); J->xx[2] = g * (-2.0 * nx * nx * ny);
            J->xy[0] = nx * ny; J->xy[1] = g * (ny - 2.0 * nx * ny * nx);       J->xy[2] = g * (nx - 2.0 * nx * ny * ny);
            J->yy[0] = ny * ny; J->yy[1] = g * (-2.0 * ny * ny * nx);           J->yy[2] = g * (2.0 * ny - 2.0 * ny * ny * ny);
        } else {
            const double ixi = rcp_sel<FAST>(xi), ic = rcp_sel<FAST>(c);
            // (3/xi - 2 q)/f^2 with 2 - xi = 3 f^2/(2 + xi)  ==>  q^2/xi: no division by f^2, no cancellation
            const double t3 = q3 * q3 * ixi;                  // multiplies f_a f_b f_k
            // d/dE
            J->xx[0] = Dxx + (f2 - 3.0 * fx * fx) * ixi;
            J->xy[0] = Dxy + (-3.0 * fx * fy) * ixi;
            J->yy[0] = Dyy + (f2 - 3.0 * fy * fy) * ixi;
            // d/dFx (k = x), d/dFy (k = y)
            J->xx[1] = ic * (t3 * fx * fx * fx - fx * ixi + q3 * 2.0 * fx);
            J->xx[2] = ic * (t3 * fx * fx * fy - fy * ixi);
            J->xy[1] = ic * (t3 * fx * fy * fx + q3 * fy);
            J->xy[2] = ic * (t3 * fx * fy * fy + q3 * fx);
            J->yy[1] = ic * (t3 * fy * fy * fx - fx * ixi);
            J->yy[2] = ic * (t3 * fy * fy * fy - fy * ixi + q3 * 2.0 * fy);
        }
    }
}

// Face coefficients a+ = l+/(l+ - l-), a- = -l-/(l+ - l-), Lambda = l+ l-/(l+ - l-), alpha (Eq. 25), sigma_f (Eq. 19).
struct Face { double ap, am, Lam, alpha, sig; };

template <bool SCHEME_DEFAULT, bool FAST = false>
__device__ __forceinline__ void face_eval(const Scheme& s, double c, double delta,
                                          double lminL, double lmaxL, double fL, double stL,
                                          double lminR, double lmaxR, double fR, double stR, Face& fc)
{
    const double fl = SCHEME_DEFAULT ? 0.0 : s.eig_floor * c;
    const double lp = dmax_sel(dmax_sel(lmaxL, lmaxR), fl);
    const double lm = dmin_sel(dmin_sel(lminL, lminR), -fl);
    const double dl = lp - lm;
    if (dl > 0.0) {
        const double idl = rcp_sel<FAST>(dl);
        fc.ap = lp * idl; fc.am = -lm * idl; fc.Lam = lp * lm * idl;
    } else { fc.ap = 0.5; fc.am = 0.5; fc.Lam = 0.0; }  // l+ = l- = 0 (f = 1 tangential to the face)
    fc.sig = 0.5 * (stL + stR);
    const double ff = 0.5 * (fL + fR);
    const int ap = SCHEME_DEFAULT ? 1 : s.ap;
    if (ap == 0) fc.alpha = 1.0;
    else {
        const double w = (ap == 2) ? 1.0 : (1.0 - ff * ff);
        fc.alpha = FAST ? rcp_fast(1.0 - 3.0 * fc.sig * delta * w * fc.Lam * rcp_fast(c)) : 1.0 / (1.0 - 3.0 * fc.sig * delta * w * fc.Lam / c);
    }
}

// State seen at (i, j), at most one step outside the grid in one direction.
__device__ __forceinline__ void fetch_cell(const Fields& F, const Grid& g, int i, int j, CellU& u)
{
    int side = -1;
    if (i < 0) side = XLO; else if (i >= g.nx) side = XHI; else if (j < 0) side = YLO; else if (j >= g.ny) side = YHI;
    if (side >= 0) {
        const int bc = g.bc[side];
        if (bc == BC_PERIODIC) { i = (i + g.nx) % g.nx; j = (j + g.ny) % g.ny; }
        else if (bc == BC_OUTFLOW) { i = min(max(i, 0), g.nx - 1); j = min(max(j, 0), g.ny - 1); }
        else {
            const int k = (side == XLO || side == XHI) ? j : i;
            u.E = F.gh[side][0][k]; u.Fx = F.gh[side][1][k]; u.Fy = F.gh[side][2][k];
            u.sa = F.gh[side][3][k]; u.st = F.gh[side][4][k]; u.idx = -1;
            return;
        }
    }
    const long long id = (long long)j * g.nx + i;
    u.E = F.E[id]; u.Fx = F.Fx[id]; u.Fy = F.Fy[id]; u.sa = F.sa[id]; u.st = F.st[id]; u.idx = id;
}

}  // namespace ark
