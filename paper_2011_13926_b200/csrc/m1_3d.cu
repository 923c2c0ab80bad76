// m1_3d.cu — the M1 radiative-transfer step in THREE space dimensions ("its extension to
// higher dimensions is straightforward"; (2+d)N unknowns): unknowns (E, Fx, Fy, Fz) per cell, 7-point stencil.
//
// Same scheme as the 2-D path, applied direction by direction: M1 closure (clamp PAPER.md:513), Eq. 14 with the
// face-normal component and the tangential magnitude, AP HLL fluxes (Eqs. 13, 25), well-balanced source (Eqs. 18-19), forward
// Euler explicit step, one Newton linearisation with the analytic pressure Jacobian solved by GMRES(m) right-preconditioned with
// the 4x4 diagonal blocks.  These are the GENERIC kernels of the 3-D path (one thread per cell, IEEE divisions and roots): they
// establish parity with the 3-D oracle; the marching organisation of the 2-D kernels is not repeated here.  The Krylov vector
// kernels (multi-dot, update, epilogues) are the 2-D path's own: they only see vectors of 4N doubles.
// Boundaries: periodic or outflow per side.  Planes [nz][ny][nx], x fastest; F = [Fx | Fy | Fz].
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <new>

#include "../../include/ark_m1.h"
#include "ark_m1_internal.h"
#include "explicit_device.cuh"

using namespace ark;

struct Grid3 { int n[3]; double d[3], c; int bc[6]; };
struct Clo3 { double f, fv[3], P[6], lmin[3], lmax[3]; };      // P: xx, xy, xz, yy, yz, zz
// index of the symmetric pair (a, b) in the order xx, xy, xz, yy, yz, zz
__host__ __device__ constexpr int sym3(int a, int b) { return a <= b ? 3 * a - a * (a - 1) / 2 + (b - a) : 3 * b - b * (b - 1) / 2 + (a - b); }

// Closure, Eq. 14 and (J != null) the pressure Jacobian dP_ab/d(E, Fx, Fy, Fz) as J[6][4], in the reduced-flux algebra of
// m1_device.cuh (no division by |F|):  P_ab = E [ (1-chi)/2 d_ab + q f_a f_b ],  q = 3/(2+xi);
//   dP_ab/dE = D_ab + (f^2 d_ab - 3 f_a f_b)/xi;  dP_ab/dF_k = [ f_a f_b f_k q^2/xi - d_ab f_k/xi + q (d_ak f_b + d_bk f_a) ]/c
__device__ __forceinline__ void closure3(double c, double E, const double F[3], Clo3& q, double* J)
{
    const double Es = (E > ARK_E_FLOOR) ? E : ARK_E_FLOOR;
    const double ice = 1.0 / (c * Es);
    double fv[3] = { F[0] * ice, F[1] * ice, F[2] * ice };
    double f2 = fv[0] * fv[0] + fv[1] * fv[1] + fv[2] * fv[2];
    const bool clamped = f2 > 1.0;
    if (clamped) { const double r = 1.0 / sqrt(f2); fv[0] *= r; fv[1] *= r; fv[2] *= r; f2 = 1.0; }
    const double xi = sqrt(4.0 - 3.0 * f2);
    const double chi = (3.0 + 4.0 * f2) / (5.0 + 2.0 * xi);
    const double q3 = 3.0 / (2.0 + xi), iso = 0.5 * (1.0 - chi);
    double D[6];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) D[sym3(a, b)] = (a == b ? iso : 0.0) + q3 * fv[a] * fv[b];
#pragma unroll
    for (int p = 0; p < 6; ++p) q.P[p] = D[p] * E;
    q.f = sqrt(f2);
#pragma unroll
    for (int a = 0; a < 3; ++a) q.fv[a] = fv[a];
    const double a_ = (xi - 1.0) * (xi + 2.0), ixi = 1.0 / xi;
    const double kk = 0.81649658092772603273 * ixi / (xi + 2.0);                                         // sqrt(2/3)/(xi (xi+2))
#pragma unroll
    for (int dir = 0; dir < 3; ++dir) {                     // Eq. 14: normal component, tangential magnitude
        const double ft2 = f2 - fv[dir] * fv[dir];
        const double root = kk * sqrt(a_ * (2.0 * a_ + 3.0 * fmax(ft2, 0.0)));
        const double mn = fv[dir] * ixi;
        q.lmax[dir] = c * (mn + root); q.lmin[dir] = c * (mn - root);
    }
    if (!J) return;
    if (clamped) {
        const double g = E / sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = a; b < 3; ++b) {
                double* Jp = J + 4 * sym3(a, b);
                Jp[0] = fv[a] * fv[b];
#pragma unroll
                for (int k = 0; k < 3; ++k) Jp[1 + k] = g * ((a == k ? fv[b] : 0.0) + (b == k ? fv[a] : 0.0) - 2.0 * fv[a] * fv[b] * fv[k]);
            }
        return;
    }
    const double t3 = q3 * q3 * ixi, ic = 1.0 / c;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) {
            double* Jp = J + 4 * sym3(a, b);
            Jp[0] = D[sym3(a, b)] + ((a == b ? f2 : 0.0) - 3.0 * fv[a] * fv[b]) * ixi;
#pragma unroll
            for (int k = 0; k < 3; ++k)
                Jp[1 + k] = ic * (t3 * fv[a] * fv[b] * fv[k] - (a == b ? fv[k] * ixi : 0.0) + q3 * ((a == k ? fv[b] : 0.0) + (b == k ? fv[a] : 0.0)));
        }
}

__device__ __forceinline__ long long nbr3(const Grid3& g, int i, int j, int k, int dir, int step)
{
    int id[3] = { i, j, k };
    id[dir] += step;
    const int n = g.n[dir];
    if (id[dir] < 0) id[dir] = (g.bc[2 * dir] == BC_PERIODIC) ? n - 1 : 0;
    else if (id[dir] >= n) id[dir] = (g.bc[2 * dir + 1] == BC_PERIODIC) ? 0 : n - 1;
    return ((long long)id[2] * g.n[1] + id[1]) * g.n[0] + id[0];
}

struct Cell3 { double E, F[3], sa, st; Clo3 q; };
__device__ __forceinline__ void load_cell3(const double* __restrict__ U, const double* __restrict__ sa, const double* __restrict__ st,
                                           long long N, long long id, double c, Cell3& u, double* J)
{
    u.E = U[id]; u.F[0] = U[N + id]; u.F[1] = U[2 * N + id]; u.F[2] = U[3 * N + id]; u.sa = sa[id]; u.st = st[id];
    closure3(c, u.E, u.F, u.q, J);
}

// Eq. 13 through a face normal to `dir` between L and R: G[0] = alpha F*, G[1..3] = P* rows (pressures as symmetric 6-vectors)
__device__ __forceinline__ void flux3(const Face& fc, int dir, double c2, const double vL[4], const double PL[6], const double vR[4], const double PR[6], double G[4])
{
    G[0] = fc.alpha * (fc.ap * vL[1 + dir] + fc.am * vR[1 + dir] + fc.Lam * (vR[0] - vL[0]));
#pragma unroll
    for (int k = 0; k < 3; ++k) G[1 + k] = c2 * (fc.ap * PL[sym3(dir, k)] + fc.am * PR[sym3(dir, k)]) + fc.Lam * (vR[1 + k] - vL[1 + k]);
}

// ---- explicit step: U^{n+1} = U^n - dt R(U^n), one thread per cell -----------------------------------------------------------
__global__ void __launch_bounds__(128) explicit3d_kernel(Grid3 g, const double* __restrict__ U, const double* __restrict__ sa, const double* __restrict__ st,
                                                         double dt, double* __restrict__ O)
{
    const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= N) return;
    const int i = (int)(id % g.n[0]), j = (int)((id / g.n[0]) % g.n[1]), k = (int)(id / ((long long)g.n[0] * g.n[1]));
    const Scheme s = { 1, 1, 0, 0, 0, 0.0, 1.0, 0, 0 };
    const double c = g.c, c2 = c * c;
    Cell3 C; load_cell3(U, sa, st, N, id, c, C, nullptr);
    const double vC[4] = { C.E, C.F[0], C.F[1], C.F[2] };
    double R[4] = { c * C.sa * C.E, 0.0, 0.0, 0.0 };
    for (int dir = 0; dir < 3; ++dir) {
        Cell3 Lo, Hi;
        load_cell3(U, sa, st, N, nbr3(g, i, j, k, dir, -1), c, Lo, nullptr);
        load_cell3(U, sa, st, N, nbr3(g, i, j, k, dir, +1), c, Hi, nullptr);
        const double vL[4] = { Lo.E, Lo.F[0], Lo.F[1], Lo.F[2] }, vH[4] = { Hi.E, Hi.F[0], Hi.F[1], Hi.F[2] };
        Face fm, fp; double Gm[4], Gp[4];
        face_eval<true>(s, c, g.d[dir], Lo.q.lmin[dir], Lo.q.lmax[dir], Lo.q.f, Lo.st, C.q.lmin[dir], C.q.lmax[dir], C.q.f, C.st, fm);
        face_eval<true>(s, c, g.d[dir], C.q.lmin[dir], C.q.lmax[dir], C.q.f, C.st, Hi.q.lmin[dir], Hi.q.lmax[dir], Hi.q.f, Hi.st, fp);
        flux3(fm, dir, c2, vL, Lo.q.P, vC, C.q.P, Gm);
        flux3(fp, dir, c2, vC, C.q.P, vH, Hi.q.P, Gp);
        const double rd = 1.0 / g.d[dir];
#pragma unroll
        for (int e = 0; e < 4; ++e) R[e] += (Gp[e] - Gm[e]) * rd;
        R[1 + dir] += 0.25 * c * (fp.sig * (vC[1 + dir] + vH[1 + dir]) + fm.sig * (vL[1 + dir] + vC[1 + dir]));     // Eqs. 18-19
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) O[e * N + id] = vC[e] - dt * R[e];
}

// ---- explicit step, two streaming passes (default): closure ONCE per cell, then the flux-form stencil ----------------------------
// Pass 1 writes, per cell, what its six faces need (13 planes): c^2 P (6), max(lambda_max, .) / min(lambda_min, .) per direction
// (6) and |f|/2, in the fast forms of the 2-D kernel (MUFU-seeded reciprocals and roots <= 1 ulp, chi = (5 - 2 xi)/3).  Pass 2
// reads the cell and its six neighbours (the x and y neighbours come out of L1, the z neighbours out of L2: two planes of the 19
// arrays are 20 MB) and evaluates each of its six faces with one reciprocal.  DRAM traffic ~ 320 B/cell against the algorithmic
// 80: it is the plain two-pass form, 4x faster than one thread doing seven closures (4.0 ms at 256^3), not a marching kernel.
struct Clo3Planes { double* p; };      // 13 planes of N doubles: P xx xy xz yy yz zz | lmin x y z | lmax x y z | f/2

__global__ void __launch_bounds__(256) closure3d_kernel(long long N, double c, const double* __restrict__ U, double* __restrict__ CL)
{
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= N) return;
    const double E = U[id], Fx = U[N + id], Fy = U[2 * N + id], Fz = U[3 * N + id];
    const double Es = dmax_sel(E, ARK_E_FLOOR);
    const double ice = rcp_fast3(c * Es);
    double fv[3] = { Fx * ice, Fy * ice, Fz * ice };
    const double f2raw = fma(fv[0], fv[0], fma(fv[1], fv[1], fma(fv[2], fv[2], 1e-300)));
    const bool huge = !(f2raw <= 1e300);
    const double rf = rsqrt_fast(huge ? 1.0 : f2raw);
    const bool clamp = f2raw > 1.0;
    const double sc = clamp ? (huge ? 0.0 : rf) : 1.0;
    fv[0] *= sc; fv[1] *= sc; fv[2] *= sc;
    const double f2 = clamp ? 1.0 : f2raw;
    CL[12 * N + id] = clamp ? 0.5 : (0.5 * f2raw) * rf;
    const double s_ = 4.0 - 3.0 * f2, rs = rsqrt_fast(s_), xi = s_ * rs;
    const double t2 = 2.0 + xi, xm1 = xi - 1.0, i2 = rcp_fast3(t2), c2 = c * c;
    const double Eq = E * ((3.0 * c2) * i2), Ei = E * ((0.33333333333333333333 * c2) * xm1);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) CL[sym3(a, b) * N + id] = fma(Eq * fv[a], fv[b], a == b ? Ei : 0.0);
    const double a_ = xm1 * t2, crs = c * rs, k = 1.41421356237309504880 * crs * i2, a23 = 0.66666666666666666667 * a_;
#pragma unroll
    for (int dir = 0; dir < 3; ++dir) {
        const double ft2 = fmax(f2 - fv[dir] * fv[dir], 0.0);
        const double root = k * sqrt_core(fma(a_, ft2 + a23, 1e-200));
        const double mn = fv[dir] * crs;
        CL[(6 + dir) * N + id] = mn - root; CL[(9 + dir) * N + id] = mn + root;
    }
}

__global__ void __launch_bounds__(128) flux3d_kernel(Grid3 g, const double* __restrict__ U, const double* __restrict__ sa, const double* __restrict__ st,
                                                     const double* __restrict__ CL, double dt, double* __restrict__ O)
{
    const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= N) return;
    const int i = (int)(id % g.n[0]), j = (int)((id / g.n[0]) % g.n[1]), k = (int)(id / ((long long)g.n[0] * g.n[1]));
    const double c = g.c;
    const double vC[4] = { U[id], U[N + id], U[2 * N + id], U[3 * N + id] };
    const double stC = st[id], fC = CL[12 * N + id];
    double R[4] = { c * sa[id] * vC[0], 0.0, 0.0, 0.0 };
#pragma unroll
    for (int dir = 0; dir < 3; ++dir) {
        const long long il = nbr3(g, i, j, k, dir, -1), ih = nbr3(g, i, j, k, dir, +1);
        const double k3h = 1.5 * g.d[dir] / c, rd = 1.0 / g.d[dir];
        double PC[3], PL[3], PH[3];
#pragma unroll
        for (int q = 0; q < 3; ++q) { PC[q] = CL[sym3(dir, q) * N + id]; PL[q] = CL[sym3(dir, q) * N + il]; PH[q] = CL[sym3(dir, q) * N + ih]; }
        const double vL[4] = { U[il], U[N + il], U[2 * N + il], U[3 * N + il] }, vH[4] = { U[ih], U[N + ih], U[2 * N + ih], U[3 * N + ih] };
        FaceF fm, fp;
        face_fast(k3h, CL[(6 + dir) * N + il], CL[(9 + dir) * N + il], CL[12 * N + il], st[il], CL[(6 + dir) * N + id], CL[(9 + dir) * N + id], fC, stC, fm);
        face_fast(k3h, CL[(6 + dir) * N + id], CL[(9 + dir) * N + id], fC, stC, CL[(6 + dir) * N + ih], CL[(9 + dir) * N + ih], CL[12 * N + ih], st[ih], fp);
        // Eq. 13 with a- = 1 - a+:  a+ x_L + a- x_R = x_R + a+ (x_L - x_R); the pressures carry c^2
        const double Gp0 = fp.alpha * fma(fp.Lam, vH[0] - vC[0], fma(fp.ap, vC[1 + dir] - vH[1 + dir], vH[1 + dir]));
        const double Gm0 = fm.alpha * fma(fm.Lam, vC[0] - vL[0], fma(fm.ap, vL[1 + dir] - vC[1 + dir], vC[1 + dir]));
        R[0] = fma(rd, Gp0 - Gm0, R[0]);
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const double Gp = fma(fp.Lam, vH[1 + q] - vC[1 + q], fma(fp.ap, PC[q] - PH[q], PH[q]));
            const double Gm = fma(fm.Lam, vC[1 + q] - vL[1 + q], fma(fm.ap, PL[q] - PC[q], PC[q]));
            R[1 + q] = fma(rd, Gp - Gm, R[1 + q]);
        }
        // Eqs. 18-19: FaceF.sig = sigma_L + sigma_R = twice the face opacity
        R[1 + dir] = fma(0.125 * c, fp.sig * (vC[1 + dir] + vH[1 + dir]) + fm.sig * (vL[1 + dir] + vC[1 + dir]), R[1 + dir]);
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) O[e * N + id] = fma(-dt, R[e], vC[e]);
}

// ---- implicit step -----------------------------------------------------------------------------------------------------------
struct Op3 {              // operator storage, planes of N doubles
    double* J;            // 24: dP_p/dU_e of the cell, p = xx, xy, xz, yy, yz, zz
    double* fP;           // 12: (a+, Lambda, alpha, c dt sigma_f/4) of the + face in x, y, z
    double* fM;           // 12: the same for the - face (stored per cell, so that boundary faces need no special case)
    double* dE;           // 1 : c dt sigma_a
    double* Minv;         // 16: inverse of the 4x4 diagonal block
    double* b;            // 4
    double* ZP;           // 10: z = M^-1 v (4) and c^2 J z (6), written by zp3d_kernel for every operator application
};

__device__ __forceinline__ void inv4(const double B[16], double I[16])      // Gauss-Jordan with partial pivoting
{
    double a[4][8];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c_ = 0; c_ < 4; ++c_) { a[r][c_] = B[4 * r + c_]; a[r][4 + c_] = (r == c_) ? 1.0 : 0.0; }
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        int piv = p;
#pragma unroll
        for (int r = p + 1; r < 4; ++r) if (fabs(a[r][p]) > fabs(a[piv][p])) piv = r;
        if (piv != p)
#pragma unroll
            for (int c_ = 0; c_ < 8; ++c_) { const double t = a[p][c_]; a[p][c_] = a[piv][c_]; a[piv][c_] = t; }
        const double ip = 1.0 / a[p][p];
#pragma unroll
        for (int c_ = 0; c_ < 8; ++c_) a[p][c_] *= ip;
#pragma unroll
        for (int r = 0; r < 4; ++r) if (r != p) {
            const double m = a[r][p];
#pragma unroll
            for (int c_ = 0; c_ < 8; ++c_) a[r][c_] -= m * a[p][c_];
        }
    }
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c_ = 0; c_ < 4; ++c_) I[4 * r + c_] = a[r][4 + c_];
}

// w * (the block multiplying THIS cell's unknowns in the flux through face fc), asLeft: the cell is the L cell of the face.
// G_L = [-alpha Lam, alpha a+ e_n ; c^2 a+ J^{n.} - Lam I_F],  G_R = [alpha Lam, alpha a- e_n ; c^2 a- J^{n.} + Lam I_F]
__device__ __forceinline__ void add_face_block(double B[16], const Face& fc, int dir, bool asLeft, double w, double c2, const double* J)
{
    const double a = asLeft ? fc.ap : fc.am, sg = asLeft ? -1.0 : 1.0;
    B[0] += w * sg * fc.alpha * fc.Lam; B[1 + dir] += w * fc.alpha * a;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double* Jp = J + 4 * sym3(dir, k);
#pragma unroll
        for (int e = 0; e < 4; ++e) B[4 * (1 + k) + e] += w * c2 * a * Jp[e];
        B[4 * (1 + k) + 1 + k] += w * sg * fc.Lam;
    }
}

__global__ void __launch_bounds__(128) assemble3d_kernel(Grid3 g, const double* __restrict__ U, const double* __restrict__ sa, const double* __restrict__ st,
                                                         double dt, Op3 op)
{
    const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= N) return;
    const int i = (int)(id % g.n[0]), j = (int)((id / g.n[0]) % g.n[1]), k = (int)(id / ((long long)g.n[0] * g.n[1]));
    const Scheme s = { 1, 1, 0, 0, 0, 0.0, 1.0, 0, 0 };
    const double c = g.c, c2 = c * c, cdt = c * dt;
    double J[24];
    Cell3 C; load_cell3(U, sa, st, N, id, c, C, J);
    double B[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) B[e] = 0.0;
    B[0] = 1.0 + cdt * C.sa; B[5] = 1.0; B[10] = 1.0; B[15] = 1.0;
    for (int dir = 0; dir < 3; ++dir) {
        const long long il = nbr3(g, i, j, k, dir, -1), ih = nbr3(g, i, j, k, dir, +1);
        Cell3 Lo, Hi;
        load_cell3(U, sa, st, N, il, c, Lo, nullptr);
        load_cell3(U, sa, st, N, ih, c, Hi, nullptr);
        Face fm, fp;
        face_eval<true>(s, c, g.d[dir], Lo.q.lmin[dir], Lo.q.lmax[dir], Lo.q.f, Lo.st, C.q.lmin[dir], C.q.lmax[dir], C.q.f, C.st, fm);
        face_eval<true>(s, c, g.d[dir], C.q.lmin[dir], C.q.lmax[dir], C.q.f, C.st, Hi.q.lmin[dir], Hi.q.lmax[dir], Hi.q.f, Hi.st, fp);
        const double rd = dt / g.d[dir], swp = 0.25 * cdt * fp.sig, swm = 0.25 * cdt * fm.sig;
        add_face_block(B, fp, dir, true, rd, c2, J);          // + rd G_L(face +)
        add_face_block(B, fm, dir, false, -rd, c2, J);        // - rd G_R(face -)
        B[4 * (1 + dir) + 1 + dir] += swp + swm;
        // a neighbour that is this very cell (outflow copy, one-cell-wide periodic direction) folds into the diagonal block
        if (ih == id) { add_face_block(B, fp, dir, false, rd, c2, J); B[4 * (1 + dir) + 1 + dir] += swp; }
        if (il == id) { add_face_block(B, fm, dir, true, -rd, c2, J); B[4 * (1 + dir) + 1 + dir] += swm; }
        op.fP[(4 * dir + 0) * N + id] = fp.ap; op.fP[(4 * dir + 1) * N + id] = fp.Lam; op.fP[(4 * dir + 2) * N + id] = fp.alpha; op.fP[(4 * dir + 3) * N + id] = swp;
        op.fM[(4 * dir + 0) * N + id] = fm.ap; op.fM[(4 * dir + 1) * N + id] = fm.Lam; op.fM[(4 * dir + 2) * N + id] = fm.alpha; op.fM[(4 * dir + 3) * N + id] = swm;
    }
    double Mi[16];
    inv4(B, Mi);
#pragma unroll
    for (int e = 0; e < 16; ++e) op.Minv[e * N + id] = Mi[e];
#pragma unroll
    for (int e = 0; e < 24; ++e) op.J[e * N + id] = J[e];
    op.dE[id] = cdt * C.sa;
    op.b[id] = C.E; op.b[N + id] = C.F[0]; op.b[2 * N + id] = C.F[1]; op.b[3 * N + id] = C.F[2];
}

// z = [M^-1] v and c^2 J z of every cell
__global__ void __launch_bounds__(256) zp3d_kernel(long long N, Op3 op, const double* __restrict__ v, int precond, double c2, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= N) return;
    const double v4[4] = { v[id], v[N + id], v[2 * N + id], v[3 * N + id] };
    double z[4];
    if (precond) {
#pragma unroll
        for (int r = 0; r < 4; ++r) z[r] = op.Minv[(4 * r) * N + id] * v4[0] + op.Minv[(4 * r + 1) * N + id] * v4[1] + op.Minv[(4 * r + 2) * N + id] * v4[2] + op.Minv[(4 * r + 3) * N + id] * v4[3];
    } else {
#pragma unroll
        for (int r = 0; r < 4; ++r) z[r] = v4[r];
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) op.ZP[r * N + id] = z[r];
#pragma unroll
    for (int p = 0; p < 6; ++p)
        op.ZP[(4 + p) * N + id] = c2 * (op.J[(4 * p) * N + id] * z[0] + op.J[(4 * p + 1) * N + id] * z[1] + op.J[(4 * p + 2) * N + id] * z[2] + op.J[(4 * p + 3) * N + id] * z[3]);
}

// out = sgn * s * (I + dt L_n) z + add, flux form, from the (z, c^2 J z) planes
__global__ void __launch_bounds__(128) op3d_kernel(Grid3 g, Op3 op, double* __restrict__ out, const double* __restrict__ scale_ptr,
                                                   const double* __restrict__ add, double sgn, double dt, const int* __restrict__ skip,
                                                   const double* __restrict__ vshift, double theta)
{
    if (skip && *skip) return;
    const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= N) return;
    const int i = (int)(id % g.n[0]), j = (int)((id / g.n[0]) % g.n[1]), k = (int)(id / ((long long)g.n[0] * g.n[1]));
    const double sc = sgn * (scale_ptr ? *scale_ptr : 1.0);
    double zC[4], PC[6];
#pragma unroll
    for (int e = 0; e < 4; ++e) zC[e] = op.ZP[e * N + id];
#pragma unroll
    for (int p = 0; p < 6; ++p) PC[p] = op.ZP[(4 + p) * N + id];
    double o[4] = { zC[0] * (1.0 + op.dE[id]), zC[1], zC[2], zC[3] };
    for (int dir = 0; dir < 3; ++dir) {
        const long long il = nbr3(g, i, j, k, dir, -1), ih = nbr3(g, i, j, k, dir, +1);
        double zL[4], zH[4], PL[6], PH[6];
#pragma unroll
        for (int e = 0; e < 4; ++e) { zL[e] = op.ZP[e * N + il]; zH[e] = op.ZP[e * N + ih]; }
#pragma unroll
        for (int p = 0; p < 6; ++p) { PL[p] = op.ZP[(4 + p) * N + il]; PH[p] = op.ZP[(4 + p) * N + ih]; }
        Face fp, fm;
        fp.ap = op.fP[(4 * dir) * N + id]; fp.Lam = op.fP[(4 * dir + 1) * N + id]; fp.alpha = op.fP[(4 * dir + 2) * N + id]; fp.am = 1.0 - fp.ap;
        fm.ap = op.fM[(4 * dir) * N + id]; fm.Lam = op.fM[(4 * dir + 1) * N + id]; fm.alpha = op.fM[(4 * dir + 2) * N + id]; fm.am = 1.0 - fm.ap;
        const double swp = op.fP[(4 * dir + 3) * N + id], swm = op.fM[(4 * dir + 3) * N + id];
        double Gp[4], Gm[4];
        flux3(fp, dir, 1.0, zC, PC, zH, PH, Gp);          // the pressures already carry c^2
        flux3(fm, dir, 1.0, zL, PL, zC, PC, Gm);
        const double rd = dt / g.d[dir];
#pragma unroll
        for (int e = 0; e < 4; ++e) o[e] += rd * (Gp[e] - Gm[e]);
        o[1 + dir] += swp * (zC[1 + dir] + zH[1 + dir]) + swm * (zL[1 + dir] + zC[1 + dir]);
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        double r = fma(sc, o[e], add ? add[e * N + id] : 0.0);
        if (vshift) r = fma(-theta, vshift[e * N + id], r);        // shifted operator (s-step Krylov basis, krylov_sstep.cu)
        out[e * N + id] = r;
    }
}

// x += M^-1 (sum_k coef_k V_k)
__global__ void __launch_bounds__(256) combine3d_kernel(long long N, const double* __restrict__ V, long long stride, const double* __restrict__ Minv,
                                                        double* __restrict__ x, GmresWork W)
{
    const int jj = W.ctl->j;
    if (jj == 0) return;
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= N) return;
    double u[4] = { 0.0, 0.0, 0.0, 0.0 };
    for (int k = 0; k < jj; ++k) {
        const double cf = W.coef[k];
        const double* v = V + k * stride;
#pragma unroll
        for (int e = 0; e < 4; ++e) u[e] += cf * v[e * N + id];
    }
#pragma unroll
    for (int r = 0; r < 4; ++r)
        x[r * N + id] += Minv[(4 * r) * N + id] * u[0] + Minv[(4 * r + 1) * N + id] * u[1] + Minv[(4 * r + 2) * N + id] * u[2] + Minv[(4 * r + 3) * N + id] * u[3];
}

// ---- handle and C ABI --------------------------------------------------------------------------------------------------------
struct ark_m1_3d {
    Grid3 g;
    long long N;
    int device, sm_count;
    cudaStream_t st;
    double* U[2]; int cur;
    double *sa, *ss_tmp, *stot;
    double* CL;               // 13 closure planes of the two-pass explicit step (lazy)
    int explicit_kernel;      // 1: two streaming passes (default), 0: one thread per cell with seven closures (IEEE forms)
    int arnoldi_block;        // 5 (default): s-step Arnoldi blocks as in the 2-D solver; 3, 4: shorter blocks; 1: one column per pass over the basis
    bool have_state;
    Op3 op;
    double* V; long long stride; int m_alloc, maxit_alloc;
    GmresWork W; void* wblock; GmresCtl* ctl_host;
    long long launches;
    char err[512];
};

static int fail3(ark_m1_3d* h, int code, const char* msg, const char* detail)
{
    if (h) snprintf(h->err, sizeof h->err, "%s%s%s", msg, detail ? ": " : "", detail ? detail : "");
    return code;
}
#define CU3(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return fail3(h, ARK_M1_E_CUDA, #call, cudaGetErrorString(e__)); } while (0)

static void free_op3(ark_m1_3d* h)
{
    cudaFree(h->op.J); cudaFree(h->op.fP); cudaFree(h->op.fM); cudaFree(h->op.dE); cudaFree(h->op.Minv); cudaFree(h->op.b); cudaFree(h->op.ZP);
    cudaFree(h->V); cudaFree(h->wblock);
    memset(&h->op, 0, sizeof h->op); h->V = nullptr; h->wblock = nullptr; h->m_alloc = 0; h->maxit_alloc = 0;
}

static int ensure3(ark_m1_3d* h, int m, int maxit)
{
    const size_t N = (size_t)h->N, n = 4 * N;
    if (h->op.J && h->m_alloc >= m && h->maxit_alloc >= maxit) return 0;
    CU3(cudaStreamSynchronize(h->st));
    if (!h->op.J) {
        const struct { double** p; size_t planes; } need[] = { { &h->op.J, 24 }, { &h->op.fP, 12 }, { &h->op.fM, 12 }, { &h->op.dE, 1 }, { &h->op.Minv, 16 }, { &h->op.b, 4 }, { &h->op.ZP, 10 } };
        for (auto& a : need) if (cudaMalloc((void**)a.p, a.planes * N * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return fail3(h, ARK_M1_E_ALLOC, "cudaMalloc (3-D operator planes)", nullptr); }
    }
    const int mm = m > h->m_alloc ? m : h->m_alloc, mi = maxit > h->maxit_alloc ? maxit : h->maxit_alloc;
    h->stride = (long long)((n + 31) / 32 * 32);
    if (mm > h->m_alloc) {
        cudaFree(h->V); h->V = nullptr;
        if (cudaMalloc((void**)&h->V, (size_t)(mm + 1) * h->stride * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return fail3(h, ARK_M1_E_ALLOC, "cudaMalloc (Krylov basis)", nullptr); }
    }
    cudaFree(h->wblock); h->wblock = nullptr;
    long long caph = (long long)mi + mi / (mm > 0 ? mm : 1) + 8;
    if (caph > (1LL << 20)) caph = (1LL << 20);
    const size_t nd = 2 * (size_t)(mm + 1) * mm + 2 * (size_t)mm + (mm + 1) + mm + 5 * (size_t)(mm + 1) + (size_t)caph + (size_t)krylov_max_blocks(h->sm_count) * MAXV
                      + 2 * (size_t)SMAX * (mm + 1) + 2 * SMAX * SMAX + (size_t)sstep_partial_doubles(h->sm_count);
    const size_t ctl_bytes = (sizeof(GmresCtl) + 255) / 256 * 256;
    if (cudaMalloc(&h->wblock, ctl_bytes + nd * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return fail3(h, ARK_M1_E_ALLOC, "cudaMalloc (solver scalars)", nullptr); }
    CU3(cudaMemset(h->wblock, 0, ctl_bytes + nd * sizeof(double)));
    GmresWork& W = h->W;
    memset(&W, 0, sizeof W);
    W.ctl = (GmresCtl*)h->wblock;
    double* p = (double*)((char*)h->wblock + ctl_bytes);
    W.H = p; p += (size_t)(mm + 1) * mm; W.cs = p; p += mm; W.sn = p; p += mm; W.g = p; p += mm + 1; W.y = p; p += mm;
    W.scale = p; p += mm + 1; W.coef = p; p += mm + 1; W.hist = p; p += caph;
    W.Hraw = p; p += (size_t)(mm + 1) * mm; W.c1 = p; p += mm + 1; W.c2 = p; p += mm + 1; W.coef2 = p; p += mm + 1;
    W.cS = p; p += (size_t)SMAX * (mm + 1); W.coefS = p; p += (size_t)SMAX * (mm + 1); W.Rb = p; p += SMAX * SMAX; W.tb = p; p += SMAX * SMAX;
    W.partialS = p; p += sstep_partial_doubles(h->sm_count);
    W.partial = p;
    W.caphist = (int)caph;
    h->m_alloc = mm; h->maxit_alloc = mi;
    return 0;
}

static int apply3(ark_m1_3d* h, const double* v, double* out, const double* scale_ptr, const double* add, double sgn, double dt, int precond, const int* stop,
                  double theta = 0.0)
{
    const long long N = h->N;
    zp3d_kernel<<<(unsigned)((N + 255) / 256), 256, 0, h->st>>>(N, h->op, v, precond, h->g.c * h->g.c, stop);
    CU3(cudaGetLastError());
    op3d_kernel<<<(unsigned)((N + 127) / 128), 128, 0, h->st>>>(h->g, h->op, out, scale_ptr, add, sgn, dt, stop, theta != 0.0 ? v : nullptr, theta);
    CU3(cudaGetLastError());
    h->launches += 2;
    return 0;
}

static int residual3(ark_m1_3d* h, double dt)        // V0 <- b - A x, ||V0|| -> DOT_RNORM epilogue
{
    int rc = apply3(h, h->U[h->cur], h->V, nullptr, h->op.b, -1.0, dt, 0, nullptr);
    if (rc) return rc;
    CU3(launch_multi_dot(h->V, h->V, h->stride, 1, 0, 4 * h->N, h->W, DOT_RNORM, h->sm_count, h->st));
    h->launches++;
    return 0;
}

extern "C" {

ark_m1_3d* ark_m1_3d_create(int nx, int ny, int nz, double dx, double dy, double dz, double c, const ark_m1_bc3* bc)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || !(c > 0)) return nullptr;
    int b[6] = { 0, 0, 0, 0, 0, 0 };
    if (bc) { b[0] = bc->xlo; b[1] = bc->xhi; b[2] = bc->ylo; b[3] = bc->yhi; b[4] = bc->zlo; b[5] = bc->zhi; }
    for (int s = 0; s < 6; ++s) if (b[s] != BC_PERIODIC && b[s] != BC_OUTFLOW) return nullptr;
    for (int a = 0; a < 3; ++a) if ((b[2 * a] == BC_PERIODIC) != (b[2 * a + 1] == BC_PERIODIC)) return nullptr;
    const long long N = (long long)nx * ny * nz;
    if ((N + 127) / 128 > 2147483647LL) return nullptr;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    ark_m1_3d* h = new (std::nothrow) ark_m1_3d;
    if (!h) return nullptr;
    memset(h, 0, sizeof *h);
    h->g.n[0] = nx; h->g.n[1] = ny; h->g.n[2] = nz; h->g.d[0] = dx; h->g.d[1] = dy; h->g.d[2] = dz; h->g.c = c;
    for (int s = 0; s < 6; ++s) h->g.bc[s] = b[s];
    h->N = N; h->device = dev; h->explicit_kernel = 1; h->arnoldi_block = 5;
    cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
    bool ok = true;
    for (int k = 0; k < 2 && ok; ++k) ok = cudaMalloc((void**)&h->U[k], 4 * (size_t)N * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->sa, (size_t)N * sizeof(double)) == cudaSuccess && cudaMalloc((void**)&h->ss_tmp, (size_t)N * sizeof(double)) == cudaSuccess
            && cudaMalloc((void**)&h->stot, (size_t)N * sizeof(double)) == cudaSuccess && cudaMallocHost((void**)&h->ctl_host, sizeof(GmresCtl)) == cudaSuccess;
    if (!ok) { cudaGetLastError(); ark_m1_3d_destroy(h); return nullptr; }
    return h;
}

void ark_m1_3d_destroy(ark_m1_3d* h)
{
    if (!h) return;
    cudaStreamSynchronize(h->st);
    free_op3(h);
    for (int k = 0; k < 2; ++k) cudaFree(h->U[k]);
    cudaFree(h->sa); cudaFree(h->ss_tmp); cudaFree(h->stot); cudaFree(h->CL);
    if (h->ctl_host) cudaFreeHost(h->ctl_host);
    cudaGetLastError();
    delete h;
}

int ark_m1_3d_set_stream(ark_m1_3d* h, void* cuda_stream)
{
    if (!h) return ARK_M1_E_ARG;
    CU3(cudaStreamSynchronize(h->st));
    h->st = (cudaStream_t)cuda_stream;
    return 0;
}

int ark_m1_3d_set_state(ark_m1_3d* h, const double* E, const double* F, const double* sigma_a, const double* sigma_s)
{
    if (!h || !E || !F || !sigma_a || !sigma_s) return ARK_M1_E_ARG;
    const size_t B = (size_t)h->N * sizeof(double);
    double* U = h->U[h->cur];
    CU3(cudaMemcpyAsync(U, E, B, cudaMemcpyDefault, h->st));
    CU3(cudaMemcpyAsync(U + h->N, F, 3 * B, cudaMemcpyDefault, h->st));
    CU3(cudaMemcpyAsync(h->sa, sigma_a, B, cudaMemcpyDefault, h->st));
    CU3(cudaMemcpyAsync(h->ss_tmp, sigma_s, B, cudaMemcpyDefault, h->st));
    CU3(launch_add_planes(h->stot, h->sa, h->ss_tmp, h->N, h->st));
    h->have_state = true;
    return 0;
}

int ark_m1_3d_set_option(ark_m1_3d* h, const char* key, double value)
{
    if (!h || !key) return ARK_M1_E_ARG;
    if (!strcmp(key, "explicit_kernel")) { if (value != 0.0 && value != 1.0) return fail3(h, ARK_M1_E_ARG, "explicit_kernel must be 0 or 1", nullptr); h->explicit_kernel = (int)value; }
    else if (!strcmp(key, "arnoldi_block")) { const int iv = (int)value; if (iv != 1 && (iv < 3 || iv > SMAX)) return fail3(h, ARK_M1_E_ARG, "arnoldi_block must be 1 or 3..5", nullptr); h->arnoldi_block = iv; }
    else return fail3(h, ARK_M1_E_ARG, "unknown option", key);
    return 0;
}

int ark_m1_3d_get_state(ark_m1_3d* h, double* E, double* F)
{
    if (!h || !E || !F) return ARK_M1_E_ARG;
    const size_t B = (size_t)h->N * sizeof(double);
    const double* U = h->U[h->cur];
    CU3(cudaMemcpyAsync(E, U, B, cudaMemcpyDefault, h->st));
    CU3(cudaMemcpyAsync(F, U + h->N, 3 * B, cudaMemcpyDefault, h->st));
    CU3(cudaStreamSynchronize(h->st));
    return 0;
}

int ark_m1_3d_step_explicit(ark_m1_3d* h, double dt)
{
    if (!h) return ARK_M1_E_ARG;
    if (!(dt > 0.0)) return fail3(h, ARK_M1_E_ARG, "step_explicit: dt must be > 0", nullptr);
    if (!h->have_state) return fail3(h, ARK_M1_E_NOTSET, "step_explicit: no state set", nullptr);
    if (h->explicit_kernel == 1) {
        if (!h->CL && cudaMalloc((void**)&h->CL, 13 * (size_t)h->N * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return fail3(h, ARK_M1_E_ALLOC, "cudaMalloc (closure planes)", nullptr); }
        closure3d_kernel<<<(unsigned)((h->N + 255) / 256), 256, 0, h->st>>>(h->N, h->g.c, h->U[h->cur], h->CL);
        CU3(cudaGetLastError());
        flux3d_kernel<<<(unsigned)((h->N + 127) / 128), 128, 0, h->st>>>(h->g, h->U[h->cur], h->sa, h->stot, h->CL, dt, h->U[h->cur ^ 1]);
        CU3(cudaGetLastError());
        h->launches += 2;
    } else {
        explicit3d_kernel<<<(unsigned)((h->N + 127) / 128), 128, 0, h->st>>>(h->g, h->U[h->cur], h->sa, h->stot, dt, h->U[h->cur ^ 1]);
        CU3(cudaGetLastError());
        h->launches++;
    }
    h->cur ^= 1;
    return 0;
}

int ark_m1_3d_step_implicit(ark_m1_3d* h, double dt, double tol, int restart, int maxit, double* final_residual)
{
    if (!h) return ARK_M1_E_ARG;
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0) return fail3(h, ARK_M1_E_ARG, "step_implicit: need dt > 0, tol > 0, restart >= 1, maxit >= 0", nullptr);
    if (!h->have_state) return fail3(h, ARK_M1_E_NOTSET, "step_implicit: no state set", nullptr);
    int rc = ensure3(h, restart, maxit);
    if (rc) return rc;
    const long long N = h->N, n = 4 * N, S = h->stride;
    const int m = restart, sm = h->sm_count;
    GmresWork W = h->W;
    const int* stop = &W.ctl->inner_stop;
    assemble3d_kernel<<<(unsigned)((N + 127) / 128), 128, 0, h->st>>>(h->g, h->U[h->cur], h->sa, h->stot, dt, h->op);
    CU3(cudaGetLastError());
    CU3(launch_begin_solve(W, tol, m, maxit, h->st));
    CU3(launch_multi_dot(h->op.b, h->op.b, 0, 1, 0, n, W, DOT_BNORM, sm, h->st));
    h->launches += 3;
    if ((rc = residual3(h, dt))) return rc;
    CU3(cudaMemcpyAsync(h->ctl_host, W.ctl, sizeof(GmresCtl), cudaMemcpyDeviceToHost, h->st));
    CU3(cudaStreamSynchronize(h->st));
    const int MV = MAXV;
    const int SB = (h->arnoldi_block >= 3 && m <= 120) ? h->arnoldi_block : 0;      // columns per s-step block (0: one column per pass)
    while (!h->ctl_host->inner_stop) {
        for (int j = 0; j < m; ++j) {
            double* w = h->V + (size_t)(j + 1) * S;
            if (SB && j + SB <= m) {
                // s-step Arnoldi block, as in the 2-D solver (krylov_sstep.cu; the vector kernels only see vectors of 4N doubles)
                for (int k = 0; k < SB; ++k)
                    if ((rc = apply3(h, h->V + (size_t)(j + k) * S, h->V + (size_t)(j + k + 1) * S, k == 0 ? W.scale + j : nullptr, nullptr, 1.0, dt, 1, stop, k == 0 ? 0.0 : 1.0))) return rc;
                const int nd = j + 1 + SB;          // the block's own slots are dotted like basis vectors: the in-block solve is predicted
                for (int c0 = 0; c0 < nd; c0 += 32) {
                    const int nv = (nd - c0) < 32 ? (nd - c0) : 32;
                    CU3(launch_dotS(w, h->V + (size_t)c0 * S, S, SB, nv, c0, n, W, sm, h->st, j));
                    h->launches++;
                }
                CU3(launch_updateS(w, h->V, S, SB, j + 1, n, W, sm, h->st));
                CU3(launch_qrS(w, S, SB, n, W, 1.0, 1, sm, h->st));
                CU3(launch_gramS(w, S, SB, n, W, sm, h->st));
                CU3(launch_qrS(w, S, SB, n, W, 1.0, 2, sm, h->st));
                h->launches += 4;
                j += SB - 1;
                continue;
            }
            if (SB && j + 1 < m) {      // columns a restart length leaves over: the two-column step
                double* w2 = h->V + (size_t)(j + 2) * S;
                if ((rc = apply3(h, h->V + (size_t)j * S, w, W.scale + j, nullptr, 1.0, dt, 1, stop))) return rc;
                if ((rc = apply3(h, w, w2, nullptr, nullptr, 1.0, dt, 1, stop))) return rc;
                const int MV2 = krylov_pair_max_vectors();
                const int nchunk2 = (j + MV2) / MV2, csize2 = (j + nchunk2) / nchunk2;
                for (int c0 = 0; c0 <= j; c0 += csize2) {
                    const int nv = (j + 1 - c0) < csize2 ? (j + 1 - c0) : csize2;
                    CU3(launch_multi_dot2(w, w2, h->V + (size_t)c0 * S, S, nv, c0, n, W, sm, h->st));
                    h->launches++;
                }
                CU3(launch_update2_all(w, w2, h->V, S, j + 1, n, W, sm, h->st));
                CU3(launch_update(w2, w, S, 1, j + 1, n, W, 1, sm, h->st, UPD_B2B));
                h->launches += 2;
                ++j;
                continue;
            }
            if ((rc = apply3(h, h->V + (size_t)j * S, w, W.scale + j, nullptr, 1.0, dt, 1, stop))) return rc;
            const int nchunk = (j + MV) / MV, csize = (j + nchunk) / nchunk;
            for (int c0 = 0; c0 <= j; c0 += csize) {
                const int nv = (j + 1 - c0) < csize ? (j + 1 - c0) : csize;
                CU3(launch_multi_dot(w, h->V + (size_t)c0 * S, S, nv, c0, n, W, DOT_H, sm, h->st));
                h->launches++;
            }
            for (int c0 = 0; c0 <= j; c0 += csize) {
                const int nv = (j + 1 - c0) < csize ? (j + 1 - c0) : csize;
                CU3(launch_update(w, h->V + (size_t)c0 * S, S, nv, c0, n, W, (c0 + csize > j) ? 1 : 0, sm, h->st));
                h->launches++;
            }
        }
        CU3(launch_solve_y(W, h->st));
        combine3d_kernel<<<(unsigned)((N + 255) / 256), 256, 0, h->st>>>(N, h->V, S, h->op.Minv, h->U[h->cur], W);
        CU3(cudaGetLastError());
        h->launches += 2;
        if ((rc = residual3(h, dt))) return rc;
        CU3(cudaMemcpyAsync(h->ctl_host, W.ctl, sizeof(GmresCtl), cudaMemcpyDeviceToHost, h->st));
        CU3(cudaStreamSynchronize(h->st));
    }
    const GmresCtl c = *h->ctl_host;
    if (c.nonfinite) return fail3(h, ARK_M1_E_NONFINITE, "step_implicit: non-finite norm in the solver", nullptr);
    if (final_residual) *final_residual = (c.bnorm > 0.0) ? c.rnorm / c.bnorm : c.rnorm;
    return c.its;
}

// out = A V (precond == 0) or A M^-1 V (precond == 1), A = I + dt L_n assembled from the stored state: the kernels the solver uses
int ark_m1_3d_apply_operator(ark_m1_3d* h, double dt, const double* Vin, double* out, int precond)
{
    if (!h || !Vin || !out) return ARK_M1_E_ARG;
    if (!(dt > 0.0)) return fail3(h, ARK_M1_E_ARG, "apply_operator: dt must be > 0", nullptr);
    if (!h->have_state) return fail3(h, ARK_M1_E_NOTSET, "apply_operator: no state set", nullptr);
    int rc = ensure3(h, 1, 1);
    if (rc) return rc;
    const size_t n = 4 * (size_t)h->N;
    assemble3d_kernel<<<(unsigned)((h->N + 127) / 128), 128, 0, h->st>>>(h->g, h->U[h->cur], h->sa, h->stot, dt, h->op);
    CU3(cudaGetLastError());
    h->launches++;
    CU3(cudaMemcpyAsync(h->V, Vin, n * sizeof(double), cudaMemcpyDefault, h->st));
    if ((rc = apply3(h, h->V, h->V + h->stride, nullptr, nullptr, 1.0, dt, precond, nullptr))) return rc;
    CU3(cudaMemcpyAsync(out, h->V + h->stride, n * sizeof(double), cudaMemcpyDefault, h->st));
    CU3(cudaStreamSynchronize(h->st));
    return 0;
}

long long ark_m1_3d_kernel_launches(const ark_m1_3d* h) { return h ? h->launches : 0; }
const char* ark_m1_3d_last_error(const ark_m1_3d* h) { return h ? h->err : "null handle"; }

}  // extern "C"
