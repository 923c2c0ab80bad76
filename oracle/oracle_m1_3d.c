/* oracle_m1_3d.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the SAME scheme as oracle_m1.c in three space dimensions ("its extension to higher
 * dimensions is straightforward"; (2+d)N unknowns): unknowns (E, Fx, Fy, Fz) per cell, a 7-point
 * stencil, every formula of the 2-D oracle applied direction by direction.  It checks the 3-D kernels of the CUDA library
 * (paper_2011_13926_b200/csrc/m1_3d.cu); it shares no code with them.  Only tests/ may build, load or call this file.
 *
 * Passages followed (PAPER.md line numbers), as in oracle_m1.c:
 *   closure chi(f), D = (1-chi)/2 I + (3chi-1)/2 n(x)n, P = D E (now a 3x3 tensor)   PAPER.md:79;  f > 1 clamp PAPER.md:513
 *   HLL-type fluxes F*, P* per face                                                  PAPER.md:162-164 (Eq. 13)
 *   eigenvalues: Eq. 14 with f_x = the face-normal component and f_y^2 = |f|^2 - f_n^2 (the tangential part)
 *   well-balanced source, face means, dimension by dimension (reading R6)            PAPER.md:193-199 (Eqs. 18, 19)
 *   AP factor alpha (Eq. 25) with the cell size of the face's direction
 *   Newton linearisation with the analytic pressure Jacobian (reading R4)
 *   right preconditioning with the (4x4) diagonal blocks, restarted GMRES            PAPER.md:267-272; north_star
 * Boundaries: periodic or outflow (zero gradient) per side.  No temperature coupling.
 *
 * Parity pins: tests/test_oracle_3d.py — a state that does not depend on z (Fz = 0) must evolve exactly like the 2-D oracle
 * (explicit and implicit), relabelling the axes must relabel the result, a slab free-streams at c along z, sums are
 * conserved, the Jacobian matches finite differences, GMRES matches a dense solve.
 *
 * Layout: planes [nz][ny][nx], x fastest.  F = [Fx | Fy | Fz].
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_API __attribute__((visibility("default")))
#define E_FLOOR 1e-300
enum { BC_PERIODIC = 0, BC_OUTFLOW = 2 };

typedef struct oracle_m1_3d {
    int n[3];            /* nx, ny, nz */
    double d[3], c;      /* dx, dy, dz */
    int bc[6];           /* xlo, xhi, ylo, yhi, zlo, zhi */
    double *U[4];        /* E, Fx, Fy, Fz */
    double *sa, *st;
    char err[256];
} oracle_m1_3d;

typedef struct {
    double E, F[3], sa, st;
    long idx;
} cell3;

typedef struct {
    double f, fv[3];          /* reduced flux after the clamp */
    double P[3][3];           /* pressure tensor */
    double lmin[3], lmax[3];  /* Eq. 14 for a face normal to x, y, z */
    double J[3][3][4];        /* dP_ab / d(E, Fx, Fy, Fz) */
} clo3;

static void closure3(double c, double E, const double F[3], clo3 *q)
{
    const double Es = (E > E_FLOOR) ? E : E_FLOOR;
    double fv[3] = { F[0] / (c * Es), F[1] / (c * Es), F[2] / (c * Es) };
    double f = sqrt(fv[0] * fv[0] + fv[1] * fv[1] + fv[2] * fv[2]);
    int clamped = 0;
    if (f > 1.0) { for (int a = 0; a < 3; ++a) fv[a] /= f; f = 1.0; clamped = 1; }
    double n[3] = { 0, 0, 0 };
    if (f > 0.0) for (int a = 0; a < 3; ++a) n[a] = fv[a] / f;
    const double xi = sqrt(4.0 - 3.0 * f * f);
    const double chi = (3.0 + 4.0 * f * f) / (5.0 + 2.0 * xi);
    const double aniso = 3.0 * f * f / (2.0 + xi);                                       /* = (3 chi - 1)/2 */
    const double iso = 0.5 * (1.0 - chi);
    q->f = f;
    double D[3][3];
    for (int a = 0; a < 3; ++a) {
        q->fv[a] = fv[a];
        for (int b = 0; b < 3; ++b) { D[a][b] = (a == b ? iso : 0.0) + aniso * n[a] * n[b]; q->P[a][b] = D[a][b] * E; }
    }
    for (int dir = 0; dir < 3; ++dir) {          /* Eq. 14: normal component and tangential magnitude */
        const double fn = fv[dir];
        double ft2 = 0.0;
        for (int a = 0; a < 3; ++a) if (a != dir) ft2 += fv[a] * fv[a];
        const double a_ = (xi - 1.0) * (xi + 2.0);
        const double root = sqrt(2.0) * sqrt(a_ * (2.0 * a_ + 3.0 * ft2)) / (sqrt(3.0) * xi * (xi + 2.0));
        q->lmax[dir] = c * (fn / xi + root);
        q->lmin[dir] = c * (fn / xi - root);
    }
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {
        const double dab = (a == b), nanb = n[a] * n[b];
        if (clamped) {
            const double Fn = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
            q->J[a][b][0] = nanb;
            for (int k = 0; k < 3; ++k) q->J[a][b][1 + k] = (E / Fn) * ((a == k) * n[b] + (b == k) * n[a] - 2.0 * nanb * n[k]);
        } else {
            const double xip = (f > 0.0) ? -3.0 * f / xi : 0.0;
            const double den = 5.0 + 2.0 * xi;
            const double chip = (8.0 * f * den - (3.0 + 4.0 * f * f) * 2.0 * xip) / (den * den);
            q->J[a][b][0] = D[a][b] + 0.5 * f * chip * (dab - 3.0 * nanb);
            const double anf = (f > 0.0) ? aniso / f : 0.0;
            for (int k = 0; k < 3; ++k)
                q->J[a][b][1 + k] = (0.5 * chip * (3.0 * nanb - dab) * n[k] + anf * ((a == k) * n[b] + (b == k) * n[a] - 2.0 * nanb * n[k])) / c;
        }
    }
}

static long wrap_index(const oracle_m1_3d *h, int i[3])
{
    for (int a = 0; a < 3; ++a) {
        const int n = h->n[a];
        if (i[a] < 0) i[a] = (h->bc[2 * a] == BC_PERIODIC) ? n - 1 : 0;
        else if (i[a] >= n) i[a] = (h->bc[2 * a + 1] == BC_PERIODIC) ? 0 : n - 1;
    }
    return ((long)i[2] * h->n[1] + i[1]) * h->n[0] + i[0];
}

static void fetch3(const oracle_m1_3d *h, int i, int j, int k, cell3 *u)
{
    int id3[3] = { i, j, k };
    const long id = wrap_index(h, id3);
    u->E = h->U[0][id]; for (int a = 0; a < 3; ++a) u->F[a] = h->U[1 + a][id];
    u->sa = h->sa[id]; u->st = h->st[id]; u->idx = id;
}

typedef struct { double ap, am, Lam, alpha, sig; } face3;

static void face_eval3(const oracle_m1_3d *h, const cell3 *L, const clo3 *qL, const cell3 *R, const clo3 *qR, int dir, face3 *fc)
{
    const double c = h->c;
    const double lp = fmax(0.0, fmax(qL->lmax[dir], qR->lmax[dir]));        /* PAPER.md:168, both neighbours (R2) */
    const double lm = fmin(0.0, fmin(qL->lmin[dir], qR->lmin[dir]));
    const double dl = lp - lm;
    if (dl > 0.0) { fc->ap = lp / dl; fc->am = -lm / dl; fc->Lam = lp * lm / dl; }
    else { fc->ap = 0.5; fc->am = 0.5; fc->Lam = 0.0; }
    fc->sig = 0.5 * (L->st + R->st);
    const double ff = 0.5 * (qL->f + qR->f);
    fc->alpha = 1.0 / (1.0 - 3.0 * fc->sig * h->d[dir] * (1.0 - ff * ff) * fc->Lam / c);     /* Eq. 25 */
}

/* Eq. 13 through a face normal to `dir`: G[0] = alpha F*, G[1..3] = P* rows for Fx, Fy, Fz.  vL, vR = (E, Fx, Fy, Fz). */
static void face_flux3(const oracle_m1_3d *h, const face3 *fc, int dir, const double vL[4], const double PL[3][3],
                       const double vR[4], const double PR[3][3], double G[4])
{
    const double c2 = h->c * h->c;
    G[0] = fc->alpha * (fc->ap * vL[1 + dir] + fc->am * vR[1 + dir] + fc->Lam * (vR[0] - vL[0]));
    for (int k = 0; k < 3; ++k) G[1 + k] = c2 * (fc->ap * PL[dir][k] + fc->am * PR[dir][k]) + fc->Lam * (vR[1 + k] - vL[1 + k]);
}

static const int DI[7][3] = { { 0, 0, 0 }, { -1, 0, 0 }, { 1, 0, 0 }, { 0, -1, 0 }, { 0, 1, 0 }, { 0, 0, -1 }, { 0, 0, 1 } };

/* lin == 0: non-linear residual R(U) of the stored state.  lin == 1: the linearised operator L_n applied to V (planes
 * [E|Fx|Fy|Fz]), coefficients frozen at the stored state, pressures replaced by J.V (reading R4). */
static void residual_cell3(const oracle_m1_3d *h, const double *V, int lin, int i, int j, int k, double R[4])
{
    const long N = (long)h->n[0] * h->n[1] * h->n[2];
    cell3 u[7]; clo3 q[7]; double v[7][4], Pv[7][3][3];
    for (int s = 0; s < 7; ++s) {
        fetch3(h, i + DI[s][0], j + DI[s][1], k + DI[s][2], &u[s]);
        closure3(h->c, u[s].E, u[s].F, &q[s]);
        if (lin) {
            for (int e = 0; e < 4; ++e) v[s][e] = V[e * N + u[s].idx];
            for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {
                double acc = 0.0;
                for (int e = 0; e < 4; ++e) acc += q[s].J[a][b][e] * v[s][e];
                Pv[s][a][b] = acc;
            }
        } else {
            v[s][0] = u[s].E; for (int a = 0; a < 3; ++a) v[s][1 + a] = u[s].F[a];
            memcpy(Pv[s], q[s].P, sizeof Pv[s]);
        }
    }
    const double c = h->c;
    R[0] = c * u[0].sa * v[0][0];                 /* -S^E = c sigma_a E */
    R[1] = R[2] = R[3] = 0.0;
    for (int dir = 0; dir < 3; ++dir) {
        const int lo = 1 + 2 * dir, hi = 2 + 2 * dir;
        face3 fm, fp; double Gm[4], Gp[4];
        face_eval3(h, &u[lo], &q[lo], &u[0], &q[0], dir, &fm);
        face_eval3(h, &u[0], &q[0], &u[hi], &q[hi], dir, &fp);
        face_flux3(h, &fm, dir, v[lo], Pv[lo], v[0], Pv[0], Gm);
        face_flux3(h, &fp, dir, v[0], Pv[0], v[hi], Pv[hi], Gp);
        for (int e = 0; e < 4; ++e) R[e] += (Gp[e] - Gm[e]) / h->d[dir];
        /* Eqs. 18-19 along this direction: -S^{F_dir} = c/4 [ sigma_+ (F_i + F_i+1) + sigma_- (F_i-1 + F_i) ] */
        R[1 + dir] += c * 0.5 * (fp.sig * 0.5 * (v[0][1 + dir] + v[hi][1 + dir]) + fm.sig * 0.5 * (v[lo][1 + dir] + v[0][1 + dir]));
    }
}

ORACLE_API int oracle3_residual(oracle_m1_3d *h, double *R)
{
    const long N = (long)h->n[0] * h->n[1] * h->n[2];
    #pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < h->n[2]; ++k) for (int j = 0; j < h->n[1]; ++j) for (int i = 0; i < h->n[0]; ++i) {
        double r[4]; residual_cell3(h, NULL, 0, i, j, k, r);
        const long id = ((long)k * h->n[1] + j) * h->n[0] + i;
        for (int e = 0; e < 4; ++e) R[e * N + id] = r[e];
    }
    return 0;
}

/* out = (I + dt L_n) V */
ORACLE_API int oracle3_apply_linear(oracle_m1_3d *h, double dt, const double *V, double *out)
{
    const long N = (long)h->n[0] * h->n[1] * h->n[2];
    #pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < h->n[2]; ++k) for (int j = 0; j < h->n[1]; ++j) for (int i = 0; i < h->n[0]; ++i) {
        double r[4]; residual_cell3(h, V, 1, i, j, k, r);
        const long id = ((long)k * h->n[1] + j) * h->n[0] + i;
        for (int e = 0; e < 4; ++e) out[e * N + id] = V[e * N + id] + dt * r[e];
    }
    return 0;
}

ORACLE_API int oracle3_step_explicit(oracle_m1_3d *h, double dt)
{
    if (!(dt > 0.0)) return -1;
    const long N = (long)h->n[0] * h->n[1] * h->n[2];
    double *R = (double *)malloc(sizeof(double) * 4 * N);
    if (!R) return -3;
    oracle3_residual(h, R);
    for (int e = 0; e < 4; ++e) for (long id = 0; id < N; ++id) h->U[e][id] -= dt * R[e * N + id];
    free(R);
    return 0;
}

/* 4x4 diagonal block of cell (i,j,k) of I + dt L_n: the operator applied to the four unit vectors of that cell, read at the
 * cell (a neighbour that IS the cell — outflow copy, one-cell-wide periodic direction — is covered, because the unit vector
 * is seen through the same fetch). */
static void diag_block3(const oracle_m1_3d *h, double dt, double *work, int i, int j, int k, double B[16])
{
    const long N = (long)h->n[0] * h->n[1] * h->n[2];
    const long id = ((long)k * h->n[1] + j) * h->n[0] + i;
    for (int e = 0; e < 4; ++e) {
        work[e * N + id] = 1.0;
        double r[4]; residual_cell3(h, work, 1, i, j, k, r);
        work[e * N + id] = 0.0;
        for (int a = 0; a < 4; ++a) B[4 * a + e] = (a == e ? 1.0 : 0.0) + dt * r[a];
    }
}

static void solve4(const double *B, const double r[4], double z[4])      /* Gaussian elimination with partial pivoting */
{
    double a[4][5];
    for (int i = 0; i < 4; ++i) { for (int k = 0; k < 4; ++k) a[i][k] = B[4 * i + k]; a[i][4] = r[i]; }
    for (int p = 0; p < 4; ++p) {
        int piv = p;
        for (int i = p + 1; i < 4; ++i) if (fabs(a[i][p]) > fabs(a[piv][p])) piv = i;
        if (piv != p) for (int k = 0; k < 5; ++k) { const double t = a[p][k]; a[p][k] = a[piv][k]; a[piv][k] = t; }
        for (int i = p + 1; i < 4; ++i) { const double m = a[i][p] / a[p][p]; for (int k = p; k < 5; ++k) a[i][k] -= m * a[p][k]; }
    }
    for (int i = 3; i >= 0; --i) { double s = a[i][4]; for (int k = i + 1; k < 4; ++k) s -= a[i][k] * z[k]; z[i] = s / a[i][i]; }
}

static double dot3(const double *a, const double *b, long n)
{
    double s = 0.0;
    for (long k = 0; k < n; ++k) s += a[k] * b[k];
    return s;
}

/* One linearised implicit step: (I + dt L_n) U^{n+1} = U^n, restarted GMRES(m), right-preconditioned by the 4x4 diagonal blocks
 * (Saad 2003, Alg. 9.5; modified Gram-Schmidt, Givens rotations), x0 = U^n, stop on ||b - A x|| <= tol ||b||. */
ORACLE_API int oracle3_step_implicit(oracle_m1_3d *h, double dt, double tol, int m, int maxit, double *final_residual)
{
    if (!(dt > 0.0) || !(tol > 0.0) || m < 1 || maxit < 0) return -1;
    const long N = (long)h->n[0] * h->n[1] * h->n[2], n = 4 * N;
    double *b = (double *)malloc(sizeof(double) * n), *x = (double *)malloc(sizeof(double) * n), *w = (double *)malloc(sizeof(double) * n);
    double *z = (double *)malloc(sizeof(double) * n), *Bd = (double *)malloc(sizeof(double) * 16 * N);
    double *V = (double *)malloc(sizeof(double) * n * (size_t)(m + 1)), *H = (double *)calloc((size_t)(m + 1) * m, sizeof(double));
    double *cs = (double *)malloc(sizeof(double) * m), *sn = (double *)malloc(sizeof(double) * m), *g = (double *)malloc(sizeof(double) * (m + 1)), *y = (double *)malloc(sizeof(double) * m);
    if (!b || !x || !w || !z || !Bd || !V || !H || !cs || !sn || !g || !y) return -3;
    for (int e = 0; e < 4; ++e) memcpy(b + e * N, h->U[e], sizeof(double) * N);
    memcpy(x, b, sizeof(double) * n);
    memset(w, 0, sizeof(double) * n);
    for (int k = 0; k < h->n[2]; ++k) for (int j = 0; j < h->n[1]; ++j) for (int i = 0; i < h->n[0]; ++i)
        diag_block3(h, dt, w, i, j, k, Bd + 16 * (((long)k * h->n[1] + j) * h->n[0] + i));
    #define HH(i, j) H[(size_t)(i) * m + (j)]
    #define PRECOND(src, dst) for (long id = 0; id < N; ++id) { double r_[4], z_[4]; for (int e = 0; e < 4; ++e) r_[e] = (src)[e * N + id]; \
                                  solve4(Bd + 16 * id, r_, z_); for (int e = 0; e < 4; ++e) (dst)[e * N + id] = z_[e]; }
    const double bnorm = sqrt(dot3(b, b, n)), target = tol * bnorm;
    int its = 0; double rnorm;
    for (;;) {
        oracle3_apply_linear(h, dt, x, w);
        for (long k = 0; k < n; ++k) w[k] = b[k] - w[k];
        rnorm = sqrt(dot3(w, w, n));
        if (rnorm <= target || its >= maxit) break;
        for (long k = 0; k < n; ++k) V[k] = w[k] / rnorm;
        for (int k = 0; k <= m; ++k) g[k] = 0.0;
        g[0] = rnorm;
        int j = 0;
        while (j < m && its < maxit) {
            double *vj = V + (size_t)j * n, *vn = V + (size_t)(j + 1) * n;
            PRECOND(vj, z)
            oracle3_apply_linear(h, dt, z, vn);
            for (int i = 0; i <= j; ++i) {
                const double *vi = V + (size_t)i * n;
                const double hij = dot3(vn, vi, n);
                HH(i, j) = hij;
                for (long k = 0; k < n; ++k) vn[k] -= hij * vi[k];
            }
            const double hn = sqrt(dot3(vn, vn, n));
            HH(j + 1, j) = hn;
            if (hn > 0.0) for (long k = 0; k < n; ++k) vn[k] /= hn;
            for (int i = 0; i < j; ++i) {
                const double t = cs[i] * HH(i, j) + sn[i] * HH(i + 1, j);
                HH(i + 1, j) = -sn[i] * HH(i, j) + cs[i] * HH(i + 1, j);
                HH(i, j) = t;
            }
            const double dd = hypot(HH(j, j), HH(j + 1, j));
            cs[j] = HH(j, j) / dd; sn[j] = HH(j + 1, j) / dd;
            HH(j, j) = dd; HH(j + 1, j) = 0.0;
            g[j + 1] = -sn[j] * g[j]; g[j] = cs[j] * g[j];
            ++j; ++its;
            if (fabs(g[j]) <= target || hn == 0.0) break;
        }
        for (int i = j - 1; i >= 0; --i) { double s = g[i]; for (int k = i + 1; k < j; ++k) s -= HH(i, k) * y[k]; y[i] = s / HH(i, i); }
        for (long k = 0; k < n; ++k) { double s = 0.0; for (int i = 0; i < j; ++i) s += y[i] * V[(size_t)i * n + k]; w[k] = s; }
        PRECOND(w, z)
        for (long k = 0; k < n; ++k) x[k] += z[k];
    }
    #undef HH
    #undef PRECOND
    for (int e = 0; e < 4; ++e) memcpy(h->U[e], x + e * N, sizeof(double) * N);
    if (final_residual) *final_residual = bnorm > 0 ? rnorm / bnorm : rnorm;
    free(b); free(x); free(w); free(z); free(Bd); free(V); free(H); free(cs); free(sn); free(g); free(y);
    return its;
}

/* Test hooks */
ORACLE_API void oracle3_closure_point(double c, double E, const double *F, double *out /* f, P[9], lmin[3], lmax[3], J[36] */)
{
    clo3 q; closure3(c, E, F, &q);
    out[0] = q.f;
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) out[1 + 3 * a + b] = q.P[a][b];
    for (int a = 0; a < 3; ++a) { out[10 + a] = q.lmin[a]; out[13 + a] = q.lmax[a]; }
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) for (int e = 0; e < 4; ++e) out[16 + 12 * a + 4 * b + e] = q.J[a][b][e];
}

ORACLE_API int oracle3_diag_blocks(oracle_m1_3d *h, double dt, double *B /* [N][16] */)
{
    const long N = (long)h->n[0] * h->n[1] * h->n[2];
    double *w = (double *)calloc((size_t)4 * N, sizeof(double));
    if (!w) return -3;
    for (int k = 0; k < h->n[2]; ++k) for (int j = 0; j < h->n[1]; ++j) for (int i = 0; i < h->n[0]; ++i)
        diag_block3(h, dt, w, i, j, k, B + 16 * (((long)k * h->n[1] + j) * h->n[0] + i));
    free(w);
    return 0;
}

ORACLE_API oracle_m1_3d *oracle3_create(int nx, int ny, int nz, double dx, double dy, double dz, double c, const int *bc6)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || !(c > 0)) return NULL;
    oracle_m1_3d *h = (oracle_m1_3d *)calloc(1, sizeof *h);
    if (!h) return NULL;
    h->n[0] = nx; h->n[1] = ny; h->n[2] = nz; h->d[0] = dx; h->d[1] = dy; h->d[2] = dz; h->c = c;
    for (int s = 0; s < 6; ++s) {
        h->bc[s] = bc6 ? bc6[s] : BC_PERIODIC;
        if (h->bc[s] != BC_PERIODIC && h->bc[s] != BC_OUTFLOW) { free(h); return NULL; }
    }
    for (int a = 0; a < 3; ++a) if ((h->bc[2 * a] == BC_PERIODIC) != (h->bc[2 * a + 1] == BC_PERIODIC)) { free(h); return NULL; }
    const size_t N = (size_t)nx * ny * nz;
    for (int e = 0; e < 4; ++e) h->U[e] = (double *)calloc(N, sizeof(double));
    h->sa = (double *)calloc(N, sizeof(double)); h->st = (double *)calloc(N, sizeof(double));
    return h;
}

ORACLE_API void oracle3_destroy(oracle_m1_3d *h)
{
    if (!h) return;
    for (int e = 0; e < 4; ++e) free(h->U[e]);
    free(h->sa); free(h->st); free(h);
}

ORACLE_API int oracle3_set_state(oracle_m1_3d *h, const double *E, const double *F, const double *sa, const double *ss)
{
    const size_t N = (size_t)h->n[0] * h->n[1] * h->n[2];
    memcpy(h->U[0], E, N * sizeof(double));
    for (int a = 0; a < 3; ++a) memcpy(h->U[1 + a], F + a * N, N * sizeof(double));
    memcpy(h->sa, sa, N * sizeof(double));
    for (size_t k = 0; k < N; ++k) h->st[k] = sa[k] + ss[k];
    return 0;
}

ORACLE_API int oracle3_get_state(oracle_m1_3d *h, double *E, double *F)
{
    const size_t N = (size_t)h->n[0] * h->n[1] * h->n[2];
    memcpy(E, h->U[0], N * sizeof(double));
    for (int a = 0; a < 3; ++a) memcpy(F + a * N, h->U[1 + a], N * sizeof(double));
    return 0;
}
