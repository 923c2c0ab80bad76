/* oracle_m1.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the radiative-transfer step of the asymptotic-preserving (AP),
 * well-balanced (WB) M1 scheme of arXiv 2011.13926 (ARK-RT), written from PAPER.md equation by equation.
 * It exists so that the CUDA library (paper_2011_13926_b200/csrc) can be checked against something that a
 * reader can compare with the paper by eye.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code with the
 * CUDA path and neither includes the other.
 *
 * Passages followed (PAPER.md line numbers):
 *   closure  chi(f), D = (1-chi)/2 I + (3chi-1)/2 n(x)n, P = D E              PAPER.md:79   (Sect. 2.2)
 *   f > 1  -> "impose f = 1 in the computation of the Eddington tensor"        PAPER.md:513  (Sect. 5.6.3)
 *   moment system, matter energy                                               PAPER.md:64-75 (Eqs. 3, 4)
 *   Godunov/HLL update with alpha                                              PAPER.md:152-157 (Eq. 12)
 *   numerical fluxes F*, P*                                                    PAPER.md:162-164 (Eq. 13)
 *   lambda^+ = max(0, lambda_max), lambda^- = min(0, lambda_min)
 *   M1 eigenvalues                                                             PAPER.md:170  (Eq. 14)
 *   cell-centred source {sigma F}_i = sigma_i F_i                              PAPER.md:185  (Eq. 16)
 *   well-balanced source, face means                                           PAPER.md:193-199 (Eqs. 18, 19)
 *   boundary form (ghost cell enters the face relation)                        PAPER.md:225-229 (Eq. 24)
 *   AP factor alpha                                                            PAPER.md:235-238 (Eq. 25 = C.9); C.7, C.8 at 771-776
 *   Newton-Raphson linearisation, (2+d)N unknowns                              PAPER.md:263  (Sect. 3.3.1)
 *   right preconditioning A K^-1 y = b, K x = y; Jacobi K = diag(A)            PAPER.md:267-272 (Eq. 27)
 *   velocity source terms S_E(u), S_F(u)                                       PAPER.md:101  (Eq. 6), 253
 *
 * Readings where the paper is silent or garbled are those of DESIGN.md ("Readings", R1..R14); the ones that
 * matter here are repeated beside the code.  north_star (BASELINE.json) replaces the paper's BiCGStab by
 * restarted GMRES, its point-Jacobi by 3x3 block-Jacobi, splits sigma into sigma_a + sigma_s, and asks for
 * one linearised solve per implicit step.
 *
 * Parity pins: tests/test_oracle_*.py (closed forms, printed values, finite differences, dense direct
 * solves, analytic diffusion, conservation, steady states).  "parity unpinned": the beam-width numbers of
 * PAPER.md:414 (no width definition given) and the absolute results of configs 3-5 (the paper prints none).
 *
 * Layout: every field is a row-major [ny][nx] plane of doubles, x fastest.  F = [Fx plane | Fy plane].
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_API __attribute__((visibility("default")))

enum { BC_PERIODIC = 0, BC_DIRICHLET = 1, BC_OUTFLOW = 2 };
enum { XLO = 0, XHI = 1, YLO = 2, YHI = 3 };
enum { PXX = 0, PXY = 1, PYY = 2 };       /* rows of the pressure Jacobian */
enum { KE = 0, KFX = 1, KFY = 2 };        /* columns: derivative with respect to E, Fx, Fy */
enum { BLK_C = 0, BLK_W = 1, BLK_E = 2, BLK_S = 3, BLK_N = 4 };

#define E_FLOOR 1e-300   /* R1: E <= 0 is only guarded in the division f = |F|/(cE) */

struct mg_hier;
typedef struct oracle_m1 {
    int nx, ny;
    double dx, dy, c;
    int bc[4];
    double *E, *Fx, *Fy, *sa, *st, *T;   /* st = sigma_a + sigma_s */
    int has_T;
    double *gh[4][5];                    /* Dirichlet ghost lines: E, Fx, Fy, sigma_a, sigma_t */
    /* scheme switches (defaults = the paper's scheme) */
    int wb;          /* 1: Eq. 18-19 (default), 0: Eq. 16 */
    int ap;          /* 1: Eq. 25 (default), 0: alpha = 1 (standard HLL), 2: Eq. C.8 */
    int eig;         /* 0: Eq. 14 (default), 1: fixed +-c, 2: fixed +-c/sqrt(3) */
    int closure;     /* 0: M1 (default), 1: P1 (chi = 1/3) */
    int lin;         /* 0: analytic pressure Jacobian (default, R4), 1: frozen Eddington tensor */
    int src_off;     /* internal (semi-implicit step): 1 drops the source terms from the residual */
    int hyp_off;     /* internal (semi-implicit step): 1 drops the flux-divergence terms from the assembled operator */
    int krylov;      /* 0: restarted GMRES (north_star, default), 1: BiCGStab (the paper's solver) */
    int precond_kind;/* 0: 3x3 block-Jacobi (north_star, default), 1: multigrid V-cycle (R15) */
    double mg_omega; /* damping of the block-Jacobi smoother, default 0.8 */
    int mg_coarse_sweeps; /* smoother sweeps on the coarsest (1x1) level, default 2 */
    struct mg_hier *mg;   /* hierarchy of the solve in progress (built by mg_build, freed after the solve) */
    double eig_floor;/* lambda^+ >= floor*c, lambda^- <= -floor*c; default 0 */
    double a_r;      /* radiation constant, default 1 */
    double *rho_cv, *ux, *uy, *source_E; /* stage-2 fields (may be NULL) */
    /* residual history of the last implicit solve (relative residual estimates) */
    double *hist; int nhist, caphist;
    char err[256];
} oracle_m1;

/* ------------------------------------------------------------------------------------------------ */
/* Per-cell quantities                                                                              */
/* ------------------------------------------------------------------------------------------------ */

typedef struct { double E, Fx, Fy, sa, st; int dirichlet_ghost; long idx; } cell_t;

typedef struct {
    double f, fx, fy;        /* reduced flux (after the f <= 1 clamp) */
    double xi, chi;
    double P[3];             /* Pxx, Pxy, Pyy */
    double lmin[2], lmax[2]; /* Eq. 14 for a face normal to x ([0]) and to y ([1]) */
    double J[3][3];          /* dP_ab/d(E,Fx,Fy), rows xx, xy, yy */
} closure_t;

/* Closure, eigenvalues and pressure Jacobian of one state.  PAPER.md:79, 170, 513. */
static void closure_eval(const oracle_m1 *h, double E, double Fx, double Fy, closure_t *q)
{
    const double c = h->c;
    const double Es = (E > E_FLOOR) ? E : E_FLOOR;           /* R1 */
    double fx = Fx / (c * Es), fy = Fy / (c * Es);
    double f = sqrt(fx * fx + fy * fy);
    int clamped = 0;
    if (f > 1.0) { fx /= f; fy /= f; f = 1.0; clamped = 1; }
    double nx = 0.0, ny = 0.0;
    if (f > 0.0) { nx = fx / f; ny = fy / f; }
    const double n[2] = { nx, ny };

    double xi, chi, aniso;       /* aniso = (3 chi - 1)/2 */
    if (h->closure == 1) {       /* P1: chi = 1/3, P = E/3 I */
        xi = 2.0; chi = 1.0 / 3.0; aniso = 0.0;
    } else {
        xi = sqrt(4.0 - 3.0 * f * f);
        chi = (3.0 + 4.0 * f * f) / (5.0 + 2.0 * xi);       /* PAPER.md:79 (R1: garbled root restored) */
        /* (3 chi - 1)/2 = 3 f^2/(2 + xi): same number, without the cancellation of 3*chi - 1 at small f */
        aniso = 3.0 * f * f / (2.0 + xi);
    }
    q->f = f; q->fx = fx; q->fy = fy; q->xi = xi; q->chi = chi;
    const double iso = 0.5 * (1.0 - chi);
    double D[3];
    D[PXX] = iso + aniso * nx * nx;
    D[PXY] =       aniso * nx * ny;
    D[PYY] = iso + aniso * ny * ny;
    for (int p = 0; p < 3; ++p) q->P[p] = D[p] * E;

    /* Eq. 14: f_x there is the component normal to the face, f_y the tangential one (R2). */
    for (int dir = 0; dir < 2; ++dir) {
        const double fn = dir == 0 ? fx : fy, ft = dir == 0 ? fy : fx;
        if (h->eig == 1) { q->lmax[dir] = c; q->lmin[dir] = -c; }
        else if (h->eig == 2 || h->closure == 1) { q->lmax[dir] = c / sqrt(3.0); q->lmin[dir] = -c / sqrt(3.0); }
        else {
            const double a = (xi - 1.0) * (xi + 2.0);
            const double root = sqrt(2.0) * sqrt(a * (2.0 * a + 3.0 * ft * ft)) / (sqrt(3.0) * xi * (xi + 2.0));
            q->lmax[dir] = c * (fn / xi + root);
            q->lmin[dir] = c * (fn / xi - root);
        }
    }

    /* Pressure Jacobian dP_ab/dU (R4).  a, b index the pair (xx, xy, yy). */
    static const int A_[3] = { 0, 0, 1 }, B_[3] = { 0, 1, 1 };
    for (int p = 0; p < 3; ++p) {
        const int a = A_[p], b = B_[p];
        const double dab = (a == b) ? 1.0 : 0.0;
        const double nanb = n[a] * n[b];
        if (h->lin == 1 || h->closure == 1) {            /* frozen Eddington tensor: P = D^n E */
            q->J[p][KE] = D[p]; q->J[p][KFX] = 0.0; q->J[p][KFY] = 0.0;
        } else if (clamped) {
            /* P = E n(x)n with n = F/|F| (the clamped closure is itself homogeneous of degree 1) */
            const double Fn = sqrt(Fx * Fx + Fy * Fy);
            q->J[p][KE] = nanb;
            for (int k = 0; k < 2; ++k) {
                const double dak = (a == k), dbk = (b == k);
                q->J[p][KFX + k] = (E / Fn) * (dak * n[b] + dbk * n[a] - 2.0 * nanb * n[k]);
            }
        } else {
            /* chi'(f) by the quotient rule on chi = (3+4f^2)/(5+2xi), xi' = -3f/xi */
            const double xip = (f > 0.0) ? -3.0 * f / xi : 0.0;
            const double den = 5.0 + 2.0 * xi;
            const double chip = (8.0 * f * den - (3.0 + 4.0 * f * f) * 2.0 * xip) / (den * den);
            /* dP_ab/dE = D_ab - f dD_ab/df = D_ab + (f chi'/2)(delta_ab - 3 n_a n_b) */
            q->J[p][KE] = D[p] + 0.5 * f * chip * (dab - 3.0 * nanb);
            /* dP_ab/dF_k = (1/c)[ (chi'/2)(3 n_a n_b - delta_ab) n_k + ((3chi-1)/(2f)) (d_ak n_b + d_bk n_a - 2 n_a n_b n_k) ] */
            const double anf = (f > 0.0) ? aniso / f : 0.0;
            for (int k = 0; k < 2; ++k) {
                const double dak = (a == k), dbk = (b == k);
                q->J[p][KFX + k] = (0.5 * chip * (3.0 * nanb - dab) * n[k]
                                    + anf * (dak * n[b] + dbk * n[a] - 2.0 * nanb * n[k])) / c;
            }
        }
    }
}

/* State and opacity seen at (i, j), one step outside the grid allowed in one direction (R9).
 * periodic: wrap; outflow: copy of the adjacent interior cell; Dirichlet: the given ghost line. */
static void fetch(const oracle_m1 *h, int i, int j, cell_t *u)
{
    const int nx = h->nx, ny = h->ny;
    int side = -1;
    if (i < 0) side = XLO; else if (i >= nx) side = XHI; else if (j < 0) side = YLO; else if (j >= ny) side = YHI;
    u->dirichlet_ghost = 0;
    if (side >= 0) {
        const int bc = h->bc[side];
        if (bc == BC_PERIODIC) { i = (i + nx) % nx; j = (j + ny) % ny; }
        else if (bc == BC_OUTFLOW) { if (i < 0) i = 0; if (i >= nx) i = nx - 1; if (j < 0) j = 0; if (j >= ny) j = ny - 1; }
        else {
            const int k = (side == XLO || side == XHI) ? j : i;
            u->E = h->gh[side][0][k]; u->Fx = h->gh[side][1][k]; u->Fy = h->gh[side][2][k];
            u->sa = h->gh[side][3][k]; u->st = h->gh[side][4][k];
            u->dirichlet_ghost = 1; u->idx = -1;
            return;
        }
    }
    const long id = (long)j * nx + i;
    u->E = h->E[id]; u->Fx = h->Fx[id]; u->Fy = h->Fy[id]; u->sa = h->sa[id]; u->st = h->st[id]; u->idx = id;
}

/* Face coefficients between a left (L) and a right (R) cell along direction dir (0: x, 1: y).
 * lambda^+-: PAPER.md:168 with both neighbours (R2); alpha: Eq. 25 with
 * sigma_{i+1/2} = (sigma_i + sigma_{i+1})/2 (Eq. 19) and f_{i+1/2} = (f_i + f_{i+1})/2 (R5). */
typedef struct { double ap, am, Lam, alpha, sig; } face_t;   /* a+ = l+/(l+ - l-), a- = -l-/(l+ - l-), Lam = l+ l-/(l+ - l-) */

static void face_eval(const oracle_m1 *h, const cell_t *L, const closure_t *qL, const cell_t *R, const closure_t *qR,
                      int dir, face_t *fc)
{
    const double c = h->c, fl = h->eig_floor * c;
    double lp = fmax(fl, fmax(qL->lmax[dir], qR->lmax[dir]));
    double lm = fmin(-fl, fmin(qL->lmin[dir], qR->lmin[dir]));
    const double dl = lp - lm;
    if (dl > 0.0) { fc->ap = lp / dl; fc->am = -lm / dl; fc->Lam = lp * lm / dl; }
    else { fc->ap = 0.5; fc->am = 0.5; fc->Lam = 0.0; }                /* R2: l+ = l- = 0 */
    fc->sig = 0.5 * (L->st + R->st);
    const double ff = 0.5 * (qL->f + qR->f);
    const double delta = dir == 0 ? h->dx : h->dy;
    if (h->ap == 0) fc->alpha = 1.0;
    else if (h->ap == 2) fc->alpha = 1.0 / (1.0 - 3.0 * fc->sig * delta * fc->Lam / c);                    /* Eq. C.8 */
    else fc->alpha = 1.0 / (1.0 - 3.0 * fc->sig * delta * (1.0 - ff * ff) * fc->Lam / c);                  /* Eq. 25 */
}

/* Numerical fluxes of Eq. 13 through the face between L and R; pressures passed in so that the same routine
 * serves the non-linear residual (P from the closure) and the linearised operator (Pi = J.U).
 * G[0] = alpha F*, G[1], G[2] = P* components for the Fx and Fy equations. */
static void face_flux(const oracle_m1 *h, const face_t *fc, int dir,
                      double EL, double FxL, double FyL, const double PL[3],
                      double ER, double FxR, double FyR, const double PR[3], double G[3])
{
    const double c2 = h->c * h->c;
    const double FnL = dir == 0 ? FxL : FyL, FnR = dir == 0 ? FxR : FyR;
    const double PnxL = dir == 0 ? PL[PXX] : PL[PXY], PnxR = dir == 0 ? PR[PXX] : PR[PXY];
    const double PnyL = dir == 0 ? PL[PXY] : PL[PYY], PnyR = dir == 0 ? PR[PXY] : PR[PYY];
    G[0] = fc->alpha * (fc->ap * FnL + fc->am * FnR + fc->Lam * (ER - EL));
    G[1] = c2 * (fc->ap * PnxL + fc->am * PnxR) + fc->Lam * (FxR - FxL);
    G[2] = c2 * (fc->ap * PnyL + fc->am * PnyR) + fc->Lam * (FyR - FyL);
}

/* ------------------------------------------------------------------------------------------------ */
/* Non-linear residual R(U) and explicit step                                                        */
/* ------------------------------------------------------------------------------------------------ */

/* R(U)_i = (G_{i+1/2} - G_{i-1/2})/dx + (H_{j+1/2} - H_{j-1/2})/dy - S  (Eq. 12 with time-n right side). */
static void residual_cell(const oracle_m1 *h, int i, int j, double R[3])
{
    cell_t u[5]; closure_t q[5];  /* 0: centre, 1: west, 2: east, 3: south, 4: north */
    fetch(h, i, j, &u[0]); fetch(h, i - 1, j, &u[1]); fetch(h, i + 1, j, &u[2]);
    fetch(h, i, j - 1, &u[3]); fetch(h, i, j + 1, &u[4]);
    for (int k = 0; k < 5; ++k) closure_eval(h, u[k].E, u[k].Fx, u[k].Fy, &q[k]);
    face_t fw, fe, fs, fn; double Gw[3], Ge[3], Hs[3], Hn[3];
    face_eval(h, &u[1], &q[1], &u[0], &q[0], 0, &fw);
    face_eval(h, &u[0], &q[0], &u[2], &q[2], 0, &fe);
    face_eval(h, &u[3], &q[3], &u[0], &q[0], 1, &fs);
    face_eval(h, &u[0], &q[0], &u[4], &q[4], 1, &fn);
    face_flux(h, &fw, 0, u[1].E, u[1].Fx, u[1].Fy, q[1].P, u[0].E, u[0].Fx, u[0].Fy, q[0].P, Gw);
    face_flux(h, &fe, 0, u[0].E, u[0].Fx, u[0].Fy, q[0].P, u[2].E, u[2].Fx, u[2].Fy, q[2].P, Ge);
    face_flux(h, &fs, 1, u[3].E, u[3].Fx, u[3].Fy, q[3].P, u[0].E, u[0].Fx, u[0].Fy, q[0].P, Hs);
    face_flux(h, &fn, 1, u[0].E, u[0].Fx, u[0].Fy, q[0].P, u[4].E, u[4].Fx, u[4].Fy, q[4].P, Hn);
    const double c = h->c;
    double SE = -c * u[0].sa * u[0].E, SFx, SFy;
    if (h->has_T) { const double T = h->T[u[0].idx]; SE += c * u[0].sa * h->a_r * T * T * T * T; }
    if (h->source_E) SE += h->source_E[u[0].idx];
    if (h->wb) {  /* Eqs. 18-19, dimension by dimension (R6) */
        SFx = -c * 0.5 * (fe.sig * 0.5 * (u[0].Fx + u[2].Fx) + fw.sig * 0.5 * (u[1].Fx + u[0].Fx));
        SFy = -c * 0.5 * (fn.sig * 0.5 * (u[0].Fy + u[4].Fy) + fs.sig * 0.5 * (u[3].Fy + u[0].Fy));
    } else {      /* Eq. 16 */
        SFx = -c * u[0].st * u[0].Fx; SFy = -c * u[0].st * u[0].Fy;
    }
    if (h->src_off) { SE = 0.0; SFx = 0.0; SFy = 0.0; }
    R[0] = (Ge[0] - Gw[0]) / h->dx + (Hn[0] - Hs[0]) / h->dy - SE;
    R[1] = (Ge[1] - Gw[1]) / h->dx + (Hn[1] - Hs[1]) / h->dy - SFx;
    R[2] = (Ge[2] - Gw[2]) / h->dx + (Hn[2] - Hs[2]) / h->dy - SFy;
}

ORACLE_API int oracle_m1_residual(oracle_m1 *h, double *RE, double *RF)
{
    const long N = (long)h->nx * h->ny;
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < h->ny; ++j)
        for (int i = 0; i < h->nx; ++i) {
            double R[3]; residual_cell(h, i, j, R);
            const long id = (long)j * h->nx + i;
            RE[id] = R[0]; RF[id] = R[1]; RF[N + id] = R[2];
        }
    return 0;
}

/* Forward Euler on the full residual (R3): U^{n+1} = U^n - dt R(U^n); with T given, Eq. 4 explicitly. */
ORACLE_API int oracle_m1_step_explicit(oracle_m1 *h, double dt)
{
    if (!(dt > 0.0)) { snprintf(h->err, sizeof h->err, "dt must be > 0"); return -1; }
    const long N = (long)h->nx * h->ny;
    double *R = (double *)malloc(sizeof(double) * 3 * N);
    if (!R) return -3;
    oracle_m1_residual(h, R, R + N);
    #pragma omp parallel for schedule(static)
    for (long id = 0; id < N; ++id) {
        if (h->has_T && !h->src_off) {
            const double T = h->T[id];
            const double rcv = h->rho_cv ? h->rho_cv[id] : 1.0;
            h->T[id] = T - dt * h->c * h->sa[id] * (h->a_r * T * T * T * T - h->E[id]) / rcv;   /* Eq. 4 */
        }
        h->E[id] -= dt * R[id]; h->Fx[id] -= dt * R[N + id]; h->Fy[id] -= dt * R[2 * N + id];
    }
    free(R);
    return 0;
}

/* ------------------------------------------------------------------------------------------------ */
/* Linearised implicit operator: flux form and assembled 5-point block matrix                        */
/* ------------------------------------------------------------------------------------------------ */

/* eta of the linearised matter coupling (R10): eta = rho c_v/(rho c_v + 4 a_r c sigma_a dt T^3); 1 without T. */
static double eta_cell(const oracle_m1 *h, long id, double dt)
{
    if (!h->has_T) return 1.0;
    const double T = h->T[id], rcv = h->rho_cv ? h->rho_cv[id] : 1.0;
    return rcv / (rcv + 4.0 * h->a_r * h->c * h->sa[id] * dt * T * T * T);
}

/* Value of a vector V = [VE | VFx | VFy] seen at (i, j) by the linear operator.
 * mode 0 (homogeneous part, the matrix): Dirichlet ghost = 0, outflow ghost = adjacent interior value.
 * mode 1 (affine part, goes to the right-hand side): interior = 0, Dirichlet ghost = boundary state. */
static void fetch_vec(const oracle_m1 *h, const double *V, int mode, int i, int j, double v[3])
{
    cell_t u; fetch(h, i, j, &u);
    const long N = (long)h->nx * h->ny;
    if (u.dirichlet_ghost) {
        if (mode == 1) { v[0] = u.E; v[1] = u.Fx; v[2] = u.Fy; } else { v[0] = v[1] = v[2] = 0.0; }
    } else if (mode == 1) { v[0] = v[1] = v[2] = 0.0; }
    else { v[0] = V[u.idx]; v[1] = V[N + u.idx]; v[2] = V[2 * N + u.idx]; }
}

static void lin_pressure(const closure_t *q, const double v[3], double Pi[3])
{
    for (int p = 0; p < 3; ++p) Pi[p] = q->J[p][KE] * v[0] + q->J[p][KFX] * v[1] + q->J[p][KFY] * v[2];
}

/* out = V + dt L_n(V) in flux form (mode 0), or out = dt L_n(ghost part) (mode 1).  Coefficients
 * (a+-, Lambda, alpha, sigma_f, J) are those of the stored state U^n (R4). */
static void apply_cell(const oracle_m1 *h, double dt, const double *V, int mode, int i, int j, double out[3])
{
    cell_t u[5]; closure_t q[5]; double v[5][3], Pi[5][3];
    const int di[5] = { 0, -1, 1, 0, 0 }, dj[5] = { 0, 0, 0, -1, 1 };
    for (int k = 0; k < 5; ++k) {
        fetch(h, i + di[k], j + dj[k], &u[k]);
        closure_eval(h, u[k].E, u[k].Fx, u[k].Fy, &q[k]);
        fetch_vec(h, V, mode, i + di[k], j + dj[k], v[k]);
        lin_pressure(&q[k], v[k], Pi[k]);
    }
    face_t fw, fe, fs, fn; double Gw[3], Ge[3], Hs[3], Hn[3];
    face_eval(h, &u[1], &q[1], &u[0], &q[0], 0, &fw);
    face_eval(h, &u[0], &q[0], &u[2], &q[2], 0, &fe);
    face_eval(h, &u[3], &q[3], &u[0], &q[0], 1, &fs);
    face_eval(h, &u[0], &q[0], &u[4], &q[4], 1, &fn);
    face_flux(h, &fw, 0, v[1][0], v[1][1], v[1][2], Pi[1], v[0][0], v[0][1], v[0][2], Pi[0], Gw);
    face_flux(h, &fe, 0, v[0][0], v[0][1], v[0][2], Pi[0], v[2][0], v[2][1], v[2][2], Pi[2], Ge);
    face_flux(h, &fs, 1, v[3][0], v[3][1], v[3][2], Pi[3], v[0][0], v[0][1], v[0][2], Pi[0], Hs);
    face_flux(h, &fn, 1, v[0][0], v[0][1], v[0][2], Pi[0], v[4][0], v[4][1], v[4][2], Pi[4], Hn);
    const double c = h->c;
    double LE = (Ge[0] - Gw[0]) / h->dx + (Hn[0] - Hs[0]) / h->dy + c * u[0].sa * eta_cell(h, u[0].idx, dt) * v[0][0];
    double LFx = (Ge[1] - Gw[1]) / h->dx + (Hn[1] - Hs[1]) / h->dy;
    double LFy = (Ge[2] - Gw[2]) / h->dx + (Hn[2] - Hs[2]) / h->dy;
    if (h->wb) {
        LFx += c * 0.5 * (fe.sig * 0.5 * (v[0][1] + v[2][1]) + fw.sig * 0.5 * (v[1][1] + v[0][1]));
        LFy += c * 0.5 * (fn.sig * 0.5 * (v[0][2] + v[4][2]) + fs.sig * 0.5 * (v[3][2] + v[0][2]));
    } else { LFx += c * u[0].st * v[0][1]; LFy += c * u[0].st * v[0][2]; }
    const double id = (mode == 0) ? 1.0 : 0.0;
    out[0] = id * v[0][0] + dt * LE; out[1] = id * v[0][1] + dt * LFx; out[2] = id * v[0][2] + dt * LFy;
}

/* Test hook: out = (I + dt L_n) V (mode 0) or dt L_n(ghost states) (mode 1), flux form. */
ORACLE_API int oracle_m1_apply_linear(oracle_m1 *h, double dt, const double *V, double *out, int mode)
{
    const long N = (long)h->nx * h->ny;
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < h->ny; ++j)
        for (int i = 0; i < h->nx; ++i) {
            double o[3]; apply_cell(h, dt, V, mode, i, j, o);
            const long id = (long)j * h->nx + i;
            out[id] = o[0]; out[N + id] = o[1]; out[2 * N + id] = o[2];
        }
    return 0;
}

/* Assembled matrix: per cell five 3x3 blocks (centre, west, east, south, north) and the column cell of each
 * (-1: no column, the block was moved to b (Dirichlet) or folded into the centre block (outflow)). */
typedef struct { double *A; long *col; double *b; long N; } system_t;

static void add_block(double *dst, const double *src) { for (int k = 0; k < 9; ++k) dst[k] += src[k]; }

/* The matrix "update" of PAPER.md:315-321: the graph is fixed, the values follow the entries listed in
 * DESIGN.md ("Implicit system"), obtained by collecting the coefficients of U_i, U_{i+-1}, U_{j+-1} in
 * apply_cell.  b = U^n + affine terms. */
static void assemble_cell(const oracle_m1 *h, double dt, const double *base, int i, int j, double A[5][9], long col[5], double b[3])
{
    cell_t u[5]; closure_t q[5];
    const int di[5] = { 0, -1, 1, 0, 0 }, dj[5] = { 0, 0, 0, -1, 1 };
    for (int k = 0; k < 5; ++k) { fetch(h, i + di[k], j + dj[k], &u[k]); closure_eval(h, u[k].E, u[k].Fx, u[k].Fy, &q[k]); }
    face_t fw, fe, fs, fn;
    face_eval(h, &u[1], &q[1], &u[0], &q[0], 0, &fw);
    face_eval(h, &u[0], &q[0], &u[2], &q[2], 0, &fe);
    face_eval(h, &u[3], &q[3], &u[0], &q[0], 1, &fs);
    face_eval(h, &u[0], &q[0], &u[4], &q[4], 1, &fn);
    const double c = h->c, c2 = c * c, rx = h->hyp_off ? 0.0 : dt / h->dx, ry = h->hyp_off ? 0.0 : dt / h->dy;
    const double eta = eta_cell(h, u[0].idx, dt);
    double se = 0, sw = 0, sn = 0, ss = 0, sc = 0;
    if (h->wb) { se = c * dt * fe.sig / 4; sw = c * dt * fw.sig / 4; sn = c * dt * fn.sig / 4; ss = c * dt * fs.sig / 4; }
    else sc = c * dt * u[0].st;
    memset(A, 0, sizeof(double) * 45);
    double *C = A[BLK_C], *W = A[BLK_W], *Eb = A[BLK_E], *S = A[BLK_S], *Nb = A[BLK_N];
    #define M(B, r, k) (B)[3 * (r) + (k)]
    /* E row */
    M(C, 0, 0) = 1.0 + c * dt * u[0].sa * eta + rx * (-fe.alpha * fe.Lam - fw.alpha * fw.Lam) + ry * (-fn.alpha * fn.Lam - fs.alpha * fs.Lam);
    M(C, 0, 1) = rx * (fe.alpha * fe.ap - fw.alpha * fw.am);
    M(C, 0, 2) = ry * (fn.alpha * fn.ap - fs.alpha * fs.am);
    M(Eb, 0, 0) = rx * fe.alpha * fe.Lam;  M(Eb, 0, 1) = rx * fe.alpha * fe.am;
    M(W, 0, 0) = rx * fw.alpha * fw.Lam;   M(W, 0, 1) = -rx * fw.alpha * fw.ap;
    M(Nb, 0, 0) = ry * fn.alpha * fn.Lam;  M(Nb, 0, 2) = ry * fn.alpha * fn.am;
    M(S, 0, 0) = ry * fs.alpha * fs.Lam;   M(S, 0, 2) = -ry * fs.alpha * fs.ap;
    /* Fx row: x-faces carry J^{xx}, y-faces carry J^{xy}; Fy row: x-faces J^{xy}, y-faces J^{yy} */
    for (int k = 0; k < 3; ++k) {
        M(C, 1, k) = c2 * (rx * (fe.ap - fw.am) * q[0].J[PXX][k] + ry * (fn.ap - fs.am) * q[0].J[PXY][k]);
        M(C, 2, k) = c2 * (rx * (fe.ap - fw.am) * q[0].J[PXY][k] + ry * (fn.ap - fs.am) * q[0].J[PYY][k]);
        M(Eb, 1, k) = c2 * rx * fe.am * q[2].J[PXX][k];  M(Eb, 2, k) = c2 * rx * fe.am * q[2].J[PXY][k];
        M(W, 1, k) = -c2 * rx * fw.ap * q[1].J[PXX][k];  M(W, 2, k) = -c2 * rx * fw.ap * q[1].J[PXY][k];
        M(Nb, 1, k) = c2 * ry * fn.am * q[4].J[PXY][k];  M(Nb, 2, k) = c2 * ry * fn.am * q[4].J[PYY][k];
        M(S, 1, k) = -c2 * ry * fs.ap * q[3].J[PXY][k];  M(S, 2, k) = -c2 * ry * fs.ap * q[3].J[PYY][k];
    }
    const double lam = 1.0 - rx * (fe.Lam + fw.Lam) - ry * (fn.Lam + fs.Lam);
    M(C, 1, 1) += lam + se + sw + sc;       M(C, 2, 2) += lam + sn + ss + sc;
    M(Eb, 1, 1) += rx * fe.Lam + se;        M(Eb, 2, 2) += rx * fe.Lam;
    M(W, 1, 1) += rx * fw.Lam + sw;         M(W, 2, 2) += rx * fw.Lam;
    M(Nb, 1, 1) += ry * fn.Lam;             M(Nb, 2, 2) += ry * fn.Lam + sn;
    M(S, 1, 1) += ry * fs.Lam;              M(S, 2, 2) += ry * fs.Lam + ss;
    #undef M
    /* right-hand side: U^n, emission and sources.  base == NULL: U^n is the stored state (one linearised step);
     * otherwise the stored state is a Newton iterate U^k that only supplies the coefficients and base = [E|Fx|Fy]
     * holds U^n (oracle_m1_step_implicit_newton below). */
    if (base) { const long N_ = (long)h->nx * h->ny; b[0] = base[u[0].idx]; b[1] = base[N_ + u[0].idx]; b[2] = base[2 * N_ + u[0].idx]; }
    else { b[0] = u[0].E; b[1] = u[0].Fx; b[2] = u[0].Fy; }
    if (h->has_T) { const double T = h->T[u[0].idx]; b[0] += c * dt * u[0].sa * eta * h->a_r * T * T * T * T; }
    if (h->source_E) b[0] += dt * h->source_E[u[0].idx];
    /* boundaries (R9) */
    col[BLK_C] = u[0].idx;
    for (int k = 1; k < 5; ++k) {
        const int ii = i + di[k], jj = j + dj[k];
        const int outside = (ii < 0 || ii >= h->nx || jj < 0 || jj >= h->ny);
        if (u[k].dirichlet_ghost) {                    /* known value: block x ghost state moves to b */
            const double g[3] = { u[k].E, u[k].Fx, u[k].Fy };
            for (int r = 0; r < 3; ++r) b[r] -= A[k][3 * r] * g[0] + A[k][3 * r + 1] * g[1] + A[k][3 * r + 2] * g[2];
            memset(A[k], 0, sizeof(double) * 9); col[k] = -1;
        } else if (outside && u[k].idx == u[0].idx) {  /* outflow ghost = this cell: fold into the centre */
            add_block(C, A[k]); memset(A[k], 0, sizeof(double) * 9); col[k] = -1;
        } else col[k] = u[k].idx;
    }
}

static int system_build(const oracle_m1 *h, double dt, const double *base, system_t *s)
{
    const long N = (long)h->nx * h->ny;
    s->N = N;
    s->A = (double *)malloc(sizeof(double) * 45 * N);
    s->col = (long *)malloc(sizeof(long) * 5 * N);
    s->b = (double *)malloc(sizeof(double) * 3 * N);
    if (!s->A || !s->col || !s->b) return -3;
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < h->ny; ++j)
        for (int i = 0; i < h->nx; ++i) {
            const long id = (long)j * h->nx + i;
            double b[3];
            assemble_cell(h, dt, base, i, j, (double (*)[9])(s->A + 45 * id), s->col + 5 * id, b);
            s->b[id] = b[0]; s->b[N + id] = b[1]; s->b[2 * N + id] = b[2];
        }
    return 0;
}
static void system_free(system_t *s) { free(s->A); free(s->col); free(s->b); }

/* Test hook: the assembled blocks A[N][5][3][3] (centre, west, east, south, north), their column cells and b. */
ORACLE_API int oracle_m1_assemble(oracle_m1 *h, double dt, double *A, long *col, double *b)
{
    system_t s; const int rc = system_build(h, dt, NULL, &s); if (rc) return rc;
    memcpy(A, s.A, sizeof(double) * 45 * s.N); memcpy(col, s.col, sizeof(long) * 5 * s.N);
    memcpy(b, s.b, sizeof(double) * 3 * s.N);
    system_free(&s); return 0;
}

/* y = A x, x and y stored as planes [E | Fx | Fy] */
static void spmv(const system_t *s, const double *x, double *y)
{
    const long N = s->N;
    #pragma omp parallel for schedule(static)
    for (long id = 0; id < N; ++id) {
        double acc[3] = { 0, 0, 0 };
        for (int k = 0; k < 5; ++k) {
            const long cj = s->col[5 * id + k]; if (cj < 0) continue;
            const double *B = s->A + 45 * id + 9 * k;
            const double v0 = x[cj], v1 = x[N + cj], v2 = x[2 * N + cj];
            for (int r = 0; r < 3; ++r) acc[r] += B[3 * r] * v0 + B[3 * r + 1] * v1 + B[3 * r + 2] * v2;
        }
        y[id] = acc[0]; y[N + id] = acc[1]; y[2 * N + id] = acc[2];
    }
}

/* z = M^-1 v, M = the 3x3 diagonal blocks of A (Eq. 27 taken block-wise): Gaussian elimination with
 * partial pivoting, cell by cell. */
static void solve3(const double *B, const double r[3], double z[3])
{
    double a[3][4];
    for (int i = 0; i < 3; ++i) { for (int k = 0; k < 3; ++k) a[i][k] = B[3 * i + k]; a[i][3] = r[i]; }
    for (int p = 0; p < 3; ++p) {
        int piv = p;
        for (int i = p + 1; i < 3; ++i) if (fabs(a[i][p]) > fabs(a[piv][p])) piv = i;
        if (piv != p) for (int k = 0; k < 4; ++k) { const double t = a[p][k]; a[p][k] = a[piv][k]; a[piv][k] = t; }
        for (int i = p + 1; i < 3; ++i) { const double m = a[i][p] / a[p][p]; for (int k = p; k < 4; ++k) a[i][k] -= m * a[p][k]; }
    }
    for (int i = 2; i >= 0; --i) { double sacc = a[i][3]; for (int k = i + 1; k < 3; ++k) sacc -= a[i][k] * z[k]; z[i] = sacc / a[i][i]; }
}
static void precond(const system_t *s, const double *v, double *z)
{
    const long N = s->N;
    #pragma omp parallel for schedule(static)
    for (long id = 0; id < N; ++id) {
        const double r[3] = { v[id], v[N + id], v[2 * N + id] }; double zz[3];
        solve3(s->A + 45 * id, r, zz);
        z[id] = zz[0]; z[N + id] = zz[1]; z[2 * N + id] = zz[2];
    }
}
/* ------------------------------------------------------------------------------------------------ */
/* Multigrid preconditioner (the five steps quoted from Saad 2003; R15)  */
/* ------------------------------------------------------------------------------------------------ */
/* The paper uses an algebraic multigrid from a library (MueLu) and does not specify it.  On this structured grid the
 * hierarchy is geometric: aggregates of 2x2 cells (the last one in a direction is 1 wide when the size is odd), down to
 * a single cell.  On every level, with D = the 3x3 diagonal blocks:
 *   restriction        R = P0^T   (sum over the aggregate; P0 = piecewise-constant injection, per component)
 *   interpolation      P = D^-1 P0   (piecewise constant in the block-Jacobi-scaled variable D x)
 *   coarse operator    R A P   ("R A P y = R r~") -- again a 5-point stencil of 3x3 blocks
 *   smoother           damped block-Jacobi, z += omega D^-1 (r - A z)   ("a simple method such as Jacobi")
 * One V-cycle, zero initial guess, one pre- and one post-smoothing sweep (steps 1-5 of PAPER.md:283-287); on the
 * coarsest level `mg_coarse_sweeps` smoother sweeps replace the direct solve of step 3. */
typedef struct mg_hier {
    int nlev;
    int nx[32], ny[32];
    system_t lev[32];            /* lev[0] aliases the fine system (not owned); b unused on coarse levels */
    double *r[32], *z[32], *t[32];   /* work vectors per level (r[0] unused) */
} mg_hier;

static void inv3(const double *B, double *Bi)   /* Bi = B^-1 by three solves (Gaussian elimination with pivoting) */
{
    for (int k = 0; k < 3; ++k) {
        const double e[3] = { k == 0, k == 1, k == 2 }; double z[3];
        solve3(B, e, z);
        for (int r = 0; r < 3; ++r) Bi[3 * r + k] = z[r];
    }
}

/* Coarse system R A P of one level. */
static int mg_coarsen(const system_t *f, int nx, int ny, system_t *c, int *cnx, int *cny)
{
    const int cx = (nx + 1) / 2, cy = (ny + 1) / 2;
    const long Nc = (long)cx * cy;
    c->N = Nc; c->b = NULL;
    c->A = (double *)calloc((size_t)45 * Nc, sizeof(double));
    c->col = (long *)malloc(sizeof(long) * 5 * Nc);
    if (!c->A || !c->col) return -3;
    for (long k = 0; k < 5 * Nc; ++k) c->col[k] = -1;
    for (long a = 0; a < Nc; ++a) c->col[5 * a + BLK_C] = a;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const long id = (long)j * nx + i, a = (long)(j / 2) * cx + i / 2;
            for (int k = 0; k < 5; ++k) {
                const long cj = f->col[5 * id + k]; if (cj < 0) continue;
                double Di[9], B[9];
                inv3(f->A + 45 * cj, Di);                       /* D^-1 of the column cell */
                const double *Ak = f->A + 45 * id + 9 * k;
                for (int r = 0; r < 3; ++r) for (int q = 0; q < 3; ++q)
                    B[3 * r + q] = Ak[3 * r] * Di[q] + Ak[3 * r + 1] * Di[3 + q] + Ak[3 * r + 2] * Di[6 + q];
                const long ac = (cj / nx / 2) * cx + (cj % nx) / 2;     /* aggregate of the column cell */
                const int kc = (ac == a) ? BLK_C : k;           /* inside the aggregate -> diagonal block */
                add_block(c->A + 45 * a + 9 * kc, B);
                c->col[5 * a + kc] = ac;
            }
        }
    *cnx = cx; *cny = cy;
    return 0;
}

static void mg_free(mg_hier *m)
{
    if (!m) return;
    for (int l = 0; l < m->nlev; ++l) {
        if (l > 0) { free(m->lev[l].A); free(m->lev[l].col); }
        free(m->r[l]); free(m->z[l]); free(m->t[l]);
    }
    free(m);
}

static mg_hier *mg_build(const oracle_m1 *h, const system_t *s)
{
    mg_hier *m = (mg_hier *)calloc(1, sizeof(mg_hier));
    if (!m) return NULL;
    m->lev[0] = *s; m->nx[0] = h->nx; m->ny[0] = h->ny; m->nlev = 1;
    while ((m->nx[m->nlev - 1] > 1 || m->ny[m->nlev - 1] > 1) && m->nlev < 32) {
        const int l = m->nlev;
        if (mg_coarsen(&m->lev[l - 1], m->nx[l - 1], m->ny[l - 1], &m->lev[l], &m->nx[l], &m->ny[l])) { m->nlev = l + 1; mg_free(m); return NULL; }
        m->nlev = l + 1;
    }
    for (int l = 0; l < m->nlev; ++l) {
        const size_t n = 3 * (size_t)m->lev[l].N;
        m->r[l] = (double *)malloc(sizeof(double) * n); m->z[l] = (double *)malloc(sizeof(double) * n); m->t[l] = (double *)malloc(sizeof(double) * n);
        if (!m->r[l] || !m->z[l] || !m->t[l]) { mg_free(m); return NULL; }
    }
    return m;
}

/* z += omega D^-1 (r - A z); `first` = 1: z = omega D^-1 r (zero initial guess).  t: work vector. */
static void mg_smooth(const system_t *s, double omega, const double *r, double *z, double *t, int first)
{
    const long n = 3 * s->N;
    if (first) { precond(s, r, z); for (long k = 0; k < n; ++k) z[k] *= omega; return; }
    spmv(s, z, t);
    for (long k = 0; k < n; ++k) t[k] = r[k] - t[k];
    double *d = (double *)malloc(sizeof(double) * n);
    precond(s, t, d);
    for (long k = 0; k < n; ++k) z[k] += omega * d[k];
    free(d);
}

/* One V-cycle on level l: z ~ A_l^-1 r (steps 1-5 of PAPER.md:283-287). */
static void mg_vcycle(const oracle_m1 *h, mg_hier *m, int l, const double *r, double *z)
{
    const system_t *s = &m->lev[l];
    const long N = s->N;
    double *t = m->t[l];
    mg_smooth(s, h->mg_omega, r, z, t, 1);                                   /* 1. pre-smoothing */
    if (l == m->nlev - 1) {                                                  /* coarsest level: more sweeps instead of a direct solve */
        for (int k = 1; k < h->mg_coarse_sweeps; ++k) mg_smooth(s, h->mg_omega, r, z, t, 0);
        return;
    }
    const int nx = m->nx[l], ny = m->ny[l], cx = m->nx[l + 1];
    const long Nc = m->lev[l + 1].N;
    double *rc = m->r[l + 1], *zc = m->z[l + 1];
    spmv(s, z, t);                                                           /* 2. residual, restricted: rc = P0^T (r - A z) */
    memset(rc, 0, sizeof(double) * 3 * Nc);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const long id = (long)j * nx + i, a = (long)(j / 2) * cx + i / 2;
            for (int q = 0; q < 3; ++q) rc[q * Nc + a] += r[q * N + id] - t[q * N + id];
        }
    mg_vcycle(h, m, l + 1, rc, zc);                                          /* 3. coarse problem, recursively */
    for (int j = 0; j < ny; ++j)                                             /* 4. interpolation: z += D^-1 P0 zc */
        for (int i = 0; i < nx; ++i) {
            const long id = (long)j * nx + i, a = (long)(j / 2) * cx + i / 2;
            const double e[3] = { zc[a], zc[Nc + a], zc[2 * Nc + a] }; double d[3];
            solve3(s->A + 45 * id, e, d);
            for (int q = 0; q < 3; ++q) z[q * N + id] += d[q];
        }
    mg_smooth(s, h->mg_omega, r, z, t, 0);                                   /* 5. post-smoothing */
}

/* The right preconditioner of the Krylov solvers: block-Jacobi (Eq. 27 block-wise) or one multigrid V-cycle. */
static void apply_precond(const oracle_m1 *h, const system_t *s, const double *v, double *z)
{
    if (h->precond_kind == 1 && h->mg) mg_vcycle(h, h->mg, 0, v, z);
    else precond(s, v, z);
}

static double dot(const double *a, const double *b, long n)
{
    double sacc = 0.0;
    #pragma omp parallel for schedule(static) reduction(+ : sacc)
    for (long k = 0; k < n; ++k) sacc += a[k] * b[k];
    return sacc;
}

static void hist_push(oracle_m1 *h, double r)
{
    if (h->nhist == h->caphist) { h->caphist = h->caphist ? 2 * h->caphist : 256; h->hist = (double *)realloc(h->hist, sizeof(double) * h->caphist); }
    h->hist[h->nhist++] = r;
}

/* Restarted GMRES(m), right-preconditioned (Saad 2003, Alg. 9.5), modified Gram-Schmidt,
 * Givens rotations.  x holds the initial guess on entry (R9: U^n) and the solution on exit.
 * Stops when ||b - A x||_2 <= tol ||b||_2 or after maxit inner iterations in total.
 * Returns the number of inner iterations; *relres = true relative residual at exit. */
static int gmres(oracle_m1 *h, const system_t *s, double *x, double tol, int m, int maxit, double *relres)
{
    const long n = 3 * s->N;
    double *V = (double *)malloc(sizeof(double) * n * (size_t)(m + 1));
    double *w = (double *)malloc(sizeof(double) * n), *z = (double *)malloc(sizeof(double) * n);
    double *H = (double *)calloc((size_t)(m + 1) * m, sizeof(double));
    double *cs = (double *)malloc(sizeof(double) * m), *sn = (double *)malloc(sizeof(double) * m);
    double *g = (double *)malloc(sizeof(double) * (m + 1)), *y = (double *)malloc(sizeof(double) * m);
    if (!V || !w || !z || !H || !cs || !sn || !g || !y) return -3;
    #define HH(i, j) H[(size_t)(i) * m + (j)]
    const double bnorm = sqrt(dot(s->b, s->b, n));
    const double target = tol * bnorm;
    int its = 0; double rnorm;
    h->nhist = 0;
    for (;;) {
        spmv(s, x, w);
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < n; ++k) w[k] = s->b[k] - w[k];
        rnorm = sqrt(dot(w, w, n));
        hist_push(h, bnorm > 0 ? rnorm / bnorm : rnorm);
        if (rnorm <= target || its >= maxit) break;
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < n; ++k) V[k] = w[k] / rnorm;
        for (int k = 0; k <= m; ++k) g[k] = 0.0;
        g[0] = rnorm;
        int j = 0;
        for (; j < m && its < maxit; ) {
            double *vj = V + (size_t)j * n, *vn = V + (size_t)(j + 1) * n;
            apply_precond(h, s, vj, z);
            spmv(s, z, vn);
            for (int i = 0; i <= j; ++i) {                       /* modified Gram-Schmidt */
                const double *vi = V + (size_t)i * n;
                const double hij = dot(vn, vi, n);
                HH(i, j) = hij;
                #pragma omp parallel for schedule(static)
                for (long k = 0; k < n; ++k) vn[k] -= hij * vi[k];
            }
            const double hn = sqrt(dot(vn, vn, n));
            HH(j + 1, j) = hn;
            if (hn > 0.0) {
                #pragma omp parallel for schedule(static)
                for (long k = 0; k < n; ++k) vn[k] /= hn;
            }
            for (int i = 0; i < j; ++i) {                        /* apply the previous rotations */
                const double t = cs[i] * HH(i, j) + sn[i] * HH(i + 1, j);
                HH(i + 1, j) = -sn[i] * HH(i, j) + cs[i] * HH(i + 1, j);
                HH(i, j) = t;
            }
            const double d = hypot(HH(j, j), HH(j + 1, j));
            cs[j] = HH(j, j) / d; sn[j] = HH(j + 1, j) / d;
            HH(j, j) = d; HH(j + 1, j) = 0.0;
            g[j + 1] = -sn[j] * g[j]; g[j] = cs[j] * g[j];
            ++j; ++its;
            hist_push(h, bnorm > 0 ? fabs(g[j]) / bnorm : fabs(g[j]));
            if (fabs(g[j]) <= target || hn == 0.0) break;
        }
        for (int i = j - 1; i >= 0; --i) {                       /* back substitution H y = g */
            double sacc = g[i];
            for (int k = i + 1; k < j; ++k) sacc -= HH(i, k) * y[k];
            y[i] = sacc / HH(i, i);
        }
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < n; ++k) { double sacc = 0.0; for (int i = 0; i < j; ++i) sacc += y[i] * V[(size_t)i * n + k]; w[k] = sacc; }
        apply_precond(h, s, w, z);                                        /* x += M^-1 (V y) */
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < n; ++k) x[k] += z[k];
    }
    #undef HH
    *relres = bnorm > 0 ? rnorm / bnorm : rnorm;
    free(V); free(w); free(z); free(H); free(cs); free(sn); free(g); free(y);
    return its;
}

/* BiCGStab (van der Vorst 1992; the paper's Krylov method, "BiCGStab"), right-preconditioned with the same
 * block-Jacobi M: p^ = M^-1 p, v = A p^, s^ = M^-1 s, t = A s^, x += alpha p^ + omega s^.
 * Stops when the recursive residual satisfies ||r|| <= tol ||b||; the TRUE residual is then recomputed and, if it is still
 * above the target (drift), the iteration restarts from it.  One iteration = two operator applications.
 * `restart` is unused.  Returns the number of iterations; *relres = true relative residual at exit. */
static int bicgstab(oracle_m1 *h, const system_t *s, double *x, double tol, int maxit, double *relres)
{
    const long n = 3 * s->N;
    double *r = (double *)malloc(sizeof(double) * n), *rh = (double *)malloc(sizeof(double) * n), *p = (double *)malloc(sizeof(double) * n);
    double *v = (double *)malloc(sizeof(double) * n), *t = (double *)malloc(sizeof(double) * n), *ph = (double *)malloc(sizeof(double) * n);
    double *sh = (double *)malloc(sizeof(double) * n);
    if (!r || !rh || !p || !v || !t || !ph || !sh) return -3;
    const double bnorm = sqrt(dot(s->b, s->b, n)), target = tol * bnorm;
    int its = 0; double rnorm;
    h->nhist = 0;
    for (;;) {
        spmv(s, x, r);
        for (long k = 0; k < n; ++k) r[k] = s->b[k] - r[k];
        rnorm = sqrt(dot(r, r, n));
        hist_push(h, bnorm > 0 ? rnorm / bnorm : rnorm);
        if (rnorm <= target || its >= maxit) break;
        memcpy(rh, r, sizeof(double) * n);
        memset(p, 0, sizeof(double) * n); memset(v, 0, sizeof(double) * n);
        double rho = 1.0, alpha = 1.0, omega = 1.0;
        const int its0 = its;
        while (its < maxit) {
            const double rho_new = dot(rh, r, n);
            if (rho_new == 0.0 || omega == 0.0) break;                 /* breakdown: restart from the true residual */
            const double beta = (rho_new / rho) * (alpha / omega);
            for (long k = 0; k < n; ++k) p[k] = r[k] + beta * (p[k] - omega * v[k]);
            apply_precond(h, s, p, ph); spmv(s, ph, v);
            const double rhv = dot(rh, v, n);
            if (rhv == 0.0) break;
            alpha = rho_new / rhv;
            for (long k = 0; k < n; ++k) r[k] -= alpha * v[k];          /* s, stored in r */
            apply_precond(h, s, r, sh); spmv(s, sh, t);
            const double tt = dot(t, t, n);
            omega = (tt > 0.0) ? dot(t, r, n) / tt : 0.0;
            for (long k = 0; k < n; ++k) { x[k] += alpha * ph[k] + omega * sh[k]; r[k] -= omega * t[k]; }
            rho = rho_new; ++its;
            const double rn = sqrt(dot(r, r, n));
            hist_push(h, bnorm > 0 ? rn / bnorm : rn);
            if (rn <= target) break;
        }
        if (its == its0) break;                                           /* no progress possible */
    }
    *relres = bnorm > 0 ? rnorm / bnorm : rnorm;
    free(r); free(rh); free(p); free(v); free(t); free(ph); free(sh);
    return its;
}

/* Krylov solve of one assembled system with the chosen method and preconditioner. */
static int solve_linear(oracle_m1 *h, const system_t *s, double *x, double tol, int restart, int maxit, double *relres)
{
    h->mg = NULL;
    if (h->precond_kind == 1 && !(h->mg = mg_build(h, s))) return -3;
    const int its = h->krylov == 1 ? bicgstab(h, s, x, tol, maxit, relres) : gmres(h, s, x, tol, restart, maxit, relres);
    mg_free(h->mg); h->mg = NULL;
    return its;
}

/* Test hooks for the multigrid preconditioner: one V-cycle z = M^-1 r on the system assembled for dt ... */
ORACLE_API int oracle_m1_mg_apply(oracle_m1 *h, double dt, const double *r, double *z)
{
    system_t s; int rc = system_build(h, dt, NULL, &s); if (rc) return rc;
    mg_hier *m = mg_build(h, &s);
    if (!m) { system_free(&s); return -3; }
    mg_vcycle(h, m, 0, r, z);
    mg_free(m); system_free(&s);
    return 0;
}
/* ... and the blocks of level `level` (0 = fine): returns the number of levels; dims = {nx, ny} of that level; A, col may
 * be NULL to query the sizes only. */
ORACLE_API int oracle_m1_mg_level(oracle_m1 *h, double dt, int level, double *A, long *col, int *dims)
{
    system_t s; int rc = system_build(h, dt, NULL, &s); if (rc) return rc;
    mg_hier *m = mg_build(h, &s);
    if (!m) { system_free(&s); return -3; }
    const int nlev = m->nlev;
    if (level >= 0 && level < nlev) {
        dims[0] = m->nx[level]; dims[1] = m->ny[level];
        if (A) memcpy(A, m->lev[level].A, sizeof(double) * 45 * m->lev[level].N);
        if (col) memcpy(col, m->lev[level].col, sizeof(long) * 5 * m->lev[level].N);
    }
    mg_free(m); system_free(&s);
    return nlev;
}

/* One linearised implicit step (R4): (I + dt L_n) U^{n+1} = U^n + affine terms; then the T update (R10). */
ORACLE_API int oracle_m1_step_implicit(oracle_m1 *h, double dt, double tol, int restart, int maxit, double *final_residual)
{
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0) { snprintf(h->err, sizeof h->err, "bad argument"); return -1; }
    system_t s; const int rc = system_build(h, dt, NULL, &s); if (rc) return rc;
    const long N = s.N;
    double *x = (double *)malloc(sizeof(double) * 3 * N);
    memcpy(x, h->E, sizeof(double) * N); memcpy(x + N, h->Fx, sizeof(double) * N); memcpy(x + 2 * N, h->Fy, sizeof(double) * N);
    double rel = 0.0;
    const int its = solve_linear(h, &s, x, tol, restart, maxit, &rel);
    if (its >= 0) {
        if (h->has_T) {
            #pragma omp parallel for schedule(static)
            for (long id = 0; id < N; ++id) {
                const double T = h->T[id], rcv = h->rho_cv ? h->rho_cv[id] : 1.0;
                const double Theta = h->a_r * T * T * T * T;
                h->T[id] = T + h->c * h->sa[id] * dt * (x[id] - Theta) / (rcv + 4.0 * h->a_r * h->c * h->sa[id] * dt * T * T * T);
            }
        }
        memcpy(h->E, x, sizeof(double) * N); memcpy(h->Fx, x + N, sizeof(double) * N); memcpy(h->Fy, x + 2 * N, sizeof(double) * N);
        if (final_residual) *final_residual = rel;
    }
    free(x); system_free(&s);
    return its;
}

/* Newton-Raphson on the implicit step ("the system is non-linear ... we use a Newton-Raphson method ... a
 * linear system has to be solved at each iteration").  With the Jacobian of DESIGN.md reading R4 (analytic pressure
 * Jacobian, derivatives of a+-, Lambda, alpha dropped) and P homogeneous of degree 1, the Newton update
 *   J_k (U^{k+1} - U^k) = -(U^k - U^n + dt R(U^k)),  J_k = I + dt L_{U^k},  L_{U^k} U^k = R(U^k)
 * is the same as   (I + dt L_{U^k}) U^{k+1} = U^n + affine terms:
 * re-assemble with the coefficients of the iterate, keep U^n on the right-hand side, start GMRES from U^k.
 * The first iteration is exactly oracle_m1_step_implicit.  Stops when ||U^{k+1} - U^k||_2 <= newton_tol ||U^{k+1}||_2
 * or after max_newton iterations.  The temperature is linearised about T^n throughout and updated once at the end.
 * Returns the total number of GMRES iterations. */
ORACLE_API int oracle_m1_step_implicit_newton(oracle_m1 *h, double dt, double tol, int restart, int maxit, double newton_tol,
                                              int max_newton, int *newton_iterations, double *final_residual, double *final_update)
{
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0 || !(newton_tol >= 0.0) || max_newton < 1) { snprintf(h->err, sizeof h->err, "bad argument"); return -1; }
    const long N = (long)h->nx * h->ny;
    double *base = (double *)malloc(sizeof(double) * 3 * N), *x = (double *)malloc(sizeof(double) * 3 * N);
    if (!base || !x) return -3;
    memcpy(base, h->E, sizeof(double) * N); memcpy(base + N, h->Fx, sizeof(double) * N); memcpy(base + 2 * N, h->Fy, sizeof(double) * N);
    int total = 0, k = 0; double rel = 0.0, upd = 0.0;
    for (k = 0; k < max_newton; ++k) {
        system_t s; const int rc = system_build(h, dt, base, &s); if (rc) { free(base); free(x); return rc; }
        memcpy(x, h->E, sizeof(double) * N); memcpy(x + N, h->Fx, sizeof(double) * N); memcpy(x + 2 * N, h->Fy, sizeof(double) * N);
        const int its = solve_linear(h, &s, x, tol, restart, maxit, &rel);
        system_free(&s);
        if (its < 0) { free(base); free(x); return its; }
        total += its;
        double d2 = 0.0, n2 = 0.0;
        for (long id = 0; id < N; ++id) {
            const double dE = x[id] - h->E[id], dFx = x[N + id] - h->Fx[id], dFy = x[2 * N + id] - h->Fy[id];
            d2 += dE * dE + dFx * dFx + dFy * dFy;
            n2 += x[id] * x[id] + x[N + id] * x[N + id] + x[2 * N + id] * x[2 * N + id];
        }
        memcpy(h->E, x, sizeof(double) * N); memcpy(h->Fx, x + N, sizeof(double) * N); memcpy(h->Fy, x + 2 * N, sizeof(double) * N);
        upd = (n2 > 0.0) ? sqrt(d2 / n2) : sqrt(d2);
        if (upd <= newton_tol) { ++k; break; }
    }
    if (h->has_T) {
        for (long id = 0; id < N; ++id) {
            const double T = h->T[id], rcv = h->rho_cv ? h->rho_cv[id] : 1.0;
            const double Theta = h->a_r * T * T * T * T;
            h->T[id] = T + h->c * h->sa[id] * dt * (h->E[id] - Theta) / (rcv + 4.0 * h->a_r * h->c * h->sa[id] * dt * T * T * T);
        }
    }
    if (newton_iterations) *newton_iterations = k;
    if (final_residual) *final_residual = rel;
    if (final_update) *final_update = upd;
    free(base); free(x);
    return total;
}

/* Semi-implicit step ("source terms remain implicit, but the hyperbolic part is time-explicit"; used by the
 * paper for the beam and shadow tests):
 *   U* = U^n - dt [flux divergence](U^n)            (Eq. 12 without its right-hand side, alpha etc. at t^n)
 *   (I + dt S) U^{n+1} = U* + affine terms          (S = the source operator: c sigma_a eta on E; the WB weights of Eqs. 18-19 or,
 *                                                    with well_balanced = 0, c sigma_t on F (Eq. 16); Eq. B.1 is its F row)
 * The second line is the assembled system of the implicit step with the flux terms switched off; it depends on the
 * opacities only, so nothing is linearised.  Solved with the same Krylov method and preconditioner. */
ORACLE_API int oracle_m1_step_semi_implicit(oracle_m1 *h, double dt, double tol, int restart, int maxit, double *final_residual)
{
    if (!(dt > 0.0) || !(tol > 0.0) || restart < 1 || maxit < 0) { snprintf(h->err, sizeof h->err, "bad argument"); return -1; }
    h->src_off = 1;
    int rc = oracle_m1_step_explicit(h, dt);
    h->src_off = 0;
    if (rc) return rc;
    h->hyp_off = 1;
    rc = oracle_m1_step_implicit(h, dt, tol, restart, maxit, final_residual);
    h->hyp_off = 0;
    return rc;
}

/* Step 3 of the operator splitting: explicit addition of the velocity-dependent sources of
 * Eq. 6, all cell-centred (R14: the WB face form is reserved for the sigma F/c term of the
 * momentum equation, which belongs to the hydro solver and is not part of this step).
 *   E  += dt * S_E,  S_E = (sigma/c) u.F + (sigma/c) E u.u + (sigma/c) u.(u.P)
 *   F  += dt * c S_F, S_F = sigma u.P + sigma a_r T^4 u + (sigma/c^2) u (u.F)                              */
ORACLE_API int oracle_m1_add_velocity_sources(oracle_m1 *h, double dt)
{
    if (!h->ux || !h->uy) { snprintf(h->err, sizeof h->err, "ux, uy not set"); return -1; }
    const long N = (long)h->nx * h->ny; const double c = h->c;
    #pragma omp parallel for schedule(static)
    for (long id = 0; id < N; ++id) {
        closure_t q; closure_eval(h, h->E[id], h->Fx[id], h->Fy[id], &q);
        const double s = h->st[id], ux = h->ux[id], uy = h->uy[id];
        const double E = h->E[id], Fx = h->Fx[id], Fy = h->Fy[id];
        const double uPx = ux * q.P[PXX] + uy * q.P[PXY], uPy = ux * q.P[PXY] + uy * q.P[PYY];
        const double uF = ux * Fx + uy * Fy, uu = ux * ux + uy * uy;
        double Th = 0.0; if (h->has_T) { const double T = h->T[id]; Th = h->a_r * T * T * T * T; }
        const double SE = (s / c) * (uF + E * uu + (ux * uPx + uy * uPy));
        const double SFx = s * uPx + s * Th * ux + (s / (c * c)) * ux * uF;
        const double SFy = s * uPy + s * Th * uy + (s / (c * c)) * uy * uF;
        h->E[id] = E + dt * SE; h->Fx[id] = Fx + dt * c * SFx; h->Fy[id] = Fy + dt * c * SFy;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------ */
/* Handle, state, options                                                                            */
/* ------------------------------------------------------------------------------------------------ */

ORACLE_API oracle_m1 *oracle_m1_create(int nx, int ny, double dx, double dy, double c, const int *bc)
{
    if (nx < 1 || ny < 1 || !(dx > 0) || !(dy > 0) || !(c > 0)) return NULL;
    oracle_m1 *h = (oracle_m1 *)calloc(1, sizeof *h);
    if (!h) return NULL;
    h->nx = nx; h->ny = ny; h->dx = dx; h->dy = dy; h->c = c;
    for (int s = 0; s < 4; ++s) h->bc[s] = bc ? bc[s] : BC_PERIODIC;
    /* periodic must be paired */
    if ((h->bc[XLO] == BC_PERIODIC) != (h->bc[XHI] == BC_PERIODIC) || (h->bc[YLO] == BC_PERIODIC) != (h->bc[YHI] == BC_PERIODIC)) { free(h); return NULL; }
    const size_t N = (size_t)nx * ny;
    h->E = (double *)calloc(N, sizeof(double)); h->Fx = (double *)calloc(N, sizeof(double)); h->Fy = (double *)calloc(N, sizeof(double));
    h->sa = (double *)calloc(N, sizeof(double)); h->st = (double *)calloc(N, sizeof(double)); h->T = (double *)calloc(N, sizeof(double));
    for (int s = 0; s < 4; ++s) { const size_t len = (s < 2) ? ny : nx; for (int k = 0; k < 5; ++k) h->gh[s][k] = (double *)calloc(len, sizeof(double)); }
    h->wb = 1; h->ap = 1; h->eig = 0; h->closure = 0; h->lin = 0; h->eig_floor = 0.0; h->a_r = 1.0; h->mg_omega = 0.8; h->mg_coarse_sweeps = 2;
    return h;
}

ORACLE_API void oracle_m1_destroy(oracle_m1 *h)
{
    if (!h) return;
    free(h->E); free(h->Fx); free(h->Fy); free(h->sa); free(h->st); free(h->T);
    for (int s = 0; s < 4; ++s) for (int k = 0; k < 5; ++k) free(h->gh[s][k]);
    free(h->rho_cv); free(h->ux); free(h->uy); free(h->source_E); free(h->hist);
    free(h);
}

ORACLE_API int oracle_m1_set_state(oracle_m1 *h, const double *E, const double *F, const double *sa, const double *ss, const double *T)
{
    const size_t N = (size_t)h->nx * h->ny;
    memcpy(h->E, E, N * sizeof(double)); memcpy(h->Fx, F, N * sizeof(double)); memcpy(h->Fy, F + N, N * sizeof(double));
    memcpy(h->sa, sa, N * sizeof(double));
    for (size_t k = 0; k < N; ++k) h->st[k] = sa[k] + ss[k];
    h->has_T = (T != NULL);
    if (T) memcpy(h->T, T, N * sizeof(double));
    return 0;
}

/* One Dirichlet ghost line on `side`: ny values for XLO/XHI, nx values for YLO/YHI; F_g = [Fx line | Fy line]. */
ORACLE_API int oracle_m1_set_boundary(oracle_m1 *h, int side, const double *E_g, const double *F_g, const double *sa_g, const double *ss_g)
{
    if (side < 0 || side > 3) return -1;
    const size_t len = (side < 2) ? h->ny : h->nx;
    memcpy(h->gh[side][0], E_g, len * sizeof(double)); memcpy(h->gh[side][1], F_g, len * sizeof(double));
    memcpy(h->gh[side][2], F_g + len, len * sizeof(double)); memcpy(h->gh[side][3], sa_g, len * sizeof(double));
    for (size_t k = 0; k < len; ++k) h->gh[side][4][k] = sa_g[k] + ss_g[k];
    return 0;
}

ORACLE_API int oracle_m1_set_option(oracle_m1 *h, const char *key, double value)
{
    if (!strcmp(key, "well_balanced")) h->wb = (value != 0.0);
    else if (!strcmp(key, "ap_mode")) h->ap = (int)value;
    else if (!strcmp(key, "eig_mode")) h->eig = (int)value;
    else if (!strcmp(key, "closure")) h->closure = (int)value;
    else if (!strcmp(key, "linearisation")) h->lin = (int)value;
    else if (!strcmp(key, "eig_floor")) h->eig_floor = value;
    else if (!strcmp(key, "krylov")) h->krylov = (int)value;
    else if (!strcmp(key, "preconditioner")) h->precond_kind = (int)value;
    else if (!strcmp(key, "mg_omega")) h->mg_omega = value;
    else if (!strcmp(key, "mg_coarse_sweeps")) h->mg_coarse_sweeps = (int)value;
    else if (!strcmp(key, "a_r")) h->a_r = value;
    else { snprintf(h->err, sizeof h->err, "unknown option %s", key); return -1; }
    return 0;
}

ORACLE_API int oracle_m1_set_field(oracle_m1 *h, const char *name, const double *plane)
{
    double **dst = NULL;
    if (!strcmp(name, "rho_cv")) dst = &h->rho_cv; else if (!strcmp(name, "ux")) dst = &h->ux;
    else if (!strcmp(name, "uy")) dst = &h->uy; else if (!strcmp(name, "source_E")) dst = &h->source_E;
    else { snprintf(h->err, sizeof h->err, "unknown field %s", name); return -1; }
    const size_t N = (size_t)h->nx * h->ny;
    if (!plane) { free(*dst); *dst = NULL; return 0; }
    if (!*dst) *dst = (double *)malloc(N * sizeof(double));
    memcpy(*dst, plane, N * sizeof(double));
    return 0;
}

ORACLE_API int oracle_m1_get_state(oracle_m1 *h, double *E, double *F, double *T)
{
    const size_t N = (size_t)h->nx * h->ny;
    memcpy(E, h->E, N * sizeof(double)); memcpy(F, h->Fx, N * sizeof(double)); memcpy(F + N, h->Fy, N * sizeof(double));
    if (T) memcpy(T, h->T, N * sizeof(double));
    return 0;
}

/* Guards of PAPER.md:245, 513: cells with E <= 0 and cells with |F| > cE (reported, never fatal). */
ORACLE_API int oracle_m1_count_unrealizable(oracle_m1 *h, long *n_E_nonpositive, long *n_f_above_one)
{
    const long N = (long)h->nx * h->ny; long a = 0, b = 0;
    for (long id = 0; id < N; ++id) {
        if (!(h->E[id] > 0.0)) ++a;
        else if (sqrt(h->Fx[id] * h->Fx[id] + h->Fy[id] * h->Fy[id]) > h->c * h->E[id]) ++b;
    }
    *n_E_nonpositive = a; *n_f_above_one = b;
    return 0;
}

/* Residual history of the last solve: entry 0 is the true relative residual of the initial guess, then one
 * implicit estimate |g_{j+1}|/||b|| per inner iteration, and one true residual at each restart. */
ORACLE_API int oracle_m1_get_history(oracle_m1 *h, double *buf, int cap)
{
    const int n = h->nhist < cap ? h->nhist : cap;
    if (buf) memcpy(buf, h->hist, sizeof(double) * n);
    return h->nhist;
}

ORACLE_API const char *oracle_m1_last_error(const oracle_m1 *h) { return h ? h->err : "null handle"; }

/* Test hook: closure of one state.  out[0..20] = f, fx, fy, xi, chi, Pxx, Pxy, Pyy,
 * lmin_x, lmax_x, lmin_y, lmax_y, J[3][3] (rows xx, xy, yy; columns E, Fx, Fy). */
ORACLE_API void oracle_m1_closure_point(oracle_m1 *h, double E, double Fx, double Fy, double *out)
{
    closure_t q; closure_eval(h, E, Fx, Fy, &q);
    out[0] = q.f; out[1] = q.fx; out[2] = q.fy; out[3] = q.xi; out[4] = q.chi;
    out[5] = q.P[0]; out[6] = q.P[1]; out[7] = q.P[2];
    out[8] = q.lmin[0]; out[9] = q.lmax[0]; out[10] = q.lmin[1]; out[11] = q.lmax[1];
    for (int p = 0; p < 3; ++p) for (int k = 0; k < 3; ++k) out[12 + 3 * p + k] = q.J[p][k];
}

/* Test hook: face coefficients between two states along dir.  out = a+, a-, Lambda, alpha, sigma_f. */
ORACLE_API void oracle_m1_face_point(oracle_m1 *h, const double *UL, const double *UR, int dir, double *out)
{
    cell_t L = { UL[0], UL[1], UL[2], UL[3], UL[4], 0, 0 }, R = { UR[0], UR[1], UR[2], UR[3], UR[4], 0, 0 };
    closure_t qL, qR; closure_eval(h, L.E, L.Fx, L.Fy, &qL); closure_eval(h, R.E, R.Fx, R.Fy, &qR);
    face_t fc; face_eval(h, &L, &qL, &R, &qR, dir, &fc);
    out[0] = fc.ap; out[1] = fc.am; out[2] = fc.Lam; out[3] = fc.alpha; out[4] = fc.sig;
}

ORACLE_API int oracle_m1_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
