// operator_mf.cu — matrix-free form of the implicit operator (row a6, option "operator" = 1).
//
// out = sgn * s * A [M^-1] v + add,  A = I + dt L_n in FLUX form (Eqs. 12-13 with the pressures
// replaced by J.z, see implicit_kernels.cu) evaluated from coefficient planes written by the assembly kernel:
//   per cell  : J (9), east-face and north-face coefficients (a+, Lambda, alpha, c dt sigma_f/4) (8), c dt sigma_a eta (1)
//   = 18 doubles against the 36 of the pre-multiplied block stencil; with M^-1 (9), v (3) and out (3):
//   264 B per cell per application instead of 336.
//
// Organisation = the explicit march kernel's: a block is ONE warp that owns a strip of 30 columns (+1 halo lane each side) and
// marches over the rows; a thread keeps z = M^-1 v and Pi = c^2 J z of its cell in rows j and j+1 in registers (the
// y-face flux needs no other thread; the north flux of row j is the south flux of row j+1); x-faces go through warp
// shuffles: take (z, Pi_xx, Pi_xy) of the east lane, compute the EAST flux, hand it to the east lane as its WEST flux.
// No shared memory, no barrier: the kernel is a latency-bound stream (ncu: 75 % of the stall samples wait for global loads),
// and many small independent blocks keep more loads in flight than a few 128-thread blocks that meet at two barriers per row
// (128 / 64 / 32 columns at 4096^2: 5.82 / 6.21 / 6.51 TB/s on the same box).
#include <string.h>
#include "krylov_device.cuh"
#include "explicit_device.cuh"

namespace ark {

static constexpr int TXO = 32;         // one warp per block: the x-face exchange is done by warp shuffles, no barrier
static constexpr int OP_RY = 32;       // rows per block (cap)
static constexpr int OP_MINB = 24;     // resident blocks per SM asked of ptxas (80 registers): 32 rows x 16 / 20 / 24 blocks: 5.96 / 6.45 / 6.51 TB/s;
                                       // 28 and 32 blocks spill (5.4-5.7); 48-256 rows: 6.15-6.48

struct ZP { double zE, zFx, zFy, Pxx, Pxy, Pyy, v0, v1, v2; };   // z = [M^-1] v, c^2 J z and the raw input v of one cell
struct FC { double ap, Lam, alpha, sw; };            // face coefficients; sw = c dt sigma_f / 4

// Linear flux through one face (normal component n, tangential t); same algebra as the explicit kernel.
#define ARK_LIN_FLUX(fc, EL, ER, FnL, FnR, FtL, FtR, PnL, PnR, PtL, PtR, G0, Gn, Gt, S)               \
    do {                                                                                             \
        const double dFn_ = (FnR) - (FnL);                                                           \
        G0 = (fc).alpha * fma((fc).Lam, (ER) - (EL), fma(-(fc).ap, dFn_, (FnR)));                    \
        Gn = fma((fc).Lam, dFn_, fma((fc).ap, (PnL) - (PnR), (PnR)));                                \
        Gt = fma((fc).Lam, (FtR) - (FtL), fma((fc).ap, (PtL) - (PtR), (PtR)));                       \
        S = (fc).sw * ((FnL) + (FnR));                                                               \
    } while (0)

// z and Pi of the cell in column (xmode, ii) and row j (j may be -1 or ny).  Dirichlet ghosts carry z = 0 (their
// contribution is in b), outflow ghosts copy the adjacent cell, periodic ghosts wrap (R9).
// Halo ghosts (BC_HALO, slab decomposition) carry the neighbour rank's (z, c^2 J z), packed by halo_pack_zp_kernel and exchanged
// before the launch: halo[0] = row below the slab, halo[1] = row above, six lines of nx doubles each.
template <bool PRECOND, typename TIN>
__device__ __forceinline__ ZP load_zp(const Grid& g, long long N, const TIN* __restrict__ v, const double* __restrict__ Minv,
                                      const double* __restrict__ J, double c2, int xmode, int ii, int j,
                                      const double* __restrict__ halo_lo, const double* __restrict__ halo_hi)
{
    ZP r; r.zE = 0.0; r.zFx = 0.0; r.zFy = 0.0; r.Pxx = 0.0; r.Pxy = 0.0; r.Pyy = 0.0; r.v0 = 0.0; r.v1 = 0.0; r.v2 = 0.0;
    if (xmode != 0) return r;
    int jj = j;
    if (j < 0 || j >= g.ny) {
        const int bc = g.bc[(j < 0) ? YLO : YHI];
        if (bc == BC_DIRICHLET) return r;
        if (bc == BC_HALO) {
            const double* hz = (j < 0) ? halo_lo : halo_hi;
            r.zE = hz[ii]; r.zFx = hz[g.nx + ii]; r.zFy = hz[2 * g.nx + ii];
            r.Pxx = hz[3 * g.nx + ii]; r.Pxy = hz[4 * g.nx + ii]; r.Pyy = hz[5 * g.nx + ii];
            return r;
        }
        jj = (bc == BC_PERIODIC) ? ((j < 0) ? g.ny - 1 : 0) : ((j < 0) ? 0 : g.ny - 1);
    }
    const long long id = (long long)jj * g.nx + ii;
    const double v0 = (double)v[id], v1 = (double)v[N + id], v2 = (double)v[2 * N + id];
    r.v0 = v0; r.v1 = v1; r.v2 = v2;
    if (PRECOND) {
        r.zE  = Minv[0 * N + id] * v0 + Minv[1 * N + id] * v1 + Minv[2 * N + id] * v2;
        r.zFx = Minv[3 * N + id] * v0 + Minv[4 * N + id] * v1 + Minv[5 * N + id] * v2;
        r.zFy = Minv[6 * N + id] * v0 + Minv[7 * N + id] * v1 + Minv[8 * N + id] * v2;
    } else { r.zE = v0; r.zFx = v1; r.zFy = v2; }
    r.Pxx = c2 * (J[0 * N + id] * r.zE + J[1 * N + id] * r.zFx + J[2 * N + id] * r.zFy);
    r.Pxy = c2 * (J[3 * N + id] * r.zE + J[4 * N + id] * r.zFx + J[5 * N + id] * r.zFy);
    r.Pyy = c2 * (J[6 * N + id] * r.zE + J[7 * N + id] * r.zFx + J[8 * N + id] * r.zFy);
    return r;
}

__device__ __forceinline__ FC load_fc(const double* __restrict__ p, long long stride, long long k)
{
    FC f; f.ap = p[k]; f.Lam = p[stride + k]; f.alpha = p[2 * stride + k]; f.sw = p[3 * stride + k];
    return f;
}

struct ZPub { double zE, zFx, zFy, Pxx, Pxy; };

// DOT (BiCGStab fusions, saving the separate reduction passes): 0 none; 1: <out, aux> -> epilogue BICG_ALPHA;
// 2: <out, v>, <out, out> -> epilogue BICG_OMEGA (v = the kernel's own input, already in registers).
// TIN = float: the input vector is a single-precision (compressed) Krylov basis vector (krylov_cb.cu); all arithmetic is fp64.
template <bool PRECOND, int DOT, typename TIN = double>
__global__ void __launch_bounds__(TXO, DOT ? 16 : OP_MINB) op_mf_kernel(Grid g, MfPlanes mf, const double* __restrict__ Minv, const TIN* __restrict__ v,
                                                    double* __restrict__ out, const double* __restrict__ scale_ptr,
                                                    const double* __restrict__ add, double sgn, const int* __restrict__ skip_flag,
                                                    int RY, double rx, double ry, double c2, const double* __restrict__ aux, GmresWork W, double theta)
{
    if (skip_flag && *skip_flag) return;
    double acc[2] = { 0.0, 0.0 };
    const int t = threadIdx.x;
    const int i = blockIdx.x * (TXO - 2) - 1 + t;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    const long long N = (long long)g.nx * g.ny;
    const bool upd = (t >= 1 && t <= TXO - 2 && i >= 0 && i < g.nx);
    // column resolution: 0 = grid column ii, 1 = Dirichlet ghost (z = 0), 2 = inactive
    int xmode = 0, ii = i;
    bool use_xlo = false;
    if (i > g.nx) xmode = 2;
    else if (i < 0 || i >= g.nx) {
        const int bc = g.bc[(i < 0) ? XLO : XHI];
        if (bc == BC_DIRICHLET) { xmode = 1; ii = 0; }
        else if (bc == BC_PERIODIC) ii = (i < 0) ? g.nx - 1 : 0;
        else ii = (i < 0) ? 0 : g.nx - 1;
        use_xlo = (i < 0) && (bc != BC_PERIODIC);
    }
    const bool east_valid = (i < g.nx) && (xmode != 2);    // this thread owns the face between columns i and i+1
    const double sc = sgn * (scale_ptr ? *scale_ptr : 1.0);

    ZP zS = load_zp<PRECOND, TIN>(g, N, v, Minv, mf.J, c2, xmode, ii, j0 - 1, mf.halo[0], mf.halo[1]);
    ZP zC = load_zp<PRECOND, TIN>(g, N, v, Minv, mf.J, c2, xmode, ii, j0, mf.halo[0], mf.halo[1]);
    double Hs0 = 0.0, Hs1 = 0.0, Hs2 = 0.0, Ss = 0.0;
    if (upd) {
        // south face of row j0: the north face of row j0-1, or the stored low-side line / the wrapped last row
        FC fs;
        if (j0 > 0) fs = load_fc(mf.fN, N, (long long)(j0 - 1) * g.nx + i);
        else if (g.bc[YLO] == BC_PERIODIC) fs = load_fc(mf.fN, N, (long long)(g.ny - 1) * g.nx + i);
        else fs = load_fc(mf.ylo, g.nx, i);
        ARK_LIN_FLUX(fs, zS.zE, zC.zE, zS.zFy, zC.zFy, zS.zFx, zC.zFx, zS.Pyy, zC.Pyy, zS.Pxy, zC.Pxy, Hs0, Hs2, Hs1, Ss);
    }

    for (int j = j0; j < j1; ++j) {
        // issue every global load of this row first (north cell, face coefficients, source weights); they are consumed
        // after the two barriers of the x-face exchange, which needs only data already in registers
        const ZP zN = load_zp<PRECOND, TIN>(g, N, v, Minv, mf.J, c2, xmode, ii, j + 1, mf.halo[0], mf.halo[1]);
        const long long id = (long long)j * g.nx + (upd ? i : 0);
        FC fn; fn.ap = 0.5; fn.Lam = 0.0; fn.alpha = 1.0; fn.sw = 0.0;
        double dE = 0.0, dF = 0.0, a0 = 0.0, a1 = 0.0, a2 = 0.0;
        if (upd) {
            fn = load_fc(mf.fN, N, id);
            dE = mf.dE[id]; dF = mf.dF[id];
            if (add) { a0 = add[id]; a1 = add[N + id]; a2 = add[2 * N + id]; }
        }
        double x0 = 0.0, x1 = 0.0, x2 = 0.0;
        if (DOT == 1 && upd) { x0 = aux[id]; x1 = aux[N + id]; x2 = aux[2 * N + id]; }
        FC fe; fe.ap = 0.5; fe.Lam = 0.0; fe.alpha = 1.0; fe.sw = 0.0;
        if (east_valid) {
            if (use_xlo || xmode == 1) { if (i < 0) fe = load_fc(mf.xlo, g.ny, j); }
            else fe = load_fc(mf.fE, N, (long long)j * g.nx + ii);
        }
        // x-face exchange inside the warp: lane t takes the x-face data of lane t+1, computes its EAST flux, and hands it to
        // lane t+1 as that lane's WEST flux
        ZPub me; me.zE = zC.zE; me.zFx = zC.zFx; me.zFy = zC.zFy; me.Pxx = zC.Pxx; me.Pxy = zC.Pxy;
        double Ge0, Ge1, Ge2, Se;
        {
            ZPub R;
            R.zE = __shfl_down_sync(0xffffffffu, me.zE, 1); R.zFx = __shfl_down_sync(0xffffffffu, me.zFx, 1); R.zFy = __shfl_down_sync(0xffffffffu, me.zFy, 1);
            R.Pxx = __shfl_down_sync(0xffffffffu, me.Pxx, 1); R.Pxy = __shfl_down_sync(0xffffffffu, me.Pxy, 1);
            ARK_LIN_FLUX(fe, me.zE, R.zE, me.zFx, R.zFx, me.zFy, R.zFy, me.Pxx, R.Pxx, me.Pxy, R.Pxy, Ge0, Ge1, Ge2, Se);
        }
        const double Gw0 = __shfl_up_sync(0xffffffffu, Ge0, 1), Gw1 = __shfl_up_sync(0xffffffffu, Ge1, 1);
        const double Gw2 = __shfl_up_sync(0xffffffffu, Ge2, 1), Sw = __shfl_up_sync(0xffffffffu, Se, 1);
        // north face (own column)
        double Hn0, Hn1, Hn2, Sn;
        ARK_LIN_FLUX(fn, zC.zE, zN.zE, zC.zFy, zN.zFy, zC.zFx, zN.zFx, zC.Pyy, zN.Pyy, zC.Pxy, zN.Pxy, Hn0, Hn2, Hn1, Sn);
        if (upd) {
            double o0 = zC.zE  + fma(rx, Ge0 - Gw0, fma(ry, Hn0 - Hs0, dE * zC.zE));
            double o1 = zC.zFx + fma(rx, Ge1 - Gw1, fma(ry, Hn1 - Hs1, fma(dF, zC.zFx, Se + Sw)));
            double o2 = zC.zFy + fma(rx, Ge2 - Gw2, fma(ry, Hn2 - Hs2, fma(dF, zC.zFy, Sn + Ss)));
            o0 = fma(sc, o0, a0); o1 = fma(sc, o1, a1); o2 = fma(sc, o2, a2);
            o0 = fma(-theta, zC.v0, o0); o1 = fma(-theta, zC.v1, o1); o2 = fma(-theta, zC.v2, o2);     // shifted operator (s-step basis)
            out[id] = o0; out[N + id] = o1; out[2 * N + id] = o2;
            if (DOT == 1) acc[0] += o0 * x0 + o1 * x1 + o2 * x2;
            if (DOT == 2) { acc[0] += o0 * zC.v0 + o1 * zC.v1 + o2 * zC.v2; acc[1] += o0 * o0 + o1 * o1 + o2 * o2; }
        }
        zC = zN;
        Hs0 = Hn0; Hs1 = Hn1; Hs2 = Hn2; Ss = Sn;
    }
    if (DOT == 1) reduce_and_finish<2, TXO>(acc, W, BICG_ALPHA, 0);
    if (DOT == 2) reduce_and_finish<2, TXO>(acc, W, BICG_OMEGA, 0);
}

// ---------------------------------------------------------------------------------------------------------
// The same operator WITHOUT the M^-1 planes (MfPlanes::rc, option "op_recompute", the default): the diagonal block of
// A = I + dt L_n is the coefficient of z_C in the flux form below, i.e. a function of the cell's J, its four faces' coefficients
// and dE (dF) — all of which this kernel loads anyway — so z = M^-1 v is obtained by building M and solving the 3 x 3 system
// in registers (76 fp64 instructions per cell) instead of loading nine more planes: 192 B per cell per application instead
// of 264.  The kernel waits for HBM (85 % of the stall samples), the arithmetic is free.
//   m00 = 1 + dE - rx (al_e L_e + al_w L_w) - ry (al_n L_n + al_s L_s)      m01 = rx (al_e a+_e - al_w a-_w)      m02 = ry (al_n a+_n - al_s a-_s)
//   rows 1, 2 = (1 + dF - rx (L_e + L_w) - ry (L_n + L_s) + source weights) e_k + c^2 [rx (a+_e - a-_w) J^{x.} + ry (a+_n - a-_s) J^{y.}]
// (assemble_march.cu's add_G terms, a- = 1 - a+).  Faces of the row AHEAD (j+1) are loaded in step j — east and north from the
// cell's own planes, west from the west lane's east face (lane 0 loads it), south = the current row's north face — and kept
// as the current row's faces of step j+1.  Cells whose diagonal block holds folded neighbours (outflow sides, R9), ghost
// rows and the two prologue rows of a block take z from the stored M^-1 as before (assembly still writes it: combine needs it).
// ---------------------------------------------------------------------------------------------------------
struct JC { double xx0, xx1, xx2, xy0, xy1, xy2, yy0, yy1, yy2; };

__device__ __forceinline__ void solve_diag(const FC& e, const FC& w, const FC& n, const FC& s, const JC& J, double dE, double dF,
                                           double rx, double ry, double c2, double v0, double v1, double v2,
                                           double& zE, double& zFx, double& zFy)
{
    const double lam = fma(rx, e.Lam + w.Lam, ry * (n.Lam + s.Lam));
    const double m00 = (1.0 + dE) - fma(rx, fma(e.alpha, e.Lam, w.alpha * w.Lam), ry * fma(n.alpha, n.Lam, s.alpha * s.Lam));
    const double m01 = rx * fma(e.alpha, e.ap, w.alpha * (w.ap - 1.0));
    const double m02 = ry * fma(n.alpha, n.ap, s.alpha * (s.ap - 1.0));
    const double ax = (c2 * rx) * ((e.ap + w.ap) - 1.0), ay = (c2 * ry) * ((n.ap + s.ap) - 1.0);
    const double dd = (1.0 + dF) - lam;
    const double m10 = fma(ax, J.xx0, ay * J.xy0), m11 = fma(ax, J.xx1, fma(ay, J.xy1, dd + (e.sw + w.sw))), m12 = fma(ax, J.xx2, ay * J.xy2);
    const double m20 = fma(ax, J.xy0, ay * J.yy0), m21 = fma(ax, J.xy1, ay * J.yy1), m22 = fma(ax, J.xy2, fma(ay, J.yy2, dd + (n.sw + s.sw)));
    const double c00 = m11 * m22 - m12 * m21, c01 = m12 * m20 - m10 * m22, c02 = m10 * m21 - m11 * m20;
    const double id = rcp_fast(m00 * c00 + m01 * c01 + m02 * c02);
    zE  = (c00 * v0 + (m02 * m21 - m01 * m22) * v1 + (m01 * m12 - m02 * m11) * v2) * id;
    zFx = (c01 * v0 + (m00 * m22 - m02 * m20) * v1 + (m02 * m10 - m00 * m12) * v2) * id;
    zFy = (c02 * v0 + (m01 * m20 - m00 * m21) * v1 + (m00 * m11 - m01 * m10) * v2) * id;
}

// The pressure Jacobian of the M1 closure from the reduced flux (closure_eval's formulas, m1_device.cuh; |f| <= 1, not clamped):
// with it the operator loads (fx, fy) instead of the nine J planes, 192 -> 136 B per cell per application.
__device__ __forceinline__ void jac_from_f(double fx, double fy, double ic, JC& J)
{
    const double f2 = fma(fx, fx, fy * fy);
    const double s = fma(-3.0, f2, 4.0);                  // xi^2 >= 1
    const double ixi = rsqrt_fast(s), xi = s * ixi;
    const double q3 = 3.0 * rcp_fast(2.0 + xi);           // (3 chi - 1)/(2 f^2) = 3/(2 + xi)
    const double iso = 0.33333333333333333333 * (xi - 1.0);   // (1 - chi)/2 with chi = (5 - 2 xi)/3
    const double qx = q3 * fx, qy = q3 * fy;
    const double Dxx = fma(qx, fx, iso), Dxy = qx * fy, Dyy = fma(qy, fy, iso);
    const double t3 = q3 * q3 * ixi;
    const double txx = t3 * fx * fx, txy = t3 * fx * fy, tyy = t3 * fy * fy, fxi = fx * ixi, fyi = fy * ixi;
    J.xx0 = fma(f2 - 3.0 * fx * fx, ixi, Dxx); J.xy0 = fma(-3.0 * fx * fy, ixi, Dxy); J.yy0 = fma(f2 - 3.0 * fy * fy, ixi, Dyy);
    J.xx1 = ic * (fma(txx, fx, 2.0 * qx) - fxi); J.xx2 = ic * fma(txx, fy, -fyi);
    J.xy1 = ic * fma(txy, fx, qy);               J.xy2 = ic * fma(txy, fy, qx);
    J.yy1 = ic * fma(tyy, fx, -fxi);             J.yy2 = ic * (fma(tyy, fy, 2.0 * qy) - fyi);
}

// 12 resident blocks per SM (160 registers) and 64 rows per block (the two prologue rows of a block take z from the stored M^-1):
// 16 blocks x 32 rows 0.630 ms, 16 x 64 0.618, 12 x 32 0.578, 12 x 64 0.573, 10 x 64 0.574, 20 x 32 (spills) 1.10 at 4096^2.
static constexpr int OP_RC_MINB = 12;
static constexpr int OP_RCJ_MINB = 14;    // with J rebuilt too (128 registers, 7 KB ring): 10 / 12 / 13 / 14 / 15 / 16 blocks: 0.508 / 0.506 / 0.482 / 0.473 / 0.487 / 0.486 ms;
                                          // rows per block 44 / 59 / 96 / 128: 0.471 / 0.474 / 0.480 / 0.498; a third ring stage 0.516
static constexpr int OP_RC_RY = 64;
static constexpr int RC_NST = 2;          // ring stages: row j+1 landed, row j+2 in flight during step j
// ring fields per cell: J (9) — or, when J is rebuilt too, the reduced flux (2) —, east face (4), north face (4), dE, v (3)
__host__ __device__ constexpr int rc_nj(bool jrc) { return jrc ? 2 : 9; }
__host__ __device__ constexpr int rc_nf(bool jrc) { return rc_nj(jrc) + 12; }

// The row after the row ahead travels HBM -> shared memory with cp.async while the block works (the explicit kernel's ring):
// a warp's row step is one long dependent chain (loads -> block -> 3 x 3 solve -> c^2 J z -> fluxes -> store), and with the loads
// issued at the start of the step that consumes them the kernel ran at 4.1 TB/s (0.79 ms, slower than loading M^-1).  Each thread
// reads back only its own slots, so cp.async.wait_group is the only synchronisation.
// Measured and not kept: a third ring stage (0.57 -> 0.91 ms: cp.async.ca holds an L1 line per request in flight and the shared-
// memory carve-out leaves too few); the same ring filled by 1-D bulk copies (cp.async.bulk + mbarrier, one 272-byte copy per plane
// row: ptxas serialises the 21 copies of a row in an ELECT loop, 0.61 / 0.63 / 0.71 ms with 2 / 3 / 4 stages); a branch-free row
// step for interior strips (0.570 against 0.574).
template <bool JRC, typename TIN>
__device__ __forceinline__ void rc_issue(double (*ring)[TXO], double* ringw, int t, const MfPlanes& mf, const TIN* __restrict__ v,
                                         long long N, long long idn, bool want)
{
    constexpr int NJ = rc_nj(JRC);
    if (want) {
        if (JRC) { cp_async8(&ring[0][t], mf.fxy + idn); cp_async8(&ring[1][t], mf.fxy + N + idn); }
        else {
#pragma unroll
            for (int e = 0; e < 9; ++e) cp_async8(&ring[e][t], mf.J + e * N + idn);
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) { cp_async8(&ring[NJ + e][t], mf.fE + e * N + idn); cp_async8(&ring[NJ + 4 + e][t], mf.fN + e * N + idn); }
        cp_async8(&ring[NJ + 8][t], mf.dE + idn);
        if (sizeof(TIN) == 8) {
#pragma unroll
            for (int e = 0; e < 3; ++e) cp_async8(&ring[NJ + 9 + e][t], reinterpret_cast<const double*>(v) + e * N + idn);
        } else {
#pragma unroll
            for (int e = 0; e < 3; ++e) {
                const unsigned int d = (unsigned int)__cvta_generic_to_shared(&ring[NJ + 9 + e][t]);
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(d), "l"(v + e * N + idn) : "memory");
            }
        }
        if (t == 0) {
#pragma unroll
            for (int e = 0; e < 4; ++e) cp_async8(&ringw[e], mf.fE + e * N + idn - 1);
        }
    }
    cp_async_commit();
}

// State a block carries from row to row: z and c^2 J z of the current row, the south flux, the current row's own faces and
// source weights.
struct RcState { ZP zC; double Hs0, Hs1, Hs2, Ss; FC fe, fn; double dE, dF; };

// Second half of a row step: east flux with the east lane's data, west flux from the west lane, north flux with the row ahead,
// the output of row j; then the row ahead becomes the current row.
template <int DOT>
__device__ __forceinline__ void rc_current_row(RcState& S, const ZP& zN, const FC& feN, const FC& fnN, double dEN, double dFN, bool upd,
                                               long long id, long long N, const double* __restrict__ add, const double* __restrict__ aux,
                                               double* __restrict__ out, double rx, double ry, double sc, double theta, double (&acc)[2])
{
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    if (upd && add) { a0 = add[id]; a1 = add[N + id]; a2 = add[2 * N + id]; }
    double x0 = 0.0, x1 = 0.0, x2 = 0.0;
    if (DOT == 1 && upd) { x0 = aux[id]; x1 = aux[N + id]; x2 = aux[2 * N + id]; }
    const ZP& zC = S.zC;
    ZPub me; me.zE = zC.zE; me.zFx = zC.zFx; me.zFy = zC.zFy; me.Pxx = zC.Pxx; me.Pxy = zC.Pxy;
    double Ge0, Ge1, Ge2, Se;
    {
        ZPub R;
        R.zE = __shfl_down_sync(0xffffffffu, me.zE, 1); R.zFx = __shfl_down_sync(0xffffffffu, me.zFx, 1); R.zFy = __shfl_down_sync(0xffffffffu, me.zFy, 1);
        R.Pxx = __shfl_down_sync(0xffffffffu, me.Pxx, 1); R.Pxy = __shfl_down_sync(0xffffffffu, me.Pxy, 1);
        ARK_LIN_FLUX(S.fe, me.zE, R.zE, me.zFx, R.zFx, me.zFy, R.zFy, me.Pxx, R.Pxx, me.Pxy, R.Pxy, Ge0, Ge1, Ge2, Se);
    }
    const double Gw0 = __shfl_up_sync(0xffffffffu, Ge0, 1), Gw1 = __shfl_up_sync(0xffffffffu, Ge1, 1);
    const double Gw2 = __shfl_up_sync(0xffffffffu, Ge2, 1), Sw = __shfl_up_sync(0xffffffffu, Se, 1);
    double Hn0, Hn1, Hn2, Sn;
    ARK_LIN_FLUX(S.fn, zC.zE, zN.zE, zC.zFy, zN.zFy, zC.zFx, zN.zFx, zC.Pyy, zN.Pyy, zC.Pxy, zN.Pxy, Hn0, Hn2, Hn1, Sn);
    if (upd) {
        double o0 = zC.zE  + fma(rx, Ge0 - Gw0, fma(ry, Hn0 - S.Hs0, S.dE * zC.zE));
        double o1 = zC.zFx + fma(rx, Ge1 - Gw1, fma(ry, Hn1 - S.Hs1, fma(S.dF, zC.zFx, Se + Sw)));
        double o2 = zC.zFy + fma(rx, Ge2 - Gw2, fma(ry, Hn2 - S.Hs2, fma(S.dF, zC.zFy, Sn + S.Ss)));
        o0 = fma(sc, o0, a0); o1 = fma(sc, o1, a1); o2 = fma(sc, o2, a2);
        o0 = fma(-theta, zC.v0, o0); o1 = fma(-theta, zC.v1, o1); o2 = fma(-theta, zC.v2, o2);     // shifted operator (s-step basis)
        out[id] = o0; out[N + id] = o1; out[2 * N + id] = o2;
        if (DOT == 1) acc[0] += o0 * x0 + o1 * x1 + o2 * x2;
        if (DOT == 2) { acc[0] += o0 * zC.v0 + o1 * zC.v1 + o2 * zC.v2; acc[1] += o0 * o0 + o1 * o1 + o2 * o2; }
    }
    S.zC = zN;
    S.Hs0 = Hn0; S.Hs1 = Hn1; S.Hs2 = Hn2; S.Ss = Sn;
    S.fe = feN; S.fn = fnN; S.dE = dEN; S.dF = dFN;
}

template <int DOT, typename TIN = double, bool JRC = false>
__global__ void __launch_bounds__(TXO, JRC ? OP_RCJ_MINB : OP_RC_MINB) op_mf_rc_kernel(Grid g, MfPlanes mf, const double* __restrict__ Minv, const TIN* __restrict__ v,
                                                    double* __restrict__ out, const double* __restrict__ scale_ptr,
                                                    const double* __restrict__ add, double sgn, const int* __restrict__ skip_flag,
                                                    int RY, double rx, double ry, double c2, const double* __restrict__ aux, GmresWork W, double theta)
{
    if (skip_flag && *skip_flag) return;
    constexpr int NJ = rc_nj(JRC), RC_NF = rc_nf(JRC);
    __shared__ double ring[RC_NST][RC_NF][TXO];     // row r lives in ring[r % RC_NST]
    __shared__ double ringw[RC_NST][4];             // lane 0: the east face of the column west of the strip
    double acc[2] = { 0.0, 0.0 };
    const int t = threadIdx.x;
    const int i = blockIdx.x * (TXO - 2) - 1 + t;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    const long long N = (long long)g.nx * g.ny;
    const bool upd = (t >= 1 && t <= TXO - 2 && i >= 0 && i < g.nx);
    int xmode = 0, ii = i;
    bool use_xlo = false;
    if (i > g.nx) xmode = 2;
    else if (i < 0 || i >= g.nx) {
        const int bc = g.bc[(i < 0) ? XLO : XHI];
        if (bc == BC_DIRICHLET) { xmode = 1; ii = 0; }
        else if (bc == BC_PERIODIC) ii = (i < 0) ? g.nx - 1 : 0;
        else ii = (i < 0) ? 0 : g.nx - 1;
        use_xlo = (i < 0) && (bc != BC_PERIODIC);
    }
    const bool east_valid = (i < g.nx) && (xmode != 2);
    // this lane's column has a plain diagonal block (no folded neighbour) and, for lane 0, a west column to take the west face from
    const bool col_ok = xmode == 0 && g.nx >= 2 && g.ny >= 2 && !(ii == 0 && g.bc[XLO] == BC_OUTFLOW) && !(ii == g.nx - 1 && g.bc[XHI] == BC_OUTFLOW)
                        && (t > 0 || ii >= 1);
    const int last_ok = (g.bc[YHI] == BC_OUTFLOW) ? g.ny - 2 : g.ny - 1;      // last row whose block is built here (block-uniform)
    const double sc = sgn * (scale_ptr ? *scale_ptr : 1.0);
    const bool has_dF = mf.has_dF != 0;
    const double ic = 1.0 / g.c;

    const int last_row = min(j1, last_ok);      // last row requested into the ring
    // request rows j0+1 .. j0+RC_NST-1 first: row j0+1 is consumed by the first row step
#pragma unroll
    for (int r = 1; r < RC_NST; ++r)
        rc_issue<JRC, TIN>(ring[(j0 + r) % RC_NST], ringw[(j0 + r) % RC_NST], t, mf, v, N, (long long)(j0 + r) * g.nx + ii, col_ok && j0 + r <= last_row);

    RcState S;
    {
        const ZP zS = load_zp<true, TIN>(g, N, v, Minv, mf.J, c2, xmode, ii, j0 - 1, mf.halo[0], mf.halo[1]);
        S.zC = load_zp<true, TIN>(g, N, v, Minv, mf.J, c2, xmode, ii, j0, mf.halo[0], mf.halo[1]);
        S.Hs0 = 0.0; S.Hs1 = 0.0; S.Hs2 = 0.0; S.Ss = 0.0;
        if (upd) {
            FC fs;
            if (j0 > 0) fs = load_fc(mf.fN, N, (long long)(j0 - 1) * g.nx + i);
            else if (g.bc[YLO] == BC_PERIODIC) fs = load_fc(mf.fN, N, (long long)(g.ny - 1) * g.nx + i);
            else fs = load_fc(mf.ylo, g.nx, i);
            ARK_LIN_FLUX(fs, zS.zE, S.zC.zE, zS.zFy, S.zC.zFy, zS.zFx, S.zC.zFx, zS.Pyy, S.zC.Pyy, zS.Pxy, S.zC.Pxy, S.Hs0, S.Hs2, S.Hs1, S.Ss);
        }
    }
    // faces and source weights of the current row (row j0 here; afterwards handed over from the row ahead)
    S.fe.ap = 0.5; S.fe.Lam = 0.0; S.fe.alpha = 1.0; S.fe.sw = 0.0;
    S.fn = S.fe;
    S.dE = 0.0; S.dF = 0.0;
    if (east_valid || col_ok) {
        if (use_xlo || xmode == 1) { if (i < 0) S.fe = load_fc(mf.xlo, g.ny, j0); }
        else S.fe = load_fc(mf.fE, N, (long long)j0 * g.nx + ii);
    }
    if (xmode == 0) {
        const long long id0 = (long long)j0 * g.nx + ii;
        S.fn = load_fc(mf.fN, N, id0);
        S.dE = mf.dE[id0];
        if (has_dF) S.dF = mf.dF[id0];
    }

    for (int j = j0; j < j1; ++j) {
        const int jn = j + 1;
        const long long id = (long long)j * g.nx + (upd ? i : 0);
        // ---- request row j+RC_NST into the slot of row j (read one step ago), then wait for row j+1
        rc_issue<JRC, TIN>(ring[j % RC_NST], ringw[j % RC_NST], t, mf, v, N, (long long)(j + RC_NST) * g.nx + ii, col_ok && j + RC_NST <= last_row);
        cp_async_wait<RC_NST - 1>();
        double (*rg)[TXO] = ring[jn % RC_NST];
        // ---- the row ahead: its faces, then z = M^-1 v either from the block built here or from the stored inverse
        FC feN; feN.ap = 0.5; feN.Lam = 0.0; feN.alpha = 1.0; feN.sw = 0.0;
        FC fnN = feN;
        double dEN = 0.0, dFN = 0.0;
        ZP zN;
        const bool row_in = jn < g.ny;                 // block-uniform
        const bool row_ok = jn <= last_ok;             // block-uniform
        const bool ringed = row_ok && col_ok;
        if (ringed) {
            feN.ap = rg[NJ][t]; feN.Lam = rg[NJ + 1][t]; feN.alpha = rg[NJ + 2][t]; feN.sw = rg[NJ + 3][t];
            fnN.ap = rg[NJ + 4][t]; fnN.Lam = rg[NJ + 5][t]; fnN.alpha = rg[NJ + 6][t]; fnN.sw = rg[NJ + 7][t];
            dEN = rg[NJ + 8][t];
            if (has_dF) dFN = mf.dF[(long long)jn * g.nx + ii];
        } else if (row_in) {
            if (east_valid || col_ok) {
                if (use_xlo || xmode == 1) { if (i < 0) feN = load_fc(mf.xlo, g.ny, jn); }
                else feN = load_fc(mf.fE, N, (long long)jn * g.nx + ii);
            }
            if (xmode == 0) {
                const long long idn = (long long)jn * g.nx + ii;
                fnN = load_fc(mf.fN, N, idn);
                dEN = mf.dE[idn];
                if (has_dF) dFN = mf.dF[idn];
            }
        }
        if (row_ok) {
            FC fwN;
            fwN.ap = __shfl_up_sync(0xffffffffu, feN.ap, 1); fwN.Lam = __shfl_up_sync(0xffffffffu, feN.Lam, 1);
            fwN.alpha = __shfl_up_sync(0xffffffffu, feN.alpha, 1); fwN.sw = __shfl_up_sync(0xffffffffu, feN.sw, 1);
            if (col_ok) {
                if (t == 0) { const double* rw = ringw[jn % RC_NST]; fwN.ap = rw[0]; fwN.Lam = rw[1]; fwN.alpha = rw[2]; fwN.sw = rw[3]; }
                JC J;
                if (JRC) {
                    const double fx = rg[0][t], fy = rg[1][t];
                    if (fx > 2.0) {      // clamped cell: its J is not the M1 closure's; take the stored one
                        const long long idn = (long long)jn * g.nx + ii;
                        J.xx0 = mf.J[0 * N + idn]; J.xx1 = mf.J[1 * N + idn]; J.xx2 = mf.J[2 * N + idn];
                        J.xy0 = mf.J[3 * N + idn]; J.xy1 = mf.J[4 * N + idn]; J.xy2 = mf.J[5 * N + idn];
                        J.yy0 = mf.J[6 * N + idn]; J.yy1 = mf.J[7 * N + idn]; J.yy2 = mf.J[8 * N + idn];
                    } else jac_from_f(fx, fy, ic, J);
                } else {
                    J.xx0 = rg[0][t]; J.xx1 = rg[1][t]; J.xx2 = rg[2][t]; J.xy0 = rg[3][t]; J.xy1 = rg[4][t]; J.xy2 = rg[5][t];
                    J.yy0 = rg[6][t]; J.yy1 = rg[7][t]; J.yy2 = rg[8][t];
                }
                if (sizeof(TIN) == 8) { zN.v0 = rg[NJ + 9][t]; zN.v1 = rg[NJ + 10][t]; zN.v2 = rg[NJ + 11][t]; }
                else {
                    zN.v0 = (double)*reinterpret_cast<const float*>(&rg[NJ + 9][t]); zN.v1 = (double)*reinterpret_cast<const float*>(&rg[NJ + 10][t]);
                    zN.v2 = (double)*reinterpret_cast<const float*>(&rg[NJ + 11][t]);
                }
                solve_diag(feN, fwN, fnN, S.fn, J, dEN, dFN, rx, ry, c2, zN.v0, zN.v1, zN.v2, zN.zE, zN.zFx, zN.zFy);
                zN.Pxx = c2 * (J.xx0 * zN.zE + J.xx1 * zN.zFx + J.xx2 * zN.zFy);
                zN.Pxy = c2 * (J.xy0 * zN.zE + J.xy1 * zN.zFx + J.xy2 * zN.zFy);
                zN.Pyy = c2 * (J.yy0 * zN.zE + J.yy1 * zN.zFx + J.yy2 * zN.zFy);
            } else zN = load_zp<true, TIN>(g, N, v, Minv, mf.J, c2, xmode, ii, jn, mf.halo[0], mf.halo[1]);
        } else zN = load_zp<true, TIN>(g, N, v, Minv, mf.J, c2, xmode, ii, jn, mf.halo[0], mf.halo[1]);
        rc_current_row<DOT>(S, zN, feN, fnN, dEN, dFN, upd, id, N, add, aux, out, rx, ry, sc, theta, acc);
    }
    cp_async_wait<0>();
    if (DOT == 1) reduce_and_finish<2, TXO>(acc, W, BICG_ALPHA, 0);
    if (DOT == 2) reduce_and_finish<2, TXO>(acc, W, BICG_OMEGA, 0);
}

// ---------------------------------------------------------------------------------------------------------
// TWO applications in one pass: out1 = s A^ v - th1 v, out2 = A^ out1 - th2 out1 (A^ = A M^-1) — the matrix-powers kernel of the
// s-step Arnoldi block (krylov_sstep.cu), which applies A^ five times in a row.  The rebuild of J and of the 3 x 3 block is ~130 of
// the operator's ~200 fp64 instructions per cell and the coefficient planes are 88 of its 136 B: both are paid ONCE for the two
// applications here (the inverse block is formed explicitly, adj(M) / det, and kept with J for one row step), 160 B per cell
// per pair instead of 272.  The second application trails the first by one row: with row j+1 built, the first application emits
// o1(j); z2(j) = M^-1(j) o1(j) and the second emits o2(j-1) from z2(j-2..j).  A strip is 28 columns (+2 halo lanes each side: o1 is
// valid on lanes 1..30, o2 on 2..29) and a block marches rows j0-1 .. j1 for the first application (rows j0-1 and j1 belong to the
// neighbours and are not stored).  rc2_body is the code for blocks that see real rows and columns only (every block of a grid
// periodic on all four sides: every column and row has a plain diagonal block, ghosts wrap); blocks that touch a Dirichlet or
// outflow side run rc2g_body further down; halo rows of a slab, op_recompute < 2 and grids under 4 x 4 take two single applications.
// ---------------------------------------------------------------------------------------------------------
// 8 resident one-warp blocks per SM (two per sub-partition, 240-255 registers, no spills).  Measured on the bench solve at 4096^2 (58 operator
// launches, 34 of them pairs, against 94 single applications at 49.2 ms): 8 blocks 38.1 ms; 12 blocks (168 registers, 216 B of spills)
// 53.6; 16 blocks 60.0; the inverse block and J parked in shared memory between the two row steps (218 registers) 39.4; rows per
// block 32 / 64 / 128: 39.4 / 38.1 / 37.9; a third ring stage 38.3.  A pair costs 0.75 ms against 2 x 0.52.
static constexpr int OP2_MINB = 8;
static constexpr int OP2_NST = 2;
static constexpr int OP2_RY = 64;
static constexpr int OP2_W = TXO - 4;

__device__ __forceinline__ void build_inv(const FC& e, const FC& w, const FC& n, const FC& s, const JC& J, double dE, double dF,
                                          double rx, double ry, double c2, double (&I)[9])
{
    const double lam = fma(rx, e.Lam + w.Lam, ry * (n.Lam + s.Lam));
    const double m00 = (1.0 + dE) - fma(rx, fma(e.alpha, e.Lam, w.alpha * w.Lam), ry * fma(n.alpha, n.Lam, s.alpha * s.Lam));
    const double m01 = rx * fma(e.alpha, e.ap, w.alpha * (w.ap - 1.0));
    const double m02 = ry * fma(n.alpha, n.ap, s.alpha * (s.ap - 1.0));
    const double ax = (c2 * rx) * ((e.ap + w.ap) - 1.0), ay = (c2 * ry) * ((n.ap + s.ap) - 1.0);
    const double dd = (1.0 + dF) - lam;
    const double m10 = fma(ax, J.xx0, ay * J.xy0), m11 = fma(ax, J.xx1, fma(ay, J.xy1, dd + (e.sw + w.sw))), m12 = fma(ax, J.xx2, ay * J.xy2);
    const double m20 = fma(ax, J.xy0, ay * J.yy0), m21 = fma(ax, J.xy1, ay * J.yy1), m22 = fma(ax, J.xy2, fma(ay, J.yy2, dd + (n.sw + s.sw)));
    const double c00 = m11 * m22 - m12 * m21, c01 = m12 * m20 - m10 * m22, c02 = m10 * m21 - m11 * m20;
    const double id = rcp_fast(m00 * c00 + m01 * c01 + m02 * c02);
    I[0] = c00 * id; I[1] = (m02 * m21 - m01 * m22) * id; I[2] = (m01 * m12 - m02 * m11) * id;
    I[3] = c01 * id; I[4] = (m00 * m22 - m02 * m20) * id; I[5] = (m02 * m10 - m00 * m12) * id;
    I[6] = c02 * id; I[7] = (m01 * m20 - m00 * m21) * id; I[8] = (m00 * m11 - m01 * m10) * id;
}

// z = I v, Pi = c^2 J z of one cell
__device__ __forceinline__ void zp_from(const double (&I)[9], const JC& J, double c2, double v0, double v1, double v2, ZP& z)
{
    z.v0 = v0; z.v1 = v1; z.v2 = v2;
    z.zE  = fma(I[0], v0, fma(I[1], v1, I[2] * v2));
    z.zFx = fma(I[3], v0, fma(I[4], v1, I[5] * v2));
    z.zFy = fma(I[6], v0, fma(I[7], v1, I[8] * v2));
    z.Pxx = c2 * (J.xx0 * z.zE + J.xx1 * z.zFx + J.xx2 * z.zFy);
    z.Pxy = c2 * (J.xy0 * z.zE + J.xy1 * z.zFx + J.xy2 * z.zFy);
    z.Pyy = c2 * (J.yy0 * z.zE + J.yy1 * z.zFx + J.yy2 * z.zFy);
}

// one row of one application (rc_current_row without the fusions): o = s (A z)(row of S) - theta v, then the row ahead becomes S's row
__device__ __forceinline__ void rc2_row(RcState& S, const ZP& zN, const FC& feN, const FC& fnN, double dEN, double dFN,
                                        double rx, double ry, double sc, double theta, double& o0, double& o1, double& o2)
{
    const ZP& zC = S.zC;
    double Ge0, Ge1, Ge2, Se;
    {
        const double RzE = __shfl_down_sync(0xffffffffu, zC.zE, 1), RzFx = __shfl_down_sync(0xffffffffu, zC.zFx, 1), RzFy = __shfl_down_sync(0xffffffffu, zC.zFy, 1);
        const double RPxx = __shfl_down_sync(0xffffffffu, zC.Pxx, 1), RPxy = __shfl_down_sync(0xffffffffu, zC.Pxy, 1);
        ARK_LIN_FLUX(S.fe, zC.zE, RzE, zC.zFx, RzFx, zC.zFy, RzFy, zC.Pxx, RPxx, zC.Pxy, RPxy, Ge0, Ge1, Ge2, Se);
    }
    const double Gw0 = __shfl_up_sync(0xffffffffu, Ge0, 1), Gw1 = __shfl_up_sync(0xffffffffu, Ge1, 1);
    const double Gw2 = __shfl_up_sync(0xffffffffu, Ge2, 1), Sw = __shfl_up_sync(0xffffffffu, Se, 1);
    double Hn0, Hn1, Hn2, Sn;
    ARK_LIN_FLUX(S.fn, zC.zE, zN.zE, zC.zFy, zN.zFy, zC.zFx, zN.zFx, zC.Pyy, zN.Pyy, zC.Pxy, zN.Pxy, Hn0, Hn2, Hn1, Sn);
    o0 = zC.zE  + fma(rx, Ge0 - Gw0, fma(ry, Hn0 - S.Hs0, S.dE * zC.zE));
    o1 = zC.zFx + fma(rx, Ge1 - Gw1, fma(ry, Hn1 - S.Hs1, fma(S.dF, zC.zFx, Se + Sw)));
    o2 = zC.zFy + fma(rx, Ge2 - Gw2, fma(ry, Hn2 - S.Hs2, fma(S.dF, zC.zFy, Sn + S.Ss)));
    o0 = fma(-theta, zC.v0, sc * o0); o1 = fma(-theta, zC.v1, sc * o1); o2 = fma(-theta, zC.v2, sc * o2);
    S.zC = zN;
    S.Hs0 = Hn0; S.Hs1 = Hn1; S.Hs2 = Hn2; S.Ss = Sn;
    S.fe = feN; S.fn = fnN; S.dE = dEN; S.dF = dFN;
}

__device__ __forceinline__ void rc2_issue(double (*ring)[TXO], double* ringw, int t, const MfPlanes& mf, const double* __restrict__ v,
                                          long long N, long long idn, long long idw, bool want)
{
    if (want) {
        cp_async8(&ring[0][t], mf.fxy + idn); cp_async8(&ring[1][t], mf.fxy + N + idn);
#pragma unroll
        for (int e = 0; e < 4; ++e) { cp_async8(&ring[2 + e][t], mf.fE + e * N + idn); cp_async8(&ring[6 + e][t], mf.fN + e * N + idn); }
        cp_async8(&ring[10][t], mf.dE + idn);
#pragma unroll
        for (int e = 0; e < 3; ++e) cp_async8(&ring[11 + e][t], v + e * N + idn);
        if (t == 0) {
#pragma unroll
            for (int e = 0; e < 4; ++e) cp_async8(&ringw[e], mf.fE + e * N + idw);
        }
    }
    cp_async_commit();
}

__device__ __forceinline__ void load_jc(const double* __restrict__ Jp, long long N, long long id, JC& J)
{
    J.xx0 = Jp[0 * N + id]; J.xx1 = Jp[1 * N + id]; J.xx2 = Jp[2 * N + id];
    J.xy0 = Jp[3 * N + id]; J.xy1 = Jp[4 * N + id]; J.xy2 = Jp[5 * N + id];
    J.yy0 = Jp[6 * N + id]; J.yy1 = Jp[7 * N + id]; J.yy2 = Jp[8 * N + id];
}

// Grids with Dirichlet or outflow sides: blocks that touch a boundary (first strip, last two strips — the last but one can hold the ghost
// lane of column nx —, first block row, last two block rows) go through op_mf_rc2g_kernel below; every other block sees real rows and
// columns only and runs this kernel's periodic code unchanged (0.75 against 0.99 ms per pair at 4096^2 for the general code).
__device__ __forceinline__ bool op2_edge_block(const Grid& g, int bx, int by, int SX, int SY)
{
    return (g.bc[YLO] != BC_PERIODIC && (by == 0 || by >= SY - 2)) || (g.bc[XLO] != BC_PERIODIC && (bx == 0 || bx >= SX - 2));
}

__device__ __forceinline__ void rc2_body(const Grid& g, const MfPlanes& mf, const double* __restrict__ Minv, const double* __restrict__ v,
                                         double* __restrict__ out1, double* __restrict__ out2, const double* __restrict__ scale_ptr,
                                         int RY, double rx, double ry, double c2, double th1, double th2)
{
    __shared__ double ring[OP2_NST][14][TXO];        // row-ahead number q lives in ring[q % OP2_NST]: (fx, fy), east face, north face, dE, v
    __shared__ double ringw[OP2_NST][4];             // lane 0: the east face of the column west of the strip
    const int t = threadIdx.x, nx = g.nx, ny = g.ny;
    const int i = blockIdx.x * OP2_W - 2 + t;
    const int ii = ((i % nx) + nx) % nx;
    const int iw = (ii == 0) ? nx - 1 : ii - 1;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, ny);
    const long long N = (long long)nx * ny;
    const bool st_lane = (t >= 2 && t <= TXO - 3 && i >= 0 && i < nx);
    const double sc = scale_ptr ? *scale_ptr : 1.0;
    const bool has_dF = mf.has_dF != 0;
    const double ic = 1.0 / g.c;
    const int qlast = j1 + 1 - j0;                  // rows ahead j0 .. j1+1 (wrapped)
#define ARK_WR(j) ((j) < 0 ? (j) + ny : ((j) >= ny ? (j) - ny : (j)))
#pragma unroll
    for (int r = 0; r < OP2_NST - 1; ++r) {
        const int rr = ARK_WR(j0 + r);
        rc2_issue(ring[r], ringw[r], t, mf, v, N, (long long)rr * nx + ii, (long long)rr * nx + iw, r <= qlast);
    }

    // first application: rows j0-2 (south of the first marched row) and j0-1 from the stored inverse
    const int rS = ARK_WR(j0 - 2), rC = ARK_WR(j0 - 1);
    const long long idC = (long long)rC * nx + ii;
    RcState S1, S2;
    {
        const ZP zS = load_zp<true, double>(g, N, v, Minv, mf.J, c2, 0, ii, rS, nullptr, nullptr);
        S1.zC = load_zp<true, double>(g, N, v, Minv, mf.J, c2, 0, ii, rC, nullptr, nullptr);
        const FC fs = load_fc(mf.fN, N, (long long)rS * nx + ii);
        ARK_LIN_FLUX(fs, zS.zE, S1.zC.zE, zS.zFy, S1.zC.zFy, zS.zFx, S1.zC.zFx, zS.Pyy, S1.zC.Pyy, zS.Pxy, S1.zC.Pxy, S1.Hs0, S1.Hs2, S1.Hs1, S1.Ss);
    }
    S1.fe = load_fc(mf.fE, N, idC);
    S1.fn = load_fc(mf.fN, N, idC);
    S1.dE = mf.dE[idC];
    S1.dF = has_dF ? mf.dF[idC] : 0.0;
    // inverse block and J of the current row of the first application (row j0-1: stored; afterwards handed over from the row ahead)
    double IC[9];
    JC Jc;
#pragma unroll
    for (int e = 0; e < 9; ++e) IC[e] = Minv[e * N + idC];
    load_jc(mf.J, N, idC, Jc);
    S2 = S1;       // (overwritten at q = 0)

    for (int q = 0; q <= qlast; ++q) {
        const int jm = j0 - 1 + q;
        const int rn = ARK_WR(jm + 1);
        {
            const int qa = q + OP2_NST - 1, r2 = ARK_WR(j0 + qa);       // the slot read one step ago
            rc2_issue(ring[qa % OP2_NST], ringw[qa % OP2_NST], t, mf, v, N, (long long)r2 * nx + ii, (long long)r2 * nx + iw, qa <= qlast);
        }
        cp_async_wait<OP2_NST - 1>();
        double (*rg)[TXO] = ring[q % OP2_NST];
        // ---- the row ahead: faces, J, inverse block, z1 = M^-1 v
        const long long idn = (long long)rn * nx + ii;
        FC feN, fnN, fwN;
        feN.ap = rg[2][t]; feN.Lam = rg[3][t]; feN.alpha = rg[4][t]; feN.sw = rg[5][t];
        fnN.ap = rg[6][t]; fnN.Lam = rg[7][t]; fnN.alpha = rg[8][t]; fnN.sw = rg[9][t];
        const double dEN = rg[10][t];
        const double dFN = has_dF ? mf.dF[idn] : 0.0;
        fwN.ap = __shfl_up_sync(0xffffffffu, feN.ap, 1); fwN.Lam = __shfl_up_sync(0xffffffffu, feN.Lam, 1);
        fwN.alpha = __shfl_up_sync(0xffffffffu, feN.alpha, 1); fwN.sw = __shfl_up_sync(0xffffffffu, feN.sw, 1);
        if (t == 0) { const double* rw = ringw[q % OP2_NST]; fwN.ap = rw[0]; fwN.Lam = rw[1]; fwN.alpha = rw[2]; fwN.sw = rw[3]; }
        JC Jn;
        {
            const double fx = rg[0][t], fy = rg[1][t];
            if (fx > 2.0) load_jc(mf.J, N, idn, Jn);      // clamped cell: the stored J
            else jac_from_f(fx, fy, ic, Jn);
        }
        double IN[9];
        build_inv(feN, fwN, fnN, S1.fn, Jn, dEN, dFN, rx, ry, c2, IN);
        ZP zN;
        zp_from(IN, Jn, c2, rg[11][t], rg[12][t], rg[13][t], zN);
        // ---- first application, row jm
        const FC fe1 = S1.fe, fn1 = S1.fn;
        const double dE1 = S1.dE, dF1 = S1.dF;
        double o0, o1, o2;
        rc2_row(S1, zN, feN, fnN, dEN, dFN, rx, ry, sc, th1, o0, o1, o2);
        if (st_lane && q >= 1 && jm < j1) {
            const long long id = (long long)jm * nx + i;
            out1[id] = o0; out1[N + id] = o1; out1[2 * N + id] = o2;
        }
        // ---- second application: z2 of row jm, then row jm-1
        ZP y;
        zp_from(IC, Jc, c2, o0, o1, o2, y);
        if (q >= 1) {
            double p0, p1, p2;
            rc2_row(S2, y, fe1, fn1, dE1, dF1, rx, ry, 1.0, th2, p0, p1, p2);
            if (st_lane && q >= 2) {
                const long long id = (long long)(jm - 1) * nx + i;
                out2[id] = p0; out2[N + id] = p1; out2[2 * N + id] = p2;
            }
        } else {
            S2.zC = y; S2.Hs0 = 0.0; S2.Hs1 = 0.0; S2.Hs2 = 0.0; S2.Ss = 0.0;
            S2.fe = fe1; S2.fn = fn1; S2.dE = dE1; S2.dF = dF1;
        }
#pragma unroll
        for (int e = 0; e < 9; ++e) IC[e] = IN[e];
        Jc = Jn;
    }
    cp_async_wait<0>();
#undef ARK_WR
}

// ---------------------------------------------------------------------------------------------------------
// The two-application kernel for grids with Dirichlet or outflow sides (any mix with periodic ones).  Same march; what the
// boundaries add:
//   columns  ghost lanes (i = -1, nx) carry z = 0 (Dirichlet) or a copy of the adjacent lane's (z, Pi) (outflow) in BOTH applications
//            (their own o1 is not a stencil result); the copy is a shuffle, done in the two edge strips only.  The west face of
//            column 0 is the boundary face of mf.xlo.  An outflow boundary column holds a folded neighbour in its diagonal block:
//            its inverse block and J come from the stored planes (as in the one-application kernel), for both applications.
//   rows     a block that starts at row 0 marches the first application from row 0 (ghost row -1 = 0 or a copy of row 0, south face
//            from mf.ylo) and starts the second with the ghost of ITS vector: z2(-1) = 0 or z2(0).  A block that ends at row ny-1
//            takes the ghost row ny as the row ahead of the first application, and one more step of the second with z2(ny) = 0 or
//            z2(ny-1).  An outflow top row uses the stored inverse.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void zp_zero(ZP& z)
{
    z.zE = 0.0; z.zFx = 0.0; z.zFy = 0.0; z.Pxx = 0.0; z.Pxy = 0.0; z.Pyy = 0.0; z.v0 = 0.0; z.v1 = 0.0; z.v2 = 0.0;
}

// lane kinds: 0 cell, 1 cell with a folded diagonal block, 2 zero ghost / inactive, 3 copy of lane t+1, 4 copy of lane t-1
__device__ __forceinline__ void fix_ghost(ZP& z, int kind)
{
    ZP a, b;
    a.zE = __shfl_down_sync(0xffffffffu, z.zE, 1); a.zFx = __shfl_down_sync(0xffffffffu, z.zFx, 1); a.zFy = __shfl_down_sync(0xffffffffu, z.zFy, 1);
    a.Pxx = __shfl_down_sync(0xffffffffu, z.Pxx, 1); a.Pxy = __shfl_down_sync(0xffffffffu, z.Pxy, 1); a.Pyy = __shfl_down_sync(0xffffffffu, z.Pyy, 1);
    b.zE = __shfl_up_sync(0xffffffffu, z.zE, 1); b.zFx = __shfl_up_sync(0xffffffffu, z.zFx, 1); b.zFy = __shfl_up_sync(0xffffffffu, z.zFy, 1);
    b.Pxx = __shfl_up_sync(0xffffffffu, z.Pxx, 1); b.Pxy = __shfl_up_sync(0xffffffffu, z.Pxy, 1); b.Pyy = __shfl_up_sync(0xffffffffu, z.Pyy, 1);
    if (kind == 2) zp_zero(z);
    else if (kind == 3) { z.zE = a.zE; z.zFx = a.zFx; z.zFy = a.zFy; z.Pxx = a.Pxx; z.Pxy = a.Pxy; z.Pyy = a.Pyy; }
    else if (kind == 4) { z.zE = b.zE; z.zFx = b.zFx; z.zFy = b.zFy; z.Pxx = b.Pxx; z.Pxy = b.Pxy; z.Pyy = b.Pyy; }
}

#define ARK_YFLUX(fc, zL, zR, H0, H1, H2, Sv) \
    ARK_LIN_FLUX(fc, (zL).zE, (zR).zE, (zL).zFy, (zR).zFy, (zL).zFx, (zR).zFx, (zL).Pyy, (zR).Pyy, (zL).Pxy, (zR).Pxy, H0, H2, H1, Sv)

__device__ __forceinline__ void rc2g_body(const Grid& g, const MfPlanes& mf, const double* __restrict__ Minv, const double* __restrict__ v,
                                          double* __restrict__ out1, double* __restrict__ out2, const double* __restrict__ scale_ptr,
                                          int RY, double rx, double ry, double c2, double th1, double th2)
{
    __shared__ double ring[OP2_NST][14][TXO];
    __shared__ double ringw[OP2_NST][4];
    const int t = threadIdx.x, nx = g.nx, ny = g.ny;
    const int i = blockIdx.x * OP2_W - 2 + t;
    const bool perx = g.bc[XLO] == BC_PERIODIC, pery = g.bc[YLO] == BC_PERIODIC;
    int ii, kind;
    if (perx) { ii = ((i % nx) + nx) % nx; kind = 0; }
    else if (i >= 0 && i < nx) { ii = i; kind = ((i == 0 && g.bc[XLO] == BC_OUTFLOW) || (i == nx - 1 && g.bc[XHI] == BC_OUTFLOW)) ? 1 : 0; }
    else if (i == -1) { ii = 0; kind = (g.bc[XLO] == BC_DIRICHLET) ? 2 : 3; }
    else if (i == nx) { ii = nx - 1; kind = (g.bc[XHI] == BC_DIRICHLET) ? 2 : 4; }
    else { ii = (i < 0) ? 0 : nx - 1; kind = 2; }
    const bool edge = __any_sync(0xffffffffu, kind >= 2);          // (warp-uniform) this strip holds ghost lanes
    const bool lghost = (!perx && i == -1);                        // its east face is the boundary face of mf.xlo
    const int iw = (ii == 0) ? (perx ? nx - 1 : 0) : ii - 1;       // column of lane 0's west face (lane 0 is never column 0 of a non-periodic grid)
    const int lxm = (kind <= 1) ? 0 : 1;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, ny);
    const long long N = (long long)nx * ny;
    const bool st_lane = (t >= 2 && t <= TXO - 3 && i >= 0 && i < nx);
    const double sc = scale_ptr ? *scale_ptr : 1.0;
    const bool has_dF = mf.has_dF != 0;
    const double ic = 1.0 / g.c;
    const int jmA = pery ? j0 - 1 : (j0 > 0 ? j0 - 1 : 0);         // rows marched by the first application: jmA .. jmB
    const int jmB = pery ? j1 : (j1 < ny ? j1 : ny - 1);
    const int nsteps = jmB - jmA + 1;
#define ARK_WR(j) ((j) < 0 ? (j) + ny : ((j) >= ny ? (j) - ny : (j)))
#define ARK_REAL(j) (pery || ((j) >= 0 && (j) < ny))
#pragma unroll
    for (int r = 0; r < OP2_NST - 1; ++r) {
        const int jr = jmA + 1 + r, rr = ARK_WR(jr);
        rc2_issue(ring[r], ringw[r], t, mf, v, N, (long long)rr * nx + ii, (long long)rr * nx + iw, r < nsteps && ARK_REAL(jr));
    }

    // ---- prologue of the first application: the row south of the first marched row, and that row, from the stored inverse
    RcState S1, S2;
    const int rA = ARK_WR(jmA);
    const long long idA = (long long)rA * nx + ii;
    {
        // (a ghost row -1 is resolved by load_zp: zero, or the copy of row 0)
        ZP zS = load_zp<true, double>(g, N, v, Minv, mf.J, c2, lxm, ii, pery ? ARK_WR(jmA - 1) : jmA - 1, nullptr, nullptr);
        S1.zC = load_zp<true, double>(g, N, v, Minv, mf.J, c2, lxm, ii, rA, nullptr, nullptr);
        if (edge) { fix_ghost(zS, kind); fix_ghost(S1.zC, kind); }
        const FC fs = (pery || jmA > 0) ? load_fc(mf.fN, N, (long long)ARK_WR(jmA - 1) * nx + ii) : load_fc(mf.ylo, nx, ii);
        ARK_YFLUX(fs, zS, S1.zC, S1.Hs0, S1.Hs1, S1.Hs2, S1.Ss);
    }
    S1.fe = lghost ? load_fc(mf.xlo, ny, rA) : load_fc(mf.fE, N, idA);
    S1.fn = load_fc(mf.fN, N, idA);
    S1.dE = mf.dE[idA];
    S1.dF = has_dF ? mf.dF[idA] : 0.0;
    double IC[9];
    JC Jc;
#pragma unroll
    for (int e = 0; e < 9; ++e) IC[e] = Minv[e * N + idA];
    load_jc(mf.J, N, idA, Jc);
    S2 = S1;       // (overwritten at q = 0)
    FC fdef; fdef.ap = 0.5; fdef.Lam = 0.0; fdef.alpha = 1.0; fdef.sw = 0.0;

    for (int q = 0; q < nsteps; ++q) {
        const int jm = jmA + q, jn = jm + 1;
        const bool real_n = ARK_REAL(jn);                            // (block-uniform) false: the row ahead is the ghost row ny
        {
            const int qa = q + OP2_NST - 1, j2 = jmA + 1 + qa, r2 = ARK_WR(j2);
            rc2_issue(ring[qa % OP2_NST], ringw[qa % OP2_NST], t, mf, v, N, (long long)r2 * nx + ii, (long long)r2 * nx + iw, qa < nsteps && ARK_REAL(j2));
        }
        cp_async_wait<OP2_NST - 1>();
        double (*rg)[TXO] = ring[q % OP2_NST];
        FC feN = fdef, fnN = fdef;
        double dEN = 0.0, dFN = 0.0;
        double IN[9];
        JC Jn;
        ZP zN;
        if (real_n) {
            const int rn = ARK_WR(jn);
            const long long idn = (long long)rn * nx + ii;
            feN.ap = rg[2][t]; feN.Lam = rg[3][t]; feN.alpha = rg[4][t]; feN.sw = rg[5][t];
            fnN.ap = rg[6][t]; fnN.Lam = rg[7][t]; fnN.alpha = rg[8][t]; fnN.sw = rg[9][t];
            dEN = rg[10][t];
            if (has_dF) dFN = mf.dF[idn];
            if (lghost) feN = load_fc(mf.xlo, ny, rn);
            FC fwN;
            fwN.ap = __shfl_up_sync(0xffffffffu, feN.ap, 1); fwN.Lam = __shfl_up_sync(0xffffffffu, feN.Lam, 1);
            fwN.alpha = __shfl_up_sync(0xffffffffu, feN.alpha, 1); fwN.sw = __shfl_up_sync(0xffffffffu, feN.sw, 1);
            if (t == 0) { const double* rw = ringw[q % OP2_NST]; fwN.ap = rw[0]; fwN.Lam = rw[1]; fwN.alpha = rw[2]; fwN.sw = rw[3]; }
            // a diagonal block that holds a folded neighbour (outflow column or outflow top row): the stored inverse and J
            const bool folded = (kind == 1) || (!pery && jn == ny - 1 && g.bc[YHI] == BC_OUTFLOW);
            if (folded) {
#pragma unroll
                for (int e = 0; e < 9; ++e) IN[e] = Minv[e * N + idn];
                load_jc(mf.J, N, idn, Jn);
            } else {
                const double fx = rg[0][t], fy = rg[1][t];
                if (fx > 2.0) load_jc(mf.J, N, idn, Jn);      // clamped cell: the stored J
                else jac_from_f(fx, fy, ic, Jn);
                build_inv(feN, fwN, fnN, S1.fn, Jn, dEN, dFN, rx, ry, c2, IN);
            }
            zp_from(IN, Jn, c2, rg[11][t], rg[12][t], rg[13][t], zN);
            if (edge) fix_ghost(zN, kind);
        } else {
            if (g.bc[YHI] == BC_DIRICHLET) zp_zero(zN); else zN = S1.zC;
#pragma unroll
            for (int e = 0; e < 9; ++e) IN[e] = 0.0;
            Jn = Jc;
        }
        // ---- first application, row jm
        const FC fe1 = S1.fe, fn1 = S1.fn;
        const double dE1 = S1.dE, dF1 = S1.dF;
        double o0, o1, o2;
        rc2_row(S1, zN, feN, fnN, dEN, dFN, rx, ry, sc, th1, o0, o1, o2);
        if (st_lane && jm >= j0 && jm < j1) {
            const long long id = (long long)jm * nx + i;
            out1[id] = o0; out1[N + id] = o1; out1[2 * N + id] = o2;
        }
        // ---- second application: z2 of row jm, then row jm-1
        ZP y;
        zp_from(IC, Jc, c2, o0, o1, o2, y);
        if (edge) fix_ghost(y, kind);
        if (q == 0) {
            S2.zC = y; S2.Hs0 = 0.0; S2.Hs1 = 0.0; S2.Hs2 = 0.0; S2.Ss = 0.0;
            S2.fe = fe1; S2.fn = fn1; S2.dE = dE1; S2.dF = dF1;
            if (jmA == j0) {       // (block-uniform) row 0 of a non-periodic grid: the ghost row of the second application's vector
                ZP yg;
                if (g.bc[YLO] == BC_DIRICHLET) zp_zero(yg); else yg = y;
                const FC fs2 = load_fc(mf.ylo, nx, ii);
                ARK_YFLUX(fs2, yg, y, S2.Hs0, S2.Hs1, S2.Hs2, S2.Ss);
            }
        } else {
            double p0, p1, p2;
            rc2_row(S2, y, fe1, fn1, dE1, dF1, rx, ry, 1.0, th2, p0, p1, p2);
            if (st_lane && jm - 1 >= j0) {
                const long long id = (long long)(jm - 1) * nx + i;
                out2[id] = p0; out2[N + id] = p1; out2[2 * N + id] = p2;
            }
        }
#pragma unroll
        for (int e = 0; e < 9; ++e) IC[e] = IN[e];
        Jc = Jn;
    }
    cp_async_wait<0>();
    if (!pery && j1 == ny) {       // (block-uniform) the last row of the second application: its row ahead is the ghost row ny
        ZP yg;
        if (g.bc[YHI] == BC_DIRICHLET) zp_zero(yg); else yg = S2.zC;
        double p0, p1, p2;
        rc2_row(S2, yg, fdef, fdef, 0.0, 0.0, rx, ry, 1.0, th2, p0, p1, p2);
        if (st_lane) {
            const long long id = (long long)(ny - 1) * nx + i;
            out2[id] = p0; out2[N + id] = p1; out2[2 * N + id] = p2;
        }
    }
#undef ARK_WR
#undef ARK_REAL
}

// MODE 0: every block runs the periodic code (grids periodic on all four sides).  1: boundary blocks run the general code, the
// others the periodic code, in ONE grid (as two launches the handful of boundary blocks were a 0.15 ms tail per pair).  2: every
// block runs the general code (grids too small to have interior blocks).
template <int MODE>
__global__ void __launch_bounds__(TXO, OP2_MINB) op_mf_rc2_kernel(Grid g, MfPlanes mf, const double* __restrict__ Minv, const double* __restrict__ v,
                                                                  double* __restrict__ out1, double* __restrict__ out2,
                                                                  const double* __restrict__ scale_ptr, const int* __restrict__ skip_flag,
                                                                  int RY, double rx, double ry, double c2, double th1, double th2)
{
    if (skip_flag && *skip_flag) return;
    if (MODE == 0) rc2_body(g, mf, Minv, v, out1, out2, scale_ptr, RY, rx, ry, c2, th1, th2);
    else if (MODE == 2) rc2g_body(g, mf, Minv, v, out1, out2, scale_ptr, RY, rx, ry, c2, th1, th2);
    else if (op2_edge_block(g, blockIdx.x, blockIdx.y, gridDim.x, gridDim.y)) rc2g_body(g, mf, Minv, v, out1, out2, scale_ptr, RY, rx, ry, c2, th1, th2);
    else rc2_body(g, mf, Minv, v, out1, out2, scale_ptr, RY, rx, ry, c2, th1, th2);
}

bool op_mf2_ok(const Grid& g, const MfPlanes& mf)
{
    if ((g.ny + OP2_RY - 1) / OP2_RY > 65535) return false;      // rows of blocks on gridDim.y
    for (int s = 0; s < 4; ++s) if (g.bc[s] != BC_PERIODIC && g.bc[s] != BC_DIRICHLET && g.bc[s] != BC_OUTFLOW) return false;      // (halo rows of a slab)
    return mf.rc && mf.rcj && g.nx >= 4 && g.ny >= 4;
}

// out1 = s A M^-1 v - th1 v, out2 = A M^-1 out1 - th2 out1 in one pass (op_mf2_ok grids only)
cudaError_t launch_op_mf2(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, double* out1, double* out2,
                          const double* scale_ptr, const int* skip_flag, int sm_count, cudaStream_t st, double th1, double th2)
{
    if (!op_mf2_ok(g, mf)) return cudaErrorNotSupported;
    const int strips = (g.nx + OP2_W - 1) / OP2_W;
    long long want = ((long long)g.ny * strips + (long long)sm_count * 64 - 1) / ((long long)sm_count * 64);
    int RY = (int)(want < 8 ? 8 : (want > OP2_RY ? OP2_RY : want));
    if (RY > g.ny) RY = g.ny;
    const dim3 grd(strips, (g.ny + RY - 1) / RY);
    const bool periodic = g.bc[XLO] == BC_PERIODIC && g.bc[XHI] == BC_PERIODIC && g.bc[YLO] == BC_PERIODIC && g.bc[YHI] == BC_PERIODIC;
    const bool interior = (g.bc[XLO] == BC_PERIODIC || grd.x >= 4) && (g.bc[YLO] == BC_PERIODIC || grd.y >= 4);      // the grid has blocks that touch no boundary
    if (periodic) op_mf_rc2_kernel<0><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out1, out2, scale_ptr, skip_flag, RY, mf.rx, mf.ry, g.c * g.c, th1, th2);
    else if (interior) op_mf_rc2_kernel<1><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out1, out2, scale_ptr, skip_flag, RY, mf.rx, mf.ry, g.c * g.c, th1, th2);
    else op_mf_rc2_kernel<2><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out1, out2, scale_ptr, skip_flag, RY, mf.rx, mf.ry, g.c * g.c, th1, th2);
    return cudaGetLastError();
}

static dim3 op_mf_grid(const Grid& g, int sm_count, int* RYout, int ry_cap = OP_RY)
{
    const int strips = (g.nx + (TXO - 2) - 1) / (TXO - 2);
    long long want = ((long long)g.ny * strips + (long long)sm_count * 64 - 1) / ((long long)sm_count * 64);
    int RY = (int)(want < 4 ? 4 : (want > ry_cap ? ry_cap : want));
    if (RY > g.ny) RY = g.ny;
    *RYout = RY;
    return dim3(strips, (g.ny + RY - 1) / RY);
}

int op_mf_blocks(const Grid& g, int sm_count) { int RY; const dim3 d = op_mf_grid(g, sm_count, &RY); return (int)(d.x * d.y); }

// v_out = A M^-1 v_in fused with the BiCGStab reduction `dot` (1: alpha with aux = r^; 2: omega)
cudaError_t launch_op_mf_dot(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, double* out,
                             const int* skip_flag, int dot, const double* aux, GmresWork W, int sm_count, cudaStream_t st)
{
    int RY; const dim3 grd = op_mf_grid(g, sm_count, &RY, mf.rc ? OP_RC_RY : OP_RY);
    const double c2 = g.c * g.c;
    if (mf.rc && mf.rcj) {
        if (dot == 1) op_mf_rc_kernel<1, double, true><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W, 0.0);
        else op_mf_rc_kernel<2, double, true><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W, 0.0);
    } else if (mf.rc) {
        if (dot == 1) op_mf_rc_kernel<1><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W, 0.0);
        else op_mf_rc_kernel<2><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W, 0.0);
    }
    else if (dot == 1) op_mf_kernel<true, 1><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W, 0.0);
    else op_mf_kernel<true, 2><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W, 0.0);
    return cudaGetLastError();
}

// out = s * A M^-1 v with v stored in single precision
cudaError_t launch_op_mf_f32(const Grid& g, const MfPlanes& mf, const double* Minv, const float* v, double* out,
                             const double* scale_ptr, const int* skip_flag, int sm_count, cudaStream_t st)
{
    int RY; const dim3 grd = op_mf_grid(g, sm_count, &RY, mf.rc ? OP_RC_RY : OP_RY);
    const double c2 = g.c * g.c;
    GmresWork none; memset(&none, 0, sizeof none);
    if (mf.rc && mf.rcj) op_mf_rc_kernel<0, float, true><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none, 0.0);
    else if (mf.rc) op_mf_rc_kernel<0, float><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none, 0.0);
    else op_mf_kernel<true, 0, float><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none, 0.0);
    return cudaGetLastError();
}

// Slab decomposition: what the neighbour ranks need of this slab for one operator application — (z, c^2 J z) of the first row
// (sent to the rank below) and of the last row (sent to the rank above): out_lo, out_hi = six lines of nx doubles each.
template <bool PRECOND>
__global__ void halo_pack_zp_kernel(Grid g, const double* __restrict__ J, const double* __restrict__ Minv, const double* __restrict__ v,
                                    double c2, double* __restrict__ out_lo, double* __restrict__ out_hi, const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    const long long N = (long long)g.nx * g.ny;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < g.nx; i += gridDim.x * blockDim.x) {
        for (int side = 0; side < 2; ++side) {
            double* o = side == 0 ? out_lo : out_hi;
            if (!o) continue;
            const ZP r = load_zp<PRECOND, double>(g, N, v, Minv, J, c2, 0, i, side == 0 ? 0 : g.ny - 1, nullptr, nullptr);
            o[i] = r.zE; o[g.nx + i] = r.zFx; o[2 * g.nx + i] = r.zFy; o[3 * g.nx + i] = r.Pxx; o[4 * g.nx + i] = r.Pxy; o[5 * g.nx + i] = r.Pyy;
        }
    }
}

cudaError_t launch_halo_pack_zp(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, int precond,
                                double* out_lo, double* out_hi, const int* skip_flag, cudaStream_t st)
{
    const int blk = 128, grd = (g.nx + blk - 1) / blk;
    const double c2 = g.c * g.c;
    if (precond) halo_pack_zp_kernel<true><<<grd, blk, 0, st>>>(g, mf.J, Minv, v, c2, out_lo, out_hi, skip_flag);
    else halo_pack_zp_kernel<false><<<grd, blk, 0, st>>>(g, mf.J, Minv, v, c2, out_lo, out_hi, skip_flag);
    return cudaGetLastError();
}

cudaError_t launch_op_mf(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, double* out,
                         const double* scale_ptr, const double* add, double sgn, const int* skip_flag, int precond,
                         int sm_count, cudaStream_t st, double theta)
{
    int RY; const dim3 grd = op_mf_grid(g, sm_count, &RY, (precond && mf.rc) ? OP_RC_RY : OP_RY);
    const double c2 = g.c * g.c;
    GmresWork none; memset(&none, 0, sizeof none);
    if (precond && mf.rc && mf.rcj) op_mf_rc_kernel<0, double, true><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, add, sgn, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none, theta);
    else if (precond && mf.rc) op_mf_rc_kernel<0><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, add, sgn, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none, theta);
    else if (precond) op_mf_kernel<true, 0><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, add, sgn, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none, theta);
    else op_mf_kernel<false, 0><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, add, sgn, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none, theta);
    return cudaGetLastError();
}

}  // namespace ark
