// multigrid.cu — geometric-aggregation multigrid V-cycle as the right preconditioner of the Krylov solvers
// (pre-smoothing, restricted residual equation "R A P y = R r~", coarse solve, interpolation,
// post-smoothing; the paper takes an algebraic multigrid from a library, reading R15 fixes this one).
//
// Everything runs in the block-Jacobi-scaled ("hat") variable of the Krylov core: on level l the operator is
//   Ahat_l = A_l D_l^-1 = I + sum_k off_k(.)            (unit diagonal blocks, four scaled neighbour blocks, like the fine level)
// so the damped block-Jacobi smoother is a damped Richardson sweep  z^ += omega (r - Ahat z^)  that never touches D, and
//   coarse operator  A_{l+1} = P0^T Ahat_l P0  (2x2 aggregates, 1 wide at an odd end; again a 5-point stencil of 3x3 blocks)
//   restriction      r_{l+1} = P0^T (r - Ahat z^)
//   interpolation    z^ += P0 e_{l+1},  e_{l+1} = D_{l+1}^-1 z^_{l+1}
// (in the unscaled variable: R = P0^T, P = D^-1 P0, smoother omega D^-1 — the form the oracle is written in).
// One V-cycle from a zero initial guess with one pre- and one post-sweep costs two stencil passes per level:
//   pass 1 (restrict)      : r_c = P0^T ((1 - omega) r - omega sum_k off_k r_nbr)            reads 36 + 3 doubles per cell
//   pass 2 (prolong+smooth): t = omega r + P0 e_c;  z^ = t + omega (r - t - sum_k off_k t_nbr)   reads 36 + 3, writes 3
// The hierarchy ends at a single cell, where `coarse_sweeps` Richardson sweeps stand in for the direct solve.
#include "implicit_device.cuh"

namespace ark {

static constexpr int MG_MINB = 3;      // resident blocks per SM asked of the pair kernels: 168 registers let ptxas issue all block loads up front (measured best of 1, 3, 4, 8)
static constexpr int MG_BY = 4;        // rows of threads per block of the V-cycle kernels (32 x MG_BY threads)

// Neighbour k (0: W, 1: E, 2: S, 3: N) of cell (i, j): its index on the level and, through `agg`, its aggregate on the next
// coarser level (cnx aggregates per row).  Non-periodic sides clamp (the block there is zero).
__device__ __forceinline__ long long mg_nbr(const Grid& g, int i, int j, int k, int cnx, long long& agg)
{
    int ii = i + (k == 0 ? -1 : (k == 1 ? 1 : 0));
    int jj = j + (k == 2 ? -1 : (k == 3 ? 1 : 0));
    if (ii < 0) ii = (g.bc[XLO] == BC_PERIODIC) ? g.nx - 1 : 0;
    if (ii >= g.nx) ii = (g.bc[XHI] == BC_PERIODIC) ? 0 : g.nx - 1;
    if (jj < 0) jj = (g.bc[YLO] == BC_PERIODIC) ? g.ny - 1 : 0;
    if (jj >= g.ny) jj = (g.bc[YHI] == BC_PERIODIC) ? 0 : g.ny - 1;
    agg = (long long)(jj >> 1) * cnx + (ii >> 1);
    return (long long)jj * g.nx + ii;
}

// ---- set-up: coarse blocks of one level --------------------------------------------------------------------------
// One thread per coarse cell: D_c = sum over the aggregate of (I + blocks whose neighbour lies in the same aggregate),
// C_k = sum of the blocks that leave the aggregate in direction k.  Writes Dinv_c = D_c^-1 and the raw C_k;
// launch_scale_offdiag then turns C_k into C_k Dinv_c(neighbour k).
__global__ void __launch_bounds__(128) mg_galerkin_kernel(Grid gf, const double* __restrict__ off, Grid gc,
                                                          double* __restrict__ coff, double* __restrict__ cDinv)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    if (I >= gc.nx || J >= gc.ny) return;
    const long long N = (long long)gf.nx * gf.ny, Nc = (long long)gc.nx * gc.ny, a = (long long)J * gc.nx + I;
    Blk D, Ck[4];
    blk_zero(D);
#pragma unroll
    for (int k = 0; k < 4; ++k) blk_zero(Ck[k]);
    for (int dj = 0; dj < 2; ++dj)
        for (int di = 0; di < 2; ++di) {
            const int i = 2 * I + di, j = 2 * J + dj;
            if (i >= gf.nx || j >= gf.ny) continue;
            const long long id = (long long)j * gf.nx + i;
            D.a[0] += 1.0; D.a[4] += 1.0; D.a[8] += 1.0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                long long anb;
                mg_nbr(gf, i, j, k, gc.nx, anb);
                const bool inside = (anb == a);
#pragma unroll
                for (int e = 0; e < 9; ++e) {
                    const double v = off[(long long)(k * 9 + e) * N + id];
                    if (inside) D.a[e] += v; else Ck[k].a[e] += v;
                }
            }
        }
    Blk Di; inv3(D, Di);
#pragma unroll
    for (int e = 0; e < 9; ++e) cDinv[e * Nc + a] = Di.a[e];
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int e = 0; e < 9; ++e) coff[(long long)(k * 9 + e) * Nc + a] = Ck[k].a[e];
}

cudaError_t launch_mg_galerkin(const Grid& gf, const double* off, const Grid& gc, double* coff, double* cDinv, float* coff32, cudaStream_t st)
{
    dim3 blk(32, 4), grd((gc.nx + 31) / 32, (gc.ny + 3) / 4);
    mg_galerkin_kernel<<<grd, blk, 0, st>>>(gf, off, gc, coff, cDinv);
    if (cudaGetLastError() != cudaSuccess) return cudaErrorLaunchFailure;
    BlockMatrix C; C.off = coff; C.C = nullptr; C.Minv = cDinv; C.b = nullptr;
    return launch_scale_offdiag(gc, C, coff32, st);
}

// ---- V-cycle pass 1: r_c = P0^T ((1 - omega) r - omega sum_k off_k r_nbr) --------------------------------------------
// Thread (i, J) handles the fine cells (i, 2J) and (i, 2J+1); lane pairs (i even, i+1) add up through a shuffle.
template <typename TB>
__global__ void __launch_bounds__(32 * MG_BY) mg_restrict_kernel(Grid g, const TB* __restrict__ off, const double* __restrict__ r,
                                                          double omega, int cnx, double* __restrict__ rc,
                                                          const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const long long N = (long long)g.nx * g.ny;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    const int cny = (g.ny + 1) / 2;
    if (i < g.nx && J < cny) {
#pragma unroll
        for (int dj = 0; dj < 2; ++dj) {
            const int j = 2 * J + dj;
            if (j >= g.ny) continue;
            const long long id = (long long)j * g.nx + i;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                long long an;
                const long long nb = mg_nbr(g, i, j, k, cnx, an);
                const double x0 = r[nb], x1 = r[N + nb], x2 = r[2 * N + nb];
                const TB* a = off + (long long)(k * 9) * N + id;
                a0 += (double)a[0 * N] * x0 + (double)a[1 * N] * x1 + (double)a[2 * N] * x2;
                a1 += (double)a[3 * N] * x0 + (double)a[4 * N] * x1 + (double)a[5 * N] * x2;
                a2 += (double)a[6 * N] * x0 + (double)a[7 * N] * x1 + (double)a[8 * N] * x2;
            }
            s0 += (1.0 - omega) * r[id] - omega * a0;
            s1 += (1.0 - omega) * r[N + id] - omega * a1;
            s2 += (1.0 - omega) * r[2 * N + id] - omega * a2;
        }
    }
    s0 += __shfl_xor_sync(0xffffffffu, s0, 1); s1 += __shfl_xor_sync(0xffffffffu, s1, 1); s2 += __shfl_xor_sync(0xffffffffu, s2, 1);
    if ((i & 1) == 0 && i < g.nx && J < cny) {
        const long long Nc = (long long)cnx * cny, a = (long long)J * cnx + (i >> 1);
        rc[a] = s0; rc[Nc + a] = s1; rc[2 * Nc + a] = s2;
    }
}

// ---- V-cycle pass 2: t = omega r + P0 e_c;  z^ = t + omega (r - t - sum_k off_k t_nbr);  out = Dinv z^ (coarse levels) or z^ ----
template <typename TB>
__global__ void __launch_bounds__(32 * MG_BY) mg_prolong_smooth_kernel(Grid g, const TB* __restrict__ off, const double* __restrict__ r,
                                                                double omega, int cnx, const double* __restrict__ ec,
                                                                const double* __restrict__ Dinv, double* __restrict__ out,
                                                                const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const long long N = (long long)g.nx * g.ny, id = (long long)j * g.nx + i;
    const long long Nc = (long long)cnx * ((g.ny + 1) / 2);
    const long long a = (long long)(j >> 1) * cnx + (i >> 1);
    const double r0 = r[id], r1 = r[N + id], r2 = r[2 * N + id];
    const double t0 = omega * r0 + ec[a], t1 = omega * r1 + ec[Nc + a], t2 = omega * r2 + ec[2 * Nc + a];
    double q0 = t0, q1 = t1, q2 = t2;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        long long an;
        const long long nb = mg_nbr(g, i, j, k, cnx, an);
        const double x0 = omega * r[nb] + ec[an], x1 = omega * r[N + nb] + ec[Nc + an], x2 = omega * r[2 * N + nb] + ec[2 * Nc + an];
        const TB* b = off + (long long)(k * 9) * N + id;
        q0 += (double)b[0 * N] * x0 + (double)b[1 * N] * x1 + (double)b[2 * N] * x2;
        q1 += (double)b[3 * N] * x0 + (double)b[4 * N] * x1 + (double)b[5 * N] * x2;
        q2 += (double)b[6 * N] * x0 + (double)b[7 * N] * x1 + (double)b[8 * N] * x2;
    }
    const double z0 = t0 + omega * (r0 - q0), z1 = t1 + omega * (r1 - q1), z2 = t2 + omega * (r2 - q2);
    if (Dinv) {
        out[id]         = Dinv[0 * N + id] * z0 + Dinv[1 * N + id] * z1 + Dinv[2 * N + id] * z2;
        out[N + id]     = Dinv[3 * N + id] * z0 + Dinv[4 * N + id] * z1 + Dinv[5 * N + id] * z2;
        out[2 * N + id] = Dinv[6 * N + id] * z0 + Dinv[7 * N + id] * z1 + Dinv[8 * N + id] * z2;
    } else {
        out[id] = z0; out[N + id] = z1; out[2 * N + id] = z2;
    }
}

// ---- pair kernels: two adjacent cells (2I, 2I+1) per thread, blocks and vectors read as 2-element vectors ----------------
// Used on every level with an even nx (all levels of a power-of-two grid): half as many load instructions per byte as the
// one-cell kernels above (which remain the path for odd nx), and the restriction needs no shuffle: a thread owns a whole aggregate.
template <typename T> struct Pair2;
template <> struct Pair2<double> { typedef double2 type; };
template <> struct Pair2<float> { typedef float2 type; };

struct V3 { double e, fx, fy; };
__device__ __forceinline__ V3 ld3(const double* __restrict__ r, long long N, long long id) { V3 v; v.e = r[id]; v.fx = r[N + id]; v.fy = r[2 * N + id]; return v; }
__device__ __forceinline__ void ld3x2(const double* __restrict__ r, long long N, long long id, V3& a, V3& b)
{
    const double2 p0 = *reinterpret_cast<const double2*>(r + id), p1 = *reinterpret_cast<const double2*>(r + N + id),
                  p2 = *reinterpret_cast<const double2*>(r + 2 * N + id);
    a.e = p0.x; b.e = p0.y; a.fx = p1.x; b.fx = p1.y; a.fy = p2.x; b.fy = p2.y;
}
// acc += off_k(a) xa and off_k(b) xb for the cell pair at id (block k), one vector load per block entry
template <typename TB>
__device__ __forceinline__ void blk2_apply(const TB* __restrict__ off, long long N, long long id, int k, const V3& xa, const V3& xb,
                                           double (&qa)[3], double (&qb)[3])
{
    typedef typename Pair2<TB>::type TB2;
    const TB* base = off + (long long)(k * 9) * N + id;
#pragma unroll
    for (int row = 0; row < 3; ++row) {
        const TB2 c0 = *reinterpret_cast<const TB2*>(base + (3 * row) * N), c1 = *reinterpret_cast<const TB2*>(base + (3 * row + 1) * N),
                  c2 = *reinterpret_cast<const TB2*>(base + (3 * row + 2) * N);
        qa[row] += (double)c0.x * xa.e + (double)c1.x * xa.fx + (double)c2.x * xa.fy;
        qb[row] += (double)c0.y * xb.e + (double)c1.y * xb.fx + (double)c2.y * xb.fy;
    }
}
// column and row neighbours of the pair (2I, 2I+1) in row j: indices on the level and aggregates on the next one
struct PairNbr { long long w, e, s, n, aw, ae, as, an; };
__device__ __forceinline__ PairNbr pair_nbr(const Grid& g, int I, int j, int cnx)
{
    PairNbr p;
    int iw = 2 * I - 1, ie = 2 * I + 2, js = j - 1, jn = j + 1;
    if (iw < 0) iw = (g.bc[XLO] == BC_PERIODIC) ? g.nx - 1 : 0;
    if (ie >= g.nx) ie = (g.bc[XHI] == BC_PERIODIC) ? 0 : g.nx - 1;
    if (js < 0) js = (g.bc[YLO] == BC_PERIODIC) ? g.ny - 1 : 0;
    if (jn >= g.ny) jn = (g.bc[YHI] == BC_PERIODIC) ? 0 : g.ny - 1;
    p.w = (long long)j * g.nx + iw; p.e = (long long)j * g.nx + ie;
    p.s = (long long)js * g.nx + 2 * I; p.n = (long long)jn * g.nx + 2 * I;
    p.aw = (long long)(j >> 1) * cnx + (iw >> 1); p.ae = (long long)(j >> 1) * cnx + (ie >> 1);
    p.as = (long long)(js >> 1) * cnx + I; p.an = (long long)(jn >> 1) * cnx + I;
    return p;
}

template <typename TB>
__global__ void __launch_bounds__(128, MG_MINB) mg_restrict2_kernel(Grid g, const TB* __restrict__ off, const double* __restrict__ r,
                                                           double omega, int cnx, double* __restrict__ rc,
                                                           const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const int cny = (g.ny + 1) / 2;
    if (I >= cnx || J >= cny) return;
    const long long N = (long long)g.nx * g.ny;
    double s[3] = { 0.0, 0.0, 0.0 };
#pragma unroll
    for (int dj = 0; dj < 2; ++dj) {
        const int j = 2 * J + dj;
        if (j >= g.ny) continue;
        const long long id = (long long)j * g.nx + 2 * I;
        const PairNbr p = pair_nbr(g, I, j, cnx);
        V3 ra, rb, sa, sb, na, nb;
        ld3x2(r, N, id, ra, rb); ld3x2(r, N, p.s, sa, sb); ld3x2(r, N, p.n, na, nb);
        const V3 rw = ld3(r, N, p.w), re = ld3(r, N, p.e);
        double qa[3] = { 0.0, 0.0, 0.0 }, qb[3] = { 0.0, 0.0, 0.0 };
        blk2_apply<TB>(off, N, id, 0, rw, ra, qa, qb);      // west: of a it is the outer column, of b it is a
        blk2_apply<TB>(off, N, id, 1, rb, re, qa, qb);      // east: of a it is b, of b the outer column
        blk2_apply<TB>(off, N, id, 2, sa, sb, qa, qb);
        blk2_apply<TB>(off, N, id, 3, na, nb, qa, qb);
        s[0] += (1.0 - omega) * (ra.e + rb.e) - omega * (qa[0] + qb[0]);
        s[1] += (1.0 - omega) * (ra.fx + rb.fx) - omega * (qa[1] + qb[1]);
        s[2] += (1.0 - omega) * (ra.fy + rb.fy) - omega * (qa[2] + qb[2]);
    }
    const long long Nc = (long long)cnx * cny, a = (long long)J * cnx + I;
    rc[a] = s[0]; rc[Nc + a] = s[1]; rc[2 * Nc + a] = s[2];
}

template <typename TB>
__global__ void __launch_bounds__(128, MG_MINB) mg_prolong_smooth2_kernel(Grid g, const TB* __restrict__ off, const double* __restrict__ r,
                                                                 double omega, int cnx, const double* __restrict__ ec,
                                                                 const double* __restrict__ Dinv, double* __restrict__ out,
                                                                 const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (I >= cnx || j >= g.ny) return;
    const long long N = (long long)g.nx * g.ny, id = (long long)j * g.nx + 2 * I;
    const long long Nc = (long long)cnx * ((g.ny + 1) / 2), ag = (long long)(j >> 1) * cnx + I;
    const PairNbr p = pair_nbr(g, I, j, cnx);
    V3 ra, rb, sa, sb, na, nb;
    ld3x2(r, N, id, ra, rb); ld3x2(r, N, p.s, sa, sb); ld3x2(r, N, p.n, na, nb);
    V3 rw = ld3(r, N, p.w), re = ld3(r, N, p.e);
    const V3 e0 = ld3(ec, Nc, ag), ew = ld3(ec, Nc, p.aw), ee = ld3(ec, Nc, p.ae), es = ld3(ec, Nc, p.as), en = ld3(ec, Nc, p.an);
    // t = omega r + P0 e_c at the pair and its six neighbours
#define ARK_T(v, c) do { (v).e = fma(omega, (v).e, (c).e); (v).fx = fma(omega, (v).fx, (c).fx); (v).fy = fma(omega, (v).fy, (c).fy); } while (0)
    V3 ta = ra, tb = rb;
    ARK_T(ta, e0); ARK_T(tb, e0); ARK_T(rw, ew); ARK_T(re, ee); ARK_T(sa, es); ARK_T(sb, es); ARK_T(na, en); ARK_T(nb, en);
#undef ARK_T
    double qa[3] = { ta.e, ta.fx, ta.fy }, qb[3] = { tb.e, tb.fx, tb.fy };
    blk2_apply<TB>(off, N, id, 0, rw, ta, qa, qb);
    blk2_apply<TB>(off, N, id, 1, tb, re, qa, qb);
    blk2_apply<TB>(off, N, id, 2, sa, sb, qa, qb);
    blk2_apply<TB>(off, N, id, 3, na, nb, qa, qb);
    const double za0 = ta.e + omega * (ra.e - qa[0]), za1 = ta.fx + omega * (ra.fx - qa[1]), za2 = ta.fy + omega * (ra.fy - qa[2]);
    const double zb0 = tb.e + omega * (rb.e - qb[0]), zb1 = tb.fx + omega * (rb.fx - qb[1]), zb2 = tb.fy + omega * (rb.fy - qb[2]);
    double2 o0, o1, o2;
    if (Dinv) {
        double2 d[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) d[e] = *reinterpret_cast<const double2*>(Dinv + e * N + id);
        o0 = make_double2(d[0].x * za0 + d[1].x * za1 + d[2].x * za2, d[0].y * zb0 + d[1].y * zb1 + d[2].y * zb2);
        o1 = make_double2(d[3].x * za0 + d[4].x * za1 + d[5].x * za2, d[3].y * zb0 + d[4].y * zb1 + d[5].y * zb2);
        o2 = make_double2(d[6].x * za0 + d[7].x * za1 + d[8].x * za2, d[6].y * zb0 + d[7].y * zb1 + d[8].y * zb2);
    } else {
        o0 = make_double2(za0, zb0); o1 = make_double2(za1, zb1); o2 = make_double2(za2, zb2);
    }
    *reinterpret_cast<double2*>(out + id) = o0; *reinterpret_cast<double2*>(out + N + id) = o1; *reinterpret_cast<double2*>(out + 2 * N + id) = o2;
}

// ---- coarsest level (a single cell): z^ = omega r, then sweeps-1 times z^ += omega (r - Ahat z^);  out = Dinv z^ ----------
template <typename TB>
__global__ void mg_coarsest_kernel(Grid g, const TB* __restrict__ off, const double* __restrict__ r, double omega, int sweeps,
                                   const double* __restrict__ Dinv, double* __restrict__ out, const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double Ah[9] = { 1, 0, 0, 0, 1, 0, 0, 0, 1 };       // N = 1: every neighbour is the cell itself (or the block is zero)
    for (int k = 0; k < 4; ++k)
        for (int e = 0; e < 9; ++e) Ah[e] += (double)off[k * 9 + e];
    const double rr[3] = { r[0], r[1], r[2] };
    double z[3] = { omega * rr[0], omega * rr[1], omega * rr[2] };
    for (int s = 1; s < sweeps; ++s) {
        double q[3];
        for (int a = 0; a < 3; ++a) q[a] = Ah[3 * a] * z[0] + Ah[3 * a + 1] * z[1] + Ah[3 * a + 2] * z[2];
        for (int a = 0; a < 3; ++a) z[a] += omega * (rr[a] - q[a]);
    }
    for (int a = 0; a < 3; ++a) out[a] = Dinv ? (Dinv[3 * a] * z[0] + Dinv[3 * a + 1] * z[1] + Dinv[3 * a + 2] * z[2]) : z[a];
}

// One V-cycle: zhat_out = Mhat^-1 r_in on level 0 (both 3N planes; may not alias).  Returns the number of launches in *nl.
// TB = float reads the single-precision copies of the blocks (option "mg_precision" = 32): the cycle is still a fixed linear
// operator evaluated in fp64, only its matrix entries are rounded to 24 bits.
template <typename TB>
static cudaError_t vcycle_t(const MgHier& H, const double* r_in, double* zhat_out, const int* skip_flag, cudaStream_t st, int* nl)
{
    int launches = 0;
    const int L = H.nlev;
    auto blocks = [](const MgLevel& lv) -> const TB* {
        if (sizeof(TB) == sizeof(float)) return reinterpret_cast<const TB*>(lv.off32);
        return reinterpret_cast<const TB*>(lv.off);
    };
    for (int l = 0; l + 1 < L; ++l) {                     // downward: restricted residuals
        const MgLevel& f = H.lev[l];
        const double* r = (l == 0) ? r_in : f.r;
        if ((f.g.nx & 1) == 0) {          // pair kernel: one thread per aggregate
            const int cnx = H.lev[l + 1].g.nx, cny = H.lev[l + 1].g.ny;
            dim3 blk(32, 4), grd((cnx + 31) / 32, (cny + 3) / 4);
            mg_restrict2_kernel<TB><<<grd, blk, 0, st>>>(f.g, blocks(f), r, H.omega, cnx, H.lev[l + 1].r, skip_flag);
        } else {
            dim3 blk(32, MG_BY), grd((f.g.nx + 31) / 32, ((f.g.ny + 1) / 2 + MG_BY - 1) / MG_BY);
            mg_restrict_kernel<TB><<<grd, blk, 0, st>>>(f.g, blocks(f), r, H.omega, H.lev[l + 1].g.nx, H.lev[l + 1].r, skip_flag);
        }
        ++launches;
    }
    {
        const MgLevel& c = H.lev[L - 1];
        const double* r = (L == 1) ? r_in : c.r;
        mg_coarsest_kernel<TB><<<1, 32, 0, st>>>(c.g, blocks(c), r, H.omega, H.coarse_sweeps, (L == 1) ? nullptr : c.Dinv,
                                                 (L == 1) ? zhat_out : c.e, skip_flag);
        ++launches;
    }
    for (int l = L - 2; l >= 0; --l) {                    // upward: interpolation + post-smoothing
        const MgLevel& f = H.lev[l];
        const double* r = (l == 0) ? r_in : f.r;
        if ((f.g.nx & 1) == 0) {
            const int cnx = H.lev[l + 1].g.nx;
            dim3 blk(32, 4), grd((cnx + 31) / 32, (f.g.ny + 3) / 4);
            mg_prolong_smooth2_kernel<TB><<<grd, blk, 0, st>>>(f.g, blocks(f), r, H.omega, cnx, H.lev[l + 1].e,
                                                               (l == 0) ? nullptr : f.Dinv, (l == 0) ? zhat_out : f.e, skip_flag);
        } else {
            dim3 blk(32, MG_BY), grd((f.g.nx + 31) / 32, (f.g.ny + MG_BY - 1) / MG_BY);
            mg_prolong_smooth_kernel<TB><<<grd, blk, 0, st>>>(f.g, blocks(f), r, H.omega, H.lev[l + 1].g.nx, H.lev[l + 1].e,
                                                              (l == 0) ? nullptr : f.Dinv, (l == 0) ? zhat_out : f.e, skip_flag);
        }
        ++launches;
    }
    if (nl) *nl = launches;
    return cudaGetLastError();
}

cudaError_t launch_mg_vcycle(const MgHier& H, const double* r_in, double* zhat_out, const int* skip_flag, cudaStream_t st, int* nl)
{
    return H.precision == 32 ? vcycle_t<float>(H, r_in, zhat_out, skip_flag, st, nl)
                             : vcycle_t<double>(H, r_in, zhat_out, skip_flag, st, nl);
}

// single-precision copy of a level's scaled blocks
__global__ void mg_to_float_kernel(const double* __restrict__ a, float* __restrict__ b, long long n)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) b[k] = (float)a[k];
}

cudaError_t launch_mg_to_float(const double* a, float* b, long long n, cudaStream_t st)
{
    const long long need = (n + 255) / 256;
    mg_to_float_kernel<<<(int)(need < current_sm_count() * 16 ? need : current_sm_count() * 16), 256, 0, st>>>(a, b, n);
    return cudaGetLastError();
}

}  // namespace ark
