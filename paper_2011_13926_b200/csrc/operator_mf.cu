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
                                                    int RY, double rx, double ry, double c2, const double* __restrict__ aux, GmresWork W)
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

static dim3 op_mf_grid(const Grid& g, int sm_count, int* RYout)
{
    const int strips = (g.nx + (TXO - 2) - 1) / (TXO - 2);
    long long want = ((long long)g.ny * strips + (long long)sm_count * 64 - 1) / ((long long)sm_count * 64);
    int RY = (int)(want < 4 ? 4 : (want > OP_RY ? OP_RY : want));
    if (RY > g.ny) RY = g.ny;
    *RYout = RY;
    return dim3(strips, (g.ny + RY - 1) / RY);
}

int op_mf_blocks(const Grid& g, int sm_count) { int RY; const dim3 d = op_mf_grid(g, sm_count, &RY); return (int)(d.x * d.y); }

// v_out = A M^-1 v_in fused with the BiCGStab reduction `dot` (1: alpha with aux = r^; 2: omega)
cudaError_t launch_op_mf_dot(const Grid& g, const MfPlanes& mf, const double* Minv, const double* v, double* out,
                             const int* skip_flag, int dot, const double* aux, GmresWork W, int sm_count, cudaStream_t st)
{
    int RY; const dim3 grd = op_mf_grid(g, sm_count, &RY);
    const double c2 = g.c * g.c;
    if (dot == 1) op_mf_kernel<true, 1><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W);
    else op_mf_kernel<true, 2><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, nullptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, aux, W);
    return cudaGetLastError();
}

// out = s * A M^-1 v with v stored in single precision
cudaError_t launch_op_mf_f32(const Grid& g, const MfPlanes& mf, const double* Minv, const float* v, double* out,
                             const double* scale_ptr, const int* skip_flag, int sm_count, cudaStream_t st)
{
    int RY; const dim3 grd = op_mf_grid(g, sm_count, &RY);
    const double c2 = g.c * g.c;
    GmresWork none; memset(&none, 0, sizeof none);
    op_mf_kernel<true, 0, float><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, nullptr, 1.0, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none);
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
                         int sm_count, cudaStream_t st)
{
    int RY; const dim3 grd = op_mf_grid(g, sm_count, &RY);
    const double c2 = g.c * g.c;
    GmresWork none; memset(&none, 0, sizeof none);
    if (precond) op_mf_kernel<true, 0><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, add, sgn, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none);
    else op_mf_kernel<false, 0><<<grd, TXO, 0, st>>>(g, mf, Minv, v, out, scale_ptr, add, sgn, skip_flag, RY, mf.rx, mf.ry, c2, nullptr, none);
    return cudaGetLastError();
}

}  // namespace ark
