// implicit_kernels.cu — row a5 (assembly of the linearised system, the paper's "matrix update")
// and the block-stencil operator of row a6.
//
// System (PAPER.md:263 Newton linearisation, one per step):
//     (I + dt L_n) U^{n+1} = U^n + affine terms,
// L_n = the flux-difference + source operator of Eq. 12 with the pressures P_ab(U) replaced by J_ab . U
// (analytic pressure Jacobian at U^n; P is homogeneous of degree 1 so J.U^n = P(U^n)) and the face coefficients
// a+-, Lambda, alpha, sigma_f frozen at t^n.
//
// Every face flux is linear in its two cell states, G = GL v_L + GR v_R with 3x3 matrices
//     GL = [ -alpha Lam , alpha a+ e_n ;  c^2 a+ J^{n.}(L) - Lam I_F ],   GR = [ alpha Lam , alpha a- e_n ;  c^2 a- J^{n.}(R) + Lam I_F ]
// (J^{n.} = rows (xx, xy) of J for an x-face, (xy, yy) for a y-face), so the five 3x3 blocks of a cell row are
//     C = I + rx (GL_e - GR_w) + ry (GL_n - GR_s) + dt S_C,  E = rx GR_e + dt S_E,  W = -rx GL_w + dt S_W,  N, S likewise,
// with S_* the WB source weights c sigma_f/4 (Eqs. 18-19; PAPER.md:677-679 fixes the 1/4) and c sigma_a eta on (E,E).
//
// Storage: structure-of-arrays planes (one plane of N doubles per block entry) so that every load is coalesced;
// the structured 5-point graph needs no index arrays ("the graph is fixed").
// Right preconditioning is folded into the stored operator: off-diagonal planes hold
// A_k M_k^-1 (M = diagonal blocks, Eq. 27 block-wise), the diagonal block of A M^-1 is the identity.
#include "implicit_device.cuh"

namespace ark {

// Tile assembly: a block owns ATX x ATY cells.  Phase 1 evaluates closure + pressure Jacobian ONCE per cell of the tile and
// of its one-cell halo (corners excluded) into shared memory; phase 2 builds the five blocks of each cell from the five
// shared entries.  (The first version evaluated five closures per cell: 3.5 ms at 4096^2; fast reciprocals: 2.4 ms.)
static constexpr int ATX = 32, ATY = 4, AW = ATX + 2, AH = ATY + 2, ACELLS = AW * AH;
enum { TC_E = 0, TC_FX, TC_FY, TC_SA, TC_ST, TC_F, TC_LMINX, TC_LMAXX, TC_LMINY, TC_LMAXY, TC_J0, TC_FIELDS = TC_J0 + 9 };

template <bool SD>
__global__ void __launch_bounds__(ATX * ATY) assemble_kernel(Grid g, Scheme s, Fields f, double dt, BlockMatrix A, MfPlanes mf,
                                                             const double* __restrict__ bsrc)
{
    extern __shared__ double tile[];                 // [TC_FIELDS][ACELLS] doubles, then ACELLS long long cell indices
    long long* tidx = reinterpret_cast<long long*>(tile + TC_FIELDS * ACELLS);
    const int i0 = blockIdx.x * ATX, j0 = blockIdx.y * ATY;
    const int tid = threadIdx.y * ATX + threadIdx.x;
    for (int cidx = tid; cidx < ACELLS; cidx += ATX * ATY) {
        const int cx = cidx % AW, cy = cidx / AW;
        const bool corner = (cx == 0 || cx == AW - 1) && (cy == 0 || cy == AH - 1);
        const int ci = i0 - 1 + cx, cj = j0 - 1 + cy;
        if (corner || ci > g.nx || cj > g.ny) continue;
        if ((ci < 0 || ci >= g.nx) && (cj < 0 || cj >= g.ny)) continue;      // domain corner ghosts are never used
        CellU u; Clo q; Jac J;
        fetch_cell(f, g, ci, cj, u);
        closure_eval<true, SD, true>(s, g.c, u.E, u.Fx, u.Fy, q, &J);
        tile[TC_E * ACELLS + cidx] = u.E; tile[TC_FX * ACELLS + cidx] = u.Fx; tile[TC_FY * ACELLS + cidx] = u.Fy;
        tile[TC_SA * ACELLS + cidx] = u.sa; tile[TC_ST * ACELLS + cidx] = u.st; tile[TC_F * ACELLS + cidx] = q.f;
        tile[TC_LMINX * ACELLS + cidx] = q.lmin[0]; tile[TC_LMAXX * ACELLS + cidx] = q.lmax[0];
        tile[TC_LMINY * ACELLS + cidx] = q.lmin[1]; tile[TC_LMAXY * ACELLS + cidx] = q.lmax[1];
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            tile[(TC_J0 + e) * ACELLS + cidx] = J.xx[e]; tile[(TC_J0 + 3 + e) * ACELLS + cidx] = J.xy[e]; tile[(TC_J0 + 6 + e) * ACELLS + cidx] = J.yy[e];
        }
        tidx[cidx] = u.idx;
    }
    __syncthreads();
    const int i = i0 + threadIdx.x, j = j0 + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const long long N = (long long)g.nx * g.ny, id = (long long)j * g.nx + i;
    CellU u[5]; Clo q[5]; Jac J[5];   // centre, west, east, south, north
    {
        const int cc = (threadIdx.y + 1) * AW + threadIdx.x + 1;
        const int where[5] = { cc, cc - 1, cc + 1, cc - AW, cc + AW };
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const int w = where[k];
            u[k].E = tile[TC_E * ACELLS + w]; u[k].Fx = tile[TC_FX * ACELLS + w]; u[k].Fy = tile[TC_FY * ACELLS + w];
            u[k].sa = tile[TC_SA * ACELLS + w]; u[k].st = tile[TC_ST * ACELLS + w]; u[k].idx = tidx[w];
            q[k].f = tile[TC_F * ACELLS + w];
            q[k].lmin[0] = tile[TC_LMINX * ACELLS + w]; q[k].lmax[0] = tile[TC_LMAXX * ACELLS + w];
            q[k].lmin[1] = tile[TC_LMINY * ACELLS + w]; q[k].lmax[1] = tile[TC_LMAXY * ACELLS + w];
#pragma unroll
            for (int e = 0; e < 3; ++e) {
                J[k].xx[e] = tile[(TC_J0 + e) * ACELLS + w]; J[k].xy[e] = tile[(TC_J0 + 3 + e) * ACELLS + w]; J[k].yy[e] = tile[(TC_J0 + 6 + e) * ACELLS + w];
            }
        }
    }
    Face fw, fe, fs, fn;
    face_eval<SD, true>(s, g.c, g.dx, q[1].lmin[0], q[1].lmax[0], q[1].f, u[1].st, q[0].lmin[0], q[0].lmax[0], q[0].f, u[0].st, fw);
    face_eval<SD, true>(s, g.c, g.dx, q[0].lmin[0], q[0].lmax[0], q[0].f, u[0].st, q[2].lmin[0], q[2].lmax[0], q[2].f, u[2].st, fe);
    face_eval<SD, true>(s, g.c, g.dy, q[3].lmin[1], q[3].lmax[1], q[3].f, u[3].st, q[0].lmin[1], q[0].lmax[1], q[0].f, u[0].st, fs);
    face_eval<SD, true>(s, g.c, g.dy, q[0].lmin[1], q[0].lmax[1], q[0].f, u[0].st, q[4].lmin[1], q[4].lmax[1], q[4].f, u[4].st, fn);

    const bool hyp = SD ? true : (s.hyp_off == 0);       // semi-implicit step: source-only system
    const double c = g.c, c2 = c * c, rx = hyp ? dt / g.dx : 0.0, ry = hyp ? dt / g.dy : 0.0;
    Blk B[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) blk_zero(B[k]);
    B[0].a[0] = 1.0; B[0].a[4] = 1.0; B[0].a[8] = 1.0;
    face_blocks(fe, 0, c2, J[0], J[2], rx, B[0], rx, B[2]);     // +rx G_e : L = centre, R = east
    face_blocks(fw, 0, c2, J[1], J[0], -rx, B[1], -rx, B[0]);   // -rx G_w : L = west,   R = centre
    face_blocks(fn, 1, c2, J[0], J[4], ry, B[0], ry, B[4]);     // +ry H_n
    face_blocks(fs, 1, c2, J[3], J[0], -ry, B[3], -ry, B[0]);   // -ry H_s

    // sources.  eta: linearised matter coupling (R10), 1 without T.
    double eta = 1.0, Theta = 0.0;
    if (f.T) {
        const double T = f.T[id], rcv = f.rho_cv ? f.rho_cv[id] : 1.0;
        eta = rcv / (rcv + 4.0 * s.a_r * c * u[0].sa * dt * T * T * T);
        Theta = s.a_r * (T * T) * (T * T);
    }
    B[0].a[0] += c * dt * u[0].sa * eta;
    const bool wb = SD ? true : (s.wb != 0);
    if (wb) {
        const double se = 0.25 * c * dt * fe.sig, sw = 0.25 * c * dt * fw.sig, sn = 0.25 * c * dt * fn.sig, ss = 0.25 * c * dt * fs.sig;
        B[0].a[4] += se + sw; B[2].a[4] += se; B[1].a[4] += sw;
        B[0].a[8] += sn + ss; B[4].a[8] += sn; B[3].a[8] += ss;
    } else {
        B[0].a[4] += c * dt * u[0].st; B[0].a[8] += c * dt * u[0].st;
    }
    // right-hand side
    double b[3] = { u[0].E, u[0].Fx, u[0].Fy };
    if (bsrc) { b[0] = bsrc[id]; b[1] = bsrc[N + id]; b[2] = bsrc[2 * N + id]; }   // Newton iterate: U^n comes from bsrc
    if (f.T) b[0] += c * dt * u[0].sa * eta * Theta;
    if (f.source_E) b[0] += dt * f.source_E[id];
    // boundaries (R9): a Dirichlet ghost is known -> block x ghost moves to b; a neighbour that is this
    // very cell (outflow copy, or a periodic direction one cell wide) folds into the diagonal block.
#pragma unroll
    for (int k = 1; k < 5; ++k) {
        if (u[k].idx < 0) {
#pragma unroll
            for (int r = 0; r < 3; ++r) b[r] -= B[k].a[3 * r] * u[k].E + B[k].a[3 * r + 1] * u[k].Fx + B[k].a[3 * r + 2] * u[k].Fy;
            blk_zero(B[k]);
        } else if (u[k].idx == id) {
#pragma unroll
            for (int e = 0; e < 9; ++e) B[0].a[e] += B[k].a[e];
            blk_zero(B[k]);
        }
    }
    Blk Mi; inv3(B[0], Mi);
    A.b[id] = b[0]; A.b[N + id] = b[1]; A.b[2 * N + id] = b[2];
#pragma unroll
    for (int e = 0; e < 9; ++e) A.Minv[e * N + id] = Mi.a[e];
    if (mf.J) {
        // matrix-free storage: the centre cell's Jacobian, its east and north face coefficients, the source weights
#pragma unroll
        for (int e = 0; e < 3; ++e) { mf.J[e * N + id] = J[0].xx[e]; mf.J[(3 + e) * N + id] = J[0].xy[e]; mf.J[(6 + e) * N + id] = J[0].yy[e]; }
        const double qw = wb ? 0.25 * c * dt : 0.0;
        mf.fE[id] = fe.ap; mf.fE[N + id] = fe.Lam; mf.fE[2 * N + id] = fe.alpha; mf.fE[3 * N + id] = qw * fe.sig;
        mf.fN[id] = fn.ap; mf.fN[N + id] = fn.Lam; mf.fN[2 * N + id] = fn.alpha; mf.fN[3 * N + id] = qw * fn.sig;
        mf.dE[id] = c * dt * u[0].sa * eta;
        mf.dF[id] = wb ? 0.0 : c * dt * u[0].st;
        if (i == 0) { mf.xlo[j] = fw.ap; mf.xlo[g.ny + j] = fw.Lam; mf.xlo[2 * g.ny + j] = fw.alpha; mf.xlo[3 * g.ny + j] = qw * fw.sig; }
        if (j == 0) { mf.ylo[i] = fs.ap; mf.ylo[g.nx + i] = fs.Lam; mf.ylo[2 * g.nx + i] = fs.alpha; mf.ylo[3 * g.nx + i] = qw * fs.sig; }
        return;
    }
#pragma unroll
    for (int e = 0; e < 9; ++e) A.C[e * N + id] = B[0].a[e];
#pragma unroll
    for (int k = 1; k < 5; ++k)
#pragma unroll
        for (int e = 0; e < 9; ++e) A.off[((k - 1) * 9 + e) * N + id] = B[k].a[e];
}

cudaError_t launch_assemble(const Grid& g, const Scheme& s, const Fields& f, double dt, BlockMatrix A, MfPlanes mf,
                            const double* bsrc, cudaStream_t st)
{
    dim3 blk(ATX, ATY), grd((g.nx + ATX - 1) / ATX, (g.ny + ATY - 1) / ATY);
    const size_t smem = (size_t)ACELLS * (TC_FIELDS * sizeof(double) + sizeof(long long));
    static bool attr_done = false;
    if (!attr_done) {
        cudaFuncSetAttribute(assemble_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaFuncSetAttribute(assemble_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr_done = true;
    }
    if (s.is_default()) assemble_kernel<true><<<grd, blk, smem, st>>>(g, s, f, dt, A, mf, bsrc);
    else assemble_kernel<false><<<grd, blk, smem, st>>>(g, s, f, dt, A, mf, bsrc);
    return cudaGetLastError();
}

// Neighbour cell of block k (0: W, 1: E, 2: S, 3: N).  Where the block is zero (Dirichlet, folded) any valid
// index will do, so non-periodic sides clamp.
__device__ __forceinline__ long long nbr_index(const Grid& g, int i, int j, int k)
{
    int ii = i + (k == 0 ? -1 : (k == 1 ? 1 : 0));
    int jj = j + (k == 2 ? -1 : (k == 3 ? 1 : 0));
    if (ii < 0) ii = (g.bc[XLO] == BC_PERIODIC) ? g.nx - 1 : 0;
    if (ii >= g.nx) ii = (g.bc[XHI] == BC_PERIODIC) ? 0 : g.nx - 1;
    if (jj < 0) jj = (g.bc[YLO] == BC_PERIODIC) ? g.ny - 1 : 0;
    if (jj >= g.ny) jj = (g.bc[YHI] == BC_PERIODIC) ? 0 : g.ny - 1;
    return (long long)jj * g.nx + ii;
}

// off_k <- off_k * Minv(neighbour k), in place; off32 (may be null) receives a single-precision copy (multigrid, mg_precision = 32).
__global__ void __launch_bounds__(128) scale_offdiag_kernel(Grid g, BlockMatrix A, float* __restrict__ off32)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const long long N = (long long)g.nx * g.ny, id = (long long)j * g.nx + i;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const long long nb = nbr_index(g, i, j, k);
        double m[9], a[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) { m[e] = A.Minv[e * N + nb]; a[e] = A.off[(k * 9 + e) * N + id]; }
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
                const double v = a[3 * r] * m[cc] + a[3 * r + 1] * m[3 + cc] + a[3 * r + 2] * m[6 + cc];
                A.off[(k * 9 + 3 * r + cc) * N + id] = v;
                if (off32) off32[(k * 9 + 3 * r + cc) * N + id] = (float)v;
            }
    }
}

cudaError_t launch_scale_offdiag(const Grid& g, BlockMatrix A, float* off32, cudaStream_t st)
{
    dim3 blk(32, 4), grd((g.nx + 31) / 32, (g.ny + 3) / 4);
    scale_offdiag_kernel<<<grd, blk, 0, st>>>(g, A, off32);
    return cudaGetLastError();
}

// t = C x (per cell 3x3)
__global__ void __launch_bounds__(256) diag_mul_kernel(long long N, const double* __restrict__ Cb, const double* __restrict__ x,
                                                       double* __restrict__ t)
{
    for (long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x; id < N; id += (long long)gridDim.x * blockDim.x) {
        const double x0 = x[id], x1 = x[N + id], x2 = x[2 * N + id];
        t[id]         = Cb[0 * N + id] * x0 + Cb[1 * N + id] * x1 + Cb[2 * N + id] * x2;
        t[N + id]     = Cb[3 * N + id] * x0 + Cb[4 * N + id] * x1 + Cb[5 * N + id] * x2;
        t[2 * N + id] = Cb[6 * N + id] * x0 + Cb[7 * N + id] * x1 + Cb[8 * N + id] * x2;
    }
}

cudaError_t launch_diag_mul(const Grid& g, const double* Cblk, const double* x, double* t, cudaStream_t st)
{
    const long long N = (long long)g.nx * g.ny;
    const int blk = 256; const int grd = (int)((N + blk - 1) / blk < current_sm_count() * 8 ? (N + blk - 1) / blk : current_sm_count() * 8);
    diag_mul_kernel<<<grd, blk, 0, st>>>(N, Cblk, x, t);
    return cudaGetLastError();
}

// out = sgn * s * (v + sum_k Ahat_k v_nbr(k)) + add      (A M^-1 has identity diagonal blocks)
__global__ void __launch_bounds__(128) spmv_hat_kernel(Grid g, const double* __restrict__ off, const double* __restrict__ v,
                                                       double* __restrict__ out, const double* __restrict__ scale_ptr,
                                                       const double* __restrict__ add, double sgn, const int* __restrict__ skip_flag)
{
    if (skip_flag && *skip_flag) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const long long N = (long long)g.nx * g.ny, id = (long long)j * g.nx + i;
    double acc0 = v[id], acc1 = v[N + id], acc2 = v[2 * N + id];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const long long nb = nbr_index(g, i, j, k);
        const double x0 = v[nb], x1 = v[N + nb], x2 = v[2 * N + nb];
        const double* a = off + (long long)(k * 9) * N + id;
        acc0 += a[0 * N] * x0 + a[1 * N] * x1 + a[2 * N] * x2;
        acc1 += a[3 * N] * x0 + a[4 * N] * x1 + a[5 * N] * x2;
        acc2 += a[6 * N] * x0 + a[7 * N] * x1 + a[8 * N] * x2;
    }
    const double sc = sgn * (scale_ptr ? *scale_ptr : 1.0);
    double o0 = sc * acc0, o1 = sc * acc1, o2 = sc * acc2;
    if (add) { o0 += add[id]; o1 += add[N + id]; o2 += add[2 * N + id]; }
    out[id] = o0; out[N + id] = o1; out[2 * N + id] = o2;
}

cudaError_t launch_spmv_hat(const Grid& g, const double* off, const double* v, double* out, const double* scale_ptr,
                            const double* add, double sgn, const int* skip_flag, cudaStream_t st)
{
    dim3 blk(32, 4), grd((g.nx + 31) / 32, (g.ny + 3) / 4);
    spmv_hat_kernel<<<grd, blk, 0, st>>>(g, off, v, out, scale_ptr, add, sgn, skip_flag);
    return cudaGetLastError();
}

// After the solve (R10): T^{n+1} = T + c sigma_a dt (E^{n+1} - a_r T^4)/(rho c_v + 4 a_r c sigma_a dt T^3)
__global__ void matter_update_kernel(long long N, double c, double a_r, double dt, const double* __restrict__ sa,
                                     const double* __restrict__ rho_cv, const double* __restrict__ Enew, double* __restrict__ T)
{
    for (long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x; id < N; id += (long long)gridDim.x * blockDim.x) {
        const double t = T[id], rcv = rho_cv ? rho_cv[id] : 1.0;
        const double Theta = a_r * (t * t) * (t * t);
        T[id] = t + c * sa[id] * dt * (Enew[id] - Theta) / (rcv + 4.0 * a_r * c * sa[id] * dt * t * t * t);
    }
}

cudaError_t launch_matter_update(const Grid& g, const Scheme& s, double dt, const double* sa, const double* rho_cv,
                                 const double* Enew, double* T, cudaStream_t st)
{
    const long long N = (long long)g.nx * g.ny;
    const int blk = 256; const int grd = (int)((N + blk - 1) / blk < current_sm_count() * 8 ? (N + blk - 1) / blk : current_sm_count() * 8);
    matter_update_kernel<<<grd, blk, 0, st>>>(N, g.c, s.a_r, dt, sa, rho_cv, Enew, T);
    return cudaGetLastError();
}

}  // namespace ark
