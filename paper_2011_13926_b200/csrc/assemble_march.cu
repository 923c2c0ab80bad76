// assemble_march.cu — row a5 for the matrix-free operator, in the explicit kernel's marching organisation.
//
// Writes, per cell: the pressure Jacobian J (9), the east- and north-face coefficients (a+, Lambda, alpha, c dt sigma_f/4) (8),
// the source weights (2), the inverse of the diagonal block M^-1 (9) and the right-hand side b (3) = 248 B out, 40 B in
// (PAPER.md:263 linearisation, 315-321 "matrix update"; formulas of implicit_kernels.cu).
// Closure + Jacobian are evaluated ONCE per cell (a thread owns a column and marches over rows), every face ONCE (north face
// from the thread's own two rows, east face from the east neighbour's data in shared memory, the west face is the west
// thread's east face).  The diagonal block needs only the cell's own J and its four faces:
//     C = I + rx (G_L(e) - G_R(w)) + ry (G_L(n) - G_R(s)) + sources          (+ folded neighbour blocks, R9)
// Dirichlet ghosts contribute to b through A_k g; with P homogeneous of degree 1 (J.g = P(g)) this needs only the ghost's
// pressure, which the halo thread / the neighbouring row has at hand.
#include "explicit_device.cuh"
#include "implicit_device.cuh"

namespace ark {

// one warp per block, like the explicit kernel: 1.104 -> 1.059 ms at 4096^2 (128 -> 64 -> 32 columns: 0.668 / 0.689 / 0.697 of HBM peak);
// with the shuffle exchange 1.008 ms = 0.73
static constexpr int TXA = 32;

struct ACell {                 // one cell: raw state, closure, Jacobian
    Raw u;
    Clo q;
    Jac J;
};
struct APub { double E, Fx, Fy, Pxx, Pxy, lmin, lmax, f, st; };
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// A_k g for a Dirichlet ghost state g on the far side of face `fc` (right == true: the ghost is the R cell of the face).
// Returns the contribution with weight w = +-dt/dx already applied, plus the WB source weight sw on the normal flux row.
__device__ __forceinline__ void ghost_term(const Face& fc, int dir, bool right, double w, double c2, double sw,
                                           double gE, double gFx, double gFy, double gPxx, double gPxy, double gPyy, double out[3])
{
    const double a = right ? fc.am : fc.ap, sg = right ? 1.0 : -1.0;
    const double Fn = dir == 0 ? gFx : gFy;
    const double Pnx = dir == 0 ? gPxx : gPxy, Pny = dir == 0 ? gPxy : gPyy;
    out[0] = w * fc.alpha * (sg * fc.Lam * gE + a * Fn);
    out[1] = w * (c2 * a * Pnx + sg * fc.Lam * gFx);
    out[2] = w * (c2 * a * Pny + sg * fc.Lam * gFy);
    out[1 + dir] += sw * Fn;
}

template <bool SD>
__global__ void __launch_bounds__(TXA) assemble_march_kernel(Grid g, Scheme s, Fields f, double dt, BlockMatrix A, MfPlanes mf,
                                                             const double* __restrict__ bsrc, int RY)
{
    const int t = threadIdx.x;
    const int i = blockIdx.x * (TXA - 2) - 1 + t;
    const int j0 = blockIdx.y * RY;
    const int j1 = min(j0 + RY, g.ny);
    const long long N = (long long)g.nx * g.ny;
    const bool upd = (t >= 1 && t <= TXA - 2 && i >= 0 && i < g.nx);
    const bool hyp = SD ? true : (s.hyp_off == 0);       // semi-implicit step: source-only system
    const double c = g.c, c2 = c * c, rx = hyp ? dt / g.dx : 0.0, ry = hyp ? dt / g.dy : 0.0, cdt = c * dt;
    const bool wb = SD ? true : (s.wb != 0);
    const double qw = wb ? 0.25 * cdt : 0.0;
    int xmode = 0, ii = i, xside = 0;
    if (i > g.nx) xmode = 2;
    else if (i < 0 || i >= g.nx) {
        xside = (i < 0) ? XLO : XHI;
        const int bc = g.bc[xside];
        if (bc == BC_DIRICHLET) { xmode = 1; ii = 0; }
        else if (bc == BC_PERIODIC) ii = (i < 0) ? g.nx - 1 : 0;
        else ii = (i < 0) ? 0 : g.nx - 1;
    }
    // which neighbours of this thread's cells are the cell itself (fold into C) or Dirichlet ghosts (move to b)
    const bool fold_w = (i == 0 && g.bc[XLO] == BC_OUTFLOW) || (g.nx == 1 && g.bc[XLO] == BC_PERIODIC);
    const bool fold_e = (i == g.nx - 1 && g.bc[XHI] == BC_OUTFLOW) || (g.nx == 1 && g.bc[XHI] == BC_PERIODIC);
    const bool dir_w = (i == 0 && g.bc[XLO] == BC_DIRICHLET), dir_e = (i == g.nx - 1 && g.bc[XHI] == BC_DIRICHLET);

    ACell S, C, Nn;
    S.u = load_row(f, g, xmode, ii, xside, j0 - 1);
    C.u = load_row(f, g, xmode, ii, xside, j0);
    Nn.u = load_row(f, g, xmode, ii, xside, j0 + 1);
    closure_eval<true, SD, true>(s, c, S.u.E, S.u.Fx, S.u.Fy, S.q, &S.J);
    closure_eval<true, SD, true>(s, c, C.u.E, C.u.Fx, C.u.Fy, C.q, &C.J);
    Face fs;
    face_eval<SD, true>(s, c, g.dy, S.q.lmin[1], S.q.lmax[1], S.q.f, S.u.st, C.q.lmin[1], C.q.lmax[1], C.q.f, C.u.st, fs);
    // the south neighbour's state and pressure (needed only if it is a Dirichlet ghost)
    double sE = S.u.E, sFx = S.u.Fx, sFy = S.u.Fy, sPxx = S.q.Pxx, sPxy = S.q.Pxy, sPyy = S.q.Pyy;

    for (int j = j0; j < j1; ++j) {
        const Raw uNN = load_row(f, g, (j + 1 < j1) ? xmode : 2, ii, xside, j + 2);
        APub me; me.E = C.u.E; me.Fx = C.u.Fx; me.Fy = C.u.Fy; me.Pxx = C.q.Pxx; me.Pxy = C.q.Pxy;
        me.lmin = C.q.lmin[0]; me.lmax = C.q.lmax[0]; me.f = C.q.f; me.st = C.u.st;
        // one-warp block: the neighbours' x-face data and the west face's coefficients travel by warp shuffles
        APub R, L;
        R.E = shfl_dn1(me.E); R.Fx = shfl_dn1(me.Fx); R.Fy = shfl_dn1(me.Fy); R.Pxx = shfl_dn1(me.Pxx); R.Pxy = shfl_dn1(me.Pxy);
        R.lmin = shfl_dn1(me.lmin); R.lmax = shfl_dn1(me.lmax); R.f = shfl_dn1(me.f); R.st = shfl_dn1(me.st);
        L.E = shfl_up1(me.E); L.Fx = shfl_up1(me.Fx); L.Fy = shfl_up1(me.Fy); L.Pxx = shfl_up1(me.Pxx); L.Pxy = shfl_up1(me.Pxy);
        closure_eval<true, SD, true>(s, c, Nn.u.E, Nn.u.Fx, Nn.u.Fy, Nn.q, &Nn.J);
        Face fn;
        face_eval<SD, true>(s, c, g.dy, C.q.lmin[1], C.q.lmax[1], C.q.f, C.u.st, Nn.q.lmin[1], Nn.q.lmax[1], Nn.q.f, Nn.u.st, fn);
        Face fe;
        face_eval<SD, true>(s, c, g.dx, me.lmin, me.lmax, me.f, me.st, R.lmin, R.lmax, R.f, R.st, fe);
        Face fw; fw.ap = shfl_up1(fe.ap); fw.am = shfl_up1(fe.am); fw.Lam = shfl_up1(fe.Lam); fw.alpha = shfl_up1(fe.alpha); fw.sig = shfl_up1(fe.sig);
        if (upd) {
            const long long id = (long long)j * g.nx + i;
            const bool fold_s = (j == 0 && g.bc[YLO] == BC_OUTFLOW) || (g.ny == 1 && g.bc[YLO] == BC_PERIODIC);
            const bool fold_n = (j == g.ny - 1 && g.bc[YHI] == BC_OUTFLOW) || (g.ny == 1 && g.bc[YHI] == BC_PERIODIC);
            const bool dir_s = (j == 0 && g.bc[YLO] == BC_DIRICHLET), dir_n = (j == g.ny - 1 && g.bc[YHI] == BC_DIRICHLET);
            const double se = qw * fe.sig, sw = qw * fw.sig, sn = qw * fn.sig, ss = qw * fs.sig;
            // diagonal block
            Blk B; blk_zero(B); B.a[0] = 1.0; B.a[4] = 1.0; B.a[8] = 1.0;
            add_G(B, fe, 0, false, rx, c2, C.J);      // +rx G_L(e)
            add_G(B, fw, 0, true, -rx, c2, C.J);      // -rx G_R(w)
            add_G(B, fn, 1, false, ry, c2, C.J);
            add_G(B, fs, 1, true, -ry, c2, C.J);
            double eta = 1.0, Theta = 0.0;
            if (f.T) {
                const double T = f.T[id], rcv = f.rho_cv ? f.rho_cv[id] : 1.0;
                eta = rcv / (rcv + 4.0 * s.a_r * c * C.u.sa * dt * T * T * T);
                Theta = s.a_r * (T * T) * (T * T);
            }
            const double dE = cdt * C.u.sa * eta;
            B.a[0] += dE;
            if (wb) { B.a[4] += se + sw; B.a[8] += sn + ss; }
            else { B.a[4] += cdt * C.u.st; B.a[8] += cdt * C.u.st; }
            // neighbours that are this very cell (outflow copy, one-cell-wide periodic direction) fold into the diagonal
            if (fold_e) { add_G(B, fe, 0, true, rx, c2, C.J); B.a[4] += se; }
            if (fold_w) { add_G(B, fw, 0, false, -rx, c2, C.J); B.a[4] += sw; }
            if (fold_n) { add_G(B, fn, 1, true, ry, c2, C.J); B.a[8] += sn; }
            if (fold_s) { add_G(B, fs, 1, false, -ry, c2, C.J); B.a[8] += ss; }
            // right-hand side
            double b0 = C.u.E, b1 = C.u.Fx, b2 = C.u.Fy;
            if (bsrc) { b0 = bsrc[id]; b1 = bsrc[N + id]; b2 = bsrc[2 * N + id]; }
            if (f.T) b0 += dE * Theta;
            if (f.source_E) b0 += dt * f.source_E[id];
            double gt[3];
            if (dir_e) { ghost_term(fe, 0, true, rx, c2, se, R.E, R.Fx, R.Fy, R.Pxx, R.Pxy, 0.0, gt); b0 -= gt[0]; b1 -= gt[1]; b2 -= gt[2]; }
            if (dir_w) { ghost_term(fw, 0, false, -rx, c2, sw, L.E, L.Fx, L.Fy, L.Pxx, L.Pxy, 0.0, gt); b0 -= gt[0]; b1 -= gt[1]; b2 -= gt[2]; }
            if (dir_n) { ghost_term(fn, 1, true, ry, c2, sn, Nn.u.E, Nn.u.Fx, Nn.u.Fy, 0.0, Nn.q.Pxy, Nn.q.Pyy, gt); b0 -= gt[0]; b1 -= gt[1]; b2 -= gt[2]; }
            if (dir_s) { ghost_term(fs, 1, false, -ry, c2, ss, sE, sFx, sFy, sPxx, sPxy, sPyy, gt); b0 -= gt[0]; b1 -= gt[1]; b2 -= gt[2]; }
            Blk Mi; inv3(B, Mi);
            A.b[id] = b0; A.b[N + id] = b1; A.b[2 * N + id] = b2;
#pragma unroll
            for (int e = 0; e < 9; ++e) A.Minv[e * N + id] = Mi.a[e];
#pragma unroll
            for (int e = 0; e < 3; ++e) { mf.J[e * N + id] = C.J.xx[e]; mf.J[(3 + e) * N + id] = C.J.xy[e]; mf.J[(6 + e) * N + id] = C.J.yy[e]; }
            mf.fE[id] = fe.ap; mf.fE[N + id] = fe.Lam; mf.fE[2 * N + id] = fe.alpha; mf.fE[3 * N + id] = se;
            mf.fN[id] = fn.ap; mf.fN[N + id] = fn.Lam; mf.fN[2 * N + id] = fn.alpha; mf.fN[3 * N + id] = sn;
            mf.dE[id] = dE;
            {   // reduced flux for the operator that rebuilds J (operator_mf.cu): the same sequence as closure_eval's, so that the
                // clamp decision is the one the stored J was formed with
                const double Es = (C.u.E > ARK_E_FLOOR) ? C.u.E : ARK_E_FLOOR;
                const double ice = rcp_sel<true>(c * Es);
                const double fx = C.u.Fx * ice, fy = C.u.Fy * ice;
                const double f2 = fx * fx + fy * fy;
                mf.fxy[id] = (f2 > 1.0) ? 4.0 : fx; mf.fxy[N + id] = fy;
            }
            mf.dF[id] = wb ? 0.0 : cdt * C.u.st;
            if (i == 0) { mf.xlo[j] = fw.ap; mf.xlo[g.ny + j] = fw.Lam; mf.xlo[2 * g.ny + j] = fw.alpha; mf.xlo[3 * g.ny + j] = sw; }
            if (j == 0) { mf.ylo[i] = fs.ap; mf.ylo[g.nx + i] = fs.Lam; mf.ylo[2 * g.nx + i] = fs.alpha; mf.ylo[3 * g.nx + i] = ss; }
        }
        // shift the window north
        sE = C.u.E; sFx = C.u.Fx; sFy = C.u.Fy; sPxx = C.q.Pxx; sPxy = C.q.Pxy; sPyy = C.q.Pyy;
        C = Nn; Nn.u = uNN; fs = fn;
    }
}

cudaError_t launch_assemble_march(const Grid& g, const Scheme& s, const Fields& f, double dt, BlockMatrix A, MfPlanes mf,
                                  const double* bsrc, int sm_count, cudaStream_t st)
{
    const int strips = (g.nx + (TXA - 2) - 1) / (TXA - 2);
    long long want = ((long long)g.ny * strips + (long long)sm_count * 8 - 1) / ((long long)sm_count * 8);
    int RY = (int)(want < 4 ? 4 : (want > 32 ? 32 : want));
    if (RY > g.ny) RY = g.ny;
    dim3 grd(strips, (g.ny + RY - 1) / RY);
    if (s.is_default()) assemble_march_kernel<true><<<grd, TXA, 0, st>>>(g, s, f, dt, A, mf, bsrc, RY);
    else assemble_march_kernel<false><<<grd, TXA, 0, st>>>(g, s, f, dt, A, mf, bsrc, RY);
    return cudaGetLastError();
}

}  // namespace ark
