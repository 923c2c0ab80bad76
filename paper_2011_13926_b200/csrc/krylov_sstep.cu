// krylov_sstep.cu — row a6: the s-step Arnoldi block of restarted GMRES(m) (option "arnoldi_block" = 3..5).
//
// Orthogonalisation against the basis is most of an iteration's traffic (PAPER.md:263-272 fixes the solver, not how its basis is
// built), and every Arnoldi column reads the whole basis twice.  A block builds SB columns per pass:
//   W_1 = A^ v_j,  W_k = (A^ - theta) W_{k-1}  (theta = 1: A^ = A M^-1 has its spectrum around 1; the shifted powers stay well
//   conditioned where the plain powers of A^ do not — numpy model of this file: in-block orthogonality defect 1e-6 against 4e-2 at s = 6);
//   C = V^T W  (ONE pass over v_0..v_j for all SB vectors: multi_dotS_kernel);
//   W' = W - V C with the Gram matrix G = W'^T W'  (ONE pass: updateS_kernel);  G = R^T R (Cholesky, on the device);
//   q~_k = W'_k - sum_{l<k} (R_lk / R_ll) q~_l element by element with the norms n_k = ||q~_k|| MEASURED (qrS_kernel), v_{j+k} = q~_k / n_k.
// The Hessenberg columns are those of Arnoldi.  With B = [v_j, W_1 .. W_{SB-1}]:  A^ B = W + theta B D (D = diag(0, 1, .., 1)),
// B = [V Q] G^ and W = [V Q] K in the orthonormal basis (K = [C; R~], R~ = the factor actually applied: R~_lk = R_lk n_l / R_ll,
// R~_kk = n_k), and A^ v_i = sum_k Hraw_ki v_k for i < j, so the new columns U_0 .. U_{SB-1} solve the triangular system
//   U_b = ( K_b + theta G^_b - Hraw(:, 0..j-1) C(0..j-1, b-1) - U_0 C(j, b-1) - sum_{1<=l<b} U_l R~(l-1, b-1) ) / R~(b-1, b-1),   U_0 = K_0,
// evaluated by the last block of the reduction (one thread per row), each followed by the Givens rotations / residual estimate /
// stop test of the one-column step (finish_column).  In exact arithmetic the iterates are GMRES(m)'s.
// Conditioning.  The pivot ratios rho_k = R_kk^2 / G_kk (the part of W'_k that is new) measure the block: the coefficients of the
// in-block solve carry a relative error of about eps / rho.  On the bench medium rho >= 0.04; on the smooth diffusive problem at
// 1024^2, whose residual falls tenfold per iteration, the first block has rho = (1, 1.6e-4, 3.5e-6, 7.9e-9, 4.0e-12) and one round
// left the basis orthogonal to 1e-5 only (29 iterations instead of 17).  A block with min rho < SS_RHO_REFINE therefore gets a SECOND
// round (gramS_kernel + qrS_kernel round 2: Gram matrix of the q~, Cholesky, solve; "CholQR2"), whose kernels return at once for every
// other block; W' = Q~ T with T = T2 T1 the product of the unit triangular factors, R~ = diag(n) T.  A pivot below SS_RHO_DROP (the
// Krylov space is exhausted inside the block, or beyond what two rounds repair) truncates the block there and ends the cycle.
// Prediction.  The dot pass also dots the block's own slots (S = W^T W, the operands already in L1), so G' = S - C^T C gives the
// Cholesky factor BEFORE the update pass; for a well-conditioned block (predicted rho >= SS_RHO_PRED) the update pass applies the
// in-block solve to the registers it holds and measures the Gram matrix of the q~; if that is orthogonal to SS_PRED_TOL the block is
// finished there and the separate in-block pass (216 of ~1900 B per cell and block) is not run (sstep_predict, sstep_pred_epilogue).
#include <stdio.h>
#include "krylov_device.cuh"

namespace ark {

static constexpr int GS_BLOCKS_PER_SM_SS = 2;   // one wave of two 256-thread blocks per SM, like the other Gram-Schmidt streams
static constexpr double SS_RHO_REFINE = 1e-5, SS_RHO_DROP = 1e-13;     // thresholds 1e-5 .. 0.5 give the same iteration counts on every system tried
// prediction of the in-block solve (sstep_predict): used when every predicted pivot ratio is at least SS_RHO_PRED and no diagonal entry of
// S - C^T C lost more than three digits; the block counts as finished when the MEASURED Gram matrix of the q~ has every
// |<q~_k, q~_l>| <= SS_PRED_TOL ||q~_k|| ||q~_l|| (what one round of the measured factorisation reaches for rho >= SS_RHO_REFINE)
static constexpr double SS_RHO_PRED = 1e-3, SS_PRED_CANCEL = 1e-3, SS_PRED_TOL = 1e-10;
static constexpr int SS_NVW = 4;              // basis vectors per warp of the dot kernel (8 warps -> 32 vectors per launch)
static constexpr int SS_CH = 8 * SS_NVW;      // basis vectors per launch of the dot kernel
__host__ __device__ constexpr int ss_ng(int s) { return s * (s + 1) / 2; }

int sstep_partial_doubles(int sm_count) { return sm_count * GS_BLOCKS_PER_SM_SS * SMAX * SS_CH; }

__device__ __forceinline__ double2 ld_cs2(const double2* p) { return __ldcs(p); }

// ---------------------------------------------------------------------------------------------------------
// Dots of SB vectors against up to 32 basis vectors in one pass.  The basis vectors are dealt to the 8 warps of a block (warp g of G
// groups takes i = g, g + G, ..): a warp keeps SB x NVW accumulators, whatever j is, and every warp of a block reads the same
// elements of W_1..W_SB (once from HBM, the rest from L1).  With fewer than 32 vectors there are fewer groups and the other warps
// take other elements (replicas of the groups).
// ---------------------------------------------------------------------------------------------------------
template <int SB, int NVW, int U>
__device__ __forceinline__ void dotS_body(const double* __restrict__ w1, const double* __restrict__ V0, long long stride, long long n2,
                                          int grp, int G, int rep, int R, int lane, int wfirst, double (&acc)[SB][SS_NVW])
{
    // vectors wfirst.. of the chunk are the block's own slots: the same lines the `a` loads of this block bring into L1, so they are
    // read through L1 (the basis streams past it)
    bool own[NVW];
#pragma unroll
    for (int q = 0; q < NVW; ++q) own[q] = (grp + q * G) >= wfirst;
    const long long tile = 32LL * U;
    for (long long t = (long long)rep * gridDim.x + blockIdx.x; t * tile < n2; t += (long long)R * gridDim.x) {
        const long long e0 = t * tile + lane;
        double2 a[U][SB], b[U][NVW];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long e = e0 + 32LL * u;
            const bool in = e < n2;
#pragma unroll
            for (int k = 0; k < SB; ++k) a[u][k] = in ? reinterpret_cast<const double2*>(w1 + k * stride)[e] : make_double2(0.0, 0.0);
#pragma unroll
            for (int q = 0; q < NVW; ++q) {
                const double2* pb = reinterpret_cast<const double2*>(V0 + (long long)(grp + q * G) * stride) + e;
                b[u][q] = in ? (own[q] ? *pb : ld_cs2(pb)) : make_double2(0.0, 0.0);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k = 0; k < SB; ++k)
#pragma unroll
                for (int q = 0; q < NVW; ++q) acc[k][q] = fma(a[u][k].y, b[u][q].y, fma(a[u][k].x, b[u][q].x, acc[k][q]));
    }
}

template <int SB> __device__ __forceinline__ void sstep_predict(const GmresWork& W, int j);

template <int SB>
__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM_SS) multi_dotS_kernel(const double* __restrict__ w1, const double* __restrict__ V0,
                                                                                    long long stride, long long n, GmresWork W, int nv, int col0, int jpred)
{
    if (W.ctl->inner_stop) return;
    __shared__ double sred[KTHREADS / 32][SB * SS_NVW];
    __shared__ bool is_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // groups: the smallest power of two that leaves a warp at most SS_NVW vectors, so that 8 / G replicas keep every warp busy and the
    // vectors per warp are as even as they can be (6 vectors: 2 groups x 3 vectors x 4 replicas, not 6 x 1 with two warps idle)
    const int G = nv <= SS_NVW ? 1 : (nv <= 2 * SS_NVW ? 2 : (nv <= 4 * SS_NVW ? 4 : 8)), R = 8 / G;
    const int grp = warp % G, rep = warp / G;
    const int nvw = (rep < R) ? (nv - grp + G - 1) / G : 0;          // vectors of this warp (0: spare warp)
    const long long n2 = n >> 1;
    const int wfirst = (jpred >= 0) ? jpred + 1 - col0 : (1 << 30);
    double acc[SB][SS_NVW];
#pragma unroll
    for (int k = 0; k < SB; ++k)
#pragma unroll
        for (int q = 0; q < SS_NVW; ++q) acc[k][q] = 0.0;
    switch (nvw) {      // loads in flight per lane: (SB + nvw) U >= 14
        case 1: dotS_body<SB, 1, 3>(w1, V0, stride, n2, grp, G, rep, R, lane, wfirst, acc); break;
        case 2: dotS_body<SB, 2, 2>(w1, V0, stride, n2, grp, G, rep, R, lane, wfirst, acc); break;
        case 3: dotS_body<SB, 3, 2>(w1, V0, stride, n2, grp, G, rep, R, lane, wfirst, acc); break;
        case 4: dotS_body<SB, 4, 2>(w1, V0, stride, n2, grp, G, rep, R, lane, wfirst, acc); break;
        default: break;
    }
#pragma unroll
    for (int k = 0; k < SB; ++k)
#pragma unroll
        for (int q = 0; q < SS_NVW; ++q) {
            const double s = warp_sum(acc[k][q]);
            if (lane == 0) sred[warp][k * SS_NVW + q] = s;
        }
    __syncthreads();
    // entry (k, i): vector i of the chunk belongs to group i % G, slot i / G; its replicas are the warps grp + G r
    const unsigned int bid = blockIdx.x, nb = gridDim.x;
    const int ent = threadIdx.x;
    if (ent < SB * SS_CH) {
        const int k = ent / SS_CH, i = ent % SS_CH;
        double s = 0.0;
        if (i < nv) { const int g = i % G, q = i / G; for (int r = 0; r < R; ++r) s += sred[g + G * r][k * SS_NVW + q]; }
        W.partialS[(size_t)bid * (SMAX * SS_CH) + ent] = s;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicInc(&W.ctl->ticket, nb - 1);
        is_last = (t == nb - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (ent < SB * SS_CH) {
        const int k = ent / SS_CH, i = ent % SS_CH;
        if (i < nv) {
            double s = 0.0;
            for (unsigned int b = 0; b < nb; ++b) s += __ldcg(&W.partialS[(size_t)b * (SMAX * SS_CH) + ent]);
            if (n & 1) s += w1[k * stride + n - 1] * V0[(long long)i * stride + n - 1];
            const int ld = W.ctl->m + 1, col = col0 + i;
            if (W.red_out) { W.red_out[k * ld + col] = s; return; }      // slab decomposition: this rank's sums; all-reduce and epilogue follow
            if (jpred >= 0 && col > jpred) W.ctl->gram[k * SMAX + (col - jpred - 1)] = s;      // a slot of the block itself: <W_k, W_l>
            else {
                const double c = s * W.scale[col];
                W.cS[k * ld + col] = c;
                W.coefS[k * ld + col] = c * W.scale[col];
            }
        }
    }
    if (W.red_out || jpred < 0 || col0 + nv != jpred + 1 + SB) return;      // (uniform) no prediction here, or more chunks of this block follow
    __syncthreads();
    sstep_predict<SB>(W, jpred);
}

// ---------------------------------------------------------------------------------------------------------
// W_k -= sum_i coefS_{i,k} V_i over all nv basis vectors in one pass (coefficients in shared memory, the basis through the registers in
// batches of SS_UB vectors), Gram matrix of the result; epilogue: Cholesky, coefficients of the in-block solve, first column of the block.
// ---------------------------------------------------------------------------------------------------------
static constexpr int SS_UB = 8;
static constexpr int SS_MAXNV = 128;

template <int SB, int NB>
__device__ __forceinline__ void updS_batch(double2 (&a)[SB], const double* __restrict__ Vb, long long stride, long long e, const double* __restrict__ cf)
{
    double2 b[NB];
#pragma unroll
    for (int q = 0; q < NB; ++q) b[q] = ld_cs2(reinterpret_cast<const double2*>(Vb + q * stride) + e);
#pragma unroll
    for (int q = 0; q < NB; ++q)
#pragma unroll
        for (int k = 0; k < SB; ++k) { const double c = cf[q * SB + k]; a[k].x = fma(-c, b[q].x, a[k].x); a[k].y = fma(-c, b[q].y, a[k].y); }
}

// Cholesky factor of a Gram matrix given as its upper triangle (row-major): t_{l,k} = R_{l,k} / R_{l,l} for l < k < nacc (0 elsewhere),
// rho_k = R_kk^2 / G_kk.  Returns the number of leading columns whose pivot is at least drop * G_kk.
template <int SB>
__device__ int sstep_factor(const double* __restrict__ G, double drop, double (&t)[SB][SB], double (&rho)[SB], double& r00)
{
    double Gm[SB][SB], R[SB][SB];
    int p = 0;
    for (int k = 0; k < SB; ++k) for (int l = k; l < SB; ++l) { Gm[k][l] = G[p]; Gm[l][k] = G[p]; ++p; }
    for (int k = 0; k < SB; ++k) for (int l = 0; l < SB; ++l) { R[k][l] = 0.0; t[k][l] = 0.0; }
    for (int k = 0; k < SB; ++k) rho[k] = 0.0;
    int nacc = SB;
    for (int k = 0; k < SB; ++k) {
        double d = Gm[k][k];
        for (int l = 0; l < k; ++l) d -= R[l][k] * R[l][k];
        if (!(d > drop * Gm[k][k]) || !isfinite(d)) { nacc = k; break; }
        rho[k] = d / Gm[k][k];
        R[k][k] = sqrt(d);
        for (int l = k + 1; l < SB; ++l) {
            double v = Gm[k][l];
            for (int q = 0; q < k; ++q) v -= R[q][k] * R[q][l];
            R[k][l] = v / R[k][k];
        }
    }
    for (int k = 0; k < nacc; ++k) for (int l = k + 1; l < nacc; ++l) t[k][l] = R[k][l] / R[k][k];
    r00 = R[0][0];
    return nacc;
}

// Prediction of the in-block solve by the dot pass (its last block, all threads).  The dot pass also dots the block's own slots like
// basis vectors, S = W^T W; with C = V^T W and V orthonormal the Gram matrix of W' = W - V C is G' = S - C^T C, so the Cholesky factor and
// the coefficients t of the solve are known BEFORE the update pass, which then applies the solve to the registers it already holds
// the block in (q~ = W' T^-1 element by element) and measures the Gram matrix of the q~.  Whatever T is, W' = Q~ T holds by
// construction and the recovery of the Hessenberg columns uses the T applied and the norms measured; T only decides how orthogonal
// the q~ are, and that is CHECKED on the measured Gram matrix (sstep_pred_epilogue): a block that passes is finished without the
// separate in-block pass (216 B per cell less), one that fails goes through the second round with the Gram matrix just measured.
template <int SB>
__device__ __forceinline__ void sstep_predict(const GmresWork& W, int j)
{
    __shared__ double Gp[SMAX * SMAX];
    GmresCtl* c = W.ctl;
    const int ld = c->m + 1;
    if (threadIdx.x < SB * SB) {
        const int k = threadIdx.x / SB, l = threadIdx.x % SB;
        double s = 0.0;
        for (int i = 0; i <= j; ++i) s = fma(W.cS[k * ld + i], W.cS[l * ld + i], s);
        Gp[k * SMAX + l] = 0.5 * (c->gram[k * SMAX + l] + c->gram[l * SMAX + k]) - s;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    double G[ss_ng(SB)], t[SB][SB], rho[SB], r00;
    int p = 0;
    bool ok = true;
    for (int k = 0; k < SB; ++k) {
        for (int l = k; l < SB; ++l) G[p++] = Gp[k * SMAX + l];
        ok = ok && (Gp[k * SMAX + k] > SS_PRED_CANCEL * c->gram[k * SMAX + k]);
    }
    const int nacc = sstep_factor<SB>(G, SS_RHO_DROP, t, rho, r00);
    ok = ok && nacc == SB;
    for (int k = 0; k < SB; ++k) ok = ok && (rho[k] >= SS_RHO_PRED);
#ifdef SS_DEBUG
    printf("pred j=%d ok=%d rho:", j, (int)ok); for (int k = 0; k < SB; ++k) printf(" %.2e", rho[k]);
    printf("  G'/S:"); for (int k = 0; k < SB; ++k) printf(" %.2e", Gp[k * SMAX + k] / c->gram[k * SMAX + k]); printf("\n");
#endif
    c->blk[5] = ok ? 1.0 : 0.0;
    c->blk[6] = 0.0;
    if (!ok) return;
    for (int k = 0; k < SB; ++k)
        for (int l = 0; l < SB; ++l) { W.tb[k * SMAX + l] = t[k][l]; W.Rb[k * SMAX + l] = (k == l) ? 1.0 : t[k][l]; }
    c->blk[3] = (double)SB;
    c->blk[4] = 0.0;
}

// the scalar part of the epilogue after the update pass (thread 0 of the last block)
template <int SB>
__device__ void sstep_first_round(const GmresWork& W, const double* __restrict__ G, const double* hcol, const double* ccs, const double* ssn)
{
    GmresCtl* c = W.ctl;
    const int j = c->j, m = c->m;
    double t[SB][SB], rho[SB], r00;
    const int nacc = sstep_factor<SB>(G, SS_RHO_DROP, t, rho, r00);
    double rmin = 1.0;
    for (int k = 0; k < nacc; ++k) rmin = rho[k] < rmin ? rho[k] : rmin;
    for (int k = 0; k < SB; ++k)
        for (int l = 0; l < SB; ++l) { W.tb[k * SMAX + l] = t[k][l]; W.Rb[k * SMAX + l] = (k == l) ? 1.0 : t[k][l]; }
    c->blk[3] = (double)nacc;
    c->blk[4] = (nacc > 1 && rmin < SS_RHO_REFINE) ? 1.0 : 0.0;
    c->blk_stat[c->blk[4] != 0.0 ? 3 : 2] += 1;
#ifdef SS_DEBUG
    printf("blk j=%d nacc=%d refine=%d rho:", j, nacc, (int)c->blk[4]); for (int k = 0; k < SB; ++k) printf(" %.2e", rho[k]); printf("\n");
#endif
    if (nacc == 0) {        // W'_1 = 0: the space is exhausted at column j (h_{j+1,j} = 0 ends the cycle like the one-column step)
        W.Hraw[(j + 1) * m + j] = 0.0;
        finish_column(W, c, j, 0.0, hcol, ccs, ssn);
        return;
    }
    c->blk[0] = r00;
    W.Hraw[(j + 1) * m + j] = r00;
    finish_column(W, c, j, r00, hcol, ccs, ssn);
    if (nacc == 1) c->inner_stop = 1;
}

// last block of the update pass (or the epilogue kernel of the slab decomposition): stage column j (the c of the first vector, also the
// raw Hessenberg column), then the scalar part
template <int SB>
__device__ __forceinline__ void sstep_update_epilogue(const GmresWork& W, const double* dres, double* hcol, double* ccs, double* ssn)
{
    const int j = W.ctl->j, m = W.ctl->m;
    for (int i = threadIdx.x; i <= j; i += blockDim.x) {
        const double h = W.cS[i];
        hcol[i] = h; W.Hraw[i * m + j] = h;
        if (i < j) { ccs[i] = W.cs[i]; ssn[i] = W.sn[i]; }
    }
    __syncthreads();
    if (threadIdx.x == 0) sstep_first_round<SB>(W, dres, hcol, ccs, ssn);
}

template <int SB> __device__ __forceinline__ void sstep_finish_block(const GmresWork& W, const double* dres, double theta);
template <int SB> __device__ __forceinline__ void sstep_second_round(const GmresWork& W, const double* dres);

// last block of an update pass that applied the predicted solve: column j from the measured ||q~_1||, then the check of the measured
// Gram matrix: orthogonal -> the remaining columns of the block here; not -> second round from this Gram matrix (qrS_kernel round 2)
template <int SB>
__device__ __forceinline__ void sstep_pred_epilogue(const GmresWork& W, const double* dres, double theta, double* hcol, double* ccs, double* ssn)
{
    __shared__ double nrm2[SMAX];
    __shared__ int verdict;          // 0: the block is orthogonal, finish it here   1: second round   2: nothing more to do
    GmresCtl* c = W.ctl;
    const int j = c->j, m = c->m;
    for (int i = threadIdx.x; i <= j; i += blockDim.x) {
        const double h = W.cS[i];
        hcol[i] = h; W.Hraw[i * m + j] = h;
        if (i < j) { ccs[i] = W.cs[i]; ssn[i] = W.sn[i]; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double Gd[SB];
        int p = 0;
        double defect = 0.0;
        for (int k = 0; k < SB; ++k) { Gd[k] = dres[p]; p += SB - k; }
        p = 0;
        for (int k = 0; k < SB; ++k)
            for (int l = k; l < SB; ++l) { if (l > k) { const double d = fabs(dres[p]) / sqrt(Gd[k] * Gd[l]); defect = (d > defect || !(d == d)) ? d : defect; } ++p; }
        const bool orth = defect <= SS_PRED_TOL;        // false for a NaN as well
#ifdef SS_DEBUG
        printf("  pred-applied j=%d defect=%.2e\n", j, defect);
#endif
        if (!(Gd[0] > 0.0)) {          // W'_1 = 0: the space is exhausted at column j
            W.Hraw[(j + 1) * m + j] = 0.0;
            finish_column(W, c, j, 0.0, hcol, ccs, ssn);
            c->blk[6] = 1.0;
            verdict = 2;
        } else {
            const double r00 = sqrt(Gd[0]);
            c->blk[0] = r00;
            W.Hraw[(j + 1) * m + j] = r00;
            finish_column(W, c, j, r00, hcol, ccs, ssn);
            if (c->inner_stop) { c->blk[6] = 1.0; verdict = 2; }
            else if (orth) {
                for (int k = 1; k < SB; ++k) nrm2[k - 1] = Gd[k];
                c->blk[6] = 1.0; c->blk_stat[0] += 1;
                verdict = 0;
            } else {
                sstep_second_round<SB>(W, dres);      // T <- T2 T1, coefficients of round 2 from the Gram matrix measured here
                c->blk[4] = 1.0; c->blk_stat[1] += 1;
                if ((int)c->blk[3] <= 1) c->inner_stop = 1;
                verdict = 1;
            }
        }
    }
    __syncthreads();
    if (verdict == 0) sstep_finish_block<SB>(W, nrm2, theta);
}

template <int SB>
__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM_SS) updateS_kernel(double* __restrict__ w1, const double* __restrict__ V0, long long stride,
                                                                                 long long n, GmresWork W, int nv, double theta)
{
    if (W.ctl->inner_stop) return;
    constexpr int NG = ss_ng(SB);
    __shared__ double cf[SS_MAXNV * SB];
    __shared__ double tsh[SMAX * SMAX];
    __shared__ double dres[MAXV];
    __shared__ double hcol[EPI_MAX + 1], ccs[EPI_MAX], ssn[EPI_MAX];
    const int ld = W.ctl->m + 1;
    const bool pred = W.ctl->blk[5] != 0.0;      // the dot pass predicted the in-block solve: apply it here
    for (int q = threadIdx.x; q < nv * SB; q += KTHREADS) cf[q] = W.coefS[(q % SB) * ld + q / SB];
    if (threadIdx.x < SMAX * SMAX) tsh[threadIdx.x] = pred ? W.tb[threadIdx.x] : 0.0;
    __syncthreads();
    double acc[NG];
#pragma unroll
    for (int p = 0; p < NG; ++p) acc[p] = 0.0;
    const long long n2 = n >> 1, T = (long long)gridDim.x * KTHREADS;
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n2; e += T) {
        double2 a[SB];
#pragma unroll
        for (int k = 0; k < SB; ++k) a[k] = ld_cs2(reinterpret_cast<const double2*>(w1 + k * stride) + e);
        int q0 = 0;
        for (; q0 + SS_UB <= nv; q0 += SS_UB) updS_batch<SB, SS_UB>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB);
        switch (nv - q0) {
            case 1: updS_batch<SB, 1>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB); break;
            case 2: updS_batch<SB, 2>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB); break;
            case 3: updS_batch<SB, 3>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB); break;
            case 4: updS_batch<SB, 4>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB); break;
            case 5: updS_batch<SB, 5>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB); break;
            case 6: updS_batch<SB, 6>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB); break;
            case 7: updS_batch<SB, 7>(a, V0 + (long long)q0 * stride, stride, e, cf + q0 * SB); break;
            default: break;
        }
        if (pred) {
#pragma unroll
            for (int k = 1; k < SB; ++k)
#pragma unroll
                for (int l = 0; l < k; ++l) { const double t = tsh[l * SMAX + k]; a[k].x = fma(-t, a[l].x, a[k].x); a[k].y = fma(-t, a[l].y, a[k].y); }
        }
        int p = 0;
#pragma unroll
        for (int k = 0; k < SB; ++k) {
            reinterpret_cast<double2*>(w1 + k * stride)[e] = a[k];
#pragma unroll
            for (int l = k; l < SB; ++l) { acc[p] = fma(a[k].y, a[l].y, fma(a[k].x, a[l].x, acc[p])); ++p; }
        }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        double a[SB];
        for (int k = 0; k < SB; ++k) { a[k] = w1[k * stride + n - 1]; for (int q = 0; q < nv; ++q) a[k] -= cf[q * SB + k] * V0[(long long)q * stride + n - 1]; }
        for (int k = 1; k < SB; ++k) for (int l = 0; l < k; ++l) a[k] -= tsh[l * SMAX + k] * a[l];
        for (int k = 0; k < SB; ++k) w1[k * stride + n - 1] = a[k];
        int p = 0;
        for (int k = 0; k < SB; ++k) for (int l = k; l < SB; ++l) acc[p++] += a[k] * a[l];
    }
    if (!reduce_to_last<NG>(acc, W, dres)) return;
    if (W.red_out) { if (threadIdx.x < NG) W.red_out[threadIdx.x] = dres[threadIdx.x]; return; }
    if (pred) sstep_pred_epilogue<SB>(W, dres, theta, hcol, ccs, ssn);
    else sstep_update_epilogue<SB>(W, dres, hcol, ccs, ssn);
}

// Columns j0+1 .. j0+nacc-1 of the Hessenberg matrix from the measured norms of the in-block solve (c->j = j0 + 1 here: the update pass
// finished column j0).  Run by one block: the last block of qrS_kernel, or the epilogue kernel of the slab decomposition.
template <int SB>
__device__ __forceinline__ void sstep_finish_block(const GmresWork& W, const double* dres, double theta)
{
    __shared__ double hcol[EPI_MAX + 1], ccs[EPI_MAX], ssn[EPI_MAX];
    __shared__ double Ush[SMAX][EPI_MAX + SMAX + 1];
    __shared__ double Rt[SMAX][SMAX], nrm[SMAX];
    __shared__ int stop_sh;
    GmresCtl* c = W.ctl;
    const int m = c->m, ld = m + 1, j0 = c->j - 1, nacc = (int)c->blk[3];
    const int rows = j0 + 1 + SB;
    if (threadIdx.x == 0) {
        // R~ = diag(n) T: the factor actually applied (W' = Q~ T with the unit triangular T of the solve(s), q_k = q~_k / n_k measured)
        nrm[0] = c->blk[0];
        for (int k = 1; k < SB; ++k) nrm[k] = sqrt(dres[k - 1]);
        for (int l = 0; l < SB; ++l)
            for (int k = 0; k < SB; ++k) Rt[l][k] = (k >= l) ? nrm[l] * W.Rb[l * SMAX + k] : 0.0;
        stop_sh = 0;
    }
    for (int i = threadIdx.x; i < c->j; i += (int)blockDim.x) { ccs[i] = W.cs[i]; ssn[i] = W.sn[i]; }
    __syncthreads();
    // U_0 = K_0 = [C(:, 0); R~(:, 0)]
    for (int r = threadIdx.x; r < rows; r += (int)blockDim.x) Ush[0][r] = (r <= j0) ? W.cS[r] : Rt[r - j0 - 1][0];
    __syncthreads();
    for (int b = 1; b < nacc; ++b) {
        const int col = j0 + b;
        const double piv = Rt[b - 1][b - 1];
        for (int r = threadIdx.x; r < rows; r += (int)blockDim.x) {
            // K_b + theta G^_b
            double s = (r <= j0) ? fma(theta, W.cS[(b - 1) * ld + r], W.cS[b * ld + r]) : fma(theta, Rt[r - j0 - 1][b - 1], Rt[r - j0 - 1][b]);
            // - Hraw(:, 0..j0-1) C(0..j0-1, b-1): row r of Hraw is non-zero from column r-1 on
            if (r <= j0) for (int i = (r > 0 ? r - 1 : 0); i < j0; ++i) s = fma(-W.Hraw[r * m + i], W.cS[(b - 1) * ld + i], s);
            s = fma(-Ush[0][r], W.cS[(b - 1) * ld + j0], s);
            for (int l = 1; l < b; ++l) s = fma(-Ush[l][r], Rt[l - 1][b - 1], s);
            const double u = s / piv;
            Ush[b][r] = u;
            if (r <= col + 1) W.Hraw[r * m + col] = u;
            if (r <= col) hcol[r] = u;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            finish_column(W, c, col, Ush[b][col + 1], hcol, ccs, ssn, nrm[b]);
            ccs[col] = W.cs[col]; ssn[col] = W.sn[col];
            stop_sh = c->inner_stop;
        }
        __syncthreads();
        if (stop_sh) break;
    }
    if (threadIdx.x == 0 && nacc < SB) c->inner_stop = 1;      // truncated block: the cycle ends here
}

// ---------------------------------------------------------------------------------------------------------
// In-block triangular solve element by element, measured norms; epilogue: the remaining columns of the block.
// ---------------------------------------------------------------------------------------------------------
template <int SB>
__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM_SS) qrS_kernel(double* __restrict__ w1, long long stride, long long n, GmresWork W, double theta, int round)
{
    if (W.ctl->inner_stop || W.ctl->blk[6] != 0.0) return;      // [6]: the update pass finished the block (predicted solve, verified)
    const bool refine = W.ctl->blk[4] != 0.0;
    if (round == 2 && !refine) return;
    if (round == 1 && W.ctl->blk[5] != 0.0) return;             // [5]: round 1 was applied by the update pass; round 2 follows
    __shared__ double tsh[SMAX * SMAX];
    __shared__ double dres[MAXV];
    if (threadIdx.x < SMAX * SMAX) tsh[threadIdx.x] = W.tb[threadIdx.x];
    __syncthreads();
    double acc[SB - 1];
#pragma unroll
    for (int k = 0; k < SB - 1; ++k) acc[k] = 0.0;
    const long long n2 = n >> 1, T = (long long)gridDim.x * KTHREADS;
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n2; e += T) {
        double2 a[SB];
#pragma unroll
        for (int k = 0; k < SB; ++k) a[k] = ld_cs2(reinterpret_cast<const double2*>(w1 + k * stride) + e);
#pragma unroll
        for (int k = 1; k < SB; ++k) {
#pragma unroll
            for (int l = 0; l < k; ++l) { const double t = tsh[l * SMAX + k]; a[k].x = fma(-t, a[l].x, a[k].x); a[k].y = fma(-t, a[l].y, a[k].y); }
            reinterpret_cast<double2*>(w1 + k * stride)[e] = a[k];
            acc[k - 1] = fma(a[k].y, a[k].y, fma(a[k].x, a[k].x, acc[k - 1]));
        }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        double a[SB];
        for (int k = 0; k < SB; ++k) a[k] = w1[k * stride + n - 1];
        for (int k = 1; k < SB; ++k) { for (int l = 0; l < k; ++l) a[k] -= tsh[l * SMAX + k] * a[l]; w1[k * stride + n - 1] = a[k]; acc[k - 1] += a[k] * a[k]; }
    }
    if (!reduce_to_last<SB - 1>(acc, W, dres)) return;
    if (W.red_out) { if (threadIdx.x < SB - 1) W.red_out[threadIdx.x] = dres[threadIdx.x]; return; }
    if (round == 1 && refine) return;        // the block goes through a second round first: its columns are finished by that round's epilogue
    sstep_finish_block<SB>(W, dres, theta);
}

// Second round for an ill-conditioned block: Gram matrix of the q~ of round 1, Cholesky, coefficients of round 2, T = T2 T1.
template <int SB>
__global__ void __launch_bounds__(KTHREADS, GS_BLOCKS_PER_SM_SS) gramS_kernel(const double* __restrict__ w1, long long stride, long long n, GmresWork W)
{
    if (W.ctl->inner_stop || W.ctl->blk[4] == 0.0 || W.ctl->blk[5] != 0.0 || W.ctl->blk[6] != 0.0) return;   // ([5]: that Gram matrix came with the update pass)
    constexpr int NG = ss_ng(SB);
    __shared__ double dres[MAXV];
    double acc[NG];
#pragma unroll
    for (int p = 0; p < NG; ++p) acc[p] = 0.0;
    const long long n2 = n >> 1, T = (long long)gridDim.x * KTHREADS;
    for (long long e = blockIdx.x * (long long)KTHREADS + threadIdx.x; e < n2; e += T) {
        double2 a[SB];
#pragma unroll
        for (int k = 0; k < SB; ++k) a[k] = ld_cs2(reinterpret_cast<const double2*>(w1 + k * stride) + e);
        int p = 0;
#pragma unroll
        for (int k = 0; k < SB; ++k)
#pragma unroll
            for (int l = k; l < SB; ++l) { acc[p] = fma(a[k].y, a[l].y, fma(a[k].x, a[l].x, acc[p])); ++p; }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        int p = 0;
        for (int k = 0; k < SB; ++k) for (int l = k; l < SB; ++l) acc[p++] += w1[k * stride + n - 1] * w1[l * stride + n - 1];
    }
    if (!reduce_to_last<NG>(acc, W, dres)) return;
    if (W.red_out) { if (threadIdx.x < NG) W.red_out[threadIdx.x] = dres[threadIdx.x]; return; }
    sstep_second_round<SB>(W, dres);
}

// Cholesky of the second round's Gram matrix, T <- T2 T1 (thread 0 of one block)
template <int SB>
__device__ __forceinline__ void sstep_second_round(const GmresWork& W, const double* dres)
{
    if (threadIdx.x == 0) {
        GmresCtl* c = W.ctl;
        double t2[SB][SB], rho[SB], r00;
        int nacc = sstep_factor<SB>(dres, SS_RHO_DROP, t2, rho, r00);
        const int nacc1 = (int)c->blk[3];
        if (nacc > nacc1) nacc = nacc1;
        // T <- T2 T1 (unit upper triangular), coefficients of round 2
        double T1[SB][SB], Tn[SB][SB];
        for (int k = 0; k < SB; ++k) for (int l = 0; l < SB; ++l) T1[k][l] = W.Rb[k * SMAX + l];
        for (int k = 0; k < SB; ++k)
            for (int l = 0; l < SB; ++l) {
                double v = 0.0;
                for (int q = k; q <= l; ++q) v += ((q == k) ? 1.0 : t2[k][q]) * T1[q][l];
                Tn[k][l] = (l >= k) ? v : 0.0;
            }
        for (int k = 0; k < SB; ++k) for (int l = 0; l < SB; ++l) { W.Rb[k * SMAX + l] = Tn[k][l]; W.tb[k * SMAX + l] = t2[k][l]; }
        c->blk[3] = (double)nacc;
#ifdef SS_DEBUG
        printf("   round 2: nacc=%d rho:", nacc); for (int k = 0; k < SB; ++k) printf(" %.2e", rho[k]); printf("\n");
#endif
    }
}

// ---------------------------------------------------------------------------------------------------------
// Slab decomposition (dist.cu): the kernels above leave this rank's sums in W.red_out; after the all-reduce over the ranks these
// one-block kernels run the epilogues on the summed values `red` (every rank holds the same solver state).
//   which 0: dots (red = [SB][m + 1] raw sums of the nv = j + 1 basis vectors)   1: update pass (Gram matrix)
//         2: in-block solve (norms; round 1 or 2)                                 3: second-round Gram matrix
// ---------------------------------------------------------------------------------------------------------
template <int SB>
__global__ void __launch_bounds__(KTHREADS) sstep_epilogue_kernel(GmresWork W, int which, int nv, const double* __restrict__ red, double theta, int round)
{
    GmresCtl* c = W.ctl;
    if (c->inner_stop) return;
    __shared__ double dres[MAXV];
    __shared__ double hcol[EPI_MAX + 1], ccs[EPI_MAX], ssn[EPI_MAX];
    const int ld = c->m + 1;
    if (which == 0) {       // round = 1: the last SB of the nv vectors are the block's own slots (W^T W) and the in-block solve is predicted
        const int jp = (round == 1) ? nv - 1 - SB : -1;
        for (int ent = threadIdx.x; ent < SB * nv; ent += KTHREADS) {
            const int k = ent / nv, i = ent % nv;
            if (jp >= 0 && i > jp) { c->gram[k * SMAX + (i - jp - 1)] = red[k * ld + i]; continue; }
            const double cc = red[k * ld + i] * W.scale[i];
            W.cS[k * ld + i] = cc; W.coefS[k * ld + i] = cc * W.scale[i];
        }
        if (jp < 0) return;
        __syncthreads();
        sstep_predict<SB>(W, jp);
        return;
    }
    const bool refine = c->blk[4] != 0.0;
    if (c->blk[6] != 0.0 && which != 1) return;                              // the update pass finished the block
    if ((which == 3 || (which == 2 && round == 2)) && !refine) return;
    if ((which == 3 || (which == 2 && round == 1)) && c->blk[5] != 0.0) return;   // round 1 and its Gram matrix came with the update pass
    const int nsum = (which == 2) ? SB - 1 : ss_ng(SB);
    if (threadIdx.x < nsum) dres[threadIdx.x] = red[threadIdx.x];
    __syncthreads();
    if (which == 1) {
        if (c->blk[5] != 0.0) sstep_pred_epilogue<SB>(W, dres, theta, hcol, ccs, ssn);
        else sstep_update_epilogue<SB>(W, dres, hcol, ccs, ssn);
    }
    else if (which == 3) sstep_second_round<SB>(W, dres);
    else { if (round == 1 && refine) return; sstep_finish_block<SB>(W, dres, theta); }
}

cudaError_t launch_sstep_epilogue(GmresWork W, int which, int sb, int nv, const double* red, double theta, int round, cudaStream_t st)
{
    switch (sb) {
        case 3: sstep_epilogue_kernel<3><<<1, KTHREADS, 0, st>>>(W, which, nv, red, theta, round); break;
        case 4: sstep_epilogue_kernel<4><<<1, KTHREADS, 0, st>>>(W, which, nv, red, theta, round); break;
        case 5: sstep_epilogue_kernel<5><<<1, KTHREADS, 0, st>>>(W, which, nv, red, theta, round); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
static int ss_grid(long long n, int sm_count)
{
    const long long need = ((n >> 1) + KTHREADS - 1) / KTHREADS;
    const long long cap = (long long)sm_count * GS_BLOCKS_PER_SM_SS;
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

cudaError_t launch_dotS(const double* w1, const double* V0, long long stride, int sb, int nv, int col0, long long n, GmresWork W, int sm_count, cudaStream_t st, int jpred)
{
    if (nv < 1 || nv > SS_CH) return cudaErrorInvalidValue;
    const int grd = ss_grid(n, sm_count);
    switch (sb) {
        case 3: multi_dotS_kernel<3><<<grd, KTHREADS, 0, st>>>(w1, V0, stride, n, W, nv, col0, jpred); break;
        case 4: multi_dotS_kernel<4><<<grd, KTHREADS, 0, st>>>(w1, V0, stride, n, W, nv, col0, jpred); break;
        case 5: multi_dotS_kernel<5><<<grd, KTHREADS, 0, st>>>(w1, V0, stride, n, W, nv, col0, jpred); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_updateS(double* w1, const double* V0, long long stride, int sb, int nv, long long n, GmresWork W, int sm_count, cudaStream_t st, double theta)
{
    if (nv < 1 || nv > SS_MAXNV) return cudaErrorInvalidValue;
    const int grd = ss_grid(n, sm_count);
    switch (sb) {
        case 3: updateS_kernel<3><<<grd, KTHREADS, 0, st>>>(w1, V0, stride, n, W, nv, theta); break;
        case 4: updateS_kernel<4><<<grd, KTHREADS, 0, st>>>(w1, V0, stride, n, W, nv, theta); break;
        case 5: updateS_kernel<5><<<grd, KTHREADS, 0, st>>>(w1, V0, stride, n, W, nv, theta); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_qrS(double* w1, long long stride, int sb, long long n, GmresWork W, double theta, int round, int sm_count, cudaStream_t st)
{
    const int grd = ss_grid(n, sm_count);
    switch (sb) {
        case 3: qrS_kernel<3><<<grd, KTHREADS, 0, st>>>(w1, stride, n, W, theta, round); break;
        case 4: qrS_kernel<4><<<grd, KTHREADS, 0, st>>>(w1, stride, n, W, theta, round); break;
        case 5: qrS_kernel<5><<<grd, KTHREADS, 0, st>>>(w1, stride, n, W, theta, round); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_gramS(const double* w1, long long stride, int sb, long long n, GmresWork W, int sm_count, cudaStream_t st)
{
    const int grd = ss_grid(n, sm_count);
    switch (sb) {
        case 3: gramS_kernel<3><<<grd, KTHREADS, 0, st>>>(w1, stride, n, W); break;
        case 4: gramS_kernel<4><<<grd, KTHREADS, 0, st>>>(w1, stride, n, W); break;
        case 5: gramS_kernel<5><<<grd, KTHREADS, 0, st>>>(w1, stride, n, W); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace ark
