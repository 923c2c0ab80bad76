// krylov_device.cuh — device pieces shared by krylov_kernels.cu and operator_mf.cu: deterministic two-stage reduction with the
// "last block done" scalar epilogues (Hessenberg/Givens for GMRES, rho/alpha/omega for BiCGStab).
#pragma once
#include "ark_m1_internal.h"

namespace ark {

static constexpr int KTHREADS = 256;
static constexpr int EPI_MAX = 128;      // Hessenberg columns up to this length are staged in shared memory for the Givens epilogue


__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ void hist_push(const GmresWork& W, GmresCtl* c, double r)
{
    if (c->nhist < W.caphist) W.hist[c->nhist] = (c->bnorm > 0.0) ? r / c->bnorm : r;
    c->nhist++;
}

// Column j of the Hessenberg matrix is complete: rows 0..j (raw, in hcol when staged, else already in W.H) and h_{j+1,j} = hn.
// Apply the rotations 0..j-1, form rotation j, advance the residual estimate and the stop flag (Saad 2003, Sect. 6.5.3).
// vnorm = norm of the stored (unnormalised) vector j+1; it differs from hn in the second column of a two-column step.
__device__ __forceinline__ void finish_column(const GmresWork& W, GmresCtl* c, int j, double hn, const double* hcol, const double* ccs,
                                              const double* ssn, double vnorm = -1.0)
{
    const int m = c->m;
    double* H = W.H;
    H[(j + 1) * m + j] = hn;
    if (hcol) {
        // column j, cs, sn were staged in shared memory by the whole block: the rotation chain runs on registers and
        // shared memory instead of a dependent global load/store pair per step (it was ~1 us per previous rotation)
        double carry = hcol[0];
        for (int i = 0; i < j; ++i) {
            const double nxt = hcol[i + 1];
            H[i * m + j] = ccs[i] * carry + ssn[i] * nxt;
            carry = -ssn[i] * carry + ccs[i] * nxt;
        }
        H[j * m + j] = carry;
    } else {
        for (int i = 0; i < j; ++i) {
            const double a = H[i * m + j], b = H[(i + 1) * m + j];
            H[i * m + j] = W.cs[i] * a + W.sn[i] * b;
            H[(i + 1) * m + j] = -W.sn[i] * a + W.cs[i] * b;
        }
    }
    const double a = H[j * m + j], b = H[(j + 1) * m + j];
    const double r = hypot(a, b);
    W.cs[j] = a / r; W.sn[j] = b / r;
    H[j * m + j] = r; H[(j + 1) * m + j] = 0.0;
    W.g[j + 1] = -W.sn[j] * W.g[j];
    W.g[j] = W.cs[j] * W.g[j];
    W.scale[j + 1] = 1.0 / (vnorm >= 0.0 ? vnorm : hn);
    c->j = j + 1; c->its += 1;
    c->est = fabs(W.g[j + 1]);
    hist_push(W, c, c->est);
    if (!isfinite(hn) || !isfinite(c->est)) c->nonfinite = 1;
    if (c->est <= c->target || hn == 0.0 || c->its >= c->maxit || j + 1 >= m || c->nonfinite) c->inner_stop = 1;
}

// Scalar epilogues, run by one thread after a reduction has produced d[0..nv).
__device__ __forceinline__ void epilogue(const GmresWork& W, int mode, const double* d, int nv, int col0,
                                         const double* hcol = nullptr, const double* ccs = nullptr, const double* ssn = nullptr)
{
    GmresCtl* c = W.ctl;
    const int m = c->m;
    if (mode == DOT_BNORM) {
        c->bnorm = sqrt(d[0]);
        c->target = c->est * c->bnorm;      // est holds tol until the first residual (set by begin_solve)
        if (!isfinite(c->bnorm)) c->nonfinite = 1;
    } else if (mode == DOT_RNORM) {         // true residual at the start of a cycle
        const double r = sqrt(d[0]);
        c->rnorm = r; c->est = r;
        hist_push(W, c, r);
        if (!isfinite(r)) c->nonfinite = 1;
        c->converged = (r <= c->target) ? 1 : 0;
        c->inner_stop = (c->converged || c->its >= c->maxit || c->nonfinite) ? 1 : 0;
        c->j = 0;
        W.scale[0] = 1.0 / r;
        W.g[0] = r;
        for (int k = 1; k <= m; ++k) W.g[k] = 0.0;
    } else if (mode == DOT_H || mode == DOT_H2) {   // h_i = <w, v_i>, v_i = scale_i V_i
        const int j = c->j;
        for (int k = 0; k < nv; ++k) {
            const int i = col0 + k;
            const double h = d[k] * W.scale[i];
            if (mode == DOT_H) W.H[i * m + j] = h; else W.H[i * m + j] += h;
            W.coef[i] = h * W.scale[i];
        }
    } else if (mode == BICG_ALPHA) {        // alpha = rho_new / <r^, v>
        const double rhv = d[0];
        if (rhv == 0.0 || !isfinite(rhv)) { c->inner_stop = 1; if (!isfinite(rhv)) c->nonfinite = 1; }
        else c->bs[BS_ALPHA] = c->bs[BS_RHO_NEW] / rhv;
    } else if (mode == BICG_OMEGA) {        // omega = <t, s> / <t, t>
        const double ts = d[0], tt = d[1];
        c->bs[BS_OMEGA] = (tt > 0.0) ? ts / tt : 0.0;
        c->bs[BS_RESTART] = (c->bs[BS_OMEGA] == 0.0 || !isfinite(c->bs[BS_OMEGA])) ? 1.0 : 0.0;
        if (!isfinite(c->bs[BS_OMEGA])) { c->nonfinite = 1; c->inner_stop = 1; }
    } else if (mode == BICG_RHO) {          // end of a BiCGStab iteration: rho <- rho_new, rho_new = <r^, r>, ||r||
        c->bs[BS_RHO] = c->bs[BS_RHO_NEW];
        c->bs[BS_RHO_NEW] = d[0];
        const double rn = sqrt(d[1]);
        c->bs[BS_RN] = rn; c->est = rn;
        c->its += 1;
        hist_push(W, c, rn);
        if (!isfinite(rn) || !isfinite(d[0])) c->nonfinite = 1;
        if (rn <= c->target || c->its >= c->maxit || d[0] == 0.0 || c->bs[BS_RESTART] != 0.0 || c->nonfinite) c->inner_stop = 1;
    } else if (mode == DOT_AUX0 || mode == DOT_AUX1) {
        c->aux[mode - DOT_AUX0] = sqrt(d[0]);
    } else if (mode == DOT_UPD) {           // h_{j+1,j} = ||w||
        finish_column(W, c, c->j, sqrt(d[0]), hcol, ccs, ssn);
    } else if (mode == DOT_B2) {            // two-column step: c1_i = <W1, v_i>, c2_i = <W2, v_i> of one chunk of the basis
        const int nb = nv / 2;              // d = [<W1, V_i>, i in the chunk | <W2, V_i>]
        for (int k = 0; k < nb; ++k) {
            const int i = col0 + k;
            const double a = d[k] * W.scale[i], b = d[nb + k] * W.scale[i];
            W.c1[i] = a; W.c2[i] = b;
            W.coef[i] = a * W.scale[i]; W.coef2[i] = b * W.scale[i];
        }
    } else if (mode == UPD_B2A) {           // first column: h_{.,j} = (c1, r11); the coefficient of the W2'' = W2' - (b/a) W1' pass
        const int j = c->j;
        const double a = d[0], b = d[1], r11 = sqrt(a);
        c->blk[0] = r11; c->blk[1] = b; c->blk[2] = a;
        W.coef[j + 1] = (a > 0.0) ? b / a : 0.0;
        W.Hraw[(j + 1) * c->m + j] = r11;
        finish_column(W, c, j, r11, hcol, ccs, ssn);
    } else if (mode == UPD_B2B) {           // second column (c->j is its index): rows 0..j of the raw column are staged in hcol
        const int j = c->j, m = c->m;
        const double hn = sqrt(d[0]) / c->blk[0];       // h_{j+1,j} = r22 / r11
        W.Hraw[(j + 1) * m + j] = hn;
        finish_column(W, c, j, hn, hcol, ccs, ssn, sqrt(d[0]));
    }
}

// The same deterministic two-stage reduction without an epilogue: returns true in the last block to finish, with the NV sums in
// dres (shared memory, visible to every thread of that block); false in every other block.  For kernels that run an epilogue of
// their own (krylov_sstep.cu).  NV <= MAXV.
template <int NV, int NT = KTHREADS>
__device__ __forceinline__ bool reduce_to_last(double (&acc)[NV], const GmresWork& W, double* dres)
{
    __shared__ double sh[NT / 32][MAXV];
    __shared__ bool is_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int bid = blockIdx.y * gridDim.x + blockIdx.x, nb = gridDim.x * gridDim.y;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double s = warp_sum(acc[k]);
        if (lane == 0) sh[warp][k] = s;
    }
    __syncthreads();
    if (threadIdx.x < NV) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < NT / 32; ++w) s += sh[w][threadIdx.x];
        W.partial[(size_t)bid * MAXV + threadIdx.x] = s;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicInc(&W.ctl->ticket, nb - 1);   // wraps to 0 after the last block
        is_last = (t == nb - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    for (int k = warp; k < NV; k += NT / 32) {
        double s = 0.0;
        for (unsigned int b = lane; b < nb; b += 32) s += __ldcg(&W.partial[(size_t)b * MAXV + k]);
        s = warp_sum(s);
        if (lane == 0) dres[k] = s;
    }
    __syncthreads();
    return true;
}

// Block reduction of acc[0..NV) -> partial[block][.]; the last block sums the partials in a fixed order and
// runs the epilogue.
// NT = threads per block; blocks may be a 2-D grid (linear block id).
// STAGE: the kernel may run the DOT_UPD epilogue, whose Hessenberg column is staged in shared memory.  Only the update kernel
// asks for it: the 3 KB of static shared memory cost the multi-dot kernels 15 % of their bandwidth (measured 6.60 -> 5.63 TB/s at
// 4096^2 when they carried it too), while the update kernel is a little faster with it.
template <int NV, int NT = KTHREADS, bool STAGE = false>
__device__ __forceinline__ void reduce_and_finish(double (&acc)[NV], const GmresWork& W, int mode, int col0)
{
    __shared__ double sh[NT / 32][MAXV];
    __shared__ double dres[MAXV];
    __shared__ bool is_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int bid = blockIdx.y * gridDim.x + blockIdx.x, nb = gridDim.x * gridDim.y;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double s = warp_sum(acc[k]);
        if (lane == 0) sh[warp][k] = s;
    }
    __syncthreads();
    if (threadIdx.x < NV) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < NT / 32; ++w) s += sh[w][threadIdx.x];
        W.partial[(size_t)bid * MAXV + threadIdx.x] = s;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicInc(&W.ctl->ticket, nb - 1);   // wraps to 0 after the last block
        is_last = (t == nb - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (int k = warp; k < NV; k += NT / 32) {
        double s = 0.0;
        for (unsigned int b = lane; b < nb; b += 32) s += __ldcg(&W.partial[(size_t)b * MAXV + k]);
        s = warp_sum(s);
        if (lane == 0) dres[k] = s;
    }
    if (W.red_out) {
        // domain-decomposed solve (dist.cu): this rank's sums go to W.red_out; the all-reduce over the ranks and the scalar
        // epilogue (launch_epilogue) follow as separate steps on the stream
        __syncthreads();
        if (threadIdx.x < NV) W.red_out[threadIdx.x] = dres[threadIdx.x];
        return;
    }
    if constexpr (STAGE) if (mode == DOT_UPD || mode == UPD_B2A || mode == UPD_B2B) {
        // stage column j of H (rows 0..j; row j+1 comes from the norm just reduced), cs and sn for the scalar epilogue
        __shared__ double hcol[EPI_MAX + 1], ccs[EPI_MAX], ssn[EPI_MAX];
        const int j = W.ctl->j, m = W.ctl->m;
        const bool staged = (j < EPI_MAX);       // the two-column step is only used with m <= EPI_MAX
        if (mode == DOT_UPD) {
            if (staged) for (int i = threadIdx.x; i <= j; i += NT) { hcol[i] = W.H[i * m + j]; if (i < j) { ccs[i] = W.cs[i]; ssn[i] = W.sn[i]; } }
        } else if (mode == UPD_B2A) {            // first column of the pair: rows 0..j are the c1 of the dot pass
            for (int i = threadIdx.x; i <= j; i += NT) {
                const double h = W.c1[i];
                hcol[i] = h; W.Hraw[i * m + j] = h;
                if (i < j) { ccs[i] = W.cs[i]; ssn[i] = W.sn[i]; }
            }
        } else {
            // second column (index j; the pair started at j-1).  A v_j = (W2 - sum_{i<j} c1_i A v_i) / r11 with W2 = V c2 + r12 v_j +
            // r22 v_{j+1} and A v_i = sum_{k<=i+1} Hraw_{k,i} v_k:  h_{k,j} = (c2ext_k - sum_{i>=k-1, i<j} Hraw_{k,i} c1_i) / r11, k <= j
            const double r11 = W.ctl->blk[0], r12 = W.ctl->blk[1] / r11;
            for (int k = threadIdx.x; k <= j; k += NT) {
                double sacc = (k < j) ? W.c2[k] : r12;
                for (int i = (k > 0 ? k - 1 : 0); i < j; ++i) sacc = fma(-W.Hraw[k * m + i], W.c1[i], sacc);
                const double h = sacc / r11;
                hcol[k] = h; W.Hraw[k * m + j] = h;
                if (k < j) { ccs[k] = W.cs[k]; ssn[k] = W.sn[k]; }
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) epilogue(W, mode, dres, NV, col0, staged ? hcol : nullptr, ccs, ssn);
        return;
    }
    __syncthreads();
    if (threadIdx.x == 0) epilogue(W, mode, dres, NV, col0);
}

}  // namespace ark
