// pipe_rates.cu — self-test that MEASURES the instruction-issue rates the explicit and assembly kernels are bound by
// (ark_m1_fp64_issue_rate, include/ark_m1.h).  The "alu" roofline of bench.py (fp64 instructions per second) and the pipe
// facts quoted in DESIGN.md section 6 come from this routine, run on the box that runs the bench.
//
// Method: every thread carries K independent dependency chains of one instruction kind and runs them for `iters` trips;
// a block times itself with clock64() between two barriers.  Throughput runs fill every SM with 2 blocks of 512 threads
// (8 warps per sub-partition, K = 8 chains each: far more independent work than any pipe latency); the latency run is one
// warp with one chain.  The operands come from kernel arguments, so nothing folds at compile time, and the results are
// summed into a sink the host never reads.
#include <cuda_runtime.h>
#include "ark_m1_internal.h"
#include "../../include/ark_m1.h"

namespace ark {

enum { OP_DFMA = 0, OP_DADD, OP_DMUL, OP_DMAX, OP_IMAD, OP_FFMA, OP_DFMA_IMAD, OP_DFMA_FFMA, OP_SHFL, OP_KINDS };

template <int OP, int K>
__global__ void __launch_bounds__(512) rate_kernel(int iters, double a, double b, int ia, long long* __restrict__ cycles, double* __restrict__ sink)
{
    double x[K]; int n[K]; float s[K];
#pragma unroll
    for (int k = 0; k < K; ++k) { x[k] = a + 1e-3 * (threadIdx.x + k); n[k] = ia + (int)threadIdx.x + k; s[k] = (float)x[k]; }
    const float fa = (float)a, fb = (float)b;
    __syncthreads();
    const long long t0 = clock64();
    // the trip is unrolled 8 times for one chain and 4 times for eight, so that the loop's own add/compare/branch is < 10 % of the stream
#pragma unroll (K == 1 ? 8 : 4)
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (OP == OP_DFMA || OP == OP_DFMA_IMAD || OP == OP_DFMA_FFMA) x[k] = fma(x[k], a, b);
            if (OP == OP_DADD) x[k] = x[k] + b;
            if (OP == OP_DMUL) x[k] = x[k] * a;
            if (OP == OP_DMAX) x[k] = dmax_sel(x[k], b) ;      // the compare+select max of the hot kernels (DSETP + 2 SEL)
            if (OP == OP_IMAD || OP == OP_DFMA_IMAD) n[k] = n[k] * ia + 12345;
            if (OP == OP_FFMA || OP == OP_DFMA_FFMA) s[k] = fmaf(s[k], fa, fb);
            if (OP == OP_SHFL) x[k] = __shfl_down_sync(0xffffffffu, x[k], 1);
        }
        if (OP == OP_DMAX) { const double t = b; b = a; a = t; }     // alternate the bound so that the select is not invariant
    }
    __syncthreads();
    const long long t1 = clock64();
    double acc = 0.0;
#pragma unroll
    for (int k = 0; k < K; ++k) acc += x[k] + (double)n[k] + (double)s[k];
    if (acc == 123.456) sink[0] = acc;                   // never true in practice; keeps the chains alive
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int OP, int K>
static cudaError_t run_rate(int blocks, int threads, int iters, long long* dcycles, double* dsink, double* mean_cycles, cudaStream_t st)
{
    rate_kernel<OP, K><<<blocks, threads, 0, st>>>(iters, 1.0000001, 1e-9, 3, dcycles, dsink);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    static long long host[4096];
    e = cudaMemcpyAsync(host, dcycles, sizeof(long long) * blocks, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return e;
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    double sum = 0.0;
    for (int k = 0; k < blocks; ++k) sum += (double)host[k];
    *mean_cycles = sum / blocks;
    return cudaSuccess;
}

}  // namespace ark

using namespace ark;

extern "C" int ark_m1_fp64_issue_rate(double* out, int cap)
{
    if (!out || cap < 12) return ARK_M1_E_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return ARK_M1_E_CUDA; }
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int BPS = 2, NT = 512, K = 8, iters = 4096;
    const int blocks = sms * BPS;
    if (blocks > 4096) return ARK_M1_E_UNSUPPORTED;
    long long* dcyc = nullptr; double* dsink = nullptr;
    if (cudaMalloc((void**)&dcyc, sizeof(long long) * blocks) != cudaSuccess || cudaMalloc((void**)&dsink, sizeof(double)) != cudaSuccess) {
        cudaGetLastError(); cudaFree(dcyc); return ARK_M1_E_ALLOC;
    }
    cudaError_t e = cudaSuccess;
    double cyc = 0.0;
    const double work = (double)BPS * NT * K * iters;       // lane-instructions per SM of one kind
    // warm-up (clocks up), then the timed kinds
#define ARK_RATE(OP, slot, perop)                                                                        \
    if (e == cudaSuccess) { e = run_rate<OP, K>(blocks, NT, iters, dcyc, dsink, &cyc, 0); out[slot] = (perop) ? work / cyc : cyc / ((double)BPS * (NT / 32) / 4.0 * K * iters); }
    ARK_RATE(OP_DFMA, 0, 1)
    ARK_RATE(OP_DFMA, 0, 1)            /* out[0]: DFMA lanes per clock per SM */
    ARK_RATE(OP_DADD, 2, 1)            /* out[2]: DADD */
    ARK_RATE(OP_DMUL, 3, 1)            /* out[3]: DMUL */
    ARK_RATE(OP_DMAX, 4, 1)            /* out[4]: compare+select max (per max) */
    ARK_RATE(OP_IMAD, 5, 1)            /* out[5]: IMAD */
    ARK_RATE(OP_FFMA, 6, 1)            /* out[6]: FFMA */
    ARK_RATE(OP_DFMA_IMAD, 7, 0)       /* out[7]: issue cycles per (DFMA + IMAD) pair per warp per sub-partition */
    ARK_RATE(OP_DFMA_FFMA, 8, 0)       /* out[8]: the same for (DFMA + FFMA) */
    ARK_RATE(OP_SHFL, 9, 1)            /* out[9]: 64-bit shuffles (two SHFL.32 each), lanes per clock per SM */
#undef ARK_RATE
    // out[1]: dependent-issue latency of DFMA (one warp, one chain)
    if (e == cudaSuccess) { e = run_rate<OP_DFMA, 1>(1, 32, iters, dcyc, dsink, &cyc, 0); out[1] = cyc / iters; }
    // out[10]: SM clock during the test, from a timed DFMA run: cycles / elapsed time
    if (e == cudaSuccess) {
        cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
        cudaEventRecord(a, 0);
        e = run_rate<OP_DFMA, K>(blocks, NT, 8 * iters, dcyc, dsink, &cyc, 0);
        cudaEventRecord(b, 0); cudaEventSynchronize(b);
        float ms = 0.f; cudaEventElapsedTime(&ms, a, b);
        out[10] = (ms > 0.f) ? cyc / (ms * 1e3) : 0.0;      // MHz (the launch overhead of a ~1 ms kernel is < 1 %)
        cudaEventDestroy(a); cudaEventDestroy(b);
    }
    out[11] = (double)sms;
    cudaFree(dcyc); cudaFree(dsink);
    if (e != cudaSuccess) { cudaGetLastError(); return ARK_M1_E_CUDA; }
    return 12;
}
