// noalloc.cu — ark_m1_count_unrealizable_noalloc: the row-a7 guard (cells with E <= 0, cells with |F| > cE)
// for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The handle path (ark_m1_count_unrealizable, explicit_kernels.cu) keeps its two counters in memory the handle cudaMalloc'ed at
// create.  This variant takes the caller's planes and the caller's output and keeps its scratch — one partial pair per block and the
// "last block done" ticket — in a file-scope __device__ array of fixed size.  Every GPU that loads libark_m1.so holds that array
// (256 KB + 256 B) until the process exits.  Nothing here calls cudaMalloc, cudaFree or a library routine
// that allocates.
//
// Consequences of the one shared array (ark_m1.h says the same):
//  * the size is bounded: one block per NOALLOC_CHUNK cells, at most NOALLOC_MAX_BLOCKS blocks -> 67 108 864 cells (8192^2);
//  * the array keeps the previous call's contents: the ticket is cleared on the stream before every launch, the partials need no
//    clearing (every block of a launch writes its own pair before it takes a ticket);
//  * two calls that overlap on the GPU (different streams, different host threads) race on it: serialise them.
//
// In host code `noalloc_scratch` is a host-side stand-in for the device array, not a device address: the address a kernel can use
// comes from cudaGetSymbolAddress, taken once per device with that device current (scratch_of below).
#include <mutex>
#include <stdarg.h>
#include <stdio.h>
#include "ark_m1_internal.h"
#include "../../include/ark_m1.h"

namespace ark {

static constexpr int NOALLOC_THREADS = 256;
static constexpr int NOALLOC_CELLS_PER_THREAD = 16;
static constexpr int NOALLOC_CHUNK = NOALLOC_THREADS * NOALLOC_CELLS_PER_THREAD;        // cells per block
static constexpr int NOALLOC_MAX_BLOCKS = 16384;
static constexpr long long NOALLOC_MAX_CELLS = (long long)NOALLOC_MAX_BLOCKS * NOALLOC_CHUNK;
static constexpr int NOALLOC_HEADER_WORDS = 32;                                        // 256 B: word 0 is the ticket
static constexpr int NOALLOC_WORDS = NOALLOC_HEADER_WORDS + 2 * NOALLOC_MAX_BLOCKS;

// [0] ticket, [1..31] unused, then partial[block][2]
static __device__ __align__(256) unsigned long long noalloc_scratch[NOALLOC_WORDS];

// counts[0] = cells with E <= 0 (or NaN), counts[1] = cells with E > 0 and |F| > cE: the same predicate, in the same arithmetic,
// as count_unrealizable_kernel.  Block b owns cells [b CHUNK, (b + 1) CHUNK); its pair goes to scratch; the last block to finish
// adds the pairs in block order and writes the caller's output.
__global__ void __launch_bounds__(NOALLOC_THREADS) count_unrealizable_noalloc_kernel(const double* E, const double* Fx, const double* Fy, long long n,
                                                                                     double c, unsigned long long* scratch, unsigned long long* out2)
{
    __shared__ unsigned int sa[NOALLOC_THREADS / 32], sb[NOALLOC_THREADS / 32];
    __shared__ bool is_last;
    unsigned long long* partial = scratch + NOALLOC_HEADER_WORDS;
    const long long base = (long long)blockIdx.x * NOALLOC_CHUNK + threadIdx.x;
    unsigned int a = 0, b = 0;
#pragma unroll
    for (int i = 0; i < NOALLOC_CELLS_PER_THREAD; ++i) {
        const long long id = base + (long long)i * NOALLOC_THREADS;
        if (id < n) {
            const double e = E[id], fx = Fx[id], fy = Fy[id];
            if (!(e > 0.0)) ++a;
            else if (sqrt(fx * fx + fy * fy) > c * e) ++b;
        }
    }
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o); }
    if ((threadIdx.x & 31) == 0) { sa[threadIdx.x >> 5] = a; sb[threadIdx.x >> 5] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long ta = 0, tb = 0;
        for (int w = 0; w < NOALLOC_THREADS / 32; ++w) { ta += sa[w]; tb += sb[w]; }
        partial[2 * blockIdx.x] = ta; partial[2 * blockIdx.x + 1] = tb;
        __threadfence();
        const unsigned long long t = atomicAdd(&scratch[0], 1ull);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    unsigned long long ta = 0, tb = 0;
    for (unsigned int k = threadIdx.x; k < gridDim.x; k += NOALLOC_THREADS) { ta += __ldcg(&partial[2 * k]); tb += __ldcg(&partial[2 * k + 1]); }
    for (int o = 16; o > 0; o >>= 1) { ta += __shfl_down_sync(0xffffffffu, ta, o); tb += __shfl_down_sync(0xffffffffu, tb, o); }
    __shared__ unsigned long long fa[NOALLOC_THREADS / 32], fb[NOALLOC_THREADS / 32];
    if ((threadIdx.x & 31) == 0) { fa[threadIdx.x >> 5] = ta; fb[threadIdx.x >> 5] = tb; }
    __syncthreads();
    if (threadIdx.x == 0) {
        ta = tb = 0;
        for (int w = 0; w < NOALLOC_THREADS / 32; ++w) { ta += fa[w]; tb += fb[w]; }
        out2[0] = ta; out2[1] = tb;
        scratch[0] = 0;                    // leave the ticket ready (the host clears it again before the next launch)
    }
}

// ---------------------------------------------------------------------------------------------------------
// Host side.
// ---------------------------------------------------------------------------------------------------------
static constexpr int NOALLOC_MAX_DEVICES = 64;
static std::mutex noalloc_mu;
static unsigned long long* noalloc_ptr[NOALLOC_MAX_DEVICES];      // device address of noalloc_scratch, per device ordinal
static thread_local char noalloc_err[256] = "";

static int noalloc_fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(noalloc_err, sizeof noalloc_err, fmt, ap);
    va_end(ap);
    return code;
}

// Device address of the scratch array on the CURRENT device; cudaGetSymbolAddress runs once per device (it may load the module:
// call ark_m1_noalloc_setup outside a capture).
static int scratch_of(unsigned long long** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return noalloc_fail(ARK_M1_E_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e)); }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return noalloc_fail(ARK_M1_E_UNSUPPORTED, "device ordinal %d beyond the %d the table holds", dev, NOALLOC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(noalloc_mu);
    if (!noalloc_ptr[dev]) {
        unsigned long long* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, noalloc_scratch);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return noalloc_fail(ARK_M1_E_CUDA, "cudaGetSymbolAddress(noalloc_scratch): %s", cudaGetErrorString(e)); }
        noalloc_ptr[dev] = p;
    }
    *out = noalloc_ptr[dev];
    return 0;
}

}  // namespace ark

using namespace ark;

extern "C" {

int ark_m1_noalloc_setup(void)
{
    unsigned long long* p = nullptr;
    return scratch_of(&p);
}

long long ark_m1_noalloc_max_cells(void) { return NOALLOC_MAX_CELLS; }

const char* ark_m1_noalloc_last_error(void) { return noalloc_err; }

int ark_m1_count_unrealizable_noalloc(const double* E, const double* Fx, const double* Fy, long long ncells, double c,
                                      unsigned long long* counts2, void* cuda_stream)
{
    if (ncells < 0 || !counts2 || (ncells > 0 && (!E || !Fx || !Fy)))
        return noalloc_fail(ARK_M1_E_ARG, "count_unrealizable_noalloc: null pointer or negative size (ncells = %lld)", ncells);
    if (ncells > NOALLOC_MAX_CELLS)
        return noalloc_fail(ARK_M1_E_UNSUPPORTED, "count_unrealizable_noalloc: ncells = %lld exceeds the %lld cells the static scratch array covers "
                            "(use ark_m1_count_unrealizable on a handle)", ncells, NOALLOC_MAX_CELLS);
    unsigned long long* scratch = nullptr;
    if (int rc = scratch_of(&scratch)) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (ncells == 0) {
        e = cudaMemsetAsync(counts2, 0, 2 * sizeof(unsigned long long), st);
        if (e != cudaSuccess) { cudaGetLastError(); return noalloc_fail(ARK_M1_E_CUDA, "cudaMemsetAsync(counts2): %s", cudaGetErrorString(e)); }
        return 0;
    }
    e = cudaMemsetAsync(scratch, 0, NOALLOC_HEADER_WORDS * sizeof(unsigned long long), st);      // the ticket must start at zero
    if (e != cudaSuccess) { cudaGetLastError(); return noalloc_fail(ARK_M1_E_CUDA, "cudaMemsetAsync(ticket): %s", cudaGetErrorString(e)); }
    const int blocks = (int)((ncells + NOALLOC_CHUNK - 1) / NOALLOC_CHUNK);
    count_unrealizable_noalloc_kernel<<<blocks, NOALLOC_THREADS, 0, st>>>(E, Fx, Fy, ncells, c, scratch, counts2);
    e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc_fail(ARK_M1_E_CUDA, "count_unrealizable_noalloc_kernel: %s", cudaGetErrorString(e));
    return 0;
}

}  // extern "C"
