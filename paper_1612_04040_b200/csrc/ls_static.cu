// ls_static.cu — ls_tube_static (include/ls_static.h): Step 1's T tube (eq. 6) with no ctx and NO allocation.
// A translation unit of its own: it shares no code with the ctx path (ls_band.cu's k_classify / k_compact / k_export_*, whose
// work memory is cudaMalloc'ed by ls_create); the kernels below are the variants of those three that keep the same work
// memory in the file-scope array g_tube_scratch.
//
//   k_tube_words    whole-grid sweep: one CTA per segment of an x-row of bricks, warp = z layer of the brick,
//                   two ballots per brick -> mask word lz (bit ly*8 + lx, ls.h) of EVERY brick, zeros included, dense by
//                   brick id, into the scratch.
//   k_tube_count    per CTA of 256 consecutive brick ids: number of bricks with a non-zero mask and their points -> scratch.
//   k_tube_scatter  ordered compaction: CTA c's base = sum of the counts of the CTAs below it (<= 256 values), block scan of
//                   the flags, ids and words to the caller's buffers in ascending brick id whatever the scheduling; CTA 0
//                   writes the totals.
// No kernel waits on another CTA (three launches instead of a grid barrier), nothing is accumulated with atomics, and every
// scratch element a call reads was written earlier by the same call: the array needs no clearing between calls.  Calls that
// overlap on the GPU race on it (ls_static.h).
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <mutex>

#include "../../include/ls_static.h"

namespace {

constexpr int kMaxBricks = LS_TUBE_STATIC_MAX_BRICKS;
constexpr int kCtaBricks = 256;                          // brick ids per CTA of k_tube_count / k_tube_scatter
constexpr int kMaxParts = kMaxBricks / kCtaBricks;       // 256 CTAs at most: one block reduce sums their counts
constexpr int kSegBricks = 32;                           // bricks of one x-row per CTA of k_tube_words
constexpr size_t kWordsOff = 0;                          // [kMaxBricks * 8] mask words, dense by brick id
constexpr size_t kPartsOff = (size_t)kMaxBricks * 8;     // [kMaxParts * 2] per CTA: T bricks, T points
constexpr size_t kScratchWords = kPartsOff + 2 * kMaxParts;
static_assert(kMaxParts == kCtaBricks, "k_tube_scatter sums the per-CTA counts with one value per thread");
static_assert(kScratchWords * 8 == LS_TUBE_STATIC_SCRATCH_BYTES, "ls_static.h states the size of the array");

// THE scratch.  In host code this name is a host-side stand-in, not a device address: only the pointer that
// cudaGetSymbolAddress returns (scratch_of_current_device) is ever passed to a kernel.
static __device__ __align__(256) unsigned long long g_tube_scratch[kScratchWords];

template <typename T> __device__ __forceinline__ T absval(T v);
template <> __device__ __forceinline__ float absval<float>(float v) { return fabsf(v); }
template <> __device__ __forceinline__ double absval<double>(double v) { return fabs(v); }

template <typename T>
__global__ void __launch_bounds__(256) k_tube_words(const T* __restrict__ phi, int nx, int ny, int nz, int NBx, int NBy,
                                                    int nseg, T gamma, unsigned long long* __restrict__ words) {
    const int seg = blockIdx.x % nseg, row = blockIdx.x / nseg;   // row = bz * NBy + by
    const int by = row % NBy, bz = row / NBy;
    const int lane = threadIdx.x & 31, lz = threadIdx.x >> 5;
    const int k = bz * 8 + lz, lx = lane & 7;
    const int b1 = min(NBx, (seg + 1) * kSegBricks);
    for (int bx = seg * kSegBricks; bx < b1; ++bx) {
        const int i = bx * 8 + lx;
        unsigned half[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {   // lane = (ly & 3) * 8 + lx of rows ly = 4h .. 4h + 3: the ballot IS the half word
            const int j = by * 8 + (lane >> 3) + 4 * h;
            bool in = false;
            if (i < nx && j < ny && k < nz) in = absval<T>(__ldg(phi + (((int64_t)k * ny + j) * nx + i))) < gamma;
            half[h] = __ballot_sync(0xffffffffu, in);
        }
        if (lane == 0) words[((int64_t)row * NBx + bx) * 8 + lz] = (unsigned long long)half[0] | ((unsigned long long)half[1] << 32);
    }
}

// Sum of v over the 256 threads of the CTA, returned to every thread.  `sh` = 8 values of shared memory.
__device__ __forceinline__ unsigned long long block_sum(unsigned long long v, unsigned long long* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();   // the previous use of sh is over
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    unsigned long long t = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) t += sh[w];
    return t;
}

__global__ void __launch_bounds__(kCtaBricks) k_tube_count(const unsigned long long* __restrict__ words, int nbricks,
                                                           unsigned long long* __restrict__ parts) {
    __shared__ unsigned long long sh[8];
    const int b = blockIdx.x * kCtaBricks + threadIdx.x;
    unsigned long long pts = 0;
    if (b < nbricks) {
#pragma unroll
        for (int w = 0; w < 8; ++w) pts += (unsigned long long)__popcll(words[(size_t)b * 8 + w]);
    }
    const unsigned long long nb = block_sum(pts != 0 ? 1ull : 0ull, sh);
    const unsigned long long np = block_sum(pts, sh);
    if (threadIdx.x == 0) {
        parts[2 * blockIdx.x] = nb;
        parts[2 * blockIdx.x + 1] = np;
    }
}

__global__ void __launch_bounds__(kCtaBricks) k_tube_scatter(const unsigned long long* __restrict__ words,
                                                             const unsigned long long* __restrict__ parts, int nbricks,
                                                             int32_t* __restrict__ T_ids, uint64_t* __restrict__ T_masks,
                                                             int64_t* __restrict__ counts) {
    __shared__ unsigned long long sh[8];
    __shared__ int warp_base[8];
    const int t = threadIdx.x, c = blockIdx.x;
    // bricks listed by the CTAs below this one (ascending ids: CTA c owns ids [256c, 256c + 256))
    const unsigned long long base = block_sum(t < c ? parts[2 * t] : 0ull, sh);
    if (c == 0) {
        const int nparts = (int)gridDim.x;
        const unsigned long long nb = block_sum(t < nparts ? parts[2 * t] : 0ull, sh);
        const unsigned long long np = block_sum(t < nparts ? parts[2 * t + 1] : 0ull, sh);
        if (t == 0) {
            counts[0] = (int64_t)np;
            counts[1] = (int64_t)nb;
        }
    }
    const int b = c * kCtaBricks + t;
    unsigned long long w[8];
    bool any = false;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        w[i] = b < nbricks ? words[(size_t)b * 8 + i] : 0ull;
        any |= w[i] != 0;
    }
    const unsigned ballot = __ballot_sync(0xffffffffu, any);
    if ((t & 31) == 0) warp_base[t >> 5] = __popc(ballot);
    __syncthreads();
    int below = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
        if (i < (t >> 5)) below += warp_base[i];
    if (any) {
        const size_t pos = (size_t)base + below + __popc(ballot & ((1u << (t & 31)) - 1u));
        T_ids[pos] = b;
#pragma unroll
        for (int i = 0; i < 8; ++i) T_masks[pos * 8 + i] = w[i];
    }
}

char g_error[256] = "";
std::mutex g_mu;
constexpr int kMaxDevices = 64;
unsigned long long* g_scratch_ptr[kMaxDevices] = {};   // device address of g_tube_scratch, per device

ls_status fail(ls_status st, const char* what, cudaError_t e) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (e != cudaSuccess)
        std::snprintf(g_error, sizeof g_error, "%s: %s", what, cudaGetErrorString(e));
    else
        std::snprintf(g_error, sizeof g_error, "%s", what);
    return st;
}

// Set-up, once per device, with that device current: the device address of the array.
ls_status scratch_of_current_device(unsigned long long** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(LS_ERR_CUDA, "ls_tube_static: cudaGetDevice", e);
    }
    if (dev < 0 || dev >= kMaxDevices) return fail(LS_ERR_CUDA, "ls_tube_static: device ordinal beyond 63", cudaSuccess);
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if (g_scratch_ptr[dev]) {
            *out = g_scratch_ptr[dev];
            return LS_OK;
        }
    }
    unsigned long long* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_tube_scratch);
    if (e != cudaSuccess || !ptr) {
        cudaGetLastError();
        return fail(LS_ERR_CUDA, "ls_tube_static: cudaGetSymbolAddress of the scratch array", e);
    }
    // load the four kernels now (lazy module loading would otherwise do it at their first launch, which may be inside a
    // stream capture)
    cudaFuncAttributes attr;
    e = cudaFuncGetAttributes(&attr, k_tube_words<float>);
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&attr, k_tube_words<double>);
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&attr, k_tube_count);
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&attr, k_tube_scatter);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(LS_ERR_CUDA, "ls_tube_static: cudaFuncGetAttributes", e);
    }
    std::lock_guard<std::mutex> lock(g_mu);
    g_scratch_ptr[dev] = ptr;
    *out = ptr;
    return LS_OK;
}

template <typename T>
ls_status run(const T* phi, int nx, int ny, int nz, int NBx, int NBy, int nbricks, T gamma, unsigned long long* scratch,
              cudaStream_t s, int32_t* T_ids, uint64_t* T_masks, int64_t* counts) {
    unsigned long long* words = scratch + kWordsOff;
    unsigned long long* parts = scratch + kPartsOff;
    const int nseg = (NBx + kSegBricks - 1) / kSegBricks;
    const int rows = nbricks / NBx;
    const int nparts = (nbricks + kCtaBricks - 1) / kCtaBricks;
    k_tube_words<T><<<(unsigned)(rows * nseg), 256, 0, s>>>(phi, nx, ny, nz, NBx, NBy, nseg, gamma, words);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(LS_ERR_CUDA, "ls_tube_static: launch of k_tube_words", e);
    k_tube_count<<<(unsigned)nparts, kCtaBricks, 0, s>>>(words, nbricks, parts);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(LS_ERR_CUDA, "ls_tube_static: launch of k_tube_count", e);
    k_tube_scatter<<<(unsigned)nparts, kCtaBricks, 0, s>>>(words, parts, nbricks, T_ids, T_masks, counts);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(LS_ERR_CUDA, "ls_tube_static: launch of k_tube_scatter", e);
    return LS_OK;
}

}  // namespace

extern "C" {

const char* ls_tube_static_error(void) { return g_error; }

ls_status ls_tube_static_setup(void) {
    unsigned long long* p = nullptr;
    return scratch_of_current_device(&p);
}

ls_status ls_tube_static(const void* phi, int32_t nx, int32_t ny, int32_t nz, ls_dtype dtype, double gamma,
                         void* cuda_stream, int32_t* T_ids, uint64_t* T_masks, int64_t* counts) {
    if (!phi || !T_ids || !T_masks || !counts) return fail(LS_ERR_ARG, "ls_tube_static: null pointer", cudaSuccess);
    if (!(gamma > 0)) return fail(LS_ERR_ARG, "ls_tube_static: gamma must be > 0", cudaSuccess);
    if (nx < 1 || ny < 1 || nz < 1) return fail(LS_ERR_DIM, "ls_tube_static: a grid dimension < 1", cudaSuccess);
    if (dtype != LS_F32 && dtype != LS_F64) return fail(LS_ERR_DTYPE, "ls_tube_static: dtype not LS_F32 / LS_F64", cudaSuccess);
    const int64_t NBx = ((int64_t)nx + 7) / 8, NBy = ((int64_t)ny + 7) / 8, NBz = ((int64_t)nz + 7) / 8;
    int64_t nbricks = NBx * NBy;                     // < 2^58: no overflow
    if (nbricks <= kMaxBricks) nbricks *= NBz;       // < 2^45
    if (nbricks > kMaxBricks) {
        std::lock_guard<std::mutex> lock(g_mu);
        std::snprintf(g_error, sizeof g_error,
                      "ls_tube_static: a %d x %d x %d grid has more 8^3 bricks than LS_TUBE_STATIC_MAX_BRICKS = %d "
                      "(the static scratch array); use ls_create + ls_build_band", nx, ny, nz, kMaxBricks);
        return LS_ERR_CAPACITY;
    }
    unsigned long long* scratch = nullptr;
    const ls_status st = scratch_of_current_device(&scratch);
    if (st != LS_OK) return st;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (dtype == LS_F32)
        return run<float>((const float*)phi, nx, ny, nz, (int)NBx, (int)NBy, (int)nbricks, (float)gamma, scratch, s, T_ids,
                          T_masks, counts);
    return run<double>((const double*)phi, nx, ny, nz, (int)NBx, (int)NBy, (int)nbricks, gamma, scratch, s, T_ids, T_masks,
                       counts);
}

}  // extern "C"
