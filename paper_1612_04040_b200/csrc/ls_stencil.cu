// ls_stencil.cu — Steps 2 and 3: the first-order upwind update of eq. 3-5
// with the cut-off of eq. 7/8, the reinitialisation sweep of
// eq. 12-13 and the clamp of eq. 10.
//
// Arithmetic contract (R18, R19): everything in T, IEEE divide / square root, no FMA contraction
// (this file is compiled with -fmad=false), differences scaled by inv_dx = 1/dx, the six squared
// terms summed pairwise by axis ((x-pair + y-pair) + z-pair).  Only the gradient norm that the sign
// of F (or of d) selects is rooted: the other one is multiplied by an exact zero in eq. 3.
#include <cstdlib>

#include "ls_internal.h"
#include "ls_math.cuh"

namespace ls {

namespace {

constexpr int kBandThreads = 256;
constexpr int kTileEdge = 10;                 // 8 + one halo cell on each side
constexpr int kTileElems = kTileEdge * kTileEdge * kTileEdge;

// Stage brick (x0,y0,z0) plus its six faces into s[z][y][x] (10^3, edges/corners skipped).
// Indices are clamped to the domain: edge replicate (R3).
template <typename T>
__device__ __forceinline__ void load_halo_tile(T* __restrict__ s, const T* __restrict__ src, const Geom& g, int x0,
                                               int y0, int z0) {
    for (int e = threadIdx.x; e < kTileElems; e += kBandThreads) {
        const int x = e % kTileEdge, r = e / kTileEdge;
        const int y = r % kTileEdge, z = r / kTileEdge;
        const int on_face = (x == 0 || x == kTileEdge - 1) + (y == 0 || y == kTileEdge - 1) +
                            (z == 0 || z == kTileEdge - 1);
        if (on_face > 1) continue;
        const int i = min(max(x0 + x - 1, 0), g.nx - 1);
        const int j = min(max(y0 + y - 1, 0), g.ny - 1);
        const int k = min(max(z0 + z - 1, 0), g.nz - 1);
        s[e] = __ldg(src + g.idx(i, j, k));
    }
}

#define LS_TILE(s, lx, ly, lz) (s)[(((lz) + 1) * kTileEdge + ((ly) + 1)) * kTileEdge + ((lx) + 1)]

// Advance over a brick list.  Writes every in-domain point of each listed brick.
template <typename T>
__global__ void __launch_bounds__(kBandThreads) k_advance_band(const T* __restrict__ phi, const T* __restrict__ F,
                                                               T* __restrict__ out, Geom g, StencilParams<T> p,
                                                               const int32_t* __restrict__ ids,
                                                               const int32_t* __restrict__ count_ptr,
                                                               const uint64_t* __restrict__ list_masks,
                                                               const uint64_t* __restrict__ tmask,
                                                               const uint8_t* __restrict__ flagT) {
    __shared__ T s[kTileElems];
    const int count = *count_ptr;
    const int lx = threadIdx.x & 7, ly = (threadIdx.x >> 3) & 7, lz0 = threadIdx.x >> 6;
    for (int li = blockIdx.x; li < count; li += gridDim.x) {
        const int b = ids[li];
        const int bx = b % g.NBx, by = (b / g.NBx) % g.NBy, bz = b / (g.NBx * g.NBy);
        const int x0 = bx * 8, y0 = by * 8, z0 = bz * 8;
        load_halo_tile(s, phi, g, x0, y0, z0);
        const bool has_T = list_masks ? true : (flagT[b] != 0);
        __syncthreads();
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int lz = lz0 + 4 * h;
            const int i = x0 + lx, j = y0 + ly, k = z0 + lz;
            if (i < g.nx && j < g.ny && k < g.nz) {
                uint64_t w = 0;
                if (has_T) w = (list_masks ? list_masks : tmask)[(int64_t)b * 8 + lz];   // both dense per brick
                const T c = LS_TILE(s, lx, ly, lz);
                T v = c;
                const int64_t at = g.idx(i, j, k);
                if ((w >> (ly * 8 + lx)) & 1ull) {
                    v = advance_value<T, false>(c, LS_TILE(s, lx - 1, ly, lz), LS_TILE(s, lx + 1, ly, lz),
                                                LS_TILE(s, lx, ly - 1, lz), LS_TILE(s, lx, ly + 1, lz),
                                                LS_TILE(s, lx, ly, lz - 1), LS_TILE(s, lx, ly, lz + 1), __ldg(F + at), p);
                }
                out[at] = v;
            }
        }
        __syncthreads();
    }
}

// One reinit sweep over the N list (see launch_reinit_band in ls_internal.h).
template <typename T, bool CLAMP, bool RESIDUAL, bool EMIT_T>
__global__ void __launch_bounds__(kBandThreads) k_reinit_band(const T* __restrict__ src, T* __restrict__ dst, Geom g,
                                                              StencilParams<T> p, const int32_t* __restrict__ ids,
                                                              const int32_t* __restrict__ count_ptr,
                                                              const uint64_t* __restrict__ masks,
                                                              unsigned long long* __restrict__ residual,
                                                              uint64_t* __restrict__ tmask, uint8_t* __restrict__ flagT) {
    __shared__ T s[kTileElems];
    __shared__ uint32_t halves[8][2];
    const int count = *count_ptr;
    const int lx = threadIdx.x & 7, ly = (threadIdx.x >> 3) & 7, lz0 = threadIdx.x >> 6;
    T rmax = T(0);
    for (int li = blockIdx.x; li < count; li += gridDim.x) {
        const int b = ids[li];
        const int bx = b % g.NBx, by = (b / g.NBx) % g.NBy, bz = b / (g.NBx * g.NBy);
        const int x0 = bx * 8, y0 = by * 8, z0 = bz * 8;
        load_halo_tile(s, src, g, x0, y0, z0);
        __syncthreads();
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int lz = lz0 + 4 * h;
            const int i = x0 + lx, j = y0 + ly, k = z0 + lz;
            const uint64_t w = masks[(int64_t)b * 8 + lz];   // dense per-brick N masks
            const unsigned rowbits = (unsigned)(w >> (ly * 8)) & 0xffu;
            const bool active = (rowbits >> lx) & 1u;
            bool tbit = false;
            if (rowbits != 0 && i < g.nx && j < g.ny && k < g.nz) {
                const T c = LS_TILE(s, lx, ly, lz);
                T v = c;
                if (active) {
                    v = reinit_value<T>(c, LS_TILE(s, lx - 1, ly, lz), LS_TILE(s, lx + 1, ly, lz),
                                        LS_TILE(s, lx, ly - 1, lz), LS_TILE(s, lx, ly + 1, lz),
                                        LS_TILE(s, lx, ly, lz - 1), LS_TILE(s, lx, ly, lz + 1), p);
                    if (RESIDUAL) rmax = fmax(rmax, mag(v - c));
                }
                if (CLAMP) v = clamp_val(v, p.gamma);
                if (EMIT_T) tbit = active && mag(v) < p.gamma;
                dst[g.idx(i, j, k)] = v;
            }
            if (EMIT_T) {
                // this warp holds rows 4*(warp&1) .. +3 of layer lz: lane == bit index within the half word
                const unsigned hw = __ballot_sync(0xffffffffu, tbit);
                if ((threadIdx.x & 31) == 0) halves[lz][(threadIdx.x >> 5) & 1] = hw;
            }
        }
        __syncthreads();
        if (EMIT_T && threadIdx.x < 32) {
            uint64_t word = 0;
            if (threadIdx.x < 8) word = (uint64_t)halves[threadIdx.x][0] | ((uint64_t)halves[threadIdx.x][1] << 32);
            const bool any = __ballot_sync(0xffffffffu, word != 0) != 0;
            if (threadIdx.x < 8 && any) tmask[(int64_t)b * 8 + threadIdx.x] = word;
            if (threadIdx.x == 0) flagT[b] = any ? 1 : 0;
        }
        if (EMIT_T) __syncthreads();
    }
    if (RESIDUAL) {
        // non-negative IEEE values order like their bit patterns
        unsigned long long bits;
        if (sizeof(T) == 4) bits = (unsigned long long)__float_as_uint((float)rmax);
        else bits = (unsigned long long)__double_as_longlong((double)rmax);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long y = __shfl_xor_sync(0xffffffffu, bits, o);
            bits = y > bits ? y : bits;
        }
        if ((threadIdx.x & 31) == 0 && bits != 0) atomicMax(residual, bits);
    }
}

template <typename T>
__global__ void __launch_bounds__(kBandThreads) k_copy_clamp_band(const T* __restrict__ src, T* __restrict__ dst, Geom g,
                                                                  T gamma, const int32_t* __restrict__ ids,
                                                                  const int32_t* __restrict__ count_ptr,
                                                                  const uint64_t* __restrict__ masks) {
    const int count = *count_ptr;
    const int lx = threadIdx.x & 7, ly = (threadIdx.x >> 3) & 7, lz0 = threadIdx.x >> 6;
    for (int li = blockIdx.x; li < count; li += gridDim.x) {
        const int b = ids[li];
        const int bx = b % g.NBx, by = (b / g.NBx) % g.NBy, bz = b / (g.NBx * g.NBy);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int lz = lz0 + 4 * h;
            const int i = bx * 8 + lx, j = by * 8 + ly, k = bz * 8 + lz;
            const uint64_t w = masks[(int64_t)b * 8 + lz];   // dense per-brick N masks
            if (((w >> (ly * 8)) & 0xffull) != 0 && i < g.nx && j < g.ny && k < g.nz) {
                const int64_t at = g.idx(i, j, k);
                dst[at] = clamp_val(src[at], gamma);
            }
        }
    }
}

// Full-domain advance, c == 1 (cfg 2).  CTA = 32(x) x 8(y) columns marching over a z chunk; the
// z-neighbours rotate through registers, x/y neighbours come through L1.
constexpr int kDenseZ = 16;
template <typename T>
__global__ void __launch_bounds__(256) k_advance_dense(const T* __restrict__ phi, const T* __restrict__ F,
                                                       T* __restrict__ out, Geom g, StencilParams<T> p) {
    const int i = blockIdx.x * 32 + threadIdx.x;
    const int j = blockIdx.y * 8 + threadIdx.y;
    const int k0 = blockIdx.z * kDenseZ;
    if (i >= g.nx || j >= g.ny) return;
    const int im = max(i - 1, 0), ip = min(i + 1, g.nx - 1);
    const int jm = max(j - 1, 0), jp = min(j + 1, g.ny - 1);
    const int k1 = min(k0 + kDenseZ, g.nz);
    T zm = __ldg(phi + g.idx(i, j, max(k0 - 1, 0)));
    T c = __ldg(phi + g.idx(i, j, k0));
    for (int k = k0; k < k1; ++k) {
        const T zp = __ldg(phi + g.idx(i, j, min(k + 1, g.nz - 1)));
        const T xm = __ldg(phi + g.idx(im, j, k)), xp = __ldg(phi + g.idx(ip, j, k));
        const T ym = __ldg(phi + g.idx(i, jm, k)), yp = __ldg(phi + g.idx(i, jp, k));
        const int64_t at = g.idx(i, j, k);
        out[at] = advance_value<T, true>(c, xm, xp, ym, yp, zm, zp, __ldg(F + at), p);
        zm = c;
        c = zp;
    }
}

// fp32 full-domain advance, two x-adjacent points per lane (nx even, 8-byte aligned fields): 64-bit loads
// (a warp row = 256 contiguous bytes), x-neighbours by warp shuffle, z-neighbours rotating through
// registers, packed arithmetic (advance_dense_pair).  CTA = 64(x) x 8(y) columns marching over a z chunk.
constexpr int kDense2Z = 32;
__global__ void __launch_bounds__(256) k_advance_dense2(const float* __restrict__ phi, const float* __restrict__ F,
                                                        float* __restrict__ out, Geom g, StencilParams<float> p) {
    const int lane = threadIdx.x;
    const int i = (blockIdx.x * 32 + lane) * 2;
    const int j = blockIdx.y * 8 + threadIdx.y;
    const int k0 = blockIdx.z * kDense2Z;
    const bool live = i < g.nx && j < g.ny;   // whole-warp shuffles below: keep dead lanes in the loop
    const int ic = live ? i : 0, jc = live ? j : 0;
    const int jm = max(jc - 1, 0), jp = min(jc + 1, g.ny - 1);
    const int il = max(ic - 1, 0), ir = min(ic + 2, g.nx - 1);
    const int k1 = min(k0 + kDense2Z, g.nz);
    // row pointers advance by one z-plane per iteration: no index arithmetic inside the loop
    const int64_t plane = (int64_t)g.nx * g.ny;
    const int64_t at0 = g.idx(ic, jc, k0);
    const float* pc = phi + at0;
    const float* pym = phi + g.idx(ic, jm, k0);
    const float* pyp = phi + g.idx(ic, jp, k0);
    const float* pl = phi + g.idx(il, jc, k0);
    const float* pr = phi + g.idx(ir, jc, k0);
    const float* pf = F + at0;
    float* po = out + at0;
    const bool edge_r = lane == 31 || ic + 2 >= g.nx;
    auto ld2 = [](const float* q) { return __ldg(reinterpret_cast<const float2*>(q)); };
    float2 zm = ld2(k0 > 0 ? pc - plane : pc);
    float2 c = ld2(pc);
    for (int k = k0; k < k1; ++k) {
        const float2 zp = ld2(k + 1 < g.nz ? pc + plane : pc);
        const float2 ym = ld2(pym), yp = ld2(pyp);
        const float2 f = ld2(pf);
        float left = __shfl_up_sync(0xffffffffu, c.y, 1), right = __shfl_down_sync(0xffffffffu, c.x, 1);
        if (lane == 0) left = __ldg(pl);
        if (edge_r) right = __ldg(pr);
        const float2 u = advance_dense_pair(c, make_float2(left, c.x), make_float2(c.y, right), ym, yp, zm, zp, f, p);
        if (live) *reinterpret_cast<float2*>(po) = u;
        zm = c;
        c = zp;
        pc += plane; pym += plane; pyp += plane; pl += plane; pr += plane; pf += plane; po += plane;
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_clamp_all(T* __restrict__ a, T* __restrict__ b, int64_t n, T gamma) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        const T v = a[p];
        const T c = clamp_val(v, gamma);
        if (c != v) {
            a[p] = c;
            if (b) b[p] = c;
        }
    }
}

// 128-bit variant for fp32 fields whose size is a multiple of 4.
__global__ void __launch_bounds__(256) k_clamp_all_v4(float4* __restrict__ a, float4* __restrict__ b, int64_t n4,
                                                      float gamma) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n4; p += stride) {
        const float4 v = a[p];
        float4 c;
        c.x = clamp_val(v.x, gamma); c.y = clamp_val(v.y, gamma);
        c.z = clamp_val(v.z, gamma); c.w = clamp_val(v.w, gamma);
        if (c.x != v.x || c.y != v.y || c.z != v.z || c.w != v.w) {
            a[p] = c;
            if (b) b[p] = c;
        }
    }
}

// Device self-check of the packed two-point arithmetic (ls_math.cuh) against the scalar IEEE functions:
// random 7-point stencils (smooth band-like values, wide-exponent values, exact zeros, flat patches),
// both halves of a pair compared bit for bit.  Counts mismatching results.
__device__ __forceinline__ uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ float test_value(uint64_t r, int kind, float centre) {
    const float u = (float)(r >> 40) * (1.0f / 16777216.0f);   // [0, 1)
    switch (kind) {
        case 0: return centre + (u - 0.5f) * 0.004f;                         // smooth field, |grad| ~ 1 at dx = 1/512
        case 1: return __uint_as_float((uint32_t)r & 0xff7fffffu);           // any finite-or-not bit pattern but NaN payloads kept rare
        case 2: return 0.0f;
        case 3: return centre;                                                // flat
        default: return (u - 0.5f) * 0.03f;
    }
}
__device__ __forceinline__ bool same_bits(float a, float b) {
    return __float_as_uint(a) == __float_as_uint(b) || (a != a && b != b);
}
__global__ void __launch_bounds__(256) k_selftest_math(uint64_t seed, int64_t n, StencilParams<float> p,
                                                       unsigned long long* mismatches, float* dbg) {
    unsigned long long bad = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        // line[h][3 + d], d in {-3: zm, -2: ym, -1: xm, 0: c, 1: xp, 2: yp, 3: zp}: a "tile" with strides sy = 2, sz = 3
        float line[16], f[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint64_t r = mix64(seed + (uint64_t)(2 * i + h) * 16);
            const int mode = (int)(r & 7);
            const float c = test_value(mix64(r), (mode == 7 || mode == 3) ? 1 : (mode == 6 ? 2 : 4), 0.f);
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                const uint64_t rk = mix64(r + 1 + k);
                int kind = 0;
                if (mode == 7) kind = 1;
                else if (mode == 3) kind = 4;
                else if (mode == 5) kind = (rk & 1) ? 3 : 0;
                else if (mode == 4) kind = (rk & 3) == 0 ? 2 : 0;
                line[8 * h + k] = k == 3 ? c : test_value(rk >> 2, kind, c);
            }
            line[8 * h + 7] = 0.f;
            const uint64_t rf = mix64(r + 9);
            f[h] = (rf & 15) == 0 ? 0.f : ((float)(rf >> 40) * (1.0f / 8388608.0f) - 1.0f);
        }
        const float* a = line;
        const float* b = line + 8;
        const float r0 = reinit_value<float>(a[3], a[2], a[4], a[1], a[5], a[0], a[6], p);
        const float r1 = reinit_value<float>(b[3], b[2], b[4], b[1], b[5], b[0], b[6], p);
        const float a0 = advance_value<float, false>(a[3], a[2], a[4], a[1], a[5], a[0], a[6], f[0], p);
        const float a1 = advance_value<float, false>(b[3], b[2], b[4], b[1], b[5], b[0], b[6], f[1], p);
        const Two<float> rp = reinit_pair<float>(line, 3, 11, 2, 3, p);
        const Two<float> ap = advance_pair<float>(line, 3, 11, 2, 3, f[0], f[1], p);
        const float e0 = advance_value<float, true>(a[3], a[2], a[4], a[1], a[5], a[0], a[6], f[0], p);
        const float e1 = advance_value<float, true>(b[3], b[2], b[4], b[1], b[5], b[0], b[6], f[1], p);
        const float2 dp = advance_dense_pair(make_float2(a[3], b[3]), make_float2(a[2], b[2]), make_float2(a[4], b[4]),
                                             make_float2(a[1], b[1]), make_float2(a[5], b[5]), make_float2(a[0], b[0]),
                                             make_float2(a[6], b[6]), make_float2(f[0], f[1]), p);
        const int br = !same_bits(rp.x, r0) + !same_bits(rp.y, r1),
                  ba = !same_bits(ap.x, a0) + !same_bits(ap.y, a1) + !same_bits(dp.x, e0) + !same_bits(dp.y, e1);
        bad += br + ba;
        if (dbg && (br | ba) && atomicAdd(mismatches + 1, 1ull) == 0) {   // first failing sample, for debugging
            for (int k = 0; k < 16; ++k) dbg[k] = line[k];
            dbg[16] = f[0]; dbg[17] = f[1]; dbg[18] = r0; dbg[19] = r1; dbg[20] = rp.x; dbg[21] = rp.y;
            dbg[22] = a0; dbg[23] = a1; dbg[24] = ap.x; dbg[25] = ap.y;
        }
    }
    if (bad) atomicAdd(mismatches, bad);
}

int band_grid() { return sm_count() * 8; }

// Debug knob: LS_DISABLE_TMA=1 forces the scalar kernels (A/B timing, parity of the two paths).
bool tma_disabled() {
    static const bool off = [] { const char* e = getenv("LS_DISABLE_TMA"); return e && e[0] == '1'; }();
    return off;
}

}  // namespace

void launch_selftest_math(uint64_t seed, int64_t n, const StencilParams<float>& p, unsigned long long* mismatches,
                          float* dbg, cudaStream_t s) {
    k_selftest_math<<<sm_count() * 8, 256, 0, s>>>(seed, n, p, mismatches, dbg);
}

int sm_count() {
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
            n = 148;
    }
    return n;
}

template <typename T>
void launch_advance_band(const T* phi, const T* F, T* out, const Geom& g, const StencilParams<T>& p,
                         const BandBuffers& bb, bool use_T_list, cudaStream_t s, int64_t* launches) {
    if (!tma_disabled() && tma_usable<T>(g, phi, F, out) &&
        launch_advance_tma<T>(phi, F, out, g, p, bb, use_T_list, s, launches))
        return;
    if (use_T_list)
        k_advance_band<T><<<band_grid(), kBandThreads, 0, s>>>(phi, F, out, g, p, bb.T_ids, &bb.counts->nT, bb.tmask,
                                                               nullptr, nullptr);
    else
        k_advance_band<T><<<band_grid(), kBandThreads, 0, s>>>(phi, F, out, g, p, bb.U_ids, &bb.counts->nU, nullptr,
                                                               bb.tmask, bb.flagT);
    if (launches) *launches += 1;
}

template <typename T>
void launch_advance_dense(const T* phi, const T* F, T* out, const Geom& g, const StencilParams<T>& p, cudaStream_t s,
                          int64_t* launches) {
    dim3 block(32, 8, 1);
    if constexpr (sizeof(T) == 4) {
        const uintptr_t bits = reinterpret_cast<uintptr_t>(phi) | reinterpret_cast<uintptr_t>(F) | reinterpret_cast<uintptr_t>(out);
        if (g.nx % 2 == 0 && (bits & 7) == 0) {
            dim3 grid2((g.nx + 63) / 64, (g.ny + 7) / 8, (g.nz + kDense2Z - 1) / kDense2Z);
            k_advance_dense2<<<grid2, block, 0, s>>>(phi, F, out, g, p);
            if (launches) *launches += 1;
            return;
        }
    }
    dim3 grid((g.nx + 31) / 32, (g.ny + 7) / 8, (g.nz + kDenseZ - 1) / kDenseZ);
    k_advance_dense<T><<<grid, block, 0, s>>>(phi, F, out, g, p);
    if (launches) *launches += 1;
}

template <typename T>
void launch_reinit_band(const T* src, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                        bool clamp, unsigned long long* residual, bool emit_T, cudaStream_t s, int64_t* launches) {
    if (!tma_disabled() && tma_usable<T>(g, src, dst, nullptr) &&
        launch_reinit_tma<T>(src, dst, g, p, bb, clamp, residual, emit_T, s, launches))
        return;
    const int grid = band_grid();
    const int32_t* cnt = &bb.counts->nN;
#define LS_LAUNCH(C, R, E)                                                                                        \
    k_reinit_band<T, C, R, E><<<grid, kBandThreads, 0, s>>>(src, dst, g, p, bb.N_ids, cnt, bb.nmask, residual,   \
                                                            bb.tmask, bb.flagT)
    if (emit_T) LS_LAUNCH(true, false, true);
    else if (residual && clamp) LS_LAUNCH(true, true, false);
    else if (residual) LS_LAUNCH(false, true, false);
    else if (clamp) LS_LAUNCH(true, false, false);
    else LS_LAUNCH(false, false, false);
#undef LS_LAUNCH
    if (launches) *launches += 1;
}

template <typename T>
void launch_copy_clamp_band(const T* src, T* dst, const Geom& g, T gamma, const BandBuffers& bb, cudaStream_t s,
                            int64_t* launches) {
    k_copy_clamp_band<T><<<band_grid(), kBandThreads, 0, s>>>(src, dst, g, gamma, bb.N_ids, &bb.counts->nN, bb.nmask);
    if (launches) *launches += 1;
}

template <typename T>
void launch_clamp_all(T* a, T* b, int64_t n, T gamma, cudaStream_t s, int64_t* launches) {
    const int grid = sm_count() * 16;
    if (sizeof(T) == 4 && n % 4 == 0 && (reinterpret_cast<uintptr_t>(a) & 15) == 0 &&
        (reinterpret_cast<uintptr_t>(b) & 15) == 0) {
        k_clamp_all_v4<<<grid, 256, 0, s>>>(reinterpret_cast<float4*>(a), reinterpret_cast<float4*>(b), n / 4,
                                            (float)gamma);
    } else {
        k_clamp_all<T><<<grid, 256, 0, s>>>(a, b, n, gamma);
    }
    if (launches) *launches += 1;
}

#define LS_INSTANTIATE(T)                                                                                          \
    template void launch_advance_band<T>(const T*, const T*, T*, const Geom&, const StencilParams<T>&,            \
                                         const BandBuffers&, bool, cudaStream_t, int64_t*);                        \
    template void launch_advance_dense<T>(const T*, const T*, T*, const Geom&, const StencilParams<T>&,           \
                                          cudaStream_t, int64_t*);                                                 \
    template void launch_reinit_band<T>(const T*, T*, const Geom&, const StencilParams<T>&, const BandBuffers&,   \
                                        bool, unsigned long long*, bool, cudaStream_t, int64_t*);                  \
    template void launch_copy_clamp_band<T>(const T*, T*, const Geom&, T, const BandBuffers&, cudaStream_t,       \
                                            int64_t*);                                                             \
    template void launch_clamp_all<T>(T*, T*, int64_t, T, cudaStream_t, int64_t*);
LS_INSTANTIATE(float)
LS_INSTANTIATE(double)

}  // namespace ls
