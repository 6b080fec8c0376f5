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

enum ScalarMode { kAdvance = 0, kReinit = 1, kCopy = 2 };

struct ScalarArgs {
    const QuadEntry* qlist;
    const int32_t* count;
    const uint64_t* nmask;        // N masks of the band the list describes
    const uint64_t* tmask_in;     // kAdvance: T masks
    const uint8_t* qflagT_in;
    const uint8_t* tgate;
    uint64_t* tmask_out;          // EMIT_T
    uint8_t* qflagT_out;
    unsigned long long* residual;
};

// Scalar band kernel for grids the tile path cannot address: one CTA per brick of a listed quad and turn, one thread
// per cell of a brick layer pair.  Same arithmetic (scalar functions of ls_math.cuh), same writes:
// every N cell of the quad gets the new value (kAdvance: N cells outside T are copied).
template <typename T, int MODE, bool CLAMP, bool RESIDUAL, bool EMIT_T>
__global__ void __launch_bounds__(kBandThreads) k_band_scalar(const T* __restrict__ src, const T* __restrict__ F,
                                                              T* __restrict__ dst, Geom g, StencilParams<T> p,
                                                              ScalarArgs a) {
    __shared__ T s[kTileElems];
    __shared__ uint32_t halves[8][2];
    const int count = *a.count;
    const int lx = threadIdx.x & 7, ly = (threadIdx.x >> 3) & 7, lz0 = threadIdx.x >> 6;
    T rmax = T(0);
    // Work unit = one brick of a listed quad (4 per list entry): the grids this path serves are small or oddly shaped,
    // and a CTA that walked the four bricks of a quad one after the other made a launch four tile-load latencies long.
    for (int wi = blockIdx.x; wi < count * 4; wi += gridDim.x) {
        const int quad = a.qlist[wi >> 2].quad, j = wi & 3;
        const int qx = quad % g.NQx, rest = quad / g.NQx, by = rest % g.NBy, bz = rest / g.NBy;
        bool tvalid = false;
        if (MODE == kAdvance) tvalid = a.qflagT_in[quad] != 0 && (a.tgate == nullptr || a.tgate[quad] != 0);
        // EMIT_T: the quad's flag only says "the T masks may hold a bit" (they are all written, zeros included), so
        // the bricks of a quad need not agree on it across CTAs
        if (EMIT_T && j == 0 && threadIdx.x == 0) a.qflagT_out[quad] = 1;
        {
            const int bx = qx * 4 + j;
            const uint64_t* nw = a.nmask + (int64_t)quad * 32 + j * 8;
            uint64_t any = 0;
#pragma unroll
            for (int z = 0; z < 8; ++z) any |= nw[z];
            if (any == 0) {   // uniform over the CTA
                if (EMIT_T && threadIdx.x < 8) a.tmask_out[(int64_t)quad * 32 + j * 8 + threadIdx.x] = 0ull;
                continue;
            }
            const int x0 = bx * 8, y0 = by * 8, z0 = bz * 8;
            __syncthreads();   // the tile of the previous brick has been read
            if (MODE != kCopy) load_halo_tile(s, src, g, x0, y0, z0);
            __syncthreads();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int lz = lz0 + 4 * h;
                const int i = x0 + lx, jj = y0 + ly, k = z0 + lz;
                const bool nbit = (nw[lz] >> (ly * 8 + lx)) & 1ull;   // in-domain by construction
                bool tbit = false;
                if (nbit) {
                    const int64_t at = g.idx(i, jj, k);
                    const T c = MODE == kCopy ? src[at] : LS_TILE(s, lx, ly, lz);
                    T v = c;
                    if (MODE == kAdvance) {
                        const bool t = tvalid && ((a.tmask_in[(int64_t)quad * 32 + j * 8 + lz] >> (ly * 8 + lx)) & 1ull);
                        if (t)
                            v = advance_value<T, false>(c, LS_TILE(s, lx - 1, ly, lz), LS_TILE(s, lx + 1, ly, lz),
                                                        LS_TILE(s, lx, ly - 1, lz), LS_TILE(s, lx, ly + 1, lz),
                                                        LS_TILE(s, lx, ly, lz - 1), LS_TILE(s, lx, ly, lz + 1), __ldg(F + at), p);
                    } else if (MODE == kReinit) {
                        v = reinit_value<T>(c, LS_TILE(s, lx - 1, ly, lz), LS_TILE(s, lx + 1, ly, lz),
                                            LS_TILE(s, lx, ly - 1, lz), LS_TILE(s, lx, ly + 1, lz),
                                            LS_TILE(s, lx, ly, lz - 1), LS_TILE(s, lx, ly, lz + 1), p);
                        if (RESIDUAL) rmax = fmax(rmax, mag(v - c));
                    }
                    if (CLAMP) v = clamp_val(v, p.gamma);
                    if (EMIT_T) tbit = mag(v) < p.gamma;
                    dst[at] = v;
                }
                if (EMIT_T) {
                    // this warp holds rows 4*(warp&1) .. +3 of layer lz: lane == bit index within the half word
                    const unsigned hw = __ballot_sync(0xffffffffu, tbit);
                    if ((threadIdx.x & 31) == 0) halves[lz][(threadIdx.x >> 5) & 1] = hw;
                }
            }
            if (EMIT_T) {
                __syncthreads();
                if (threadIdx.x < 8) {
                    const uint64_t word = (uint64_t)halves[threadIdx.x][0] | ((uint64_t)halves[threadIdx.x][1] << 32);
                    a.tmask_out[(int64_t)quad * 32 + j * 8 + threadIdx.x] = word;
                }
            }
        }
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
        if ((threadIdx.x & 31) == 0 && bits != 0) atomicMax(a.residual, bits);
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
        // The item under test: cells 0,1 = the two random stencils, cells 2,3 = the same two swapped, so both
        // packed pairs and both halves see every sample; x neighbours of an item are its own cells, which the
        // scalar reference below reads the same way.
        const float* A = line;
        const float* B = line + 8;
        Item4<float> it;
        const float* src[4] = {A, B, B, A};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            it.c[e] = src[e][3]; it.ym[e] = src[e][1]; it.yp[e] = src[e][5]; it.zm[e] = src[e][0]; it.zp[e] = src[e][6];
        }
        it.xm = A[2];
        it.xp = A[4];
        const float ff[4] = {f[0], f[1], f[1], f[0]};
        float rr[4], ra[4], rd[4], pr_[4], pa_[4], pd_[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float l = it.left(e), r = it.right(e);
            rr[e] = reinit_value<float>(it.c[e], l, r, it.ym[e], it.yp[e], it.zm[e], it.zp[e], p);
            ra[e] = advance_value<float, false>(it.c[e], l, r, it.ym[e], it.yp[e], it.zm[e], it.zp[e], ff[e], p);
            rd[e] = advance_value<float, true>(it.c[e], l, r, it.ym[e], it.yp[e], it.zm[e], it.zp[e], ff[e], p);
        }
        reinit_item<float>(it, p, pr_);
        advance_item<float, false>(it, ff, p, pa_);
        advance_item<float, true>(it, ff, p, pd_);
        int br = 0, ba = 0;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            br += !same_bits(pr_[e], rr[e]);
            ba += !same_bits(pa_[e], ra[e]) + !same_bits(pd_[e], rd[e]);
        }
        bad += br + ba;
        if (dbg && (br | ba) && atomicAdd(mismatches + 1, 1ull) == 0) {   // first failing sample, for debugging
            for (int k = 0; k < 16; ++k) dbg[k] = line[k];
            dbg[16] = f[0]; dbg[17] = f[1];
            for (int e = 0; e < 4; ++e) { dbg[18 + e] = rr[e]; dbg[22 + e] = pr_[e]; }
            dbg[26] = ra[0]; dbg[27] = pa_[0]; dbg[28] = ra[1]; dbg[29] = pa_[1]; dbg[30] = rd[0]; dbg[31] = pd_[0];
        }
    }
    if (bad) atomicAdd(mismatches, bad);
}

int band_grid() { return sm_count() * 8; }

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
void launch_band_scalar(const T* src, const T* F, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                        const BandOp& op, cudaStream_t s, int64_t* launches) {
    ScalarArgs a;
    a.qlist = bb.qlist[op.list];
    a.count = &bb.counts->nQ[op.list];
    a.nmask = bb.nmask;
    a.tmask_in = bb.tmask[bb.tb];
    a.qflagT_in = bb.qflagT[bb.tb];
    a.tgate = op.tgate;
    a.tmask_out = bb.tmask[bb.tb ^ 1];
    a.qflagT_out = bb.qflagT[bb.tb ^ 1];
    a.residual = op.residual;
    const int grid = band_grid();
#define LS_LAUNCH(M, C, R, E) k_band_scalar<T, M, C, R, E><<<grid, kBandThreads, 0, s>>>(src, F, dst, g, p, a)
    if (op.advance) LS_LAUNCH(kAdvance, false, false, false);
    else if (op.copy) {
        if (op.emit_T) LS_LAUNCH(kCopy, true, false, true);
        else if (op.clamp) LS_LAUNCH(kCopy, true, false, false);
        else LS_LAUNCH(kCopy, false, false, false);
    } else if (op.emit_T) LS_LAUNCH(kReinit, true, false, true);
    else if (op.residual && op.clamp) LS_LAUNCH(kReinit, true, true, false);
    else if (op.residual) LS_LAUNCH(kReinit, false, true, false);
    else if (op.clamp) LS_LAUNCH(kReinit, true, false, false);
    else LS_LAUNCH(kReinit, false, false, false);
#undef LS_LAUNCH
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
    template void launch_band_scalar<T>(const T*, const T*, T*, const Geom&, const StencilParams<T>&,             \
                                        const BandBuffers&, const BandOp&, cudaStream_t, int64_t*);                \
    template void launch_advance_dense<T>(const T*, const T*, T*, const Geom&, const StencilParams<T>&,           \
                                          cudaStream_t, int64_t*);                                                 \
    template void launch_clamp_all<T>(T*, T*, int64_t, T, cudaStream_t, int64_t*);
LS_INSTANTIATE(float)
LS_INSTANTIATE(double)

}  // namespace ls
