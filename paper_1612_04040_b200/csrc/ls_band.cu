// ls_band.cu — Step 1: tubes T (eq. 6) and N (eq. 11) as
// ascending lists of 8^3 bricks with 512-bit masks.
//
// Kernels
//   k_classify        whole-grid sweep, 32x8x8 points per CTA, 128-bit coalesced loads;
//                     T bits are assembled into brick mask words with warp REDUX (no atomics).
//   k_dilate          N words = T | shifted T | neighbour-brick faces; one thread per brick, gated by the 7 flag
//                     bytes of the brick and its face neighbours; also counts |T| and |N|.
//   k_count / k_scan_partials / k_scatter
//                     ordered stream compaction of the brick flags by a two-level prefix sum, so the
//                     lists are ascending in brick id whatever the CTA scheduling (R20).
//                     (k_scan_partials also folds the point counters and adds |T| + iters*|N| to the work counter)
//   k_gather_masks    list-ordered mask copies for ls_band_export (T: snapshot per build, N: on demand).
// Data: per-brick byte flags (nbricks B) and dense mask words (64 B per brick, written only for
// non-empty bricks) live in the ctx; the compacted lists are what the stencil kernels iterate.
#include "ls_internal.h"

namespace ls {

namespace {

constexpr int kScanThreads = 256;
constexpr int kItemsPerThread = 16;
constexpr int kScanTile = kScanThreads * kItemsPerThread;  // 4096 bricks per CTA

constexpr uint64_t COL0 = 0x0101010101010101ull;  // lx == 0 in every row
constexpr uint64_t COL7 = 0x8080808080808080ull;  // lx == 7 in every row

template <typename T> __device__ __forceinline__ T absval(T v);
template <> __device__ __forceinline__ float absval<float>(float v) { return fabsf(v); }
template <> __device__ __forceinline__ double absval<double>(double v) { return fabs(v); }

// One CTA = 32(x) x 8(y) x 8(z) points = 4 bricks in a row.  Warp w owns z-layer w; lane l owns the
// 4 consecutive x cells x4 = l&7 of row y = (l>>3) + 4h, h = 0,1.  With VEC the 4 cells are one
// 128-bit load and a warp load covers 4 full 128-byte lines.
template <typename T, bool VEC>
__global__ void __launch_bounds__(256) k_classify(const T* __restrict__ phi, Geom g, int ntx, T gamma,
                                                  uint64_t* __restrict__ tmask, uint8_t* __restrict__ flagT) {
    __shared__ uint32_t half_words[8][4][2];  // [lz][brick in tile][low/high 32 bits]
    const int tile = blockIdx.x;
    const int tx = tile % ntx;
    const int by = (tile / ntx) % g.NBy;
    const int bz = tile / (ntx * g.NBy);
    const int lane = threadIdx.x & 31, lz = threadIdx.x >> 5;
    const int k = bz * 8 + lz;
    const int x4 = lane & 7;
    const int i0 = tx * 32 + x4 * 4;
    const int q = x4 >> 1;                                  // brick of the tile this lane feeds
    const unsigned group = 0x03030303u << (2 * q);          // the 8 lanes feeding the same 32-bit half

#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int ly = (lane >> 3) + 4 * h;
        const int j = by * 8 + ly;
        unsigned bits = 0;
        if (k < g.nz && j < g.ny && i0 < g.nx) {
            const T* row = phi + g.idx(0, j, k);
            if (VEC) {  // nx % 4 == 0 here, so i0 + 3 < nx
                if (sizeof(T) == 4) {
                    const float4 v = __ldg(reinterpret_cast<const float4*>(row + i0));
                    bits = (absval<T>((T)v.x) < gamma ? 1u : 0u) | (absval<T>((T)v.y) < gamma ? 2u : 0u) |
                           (absval<T>((T)v.z) < gamma ? 4u : 0u) | (absval<T>((T)v.w) < gamma ? 8u : 0u);
                } else {
                    const double2 a = __ldg(reinterpret_cast<const double2*>(row + i0));
                    const double2 b = __ldg(reinterpret_cast<const double2*>(row + i0 + 2));
                    bits = (absval<T>((T)a.x) < gamma ? 1u : 0u) | (absval<T>((T)a.y) < gamma ? 2u : 0u) |
                           (absval<T>((T)b.x) < gamma ? 4u : 0u) | (absval<T>((T)b.y) < gamma ? 8u : 0u);
                }
            } else {
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    if (i0 + e < g.nx && absval<T>(__ldg(row + i0 + e)) < gamma) bits |= 1u << e;
            }
        }
        // bit position inside the 32-bit half: row (ly & 3), columns (x4 & 1)*4 ..
        const unsigned v = bits << ((ly & 3) * 8 + (x4 & 1) * 4);
        const unsigned r = __reduce_or_sync(group, v);
        if ((lane & 0x19) == 0) half_words[lz][q][h] = r;   // lanes 0,2,4,6: first lane of each group
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        const int qq = threadIdx.x >> 3, z = threadIdx.x & 7;
        const uint64_t word = (uint64_t)half_words[z][qq][0] | ((uint64_t)half_words[z][qq][1] << 32);
        const unsigned nz_lanes = __ballot_sync(0xffffffffu, word != 0);
        const bool brick_any = ((nz_lanes >> (qq * 8)) & 0xffu) != 0;
        const int bx = tx * 4 + qq;
        if (bx < g.NBx) {
            const int b = (bz * g.NBy + by) * g.NBx + bx;
            if (brick_any) tmask[(int64_t)b * 8 + z] = word;
            if (z == 0) flagT[b] = brick_any ? 1 : 0;
        }
    }
}

// Bits of the cells of brick (bx,by,bz), word lz, that lie inside the domain.
__device__ __forceinline__ uint64_t domain_word(const Geom& g, int bx, int by, int bz, int lz) {
    if (bz * 8 + lz >= g.nz) return 0;
    const int vx = min(8, g.nx - bx * 8), vy = min(8, g.ny - by * 8);
    const uint64_t rowbits = (1ull << vx) - 1ull;            // vx <= 8
    uint64_t w = rowbits * COL0;                             // replicate into all 8 rows
    if (vy < 8) w &= (1ull << (8 * vy)) - 1ull;
    return w;
}

// eq. 11 (R6): N = T or any in-domain face neighbour in T.  One thread per brick: 7 flag bytes decide
// whether the brick can hold N points at all (3 % of the bricks of cfg 4 can); only those touch masks.
// Also counts |T| and |N| into the accumulators of Counts (integer adds commute: order independent).
__global__ void __launch_bounds__(256) k_dilate(Geom g, const uint64_t* __restrict__ tmask,
                                                const uint8_t* __restrict__ flagT, uint64_t* __restrict__ nmask,
                                                uint8_t* __restrict__ flagN, Counts* __restrict__ counts) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned ptsT = 0, ptsN = 0;
    if (b < g.nbricks) {
        const int bx = b % g.NBx, by = (b / g.NBx) % g.NBy, bz = b / (g.NBx * g.NBy);
        const int sx = 1, sy = g.NBx, sz = g.NBx * g.NBy;
        const bool self = flagT[b] != 0;
        const bool xm = bx > 0 && flagT[b - sx], xp = bx < g.NBx - 1 && flagT[b + sx];
        const bool ym = by > 0 && flagT[b - sy], yp = by < g.NBy - 1 && flagT[b + sy];
        const bool zm = bz > 0 && flagT[b - sz], zp = bz < g.NBz - 1 && flagT[b + sz];
        bool any = false;
        if (self | xm | xp | ym | yp | zm | zp) {
            uint64_t own[8];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                ulonglong2 v = make_ulonglong2(0ull, 0ull);
                if (self) v = reinterpret_cast<const ulonglong2*>(tmask + (int64_t)b * 8)[i];
                own[2 * i] = v.x;
                own[2 * i + 1] = v.y;
            }
            const uint64_t below = zm ? tmask[(int64_t)(b - sz) * 8 + 7] : 0ull;
            const uint64_t above = zp ? tmask[(int64_t)(b + sz) * 8 + 0] : 0ull;
            const uint64_t* txm = tmask + (int64_t)(b - sx) * 8;
            const uint64_t* txp = tmask + (int64_t)(b + sx) * 8;
            const uint64_t* tym = tmask + (int64_t)(b - sy) * 8;
            const uint64_t* typ = tmask + (int64_t)(b + sy) * 8;
            uint64_t out[8];
#pragma unroll
            for (int lz = 0; lz < 8; ++lz) {
                const uint64_t w = own[lz];
                uint64_t n = w | ((w << 1) & ~COL0) | ((w >> 1) & ~COL7) | (w << 8) | (w >> 8);
                n |= lz > 0 ? own[lz - 1] : below;
                n |= lz < 7 ? own[lz + 1] : above;
                if (xm) n |= (txm[lz] >> 7) & COL0;   // their lx=7 -> our lx=0
                if (xp) n |= (txp[lz] & COL0) << 7;   // their lx=0 -> our lx=7
                if (ym) n |= tym[lz] >> 56;           // their ly=7 -> our ly=0
                if (yp) n |= (typ[lz] & 0xffull) << 56;
                n &= domain_word(g, bx, by, bz, lz);
                out[lz] = n;
                any = any || n != 0;
                ptsN += __popcll(n);
                ptsT += __popcll(w);
            }
            if (any) {
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    reinterpret_cast<ulonglong2*>(nmask + (int64_t)b * 8)[i] = make_ulonglong2(out[2 * i], out[2 * i + 1]);
            }
        }
        flagN[b] = any ? 1 : 0;
    }
    ptsT = __reduce_add_sync(0xffffffffu, ptsT);
    ptsN = __reduce_add_sync(0xffffffffu, ptsN);
    if ((threadIdx.x & 31) == 0) {
        if (ptsT) atomicAdd(&counts->acc_T, (unsigned long long)ptsT);
        if (ptsN) atomicAdd(&counts->acc_N, (unsigned long long)ptsN);
    }
}

__device__ __forceinline__ int warp_sum(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Flags of this thread's 16 consecutive bricks (arrays are padded to a multiple of kScanTile with 0).
__device__ __forceinline__ void load_flags(const uint8_t* fT, const uint8_t* fN, const uint8_t* fP, int base,
                                           uint32_t& mT, uint32_t& mN, uint32_t& mU) {
    const uint4 a = *reinterpret_cast<const uint4*>(fT + base);
    const uint4 b = *reinterpret_cast<const uint4*>(fN + base);
    const uint4 c = *reinterpret_cast<const uint4*>(fP + base);
    const uint32_t wa[4] = {a.x, a.y, a.z, a.w}, wb[4] = {b.x, b.y, b.z, b.w}, wc[4] = {c.x, c.y, c.z, c.w};
    mT = mN = mU = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const uint32_t t = (wa[i >> 2] >> ((i & 3) * 8)) & 0xffu;
        const uint32_t n = (wb[i >> 2] >> ((i & 3) * 8)) & 0xffu;
        const uint32_t p = (wc[i >> 2] >> ((i & 3) * 8)) & 0xffu;
        mT |= (t ? 1u : 0u) << i;
        mN |= (n ? 1u : 0u) << i;
        mU |= ((n | p) ? 1u : 0u) << i;
    }
}

__global__ void __launch_bounds__(kScanThreads) k_count(const uint8_t* __restrict__ fT, const uint8_t* __restrict__ fN,
                                                        const uint8_t* __restrict__ fP, int32_t* __restrict__ partials,
                                                        int npartials) {
    __shared__ int red[3][kScanThreads / 32];
    uint32_t mT, mN, mU;
    load_flags(fT, fN, fP, blockIdx.x * kScanTile + threadIdx.x * kItemsPerThread, mT, mN, mU);
    const int cT = warp_sum(__popc(mT)), cN = warp_sum(__popc(mN)), cU = warp_sum(__popc(mU));
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { red[0][w] = cT; red[1][w] = cN; red[2][w] = cU; }
    __syncthreads();
    if (threadIdx.x < 3) {
        int s = 0;
        for (int i = 0; i < kScanThreads / 32; ++i) s += red[threadIdx.x][i];
        partials[threadIdx.x * npartials + blockIdx.x] = s;
    }
}

// Exclusive scan of the per-CTA counts of each list, in place; totals go to Counts.  One CTA.
__global__ void __launch_bounds__(1024) k_scan_partials(int32_t* __restrict__ partials, int npartials,
                                                         Counts* __restrict__ counts, int iters, int count_step) {
    __shared__ int wsum[32];
    __shared__ int carry_s;
    for (int l = 0; l < 3; ++l) {
        int32_t* p = partials + l * npartials;
        if (threadIdx.x == 0) carry_s = 0;
        __syncthreads();
        for (int base = 0; base < npartials; base += 1024) {
            const int i = base + threadIdx.x;
            const int v = i < npartials ? p[i] : 0;
            int incl = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, incl, o);
                if ((threadIdx.x & 31) >= o) incl += y;
            }
            if ((threadIdx.x & 31) == 31) wsum[threadIdx.x >> 5] = incl;
            __syncthreads();
            if (threadIdx.x < 32) {
                int s = wsum[threadIdx.x];
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int y = __shfl_up_sync(0xffffffffu, s, o);
                    if (threadIdx.x >= o) s += y;
                }
                wsum[threadIdx.x] = s;  // inclusive over warps
            }
            __syncthreads();
            const int warp_off = (threadIdx.x >> 5) ? wsum[(threadIdx.x >> 5) - 1] : 0;
            const int carry = carry_s;
            if (i < npartials) p[i] = carry + warp_off + incl - v;
            __syncthreads();
            if (threadIdx.x == 0) carry_s = carry + wsum[31];
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            if (l == 0) counts->nT = carry_s;
            if (l == 1) counts->nN = carry_s;
            if (l == 2) counts->nU = carry_s;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {   // fold the point counters of this build (k_dilate has finished: stream order)
        counts->nT_pts = counts->acc_T;
        counts->nN_pts = counts->acc_N;
        counts->acc_T = 0;
        counts->acc_N = 0;
        if (count_step) {
            counts->updates += counts->nT_pts + (unsigned long long)iters * counts->nN_pts;
            counts->steps += 1;
        }
    }
}

// Ordered scatter of the brick ids (and packed positions) of the three lists.
__global__ void __launch_bounds__(kScanThreads) k_scatter(const uint8_t* __restrict__ fT, const uint8_t* __restrict__ fN,
                                                          const uint8_t* __restrict__ fP,
                                                          const int32_t* __restrict__ partials, int npartials,
                                                          BandBuffers bb, Geom g) {
    __shared__ int wtot[3][kScanThreads / 32];
    const int base = blockIdx.x * kScanTile + threadIdx.x * kItemsPerThread;
    uint32_t m[3];
    load_flags(fT, fN, fP, base, m[0], m[1], m[2]);
    int excl[3];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int l = 0; l < 3; ++l) {
        const int c = __popc(m[l]);
        int incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        if (lane == 31) wtot[l][w] = incl;
        excl[l] = incl - c;
    }
    __syncthreads();
    if ((m[0] | m[1] | m[2]) == 0) return;   // no barrier or warp collective below
#pragma unroll
    for (int l = 0; l < 3; ++l) {
        int off = partials[l * npartials + blockIdx.x];
        for (int i = 0; i < w; ++i) off += wtot[l][i];
        excl[l] += off;
    }
    int bx = base % g.NBx, by = (base / g.NBx) % g.NBy, bz = base / (g.NBx * g.NBy);
    for (int i = 0; i < kItemsPerThread; ++i) {
        const int b = base + i;
        const int pos = bx | (by << g.pos_sy) | (bz << g.pos_sz);
        if (++bx == g.NBx) { bx = 0; if (++by == g.NBy) { by = 0; ++bz; } }
        if ((m[0] >> i) & 1u) { bb.T_ids[excl[0]] = b; bb.T_pos[excl[0]++] = pos; }
        if ((m[1] >> i) & 1u) { bb.N_ids[excl[1]] = b; bb.N_pos[excl[1]++] = pos; }
        if ((m[2] >> i) & 1u) { bb.U_ids[excl[2]] = b; bb.U_pos[excl[2]++] = pos; }
    }
}

// List-ordered copies of the dense masks (ls_band_export only): one thread per (list entry, word).
__global__ void __launch_bounds__(256) k_gather_masks(const int32_t* __restrict__ ids, const int32_t* __restrict__ count_ptr,
                                                      const uint64_t* __restrict__ dense, uint64_t* __restrict__ out) {
    const int64_t n = (int64_t)*count_ptr * 8;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x)
        out[t] = dense[(int64_t)ids[t >> 3] * 8 + (t & 7)];
}

}  // namespace

template <typename T>
void launch_classify(const T* phi, const Geom& g, T gamma, const BandBuffers& bb, cudaStream_t s, int64_t* launches) {
    const int ntx = (g.NBx + 3) / 4;
    const int64_t ntiles = (int64_t)ntx * g.NBy * g.NBz;
    const bool vec = (g.nx % 4 == 0) && ((reinterpret_cast<uintptr_t>(phi) & 15) == 0);
    if (vec)
        k_classify<T, true><<<(unsigned)ntiles, 256, 0, s>>>(phi, g, ntx, gamma, bb.tmask, bb.flagT);
    else
        k_classify<T, false><<<(unsigned)ntiles, 256, 0, s>>>(phi, g, ntx, gamma, bb.tmask, bb.flagT);
    if (launches) *launches += 1;
}

void launch_dilate_compact(const Geom& g, const BandBuffers& bb, int iters, bool count_step, cudaStream_t s,
                           int64_t* launches) {
    k_dilate<<<(unsigned)((g.nbricks + 255) / 256), 256, 0, s>>>(g, bb.tmask, bb.flagT, bb.nmask, bb.flagN, bb.counts);
    k_count<<<bb.npartials, kScanThreads, 0, s>>>(bb.flagT, bb.flagN, bb.flagNprev, bb.partials, bb.npartials);
    k_scan_partials<<<1, 1024, 0, s>>>(bb.partials, bb.npartials, bb.counts, iters, count_step ? 1 : 0);
    k_scatter<<<bb.npartials, kScanThreads, 0, s>>>(bb.flagT, bb.flagN, bb.flagNprev, bb.partials, bb.npartials, bb, g);
    // Snapshot of the T masks in list order: the last reinit sweep of an incremental step overwrites the
    // dense T masks with those of phi^{n+1}, while ls_band_export reports the band of phi^n.
    k_gather_masks<<<sm_count() * 2, 256, 0, s>>>(bb.T_ids, &bb.counts->nT, bb.tmask, bb.T_masks);
    if (launches) *launches += 5;
}

void launch_gather_masks(const BandBuffers& bb, cudaStream_t s, int64_t* launches) {
    k_gather_masks<<<sm_count() * 4, 256, 0, s>>>(bb.N_ids, &bb.counts->nN, bb.nmask, bb.N_masks);
    if (launches) *launches += 1;
}

int scan_tile() { return kScanTile; }

template void launch_classify<float>(const float*, const Geom&, float, const BandBuffers&, cudaStream_t, int64_t*);
template void launch_classify<double>(const double*, const Geom&, double, const BandBuffers&, cudaStream_t, int64_t*);

}  // namespace ls
