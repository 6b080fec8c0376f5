// ls_tma.cu — the band kernels of Steps 2 and 3 as persistent, TMA-fed pipelines.
//
// Data flow per brick (8^3 points of a listed brick plus its one-cell halo):
//   producer (thread 0)  one cp.async.bulk.tensor.3d box load of the halo tile straight from the dense
//                        x-fastest field into shared memory, plus the brick's 64-byte
//                        mask (and, for Advance, the 8^3 box of F), all completing on one mbarrier;
//                        kStages bricks are in flight per CTA
//   consumers (8 warps)  wait on the mbarrier; replicate edge values into out-of-domain halo cells
//                        (R3; TMA zero-fills them); compact the brick's active points into a list with
//                        ballot/popc ranks so warps run full; evaluate eq. 3-8 / eq. 12-13 once per
//                        active point from the tile; write results back into the tile; store whole
//                        32-byte rows with 128-bit stores.
// The arithmetic is that of ls_math.cuh (IEEE, no FMA contraction): results are bit-identical to the
// scalar kernels of ls_stencil.cu, which remain the path for grids TMA cannot address
// (nx*sizeof(T) not a multiple of 16, or unaligned fields).
#include <cuda.h>

#include "ls_internal.h"
#include "ls_math.cuh"

namespace ls {

namespace {

constexpr int kThreads = 256;
constexpr int kStages = 3;
constexpr int kPY = 10;   // tile extent in y and z: 8 + one halo cell on each side

template <typename T> struct TileCfg;
// TMA needs every box row to start on a 16-byte boundary of the field and to span a multiple of 16
// bytes (an unaligned start coordinate faults with "illegal instruction" on sm_100a): fp32 loads 16
// cells starting four left of the brick, fp64 loads 12 cells starting two left.
template <> struct TileCfg<float> { static constexpr int XOFF = 4, PX = 16; };
template <> struct TileCfg<double> { static constexpr int XOFF = 2, PX = 12; };

constexpr int round128(int x) { return (x + 127) / 128 * 128; }

// One pipeline stage in shared memory: [halo tile][F brick (Advance only)][mask 64 B][header 64 B].
template <typename T, bool WITH_F>
struct Stage {
    static constexpr int PX = TileCfg<T>::PX;
    static constexpr int XOFF = TileCfg<T>::XOFF;
    static constexpr int ELEMS = PX * kPY * kPY;
    static constexpr int TILE_BYTES = ELEMS * (int)sizeof(T);
    static constexpr int F_BYTES = 512 * (int)sizeof(T);
    static constexpr int OFF_F = round128(TILE_BYTES);
    static constexpr int OFF_MASK = OFF_F + (WITH_F ? F_BYTES : 0);
    static constexpr int OFF_HDR = OFF_MASK + 64;
    static constexpr int BYTES = OFF_HDR + 64;
    static_assert(BYTES % 128 == 0, "stages must keep 128-byte alignment");
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LS_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LS_DONE;\n"
        "bra LS_WAIT;\n"
        "LS_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z)
        : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

struct BrickPos {
    int b, x0, y0, z0;
};
__device__ __forceinline__ BrickPos brick_pos(const Geom& g, int b) {
    BrickPos q;
    q.b = b;
    const int bx = b % g.NBx, r = b / g.NBx;
    q.x0 = bx * 8;
    q.y0 = (r % g.NBy) * 8;
    q.z0 = (r / g.NBy) * 8;
    return q;
}

// R3: TMA zero-fills cells outside the domain; give them the value of the nearest in-domain cell
// (edge replicate).  Sources are in-domain cells, destinations are not: no ordering needed inside.
template <typename T, int PX, int XOFF>
__device__ __forceinline__ void patch_boundary(T* tile, const Geom& g, const BrickPos& q) {
    const bool edge = q.x0 == 0 || q.y0 == 0 || q.z0 == 0 || q.x0 + 8 >= g.nx || q.y0 + 8 >= g.ny || q.z0 + 8 >= g.nz;
    if (!edge) return;   // uniform over the CTA
    const int ox = q.x0 - XOFF, oy = q.y0 - 1, oz = q.z0 - 1;
    for (int e = threadIdx.x; e < PX * kPY * kPY; e += kThreads) {
        const int x = e % PX, r = e / PX, y = r % kPY, z = r / kPY;
        const int gx = ox + x, gy = oy + y, gz = oz + z;
        const int cx = min(max(gx, 0), g.nx - 1), cy = min(max(gy, 0), g.ny - 1), cz = min(max(gz, 0), g.nz - 1);
        if (cx != gx || cy != gy || cz != gz) {
            const int sx = cx - ox, sy = cy - oy, sz = cz - oz;
            if (sx >= 0 && sx < PX && sy < kPY && sz < kPY) tile[e] = tile[(sz * kPY + sy) * PX + sx];
        }
    }
    __syncthreads();
}

// Compact the set bits of the brick mask into `list` (tile offsets of the active points, ascending
// point order) and return their number.  Warp w owns mask word w (layer lz = w): lane l holds bit l of
// the low half (row l>>3) and of the high half (row 4 + (l>>3)).
template <int PX, int XOFF>
__device__ __forceinline__ int build_list(const uint64_t* mk, uint16_t* list, uint32_t& lo, uint32_t& hi, int& off_lo) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint64_t word = mk[w];
    lo = (uint32_t)word;
    hi = (uint32_t)(word >> 32);
    const int pc = lane < 8 ? __popcll(mk[lane]) : 0;
    int incl = pc;
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 7);
    const int base = __shfl_sync(0xffffffffu, incl - pc, w);
    const uint32_t lt = (1u << lane) - 1u;
    off_lo = ((w + 1) * kPY + (lane >> 3) + 1) * PX + (lane & 7) + XOFF;
    if ((lo >> lane) & 1u) list[base + __popc(lo & lt)] = (uint16_t)off_lo;
    if ((hi >> lane) & 1u) list[base + __popc(lo) + __popc(hi & lt)] = (uint16_t)(off_lo + 4 * PX);
    return total;
}

// Store rows of the brick from the tile to dst with 128-bit stores.  A row (8 cells, 32 B in fp32)
// is written if `all_rows` or it holds a mask bit, and lies inside the domain.
template <typename T, int PX, int XOFF>
__device__ __forceinline__ void store_rows(const T* tile, const uint64_t* mk, bool all_rows, T* __restrict__ dst,
                                           const Geom& g, const BrickPos& q) {
    constexpr int VEC = 16 / (int)sizeof(T);   // cells per 128-bit store
    constexpr int PARTS = 8 / VEC;             // stores per row
    const int t = threadIdx.x;
    if (t >= 64 * PARTS) return;
    const int row = t / PARTS, part = t % PARTS;
    const int lz = row >> 3, ly = row & 7;
    const bool want = all_rows || ((mk[lz] >> (8 * ly)) & 0xffull) != 0;
    const int i = q.x0 + part * VEC, j = q.y0 + ly, k = q.z0 + lz;
    if (!want || i >= g.nx || j >= g.ny || k >= g.nz) return;   // nx % VEC == 0: a part is all in or all out
    const T* s = tile + ((lz + 1) * kPY + (ly + 1)) * PX + XOFF + part * VEC;
    T* d = dst + g.idx(i, j, k);
    *reinterpret_cast<int4*>(d) = *reinterpret_cast<const int4*>(s);   // XOFF*sizeof(T) == 16: aligned
}

// ---------------------------------------------------------------------------------------------
// Step 3: one reinitialisation sweep over the N list (eq. 12-13), see launch_reinit_band.
// ---------------------------------------------------------------------------------------------
template <typename T, bool CLAMP, bool RESIDUAL, bool EMIT_T>
__global__ void __launch_bounds__(kThreads, 6)
k_reinit_tma(const __grid_constant__ CUtensorMap tm_src, T* __restrict__ dst, Geom g, StencilParams<T> p,
             const int32_t* __restrict__ ids, const int32_t* __restrict__ count_ptr,
             const uint64_t* __restrict__ masks, unsigned long long* __restrict__ residual,
             uint64_t* __restrict__ tmask, uint8_t* __restrict__ flagT) {
    using S = Stage<T, false>;
    constexpr int PX = S::PX, XOFF = S::XOFF;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint64_t full[kStages];
    __shared__ uint16_t list[512];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int count = *count_ptr;
    const int G = gridDim.x;
    const int mine = (int)blockIdx.x < count ? (count - (int)blockIdx.x + G - 1) / G : 0;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        fence_barrier_init();
    }
    __syncthreads();

    auto issue = [&](int n, int b) {   // thread 0: start the loads of my n-th brick (list index li, id b)
        const int li = blockIdx.x + n * G;
        unsigned char* st = smem + (n % kStages) * S::BYTES;
        uint64_t* bar = &full[n % kStages];
        const BrickPos q = brick_pos(g, b);
        *reinterpret_cast<int*>(st + S::OFF_HDR) = b;
        mbar_expect_tx(bar, S::TILE_BYTES + 64);
        tma_load_3d(st, &tm_src, bar, q.x0 - XOFF, q.y0 - 1, q.z0 - 1);
        bulk_load(st + S::OFF_MASK, masks + (int64_t)li * 8, 64, bar);
    };
    int b_next = 0;   // id of my brick number (n + kStages - 1), prefetched one iteration ahead
    if (tid == 0) {
        for (int n = 0; n < kStages - 1 && n < mine; ++n) issue(n, ids[blockIdx.x + n * G]);
        if (kStages - 1 < mine) b_next = ids[blockIdx.x + (kStages - 1) * G];
    }

    T rmax = T(0);
    for (int n = 0; n < mine; ++n) {
        if (tid == 0 && n + kStages - 1 < mine) {
            issue(n + kStages - 1, b_next);
            if (n + kStages < mine) b_next = ids[blockIdx.x + (n + kStages) * G];
        }
        unsigned char* st = smem + (n % kStages) * S::BYTES;
        T* tile = reinterpret_cast<T*>(st);
        const uint64_t* mk = reinterpret_cast<const uint64_t*>(st + S::OFF_MASK);
        mbar_wait(&full[n % kStages], (uint32_t)((n / kStages) & 1));
        const BrickPos q = brick_pos(g, *reinterpret_cast<const int*>(st + S::OFF_HDR));
        patch_boundary<T, PX, XOFF>(tile, g, q);

        uint32_t lo, hi;
        int off_lo;
        const int total = build_list<PX, XOFF>(mk, list, lo, hi, off_lo);
        __syncthreads();

        T v[2];
        int off[2];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int e = tid + r * kThreads;
            off[r] = -1;
            if (e < total) {
                const int o = list[e];
                off[r] = o;
                const T c = tile[o];
                T u = reinit_value<T>(c, tile[o - 1], tile[o + 1], tile[o - PX], tile[o + PX], tile[o - kPY * PX],
                                      tile[o + kPY * PX], p);
                if (RESIDUAL) rmax = fmax(rmax, mag(u - c));
                if (CLAMP) u = clamp_val(u, p.gamma);
                v[r] = u;
            }
        }
        __syncthreads();   // every neighbour read of iteration k is done: write iteration k+1 in place
#pragma unroll
        for (int r = 0; r < 2; ++r)
            if (off[r] >= 0) tile[off[r]] = v[r];
        fence_proxy_async();   // the next TMA load into this stage must order after these generic writes
        __syncthreads();

        store_rows<T, PX, XOFF>(tile, mk, false, dst, g, q);
        if (EMIT_T) {
            // T mask of phi^{n+1} = clamp(d) on this brick: T^{n+1} is a subset of N^n
            const bool tl = ((lo >> lane) & 1u) && mag(tile[off_lo]) < p.gamma;
            const bool th = ((hi >> lane) & 1u) && mag(tile[off_lo + 4 * PX]) < p.gamma;
            const uint32_t bl = __ballot_sync(0xffffffffu, tl), bh = __ballot_sync(0xffffffffu, th);
            const uint64_t word = (uint64_t)bl | ((uint64_t)bh << 32);
            if (lane == 0) tmask[(int64_t)q.b * 8 + w] = word;
            const int any = __syncthreads_or(word != 0);
            if (tid == 0) flagT[q.b] = any ? 1 : 0;
        } else {
            __syncthreads();   // stage is free for the producer
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
        if (lane == 0 && bits != 0) atomicMax(residual, bits);
    }
}

// ---------------------------------------------------------------------------------------------
// Step 2: Advance (eq. 3 with eq. 8) over a brick list; writes every in-domain point of each brick.
//   dense_tmask != null: U list, T masks from the dense per-brick arrays (bricks without T are copied)
//   dense_tmask == null: T list with its list-ordered masks
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(kThreads, 5)
k_advance_tma(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_F,
              T* __restrict__ out, Geom g, StencilParams<T> p, const int32_t* __restrict__ ids,
              const int32_t* __restrict__ count_ptr, const uint64_t* __restrict__ list_masks,
              const uint64_t* __restrict__ dense_tmask, const uint8_t* __restrict__ flagT) {
    using S = Stage<T, true>;
    constexpr int PX = S::PX, XOFF = S::XOFF;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint64_t full[kStages];
    __shared__ uint16_t list[512];
    const int tid = threadIdx.x;
    const int count = *count_ptr;
    const int G = gridDim.x;
    const int mine = (int)blockIdx.x < count ? (count - (int)blockIdx.x + G - 1) / G : 0;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        fence_barrier_init();
    }
    __syncthreads();

    auto issue = [&](int n, int b, bool has_T) {
        const int li = blockIdx.x + n * G;
        unsigned char* st = smem + (n % kStages) * S::BYTES;
        uint64_t* bar = &full[n % kStages];
        const BrickPos q = brick_pos(g, b);
        int* hdr = reinterpret_cast<int*>(st + S::OFF_HDR);
        hdr[0] = b;
        hdr[1] = has_T ? 1 : 0;
        mbar_expect_tx(bar, has_T ? S::TILE_BYTES + S::F_BYTES + 64 : S::TILE_BYTES);
        tma_load_3d(st, &tm_phi, bar, q.x0 - XOFF, q.y0 - 1, q.z0 - 1);
        if (has_T) {
            tma_load_3d(st + S::OFF_F, &tm_F, bar, q.x0, q.y0, q.z0);
            const uint64_t* m = dense_tmask ? dense_tmask + (int64_t)b * 8 : list_masks + (int64_t)li * 8;
            bulk_load(st + S::OFF_MASK, m, 64, bar);
        }
    };
    auto fetch = [&](int n, int& b, bool& has_T) {
        b = ids[blockIdx.x + n * G];
        has_T = dense_tmask ? flagT[b] != 0 : true;
    };
    int b_next = 0;
    bool t_next = false;
    if (tid == 0) {
        for (int n = 0; n < kStages - 1 && n < mine; ++n) {
            int b;
            bool h;
            fetch(n, b, h);
            issue(n, b, h);
        }
        if (kStages - 1 < mine) fetch(kStages - 1, b_next, t_next);
    }

    for (int n = 0; n < mine; ++n) {
        if (tid == 0 && n + kStages - 1 < mine) {
            issue(n + kStages - 1, b_next, t_next);
            if (n + kStages < mine) fetch(n + kStages, b_next, t_next);
        }
        unsigned char* st = smem + (n % kStages) * S::BYTES;
        T* tile = reinterpret_cast<T*>(st);
        const T* Fb = reinterpret_cast<const T*>(st + S::OFF_F);
        const uint64_t* mk = reinterpret_cast<const uint64_t*>(st + S::OFF_MASK);
        mbar_wait(&full[n % kStages], (uint32_t)((n / kStages) & 1));
        const int* hdr = reinterpret_cast<const int*>(st + S::OFF_HDR);
        const BrickPos q = brick_pos(g, hdr[0]);
        const bool has_T = hdr[1] != 0;
        patch_boundary<T, PX, XOFF>(tile, g, q);

        if (has_T) {   // uniform over the CTA
            uint32_t lo, hi;
            int off_lo;
            const int total = build_list<PX, XOFF>(mk, list, lo, hi, off_lo);
            __syncthreads();
            T v[2];
            int off[2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int e = tid + r * kThreads;
                off[r] = -1;
                if (e < total) {
                    const int o = list[e];
                    off[r] = o;
                    // tile offset -> brick-local (lx, ly, lz) -> index into the dense 8^3 F box
                    const int x = o % PX - XOFF, rr = o / PX, y = rr % kPY - 1, z = rr / kPY - 1;
                    const T f = Fb[(z * 8 + y) * 8 + x];
                    v[r] = advance_value<T, false>(tile[o], tile[o - 1], tile[o + 1], tile[o - PX], tile[o + PX],
                                                   tile[o - kPY * PX], tile[o + kPY * PX], f, p);
                }
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 2; ++r)
                if (off[r] >= 0) tile[off[r]] = v[r];
            fence_proxy_async();
            __syncthreads();
        }
        store_rows<T, PX, XOFF>(tile, mk, true, out, g, q);
        __syncthreads();
    }
}

int tma_grid(int ctas_per_sm) { return sm_count() * ctas_per_sm; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
            qr == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        else
            cudaGetLastError();
    }
    return fn;
}

// Tensor map of a dense nx*ny*nz field with an (bx, by, bz) box; zero fill outside the domain.
template <typename T>
bool make_map(CUtensorMap* m, const void* field, const Geom& g, int bx, int by, int bz) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz};
    const cuuint64_t strides[2] = {(cuuint64_t)g.nx * sizeof(T), (cuuint64_t)g.nx * g.ny * sizeof(T)};
    const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz};
    const cuuint32_t es[3] = {1, 1, 1};
    const CUtensorMapDataType dt = sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    return fn(m, dt, 3, const_cast<void*>(field), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <typename K>
void prefer_smem(K kernel) {
    cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

}  // namespace

template <typename T>
bool tma_usable(const Geom& g, const void* a, const void* b, const void* c) {
    if (((size_t)g.nx * sizeof(T)) % 16 != 0) return false;
    if (((size_t)g.nx * g.ny * sizeof(T)) >= ((size_t)1 << 40)) return false;
    const uintptr_t bits = reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(c);
    return (bits & 15) == 0 && encode_fn() != nullptr;
}

template <typename T>
bool launch_reinit_tma(const T* src, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                       bool clamp, unsigned long long* residual, bool emit_T, cudaStream_t s, int64_t* launches) {
    using S = Stage<T, false>;
    CUtensorMap tm;
    if (!make_map<T>(&tm, src, g, S::PX, kPY, kPY)) return false;
    const int grid = tma_grid(6);
    const size_t shm = (size_t)kStages * S::BYTES;
    const int32_t* cnt = &bb.counts->nN;
#define LS_LAUNCH(C, R, E)                                                                                       \
    do {                                                                                                         \
        static bool once = (prefer_smem(k_reinit_tma<T, C, R, E>), true);                                        \
        (void)once;                                                                                              \
        k_reinit_tma<T, C, R, E><<<grid, kThreads, shm, s>>>(tm, dst, g, p, bb.N_ids, cnt, bb.N_masks, residual, \
                                                             bb.tmask, bb.flagT);                                \
    } while (0)
    if (emit_T) LS_LAUNCH(true, false, true);
    else if (residual && clamp) LS_LAUNCH(true, true, false);
    else if (residual) LS_LAUNCH(false, true, false);
    else if (clamp) LS_LAUNCH(true, false, false);
    else LS_LAUNCH(false, false, false);
#undef LS_LAUNCH
    if (launches) *launches += 1;
    return true;
}

template <typename T>
bool launch_advance_tma(const T* phi, const T* F, T* out, const Geom& g, const StencilParams<T>& p,
                        const BandBuffers& bb, bool use_T_list, cudaStream_t s, int64_t* launches) {
    using S = Stage<T, true>;
    CUtensorMap tm_phi, tm_F;
    if (!make_map<T>(&tm_phi, phi, g, S::PX, kPY, kPY) || !make_map<T>(&tm_F, F, g, 8, 8, 8)) return false;
    static bool once = (prefer_smem(k_advance_tma<T>), true);
    (void)once;
    const int grid = tma_grid(5);
    const size_t shm = (size_t)kStages * S::BYTES;
    if (use_T_list)
        k_advance_tma<T><<<grid, kThreads, shm, s>>>(tm_phi, tm_F, out, g, p, bb.T_ids, &bb.counts->nT, bb.T_masks,
                                                     nullptr, nullptr);
    else
        k_advance_tma<T><<<grid, kThreads, shm, s>>>(tm_phi, tm_F, out, g, p, bb.U_ids, &bb.counts->nU, nullptr,
                                                     bb.tmask, bb.flagT);
    if (launches) *launches += 1;
    return true;
}

#define LS_INSTANTIATE(T)                                                                                        \
    template bool tma_usable<T>(const Geom&, const void*, const void*, const void*);                             \
    template bool launch_reinit_tma<T>(const T*, T*, const Geom&, const StencilParams<T>&, const BandBuffers&,  \
                                       bool, unsigned long long*, bool, cudaStream_t, int64_t*);                 \
    template bool launch_advance_tma<T>(const T*, const T*, T*, const Geom&, const StencilParams<T>&,           \
                                        const BandBuffers&, bool, cudaStream_t, int64_t*);
LS_INSTANTIATE(float)
LS_INSTANTIATE(double)

}  // namespace ls
