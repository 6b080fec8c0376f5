// ls_tma.cu — the band kernels of Steps 2 and 3 as persistent, TMA-fed pipelines.
//
// Data flow per brick (8^3 points of a listed brick plus its one-cell halo):
//   producer (thread 0)  one cp.async.bulk.tensor.3d box load of the halo tile straight from the dense
//                        x-fastest field into shared memory, plus the brick's 64-byte
//                        mask (and, for Advance, the 8^3 box of F), all completing on one mbarrier;
//                        kStages bricks are in flight per CTA
//   consumers (4 warps)  wait on the mbarrier; replicate edge values into out-of-domain halo cells
//                        (R3; TMA zero-fills them); compact the brick's active points into a list with
//                        popc / REDUX ranks so warps run full; evaluate eq. 3-8 / eq. 12-13 for two points
//                        per lane (packed fp32 arithmetic) from the tile into an 8^3 out-brick (Jacobi);
//                        store whole 32-byte rows with 128-bit stores, merging out-brick and tile values.
//                        Two CTA barriers per brick (list complete; out-brick complete).
// The arithmetic is that of ls_math.cuh (IEEE, no FMA contraction): results are bit-identical to the
// scalar kernels of ls_stencil.cu, which remain the path for grids TMA cannot address
// (nx*sizeof(T) not a multiple of 16, or unaligned fields).
#include <cuda.h>

#include "ls_internal.h"
#include "ls_math.cuh"

namespace ls {

namespace {

constexpr int kThreads = 128;   // 4 warps: the per-brick bookkeeping every warp repeats is paid 4x, not 8x
constexpr int kStages = 3;
constexpr int kPY = 10;   // tile extent in y and z: 8 + one halo cell on each side
constexpr int kListBytes = 512 * 4;
constexpr int kBarBytes = 64;   // mbarriers

template <typename T> struct TileCfg;
// TMA needs every box row to start on a 16-byte boundary of the field and to span a multiple of 16
// bytes (an unaligned start coordinate faults with "illegal instruction" on sm_100a): fp32 loads 16
// cells starting four left of the brick, fp64 loads 12 cells starting two left.
template <> struct TileCfg<float> { static constexpr int XOFF = 4, PX = 16; };
template <> struct TileCfg<double> { static constexpr int XOFF = 2, PX = 12; };

constexpr int round128(int x) { return (x + 127) / 128 * 128; }

// Header of a stage, written by the producer thread before it starts the loads of the stage.
struct alignas(16) Hdr {
    int b;          // brick id
    int x0, y0, z0; // first cell of the brick
    long long org;  // element offset of that cell in the dense field
    int edge;       // brick touches the domain boundary (halo needs patching, rows may be partial)
    int has_T;      // Advance: the brick holds T points (mask and F were loaded)
};

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
    static_assert(sizeof(Hdr) <= 64, "header slot");
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LS_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LS_DONE;\n"
        "bra LS_WAIT;\n"
        "LS_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(x), "r"(y), "r"(z)
        : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// Producer side: decode the packed brick position (Geom::pos_*), fill the header.
__device__ __forceinline__ void fill_hdr(Hdr* h, const Geom& g, int b, int pos, bool has_T) {
    const int bx = pos & g.pos_mx, by = (pos >> g.pos_sy) & g.pos_my, bz = pos >> g.pos_sz;
    h->b = b;
    h->x0 = bx * 8;
    h->y0 = by * 8;
    h->z0 = bz * 8;
    h->org = g.idx(bx * 8, by * 8, bz * 8);
    h->edge = (bx == 0) | (by == 0) | (bz == 0) | (bx == g.NBx - 1) | (by == g.NBy - 1) | (bz == g.NBz - 1);
    h->has_T = has_T ? 1 : 0;
}

// R3: TMA zero-fills cells outside the domain; give them the value of the nearest in-domain cell
// (edge replicate).  Sources are in-domain cells, destinations are not: no ordering needed inside.
// Only called for bricks on the domain boundary (block-uniform).
template <typename T, int PX, int XOFF>
__device__ __noinline__ void patch_boundary(T* tile, const Geom& g, int x0, int y0, int z0) {
    const int ox = x0 - XOFF, oy = y0 - 1, oz = z0 - 1;
    for (int e = threadIdx.x; e < PX * kPY * kPY; e += kThreads) {
        const int x = e % PX, r = e / PX, y = r % kPY, z = r / kPY;
        const int gx = ox + x, gy = oy + y, gz = oz + z;
        const int cx = min(max(gx, 0), g.nx - 1), cy = min(max(gy, 0), g.ny - 1), cz = min(max(gz, 0), g.nz - 1);
        if (cx != gx || cy != gy || cz != gz) {
            const int sx = cx - ox, sy = cy - oy, sz = cz - oz;
            if (sx >= 0 && sx < PX && sy < kPY && sz < kPY) tile[e] = tile[(sz * kPY + sy) * PX + sx];
        }
    }
    fence_proxy_async();   // generic writes into a tile a later TMA load overwrites
    __syncthreads();
}

// Compact the set bits of the brick mask into `list` (ascending point order) and return their number.
// Entry = tile offset of the point | brick-local index (lz*64 + ly*8 + lx) << 16.
// Warp w owns mask words 2w and 2w+1 (layers lz): lane l holds bit l of the low half (row l>>3) and
// of the high half (row 4 + (l>>3)) of each.
template <int PX, int XOFF>
__device__ __forceinline__ int build_list(const uint64_t* mk, uint32_t* list) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned pc = lane < 8 ? __popcll(mk[lane]) : 0;
    const int total = (int)__reduce_add_sync(0xffffffffu, pc);
    int base = (int)__reduce_add_sync(0xffffffffu, lane < 2 * w ? pc : 0u);   // points in layers below 2w
    const ulonglong2 words = *reinterpret_cast<const ulonglong2*>(mk + 2 * w);
    const uint32_t lt = (1u << lane) - 1u;
    const uint32_t e0 = (uint32_t)((2 * w + 1) * kPY * PX + ((lane >> 3) + 1) * PX + (lane & 7) + XOFF) |
                        (uint32_t)(2 * w * 64 + lane) << 16;   // layer 2w, low half (rows 0-3)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const uint64_t word = h ? words.y : words.x;
        const uint32_t lo = (uint32_t)word, hi = (uint32_t)(word >> 32);
        const uint32_t e_lo = e0 + h * (uint32_t)(kPY * PX + (64 << 16));
        const int nlo = __popc(lo);
        if ((lo >> lane) & 1u) list[base + __popc(lo & lt)] = e_lo;
        if ((hi >> lane) & 1u) list[base + nlo + __popc(hi & lt)] = e_lo + (uint32_t)(4 * PX + (32 << 16));
        base += nlo + __popc(hi);
    }
    return total;
}

// Per-thread constants of the row store: thread t owns 128-bit part `part` of brick row `row`
// (fp32: 64 rows x 2 parts = 128 threads, one pass; fp64: 64 rows x 4 parts, two passes).
template <typename T>
struct RowSlot {
    int row;        // lz*8 + ly
    int toff;       // tile offset of the first cell of the part
    long long goff; // element offset from the brick origin
    int lx0, ly, lz;
};
template <typename T, int PX, int XOFF>
__device__ __forceinline__ RowSlot<T> row_slot(const Geom& g, int t) {
    constexpr int VEC = 16 / (int)sizeof(T), PARTS = 8 / VEC;
    RowSlot<T> r;
    r.row = t / PARTS;
    const int part = t % PARTS;
    r.lz = r.row >> 3;
    r.ly = r.row & 7;
    r.lx0 = part * VEC;
    r.toff = ((r.lz + 1) * kPY + (r.ly + 1)) * PX + XOFF + part * VEC;
    r.goff = ((long long)r.lz * g.ny + r.ly) * g.nx + part * VEC;
    return r;
}
// Store the part: new values (out brick, indexed by brick-local cell) where the mask bit is set, the
// tile's values elsewhere.  Rows without a mask bit are skipped unless all_rows (then copied from the tile).
template <typename T>
__device__ __forceinline__ void store_part(const T* tile, const T* outb, const unsigned char* mk8, bool have_mask,
                                           bool all_rows, T* __restrict__ dst, const Geom& g, const Hdr& h,
                                           const RowSlot<T>& r) {
    constexpr int VEC = 16 / (int)sizeof(T);
    const unsigned m = have_mask ? mk8[r.row] : 0u;
    if (!all_rows && m == 0) return;
    if (h.edge && (h.x0 + r.lx0 >= g.nx || h.y0 + r.ly >= g.ny || h.z0 + r.lz >= g.nz)) return;   // nx % VEC == 0
    union V { int4 q; T e[VEC]; } a, b;
    a.q = *reinterpret_cast<const int4*>(tile + r.toff);
    const unsigned nib = (m >> r.lx0) & ((1u << VEC) - 1u);
    if (nib) {
        b.q = *reinterpret_cast<const int4*>(outb + r.row * 8 + r.lx0);
#pragma unroll
        for (int e = 0; e < VEC; ++e)
            if ((nib >> e) & 1u) a.e[e] = b.e[e];
    }
    *reinterpret_cast<int4*>(dst + h.org + r.goff) = a.q;
}

// ---------------------------------------------------------------------------------------------
// Step 3: one reinitialisation sweep over the N list (eq. 12-13), see launch_reinit_band.
// ---------------------------------------------------------------------------------------------
template <typename T, bool CLAMP, bool RESIDUAL, bool EMIT_T>
__global__ void __launch_bounds__(kThreads)
k_reinit_tma(const __grid_constant__ CUtensorMap tm_src, T* __restrict__ dst, Geom g, StencilParams<T> p,
             const int32_t* __restrict__ ids, const int32_t* __restrict__ poss, const int32_t* __restrict__ count_ptr,
             const uint64_t* __restrict__ masks, unsigned long long* __restrict__ residual,
             uint64_t* __restrict__ tmask, uint8_t* __restrict__ flagT) {
    using S = Stage<T, false>;
    constexpr int PX = S::PX, XOFF = S::XOFF;
    constexpr int SY = PX, SZ = kPY * PX;
    constexpr int PASSES = (64 * (8 / (16 / (int)sizeof(T)))) / kThreads;   // row-store passes: 1 (fp32), 2 (fp64)
    // dynamic shared memory: [kStages stages][list 2 KB][out brick 8^3][mbarriers] — one base register for all
    extern __shared__ __align__(128) unsigned char smem[];
    uint32_t* list = reinterpret_cast<uint32_t*>(smem + kStages * S::BYTES);
    T* outb = reinterpret_cast<T*>(smem + kStages * S::BYTES + kListBytes);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int count = *count_ptr;
    const int G = gridDim.x;
    const int mine = (int)blockIdx.x < count ? (count - (int)blockIdx.x + G - 1) / G : 0;
    const uint32_t smem_base = smem_u32(smem), bar_base = smem_base + kStages * S::BYTES + kListBytes + 512 * (int)sizeof(T);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(bar_base + 8 * s, 1);
        fence_barrier_init();
    }
    __syncthreads();

    RowSlot<T> rs[PASSES];
#pragma unroll
    for (int q = 0; q < PASSES; ++q) rs[q] = row_slot<T, PX, XOFF>(g, tid + q * kThreads);

    // producer state (thread 0): next list index to issue and the stage it goes to
    int p_li = blockIdx.x, p_slot = 0, p_left = mine;
    auto issue = [&]() {
        const int b = ids[p_li], pos = poss[p_li];
        Hdr* h = reinterpret_cast<Hdr*>(smem + p_slot * S::BYTES + S::OFF_HDR);
        fill_hdr(h, g, b, pos, true);
        if (EMIT_T) flagT[b] = 0;
        const uint32_t st = smem_base + p_slot * S::BYTES, bar = bar_base + 8 * p_slot;
        mbar_expect_tx(bar, S::TILE_BYTES + 64);
        tma_load_3d(st, &tm_src, bar, h->x0 - XOFF, h->y0 - 1, h->z0 - 1);
        bulk_load(st + S::OFF_MASK, masks + (int64_t)b * 8, 64, bar);   // dense per-brick N masks
        p_li += G;
        p_slot = p_slot == kStages - 1 ? 0 : p_slot + 1;
        --p_left;
    };
    if (tid == 0)
        for (int n = 0; n < kStages - 1 && p_left > 0; ++n) issue();

    T rmax = T(0);
    int slot = 0;
    uint32_t phase = 0;
    for (int n = 0; n < mine; ++n) {
        unsigned char* st = smem + slot * S::BYTES;
        const T* tile = reinterpret_cast<const T*>(st);
        const uint64_t* mk = reinterpret_cast<const uint64_t*>(st + S::OFF_MASK);
        mbar_wait(bar_base + 8 * slot, phase);
        const Hdr h = *reinterpret_cast<const Hdr*>(st + S::OFF_HDR);
        if (h.edge) patch_boundary<T, PX, XOFF>(reinterpret_cast<T*>(st), g, h.x0, h.y0, h.z0);

        const int total = build_list<PX, XOFF>(mk, list);
        __syncthreads();   // B1: list complete; every thread is done with brick n-1 (its stage, list, out brick)
        if (tid == 0 && p_left > 0) issue();   // refill the stage brick n-1 used

        // two points per thread and round; at most 512 points = 2 rounds of 128 pairs.  Jacobi: reads come
        // from the tile (iteration k), results go to the out brick (iteration k+1).
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            // lane l of warp w takes list entries e and e + 32: each shared-memory load of a warp then covers
            // 32 CONSECUTIVE points (4 brick rows), the least bank-conflicting set this tile pitch allows
            // round 1 deals its (usually few) entries to warp 3 first: warp 0 also runs the producer
            const int e = r * 2 * kThreads + 64 * (r ? kThreads / 32 - 1 - w : w) + lane;
            if (e < total) {
                uint2 ent;
                ent.x = list[e];
                ent.y = e + 32 < total ? list[e + 32] : ent.x;   // tail: evaluate the point twice
                const int o0 = (int)(ent.x & 0xffffu), o1 = (int)(ent.y & 0xffffu);
                Two<T> u = reinit_pair<T>(tile, o0, o1, SY, SZ, p);
                if (RESIDUAL) rmax = fmax(rmax, fmax(mag(u.x - tile[o0]), mag(u.y - tile[o1])));
                if (CLAMP) { u.x = clamp_val(u.x, p.gamma); u.y = clamp_val(u.y, p.gamma); }
                outb[ent.x >> 16] = u.x;
                outb[ent.y >> 16] = u.y;
            }
        }
        __syncthreads();   // B2: out brick complete

#pragma unroll
        for (int q = 0; q < PASSES; ++q)
            store_part<T>(tile, outb, reinterpret_cast<const unsigned char*>(mk), true, false, dst, g, h, rs[q]);
        if (EMIT_T) {
            // T mask of phi^{n+1} = clamp(d) on this brick: T^{n+1} is a subset of N^n
            bool any = false;
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const int lz = 2 * w + hh;
                const uint64_t word = mk[lz];
                const bool tl = ((uint32_t)word >> lane) & 1u ? mag(outb[lz * 64 + lane]) < p.gamma : false;
                const bool th = ((uint32_t)(word >> 32) >> lane) & 1u ? mag(outb[lz * 64 + 32 + lane]) < p.gamma : false;
                const uint32_t bl = __ballot_sync(0xffffffffu, tl), bh = __ballot_sync(0xffffffffu, th);
                const uint64_t tw = (uint64_t)bl | ((uint64_t)bh << 32);
                if (lane == 0) tmask[(int64_t)h.b * 8 + lz] = tw;
                any = any || tw != 0;
            }
            if (lane == 0 && any) flagT[h.b] = 1;   // zeroed by the producer when it issued the brick (barriers in between)
        }
        if (++slot == kStages) { slot = 0; phase ^= 1u; }
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
__global__ void __launch_bounds__(kThreads)
k_advance_tma(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_F,
              T* __restrict__ out, Geom g, StencilParams<T> p, const int32_t* __restrict__ ids,
              const int32_t* __restrict__ poss, const int32_t* __restrict__ count_ptr,
              const uint64_t* __restrict__ list_masks, const uint64_t* __restrict__ dense_tmask,
              const uint8_t* __restrict__ flagT) {
    using S = Stage<T, true>;
    constexpr int PX = S::PX, XOFF = S::XOFF;
    constexpr int SY = PX, SZ = kPY * PX;
    constexpr int PASSES = (64 * (8 / (16 / (int)sizeof(T)))) / kThreads;
    // dynamic shared memory: [kStages stages][list 2 KB][out brick 8^3][mbarriers] — one base register for all
    extern __shared__ __align__(128) unsigned char smem[];
    uint32_t* list = reinterpret_cast<uint32_t*>(smem + kStages * S::BYTES);
    T* outb = reinterpret_cast<T*>(smem + kStages * S::BYTES + kListBytes);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int count = *count_ptr;
    const int G = gridDim.x;
    const int mine = (int)blockIdx.x < count ? (count - (int)blockIdx.x + G - 1) / G : 0;
    const uint32_t smem_base = smem_u32(smem), bar_base = smem_base + kStages * S::BYTES + kListBytes + 512 * (int)sizeof(T);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(bar_base + 8 * s, 1);
        fence_barrier_init();
    }
    __syncthreads();

    RowSlot<T> rs[PASSES];
#pragma unroll
    for (int q = 0; q < PASSES; ++q) rs[q] = row_slot<T, PX, XOFF>(g, tid + q * kThreads);

    int p_li = blockIdx.x, p_slot = 0, p_left = mine;
    auto issue = [&]() {
        const int b = ids[p_li], pos = poss[p_li];
        const bool has_T = dense_tmask ? flagT[b] != 0 : true;
        Hdr* h = reinterpret_cast<Hdr*>(smem + p_slot * S::BYTES + S::OFF_HDR);
        fill_hdr(h, g, b, pos, has_T);
        const uint32_t st = smem_base + p_slot * S::BYTES, bar = bar_base + 8 * p_slot;
        mbar_expect_tx(bar, has_T ? S::TILE_BYTES + S::F_BYTES + 64 : S::TILE_BYTES);
        tma_load_3d(st, &tm_phi, bar, h->x0 - XOFF, h->y0 - 1, h->z0 - 1);
        if (has_T) {
            tma_load_3d(st + S::OFF_F, &tm_F, bar, h->x0, h->y0, h->z0);
            const uint64_t* m = (dense_tmask ? dense_tmask : list_masks) + (int64_t)b * 8;   // both dense per brick
            bulk_load(st + S::OFF_MASK, m, 64, bar);
        }
        p_li += G;
        p_slot = p_slot == kStages - 1 ? 0 : p_slot + 1;
        --p_left;
    };
    if (tid == 0)
        for (int n = 0; n < kStages - 1 && p_left > 0; ++n) issue();

    int slot = 0;
    uint32_t phase = 0;
    for (int n = 0; n < mine; ++n) {
        unsigned char* st = smem + slot * S::BYTES;
        const T* tile = reinterpret_cast<const T*>(st);
        const T* Fb = reinterpret_cast<const T*>(st + S::OFF_F);
        const uint64_t* mk = reinterpret_cast<const uint64_t*>(st + S::OFF_MASK);
        mbar_wait(bar_base + 8 * slot, phase);
        const Hdr h = *reinterpret_cast<const Hdr*>(st + S::OFF_HDR);
        if (h.edge) patch_boundary<T, PX, XOFF>(reinterpret_cast<T*>(st), g, h.x0, h.y0, h.z0);

        int total = 0;
        if (h.has_T) total = build_list<PX, XOFF>(mk, list);   // uniform over the CTA
        __syncthreads();   // B1: list complete; every thread is done with brick n-1
        if (tid == 0 && p_left > 0) issue();
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int e = r * 2 * kThreads + 64 * (r ? kThreads / 32 - 1 - w : w) + lane;   // see k_reinit_tma
            if (e < total) {
                uint2 ent;
                ent.x = list[e];
                ent.y = e + 32 < total ? list[e + 32] : ent.x;
                const Two<T> u = advance_pair<T>(tile, (int)(ent.x & 0xffffu), (int)(ent.y & 0xffffu), SY, SZ,
                                                 Fb[ent.x >> 16], Fb[ent.y >> 16], p);
                outb[ent.x >> 16] = u.x;
                outb[ent.y >> 16] = u.y;
            }
        }
        __syncthreads();   // B2: out brick complete
#pragma unroll
        for (int q = 0; q < PASSES; ++q)
            store_part<T>(tile, outb, reinterpret_cast<const unsigned char*>(mk), h.has_T != 0, true, out, g, h, rs[q]);
        if (++slot == kStages) { slot = 0; phase ^= 1u; }
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

// Persistent grid of a band kernel: the largest shared-memory carve-out, then as many CTAs as fit on an SM.
template <typename K>
int persistent_grid(K kernel, size_t dyn_smem) {
    cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, dyn_smem) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    return tma_grid(per_sm);
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
    const size_t shm = (size_t)kStages * S::BYTES + kListBytes + 512 * sizeof(T) + kBarBytes;
    const int32_t* cnt = &bb.counts->nN;
#define LS_LAUNCH(C, R, E)                                                                                       \
    do {                                                                                                         \
        static const int grid = persistent_grid(k_reinit_tma<T, C, R, E>, shm);                                  \
        k_reinit_tma<T, C, R, E><<<grid, kThreads, shm, s>>>(tm, dst, g, p, bb.N_ids, bb.N_pos, cnt, bb.nmask,      \
                                                             residual, bb.tmask, bb.flagT);                      \
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
    const size_t shm = (size_t)kStages * S::BYTES + kListBytes + 512 * sizeof(T) + kBarBytes;
    static const int grid = persistent_grid(k_advance_tma<T>, shm);
    if (use_T_list)
        k_advance_tma<T><<<grid, kThreads, shm, s>>>(tm_phi, tm_F, out, g, p, bb.T_ids, bb.T_pos, &bb.counts->nT,
                                                     bb.tmask, nullptr, nullptr);
    else
        k_advance_tma<T><<<grid, kThreads, shm, s>>>(tm_phi, tm_F, out, g, p, bb.U_ids, bb.U_pos, &bb.counts->nU,
                                                     nullptr, bb.tmask, bb.flagT);
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
