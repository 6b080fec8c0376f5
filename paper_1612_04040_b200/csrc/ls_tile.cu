// ls_tile.cu — the band kernels of Steps 2 and 3: persistent, warp-specialised, fed by asynchronous
// copies through an mbarrier pipeline.
//
// Tile = one QUAD (four x-adjacent 8^3 bricks, 32 x 8 x 8 points; ls_internal.h).  In shared memory:
//   M  [8+2K][8+2K][32]   the quad and K halo rows in y and z: every row is one aligned 128-byte line (fp32)
//   L, R [6+2K][6+2K][XW] the x halo, one 16-byte piece per row (fp32: 4 cells, fp64: 2)
// K = number of operations fused in the launch: K = 1 is Advance or one reinit sweep (the default); K = 2 is two
// sweeps (temporal blocking of eq. 12's pseudo-time iterations): sweep 1 is evaluated on the
// quad's N points AND on the N points of the one-cell ring around it (neighbour quads' masks), kept in
// registers until every read of iteration k is done, written back IN PLACE, and sweep 2 then runs on the
// quad's own points.  Jacobi order is preserved exactly, so K = 2 equals two K = 1 launches bit for bit.
//
//   producer warps, K = 1 (one whole warp per pipeline stage)   draw one quad at a time from the ordered quad list
//        through a device ticket counter, read its list entry and load map, and GATHER only the 32-byte sectors
//        the quad's N points read with 16-byte cp.async (LDGSTS), two lanes per sector (half the DRAM reads of a
//        whole-box load); the quad's precomputed item list comes by cp.async.bulk (UBLKCP); Advance also gathers
//        the F rows of bricks that hold band points and takes the quad's 32 T mask words by cp.async.bulk.
//   producer, K = 2 (one elected lane)   issues three cp.async.bulk.tensor.3d box loads (M, L, R: UTMALDG) straight
//        from the dense x-fastest field, the item list and the N masks of the six neighbour quads.
//        Either way everything completes on the stage's "full" mbarrier, and the stage's "empty" mbarrier gates its reuse.
//   consumer warps   wait on "full"; edge-replicate the out-of-domain halo of tiles that reach outside the domain
//        (R3); lane l evaluates items l, l+NC, ...: one item = 4 x-consecutive cells = 5 LDS.128 + 2 LDS.32, two
//        packed fp32 pairs through eq. 3-8 / eq. 12-13 (ls_math.cuh), one 16-byte store to the other global buffer.
//        K = 1 needs no CTA barrier per tile: each warp arrives on "empty" when it is done with the stage.
// The arithmetic is bit-identical to the scalar kernels of ls_stencil.cu, which remain the path for grids the
// tile path cannot address (nx not a multiple of 4, unaligned fields).
#include <cuda.h>

#include <cstring>

#include "ls_internal.h"
#include "ls_math.cuh"

namespace ls {

namespace {

constexpr int kChunk = 4;                   // quads per ticket

constexpr int round128(int x) { return (x + 127) / 128 * 128; }

// Header of a stage, written by the producer before it starts the loads of the stage.
struct alignas(16) Hdr {
    int quad;       // quad id; -1: no more work
    int nitems;
    int x0, y0, z0; // first cell of the quad
    int edge;       // tile reaches outside the domain (halo needs patching)
    long long org;  // element offset of the first cell in the dense field
    int tvalid;     // Advance: T masks were loaded (else the quad holds no T point)
    int ring_n;     // K = 2: entries of the ring list (consumers count them up from 0)
    int haveL, haveR;   // the x halo pieces were loaded
};

// One pipeline stage in shared memory.
template <typename T, int K, bool ADV>
struct Stage {
    static constexpr int XW = 16 / (int)sizeof(T);
    static constexpr int PY = 8 + 2 * K;
    static constexpr int PH = 6 + 2 * K;
    static constexpr int M_BYTES = PY * PY * 32 * (int)sizeof(T);
    static constexpr int H_BYTES = PH * PH * 16;
    static constexpr int OFF_L = round128(M_BYTES);
    static constexpr int OFF_R = OFF_L + round128(H_BYTES);
    static constexpr int OFF_F = OFF_R + round128(H_BYTES);
    static constexpr int F_BYTES = ADV ? 2048 * (int)sizeof(T) : 0;
    static constexpr int OFF_ITEMS = OFF_F + F_BYTES;
    static constexpr int OFF_TM = OFF_ITEMS + kItemsPerQuad * 2;
    static constexpr int TM_BYTES = ADV ? 256 : 0;
    static constexpr int OFF_NB = OFF_TM + TM_BYTES;            // K = 2: y-, y+, z-, z+ quads (256 B each), left quad's
    static constexpr int NB_BYTES = K > 1 ? 4 * 256 + 2 * 64 : 0;   // brick 3 and right quad's brick 0 (64 B each)
    static constexpr int OFF_RING = OFF_NB + NB_BYTES;
    static constexpr int RING_BYTES = K > 1 ? 256 * 4 : 0;
    static constexpr int OFF_HDR = OFF_RING + RING_BYTES;
    static constexpr int BYTES = round128(OFF_HDR + (int)sizeof(Hdr));
    static_assert(sizeof(Hdr) <= 64, "header slot");
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// (with a suspend-time hint the hardware parks the waiting warp; a bare try_wait loop returns at once and spins, and the
// spinning takes issue slots from the warps of the other CTAs on the SM: 22 M of 73 M warp instructions of a sweep, measured)
#ifndef LS_WAIT_HINT_NS
#define LS_WAIT_HINT_NS 20000u
#endif
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LS_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra LS_DONE;\n"
        "bra LS_WAIT;\n"
        "LS_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity), "r"(LS_WAIT_HINT_NS)
        : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
template <int NC>
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(NC) : "memory"); }

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(x), "r"(y), "r"(z)
        : "memory");
}
// 16-byte asynchronous copy global -> shared (LDGSTS, L2 only), and the arrive that fires when all of this
// thread's earlier ones have landed (the barrier's expected count includes it: .noinc).
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_arrive(uint32_t bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// The three arrays of a tile.  Coordinates are relative to the quad's first cell.
template <typename T, int K>
struct Tile {
    static constexpr int XW = 16 / (int)sizeof(T), PY = 8 + 2 * K, PH = 6 + 2 * K;
    T* M;
    T* L;
    T* R;
    // offset in M of cell (x, y, z), x in [0, 32), y, z in [-K, 8 + K)
    __device__ __forceinline__ static int om(int x, int y, int z) { return ((z + K) * PY + (y + K)) * 32 + x; }
    // offset in L / R of column c of row (y, z), y, z in [-(K-1), 8 + K - 1)
    __device__ __forceinline__ static int oh(int c, int y, int z) { return ((z + K - 1) * PH + (y + K - 1)) * XW + c; }
    // any cell of the tile's cover: x in [-XW, 32 + XW) (x outside [0, 32) only for rows L / R hold)
    __device__ __forceinline__ T& at(int x, int y, int z) const {
        if (x < 0) return L[oh(x + XW, y, z)];
        if (x >= 32) return R[oh(x - 32, y, z)];
        return M[om(x, y, z)];
    }
};

// R3: TMA zero-fills cells outside the domain; give them the value of the nearest in-domain cell (edge
// replicate).  Sources are in-domain cells, destinations are not: no ordering needed inside.  Only called for
// tiles that reach outside the domain (uniform over the consumers).  Ends with a consumer barrier.
template <typename T, int K, int NC>
__device__ __noinline__ void patch_boundary(const Tile<T, K>& t, const Geom& g, int x0, int y0, int z0, int ctid) {
    constexpr int XW = Tile<T, K>::XW, PY = Tile<T, K>::PY, PH = Tile<T, K>::PH;
    auto fix = [&](int x, int y, int z) {
        const int gx = x0 + x, gy = y0 + y, gz = z0 + z;
        const int cx = min(max(gx, 0), g.nx - 1), cy = min(max(gy, 0), g.ny - 1), cz = min(max(gz, 0), g.nz - 1);
        if (cx != gx || cy != gy || cz != gz) {
            const int sx = cx - x0, sy = cy - y0, sz = cz - z0;
            // the nearest in-domain cell lies in the tile's cover unless the tile misses the domain in x by more
            // than its halo (cannot happen: a listed quad holds in-domain cells)
            if (sx >= -XW && sx < 32 + XW) t.at(x, y, z) = t.at(sx, sy, sz);
        }
    };
    for (int e = ctid; e < PY * PY * 32; e += NC) fix(e & 31, (e >> 5) % PY - K, (e >> 5) / PY - K);
    for (int e = ctid; e < PH * PH * XW * 2; e += NC) {
        const int side = e / (PH * PH * XW), r = e % (PH * PH * XW);
        const int c = r % XW, row = r / XW;
        fix(side ? 32 + c : c - XW, row % PH - (K - 1), row / PH - (K - 1));
    }
    fence_proxy_async();   // generic writes into a tile a later TMA load overwrites
    consumer_sync<NC>();
}

// The stencil of the item at group xq (0..7) of row (y, z) of the quad.
template <typename T, int K>
__device__ __forceinline__ void load_item(const Tile<T, K>& t, int xq, int y, int z, Item4<T>& s) {
    constexpr int SY = 32, SZ = 32 * Tile<T, K>::PY, XW = Tile<T, K>::XW;
    const int o = Tile<T, K>::om(xq * 4, y, z);
    const T* tile = t.M;
    if (sizeof(T) == 4) {
        union V { float4 q; T e[4]; } c, ym, yp, zm, zp;
        c.q = *reinterpret_cast<const float4*>(tile + o);
        ym.q = *reinterpret_cast<const float4*>(tile + o - SY);
        yp.q = *reinterpret_cast<const float4*>(tile + o + SY);
        zm.q = *reinterpret_cast<const float4*>(tile + o - SZ);
        zp.q = *reinterpret_cast<const float4*>(tile + o + SZ);
#pragma unroll
        for (int e = 0; e < 4; ++e) { s.c[e] = c.e[e]; s.ym[e] = ym.e[e]; s.yp[e] = yp.e[e]; s.zm[e] = zm.e[e]; s.zp[e] = zp.e[e]; }
    } else {
        union V { double2 q[2]; T e[4]; } c, ym, yp, zm, zp;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            c.q[h] = *reinterpret_cast<const double2*>(tile + o + 2 * h);
            ym.q[h] = *reinterpret_cast<const double2*>(tile + o - SY + 2 * h);
            yp.q[h] = *reinterpret_cast<const double2*>(tile + o + SY + 2 * h);
            zm.q[h] = *reinterpret_cast<const double2*>(tile + o - SZ + 2 * h);
            zp.q[h] = *reinterpret_cast<const double2*>(tile + o + SZ + 2 * h);
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) { s.c[e] = c.e[e]; s.ym[e] = ym.e[e]; s.yp[e] = yp.e[e]; s.zm[e] = zm.e[e]; s.zp[e] = zp.e[e]; }
    }
    const int h = Tile<T, K>::oh(0, y, z);
    const T* pm = xq > 0 ? tile + o - 1 : t.L + h + XW - 1;
    const T* pp = xq < 7 ? tile + o + 4 : t.R + h;
    s.xm = *pm;
    s.xp = *pp;
}
template <typename T>
__device__ __forceinline__ void store4(T* p, const T v[4]) {
    if (sizeof(T) == 4) {
        *reinterpret_cast<float4*>(p) = make_float4((float)v[0], (float)v[1], (float)v[2], (float)v[3]);
    } else {
        reinterpret_cast<double2*>(p)[0] = make_double2((double)v[0], (double)v[1]);
        reinterpret_cast<double2*>(p)[1] = make_double2((double)v[2], (double)v[3]);
    }
}

struct TileArgs {
    const QuadEntry* qlist;
    const int32_t* count;
    const uint16_t* items;
    const uint8_t* qneed;         // K = 1: load maps (ls_internal.h)
    const uint64_t* nmask;        // K = 2: N masks of the band (zero for quads outside it)
    const void* zero_page;        // 256 zero bytes (neighbour quads outside the domain)
    const uint64_t* tmask_in;     // Advance: T masks of the band (tmask[tb])
    const uint8_t* qflagT_in;
    const uint8_t* tgate;         // null or validity gate of tmask_in
    uint64_t* tmask_out;          // EMIT_T: tmask[tb ^ 1]
    uint8_t* qflagT_out;
    unsigned long long* residual;
    const void* src;              // K = 1: the field the tiles are gathered from, and F (Advance)
    const void* F;
    unsigned int* ticket;         // [0] next list index, [1] CTAs done (self-resetting)
    int reverse;                  // walk the list from its end
};

// ---------------------------------------------------------------------------------------------
// One launch = Advance (ADV, K = 1), or K reinit sweeps, on every listed quad; results of the last operation
// are written to `dst` at the item cells.  NCW consumer warps + 1 producer warp.
// ---------------------------------------------------------------------------------------------
template <typename T, bool ADV, int K, bool CLAMP, bool RESIDUAL, bool EMIT_T, int STAGES, int NCW, int NPW>
__global__ void __launch_bounds__((NCW + NPW) * 32)
k_band_tile(const __grid_constant__ CUtensorMap tm_M, const __grid_constant__ CUtensorMap tm_H,
            const __grid_constant__ CUtensorMap tm_F, T* __restrict__ dst, Geom g, StencilParams<T> pa,
            StencilParams<T> pr, TileArgs a) {
    static_assert(K == 1 || (K == 2 && !ADV && NCW == 8 && NPW == 1), "K = 2: two reinit sweeps, 256 consumers");
    static_assert(K != 1 || NPW == STAGES || NPW == 1, "K = 1: one producer warp per stage, or one for all stages");
    using S = Stage<T, K, ADV>;
    using TL = Tile<T, K>;
    constexpr int NC = NCW * 32, XW = S::XW;
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t smem_base = smem_u32(smem);
    // after the stages: T staging of EMIT_T (2 x 512 B: one byte per item position), then the mbarriers
    // (full[STAGES], empty[STAGES])
    constexpr int TS_BYTES = EMIT_T ? 1024 : 0;
    unsigned char* tstage = smem + STAGES * S::BYTES;
    const uint32_t bar_full = smem_base + STAGES * S::BYTES + TS_BYTES, bar_empty = bar_full + 8 * STAGES;
    // Small bands (cfg 1, the paper's 101^3): most CTAs of the persistent grid have nothing to do.  They leave before
    // touching shared memory — only the scheduler's "producer warps done" count must still see them.
    const int count = *a.count;
    if ((int)blockIdx.x >= count) {
        if (tid == 0) {
            __threadfence();
            if (atomicAdd(a.ticket + 1, (unsigned)NPW) + NPW == gridDim.x * NPW) { a.ticket[0] = 0u; a.ticket[1] = 0u; }
        }
        return;
    }
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) { mbar_init(bar_full + 8 * s, K == 1 ? 33 : 1); mbar_init(bar_empty + 8 * s, NCW); }
        fence_barrier_init();
    }
    if (EMIT_T && tid < 64) reinterpret_cast<uint4*>(tstage)[tid] = make_uint4(0u, 0u, 0u, 0u);
    // K = 1 fetches only the chunks its items read; the rest of a stage keeps what earlier tiles left there, which
    // only feeds results that are thrown away (cells of an item outside N).  Start from zeros, not from whatever
    // bit patterns the last kernel left in shared memory (a NaN would send a lane down the scalar slow path).
    for (int i = tid; i < STAGES * S::BYTES / 16; i += (NCW + NPW) * 32) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();

    if (warp >= NCW && K == 1) {
        // ------------------------------ producer, K = 1: sparse gather ------------------------------
        // The whole warp works.  Lane pair (2s, 2s+1) owns tile rows s, s+16, ..., s+96 (of 10 x 10): per needed
        // chunk of a row each lane of the pair copies one 16-byte half with cp.async (the two halves of a 32-byte
        // sector leave in one instruction and coalesce into one sector request); lane 2s also copies the row's left
        // x-halo piece, lane 2s+1 the right one.  Which chunks: the load map the band builder wrote (kNeedBytes).
        // One producer warp per stage: warp p fills stage p only, with tiles it draws itself from the ticket counter,
        // so it has STAGES tile periods for each tile it issues.
        constexpr int NPASS = 7;
        const int half = lane & 1, rslot = lane >> 1;
        const T* src = reinterpret_cast<const T*>(a.src);
        const T* Fsrc = reinterpret_cast<const T*>(a.F);
        struct Need { uint32_t lo, hi, own; };   // need bytes of passes 0-3, 4-6; own nibbles of the 4 F passes
        auto load_entry = [&](int idx) -> QuadEntry {
            QuadEntry e;
            e.quad = -1; e.nitems = 0;
            if (idx >= 0) e = a.qlist[a.reverse ? count - 1 - idx : idx];
            return e;
        };
        auto load_need = [&](int quad) -> Need {
            Need n;
            n.lo = n.hi = n.own = 0;
            if (quad >= 0) {
                const uint8_t* nd = a.qneed + (int64_t)quad * kNeedBytes;
                n.lo = (uint32_t)nd[rslot] | ((uint32_t)nd[rslot + 16] << 8) | ((uint32_t)nd[rslot + 32] << 16) |
                       ((uint32_t)nd[rslot + 48] << 24);
                n.hi = (uint32_t)nd[rslot + 64] | ((uint32_t)nd[rslot + 80] << 8) |
                       ((uint32_t)(rslot < 4 ? nd[rslot + 96] : 0) << 16);
                if (ADV)
                    n.own = (uint32_t)nd[112 + rslot] | ((uint32_t)nd[112 + 16 + rslot] << 8) |
                            ((uint32_t)nd[112 + 32 + rslot] << 16) | ((uint32_t)nd[112 + 48 + rslot] << 24);
            }
            return n;
        };
        // per-lane constants of the 7 passes: element offset of the row from the quad's first cell, byte offset of
        // the row in M, byte offset of its piece in L / R (quad rows only)
        int64_t rowoff[NPASS];
        uint32_t m_off[NPASS], h_off[NPASS];
#pragma unroll
        for (int k = 0; k < NPASS; ++k) {
            const int r = min(rslot + 16 * k, 99), y = r % 10 - 1, z = r / 10 - 1;
            rowoff[k] = ((int64_t)z * g.ny + y) * g.nx;
            m_off[k] = (uint32_t)(r * 32 * (int)sizeof(T));
            h_off[k] = (uint32_t)(((z & 7) * 8 + (y & 7)) * 16);
        }
        int64_t frowoff[4];   // Advance: rows of the F box
#pragma unroll
        for (int k = 0; k < 4; ++k) frowoff[k] = ((int64_t)((rslot + 16 * k) >> 3) * g.ny + ((rslot + 16 * k) & 7)) * g.nx;
        // Scheduling is dynamic, one tile per ticket, and nothing is drawn ahead: a warp takes its next ticket right
        // after it has fired a tile, and the three dependent round trips (ticket, list entry, load map) run while
        // the consumers work through the other stages.  Tiles cost between 1 and 512 items, so any tile reserved
        // early is load imbalance at the end of the launch: with tickets drawn in chunks and one chunk ahead, two
        // thirds of the list were handed out in the first microsecond and the slowest CTA ran 1.4x the mean.
        // NPW == STAGES: warp p owns stage p.  NPW == 1: one warp fills the stages in turn (smaller CTAs, more of them
        // per SM: what hides the consumers' latencies is the number of consumer warps on the SM).
        int issued = 0;
        for (;;) {
            const int slot = NPW == 1 ? issued % STAGES : warp - NCW;
            const int fill = NPW == 1 ? issued / STAGES : issued;          // fills of this stage so far
            const uint32_t st = smem_base + slot * S::BYTES, bar = bar_full + 8 * slot;
            Hdr* const h = reinterpret_cast<Hdr*>(smem + slot * S::BYTES + S::OFF_HDR);
            int idx = 0;
            if (lane == 0) idx = (int)atomicAdd(a.ticket, 1u);
            idx = __shfl_sync(0xffffffffu, idx, 0);
            if (idx >= count) break;
            const QuadEntry e_cur = load_entry(idx);
            const Need n_cur = load_need(e_cur.quad);
            // ---- prepare (the stage is usually still busy: this is hidden behind the wait below) ----
            const int quad = e_cur.quad;
            const int qx = quad % g.NQx, rest = quad / g.NQx, by = rest % g.NBy, bz = rest / g.NBy;
            const int64_t org = g.idx(qx * 32, by * 8, bz * 8);
            bool tv = false;
            if (ADV) tv = a.qflagT_in[quad] != 0 && (a.tgate == nullptr || a.tgate[quad] != 0);
            const int nitems = e_cur.nitems & 0xffff;
            const uint32_t item_bytes = (uint32_t)((nitems * 2 + 15) & ~15);
            const int edge = (qx == 0) | (by == 0) | (bz == 0) | (qx * 32 + 32 + XW > g.nx) | (by * 8 + 8 + K > g.ny) |
                             (bz * 8 + 8 + K > g.nz);
            const int avail = g.nx - qx * 32;   // cells of this quad's rows that exist (the domain may cut the last quad)
            const T* qsrc = src + org;
            const uint16_t* item_src = a.items + (int64_t)quad * kItemsPerQuad;
            // ---- the stage's previous tenant has been consumed ----
            if (fill >= 1) mbar_wait(bar_empty + 8 * slot, (uint32_t)((fill - 1) & 1));
            // ---- fire ----
            if (lane == 0) {
                h->quad = quad;
                h->nitems = nitems;
                h->x0 = qx * 32; h->y0 = by * 8; h->z0 = bz * 8;
                h->org = org;
                h->edge = edge;
                h->tvalid = tv ? 1 : 0;
                mbar_expect_tx(bar, item_bytes + (ADV && tv ? 256 : 0));
                bulk_load(st + S::OFF_ITEMS, item_src, item_bytes, bar);
                if (ADV && tv) bulk_load(st + S::OFF_TM, a.tmask_in + (int64_t)quad * 32, 256, bar);
            }
#pragma unroll
            for (int k = 0; k < NPASS; ++k) {
                const uint32_t need = ((k < 4 ? n_cur.lo : n_cur.hi) >> (8 * (k & 3))) & 0xffu;
                if (need) {
                    const T* row = qsrc + rowoff[k];
                    const uint32_t m = st + m_off[k];
                    if ((need & 1u) && half == 0) cp_async16(st + S::OFF_L + h_off[k], row - XW);
                    if ((need & 32u) && half == 1) cp_async16(st + S::OFF_R + h_off[k], row + 32);
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch)
                        if (need & (2u << ch)) {
#pragma unroll
                            for (int q = 0; q < 4 / XW; ++q) {   // fp32: one 32-byte sector per chunk; fp64: two
                                const int c0 = ch * 8 + (q * 2 + half) * XW;
                                if (c0 < avail) cp_async16(m + c0 * (int)sizeof(T), row + c0);
                            }
                        }
                }
            }
            if (ADV && tv) {
                const T* qF = Fsrc + org;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t own = (n_cur.own >> (8 * k)) & 0xfu;
                    const T* row = qF + frowoff[k];
                    const uint32_t f = st + S::OFF_F + (uint32_t)((rslot + 16 * k) * 32 * (int)sizeof(T));
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch)
                        if (own & (1u << ch)) {
#pragma unroll
                            for (int q = 0; q < 4 / XW; ++q) {
                                const int c0 = ch * 8 + (q * 2 + half) * XW;
                                if (c0 < avail) cp_async16(f + c0 * (int)sizeof(T), row + c0);
                            }
                        }
                }
            }
            cp_async_arrive(bar);
            ++issued;
        }
        // sentinel: this stage gets no more work (NPW == 1: nor do the others, the consumers stop at the first one)
        {
            const int slot = NPW == 1 ? issued % STAGES : warp - NCW;
            const int fill = NPW == 1 ? issued / STAGES : issued;
            if (fill >= 1) mbar_wait(bar_empty + 8 * slot, (uint32_t)((fill - 1) & 1));
            if (lane == 0) {
                reinterpret_cast<Hdr*>(smem + slot * S::BYTES + S::OFF_HDR)->quad = -1;
                mbar_expect_tx(bar_full + 8 * slot, 0);
            }
            cp_async_arrive(bar_full + 8 * slot);
        }
        // self-resetting scheduler: the last producer warp to finish fetching zeroes the counters for the next launch
        if (lane == 0) {
            __threadfence();
            if (atomicAdd(a.ticket + 1, 1u) == gridDim.x * NPW - 1) { a.ticket[0] = 0u; a.ticket[1] = 0u; }
        }
        return;
    }
    if (warp == NCW) {
        // ------------------------------ producer, K = 2: one elected lane, TMA boxes ------------------------------
        if (lane != 0) return;
        int slot = 0, issued = 0;
        auto acquire = [&]() {   // the stage's previous tenant has been consumed
            if (issued >= STAGES) mbar_wait(bar_empty + 8 * slot, (uint32_t)((issued / STAGES - 1) & 1));
        };
        auto issue = [&](const QuadEntry e) {
            acquire();
            const int quad = e.quad;
            const int qx = quad % g.NQx, rest = quad / g.NQx, by = rest % g.NBy, bz = rest / g.NBy;
            Hdr* h = reinterpret_cast<Hdr*>(smem + slot * S::BYTES + S::OFF_HDR);
            const int nitems = e.nitems & 0xffff;
            // K = 1: the x halo is read only by items on that edge (band builder's flags); K = 2: always (ring cells)
            const bool haveL = K > 1 || ((e.nitems >> 16) & 1), haveR = K > 1 || ((e.nitems >> 17) & 1);
            h->quad = quad;
            h->nitems = nitems;
            h->x0 = qx * 32; h->y0 = by * 8; h->z0 = bz * 8;
            h->org = g.idx(qx * 32, by * 8, bz * 8);
            h->edge = (qx == 0) | (by == 0) | (bz == 0) | (qx * 32 + 32 + XW > g.nx) | (by * 8 + 8 + K > g.ny) |
                      (bz * 8 + 8 + K > g.nz);
            h->ring_n = 0;
            h->haveL = haveL;
            h->haveR = haveR;
            const uint32_t st = smem_base + slot * S::BYTES, bar = bar_full + 8 * slot;
            const uint32_t item_bytes = (uint32_t)((nitems * 2 + 15) & ~15);
            bool tv = false;
            if (ADV) tv = a.qflagT_in[quad] != 0 && (a.tgate == nullptr || a.tgate[quad] != 0);
            h->tvalid = tv ? 1 : 0;
            mbar_expect_tx(bar, S::M_BYTES + (haveL ? S::H_BYTES : 0) + (haveR ? S::H_BYTES : 0) + item_bytes +
                                    (ADV && tv ? S::F_BYTES + 256 : 0) + S::NB_BYTES);
            tma_load_3d(st, &tm_M, bar, h->x0, h->y0 - K, h->z0 - K);
            if (haveL) tma_load_3d(st + S::OFF_L, &tm_H, bar, h->x0 - XW, h->y0 - (K - 1), h->z0 - (K - 1));
            if (haveR) tma_load_3d(st + S::OFF_R, &tm_H, bar, h->x0 + 32, h->y0 - (K - 1), h->z0 - (K - 1));
            bulk_load(st + S::OFF_ITEMS, a.items + (int64_t)quad * kItemsPerQuad, item_bytes, bar);
            if (ADV && tv) {
                tma_load_3d(st + S::OFF_F, &tm_F, bar, h->x0, h->y0, h->z0);
                bulk_load(st + S::OFF_TM, a.tmask_in + (int64_t)quad * 32, 256, bar);
            }
            if (K > 1) {
                const int syq = g.NQx, szq = g.NQx * g.NBy;
                const uint64_t* z = reinterpret_cast<const uint64_t*>(a.zero_page);
                const uint32_t nb = st + S::OFF_NB;
                bulk_load(nb, by > 0 ? a.nmask + (int64_t)(quad - syq) * 32 : z, 256, bar);
                bulk_load(nb + 256, by < g.NBy - 1 ? a.nmask + (int64_t)(quad + syq) * 32 : z, 256, bar);
                bulk_load(nb + 512, bz > 0 ? a.nmask + (int64_t)(quad - szq) * 32 : z, 256, bar);
                bulk_load(nb + 768, bz < g.NBz - 1 ? a.nmask + (int64_t)(quad + szq) * 32 : z, 256, bar);
                bulk_load(nb + 1024, qx > 0 ? a.nmask + (int64_t)(quad - 1) * 32 + 24 : z, 64, bar);
                bulk_load(nb + 1088, qx < g.NQx - 1 ? a.nmask + (int64_t)(quad + 1) * 32 : z, 64, bar);
            }
            ++issued;
            slot = slot == STAGES - 1 ? 0 : slot + 1;
        };
        auto fetch = [&](int base, QuadEntry* e) {
#pragma unroll
            for (int i = 0; i < kChunk; ++i)
                if (base + i < count) e[i] = a.qlist[a.reverse ? count - 1 - (base + i) : base + i];
        };
        int base = (int)atomicAdd(a.ticket, (unsigned)kChunk);
        QuadEntry cur[kChunk], nxt[kChunk];
        fetch(base, cur);
        while (base < count) {
            const int nbase = (int)atomicAdd(a.ticket, (unsigned)kChunk);
            fetch(nbase, nxt);
#pragma unroll 1
            for (int i = 0; i < kChunk; ++i)
                if (base + i < count) issue(cur[i]);
#pragma unroll
            for (int i = 0; i < kChunk; ++i) cur[i] = nxt[i];
            base = nbase;
        }
        // sentinel: no more work
        acquire();
        reinterpret_cast<Hdr*>(smem + slot * S::BYTES + S::OFF_HDR)->quad = -1;
        mbar_arrive(bar_full + 8 * slot);
        // self-resetting scheduler: the last CTA to finish fetching zeroes the counters for the next launch
        __threadfence();
        if (atomicAdd(a.ticket + 1, 1u) == gridDim.x - 1) { a.ticket[0] = 0u; a.ticket[1] = 0u; }
        return;
    }

    // ------------------------------ consumers ------------------------------
    const int ctid = tid;   // 0 .. NC-1
    T rmax = T(0);
    int slot = 0, par = 0;
    uint32_t phases = 0;                       // parity of each stage's "full" barrier
    uint32_t alive = (1u << STAGES) - 1u;      // stages whose producer has not sent its sentinel yet
    int rot = 0;                               // tiles done: rotates which warp takes the first items of a tile
    auto next_slot = [&]() { slot = slot == STAGES - 1 ? 0 : slot + 1; };
    for (;;) {
        if (!((alive >> slot) & 1u)) { next_slot(); continue; }
        unsigned char* st = smem + slot * S::BYTES;
        mbar_wait(bar_full + 8 * slot, (phases >> slot) & 1u);
        phases ^= 1u << slot;
        Hdr* hp = reinterpret_cast<Hdr*>(st + S::OFF_HDR);
        const int quad = hp->quad;
        if (quad < 0) {   // one producer per stage: this stage's producer is done; a single producer: all work is done
            alive &= ~(1u << slot);
            if (NPW == 1 || alive == 0) break;
            next_slot();
            continue;
        }
        const int nitems = hp->nitems, edge = hp->edge;
        TL t;
        t.M = reinterpret_cast<T*>(st);
        t.L = reinterpret_cast<T*>(st + S::OFF_L);
        t.R = reinterpret_cast<T*>(st + S::OFF_R);
        if (edge) patch_boundary<T, K, NC>(t, g, hp->x0, hp->y0, hp->z0, ctid);
        const uint16_t* items = reinterpret_cast<const uint16_t*>(st + S::OFF_ITEMS);

        if (K == 2) {
            // ---- sweep 1 on the quad's N points and on the N points of the one-cell ring around it ----
            const unsigned char* nb = st + S::OFF_NB;
            uint32_t* ring = reinterpret_cast<uint32_t*>(st + S::OFF_RING);
            {   // ring list: one candidate group per consumer: face f (y-, y+, z-, z+), row r of the face, group xq
                const int f = ctid >> 6, r = (ctid >> 3) & 7, xq = ctid & 7, j = xq >> 1;
                int y, z, byte;
                if (f == 0) { y = -1; z = r; byte = j * 64 + r * 8 + 7; }
                else if (f == 1) { y = 8; z = r; byte = 256 + j * 64 + r * 8; }
                else if (f == 2) { y = r; z = -1; byte = 512 + j * 64 + 56 + r; }
                else { y = r; z = 8; byte = 768 + j * 64 + r; }
                const unsigned nib = ((unsigned)nb[byte] >> ((xq & 1) * 4)) & 0xfu;
                const unsigned vote = __ballot_sync(0xffffffffu, nib != 0);
                int wbase = 0;
                if (lane == 0 && vote) wbase = atomicAdd(&hp->ring_n, __popc(vote));
                wbase = __shfl_sync(0xffffffffu, wbase, 0);
                if (nib) ring[wbase + __popc(vote & ((1u << lane) - 1u))] = (uint32_t)(xq | ((y + 1) << 4) | ((z + 1) << 8) | (nib << 12));
            }
            consumer_sync<NC>();
            const int n1 = hp->ring_n, ntot = nitems + n1;
            constexpr int R1 = (kItemsPerQuad + 256 + NC - 1) / NC;   // rounds that cover the largest tile
            T keep[R1][4];
            int where[R1];
#pragma unroll
            for (int r = 0; r < R1; ++r) {
                const int p = ctid + r * NC;
                where[r] = -1;
                if (p < ntot) {
                    int xq, y, z;
                    unsigned nib;
                    if (p < nitems) {
                        const unsigned it = items[p];
                        nib = it >> 9; z = (it >> 6) & 7; y = (it >> 3) & 7; xq = it & 7;
                    } else {
                        const uint32_t e = ring[p - nitems];
                        xq = e & 7; y = (int)((e >> 4) & 15) - 1; z = (int)((e >> 8) & 15) - 1; nib = e >> 12;
                    }
                    Item4<T> s;
                    load_item<T, K>(t, xq, y, z, s);
                    T v[4];
                    reinit_item<T>(s, pr, v);
#pragma unroll
                    for (int e = 0; e < 4; ++e) keep[r][e] = ((nib >> e) & 1u) ? v[e] : s.c[e];
                    where[r] = TL::om(xq * 4, y, z);
                }
            }
            // x ring: cells x = -1 and x = 32 of the quad's own rows, one row per thread of the first two warps
            T xl = T(0), xr = T(0);
            bool nl = false, nr = false;
            int row_y = 0, row_z = 0;
            if (ctid < 64) {
                row_z = ctid >> 3; row_y = ctid & 7;
                nl = (nb[1024 + row_z * 8 + row_y] >> 7) & 1;
                nr = nb[1088 + row_z * 8 + row_y] & 1;
                if (nl) {
                    const int h = TL::oh(XW - 1, row_y, row_z);
                    xl = reinit_value<T>(t.L[h], t.L[h - 1], t.M[TL::om(0, row_y, row_z)], t.L[h - XW], t.L[h + XW],
                                         t.L[h - XW * TL::PH], t.L[h + XW * TL::PH], pr);
                }
                if (nr) {
                    const int h = TL::oh(0, row_y, row_z);
                    xr = reinit_value<T>(t.R[h], t.M[TL::om(31, row_y, row_z)], t.R[h + 1], t.R[h - XW], t.R[h + XW],
                                         t.R[h - XW * TL::PH], t.R[h + XW * TL::PH], pr);
                }
            }
            consumer_sync<NC>();   // every read of iteration k is done: write iteration k+1 in place
#pragma unroll
            for (int r = 0; r < R1; ++r)
                if (where[r] >= 0) store4<T>(t.M + where[r], keep[r]);
            if (nl) t.L[TL::oh(XW - 1, row_y, row_z)] = xl;
            if (nr) t.R[TL::oh(0, row_y, row_z)] = xr;
            fence_proxy_async();   // generic writes into a tile a later TMA load overwrites
            consumer_sync<NC>();
            if (edge) patch_boundary<T, K, NC>(t, g, hp->x0, hp->y0, hp->z0, ctid);   // edge replicate of iteration k+1
        }

        // ---- the launch's last operation on the quad's own items: results to the other global buffer ----
        const unsigned char* tm8 = st + S::OFF_TM;
        const T* Fb = reinterpret_cast<const T*>(st + S::OFF_F);
        T* out_base = dst + hp->org;
        const int tvalid = hp->tvalid;
        // A tile's items rarely fill a whole number of rounds: the warp that takes the first 32 items of every
        // round works longest.  Rotating that role from tile to tile evens the warps out over a few tiles (the
        // stages let them drift apart that far), so none of them ends up waiting for the slowest one.
        const int vtid = (((warp + rot) & (NCW - 1)) << 5) | lane;
        for (int p = vtid; p < nitems; p += NC) {
            const unsigned it = items[p];
            const unsigned nib = it >> 9;
            const int lz = (it >> 6) & 7, ly = (it >> 3) & 7, xq = it & 7;
            Item4<T> s;
            load_item<T, K>(t, xq, ly, lz, s);
            T v[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] = s.c[e];
            unsigned act = nib;   // cells whose value this launch changes
            if (ADV) {
                act = tvalid ? ((unsigned)tm8[(xq >> 1) * 64 + lz * 8 + ly] >> ((xq & 1) * 4)) & 0xfu : 0u;
                if (act) {
                    T f[4];
                    if (sizeof(T) == 4) {
                        const float4 fq = *reinterpret_cast<const float4*>(Fb + (lz * 8 + ly) * 32 + xq * 4);
                        f[0] = (T)fq.x; f[1] = (T)fq.y; f[2] = (T)fq.z; f[3] = (T)fq.w;
                    } else {
#pragma unroll
                        for (int e = 0; e < 4; ++e) f[e] = Fb[(lz * 8 + ly) * 32 + xq * 4 + e];
                    }
                    advance_item<T, false>(s, f, pa, v);
                }
            } else {
                reinit_item<T>(s, pr, v);
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const bool on = (act >> e) & 1u;
                if (RESIDUAL && on) rmax = fmax(rmax, mag(v[e] - s.c[e]));
                v[e] = on ? v[e] : s.c[e];
                if (CLAMP) v[e] = clamp_val(v[e], pr.gamma);
            }
            if (EMIT_T) {   // T of phi^{n+1} = clamp(d) at the item's N cells: one staging byte per item, no atomics
                unsigned tn = 0;
#pragma unroll
                for (int e = 0; e < 4; ++e) tn |= (((nib >> e) & 1u) && mag(v[e]) < pr.gamma) ? (1u << e) : 0u;
                tstage[par * 512 + (it & 511u)] = (unsigned char)tn;
            }
            store4<T>(out_base + (int64_t)(lz * g.ny + ly) * g.nx + xq * 4, v);
        }
        if (EMIT_T) {
            // T masks of phi^{n+1} = clamp(d) on this quad: T^{n+1} is a subset of N^n
            consumer_sync<NC>();   // every item's bits are in
            if (ctid < 32) {
                // lane (j, lz) packs the staging bytes of its brick layer (two item nibbles per mask byte) into word lz
                // of brick j, then clears them for the tile after the next one (a consumer_sync lies in between)
                unsigned char* ts = tstage + par * 512;
                const int j = ctid >> 3, lz = ctid & 7;
                uint64_t word = 0ull;
#pragma unroll
                for (int ly = 0; ly < 8; ++ly) {
                    const unsigned two = *reinterpret_cast<const unsigned short*>(ts + lz * 64 + ly * 8 + 2 * j);
                    word |= (uint64_t)((two & 0xfu) | ((two >> 4) & 0xf0u)) << (8 * ly);
                }
                __syncwarp();
                reinterpret_cast<uint4*>(ts)[ctid] = make_uint4(0u, 0u, 0u, 0u);
                a.tmask_out[(int64_t)quad * 32 + ctid] = word;
                const unsigned any = __ballot_sync(0xffffffffu, word != 0ull);
                if (ctid == 0) a.qflagT_out[quad] = any ? 1 : 0;
            }
            par ^= 1;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
        ++rot;
        next_slot();
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
        if (lane == 0 && bits != 0) atomicMax(a.residual, bits);
    }
}

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
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Persistent grid of a band kernel: the largest shared-memory carve-out, then as many CTAs as fit on an SM.
template <typename Kn>
int persistent_grid(Kn kernel, int threads, size_t dyn_smem) {
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem);
    cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, dyn_smem) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    return sm_count() * per_sm;
}

struct Maps { CUtensorMap M, H, F; };

template <typename T, bool ADV, int K, bool CLAMP, bool RESIDUAL, bool EMIT_T>
void launch_variant(const Maps& m, T* dst, const Geom& g, const StencilParams<T>& pa, const StencilParams<T>& pr,
                    const TileArgs& a, cudaStream_t s) {
#ifndef LS_K1_STAGES
#define LS_K1_STAGES 2
#endif
#ifndef LS_K1_NPW
#define LS_K1_NPW 0   // 0: one producer warp per stage
#endif
#ifndef LS_F64_NCW
#define LS_F64_NCW 8
#endif
#ifndef LS_F64_STAGES
#define LS_F64_STAGES 2
#endif
    // consumer warps per CTA: four is the measured optimum in fp32; fp64 needs 80 registers and 29 KB
    // per stage, so few CTAs fit an SM and eight consumer warps each keep more of them in flight (78.7 against 82.5 us)
    constexpr int NCW = K > 1 ? 8 : (sizeof(T) == 8 ? LS_F64_NCW : 4);
#ifndef LS_ADV_STAGES
#define LS_ADV_STAGES 2
#endif
    constexpr int STAGES = K > 1 ? 2 : (sizeof(T) == 8 ? LS_F64_STAGES : (ADV ? LS_ADV_STAGES : LS_K1_STAGES));
    // K = 1: gather warps (one per stage, or one for all stages); K = 2: one lane issuing TMA boxes
    constexpr int NPW = K > 1 ? 1 : (LS_K1_NPW ? LS_K1_NPW : STAGES);
    using S = Stage<T, K, ADV>;
    const size_t shm = (size_t)STAGES * S::BYTES + (EMIT_T ? 1024 : 0) + 16 * STAGES;
    auto kern = k_band_tile<T, ADV, K, CLAMP, RESIDUAL, EMIT_T, STAGES, NCW, NPW>;
    // (the grid is sized once per process for the device current at the first launch: every B200 is alike)
    static const int grid = persistent_grid(kern, (NCW + NPW) * 32, shm);
    kern<<<grid, (NCW + NPW) * 32, shm, s>>>(m.M, m.H, m.F, dst, g, pa, pr, a);
}

}  // namespace

template <typename T>
bool tile_usable(const Geom& g, const void* a, const void* b, const void* c) {
    if (g.nx % 4 != 0) return false;                                        // items are aligned groups of 4 cells
    if (((size_t)g.nx * g.ny * sizeof(T)) >= ((size_t)1 << 40)) return false;   // tensor-map stride limit
    const uintptr_t bits = reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(c);
    return (bits & 15) == 0 && encode_fn() != nullptr;
}

template <typename T>
bool launch_band_tile(const T* src, const T* F, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                      const BandOp& op, cudaStream_t s, int64_t* launches) {
    const int K = (op.advance ? 1 : 0) + op.sweeps;
    if (K < 1 || K > 2 || (op.advance && K != 1)) return false;
    constexpr int XW = 16 / (int)sizeof(T);
    Maps m;
    std::memset(&m, 0, sizeof m);
    if (K == 2) {   // only the two-sweep kernels load whole boxes by TMA; the gather kernels take no tensor map
        if (!make_map<T>(&m.M, src, g, 32, 8 + 2 * K, 8 + 2 * K)) return false;
        if (!make_map<T>(&m.H, src, g, XW, 6 + 2 * K, 6 + 2 * K)) return false;
        m.F = m.M;
    }
    TileArgs a;
    a.qlist = bb.qlist[op.list];
    a.count = &bb.counts->nQ[op.list];
    a.items = bb.items[op.list];
    a.qneed = bb.qneed[op.list];
    a.nmask = bb.nmask;
    a.zero_page = bb.zero_page;
    a.tmask_in = bb.tmask[bb.tb];
    a.qflagT_in = bb.qflagT[bb.tb];
    a.tgate = op.tgate;
    a.tmask_out = bb.tmask[bb.tb ^ 1];
    a.qflagT_out = bb.qflagT[bb.tb ^ 1];
    a.residual = op.residual;
    a.src = src;
    a.F = F;
    a.ticket = bb.counts->ticket;
    a.reverse = op.reverse ? 1 : 0;
#define LS_VARIANTS(KK)                                                                                      \
    do {                                                                                                     \
        if (op.emit_T) launch_variant<T, false, KK, true, false, true>(m, dst, g, p, p, a, s);               \
        else if (op.residual && op.clamp) launch_variant<T, false, KK, true, true, false>(m, dst, g, p, p, a, s);  \
        else if (op.residual) launch_variant<T, false, KK, false, true, false>(m, dst, g, p, p, a, s);       \
        else if (op.clamp) launch_variant<T, false, KK, true, false, false>(m, dst, g, p, p, a, s);          \
        else launch_variant<T, false, KK, false, false, false>(m, dst, g, p, p, a, s);                       \
    } while (0)
    if (op.advance) launch_variant<T, true, 1, false, false, false>(m, dst, g, p, p, a, s);
    else if (K == 2) LS_VARIANTS(2);
    else LS_VARIANTS(1);
#undef LS_VARIANTS
    if (launches) *launches += 1;
    return true;
}

#define LS_INSTANTIATE(T)                                                                                       \
    template bool tile_usable<T>(const Geom&, const void*, const void*, const void*);                           \
    template bool launch_band_tile<T>(const T*, const T*, T*, const Geom&, const StencilParams<T>&,            \
                                      const BandBuffers&, const BandOp&, cudaStream_t, int64_t*);
LS_INSTANTIATE(float)
LS_INSTANTIATE(double)

}  // namespace ls
