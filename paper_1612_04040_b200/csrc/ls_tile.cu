// ls_tile.cu — the band kernels of Steps 2 and 3: persistent, warp-specialised, TMA-fed.
//
// Tile = one QUAD (four x-adjacent 8^3 bricks, 32 x 8 x 8 points; ls_internal.h) plus a halo of K cells in
// y and z and of one 16-byte piece in x (fp32: 4 cells, fp64: 2), K = number of operations fused in the
// launch (Advance and / or reinit sweeps: temporal blocking).  Every tile row is
// 160 (fp32) / 288 (fp64) contiguous bytes of a field row that starts 16 bytes before a 128-byte line.
//
//   producer warp (one elected lane)   takes quads from the ordered quad list through a device ticket
//        counter (chunks of 4), and per quad issues ONE cp.async.bulk.tensor.3d box load of the halo tile
//        straight from the dense x-fastest field, one cp.async.bulk of the quad's
//        precomputed item list (and, for Advance, the 32x8x8 box of F and the quad's 32 T mask words), all
//        completing on the stage's "full" mbarrier; it waits on the stage's "empty" mbarrier before reuse.
//   4 consumer warps   wait on "full"; edge-replicate the out-of-domain halo (R3; TMA zero-fills it);
//        lane l evaluates items l, l+128, ...: one item = 4 x-consecutive cells = 5 LDS.128 + 2 LDS.32,
//        two packed fp32 pairs through eq. 3-8 / eq. 12-13 (ls_math.cuh), one 16-byte store — Jacobi: reads
//        come from the tile, results go to the other global buffer (K = 1) or to the second tile buffer
//        (K > 1).  No CTA barrier per tile: each warp arrives on "empty" when it is done with the stage.
// The arithmetic is bit-identical to the scalar kernels of ls_stencil.cu, which remain the path for grids the
// tile path cannot address (nx not a multiple of 4, unaligned fields).
#include <cuda.h>

#include "ls_internal.h"
#include "ls_math.cuh"

namespace ls {

namespace {

constexpr int kConsumerWarps = 4;
constexpr int kConsumers = kConsumerWarps * 32;
constexpr int kThreads = kConsumers + 32;   // + the producer warp
constexpr int kChunk = 4;                   // quads per ticket

template <typename T> struct XHalo;
template <> struct XHalo<float> { static constexpr int XH = 4; };
template <> struct XHalo<double> { static constexpr int XH = 2; };

constexpr int round128(int x) { return (x + 127) / 128 * 128; }

// Header of a stage, written by the producer before it starts the loads of the stage.
struct alignas(16) Hdr {
    int quad;       // quad id; -1: no more work
    int nitems;
    int x0, y0, z0; // first cell of the quad
    int edge;       // tile reaches outside the domain (halo needs patching)
    long long org;  // element offset of the first cell in the dense field
    int tvalid;     // Advance: T masks were loaded (else the quad holds no T point)
    int pad;
};

// One pipeline stage in shared memory.
template <typename T, int K, bool ADV>
struct Stage {
    static constexpr int XH = XHalo<T>::XH;
    static constexpr int PX = 32 + 2 * XH;
    static constexpr int PY = 8 + 2 * K;
    static constexpr int ELEMS = PX * PY * PY;
    static constexpr int TILE_BYTES = ELEMS * (int)sizeof(T);
    static constexpr int OFF_TILE2 = round128(TILE_BYTES);                       // second tile buffer (K > 1)
    static constexpr int OFF_F = OFF_TILE2 + (K > 1 ? round128(TILE_BYTES) : 0);
    static constexpr int F_BYTES = ADV ? 2048 * (int)sizeof(T) : 0;
    static constexpr int OFF_ITEMS = OFF_F + F_BYTES;
    static constexpr int ITEM_BYTES = kItemsPerQuad * 2;
    static constexpr int OFF_TM = OFF_ITEMS + ITEM_BYTES;
    static constexpr int TM_BYTES = ADV ? 256 : 0;
    static constexpr int OFF_HDR = OFF_TM + TM_BYTES;
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
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory"); }

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

// R3: TMA zero-fills cells outside the domain; give them the value of the nearest in-domain cell (edge
// replicate).  Sources are in-domain cells, destinations are not: no ordering needed inside.  Only called for
// tiles that reach outside the domain (uniform over the consumers).  `tile` may be either tile buffer.
template <typename T, int PX, int PY, int XH, int K>
__device__ __noinline__ void patch_boundary(T* tile, const Geom& g, int x0, int y0, int z0, int ctid) {
    const int ox = x0 - XH, oy = y0 - K, oz = z0 - K;
    for (int e = ctid; e < PX * PY * PY; e += kConsumers) {
        const int x = e % PX, r = e / PX, y = r % PY, z = r / PY;
        const int gx = ox + x, gy = oy + y, gz = oz + z;
        const int cx = min(max(gx, 0), g.nx - 1), cy = min(max(gy, 0), g.ny - 1), cz = min(max(gz, 0), g.nz - 1);
        if (cx != gx || cy != gy || cz != gz) {
            const int sx = cx - ox, sy = cy - oy, sz = cz - oz;
            if (sx >= 0 && sx < PX && sy >= 0 && sy < PY && sz >= 0 && sz < PY) tile[e] = tile[(sz * PY + sy) * PX + sx];
        }
    }
    fence_proxy_async();   // generic writes into a tile a later TMA load overwrites
    consumer_sync();
}

// The stencil of the item whose first cell sits at tile offset o.
template <typename T, int PX, int PY>
__device__ __forceinline__ void load_item(const T* tile, int o, Item4<T>& s) {
    constexpr int SY = PX, SZ = PX * PY;
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
    s.xm = tile[o - 1];
    s.xp = tile[o + 4];
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
    const uint64_t* tmask_in;     // Advance: T masks of the band (tmask[tb])
    const uint8_t* qflagT_in;
    const uint8_t* tgate;         // null or validity gate of tmask_in
    uint64_t* tmask_out;          // EMIT_T: tmask[tb ^ 1]
    uint8_t* qflagT_out;
    unsigned long long* residual;
    unsigned int* ticket;         // [0] next list index, [1] CTAs done (self-resetting)
    int reverse;                  // walk the list from its end (L2 reuse between consecutive sweeps)
};

// ---------------------------------------------------------------------------------------------
// One launch = (ADV ? Advance : nothing) followed by SWEEPS reinit sweeps on every listed quad, K = ADV + SWEEPS
// operations deep, results of the last operation written to `dst` at the item cells.
// ---------------------------------------------------------------------------------------------
template <typename T, bool ADV, int SWEEPS, bool CLAMP, bool RESIDUAL, bool EMIT_T, int STAGES>
__global__ void __launch_bounds__(kThreads)
k_band_tile(const __grid_constant__ CUtensorMap tm_src, const __grid_constant__ CUtensorMap tm_F, T* __restrict__ dst,
            Geom g, StencilParams<T> pa, StencilParams<T> pr, TileArgs a) {
    constexpr int K = (ADV ? 1 : 0) + SWEEPS;
    static_assert(K == 1, "temporal blocking (K > 1) is built by k_band_tile_multi");
    using S = Stage<T, K, ADV>;
    constexpr int PX = S::PX, PY = S::PY, XH = S::XH;
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t smem_base = smem_u32(smem);
    // after the stages: T staging of EMIT_T (2 x 256 B), then the mbarriers (full[STAGES], empty[STAGES])
    uint32_t* tstage = reinterpret_cast<uint32_t*>(smem + STAGES * S::BYTES);
    const uint32_t bar_full = smem_base + STAGES * S::BYTES + 512, bar_empty = bar_full + 8 * STAGES;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, kConsumerWarps); }
        fence_barrier_init();
    }
    if (EMIT_T && tid < 128) tstage[tid] = 0u;
    __syncthreads();
    const int count = *a.count;

    if (warp == kConsumerWarps) {
        // ------------------------------ producer ------------------------------
        if (lane != 0) return;
        int slot = 0, issued = 0;
        auto acquire = [&]() {   // the stage's previous tenant has been consumed
            if (issued >= STAGES) mbar_wait(bar_empty + 8 * slot, (uint32_t)((issued / STAGES - 1) & 1));
        };
        auto advance_slot = [&]() { ++issued; slot = slot == STAGES - 1 ? 0 : slot + 1; };
        auto issue = [&](const QuadEntry e) {
            acquire();
            const int quad = e.quad;
            const int qx = quad % g.NQx, rest = quad / g.NQx, by = rest % g.NBy, bz = rest / g.NBy;
            Hdr* h = reinterpret_cast<Hdr*>(smem + slot * S::BYTES + S::OFF_HDR);
            h->quad = quad;
            h->nitems = e.nitems;
            h->x0 = qx * 32; h->y0 = by * 8; h->z0 = bz * 8;
            h->org = g.idx(qx * 32, by * 8, bz * 8);
            h->edge = (qx == 0) | (by == 0) | (bz == 0) | (qx * 32 + 32 + XH > g.nx) | (by * 8 + 8 + K > g.ny) |
                      (bz * 8 + 8 + K > g.nz);
            const uint32_t st = smem_base + slot * S::BYTES, bar = bar_full + 8 * slot;
            const uint32_t item_bytes = (uint32_t)((e.nitems * 2 + 15) & ~15);
            bool tv = false;
            if (ADV) tv = a.qflagT_in[quad] != 0 && (a.tgate == nullptr || a.tgate[quad] != 0);
            h->tvalid = tv ? 1 : 0;
            mbar_expect_tx(bar, S::TILE_BYTES + item_bytes + (ADV && tv ? S::F_BYTES + 256 : 0));
            tma_load_3d(st, &tm_src, bar, h->x0 - XH, h->y0 - K, h->z0 - K);
            bulk_load(st + S::OFF_ITEMS, a.items + (int64_t)quad * kItemsPerQuad, item_bytes, bar);
            if (ADV && tv) {
                tma_load_3d(st + S::OFF_F, &tm_F, bar, h->x0, h->y0, h->z0);
                bulk_load(st + S::OFF_TM, a.tmask_in + (int64_t)quad * 32, 256, bar);
            }
            advance_slot();
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
#pragma unroll
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
    const int ctid = tid;   // 0..127
    T rmax = T(0);
    int slot = 0, par = 0;
    uint32_t phase = 0;
    for (;;) {
        unsigned char* st = smem + slot * S::BYTES;
        mbar_wait(bar_full + 8 * slot, phase);
        const Hdr h = *reinterpret_cast<const Hdr*>(st + S::OFF_HDR);
        if (h.quad < 0) break;
        T* tile = reinterpret_cast<T*>(st);
        if (h.edge) patch_boundary<T, PX, PY, XH, K>(tile, g, h.x0, h.y0, h.z0, ctid);
        const uint16_t* items = reinterpret_cast<const uint16_t*>(st + S::OFF_ITEMS);
        const unsigned char* tm8 = st + S::OFF_TM;
        const T* Fb = reinterpret_cast<const T*>(st + S::OFF_F);
        T* out_base = dst + h.org;
        for (int p = ctid; p < h.nitems; p += kConsumers) {
            const unsigned it = items[p];
            const unsigned nib = it >> 9;
            const int lz = (it >> 6) & 7, ly = (it >> 3) & 7, xq = it & 7;
            const int o = ((lz + K) * PY + (ly + K)) * PX + XH + xq * 4;
            Item4<T> s;
            load_item<T, PX, PY>(tile, o, s);
            T v[4];
            unsigned act = nib;   // cells whose value this launch changes
            if (ADV) {
                act = h.tvalid ? ((unsigned)tm8[(xq >> 1) * 64 + lz * 8 + ly] >> ((xq & 1) * 4)) & 0xfu : 0u;
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
            if (EMIT_T) {
                unsigned tn = 0;
#pragma unroll
                for (int e = 0; e < 4; ++e) tn |= (((nib >> e) & 1u) && mag(v[e]) < pr.gamma) ? (1u << e) : 0u;
                if (tn) atomicOr(tstage + par * 64 + ((xq >> 1) * 8 + lz) * 2 + (ly >> 2), tn << ((ly & 3) * 8 + (xq & 1) * 4));
            }
            store4<T>(out_base + (int64_t)(lz * g.ny + ly) * g.nx + xq * 4, v);
        }
        if (EMIT_T) {
            // T masks of phi^{n+1} = clamp(d) on this quad: T^{n+1} is a subset of N^n
            consumer_sync();   // every item's bits are in
            if (ctid < 32) {
                uint64_t* w64 = reinterpret_cast<uint64_t*>(tstage + par * 64);
                const uint64_t word = w64[ctid];
                w64[ctid] = 0ull;   // ready for the tile after the next one (a consumer_sync lies in between)
                a.tmask_out[(int64_t)h.quad * 32 + ctid] = word;
                const unsigned any = __ballot_sync(0xffffffffu, word != 0ull);
                if (ctid == 0) a.qflagT_out[h.quad] = any ? 1 : 0;
            }
            par ^= 1;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
        if (++slot == STAGES) { slot = 0; phase ^= 1u; }
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
int persistent_grid(Kn kernel, size_t dyn_smem) {
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem);
    cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, dyn_smem) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    return sm_count() * per_sm;
}

template <typename T, bool ADV, int SWEEPS, bool CLAMP, bool RESIDUAL, bool EMIT_T>
void launch_variant(const CUtensorMap& tm_src, const CUtensorMap& tm_F, T* dst, const Geom& g, const StencilParams<T>& pa,
                    const StencilParams<T>& pr, const TileArgs& a, cudaStream_t s) {
    constexpr int K = (ADV ? 1 : 0) + SWEEPS;
    constexpr int STAGES = (ADV || sizeof(T) == 8) ? 2 : 3;
    using S = Stage<T, K, ADV>;
    const size_t shm = (size_t)STAGES * S::BYTES + 512 + 16 * STAGES;
    auto kern = k_band_tile<T, ADV, SWEEPS, CLAMP, RESIDUAL, EMIT_T, STAGES>;
    static const int grid = persistent_grid(kern, shm);
    kern<<<grid, kThreads, shm, s>>>(tm_src, tm_F, dst, g, pa, pr, a);
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
    if (K != 1) return false;
    constexpr int XH = XHalo<T>::XH;
    CUtensorMap tm_src, tm_F;
    if (!make_map<T>(&tm_src, src, g, 32 + 2 * XH, 8 + 2 * K, 8 + 2 * K)) return false;
    if (op.advance) {
        if (!make_map<T>(&tm_F, F, g, 32, 8, 8)) return false;
    } else {
        tm_F = tm_src;
    }
    TileArgs a;
    a.qlist = bb.qlist[op.list];
    a.count = &bb.counts->nQ[op.list];
    a.items = bb.items[op.list];
    a.tmask_in = bb.tmask[bb.tb];
    a.qflagT_in = bb.qflagT[bb.tb];
    a.tgate = op.tgate;
    a.tmask_out = bb.tmask[bb.tb ^ 1];
    a.qflagT_out = bb.qflagT[bb.tb ^ 1];
    a.residual = op.residual;
    a.ticket = bb.counts->ticket;
    a.reverse = op.reverse ? 1 : 0;
    if (op.advance) launch_variant<T, true, 0, false, false, false>(tm_src, tm_F, dst, g, p, p, a, s);
    else if (op.emit_T) launch_variant<T, false, 1, true, false, true>(tm_src, tm_F, dst, g, p, p, a, s);
    else if (op.residual && op.clamp) launch_variant<T, false, 1, true, true, false>(tm_src, tm_F, dst, g, p, p, a, s);
    else if (op.residual) launch_variant<T, false, 1, false, true, false>(tm_src, tm_F, dst, g, p, p, a, s);
    else if (op.clamp) launch_variant<T, false, 1, true, false, false>(tm_src, tm_F, dst, g, p, p, a, s);
    else launch_variant<T, false, 1, false, false, false>(tm_src, tm_F, dst, g, p, p, a, s);
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
