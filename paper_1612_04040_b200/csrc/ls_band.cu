// ls_band.cu — Step 1: tubes T (eq. 6) and N (eq. 11).
//
// Kernels
//   k_classify        whole-grid sweep, one CTA per x-row of quads (32x8x8 points each), 128-bit
//                     coalesced loads; T bits are assembled into brick mask words with warp REDUX (no atomics).
//   k_dilate_items    one WARP per candidate quad: lane (j, lz) builds N word lz of brick j from its own T
//                     word, its neighbours' words by shuffle, and the facing bit planes of the six
//                     neighbour quads (eq. 11, R6); then the quad's item list (ls_internal.h) by a warp
//                     scan.  Candidates: every quad (first build, LS_REBUILD_FULL) or, incrementally, the
//                     quads of the previous band and their face neighbours (T^{n+1} is a subset of N^n,
//                     PAPER.md:65) — O(band), not O(grid).  Counts |T| and |N| (integer adds commute).
//   k_compact         ordered stream compaction of the quad flags into the quad list: per-CTA counts, one
//                     grid barrier, exclusive scan, scatter — ascending quad id whatever the scheduling
//                     (R20: no atomics-order dependence).  Also folds the point counters.
//   k_export_*        brick lists in ls.h's format (ascending brick id + 8 mask words per brick) for
//                     ls_band_counts / ls_band_export, derived from the quad list on demand.
#include "ls_internal.h"

namespace ls {

namespace {

constexpr uint64_t COL0 = 0x0101010101010101ull;  // lx == 0 in every row
constexpr uint64_t COL7 = 0x8080808080808080ull;  // lx == 7 in every row

template <typename T> __device__ __forceinline__ T absval(T v);
template <> __device__ __forceinline__ float absval<float>(float v) { return fabsf(v); }
template <> __device__ __forceinline__ double absval<double>(double v) { return fabs(v); }

// One CTA = one x-row of quads (by, bz), a segment of `qper` of them; one quad = 32(x) x 8(y) x 8(z) points.  Warp w owns
// z-layer w; lane l owns the 4 consecutive x cells x4 = l&7 of row y = (l>>3) + 4h, h = 0,1.  With VEC the 4 cells are one
// 128-bit load and a warp load covers 4 full 128-byte lines.  The CTA walks its quads along x, so the coordinates and row
// pointers are set up once and a quad costs two loads, eight compares and two REDUX per lane (round 1 launched one CTA per
// quad: the set-up made it issue bound at 55 % of the copy bandwidth).  Writes all 32 mask words of every quad (zeros
// included) and its flag.
template <typename T, bool VEC>
__global__ void __launch_bounds__(256) k_classify(const T* __restrict__ phi, Geom g, T gamma, int qper,
                                                  uint64_t* __restrict__ tmask, uint8_t* __restrict__ qflagT) {
    __shared__ uint32_t half_words[2][8][4][2];  // [parity of the quad][lz][brick in quad][low/high 32 bits]
    const int nseg = (g.NQx + qper - 1) / qper;
    const int seg = blockIdx.x % nseg, rowid = blockIdx.x / nseg;   // rowid = bz * NBy + by
    const int by = rowid % g.NBy, bz = rowid / g.NBy;
    const int lane = threadIdx.x & 31, lz = threadIdx.x >> 5;
    const int k = bz * 8 + lz;
    const int x4 = lane & 7;
    const int q = x4 >> 1;                                  // brick of the quad this lane feeds
    const unsigned group = 0x03030303u << (2 * q);          // the 8 lanes feeding the same 32-bit half
    const T* row[2];
    bool row_ok[2];
    unsigned shift[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int ly = (lane >> 3) + 4 * h;
        const int j = by * 8 + ly;
        row_ok[h] = k < g.nz && j < g.ny;
        row[h] = phi + g.idx(0, row_ok[h] ? j : 0, row_ok[h] ? k : 0);
        shift[h] = (ly & 3) * 8 + (x4 & 1) * 4;             // bit position inside the 32-bit half: row (ly & 3), columns (x4 & 1)*4 ..
    }
    const int q0 = seg * qper, q1 = min(g.NQx, q0 + qper);
    for (int qx = q0; qx < q1; ++qx) {
        const int i0 = qx * 32 + x4 * 4;
        const int par = (qx - q0) & 1;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            unsigned bits = 0;
            if (row_ok[h] && i0 < g.nx) {
                if (VEC) {  // nx % 4 == 0 here, so i0 + 3 < nx
                    if (sizeof(T) == 4) {
                        const float4 v = __ldg(reinterpret_cast<const float4*>(row[h] + i0));
                        bits = (absval<T>((T)v.x) < gamma ? 1u : 0u) | (absval<T>((T)v.y) < gamma ? 2u : 0u) |
                               (absval<T>((T)v.z) < gamma ? 4u : 0u) | (absval<T>((T)v.w) < gamma ? 8u : 0u);
                    } else {
                        const double2 a = __ldg(reinterpret_cast<const double2*>(row[h] + i0));
                        const double2 b = __ldg(reinterpret_cast<const double2*>(row[h] + i0 + 2));
                        bits = (absval<T>((T)a.x) < gamma ? 1u : 0u) | (absval<T>((T)a.y) < gamma ? 2u : 0u) |
                               (absval<T>((T)b.x) < gamma ? 4u : 0u) | (absval<T>((T)b.y) < gamma ? 8u : 0u);
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < 4; ++e)
                        if (i0 + e < g.nx && absval<T>(__ldg(row[h] + i0 + e)) < gamma) bits |= 1u << e;
                }
            }
            const unsigned r = __reduce_or_sync(group, bits << shift[h]);
            if ((lane & 0x19) == 0) half_words[par][lz][q][h] = r;   // lanes 0,2,4,6: first lane of each group
        }
        __syncthreads();   // (the other parity's words were read before the previous barrier's successor: see below)
        if (threadIdx.x < 32) {
            // warp 0 assembles the quad's 32 words; it reaches the next barrier only after these reads, and the words of
            // this parity are next written two quads later, after that barrier
            const int qq = threadIdx.x >> 3, z = threadIdx.x & 7;
            const uint64_t word = (uint64_t)half_words[par][z][qq][0] | ((uint64_t)half_words[par][z][qq][1] << 32);
            const unsigned nz_lanes = __ballot_sync(0xffffffffu, word != 0);
            const int64_t quad = (int64_t)rowid * g.NQx + qx;
            tmask[quad * 32 + threadIdx.x] = word;
            if (threadIdx.x == 0) qflagT[quad] = nz_lanes ? 1 : 0;
        }
    }
}

// Bits of the cells of brick (bx,by,bz), word lz, that lie inside the domain.
__device__ __forceinline__ uint64_t domain_word(const Geom& g, int bx, int by, int bz, int lz) {
    if (bx >= g.NBx || bz * 8 + lz >= g.nz) return 0;
    const int vx = min(8, g.nx - bx * 8), vy = min(8, g.ny - by * 8);
    const uint64_t rowbits = (1ull << vx) - 1ull;            // vx <= 8
    uint64_t w = rowbits * COL0;                             // replicate into all 8 rows
    if (vy < 8) w &= (1ull << (8 * vy)) - 1ull;
    return w;
}

struct DilateArgs {
    const uint64_t* tmask;     // T masks to dilate
    const uint8_t* qflagT;
    const uint8_t* tgate;      // null: T valid for every quad; else T valid only where tgate != 0 (= qflagN of the previous band)
    const uint8_t* prevN;      // qflagN of the previous band (list buffer lb)
    const QuadEntry* prevList; // its quad list ...
    const int32_t* prevCount;  // ... and length
    const QuadEntry* staleList;// quad list last stored in the buffer being rebuilt (its flags must be cleared) ...
    const int32_t* staleCount; // ... and length
    uint64_t* nmask;
    uint8_t* qflagN;           // out: flags of the band being built
    int32_t* qcount;           // out: items per quad
    uint16_t* items;           // out: item lists
    uint8_t* qneed;            // out: load maps
    Counts* counts;
};

constexpr int kDilateWarps = 4;

// Which quad does candidate `wid` stand for?  -1: none (out of range, or another candidate owns the quad).
// Incremental candidates: (entry e of the previous list, direction d = self, -x, +x, -y, +y, -z, +z), then the
// quads of the stale list.  A quad is processed by exactly one candidate: the first (e, d) in direction order
// that reaches it; stale entries only if no (e, d) reaches them.
__device__ __forceinline__ int candidate_quad(const Geom& g, const DilateArgs& a, int64_t wid, int nprev, int nstale) {
    const int sxq = 1, syq = g.NQx, szq = g.NQx * g.NBy;
    const int dq[7] = {0, -sxq, sxq, -syq, syq, -szq, szq};
    if (wid < (int64_t)nprev * 7) {
        const int e = (int)(wid / 7), d = (int)(wid % 7);
        const int sq = a.prevList[e].quad;
        const int qx = sq % g.NQx, by = (sq / g.NQx) % g.NBy, bz = sq / szq;
        const bool inside = d == 0 || (d == 1 && qx > 0) || (d == 2 && qx < g.NQx - 1) || (d == 3 && by > 0) ||
                            (d == 4 && by < g.NBy - 1) || (d == 5 && bz > 0) || (d == 6 && bz < g.NBz - 1);
        if (!inside) return -1;
        const int c = sq + dq[d];
        if (d != 0) {
            if (a.prevN[c]) return -1;   // reached by its own (e', self)
            const int cx = c % g.NQx, cy = (c / g.NQx) % g.NBy, cz = c / szq;
            for (int dd = 1; dd < d; ++dd) {   // an earlier direction dd reaches c from the source c - dq[dd]
                const bool in2 = (dd == 1 && cx < g.NQx - 1) || (dd == 2 && cx > 0) || (dd == 3 && cy < g.NBy - 1) ||
                                 (dd == 4 && cy > 0) || (dd == 5 && cz < g.NBz - 1) || (dd == 6 && cz > 0);
                if (in2 && a.prevN[c - dq[dd]]) return -1;
            }
        }
        return c;
    }
    if (wid < (int64_t)nprev * 7 + nstale) {
        const int c = a.staleList[(int)(wid - (int64_t)nprev * 7)].quad;
        const int cx = c % g.NQx, cy = (c / g.NQx) % g.NBy, cz = c / szq;
        bool reached = a.prevN[c] != 0;
        reached = reached || (cx > 0 && a.prevN[c - sxq]) || (cx < g.NQx - 1 && a.prevN[c + sxq]);
        reached = reached || (cy > 0 && a.prevN[c - syq]) || (cy < g.NBy - 1 && a.prevN[c + syq]);
        reached = reached || (cz > 0 && a.prevN[c - szq]) || (cz < g.NBz - 1 && a.prevN[c + szq]);
        return reached ? -1 : c;
    }
    return -1;
}

// eq. 11 (R6): N = T or any in-domain face neighbour in T.  Persistent warps, one candidate quad per warp and turn.
template <bool INCREMENTAL>
__global__ void __launch_bounds__(kDilateWarps * 32) k_dilate_items(Geom g, DilateArgs a) {
    __shared__ __align__(16) uint64_t s_words[kDilateWarps][32];
    __shared__ __align__(16) uint16_t s_items[kDilateWarps][kItemsPerQuad];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int sxq = 1, syq = g.NQx, szq = g.NQx * g.NBy;
    const int nprev = INCREMENTAL ? *a.prevCount : 0, nstale = INCREMENTAL ? *a.staleCount : 0;
    const int64_t ncand = INCREMENTAL ? (int64_t)nprev * 7 + nstale : (int64_t)g.nquads;
    const int64_t nwarps = (int64_t)gridDim.x * kDilateWarps;
    // T masks are valid for quad q if its flag is set and (incremental builds) it lay in the previous band.  Both
    // bytes are loaded unconditionally (no dependent branch between them): what this kernel waits for is the flags.
    const uint8_t* gate = a.tgate != nullptr ? a.tgate : a.qflagT;
    auto tvalid = [&](bool inside, int q) -> unsigned { return inside ? ((a.qflagT[q] != 0) & (gate[q] != 0) ? 1u : 0u) : 0u; };
    // A warp turn takes up to 32 consecutive candidates: each lane resolves one (which quad, does another candidate own
    // it, which of the quad and its six face neighbours hold valid T masks) with its flag loads in flight together;
    // the quads that can hold an N point are then processed one after the other by the whole warp.
    // On a short candidate list a turn takes fewer than 32 (`per`), so that the quads to process — a serial loop per
    // warp — spread over all warps of the grid instead of piling up on the first ncand / 32 of them.
    const int per = (int)(ncand >= nwarps * 32 ? 32 : (ncand + nwarps - 1) / nwarps < 1 ? 1 : (ncand + nwarps - 1) / nwarps);
    for (int64_t w0 = ((int64_t)blockIdx.x * kDilateWarps + wib) * per; w0 < ncand; w0 += nwarps * per) {
    int mine = -1, my_x = 0, my_y = 0, my_z = 0;
    unsigned my_valid = 0;   // bit 0: the quad itself, bits 1..6: its -x, +x, -y, +y, -z, +z neighbour
    {
        const int64_t wid = w0 + lane;
        int c = -1;
        if (lane < per && wid < ncand) c = INCREMENTAL ? candidate_quad(g, a, wid, nprev, nstale) : (int)wid;
        if (c >= 0) {
            const int cx = c % g.NQx, cy = (c / g.NQx) % g.NBy, cz = c / szq;
            my_x = cx; my_y = cy; my_z = cz;
            my_valid = tvalid(true, c) | (tvalid(cx > 0, c - sxq) << 1) | (tvalid(cx < g.NQx - 1, c + sxq) << 2) |
                       (tvalid(cy > 0, c - syq) << 3) | (tvalid(cy < g.NBy - 1, c + syq) << 4) |
                       (tvalid(cz > 0, c - szq) << 5) | (tvalid(cz < g.NBz - 1, c + szq) << 6);
            if (my_valid) {
                mine = c;
            } else {
                // no T point in reach: the quad is outside N.  Its masks are already zero unless it was in the
                // previous band (or, when rebuilding incrementally, in the stale band of this buffer).
                if (INCREMENTAL || a.prevN[c]) {
                    uint4* z = reinterpret_cast<uint4*>(a.nmask + (int64_t)c * 32);
#pragma unroll
                    for (int i = 0; i < 16; ++i) z[i] = make_uint4(0u, 0u, 0u, 0u);
                }
                a.qflagN[c] = 0;
                a.qcount[c] = 0;
            }
        }
    }
    unsigned todo = __ballot_sync(0xffffffffu, mine >= 0);
    while (todo) {
    const int src_lane = __ffs(todo) - 1;
    todo &= todo - 1;
    const int c = __shfl_sync(0xffffffffu, mine, src_lane);
    const int qx = __shfl_sync(0xffffffffu, my_x, src_lane), by = __shfl_sync(0xffffffffu, my_y, src_lane);
    const int bz = __shfl_sync(0xffffffffu, my_z, src_lane);
    const unsigned vm = __shfl_sync(0xffffffffu, my_valid, src_lane);
    __syncwarp();   // the staging of the previous quad has been copied out
    const bool vs = vm & 1u, vxm = vm & 2u, vxp = vm & 4u, vym = vm & 8u, vyp = vm & 16u, vzm = vm & 32u, vzp = vm & 64u;
    const int j = lane >> 3, lz = lane & 7;   // brick of the quad, word of the brick
    const uint64_t w = vs ? a.tmask[(int64_t)c * 32 + lane] : 0ull;
    uint64_t n = w | ((w << 1) & ~COL0) | ((w >> 1) & ~COL7) | (w << 8) | (w >> 8);
    // z neighbours: the lane below / above, or the facing word of the quad below / above
    {
        uint64_t dn = __shfl_up_sync(0xffffffffu, w, 1), up = __shfl_down_sync(0xffffffffu, w, 1);
        if (lz == 0) dn = vzm ? a.tmask[(int64_t)(c - szq) * 32 + j * 8 + 7] : 0ull;
        if (lz == 7) up = vzp ? a.tmask[(int64_t)(c + szq) * 32 + j * 8 + 0] : 0ull;
        n |= dn | up;
    }
    // x neighbours: brick j-1 / j+1 of this quad (8 lanes away), or brick 3 / 0 of the quad to the left / right
    {
        uint64_t lf = __shfl_up_sync(0xffffffffu, w, 8), rt = __shfl_down_sync(0xffffffffu, w, 8);
        if (j == 0) lf = vxm ? a.tmask[(int64_t)(c - sxq) * 32 + 24 + lz] : 0ull;
        if (j == 3) rt = vxp ? a.tmask[(int64_t)(c + sxq) * 32 + lz] : 0ull;
        n |= (lf >> 7) & COL0;     // their lx = 7 -> our lx = 0
        n |= (rt & COL0) << 7;     // their lx = 0 -> our lx = 7
    }
    if (vym) n |= a.tmask[(int64_t)(c - syq) * 32 + lane] >> 56;              // their ly = 7 -> our ly = 0
    if (vyp) n |= (a.tmask[(int64_t)(c + syq) * 32 + lane] & 0xffull) << 56;  // their ly = 0 -> our ly = 7
    n &= domain_word(g, qx * 4 + j, by, bz, lz);
    a.nmask[(int64_t)c * 32 + lane] = n;
    // |T|, |N|
    {
        const unsigned pT = __reduce_add_sync(0xffffffffu, (unsigned)__popcll(w));
        const unsigned pN = __reduce_add_sync(0xffffffffu, (unsigned)__popcll(n));
        if (lane == 0) {
            if (pT) atomicAdd(&a.counts->acc_T, (unsigned long long)pT);
            if (pN) atomicAdd(&a.counts->acc_N, (unsigned long long)pN);
        }
    }
    // Item list in row-major order (lz, ly, xq): lane l takes rows (lz = l >> 2, ly = 2*(l & 3) + {0, 1}); a row's
    // 32 bits are byte ly of word lz of the four bricks.
    s_words[wib][lane] = n;
    __syncwarp();
    const unsigned char* sb = reinterpret_cast<const unsigned char*>(s_words[wib]);
    const int rz = lane >> 2, ry = (lane & 3) * 2;
    uint32_t row[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int o = rz * 8 + ry + r;
        row[r] = (uint32_t)sb[o] | ((uint32_t)sb[64 + o] << 8) | ((uint32_t)sb[128 + o] << 16) | ((uint32_t)sb[192 + o] << 24);
    }
    int cnt = 0;
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int x = 0; x < 8; ++x) cnt += ((row[r] >> (4 * x)) & 0xfu) ? 1 : 0;
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    int pos = incl - cnt;
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            const uint32_t nib = (row[r] >> (4 * x)) & 0xfu;
            if (nib) s_items[wib][pos++] = (uint16_t)((rz * 64 + (ry + r) * 8 + x) | (nib << 9));
        }
    __syncwarp();
    // copy out in 16-byte pieces (the tail piece may carry unused entries; the slot is 1 KiB)
    {
        const uint4* src = reinterpret_cast<const uint4*>(s_items[wib]);
        uint4* dst = reinterpret_cast<uint4*>(a.items + (int64_t)c * kItemsPerQuad);
        const int pieces = (total + 7) >> 3;
        for (int i = lane; i < pieces; i += 32) dst[i] = src[i];
    }
    // Load map (kNeedBytes, ls_internal.h): a chunk is needed if an N point of the quad reads one of its cells:
    // its own chunk, the same chunk one row up / down in y or z, or — for a point in the first / last cell of a
    // chunk — the chunk next to it in x.  Pieces outside the domain are never needed (edge replicate patches them).
    // Lane (j, lz) reduces its word to three 8-bit masks over y: R = rows of brick j, layer lz that hold an N point,
    // E0 / E7 = rows whose first / last cell is one; the needs of the chunks of brick j in layer lz are then
    // D = R | R<<1 | R>>1 | R(lz-1) | R(lz+1) | E7(j-1) | E0(j+1), and a transposition through shared memory
    // turns the per-(j, lz) masks over y into the per-row bytes over chunks.
    {
        auto gather = [](uint64_t m) -> unsigned {   // bit 0 of each byte -> one 8-bit mask
            return (unsigned)(((m & COL0) * 0x0102040810204080ull) >> 56);
        };
        uint64_t f = n | (n >> 4);
        f |= f >> 2;
        f |= f >> 1;
        const unsigned R = gather(f), E0 = gather(n), E7 = gather(n >> 7);
        const unsigned Rdn = __shfl_up_sync(0xffffffffu, R, 1), Rup = __shfl_down_sync(0xffffffffu, R, 1);
        const unsigned E7l = __shfl_up_sync(0xffffffffu, E7, 8), E0r = __shfl_down_sync(0xffffffffu, E0, 8);
        unsigned D = R | ((R << 1) & 0xffu) | (R >> 1);
        if (lz > 0) D |= Rdn;
        if (lz < 7) D |= Rup;
        if (j > 0) D |= E7l;
        if (j < 3) D |= E0r;
        __syncwarp();   // s_words (read as `sb` above) is reused as the transposition buffer
        unsigned char* tb = reinterpret_cast<unsigned char*>(s_words[wib]);   // [0,32) D(j,lz)  [32,64) R(j,lz)  [64,72) E0(0,lz)  [72,80) E7(3,lz)
        tb[lane] = (unsigned char)D;
        tb[32 + lane] = (unsigned char)R;
        if (j == 0) tb[64 + lz] = (unsigned char)E0;
        if (j == 3) tb[72 + lz] = (unsigned char)E7;
        __syncwarp();
        // Per tile row (y, z): which sectors are needed.  Lanes 0..31 take the 64 quad rows two at a time (z = lane / 4,
        // y = 2 (lane % 4) + {0, 1}); then one halo row each: y = -1, y = 8 (read by the quad row next to them), z = -1,
        // z = 8 (corner rows are never read).  Pieces outside the domain are never needed (edge replicate patches them).
        uint8_t* need_out = a.qneed + (int64_t)c * kNeedBytes;
        unsigned xclip = 0x3fu;   // sectors of a row that lie inside the domain in x
        if (qx == 0) xclip &= ~1u;
#pragma unroll
        for (int ch = 0; ch < 5; ++ch)
            if (qx * 32 + ch * 8 >= g.nx) xclip &= ~(2u << ch);
        {
            const int z = lane >> 2, y0 = (lane & 3) * 2;
            const unsigned d0 = tb[z], d1 = tb[8 + z], d2 = tb[16 + z], d3 = tb[24 + z], e0 = tb[64 + z], e7 = tb[72 + z];
            const unsigned r0 = tb[32 + z], r1 = tb[40 + z], r2 = tb[48 + z], r3 = tb[56 + z];
            const bool zin = bz * 8 + z < g.nz;
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int y = y0 + k;
                unsigned need = ((e0 >> y) & 1u) | (((d0 >> y) & 1u) << 1) | (((d1 >> y) & 1u) << 2) | (((d2 >> y) & 1u) << 3) |
                                (((d3 >> y) & 1u) << 4) | (((e7 >> y) & 1u) << 5);
                if (!zin || by * 8 + y >= g.ny) need = 0;
                need_out[(z + 1) * 10 + (y + 1)] = (uint8_t)(need & xclip);
                const unsigned own = ((r0 >> y) & 1u) | (((r1 >> y) & 1u) << 1) | (((r2 >> y) & 1u) << 2) | (((r3 >> y) & 1u) << 3);
                need_out[112 + z * 8 + y] = (uint8_t)own;
            }
        }
        {
            const int kind = lane >> 3, i = lane & 7;   // 0: y = -1, 1: y = 8 (i = z);  2: z = -1, 3: z = 8 (i = y)
            const int zr = kind < 2 ? i : (kind == 2 ? 0 : 7);              // the layer whose rows read this halo row
            const int sh = kind < 2 ? (kind == 0 ? 0 : 7) : i;              // the row of that layer which does
            unsigned need = 0;
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) need |= (((unsigned)tb[32 + jj * 8 + zr] >> sh) & 1u) << (1 + jj);
            const int y = kind < 2 ? (kind == 0 ? -1 : 8) : i, z = kind < 2 ? i : (kind == 2 ? -1 : 8);
            const int gy = by * 8 + y, gz = bz * 8 + z;
            if (gy < 0 || gy >= g.ny || gz < 0 || gz >= g.nz) need = 0;
            need_out[(z + 1) * 10 + (y + 1)] = (uint8_t)(need & xclip);
            if (lane < 4) need_out[(lane >> 1) * 90 + (lane & 1) * 9] = 0;   // the four corner rows
        }
    }
    // does an N point sit on the quad's low-x / high-x face?  (the band kernels load that x halo only then)
    const unsigned faceL = __ballot_sync(0xffffffffu, j == 0 && (n & COL0) != 0);
    const unsigned faceR = __ballot_sync(0xffffffffu, j == 3 && (n & COL7) != 0);
    if (lane == 0) { a.qflagN[c] = total ? 1 : 0; a.qcount[c] = total | (faceL ? 1 << 16 : 0) | (faceR ? 1 << 17 : 0); }
    }   // quads of this turn
    }   // turns
}

// ---- ordered compaction of the quad flags --------------------------------------------------------
constexpr int kCompactThreads = 1024;
constexpr int kFlagsPerThread = 16;
constexpr int kCompactTile = kCompactThreads * kFlagsPerThread;

__device__ __forceinline__ uint32_t flag_bits16(const uint8_t* flags, int64_t base, int64_t n) {
    uint32_t m = 0;
    if (base + 16 <= n) {
        const uint4 v = *reinterpret_cast<const uint4*>(flags + base);
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 16; ++i) m |= (((w[i >> 2] >> ((i & 3) * 8)) & 0xffu) ? 1u : 0u) << i;
    } else {
        for (int i = 0; i < 16; ++i)
            if (base + i < n && flags[base + i]) m |= 1u << i;
    }
    return m;
}

// CTA-wide exclusive scan of one int per thread; returns the exclusive prefix, *total = CTA sum.
__device__ __forceinline__ int cta_exclusive_scan(int v, int* s_warp, int* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    __syncthreads();   // s_warp may still be read from a previous call
    if (lane == 31) s_warp[w] = incl;
    __syncthreads();
    if (w == 0) {
        const int x = s_warp[lane];
        int s = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        s_warp[lane] = s - x;          // exclusive over warps
        if (lane == 31) s_warp[32] = s; // CTA total
    }
    __syncthreads();
    *total = s_warp[32];
    return s_warp[w] + incl - v;
}

// All CTAs of the grid are co-resident (grid <= SM count, one CTA per SM fits): phase 1 counts, a grid
// barrier on a monotone counter, phase 2 scans and scatters.  Output order = ascending quad id.
__global__ void __launch_bounds__(kCompactThreads) k_compact(const uint8_t* __restrict__ qflagN,
                                                             const int32_t* __restrict__ qcount, int nquads,
                                                             QuadEntry* __restrict__ qlist, int32_t* __restrict__ partials,
                                                             Counts* __restrict__ counts, int which,
                                                             unsigned long long bar_target, int iters, int count_step) {
    __shared__ int s_warp[33];
    const int G = gridDim.x;
    const int64_t ntiles = ((int64_t)nquads + kCompactTile - 1) / kCompactTile;
    const int64_t tiles_per = (ntiles + G - 1) / G;
    const int64_t t0 = (int64_t)blockIdx.x * tiles_per, t1 = min(ntiles, t0 + tiles_per);
    // phase 1: flags of my range
    int mine = 0;
    for (int64_t t = t0; t < t1; ++t)
        mine += __popc(flag_bits16(qflagN, t * kCompactTile + (int64_t)threadIdx.x * kFlagsPerThread, nquads));
    int total;
    cta_exclusive_scan(mine, s_warp, &total);
    if (G > 1) {   // a single CTA (small grids) has nobody to wait for
        if (threadIdx.x == 0) {
            partials[blockIdx.x] = total;
            __threadfence();
            atomicAdd(&counts->bar, 1ull);
            while (*reinterpret_cast<volatile unsigned long long*>(&counts->bar) < bar_target) {}
            __threadfence();
        }
        __syncthreads();
    }
    // phase 2: my base = sum of the partials before me
    int base = 0;
    {
        int v = 0;
        for (int i = threadIdx.x; i < (int)blockIdx.x; i += kCompactThreads) v += __ldcg(partials + i);
        int dummy;
        cta_exclusive_scan(v, s_warp, &dummy);
        base = dummy;
    }
    if (blockIdx.x == G - 1 && threadIdx.x == 0) {
        counts->nQ[which] = base + total;
        // fold the point counters of this build (k_dilate_items has finished: stream order)
        counts->nT_pts = counts->acc_T;
        counts->nN_pts = counts->acc_N;
        counts->acc_T = 0;
        counts->acc_N = 0;
        if (count_step) {
            counts->updates += counts->nT_pts + (unsigned long long)iters * counts->nN_pts;
            counts->steps += 1;
        }
        for (int i = 0; i < kTickets; ++i) counts->ticket[i] = 0;
    }
    for (int64_t t = t0; t < t1; ++t) {
        const int64_t first = t * kCompactTile + (int64_t)threadIdx.x * kFlagsPerThread;
        const uint32_t m = flag_bits16(qflagN, first, nquads);
        int tile_total;
        int pos = base + cta_exclusive_scan(__popc(m), s_warp, &tile_total);
        uint32_t mm = m;
        while (mm) {
            const int i = __ffs(mm) - 1;
            mm &= mm - 1;
            QuadEntry e;
            e.quad = (int)(first + i);
            e.nitems = qcount[first + i];
            qlist[pos++] = e;
        }
        base += tile_total;
    }
}

// ---- export: brick lists in ls.h's format --------------------------------------------------------
struct ExportArgs {
    const QuadEntry* qlist;
    const int32_t* count;
    const uint64_t* tmask;
    const uint8_t* qflagT;
    const uint8_t* tgate;
    const uint64_t* nmask;
    int32_t* ex_cnt;   // [2][nquads]: per list entry, T bricks / N bricks, then exclusive scans
    int32_t* T_ids;
    int32_t* N_ids;
    uint64_t* T_masks;
    uint64_t* N_masks;
    Counts* counts;
    int nquads;
};

// per list entry: which of the quad's 4 bricks hold T / N points (bit j)
__device__ __forceinline__ void quad_brick_bits(const ExportArgs& a, int quad, unsigned& bT, unsigned& bN) {
    bT = bN = 0;
    const bool tv = a.qflagT[quad] != 0 && (a.tgate == nullptr || a.tgate[quad] != 0);
    for (int j = 0; j < 4; ++j) {
        uint64_t t = 0, n = 0;
        for (int z = 0; z < 8; ++z) {
            if (tv) t |= a.tmask[(int64_t)quad * 32 + j * 8 + z];
            n |= a.nmask[(int64_t)quad * 32 + j * 8 + z];
        }
        bT |= (t ? 1u : 0u) << j;
        bN |= (n ? 1u : 0u) << j;
    }
}

__global__ void __launch_bounds__(256) k_export_count(ExportArgs a) {
    const int n = *a.count;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        unsigned bT, bN;
        quad_brick_bits(a, a.qlist[e].quad, bT, bN);
        a.ex_cnt[e] = __popc(bT);
        a.ex_cnt[a.nquads + e] = __popc(bN);
    }
}

// exclusive scans of the two count arrays, in place; one CTA.
__global__ void __launch_bounds__(1024) k_export_scan(ExportArgs a) {
    __shared__ int s_warp[33];
    const int n = *a.count;
    for (int l = 0; l < 2; ++l) {
        int32_t* p = a.ex_cnt + (int64_t)l * a.nquads;
        int carry = 0;
        for (int base = 0; base < n; base += 1024) {
            const int i = base + threadIdx.x;
            const int v = i < n ? p[i] : 0;
            int total;
            const int ex = cta_exclusive_scan(v, s_warp, &total);
            if (i < n) p[i] = carry + ex;
            carry += total;
        }
        if (threadIdx.x == 0) {
            if (l == 0) a.counts->nT_bricks = carry;
            else a.counts->nN_bricks = carry;
        }
    }
}

__global__ void __launch_bounds__(256) k_export_scatter(ExportArgs a, Geom g, int with_masks) {
    const int n = *a.count;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const int quad = a.qlist[e].quad;
        unsigned bT, bN;
        quad_brick_bits(a, quad, bT, bN);
        const int qx = quad % g.NQx, rest = quad / g.NQx;   // rest = bz*NBy + by
        int pT = a.ex_cnt[e], pN = a.ex_cnt[a.nquads + e];
        for (int j = 0; j < 4; ++j) {
            const int b = rest * g.NBx + qx * 4 + j;   // true brick id (ls.h)
            if ((bT >> j) & 1u) {
                a.T_ids[pT] = b;
                if (with_masks)
                    for (int z = 0; z < 8; ++z) a.T_masks[(int64_t)pT * 8 + z] = a.tmask[(int64_t)quad * 32 + j * 8 + z];
                ++pT;
            }
            if ((bN >> j) & 1u) {
                a.N_ids[pN] = b;
                if (with_masks)
                    for (int z = 0; z < 8; ++z) a.N_masks[(int64_t)pN * 8 + z] = a.nmask[(int64_t)quad * 32 + j * 8 + z];
                ++pN;
            }
        }
    }
}

}  // namespace

template <typename T>
void launch_classify(const T* phi, const Geom& g, T gamma, BandBuffers& bb, cudaStream_t s, int64_t* launches) {
    const bool vec = (g.nx % 4 == 0) && ((reinterpret_cast<uintptr_t>(phi) & 15) == 0);
    // one CTA per x-row of quads, split into segments while that leaves fewer CTAs than a few waves of the GPU
    const int rows = g.NBy * g.NBz;
    int qper = g.NQx;
    while (qper > 4 && (int64_t)rows * ((g.NQx + qper - 1) / qper) < (int64_t)sm_count() * 16) qper = (qper + 1) / 2;
    const unsigned grid = (unsigned)(rows * ((g.NQx + qper - 1) / qper));
    if (vec)
        k_classify<T, true><<<grid, 256, 0, s>>>(phi, g, gamma, qper, bb.tmask[bb.tb], bb.qflagT[bb.tb]);
    else
        k_classify<T, false><<<grid, 256, 0, s>>>(phi, g, gamma, qper, bb.tmask[bb.tb], bb.qflagT[bb.tb]);
    bb.tvalid_all = true;
    if (launches) *launches += 1;
}

void launch_build_lists(const Geom& g, BandBuffers& bb, bool incremental, int iters, bool count_step, cudaStream_t s,
                        int64_t* launches) {
    const int pv = bb.lb, cr = bb.lb ^ 1;
    DilateArgs a;
    a.tmask = bb.tmask[bb.tb];
    a.qflagT = bb.qflagT[bb.tb];
    a.tgate = bb.tvalid_all ? nullptr : bb.qflagN[pv];
    a.prevN = bb.qflagN[pv];
    a.prevList = bb.qlist[pv];
    a.prevCount = &bb.counts->nQ[pv];
    a.staleList = bb.qlist[cr];
    a.staleCount = &bb.counts->nQ[cr];
    a.nmask = bb.nmask;
    a.qflagN = bb.qflagN[cr];
    a.qcount = bb.qcount;
    a.items = bb.items[cr];
    a.qneed = bb.qneed[cr];
    a.counts = bb.counts;
    // Persistent warps: the candidate count lives on the device (ls_step never synchronises).
    const unsigned blocks = (unsigned)(sm_count() * 8);
    if (incremental)
        k_dilate_items<true><<<blocks, kDilateWarps * 32, 0, s>>>(g, a);
    else
        k_dilate_items<false><<<blocks, kDilateWarps * 32, 0, s>>>(g, a);
    bb.bar_epoch += 1;
    k_compact<<<bb.compact_grid, kCompactThreads, 0, s>>>(bb.qflagN[cr], bb.qcount, g.nquads, bb.qlist[cr], bb.partials,
                                                          bb.counts, cr, bb.bar_epoch * (unsigned long long)bb.compact_grid,
                                                          iters, count_step ? 1 : 0);
    bb.lb = cr;
    if (launches) *launches += 2;
}

bool launch_export(const Geom& g, BandBuffers& bb, bool with_masks, cudaStream_t s, int64_t* launches) {
    if (!bb.ex_cnt) {
        cudaError_t e = cudaMalloc((void**)&bb.ex_cnt, (size_t)g.nquads * 2 * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMalloc((void**)&bb.T_ids, (size_t)g.nquads * 4 * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMalloc((void**)&bb.N_ids, (size_t)g.nquads * 4 * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMalloc((void**)&bb.T_masks, (size_t)g.nquads * 32 * sizeof(uint64_t));
        if (e == cudaSuccess) e = cudaMalloc((void**)&bb.N_masks, (size_t)g.nquads * 32 * sizeof(uint64_t));
        if (e != cudaSuccess) { cudaGetLastError(); return false; }
    }
    ExportArgs a;
    a.qlist = bb.qlist[bb.lb];
    a.count = &bb.counts->nQ[bb.lb];
    a.tmask = bb.tmask[bb.tb];
    a.qflagT = bb.qflagT[bb.tb];
    a.tgate = bb.tvalid_all ? nullptr : bb.qflagN[bb.lb ^ 1];
    a.nmask = bb.nmask;
    a.ex_cnt = bb.ex_cnt;
    a.T_ids = bb.T_ids;
    a.N_ids = bb.N_ids;
    a.T_masks = bb.T_masks;
    a.N_masks = bb.N_masks;
    a.counts = bb.counts;
    a.nquads = g.nquads;
    const int grid = sm_count() * 4;
    k_export_count<<<grid, 256, 0, s>>>(a);
    k_export_scan<<<1, 1024, 0, s>>>(a);
    k_export_scatter<<<grid, 256, 0, s>>>(a, g, with_masks ? 1 : 0);
    if (launches) *launches += 3;
    return true;
}

// |T| + iters * |N| of the band last built, over the z layers [z0, z1) only, added to `out->updates` (and `add_steps` to
// out->steps): the z-slab pipeline of ls_step_host runs the step on windows with halo layers and must count each point of
// the grid once.  One thread per mask word (quad, brick j, lz); integer adds commute.
__global__ void __launch_bounds__(256) k_count_layers(const uint64_t* __restrict__ tmask, const uint64_t* __restrict__ nmask,
                                                      Geom g, int z0, int z1, int iters, int add_steps, Counts* out) {
    __shared__ unsigned long long sh[8];
    const int64_t nwords = (int64_t)g.nquads * 32;
    unsigned long long v = 0;
    for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < nwords; w += (int64_t)gridDim.x * blockDim.x) {
        const int quad = (int)(w >> 5), lz = (int)(w & 7);
        const int z = (quad / (g.NQx * g.NBy)) * 8 + lz;
        if (z >= z0 && z < z1)
            v += (unsigned long long)__popcll(tmask[w]) + (unsigned long long)iters * (unsigned long long)__popcll(nmask[w]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int i = 0; i < 8; ++i) t += sh[i];
        if (t) atomicAdd(&out->updates, t);
        if (blockIdx.x == 0 && add_steps) atomicAdd(&out->steps, (unsigned long long)add_steps);
    }
}

void launch_count_layers(const Geom& g, const BandBuffers& bb, int z0, int z1, int iters, int add_steps, Counts* out,
                         cudaStream_t s, int64_t* launches) {
    const int64_t nwords = (int64_t)g.nquads * 32;
    const int64_t want = (nwords + 255) / 256, cap = (int64_t)sm_count() * 8;
    const int grid = (int)(want < cap ? want : cap);
    k_count_layers<<<grid, 256, 0, s>>>(bb.tmask[bb.tb], bb.nmask, g, z0, z1, iters, add_steps, out);
    if (launches) *launches += 1;
}

template void launch_classify<float>(const float*, const Geom&, float, BandBuffers&, cudaStream_t, int64_t*);
template void launch_classify<double>(const double*, const Geom&, double, BandBuffers&, cudaStream_t, int64_t*);

}  // namespace ls
