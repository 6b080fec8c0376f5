// ls_internal.h — shared declarations of the CUDA path (libls.so).  Not part of the public ABI.
// Nothing here is shared with oracle/ (the CPU oracle is an independent restatement of the paper).
//
// Band representation.  The grid is cut into 8^3 bricks (R20) and bricks into
// QUADS: four x-adjacent bricks, 32 x 8 x 8 points, whose rows are whole 128-byte lines of an fp32
// field.  A quad is the tile of the band kernels.  Per quad the ctx keeps
//   * 32 T mask words and 32 N mask words (brick j = 0..3, word lz = 0..7, bit ly*8 + lx), dense by
//     padded brick id  pb = 4*quad + j  (so a quad's masks are 256 contiguous bytes),
//   * an ITEM LIST of the band N: one uint16 per aligned group of four x-consecutive cells that holds
//     at least one N point (code = lz*64 + ly*8 + xq, xq = 0..7 the group within the 32-cell row;
//     bits 9..12 = which of the four cells are in N).  One lane of a band kernel evaluates one item
//     (two packed fp32 pairs), so lanes are 92 % full although a brick is only 56 % N points.
// Lists of quads (ascending quad id; built by an ordered scan, no atomics-order dependence) drive the
// band kernels; brick lists in the paper's / ls.h's format are derived on demand for ls_band_export.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ls {

// Grid geometry (x fastest), its 8^3 bricks (R20) and quads of bricks.
struct Geom {
    int nx, ny, nz;
    int NBx, NBy, NBz;   // bricks per axis
    int NQx;             // quads per x row = ceil(NBx / 4)
    int nbricks;         // NBx*NBy*NBz (true brick ids of ls.h)
    int nquads;          // NQx*NBy*NBz
    __host__ __device__ inline int64_t idx(int i, int j, int k) const {
        return ((int64_t)k * ny + j) * nx + i;
    }
};

constexpr int kItemsPerQuad = 512;   // 64 rows x 8 groups of 4 cells
// Load map of a quad's tile (one-sweep band kernels): which 32-byte brick rows ("chunks") of the 10 x 10 tile
// rows hold a cell that some N point of the quad reads — the band kernels fetch only those.
//   [0, 100)    need byte of tile row rz*10 + ry (rz = z + 1, ry = y + 1): bit 0 = the x-halo piece left of the
//               quad, bits 1..4 = chunks 0..3 of the quad, bit 5 = the x-halo piece right of it
//   [112, 176)  own byte of quad row z*8 + y: bit j = brick j has an N point in that row (Advance reads F there)
constexpr int kNeedBytes = 176;
constexpr int kTickets = 16;

// One entry of a quad list.
struct QuadEntry {
    int32_t quad;    // quad id
    int32_t nitems;  // items in its list (1..512) | x-face flags, see BandBuffers::qcount
};

// Device-resident counters, written by the band builder, read by the band kernels (so the host
// never needs them inside ls_step).
struct Counts {
    int32_t nQ[2];         // quads in the N quad list of each list buffer
    unsigned long long nT_pts, nN_pts;  // |T|, |N| of the band last built
    unsigned long long acc_T, acc_N;    // accumulators of the build in flight, folded by k_compact
    unsigned long long updates;         // sum over steps of |T| + iters*|N|
    unsigned long long steps;
    unsigned long long bar;             // grid barrier of k_compact (monotone)
    unsigned int ticket[kTickets];      // dynamic tile schedulers of the band kernels of one step
    // export scratch (ls_band_counts / ls_band_export)
    int32_t nT_bricks, nN_bricks;
};

// Everything the band builder owns, as raw device pointers.  [2] = double buffered by step parity.
struct BandBuffers {
    uint64_t* tmask[2];   // [nquads*32] T mask words.  Buffer `tb` holds T of the band last built; the last
                          // sweep of an incremental step writes T of phi^{n+1} into the other one, which the
                          // next step adopts (tb ^= 1) before its Advance.
    uint8_t* qflagT[2];   // [nquads] quad holds a T point (valid as tmask is, see tvalid_all)
    uint64_t* nmask;      // [nquads*32] N mask words of the band last built; all-zero for quads outside N
    uint8_t* qflagN[2];   // [nquads] quad holds an N point, per list buffer
    uint16_t* items[2];   // [nquads*512] item lists, dense by quad id, per list buffer
    uint8_t* qneed[2];    // [nquads*kNeedBytes] load maps, dense by quad id, per list buffer
    int32_t* qcount;      // [nquads] items of the quad in the band being built (bits 0-15) | N point on the quad's
                          // low-x face (bit 16) / high-x face (bit 17): the band kernels load that x halo only then
    void* zero_page;      // 256 zero bytes
    QuadEntry* qlist[2];  // [nquads] N quad list per list buffer
    int32_t* partials;    // [<= 1024] per-CTA counts of k_compact
    Counts* counts;
    // export scratch, allocated on first use: brick-level lists in ls.h's format
    int32_t* ex_cnt;      // [2*nquads] per listed quad: T bricks, N bricks (then their exclusive scans)
    int32_t* T_ids;
    int32_t* N_ids;
    uint64_t* T_masks;
    uint64_t* N_masks;
    // host-side state
    int tb;               // T buffer of the band last built
    int lb;               // list buffer of the band last built
    bool tvalid_all;      // tmask[tb] / qflagT[tb] valid for every quad (after a whole-grid classify); otherwise
                          // only for quads with qflagN[lb ^ 1] (emitted by the last sweep over that band)
    unsigned long long bar_epoch;   // launches of k_compact so far
    int compact_grid;
};

// ---- band builder (ls_band.cu) --------------------------------------------------------------
// Whole-grid classification |phi| < gamma into tmask[bb.tb] / qflagT[bb.tb] (eq. 6); sets tvalid_all.
template <typename T>
void launch_classify(const T* phi, const Geom& g, T gamma, BandBuffers& bb, cudaStream_t s, int64_t* launches);
// N = one-cell face dilation of T (eq. 11) for every quad that can hold N points, item lists, then the
// ordered quad list, into list buffer lb ^ 1, which becomes lb.  `incremental`: visit only the quads of the
// previous band and their face neighbours (T^{n+1} is a subset of N^n); else every quad.
// `iters` only feeds the update counter (|T| + iters*|N|).
void launch_build_lists(const Geom& g, BandBuffers& bb, bool incremental, int iters, bool count_step, cudaStream_t s,
                        int64_t* launches);
// Brick lists of the band last built in ls.h's format into T_ids / T_masks / N_ids / N_masks and the brick
// counts into Counts (allocates the export scratch on first use; returns false if that fails).
bool launch_export(const Geom& g, BandBuffers& bb, bool with_masks, cudaStream_t s, int64_t* launches);

// Adds |T| + iters * |N| of the band last built, restricted to the z layers [z0, z1), to out->updates and add_steps to
// out->steps (`out` may belong to another ctx: the z-slab pipeline of ls_step_host counts each grid point once).
// Requires tmask[tb] valid for every quad (a whole-grid classify built the band).
void launch_count_layers(const Geom& g, const BandBuffers& bb, int z0, int z1, int iters, int add_steps, Counts* out,
                         cudaStream_t s, int64_t* launches);

// ---- stencil parameters -----------------------------------------------------------------------
template <typename T>
struct StencilParams {
    T inv_dx;      // 1/dx
    T half_inv_dx; // inv_dx / 2 (exact)
    T dx2;         // dx*dx
    T dt;          // dt (advance) or dtau (reinit)
    T beta, gamma, three_beta, inv3;  // eq. 7 constants, inv3 = 1/((gamma-beta)^3)
};

// What one launch of a band kernel does to the band (ls_tile.cu, ls_stencil.cu).
struct BandOp {
    bool advance = false;   // Step 2 (eq. 3/8) on the T bits of the items; other cells of an item are copied
    int sweeps = 0;         // Step 3 sweeps (eq. 12-13) fused after it (temporal blocking); advance + sweeps >= 1
    bool copy = false;      // neither: dst = src on the item cells (scalar path only; with clamp: eq. 10)
    bool clamp = false;     // eq. 10 on the values written
    bool emit_T = false;    // also emit the T masks of the values written into tmask[tb ^ 1] (requires clamp)
    unsigned long long* residual = nullptr;   // max |d_new - d_old| over N of the LAST sweep, as ordered bits
    int list = 0;           // list buffer to iterate (quads + items)
    const uint8_t* tgate = nullptr;   // advance: null, or tmask[tb] is valid only for quads with tgate != 0
    bool reverse = false;   // walk the list from its end (L2 reuse between consecutive launches)
};

// Band kernel over a quad list: reads `src` (and F), writes the item cells of `dst`.
// Returns false if the tile path cannot address the grid (caller falls back to the scalar kernels).
template <typename T>
bool launch_band_tile(const T* src, const T* F, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                      const BandOp& op, cudaStream_t s, int64_t* launches);
template <typename T>
bool tile_usable(const Geom& g, const void* a, const void* b, const void* c);
// Scalar fallback (any nx, any alignment): one launch = advance OR one sweep OR a copy (even `iters`: eq. 10 only).
template <typename T>
void launch_band_scalar(const T* src, const T* F, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                        const BandOp& op, cudaStream_t s, int64_t* launches);

// Dense full-domain advance (c == 1), cfg 2.
template <typename T>
void launch_advance_dense(const T* phi, const T* F, T* out, const Geom& g, const StencilParams<T>& p,
                          cudaStream_t s, int64_t* launches);
// eq. 10 at every point of a; where the value changes it is also written to b (b may be null).
template <typename T>
void launch_clamp_all(T* a, T* b, int64_t n, T gamma, cudaStream_t s, int64_t* launches);

// Bit-for-bit check of the packed arithmetic against the scalar functions on n random stencil samples.
// mismatches: 2 counters (differing results; differing samples); dbg: 32 floats of the first differing sample or null.
void launch_selftest_math(uint64_t seed, int64_t n, const StencilParams<float>& p, unsigned long long* mismatches,
                          float* dbg, cudaStream_t s);

int sm_count();

}  // namespace ls
