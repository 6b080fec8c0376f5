// ls_internal.h — shared declarations of the CUDA path (libls.so).  Not part of the public ABI.
// Nothing here is shared with oracle/ (the CPU oracle is an independent restatement of the paper).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ls {

// Grid geometry (x fastest) and its 8^3 brick decomposition (R20).
struct Geom {
    int nx, ny, nz;
    int NBx, NBy, NBz;
    int nbricks;
    // packed brick position of the list entries (T_pos / N_pos / U_pos): bx | by << pos_sy | bz << pos_sz
    int pos_mx, pos_my, pos_sy, pos_sz;
    __host__ __device__ inline int64_t idx(int i, int j, int k) const {
        return ((int64_t)k * ny + j) * nx + i;
    }
};

// Device-resident counters, written by the band builder, read by the band kernels (grid-stride
// loops bound by these counts, so the host never needs them inside ls_step).
struct Counts {
    int32_t nT;            // bricks in the T list
    int32_t nN;            // bricks in the N list
    int32_t nU;            // bricks in the U list (N of this step  ∪  N of the previous step)
    int32_t pad;
    unsigned long long nT_pts, nN_pts;  // |T|, |N|
    unsigned long long acc_T, acc_N;    // accumulators of the build in flight (k_dilate), folded by k_scan_partials
    unsigned long long updates;         // sum over steps of |T| + iters*|N|
    unsigned long long steps;
};

// Everything the band builder owns, as raw device pointers.
struct BandBuffers {
    uint64_t* tmask;   // [nbricks*8] dense T mask words; valid only where flagT != 0
    uint64_t* nmask;   // [nbricks*8] dense N mask words; valid only where flagN != 0
    uint8_t* flagT;    // [nbricks]
    uint8_t* flagN;    // [nbricks] N flags of the band being built
    uint8_t* flagNprev;// [nbricks] N flags of the previous step's band (all 0 at the start of a call)
    int32_t* T_ids;    // [nbricks]
    uint64_t* T_masks; // [nbricks*8] list-ordered snapshot of the T masks (export); N_masks: filled at export
    int32_t* N_ids;
    uint64_t* N_masks;
    int32_t* U_ids;
    int32_t* T_pos;    // [nbricks] packed (bx, by, bz) of each list entry, see Geom::pos_*
    int32_t* N_pos;
    int32_t* U_pos;
    int32_t* partials; // [3 * npartials] per-CTA flag counts, then their exclusive scans
    int npartials;
    Counts* counts;
};

// ---- band builder (ls_band.cu) --------------------------------------------------------------
// Full-grid classification |phi| < gamma into per-brick T masks (eq. 6).
template <typename T>
void launch_classify(const T* phi, const Geom& g, T gamma, const BandBuffers& bb, cudaStream_t s, int64_t* launches);
// N = one-cell face dilation of T (eq. 11), then ordered compaction of the T, N and U lists.
// `iters` only feeds the update counter (|T| + iters*|N|).
void launch_dilate_compact(const Geom& g, const BandBuffers& bb, int iters, bool count_step, cudaStream_t s,
                           int64_t* launches);

// List-ordered copy N_masks of the dense N masks of the band last built (for ls_band_export; T_masks is
// snapshotted by launch_dilate_compact).
void launch_gather_masks(const BandBuffers& bb, cudaStream_t s, int64_t* launches);

// ---- stencil kernels (ls_stencil.cu) --------------------------------------------------------
template <typename T>
struct StencilParams {
    T inv_dx;      // 1/dx
    T dx2;         // dx*dx
    T dt;          // dt (advance) or dtau (reinit)
    T beta, gamma, three_beta, inv3;  // eq. 7 constants, inv3 = 1/((gamma-beta)^3)
};

// Advance over the U list: writes every in-domain point of each listed brick (T points by eq. 8,
// the rest copied).  src = phi^n, dst = phi_bar.
template <typename T>
void launch_advance_band(const T* phi, const T* F, T* out, const Geom& g, const StencilParams<T>& p,
                         const BandBuffers& bb, bool use_T_list, cudaStream_t s, int64_t* launches);
// Dense full-domain advance (c == 1), cfg 2.
template <typename T>
void launch_advance_dense(const T* phi, const T* F, T* out, const Geom& g, const StencilParams<T>& p,
                          cudaStream_t s, int64_t* launches);
// One reinit sweep over the N list: dst(x) = update(src)(x) for x in N; rows of a listed brick that
// hold an N point are written whole (non-N points of such a row keep src's value).
//   clamp        : apply eq. 10 to the values written (last sweep of a step)
//   residual     : if non-null, atomically max-accumulates |dst - src| over N as ordered bits
//   emit_T       : if true, also emits the T mask words / flagT of phi^{n+1} = clamp(dst) per N brick
//                  (incremental rebuild; requires clamp)
template <typename T>
void launch_reinit_band(const T* src, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                        bool clamp, unsigned long long* residual, bool emit_T, cudaStream_t s, int64_t* launches);
// dst(x) = clamp(src(x)) on the rows of N bricks that hold N points (even `iters`, iters = 0).
template <typename T>
void launch_copy_clamp_band(const T* src, T* dst, const Geom& g, T gamma, const BandBuffers& bb, cudaStream_t s,
                            int64_t* launches);
// eq. 10 at every point of a; where the value changes it is also written to b (b may be null).
template <typename T>
void launch_clamp_all(T* a, T* b, int64_t n, T gamma, cudaStream_t s, int64_t* launches);

// ---- TMA-pipelined band kernels (ls_tma.cu) ---------------------------------------------------
// Usable when every field row starts on a 16-byte boundary (nx*sizeof(T) % 16 == 0, aligned bases) and
// the driver exposes cuTensorMapEncodeTiled.  The launchers return false (nothing enqueued) if the
// tensor map cannot be built; the callers then take the scalar kernels of ls_stencil.cu.
template <typename T>
bool tma_usable(const Geom& g, const void* a, const void* b, const void* c);
template <typename T>
bool launch_reinit_tma(const T* src, T* dst, const Geom& g, const StencilParams<T>& p, const BandBuffers& bb,
                       bool clamp, unsigned long long* residual, bool emit_T, cudaStream_t s, int64_t* launches);
template <typename T>
bool launch_advance_tma(const T* phi, const T* F, T* out, const Geom& g, const StencilParams<T>& p,
                        const BandBuffers& bb, bool use_T_list, cudaStream_t s, int64_t* launches);

// Bit-for-bit check of the packed pair arithmetic against the scalar functions on n random stencil pairs.
// mismatches: 2 counters (differing results; differing samples); dbg: 26 floats of the first differing sample or null.
void launch_selftest_math(uint64_t seed, int64_t n, const StencilParams<float>& p, unsigned long long* mismatches,
                          float* dbg, cudaStream_t s);

int sm_count();

}  // namespace ls
