/* ls_static.h — the ONE entry point of libls.so that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc — code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it.  Every other entry point of ls.h works on an ls_ctx whose ls_create (and the first ls_step / export)
 * allocates device memory.  ls_tube_static computes the T tube of Step 1 (eq. 6, PAPER.md:43:
 * T = {|phi| < gamma}, found by scanning the whole grid) with no ctx: its work memory — the dense
 * per-brick mask words that ls_build_band keeps in ctx-owned buffers, and the per-CTA counts of the ordered
 * compaction — is a file-scope `static __device__` array inside libls.so.
 *
 * The limit: LS_TUBE_STATIC_MAX_BRICKS 8x8x8 bricks per call (65536: e.g. 320 x 320 x 320, 256 x 256 x 512 or
 * 512 x 512 x 128 points).  The array is LS_TUBE_STATIC_SCRATCH_BYTES (4 MiB + 4 KiB); every GPU that loads
 * libls.so holds it from the load of the module until the process exits, whether or not this call is used.
 *
 * Sharing: there is ONE array per device and every call on that device uses it.  It keeps the last call's
 * contents; a call reads only what the same call wrote before (all words of all its bricks, zeros included, and
 * all its per-CTA counts), so nothing has to be cleared and a smaller grid after a larger one is safe.  Two calls
 * that overlap on the GPU (different streams, or two graphs replayed concurrently) RACE on the array: the caller
 * serialises them (same stream, or an event between them).
 *
 * Conventions of ls.h hold (field layout, brick ids, mask words, DEVICE pointers owned by the caller).
 */
#ifndef LS_STATIC_H_
#define LS_STATIC_H_

#include "ls.h"

#ifdef __cplusplus
extern "C" {
#endif

#define LS_TUBE_STATIC_MAX_BRICKS 65536
#define LS_TUBE_STATIC_SCRATCH_BYTES (LS_TUBE_STATIC_MAX_BRICKS * 64 + 4096)

/* Resolve the device address of the static array for the CURRENT device (cudaGetSymbolAddress; the first CUDA
 * call of a process on a device also creates its context and loads the module).  Optional: ls_tube_static does it
 * on its first call per device; call it yourself before a stream capture begins.  No allocation. */
ls_status ls_tube_static_setup(void);

/* T = {|phi| < gamma} of an nx*ny*nz field of `dtype` on the current device, as ls_build_band + ls_band_export
 * return it: the ascending ids of the bricks that hold at least one T point and their 8 mask words each.
 *   phi      DEVICE, read only, nx*ny*nz elements, x fastest (any alignment of the element type).
 *   gamma    > 0 (NaN rejected), rounded once to the field type; +inf puts every in-domain point in T.
 *   T_ids    DEVICE out, capacity nbricks = ceil(nx/8)*ceil(ny/8)*ceil(nz/8) int32; the first counts[1] are written.
 *   T_masks  DEVICE out, capacity 8*nbricks uint64; the first 8*counts[1] are written.
 *   counts   DEVICE out, 2 x int64: [0] = |T| (points), [1] = number of T bricks.
 * Enqueues three kernels on `cuda_stream` (a cudaStream_t cast to void*, NULL = the legacy default stream) and
 * returns without waiting; no host synchronisation, no cudaMalloc / cudaFree / allocating library routine, on any
 * call.  Errors: LS_ERR_ARG (null pointer, gamma not > 0), LS_ERR_DIM (a dimension < 1), LS_ERR_DTYPE,
 * LS_ERR_CAPACITY (more than LS_TUBE_STATIC_MAX_BRICKS bricks: checked before any CUDA call; use ls_build_band),
 * LS_ERR_CUDA (ls_tube_static_error has the text).  Nothing is enqueued when an error is returned. */
ls_status ls_tube_static(const void* phi, int32_t nx, int32_t ny, int32_t nz, ls_dtype dtype, double gamma,
                         void* cuda_stream, int32_t* T_ids, uint64_t* T_masks, int64_t* counts);

/* Text of the last error ls_tube_static / ls_tube_static_setup returned in this process (static storage; "" if none). */
const char* ls_tube_static_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LS_STATIC_H_ */
