// ls_api.cu — the C ABI of include/ls.h: context, argument checks, and the host driver of the
// Step 1-3 loop on one stream.  Every step of the path runs in the kernels of
// ls_band.cu / ls_tile.cu / ls_stencil.cu; this file only sequences launches.  There is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <vector>

#include "../../include/ls.h"
#include "ls_internal.h"

struct HostPipe;

struct ls_ctx {
    ls::Geom g;
    ls_dtype dtype;
    cudaStream_t stream;
    ls::BandBuffers bb;
    void* scratch;        // one field, second Jacobi buffer (lazy)
    void* dev_phi;        // ls_step_host staging (lazy)
    void* dev_F;
    bool dev_F_valid;     // dev_F holds the F of the last ls_step_host call that passed one
    struct HostPipe* pipe;   // ls_step_host: the z-slab pipeline of one-step calls on large grids (lazy)
    void* snap[2];        // ls_step_snapshots: device snapshot slots (lazy)
    cudaStream_t copy_stream;   // ... and the stream / events of the device-to-host copies (lazy)
    cudaEvent_t snap_ready[2], snap_free[2];
    unsigned long long* residual;  // device
    ls::Counts* host_counts;       // pinned
    unsigned long long* host_residual;  // pinned
    bool band_valid;
    int64_t launches;
    int64_t dense_updates;
    size_t elem;          // sizeof field element
    int64_t n;            // nx*ny*nz
    // chained stepping (ls_params::chained): what the last ls_step left behind
    const void* chain_phi;   // phi buffer the ctx state is consistent with (null: none)
    double chain_gamma;
    bool chain_have_T;       // tmask[tb ^ 1] holds the T masks of the current phi (emitted by the last sweep)
    bool flip;               // list walking direction of the next band launch
    int64_t tile_min_cells;  // ls_tile_threshold
    // per-kernel device timing (ls_profile_*)
    bool prof_on;
    struct ProfRec { int kind; cudaEvent_t a, b; };
    std::vector<ProfRec>* prof_recs;    // brackets recorded since the last read
    std::vector<cudaEvent_t>* prof_pool;  // idle events
    double prof_ms[LS_K_KINDS];
    int64_t prof_n[LS_K_KINDS];
};

namespace {

char g_cuda_error[512] = "";

ls_status cuda_fail(cudaError_t e, const char* what) {
    std::snprintf(g_cuda_error, sizeof g_cuda_error, "%s: %s", what, cudaGetErrorString(e));
    return LS_ERR_CUDA;
}

#define LS_CK(call)                                             \
    do {                                                        \
        cudaError_t e_ = (call);                                \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);     \
    } while (0)

#define LS_CK_LAUNCH()                                                   \
    do {                                                                 \
        cudaError_t e_ = cudaPeekAtLastError();                          \
        if (e_ != cudaSuccess) { cudaGetLastError(); return cuda_fail(e_, "kernel launch"); } \
    } while (0)

// Bracket the launches enqueued during its lifetime with two events on the ctx stream.
struct ProfScope {
    ls_ctx* c;
    ls_ctx::ProfRec r;
    bool live;
    ProfScope(ls_ctx* ctx, int kind) : c(ctx), live(false) {
        if (!c->prof_on) return;
        auto get = [&](cudaEvent_t* e) {
            if (!c->prof_pool->empty()) { *e = c->prof_pool->back(); c->prof_pool->pop_back(); return true; }
            return cudaEventCreate(e) == cudaSuccess;
        };
        r.kind = kind;
        if (!get(&r.a)) return;
        if (!get(&r.b)) { c->prof_pool->push_back(r.a); return; }
        cudaEventRecord(r.a, c->stream);
        live = true;
    }
    ~ProfScope() {
        if (!live) return;
        cudaEventRecord(r.b, c->stream);
        c->prof_recs->push_back(r);
    }
};

// Fold finished brackets into the totals.  Synchronises the stream.
ls_status prof_collect(ls_ctx* c) {
    if (c->prof_recs->empty()) return LS_OK;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    for (auto& r : *c->prof_recs) {
        float ms = 0.f;
        if (e == cudaSuccess && cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) {
            c->prof_ms[r.kind] += ms;
            c->prof_n[r.kind] += 1;
        }
        c->prof_pool->push_back(r.a);
        c->prof_pool->push_back(r.b);
    }
    c->prof_recs->clear();
    if (e != cudaSuccess) return cuda_fail(e, "ls_profile: cudaStreamSynchronize");
    return LS_OK;
}

template <typename T>
ls::StencilParams<T> make_params(double dx, double dt, double beta, double gamma) {
    // R18: each scalar is rounded to T once; derived constants are formed in T.
    ls::StencilParams<T> p;
    const T dxT = (T)dx;
    p.inv_dx = T(1) / dxT;
    p.half_inv_dx = p.inv_dx * T(0.5);
    p.dx2 = dxT * dxT;
    p.dt = (T)dt;
    p.beta = (T)beta;
    p.gamma = (T)gamma;
    p.three_beta = T(3) * p.beta;
    const T w = p.gamma - p.beta;
    p.inv3 = T(1) / ((w * w) * w);
    return p;
}

ls_status ensure_field(ls_ctx* c, void** field) {
    if (*field) return LS_OK;
    cudaError_t e = cudaMalloc(field, (size_t)c->n * c->elem);
    if (e != cudaSuccess) { cudaGetLastError(); *field = nullptr; return LS_ERR_ALLOC; }
    return LS_OK;
}

bool bad_band_params(double dx, double beta, double gamma) {
    if (!(dx > 0) || std::isnan(beta) || std::isnan(gamma)) return true;
    if (std::isinf(beta) && std::isinf(gamma) && beta > 0 && gamma > 0) return false;
    return !(beta > 0 && beta < gamma);
}

// Default of ls_tile_threshold: grids below it take the scalar band kernels.  A tiled launch costs ~12 us before its
// first tile is through the pipeline (ticket -> list entry -> item list -> gather -> compute), which is more than the
// scalar kernel's whole run time on a small band: cfg 1 shapes on a B200, us per step tiled / scalar: 64^3 104 / 56,
// 96^3 109 / 69, 128^3 114 / 88, 160^3 118 / 117, 200^3 116 / 157, 256^3 119 / 223.
#ifndef LS_TILE_MIN_CELLS
#define LS_TILE_MIN_CELLS 4000000
#endif

// One band launch: the tile kernels where they can address the grid, else the scalar kernels.
template <typename T>
void band_launch(ls_ctx* c, const T* src, const T* F, T* dst, const ls::StencilParams<T>& p, ls::BandOp op) {
    op.reverse = c->flip;
    c->flip = !c->flip;
    if (!op.copy && c->n >= c->tile_min_cells && ls::tile_usable<T>(c->g, src, F, dst) &&
        ls::launch_band_tile<T>(src, F, dst, c->g, p, c->bb, op, c->stream, &c->launches))
        return;
    ls::launch_band_scalar<T>(src, F, dst, c->g, p, c->bb, op, c->stream, &c->launches);
}

// Step 1.  classify: scan the whole grid for T (else tmask[tb] already holds T of phi, emitted by the last
// sweep of the previous step); incremental: candidates from the previous band only.
ls_status build_band_impl(ls_ctx* c, const void* phi, double gamma, int iters, bool count_step, bool classify,
                          bool incremental) {
    if (classify) {
        ProfScope ps(c, LS_K_CLASSIFY);
        if (c->dtype == LS_F32)
            ls::launch_classify<float>((const float*)phi, c->g, (float)gamma, c->bb, c->stream, &c->launches);
        else
            ls::launch_classify<double>((const double*)phi, c->g, gamma, c->bb, c->stream, &c->launches);
    }
    {
        ProfScope ps(c, LS_K_BAND);
        ls::launch_build_lists(c->g, c->bb, incremental, iters, count_step, c->stream, &c->launches);
    }
    LS_CK_LAUNCH();
    c->band_valid = true;
    return LS_OK;
}

// Steps 1-3, n_steps times.  Two Jacobi buffers: the caller's phi and the ctx scratch field S.
//   Advance phi -> S, sweeps S -> phi -> S ..., the last one landing in phi (even `iters`: a band copy).
// Only item cells are written, so the buffers must agree wherever a later launch reads a halo.  Invariant at
// the start of a chained step n: S == phi^n except on the item cells of the band of step n-1 (they hold the
// next-to-last iterate).  Since T^n is a subset of N^{n-1}, Advance of step n walks the items of
// the PREVIOUS band: T cells get eq. 8, the other cells are copied — which repairs S exactly where it is stale.
// The first step of an unchained call starts from S = phi (one whole-field copy) and walks its own band.
template <typename T>
ls_status step_impl(ls_ctx* c, T* phi, const T* F, const ls_params* p, int n_steps) {
    ls_status st = ensure_field(c, &c->scratch);
    if (st != LS_OK) return st;
    T* S = (T*)c->scratch;
    const ls::StencilParams<T> adv = make_params<T>(p->dx, p->dt, p->beta, p->gamma);
    const ls::StencilParams<T> rei = make_params<T>(p->dx, p->dtau, p->beta, p->gamma);
    const T gammaT = (T)p->gamma;
    cudaStream_t s = c->stream;
    const bool incremental = p->rebuild == LS_REBUILD_INCREMENTAL;
    const bool chained = p->chained && c->chain_phi == (const void*)phi && c->chain_gamma == p->gamma;
    bool have_T = chained && c->chain_have_T && incremental;
    c->chain_phi = nullptr;   // re-established only when the whole call was enqueued
    if (!chained) {
        ProfScope ps(c, LS_K_COPY);
        LS_CK(cudaMemcpyAsync(S, phi, (size_t)c->n * sizeof(T), cudaMemcpyDeviceToDevice, s));
    }
    for (int step = 0; step < n_steps; ++step) {
        const bool have_prev = chained || step > 0;   // S is stale on the previous band's items
        if (have_T) {   // the last sweep left T of phi^n in the other T buffer, valid on the quads of the band it walked
            c->bb.tb ^= 1;
            c->bb.tvalid_all = false;
        }
        ls::BandOp a;
        a.advance = true;
        if (have_prev) {
            // Step 2 first (it needs T^n and the PREVIOUS band's lists), then Step 1 for the sweeps
            if (!have_T) {
                ProfScope ps(c, LS_K_CLASSIFY);
                ls::launch_classify<T>(phi, c->g, gammaT, c->bb, s, &c->launches);
            }
            a.list = c->bb.lb;
            {
                ProfScope ps(c, LS_K_ADVANCE);
                band_launch<T>(c, phi, F, S, adv, a);
            }
            st = build_band_impl(c, phi, p->gamma, p->iters, true, false, have_T);
            if (st != LS_OK) return st;
        } else {
            st = build_band_impl(c, phi, p->gamma, p->iters, true, true, false);   // Step 1 (whole grid)
            if (st != LS_OK) return st;
            a.list = c->bb.lb;
            ProfScope ps(c, LS_K_ADVANCE);
            band_launch<T>(c, phi, F, S, adv, a);                                   // Step 2: phi -> S
        }
        T* src = S;
        T* dst = phi;
        bool emitted = false;
        // Step 3: `iters` sweeps in launches of 2 (temporal blocking, tile path only) or 1.  The number of
        // launches should be odd so that the last one lands in phi; if it cannot be (iters == 0, or an even
        // count on the scalar path), the band copy below moves the result.
        const bool can_fuse = p->fuse == 2 && c->n >= c->tile_min_cells && ls::tile_usable<T>(c->g, phi, S, (const void*)nullptr);
        int pairs = can_fuse ? p->iters / 2 : 0, singles = p->iters - 2 * pairs;
        if (pairs > 0 && ((pairs + singles) & 1) == 0) { pairs -= 1; singles += 2; }
        for (int l = 0; l < pairs + singles; ++l) {
            const bool last = l == pairs + singles - 1 && dst == phi;
            ls::BandOp r;
            r.sweeps = l < pairs ? 2 : 1;
            r.list = c->bb.lb;
            r.clamp = last;
            r.emit_T = last && incremental;
            emitted = emitted || r.emit_T;
            ProfScope ps(c, LS_K_REINIT);
            band_launch<T>(c, src, (const T*)nullptr, dst, rei, r);
            T* t = src; src = dst; dst = t;
        }
        if (src != phi) {  // even iters: the result sits in S
            ls::BandOp r;
            r.copy = true;
            r.list = c->bb.lb;
            r.clamp = true;
            r.emit_T = incremental;
            emitted = r.emit_T;
            ProfScope ps(c, LS_K_CLAMP);
            band_launch<T>(c, S, (const T*)nullptr, phi, rei, r);
        }
        if (!have_prev) {  // eq. 10 at every point (R14); afterwards points off N already hold +-gamma
            ProfScope ps(c, LS_K_CLAMP);
            ls::launch_clamp_all<T>(phi, S, c->n, gammaT, s, &c->launches);
        }
        LS_CK_LAUNCH();
        have_T = emitted;
    }
    c->chain_phi = phi;
    c->chain_gamma = p->gamma;
    c->chain_have_T = have_T;
    return LS_OK;
}

ls_status check_step_args(ls_ctx* c, const void* phi, const void* F, const ls_params* p, int n_steps) {
    if (!c || !phi || !F || !p) return LS_ERR_ARG;
    if (n_steps < 0 || p->iters < 0) return LS_ERR_ARG;
    if (!(p->dx > 0) || !(p->beta > 0) || !(p->beta < p->gamma) || std::isinf(p->gamma)) return LS_ERR_ARG;
    if (p->rebuild != LS_REBUILD_FULL && p->rebuild != LS_REBUILD_INCREMENTAL) return LS_ERR_ARG;
    if ((p->chained != 0 && p->chained != 1) || p->fuse < 0 || p->fuse > 2) return LS_ERR_ARG;
    return LS_OK;
}

}  // namespace

// ---- ls_step_host, one step per call on a large grid: z-slab pipeline ---------------------------------------------
// A one-step call moves the whole field host -> device -> host (2 x 4.3 GB at cfg 4: ~78 ms each way) around ~5 ms of
// GPU work; on one stream the three phases run one after the other.  One narrow-band step has a finite domain of
// dependence: Advance reads the face neighbours of a point, each of the `iters` Jacobi sweeps one more layer, the T / N
// membership one layer, eq. 10 none (eq. 3-5, 11, 12) — phi^{n+1} on the layers [z0, z1) is a
// function of phi^n on [z0 - h, z1 + h), h = iters + 1.  So the field is cut into z-slabs (the paper's own decomposition
// axis is a slab cut too): slab k's layers are uploaded ONCE into the full staging field, the step runs on
// a window of the staging field that holds the slab plus h layers on each side (copied device-to-device into a window
// buffer: the staging field must stay phi^n for the neighbouring windows), on a child ctx of the window's shape, and the
// slab's layers of the result go back to the host while later slabs are still arriving: H2D, compute and D2H overlap on
// three streams.  The window's z ends are the child's domain boundary (edge replicate, R3): exact where they are the
// grid's own boundary, wrong within iters layers of an artificial cut — layers that are never returned.  Results are
// bit-identical to the unsliced call; every window has the same shape (the first and last are shifted inwards).
struct HostPipe {
    ls_ctx* child;
    int L, zs, h;                 // window layers, slab layers, halo layers
    void* buf[3];                 // window fields
    cudaStream_t up, cs, down;
    cudaEvent_t start, done[3], freed[3];
    std::vector<cudaEvent_t>* uploaded;   // one per slab
};

namespace {

void pipe_destroy(HostPipe* hp) {
    if (!hp) return;
    if (hp->child) ls_destroy(hp->child);
    for (void* b : hp->buf)
        if (b) cudaFree(b);
    if (hp->up) cudaStreamDestroy(hp->up);
    if (hp->cs) cudaStreamDestroy(hp->cs);
    if (hp->down) cudaStreamDestroy(hp->down);
    if (hp->start) cudaEventDestroy(hp->start);
    for (int i = 0; i < 3; ++i) {
        if (hp->done[i]) cudaEventDestroy(hp->done[i]);
        if (hp->freed[i]) cudaEventDestroy(hp->freed[i]);
    }
    if (hp->uploaded) {
        for (cudaEvent_t e : *hp->uploaded) cudaEventDestroy(e);
        delete hp->uploaded;
    }
    cudaGetLastError();
    delete hp;
}

// Slab thickness for a one-step call, or 0 when the call should run unsliced (small field, few layers, not one step).
int pipe_slab_layers(const ls_ctx* c, const ls_params* p, int n_steps) {
    if (n_steps != 1) return 0;
    const size_t plane = (size_t)c->g.nx * c->g.ny * c->elem;
    if (plane * (size_t)c->g.nz < ((size_t)64 << 20)) return 0;        // transfers too short to be worth the windows
    const int64_t h = (int64_t)p->iters + 1;
    int64_t zs = (int64_t)((((size_t)16 << 20) + plane - 1) / plane);   // >= 16 MiB per slab
    if (zs < 4 * h) zs = 4 * h;                                        // <= 1.5 x redundant compute
    if (zs < 8) zs = 8;
    if (zs + 2 * h > c->g.nz || 2 * zs > c->g.nz) return 0;            // window must fit; at least two slabs
    return (int)zs;
}

ls_status pipe_ensure(ls_ctx* c, int zs, int h) {
    const int L = zs + 2 * h;
    if (c->pipe && c->pipe->L == L && c->pipe->zs == zs) return LS_OK;
    pipe_destroy(c->pipe);
    c->pipe = nullptr;
    HostPipe* hp = new (std::nothrow) HostPipe();
    if (!hp) return LS_ERR_ALLOC;
    std::memset(hp, 0, sizeof *hp);
    hp->L = L; hp->zs = zs; hp->h = h;
    hp->uploaded = new (std::nothrow) std::vector<cudaEvent_t>();
    cudaError_t e = hp->uploaded ? cudaSuccess : cudaErrorMemoryAllocation;
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hp->up, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hp->cs, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hp->down, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hp->start, cudaEventDisableTiming);
    for (int i = 0; i < 3 && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&hp->done[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hp->freed[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaMalloc(&hp->buf[i], (size_t)c->g.nx * c->g.ny * L * c->elem);
    }
    const int K = (c->g.nz + zs - 1) / zs;
    for (int k = 0; k < K && e == cudaSuccess; ++k) {
        cudaEvent_t ev;
        e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
        if (e == cudaSuccess) hp->uploaded->push_back(ev);
    }
    ls_status st = LS_OK;
    if (e != cudaSuccess) {
        st = e == cudaErrorMemoryAllocation ? LS_ERR_ALLOC : cuda_fail(e, "ls_step_host: slab pipeline set-up");
        cudaGetLastError();
    } else {
        st = ls_create(c->g.nx, c->g.ny, L, c->dtype, (void*)hp->cs, &hp->child);
    }
    if (st != LS_OK) { pipe_destroy(hp); return st; }
    c->pipe = hp;
    return LS_OK;
}

// The sliced one-step call.  c->dev_phi / c->dev_F are allocated, F is on the device (this call's upload, if any, is queued
// on c->stream).  Synchronises; on a failure it still drains its streams before it returns the first error.
ls_status step_host_sliced(ls_ctx* c, void* phi_host, const ls_params* p, int zs) {
    const int h = p->iters + 1;
    ls_status st = pipe_ensure(c, zs, h);
    if (st != LS_OK) return st;
    HostPipe* hp = c->pipe;
    ls_ctx* ch = hp->child;
    ch->tile_min_cells = c->tile_min_cells <= c->n ? 0 : ch->n + 1;   // the windows take the path the whole grid would
    const int nz = c->g.nz, L = hp->L, K = (nz + zs - 1) / zs;
    const size_t plane = (size_t)c->g.nx * c->g.ny * c->elem;
    ls_params q = *p;
    q.chained = 0;
    cudaError_t ce = cudaSuccess;
    const char* what = "";
    auto ck = [&](cudaError_t e, const char* w) { if (ce == cudaSuccess && e != cudaSuccess) { ce = e; what = w; } return e == cudaSuccess; };
    const int64_t child_launches0 = ch->launches;
    int64_t extra_launches = 0;
    bool ok = ck(cudaEventRecord(hp->start, c->stream), "cudaEventRecord") &&
              ck(cudaStreamWaitEvent(hp->up, hp->start, 0), "cudaStreamWaitEvent") &&
              ck(cudaStreamWaitEvent(hp->cs, hp->start, 0), "cudaStreamWaitEvent") &&
              ck(cudaStreamWaitEvent(hp->down, hp->start, 0), "cudaStreamWaitEvent");
    // every layer goes up once, slab by slab
    for (int k = 0; k < K && ok; ++k) {
        const int z0 = k * zs, z1 = std::min(nz, z0 + zs);
        ok = ck(cudaMemcpyAsync((char*)c->dev_phi + z0 * plane, (const char*)phi_host + z0 * plane, (z1 - z0) * plane,
                                cudaMemcpyHostToDevice, hp->up), "slab upload") &&
             ck(cudaEventRecord((*hp->uploaded)[k], hp->up), "cudaEventRecord");
    }
    for (int k = 0; k < K && ok && st == LS_OK; ++k) {
        const int z0 = k * zs, z1 = std::min(nz, z0 + zs), b = k % 3;
        const int lo = std::max(0, std::min(z0 - h, nz - L));       // window [lo, lo + L): same shape for every slab
        const int last_slab = (lo + L - 1) / zs;                    // uploads are ordered: the last slab it touches
        ok = ck(cudaStreamWaitEvent(hp->cs, (*hp->uploaded)[last_slab], 0), "cudaStreamWaitEvent");
        if (ok && k >= 3) ok = ck(cudaStreamWaitEvent(hp->cs, hp->freed[b], 0), "cudaStreamWaitEvent");   // its download has drained
        if (!ok) break;
        ok = ck(cudaMemcpyAsync(hp->buf[b], (const char*)c->dev_phi + lo * plane, L * plane, cudaMemcpyDeviceToDevice, hp->cs),
                "window copy");
        if (!ok) break;
        const void* Fwin = (const char*)c->dev_F + lo * plane;
        st = c->dtype == LS_F32 ? step_impl<float>(ch, (float*)hp->buf[b], (const float*)Fwin, &q, 1)
                                : step_impl<double>(ch, (double*)hp->buf[b], (const double*)Fwin, &q, 1);
        if (st != LS_OK) break;
        // work counters of the parent: each grid point once (the window's halo layers are some other slab's)
        ls::launch_count_layers(ch->g, ch->bb, z0 - lo, z1 - lo, p->iters, k == 0 ? 1 : 0, c->bb.counts, hp->cs, &extra_launches);
        ok = ck(cudaPeekAtLastError(), "kernel launch") && ck(cudaEventRecord(hp->done[b], hp->cs), "cudaEventRecord") &&
             ck(cudaStreamWaitEvent(hp->down, hp->done[b], 0), "cudaStreamWaitEvent") &&
             ck(cudaMemcpyAsync((char*)phi_host + z0 * plane, (const char*)hp->buf[b] + (size_t)(z0 - lo) * plane,
                                (z1 - z0) * plane, cudaMemcpyDeviceToHost, hp->down), "slab download") &&
             ck(cudaEventRecord(hp->freed[b], hp->down), "cudaEventRecord");
    }
    ck(cudaStreamSynchronize(hp->up), "cudaStreamSynchronize");
    ck(cudaStreamSynchronize(hp->cs), "cudaStreamSynchronize");
    ck(cudaStreamSynchronize(hp->down), "cudaStreamSynchronize");
    c->launches += ch->launches - child_launches0 + extra_launches;
    c->band_valid = false;      // the windows' bands live in the child ctx; this ctx holds none
    c->chain_phi = nullptr;
    if (st != LS_OK) return st;
    if (ce != cudaSuccess) { cudaGetLastError(); return cuda_fail(ce, what); }
    return LS_OK;
}

}  // namespace

extern "C" {

const char* ls_status_str(ls_status s) {
    switch (s) {
        case LS_OK: return "LS_OK";
        case LS_ERR_ARG: return "LS_ERR_ARG";
        case LS_ERR_DIM: return "LS_ERR_DIM";
        case LS_ERR_DTYPE: return "LS_ERR_DTYPE";
        case LS_ERR_ALLOC: return "LS_ERR_ALLOC";
        case LS_ERR_CUDA: return "LS_ERR_CUDA";
        case LS_ERR_CAPACITY: return "LS_ERR_CAPACITY";
        case LS_NOT_CONVERGED: return "LS_NOT_CONVERGED";
        case LS_ERR_STATE: return "LS_ERR_STATE";
    }
    return "LS_UNKNOWN";
}

const char* ls_last_cuda_error(void) { return g_cuda_error; }

ls_status ls_create(int32_t nx, int32_t ny, int32_t nz, ls_dtype dtype, void* cuda_stream, ls_ctx** out) {
    if (!out) return LS_ERR_ARG;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return LS_ERR_DIM;
    if (dtype != LS_F32 && dtype != LS_F64) return LS_ERR_DTYPE;
    const int64_t NBx = (nx + 7) / 8, NBy = (ny + 7) / 8, NBz = (nz + 7) / 8;
    const int64_t nbricks = NBx * NBy * NBz;
    const int64_t NQx = (NBx + 3) / 4, nquads = NQx * NBy * NBz;
    if (nbricks > (int64_t)1 << 27) return LS_ERR_DIM;   // brick ids, quad ids and 32*quad stay in range
    int ndev = 0;
    LS_CK(cudaGetDeviceCount(&ndev));
    ls_ctx* c = new (std::nothrow) ls_ctx();
    if (!c) return LS_ERR_ALLOC;
    std::memset(c, 0, sizeof *c);
    c->g = ls::Geom{nx, ny, nz, (int)NBx, (int)NBy, (int)NBz, (int)NQx, (int)nbricks, (int)nquads};
    c->dtype = dtype;
    c->stream = (cudaStream_t)cuda_stream;
    c->elem = dtype == LS_F32 ? 4 : 8;
    c->n = (int64_t)nx * ny * nz;
    c->tile_min_cells = LS_TILE_MIN_CELLS;
    c->prof_recs = new (std::nothrow) std::vector<ls_ctx::ProfRec>();
    c->prof_pool = new (std::nothrow) std::vector<cudaEvent_t>();
    if (!c->prof_recs || !c->prof_pool) { delete c->prof_recs; delete c->prof_pool; delete c; return LS_ERR_ALLOC; }
    ls::BandBuffers& bb = c->bb;
    bb.compact_grid = (int)std::min<int64_t>(ls::sm_count(), std::max<int64_t>(1, (nquads + 16383) / 16384));
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void** p, size_t bytes, bool zero) {
        if (e != cudaSuccess) return;
        e = cudaMalloc(p, bytes);
        if (e == cudaSuccess && zero) e = cudaMemsetAsync(*p, 0, bytes, c->stream);
    };
    const size_t nq = (size_t)nquads;
    for (int i = 0; i < 2; ++i) {
        alloc((void**)&bb.tmask[i], nq * 32 * sizeof(uint64_t), false);
        alloc((void**)&bb.qflagT[i], nq + 16, true);
        alloc((void**)&bb.qflagN[i], nq + 16, true);          // invariant: 1 exactly at the quads of qlist[i]
        alloc((void**)&bb.items[i], nq * ls::kItemsPerQuad * sizeof(uint16_t), false);
        alloc((void**)&bb.qlist[i], nq * sizeof(ls::QuadEntry), false);
        alloc((void**)&bb.qneed[i], nq * ls::kNeedBytes, false);
    }
    alloc((void**)&bb.nmask, nq * 32 * sizeof(uint64_t), true);   // invariant: zero outside the band last built
    alloc((void**)&bb.qcount, nq * sizeof(int32_t), true);
    alloc((void**)&bb.partials, 1024 * sizeof(int32_t), true);
    alloc((void**)&bb.zero_page, 256, true);
    alloc((void**)&bb.counts, sizeof(ls::Counts), true);
    alloc((void**)&c->residual, 8, true);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&c->host_counts, sizeof(ls::Counts));
    if (e == cudaSuccess) e = cudaMallocHost((void**)&c->host_residual, 8);
    if (e != cudaSuccess) {
        const bool oom = e == cudaErrorMemoryAllocation;
        cuda_fail(e, "ls_create allocation");
        cudaGetLastError();
        ls_destroy(c);
        return oom ? LS_ERR_ALLOC : LS_ERR_CUDA;
    }
    *out = c;
    return LS_OK;
}

ls_status ls_destroy(ls_ctx* c) {
    if (!c) return LS_OK;
    cudaStreamSynchronize(c->stream);
    ls::BandBuffers& bb = c->bb;
    void* dev[] = {bb.tmask[0], bb.tmask[1], bb.qflagT[0], bb.qflagT[1], bb.qflagN[0], bb.qflagN[1], bb.items[0], bb.items[1],
                   bb.qlist[0], bb.qlist[1], bb.qneed[0], bb.qneed[1], bb.nmask, bb.qcount, bb.partials, bb.zero_page, bb.counts, bb.ex_cnt, bb.T_ids, bb.N_ids,
                   bb.T_masks, bb.N_masks, c->residual, c->scratch, c->dev_phi, c->dev_F, c->snap[0], c->snap[1]};
    for (void* p : dev)
        if (p) cudaFree(p);
    pipe_destroy(c->pipe);
    if (c->copy_stream) {
        cudaStreamSynchronize(c->copy_stream);
        cudaStreamDestroy(c->copy_stream);
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->snap_ready[i]); cudaEventDestroy(c->snap_free[i]); }
    }
    if (c->host_counts) cudaFreeHost(c->host_counts);
    if (c->host_residual) cudaFreeHost(c->host_residual);
    for (auto& r : *c->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (cudaEvent_t e : *c->prof_pool) cudaEventDestroy(e);
    delete c->prof_recs;
    delete c->prof_pool;
    cudaGetLastError();
    delete c;
    return LS_OK;
}

ls_status ls_build_band(ls_ctx* c, const void* phi, double dx, double gamma) {
    if (!c || !phi) return LS_ERR_ARG;
    if (!(dx > 0) || !(gamma > 0)) return LS_ERR_ARG;
    c->chain_phi = nullptr;
    return build_band_impl(c, phi, gamma, 0, false, true, false);
}

ls_status ls_band_counts(ls_ctx* c, int64_t* nT_points, int64_t* nN_points, int32_t* nT_bricks, int32_t* nN_bricks) {
    if (!c) return LS_ERR_ARG;
    if (!c->band_valid) return LS_ERR_STATE;
    if (nT_bricks || nN_bricks) {   // brick counts are derived from the quad list on demand
        if (!ls::launch_export(c->g, c->bb, false, c->stream, &c->launches)) return LS_ERR_ALLOC;
        LS_CK_LAUNCH();
    }
    LS_CK(cudaMemcpyAsync(c->host_counts, c->bb.counts, sizeof(ls::Counts), cudaMemcpyDeviceToHost, c->stream));
    LS_CK(cudaStreamSynchronize(c->stream));
    if (nT_points) *nT_points = (int64_t)c->host_counts->nT_pts;
    if (nN_points) *nN_points = (int64_t)c->host_counts->nN_pts;
    if (nT_bricks) *nT_bricks = c->host_counts->nT_bricks;
    if (nN_bricks) *nN_bricks = c->host_counts->nN_bricks;
    return LS_OK;
}

ls_status ls_band_export(ls_ctx* c, int32_t* T_ids, uint64_t* T_masks, int32_t* N_ids, uint64_t* N_masks) {
    if (!c) return LS_ERR_ARG;
    if (!c->band_valid) return LS_ERR_STATE;
    cudaStream_t s = c->stream;
    if (!ls::launch_export(c->g, c->bb, true, s, &c->launches)) return LS_ERR_ALLOC;
    LS_CK_LAUNCH();
    LS_CK(cudaMemcpyAsync(c->host_counts, c->bb.counts, sizeof(ls::Counts), cudaMemcpyDeviceToHost, s));
    LS_CK(cudaStreamSynchronize(s));
    const int32_t nT = c->host_counts->nT_bricks, nN = c->host_counts->nN_bricks;
    if (T_ids && nT) LS_CK(cudaMemcpyAsync(T_ids, c->bb.T_ids, (size_t)nT * 4, cudaMemcpyDeviceToHost, s));
    if (T_masks && nT) LS_CK(cudaMemcpyAsync(T_masks, c->bb.T_masks, (size_t)nT * 64, cudaMemcpyDeviceToHost, s));
    if (N_ids && nN) LS_CK(cudaMemcpyAsync(N_ids, c->bb.N_ids, (size_t)nN * 4, cudaMemcpyDeviceToHost, s));
    if (N_masks && nN) LS_CK(cudaMemcpyAsync(N_masks, c->bb.N_masks, (size_t)nN * 64, cudaMemcpyDeviceToHost, s));
    LS_CK(cudaStreamSynchronize(s));
    return LS_OK;
}

ls_status ls_advance(ls_ctx* c, const void* phi, const void* F, double dt, double dx, double beta, double gamma,
                     void* out) {
    if (!c || !phi || !F || !out || out == phi) return LS_ERR_ARG;
    if (bad_band_params(dx, beta, gamma)) return LS_ERR_ARG;
    const bool dense = std::isinf(beta) && std::isinf(gamma);
    cudaStream_t s = c->stream;
    if (dense) {
        ProfScope ps(c, LS_K_ADVANCE);
        if (c->dtype == LS_F32)
            ls::launch_advance_dense<float>((const float*)phi, (const float*)F, (float*)out, c->g,
                                            make_params<float>(dx, dt, beta, gamma), s, &c->launches);
        else
            ls::launch_advance_dense<double>((const double*)phi, (const double*)F, (double*)out, c->g,
                                             make_params<double>(dx, dt, beta, gamma), s, &c->launches);
        LS_CK_LAUNCH();
        c->dense_updates += c->n;
        return LS_OK;
    }
    if (!c->band_valid) return LS_ERR_STATE;
    // out = phi everywhere, then eq. 8 on the T bricks.
    {
        ProfScope ps(c, LS_K_COPY);
        LS_CK(cudaMemcpyAsync(out, phi, (size_t)c->n * c->elem, cudaMemcpyDeviceToDevice, s));
    }
    ProfScope ps(c, LS_K_ADVANCE);
    ls::BandOp a;
    a.advance = true;
    a.list = c->bb.lb;
    // T of the band last built: emitted masks are valid only on the quads of the band before it
    a.tgate = c->bb.tvalid_all ? nullptr : c->bb.qflagN[c->bb.lb ^ 1];
    if (c->dtype == LS_F32)
        band_launch<float>(c, (const float*)phi, (const float*)F, (float*)out, make_params<float>(dx, dt, beta, gamma), a);
    else
        band_launch<double>(c, (const double*)phi, (const double*)F, (double*)out,
                            make_params<double>(dx, dt, beta, gamma), a);
    LS_CK_LAUNCH();
    return LS_OK;
}

}  // extern "C"

namespace {

// Shared body of ls_reinit (tol < 0: fixed count) and ls_reinit_tol.
template <typename T>
ls_status reinit_impl(ls_ctx* c, T* d, const T* phi_bar, double dtau, double dx, double gamma, int iters, double tol,
                      int check_every, int32_t* iters_done, double* residual_out) {
    ls_status st = ensure_field(c, &c->scratch);
    if (st != LS_OK) return st;
    T* S = (T*)c->scratch;
    cudaStream_t s = c->stream;
    const size_t bytes = (size_t)c->n * sizeof(T);
    const ls::StencilParams<T> rei = make_params<T>(dx, dtau, gamma * 0.5, gamma);
    c->chain_phi = nullptr;   // the scratch field is reused here
    {
        ProfScope ps(c, LS_K_COPY);
        LS_CK(cudaMemcpyAsync(d, phi_bar, bytes, cudaMemcpyDeviceToDevice, s));
        LS_CK(cudaMemcpyAsync(S, phi_bar, bytes, cudaMemcpyDeviceToDevice, s));
    }
    const bool to_tol = tol >= 0;
    // fixed count: choose the first source so that the last sweep writes d
    T* src = (!to_tol && (iters & 1)) ? S : d;
    T* dst = src == d ? S : d;
    int k = 0;
    double r = 0.0;
    bool converged = false;
    while (k < iters) {
        ++k;
        const bool check = to_tol && (k % check_every == 0 || k == iters);
        if (check) LS_CK(cudaMemsetAsync(c->residual, 0, 8, s));
        {
            ProfScope ps(c, LS_K_REINIT);
            ls::BandOp r;
            r.sweeps = 1;
            r.list = c->bb.lb;
            r.residual = check ? c->residual : nullptr;
            band_launch<T>(c, src, (const T*)nullptr, dst, rei, r);
        }
        T* t = src; src = dst; dst = t;
        if (check) {
            LS_CK_LAUNCH();
            LS_CK(cudaMemcpyAsync(c->host_residual, c->residual, 8, cudaMemcpyDeviceToHost, s));
            LS_CK(cudaStreamSynchronize(s));
            const unsigned long long bits = *c->host_residual;
            if (sizeof(T) == 4) { uint32_t b32 = (uint32_t)bits; float f; std::memcpy(&f, &b32, 4); r = f; }
            else std::memcpy(&r, &bits, 8);
            if (k % check_every == 0 && r < tol) { converged = true; break; }
        }
    }
    LS_CK_LAUNCH();
    if (src != d) {   // result is in `src`
        ProfScope ps(c, LS_K_COPY);
        LS_CK(cudaMemcpyAsync(d, src, bytes, cudaMemcpyDeviceToDevice, s));
    }
    {
        ProfScope ps(c, LS_K_CLAMP);
        ls::launch_clamp_all<T>(d, (T*)nullptr, c->n, (T)gamma, s, &c->launches);          // eq. 10 everywhere
    }
    LS_CK_LAUNCH();
    if (iters_done) *iters_done = k;
    if (residual_out) *residual_out = r;
    if (to_tol && !converged) return LS_NOT_CONVERGED;
    return LS_OK;
}

}  // namespace

extern "C" {

ls_status ls_reinit(ls_ctx* c, void* d, const void* phi_bar, double dtau, double dx, double gamma, int32_t iters) {
    if (!c || !d || !phi_bar || d == phi_bar) return LS_ERR_ARG;
    if (!(dx > 0) || !(gamma > 0) || std::isinf(gamma) || iters < 0) return LS_ERR_ARG;
    if (!c->band_valid) return LS_ERR_STATE;
    if (c->dtype == LS_F32)
        return reinit_impl<float>(c, (float*)d, (const float*)phi_bar, dtau, dx, gamma, iters, -1.0, 1, nullptr, nullptr);
    return reinit_impl<double>(c, (double*)d, (const double*)phi_bar, dtau, dx, gamma, iters, -1.0, 1, nullptr, nullptr);
}

ls_status ls_reinit_tol(ls_ctx* c, void* d, const void* phi_bar, double dtau, double dx, double gamma, double tol,
                        int32_t max_iters, int32_t check_every, int32_t* iters_done, double* residual) {
    if (!c || !d || !phi_bar || d == phi_bar) return LS_ERR_ARG;
    if (!(dx > 0) || !(gamma > 0) || std::isinf(gamma) || max_iters < 0 || check_every < 1 || !(tol >= 0))
        return LS_ERR_ARG;
    if (!c->band_valid) return LS_ERR_STATE;
    if (c->dtype == LS_F32)
        return reinit_impl<float>(c, (float*)d, (const float*)phi_bar, dtau, dx, gamma, max_iters, tol, check_every,
                                  iters_done, residual);
    return reinit_impl<double>(c, (double*)d, (const double*)phi_bar, dtau, dx, gamma, max_iters, tol, check_every,
                               iters_done, residual);
}

ls_status ls_step(ls_ctx* c, void* phi, const void* F, const ls_params* p, int32_t n_steps) {
    ls_status st = check_step_args(c, phi, F, p, n_steps);
    if (st != LS_OK) return st;
    if (n_steps == 0) return LS_OK;
    if (c->dtype == LS_F32) return step_impl<float>(c, (float*)phi, (const float*)F, p, n_steps);
    return step_impl<double>(c, (double*)phi, (const double*)F, p, n_steps);
}

ls_status ls_step_host(ls_ctx* c, void* phi_host, const void* F_host, const ls_params* p, int32_t n_steps) {
    // F_host == NULL: reuse the F uploaded by the last call that passed one (R17: F is static)
    if (!F_host && c && !c->dev_F_valid) return LS_ERR_STATE;
    ls_status st = check_step_args(c, phi_host, F_host ? F_host : (const void*)phi_host, p, n_steps);
    if (st != LS_OK) return st;
    if ((st = ensure_field(c, &c->dev_phi)) != LS_OK) return st;
    if ((st = ensure_field(c, &c->dev_F)) != LS_OK) return st;
    const size_t bytes = (size_t)c->n * c->elem;
    const int zs = pipe_slab_layers(c, p, n_steps);
    if (F_host) {
        c->dev_F_valid = false;
        LS_CK(cudaMemcpyAsync(c->dev_F, F_host, bytes, cudaMemcpyHostToDevice, c->stream));
        c->dev_F_valid = true;
    }
    if (zs > 0) return step_host_sliced(c, phi_host, p, zs);   // one step, large grid: H2D / compute / D2H overlapped by z-slabs
    LS_CK(cudaMemcpyAsync(c->dev_phi, phi_host, bytes, cudaMemcpyHostToDevice, c->stream));
    if (n_steps > 0) {
        ls_params q = *p;
        q.chained = 0;   // the staging field was just overwritten
        st = c->dtype == LS_F32 ? step_impl<float>(c, (float*)c->dev_phi, (const float*)c->dev_F, &q, n_steps)
                                : step_impl<double>(c, (double*)c->dev_phi, (const double*)c->dev_F, &q, n_steps);
        if (st != LS_OK) return st;
    }
    LS_CK(cudaMemcpyAsync(phi_host, c->dev_phi, bytes, cudaMemcpyDeviceToHost, c->stream));
    LS_CK(cudaStreamSynchronize(c->stream));
    return LS_OK;
}

ls_status ls_step_snapshots(ls_ctx* c, void* phi, const void* F, const ls_params* p, int32_t n_steps, int32_t every,
                            void* host_out, int32_t* n_written) {
    ls_status st = check_step_args(c, phi, F, p, n_steps);
    if (st != LS_OK) return st;
    if (every < 1 || (!host_out && n_steps >= every)) return LS_ERR_ARG;
    if (n_written) *n_written = 0;
    if (n_steps == 0) return LS_OK;
    const size_t bytes = (size_t)c->n * c->elem;
    if (!c->copy_stream) {
        LS_CK(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            LS_CK(cudaEventCreateWithFlags(&c->snap_ready[i], cudaEventDisableTiming));
            LS_CK(cudaEventCreateWithFlags(&c->snap_free[i], cudaEventDisableTiming));
        }
    }
    if ((st = ensure_field(c, &c->snap[0])) != LS_OK) return st;
    if ((st = ensure_field(c, &c->snap[1])) != LS_OK) return st;
    ls_params q = *p;
    int k = 0;   // snapshots taken
    cudaError_t ce = cudaSuccess;
    const char* what = "";
    auto ck = [&](cudaError_t e, const char* w) { if (ce == cudaSuccess && e != cudaSuccess) { ce = e; what = w; } return e == cudaSuccess; };
    // On any failure: leave the loop, then ALWAYS drain both streams (copies into the caller's host_out may be in flight)
    // and report how many snapshots were written before returning the first error.
    for (int s = 0; s < n_steps && st == LS_OK && ce == cudaSuccess; ++s) {
        st = c->dtype == LS_F32 ? step_impl<float>(c, (float*)phi, (const float*)F, &q, 1)
                                : step_impl<double>(c, (double*)phi, (const double*)F, &q, 1);
        if (st != LS_OK) break;
        q.chained = 1;   // same buffer, untouched in between
        if ((s + 1) % every == 0) {
            const int slot = k & 1;
            if (k >= 2 && !ck(cudaStreamWaitEvent(c->stream, c->snap_free[slot], 0), "cudaStreamWaitEvent")) break;   // its last D2H has drained
            {
                ProfScope ps(c, LS_K_COPY);
                if (!ck(cudaMemcpyAsync(c->snap[slot], phi, bytes, cudaMemcpyDeviceToDevice, c->stream), "snapshot copy")) break;
            }
            if (!ck(cudaEventRecord(c->snap_ready[slot], c->stream), "cudaEventRecord")) break;
            if (!ck(cudaStreamWaitEvent(c->copy_stream, c->snap_ready[slot], 0), "cudaStreamWaitEvent")) break;
            if (!ck(cudaMemcpyAsync((char*)host_out + (size_t)k * bytes, c->snap[slot], bytes, cudaMemcpyDeviceToHost,
                                    c->copy_stream), "snapshot download")) break;
            if (!ck(cudaEventRecord(c->snap_free[slot], c->copy_stream), "cudaEventRecord")) break;
            ++k;
        }
    }
    cudaError_t e1 = cudaStreamSynchronize(c->stream), e2 = cudaStreamSynchronize(c->copy_stream);
    if (n_written) *n_written = k;
    if (ce != cudaSuccess) return cuda_fail(ce, what);
    if (e1 != cudaSuccess) return cuda_fail(e1, "ls_step_snapshots: cudaStreamSynchronize");
    if (e2 != cudaSuccess) return cuda_fail(e2, "ls_step_snapshots: cudaStreamSynchronize(copy)");
    return st;
}

ls_status ls_stats(ls_ctx* c, int64_t* point_updates, int64_t* steps, int64_t* kernel_launches) {
    if (!c) return LS_ERR_ARG;
    LS_CK(cudaMemcpyAsync(c->host_counts, c->bb.counts, sizeof(ls::Counts), cudaMemcpyDeviceToHost, c->stream));
    LS_CK(cudaStreamSynchronize(c->stream));
    if (point_updates) *point_updates = (int64_t)c->host_counts->updates + c->dense_updates;
    if (steps) *steps = (int64_t)c->host_counts->steps;
    if (kernel_launches) *kernel_launches = c->launches;
    return LS_OK;
}

ls_status ls_tile_threshold(ls_ctx* c, int64_t min_cells) {
    if (!c) return LS_ERR_ARG;
    c->tile_min_cells = min_cells < 0 ? (int64_t)LS_TILE_MIN_CELLS : min_cells;
    return LS_OK;
}

ls_status ls_profile_enable(ls_ctx* c, int32_t on) {
    if (!c) return LS_ERR_ARG;
    c->prof_on = on != 0;
    return LS_OK;
}

ls_status ls_profile_read(ls_ctx* c, int32_t kind, double* ms_total, int64_t* launches) {
    if (!c || kind < 0 || kind >= LS_K_KINDS) return LS_ERR_ARG;
    ls_status st = prof_collect(c);
    if (st != LS_OK) return st;
    if (ms_total) *ms_total = c->prof_ms[kind];
    if (launches) *launches = c->prof_n[kind];
    return LS_OK;
}

ls_status ls_profile_reset(ls_ctx* c) {
    if (!c) return LS_ERR_ARG;
    ls_status st = prof_collect(c);
    for (int k = 0; k < LS_K_KINDS; ++k) { c->prof_ms[k] = 0.0; c->prof_n[k] = 0; }
    return st;
}

ls_status ls_selftest_math(void* cuda_stream, uint64_t seed, int64_t n, double dx, double dt, double beta,
                           double gamma, int64_t* mismatches) {
    if (!mismatches || n < 0 || bad_band_params(dx, beta, gamma) || std::isinf(gamma)) return LS_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    unsigned long long* d = nullptr;
    LS_CK(cudaMalloc((void**)&d, 16 + 32 * sizeof(float)));
    float* dbg = reinterpret_cast<float*>(d + 2);
    cudaError_t e = cudaMemsetAsync(d, 0, 16 + 32 * sizeof(float), s);
    struct { unsigned long long n[2]; float v[32]; } out;
    std::memset(&out, 0, sizeof out);
    if (e == cudaSuccess) {
        ls::launch_selftest_math(seed, n, make_params<float>(dx, dt, beta, gamma), d, dbg, s);
        e = cudaPeekAtLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&out, d, sizeof out, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(d);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e, "ls_selftest_math"); }
    const unsigned long long h = out.n[0];
#ifdef LS_DEBUG
    if (h) {   // first differing sample: stencils (zm ym xm c xp yp zp) x2, F, scalar / packed results
        std::fprintf(stderr, "ls_selftest_math: %llu results differ; first sample:\n", h);
        for (int k = 0; k < 32; ++k) {
            unsigned bits;
            std::memcpy(&bits, &out.v[k], 4);
            std::fprintf(stderr, "  [%2d] %.9g (0x%08x)\n", k, out.v[k], bits);
        }
    }
#endif
    *mismatches = (int64_t)h;
    return LS_OK;
}

ls_status ls_stats_reset(ls_ctx* c) {
    if (!c) return LS_ERR_ARG;
    LS_CK(cudaMemsetAsync((char*)c->bb.counts + offsetof(ls::Counts, updates), 0, 16, c->stream));
    c->launches = 0;
    c->dense_updates = 0;
    return LS_OK;
}

}  // extern "C"
