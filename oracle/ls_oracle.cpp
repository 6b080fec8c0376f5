// ls_oracle.cpp — CPU ORACLE for the narrow-band level-set hot path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference leg may load it.  It shares no code,
// header, table or helper with paper_1612_04040_b200/csrc (the CUDA path); the two
// never include or import each other.
//
// It is the paper's algorithm written out step by step, in the paper's order
// (Steps 1-3), with plain nested loops over (k, j, i):
//   O1  neighbour access, edge replicate               (reading R3)
//   O2  one-sided differences D^{-x}, D^{+x}, ...      (eq. 3-5 notation; R1)
//   O3  upwind sums q+ = (nabla+)^2, q- = (nabla-)^2   (eq. 4, 5; R2, R19)
//   O4  cut-off c(phi)                                 (eq. 7; R5)
//   O5  tubes T and N, 8^3 brick lists                 (eq. 6, eq. 11; R6, R20)
//   O6  Advance                                        (eq. 3 with eq. 8; R8, R15)
//   O7  Reinitialisation iteration                     (eq. 12-13; R9-R12, R15)
//   O8  one narrow-band step, clamp of eq. 10          (R7, R14)
// No blocking, fusion or reordering beyond what those passages state.  All per-point
// arithmetic is in T (float or double); parameters arrive as double and are rounded to T
// once (R18).  Build with -ffp-contract=off (no FMA contraction).
//
// Parity pins: tests/test_oracle_pins.py (I1-I14 of DESIGN.md).  Unpinned by anything the
// paper prints ("parity unpinned"): the choice of face- vs box-neighbourhood in eq. 11 (R6),
// the meaning of |Dd| in eq. 13 (R10), and the domain-boundary rule (R3).  DESIGN.md lists them.
//
// `#pragma omp parallel for` on the outer loops only changes who executes an iteration;
// every output element is still produced by exactly one iteration, from the same inputs,
// so results are identical for any thread count.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Dims {
    int nx, ny, nz;
    int64_t idx(int i, int j, int k) const { return ((int64_t)k * ny + j) * nx + i; }
    int64_t size() const { return (int64_t)nx * ny * nz; }
};

// max(x,0) and min(x,0) of eq. 3-5
template <class T> inline T pos(T x) { return x > T(0) ? x : T(0); }
template <class T> inline T neg(T x) { return x < T(0) ? x : T(0); }

// O1: phi(i,j,k) with indices clamped to the domain (edge replicate, R3)
template <class T>
inline T at(const T* phi, const Dims& g, int i, int j, int k) {
    if (i < 0) i = 0; if (i > g.nx - 1) i = g.nx - 1;
    if (j < 0) j = 0; if (j > g.ny - 1) j = g.ny - 1;
    if (k < 0) k = 0; if (k > g.nz - 1) k = g.nz - 1;
    return phi[g.idx(i, j, k)];
}

// O2 + O3: q+ = (nabla+)^2 of eq. 4 and q- = (nabla-)^2 of eq. 5 at (i,j,k)
template <class T>
inline void upwind_q(const T* phi, const Dims& g, int i, int j, int k, T inv, T& qp, T& qm) {
    const T c = at(phi, g, i, j, k);
    const T Dmx = (c - at(phi, g, i - 1, j, k)) * inv;
    const T Dpx = (at(phi, g, i + 1, j, k) - c) * inv;
    const T Dmy = (c - at(phi, g, i, j - 1, k)) * inv;
    const T Dpy = (at(phi, g, i, j + 1, k) - c) * inv;
    const T Dmz = (c - at(phi, g, i, j, k - 1)) * inv;
    const T Dpz = (at(phi, g, i, j, k + 1) - c) * inv;
    // eq. 4, summed pairwise by axis: ((x-pair) + (y-pair)) + (z-pair)   (R19)
    qp = ((pos(Dmx) * pos(Dmx) + neg(Dpx) * neg(Dpx)) +
          (pos(Dmy) * pos(Dmy) + neg(Dpy) * neg(Dpy))) +
         (pos(Dmz) * pos(Dmz) + neg(Dpz) * neg(Dpz));
    // eq. 5
    qm = ((pos(Dpx) * pos(Dpx) + neg(Dmx) * neg(Dmx)) +
          (pos(Dpy) * pos(Dpy) + neg(Dmy) * neg(Dmy))) +
         (pos(Dpz) * pos(Dpz) + neg(Dmz) * neg(Dmz));
}

// O4: eq. 7.  beta = gamma = +inf: the first branch always fires (full-domain mode).
template <class T>
struct Cutoff {
    T beta, gamma, three_beta, inv3;
    Cutoff(double b, double gm) {
        beta = (T)b; gamma = (T)gm;
        three_beta = T(3) * beta;
        const T w = gamma - beta;
        inv3 = T(1) / ((w * w) * w);
    }
    T operator()(T phi_c) const {
        const T a = std::fabs(phi_c);
        if (a <= beta) return T(1);
        if (a <= gamma) {
            const T t = a - gamma;
            return ((t * t) * (((T(2) * a) + gamma) - three_beta)) * inv3;
        }
        return T(0);
    }
};

// O6 at one point: phi_bar = phi - dt * (c(phi) * [max(F,0) nabla+ + min(F,0) nabla-])
template <class T>
inline T advance_point(const T* phi, const T* F, const Dims& g, int i, int j, int k,
                       T inv, T dt, const Cutoff<T>& cut) {
    T qp, qm;
    upwind_q(phi, g, i, j, k, inv, qp, qm);
    const T gp = std::sqrt(qp), gm = std::sqrt(qm);
    const T c = phi[g.idx(i, j, k)];
    const T f = F[g.idx(i, j, k)];
    const T H = pos(f) * gp + neg(f) * gm;
    return c - dt * (cut(c) * H);
}

// O7 at one point: d' = d - dtau * [max(S,0)(nabla+ - 1) + min(S,0)(nabla- - 1)],
// S = d / sqrt(d^2 + |Dd|^2 dx^2), |Dd|^2 = q+ if d>0, q- if d<0 (R10); S = 0 if the root is 0 (R12)
template <class T>
inline T reinit_point(const T* d, const Dims& g, int i, int j, int k, T inv, T dx, T dtau) {
    T qp, qm;
    upwind_q(d, g, i, j, k, inv, qp, qm);
    const T gp = std::sqrt(qp), gm = std::sqrt(qm);
    const T c = d[g.idx(i, j, k)];
    const T q = c > T(0) ? qp : (c < T(0) ? qm : T(0));
    const T den = std::sqrt(c * c + q * (dx * dx));
    const T S = den == T(0) ? T(0) : c / den;
    const T U = pos(S) * (gp - T(1)) + neg(S) * (gm - T(1));
    return c - dtau * U;
}

// O5: point masks.  T = {|phi| < gamma} (eq. 6); N = T or a face neighbour inside the domain in T (eq. 11, R6)
template <class T>
void band_masks(const T* phi, const Dims& g, double gamma_d, uint8_t* Tm, uint8_t* Nm) {
    const T gamma = (T)gamma_d;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i)
                Tm[g.idx(i, j, k)] = std::fabs(phi[g.idx(i, j, k)]) < gamma ? 1 : 0;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                uint8_t m = Tm[g.idx(i, j, k)];
                if (i > 0) m |= Tm[g.idx(i - 1, j, k)];
                if (i < g.nx - 1) m |= Tm[g.idx(i + 1, j, k)];
                if (j > 0) m |= Tm[g.idx(i, j - 1, k)];
                if (j < g.ny - 1) m |= Tm[g.idx(i, j + 1, k)];
                if (k > 0) m |= Tm[g.idx(i, j, k - 1)];
                if (k < g.nz - 1) m |= Tm[g.idx(i, j, k + 1)];
                Nm[g.idx(i, j, k)] = m;
            }
}

// O5: 8^3 brick list of a point mask.  Brick id b = (bz*NBy + by)*NBx + bx; word lz, bit ly*8+lx (R20).
// Returns the number of non-empty bricks; writes at most `cap` entries (ascending id).
int64_t brick_list(const uint8_t* mask, const Dims& g, int32_t* ids, uint64_t* words, int64_t cap,
                   int64_t* n_points) {
    const int NBx = (g.nx + 7) / 8, NBy = (g.ny + 7) / 8, NBz = (g.nz + 7) / 8;
    int64_t count = 0, pts = 0;
    for (int bz = 0; bz < NBz; ++bz)
        for (int by = 0; by < NBy; ++by)
            for (int bx = 0; bx < NBx; ++bx) {
                uint64_t w[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                bool any = false;
                for (int lz = 0; lz < 8; ++lz)
                    for (int ly = 0; ly < 8; ++ly)
                        for (int lx = 0; lx < 8; ++lx) {
                            const int i = bx * 8 + lx, j = by * 8 + ly, k = bz * 8 + lz;
                            if (i < g.nx && j < g.ny && k < g.nz && mask[g.idx(i, j, k)]) {
                                w[lz] |= (uint64_t)1 << (ly * 8 + lx);
                                any = true;
                                ++pts;
                            }
                        }
                if (any) {
                    if (ids && count < cap) {
                        ids[count] = (bz * NBy + by) * NBx + bx;
                        if (words) std::memcpy(words + 8 * count, w, sizeof w);
                    }
                    ++count;
                }
            }
    if (n_points) *n_points = pts;
    return count;
}

// O6 over the grid: mask == nullptr means every point (full-domain mode, cfg 2)
template <class T>
void advance(const T* phi, const T* F, const uint8_t* Tm, const Dims& g, double dt_d, double dx_d,
             double beta_d, double gamma_d, T* out) {
    const T dx = (T)dx_d, dt = (T)dt_d, inv = T(1) / dx;
    const Cutoff<T> cut(beta_d, gamma_d);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                const int64_t p = g.idx(i, j, k);
                out[p] = (!Tm || Tm[p]) ? advance_point(phi, F, g, i, j, k, inv, dt, cut) : phi[p];
            }
}

// O7 over the grid; returns r = max_{x in N} |d' - d|
template <class T>
double reinit_iter(const T* d, const uint8_t* Nm, const Dims& g, double dtau_d, double dx_d, T* out) {
    const T dx = (T)dx_d, dtau = (T)dtau_d, inv = T(1) / dx;
    double res = 0.0;
#pragma omp parallel for schedule(static) reduction(max : res)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                const int64_t p = g.idx(i, j, k);
                if (Nm[p]) {
                    const T v = reinit_point(d, g, i, j, k, inv, dx, dtau);
                    const double r = std::fabs((double)(v - d[p]));
                    if (r > res) res = r;
                    out[p] = v;
                } else {
                    out[p] = d[p];
                }
            }
    return res;
}

// eq. 10 on every point (R14)
template <class T>
void clamp_all(T* d, int64_t n, double gamma_d) {
    const T gamma = (T)gamma_d;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        T v = d[p];
        if (v < -gamma) v = -gamma;
        if (v > gamma) v = gamma;
        d[p] = v;
    }
}

// List-driven variants (the paper's "active points are stored in an array").
// Same per-point functions, iterated over the brick list instead of the whole grid; points
// not listed are NOT touched, so `out` must already hold a copy of the input there.
template <class T, class Fn>
void for_each_listed(const Dims& g, const int32_t* ids, const uint64_t* words, int64_t nb, Fn fn) {
    const int NBx = (g.nx + 7) / 8, NBy = (g.ny + 7) / 8;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t n = 0; n < nb; ++n) {
        const int b = ids[n];
        const int bx = b % NBx, by = (b / NBx) % NBy, bz = b / (NBx * NBy);
        for (int lz = 0; lz < 8; ++lz) {
            const uint64_t w = words[8 * n + lz];
            if (!w) continue;
            for (int ly = 0; ly < 8; ++ly)
                for (int lx = 0; lx < 8; ++lx)
                    if ((w >> (ly * 8 + lx)) & 1) fn(bx * 8 + lx, by * 8 + ly, bz * 8 + lz);
        }
    }
}

template <class T>
void advance_list(const T* phi, const T* F, const int32_t* ids, const uint64_t* words, int64_t nb,
                  const Dims& g, double dt_d, double dx_d, double beta_d, double gamma_d, T* out) {
    const T dx = (T)dx_d, dt = (T)dt_d, inv = T(1) / dx;
    const Cutoff<T> cut(beta_d, gamma_d);
    for_each_listed<T>(g, ids, words, nb, [&](int i, int j, int k) {
        out[g.idx(i, j, k)] = advance_point(phi, F, g, i, j, k, inv, dt, cut);
    });
}

template <class T>
void reinit_iter_list(const T* d, const int32_t* ids, const uint64_t* words, int64_t nb, const Dims& g,
                      double dtau_d, double dx_d, T* out) {
    const T dx = (T)dx_d, dtau = (T)dtau_d, inv = T(1) / dx;
    for_each_listed<T>(g, ids, words, nb, [&](int i, int j, int k) {
        out[g.idx(i, j, k)] = reinit_point(d, g, i, j, k, inv, dx, dtau);
    });
}

// O8: `n_steps` narrow-band steps in place on phi.  Full-grid masked evaluation (use_lists = 0)
// or the list-driven evaluation (use_lists = 1); the two must agree bit for bit (pin I14).
// updates += |T| + iters*|N| per step.  Returns 0, or -1 on allocation failure.
template <class T>
int step(T* phi, const T* F, const Dims& g, double dx, double dt, double dtau, double beta, double gamma,
         int iters, int n_steps, int use_lists, int64_t* updates) {
    const int64_t n = g.size();
    std::vector<T> a, b;
    std::vector<uint8_t> Tm, Nm;
    try {
        a.resize(n); b.resize(n); Tm.resize(n); Nm.resize(n);
    } catch (...) { return -1; }
    int64_t upd = 0;
    for (int s = 0; s < n_steps; ++s) {
        band_masks(phi, g, gamma, Tm.data(), Nm.data());              // Step 1 (R7: both from phi^n)
        int64_t nT = 0, nN = 0;
        if (!use_lists) {
            for (int64_t p = 0; p < n; ++p) { nT += Tm[p]; nN += Nm[p]; }
            advance(phi, F, Tm.data(), g, dt, dx, beta, gamma, a.data());   // Step 2
            T* cur = a.data(); T* nxt = b.data();
            for (int it = 0; it < iters; ++it) {                            // Step 3
                reinit_iter(cur, Nm.data(), g, dtau, dx, nxt);
                T* t = cur; cur = nxt; nxt = t;
            }
            std::memcpy(phi, cur, n * sizeof(T));
        } else {
            const int64_t capT = brick_list(Tm.data(), g, nullptr, nullptr, 0, &nT);
            const int64_t capN = brick_list(Nm.data(), g, nullptr, nullptr, 0, &nN);
            std::vector<int32_t> Tid(capT), Nid(capN);
            std::vector<uint64_t> Tw(8 * capT), Nw(8 * capN);
            brick_list(Tm.data(), g, Tid.data(), Tw.data(), capT, nullptr);
            brick_list(Nm.data(), g, Nid.data(), Nw.data(), capN, nullptr);
            std::memcpy(a.data(), phi, n * sizeof(T));
            advance_list(phi, F, Tid.data(), Tw.data(), capT, g, dt, dx, beta, gamma, a.data());
            std::memcpy(b.data(), a.data(), n * sizeof(T));
            T* cur = a.data(); T* nxt = b.data();
            for (int it = 0; it < iters; ++it) {
                // every sweep rewrites all of N in `nxt`; off N both buffers hold phi_bar
                reinit_iter_list(cur, Nid.data(), Nw.data(), capN, g, dtau, dx, nxt);
                T* t = cur; cur = nxt; nxt = t;
            }
            std::memcpy(phi, cur, n * sizeof(T));
        }
        clamp_all(phi, n, gamma);                                           // eq. 10 everywhere (R14)
        upd += nT + (int64_t)iters * nN;
    }
    if (updates) *updates = upd;
    return 0;
}

// cfg 5 (R13, R25): reinit on the N of `phi` until r_k < tol at a k that is a multiple of check_every.
// d (out) holds the clamped result.  Returns iterations done; *converged says whether tol was met.
template <class T>
int reinit_tol(const T* phi_bar, T* d, const Dims& g, double dtau, double dx, double gamma, double tol,
               int max_iters, int check_every, double* residual, int* converged) {
    const int64_t n = g.size();
    std::vector<uint8_t> Tm(n), Nm(n);
    band_masks(phi_bar, g, gamma, Tm.data(), Nm.data());
    std::vector<T> other(n);
    std::memcpy(d, phi_bar, n * sizeof(T));
    T* cur = d; T* nxt = other.data();
    int k = 0; double r = 0.0; *converged = 0;
    while (k < max_iters) {
        r = reinit_iter(cur, Nm.data(), g, dtau, dx, nxt);
        T* t = cur; cur = nxt; nxt = t;
        ++k;
        if (k % check_every == 0 && r < tol) { *converged = 1; break; }
    }
    if (cur != d) std::memcpy(d, cur, n * sizeof(T));
    clamp_all(d, n, gamma);
    if (residual) *residual = r;
    return k;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C entry points for the ctypes wrapper (oracle/ls_oracle.py).  _f32 / _f64 pick T.
// ---------------------------------------------------------------------------------------------
#define ORC_INSTANTIATE(SUF, T)                                                                              \
    extern "C" double orc_cutoff_##SUF(double phi_c, double beta, double gamma) {                           \
        return (double)Cutoff<T>(beta, gamma)((T)phi_c);                                                     \
    }                                                                                                        \
    extern "C" void orc_upwind_q_##SUF(const T* phi, int nx, int ny, int nz, int i, int j, int k, double dx, \
                                       double* qp, double* qm) {                                             \
        Dims g{nx, ny, nz}; T a, b;                                                                          \
        upwind_q<T>(phi, g, i, j, k, T(1) / (T)dx, a, b);                                                    \
        *qp = (double)a; *qm = (double)b;                                                                    \
    }                                                                                                        \
    extern "C" void orc_band_masks_##SUF(const T* phi, int nx, int ny, int nz, double gamma, uint8_t* Tm,   \
                                         uint8_t* Nm) {                                                      \
        band_masks<T>(phi, Dims{nx, ny, nz}, gamma, Tm, Nm);                                                 \
    }                                                                                                        \
    extern "C" void orc_advance_##SUF(const T* phi, const T* F, const uint8_t* Tm, int nx, int ny, int nz,  \
                                      double dt, double dx, double beta, double gamma, T* out) {             \
        advance<T>(phi, F, Tm, Dims{nx, ny, nz}, dt, dx, beta, gamma, out);                                  \
    }                                                                                                        \
    extern "C" double orc_advance_point_##SUF(const T* phi, const T* F, int nx, int ny, int nz, int i,      \
                                              int j, int k, double dt, double dx, double beta,              \
                                              double gamma) {                                                \
        Dims g{nx, ny, nz};                                                                                  \
        return (double)advance_point<T>(phi, F, g, i, j, k, T(1) / (T)dx, (T)dt, Cutoff<T>(beta, gamma));    \
    }                                                                                                        \
    extern "C" double orc_reinit_iter_##SUF(const T* d, const uint8_t* Nm, int nx, int ny, int nz,          \
                                            double dtau, double dx, T* out) {                                \
        return reinit_iter<T>(d, Nm, Dims{nx, ny, nz}, dtau, dx, out);                                       \
    }                                                                                                        \
    extern "C" double orc_reinit_point_##SUF(const T* d, int nx, int ny, int nz, int i, int j, int k,       \
                                             double dtau, double dx) {                                       \
        Dims g{nx, ny, nz};                                                                                  \
        return (double)reinit_point<T>(d, g, i, j, k, T(1) / (T)dx, (T)dx, (T)dtau);                         \
    }                                                                                                        \
    extern "C" void orc_clamp_##SUF(T* d, int64_t n, double gamma) { clamp_all<T>(d, n, gamma); }            \
    extern "C" void orc_advance_list_##SUF(const T* phi, const T* F, const int32_t* ids,                    \
                                           const uint64_t* words, int64_t nb, int nx, int ny, int nz,       \
                                           double dt, double dx, double beta, double gamma, T* out) {       \
        advance_list<T>(phi, F, ids, words, nb, Dims{nx, ny, nz}, dt, dx, beta, gamma, out);                 \
    }                                                                                                        \
    extern "C" void orc_reinit_iter_list_##SUF(const T* d, const int32_t* ids, const uint64_t* words,       \
                                               int64_t nb, int nx, int ny, int nz, double dtau, double dx,  \
                                               T* out) {                                                     \
        reinit_iter_list<T>(d, ids, words, nb, Dims{nx, ny, nz}, dtau, dx, out);                             \
    }                                                                                                        \
    extern "C" int orc_step_##SUF(T* phi, const T* F, int nx, int ny, int nz, double dx, double dt,         \
                                  double dtau, double beta, double gamma, int iters, int n_steps,           \
                                  int use_lists, int64_t* updates) {                                         \
        return step<T>(phi, F, Dims{nx, ny, nz}, dx, dt, dtau, beta, gamma, iters, n_steps, use_lists,       \
                       updates);                                                                             \
    }                                                                                                        \
    extern "C" int orc_reinit_tol_##SUF(const T* phi_bar, T* d, int nx, int ny, int nz, double dtau,        \
                                        double dx, double gamma, double tol, int max_iters,                 \
                                        int check_every, double* residual, int* converged) {                \
        return reinit_tol<T>(phi_bar, d, Dims{nx, ny, nz}, dtau, dx, gamma, tol, max_iters, check_every,     \
                             residual, converged);                                                           \
    }

ORC_INSTANTIATE(f32, float)
ORC_INSTANTIATE(f64, double)

extern "C" int64_t orc_brick_list(const uint8_t* mask, int nx, int ny, int nz, int32_t* ids, uint64_t* words,
                                  int64_t cap, int64_t* n_points) {
    return brick_list(mask, Dims{nx, ny, nz}, ids, words, cap, n_points);
}

extern "C" int orc_max_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

extern "C" void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
