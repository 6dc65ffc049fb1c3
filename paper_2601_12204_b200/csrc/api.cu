// api.cu -- the C ABI of include/burgers.h: argument validation, plan selection, dispatch,
// and the host-buffer (end-to-end) variants.  No arithmetic of the method lives here.
#include <algorithm>
#include <cmath>
#include <mutex>
#include <cstdint>

#include "common.cuh"

using namespace burgers;

namespace {

int check_common(const void *u, const void *nu, const void *dt, int64_t B, int64_t N, double L,
                 int64_t n_steps, int bc) {
    if (!u || !nu || !dt) return BURGERS_ERR_NULL;
    if (B < 1 || N < 3 || n_steps < 0) return BURGERS_ERR_SHAPE;
    if (bc != BURGERS_BC_PERIODIC && bc != BURGERS_BC_DIRICHLET) return BURGERS_ERR_ENUM;
    if (!(L > 0.0) || !std::isfinite(L)) return BURGERS_ERR_VALUE;
    return BURGERS_OK;
}

bool scheme_ok(int scheme) { return scheme == BURGERS_SCHEME_EULER || scheme == BURGERS_SCHEME_RK4; }

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// AUTO plan of the BTCS op: one long system -> LONG; a system that fits one
// CTA -> HYBRID; anything else -> THOMAS.
int btcs_auto_plan(int is_f64, int64_t B, int64_t N, int bc) {
    if (btcs_hybrid_fits(is_f64, N, bc) && B < 200000) return BURGERS_PLAN_HYBRID;
    if (btcs_long_fits(is_f64, B, N, bc) && B < 65536) return BURGERS_PLAN_LONG;
    return BURGERS_PLAN_THOMAS;
}

template <typename T>
int explicit_call(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps,
                  int bc, int scheme, int plan, int tblock, int ppt, void *ws, size_t ws_bytes,
                  void *stream, T *snaps = nullptr, int64_t snap_every = 0) {
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (!scheme_ok(scheme)) return BURGERS_ERR_ENUM;
    if (plan != BURGERS_PLAN_AUTO && plan != BURGERS_PLAN_RESIDENT && plan != BURGERS_PLAN_TILED)
        return BURGERS_ERR_ENUM;
    ExplicitGeom g;
    st = explicit_geometry(sizeof(T) == 8, B, N, bc, scheme, plan, tblock, ppt, &g);
    if (st != BURGERS_OK) return st;
    if (g.plan == BURGERS_PLAN_TILED) {
        const size_t need = (size_t)B * (size_t)N * sizeof(T);
        if (!ws || ws_bytes < need) return BURGERS_ERR_WORKSPACE;
    }
    return launch_explicit<T>(u, B, N, grid_dx(N, L, bc), nu, dt, n_steps, bc, scheme, g, (T *)ws, snaps,
                              snap_every, (cudaStream_t)stream);
}

template <typename T>
int btcs_call(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc,
              int plan, void *ws, size_t ws_bytes, void *stream) {
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    const int is_f64 = sizeof(T) == 8;
    if (plan == BURGERS_PLAN_AUTO) plan = btcs_auto_plan(is_f64, B, N, bc);
    const double dx = grid_dx(N, L, bc);
    cudaStream_t s = (cudaStream_t)stream;
    switch (plan) {
        case BURGERS_PLAN_THOMAS: {
            const size_t need = btcs_thomas_ws_elems(B, N, bc) * sizeof(T);
            if (!ws || ws_bytes < need) return BURGERS_ERR_WORKSPACE;
            return launch_btcs_thomas<T>(u, B, N, dx, nu, dt, n_steps, bc, (T *)ws, s);
        }
        case BURGERS_PLAN_HYBRID:
            if (!btcs_hybrid_fits(is_f64, N, bc)) return BURGERS_ERR_PLAN;
            return launch_btcs_hybrid<T>(u, B, N, dx, nu, dt, n_steps, bc, s);
        case BURGERS_PLAN_LONG:
        case BURGERS_PLAN_LONG_GENERAL: {
            if (!btcs_long_fits(is_f64, B, N, bc)) return BURGERS_ERR_PLAN;
            const size_t need = btcs_long_ws_bytes((int)sizeof(T), B, N);
            if (!ws || ws_bytes < need) return BURGERS_ERR_WORKSPACE;
            return launch_btcs_long<T>(u, B, N, dx, nu, dt, n_steps, bc, ws,
                                       plan == BURGERS_PLAN_LONG_GENERAL, s);
        }
    }
    return BURGERS_ERR_ENUM;
}

template <typename T>
int cfl_call(const T *u, int64_t B, int64_t N, double L, const T *nu, double C, int bc, T *dt_out, void *stream);

// Adaptive time step (SURVEY 8(f) NEXT-4a): n_outer times { dt = dt_from_cfl(u); m explicit steps with it;
// t += m dt }, all enqueued on the stream, no host synchronisation; the CFL evaluation is fused into the kernels
// of both explicit plans.
inline size_t tiled_adapt_slot_bytes(int64_t B) { return align_up((size_t)3 * (size_t)B * sizeof(unsigned long long), 256); }

template <typename T>
int adaptive_call(T *u, int64_t B, int64_t N, double L, const T *nu, double C, int64_t n_outer, int64_t m_steps,
                  int bc, int scheme, T *dt_scratch, double *t_out, void *ws, size_t ws_bytes, void *stream) {
    if (!dt_scratch) return BURGERS_ERR_NULL;
    if (n_outer < 0 || m_steps < 1) return BURGERS_ERR_SHAPE;
    int st = check_common(u, nu, dt_scratch, B, N, L, 0, bc);
    if (st != BURGERS_OK) return st;
    if (!scheme_ok(scheme)) return BURGERS_ERR_ENUM;
    if (!(C > 0.0) || !std::isfinite(C)) return BURGERS_ERR_VALUE;
    cudaStream_t s = (cudaStream_t)stream;
    if (t_out && cudaMemsetAsync(t_out, 0, (size_t)B * sizeof(double), s) != cudaSuccess) return BURGERS_ERR_CUDA;
    // RESIDENT plan: one launch, the CFL evaluation fused into the time loop of the kernel
    ExplicitGeom g;
    st = explicit_geometry(sizeof(T) == 8, B, N, bc, scheme, BURGERS_PLAN_AUTO, 0, 0, &g);
    if (st != BURGERS_OK) return st;
    if (g.plan == BURGERS_PLAN_RESIDENT && n_outer <= INT64_MAX / m_steps) {
        if (n_outer == 0) return BURGERS_OK;
        const ExplicitAdapt<T> ad{m_steps, C, t_out, dt_scratch};
        return launch_explicit<T>(u, B, N, grid_dx(N, L, bc), nu, dt_scratch, n_outer * m_steps, bc, scheme, g, (T *)ws,
                                  nullptr, 0, s, &ad);
    }
    // TILED plan: the CFL reduction rides on the launches themselves (explicit_impl.cuh, TADAPT): the last launch of a
    // segment leaves max |u| of the state it stores in one of three rotating slots behind the ping-pong buffer, the
    // launches of the next segment evaluate dt from it.  Only the first dt comes from the CFL kernel.
    if (n_outer == 0) return BURGERS_OK;
    const size_t state_b = align_up((size_t)B * (size_t)N * sizeof(T), 256);
    if (!ws || ws_bytes < state_b + tiled_adapt_slot_bytes(B)) return BURGERS_ERR_WORKSPACE;
    unsigned long long *slots = reinterpret_cast<unsigned long long *>(static_cast<unsigned char *>(ws) + state_b);
    st = cfl_call<T>(u, B, N, L, nu, C, bc, dt_scratch, stream);
    if (st != BURGERS_OK) return st;
    if (cudaMemsetAsync(slots, 0, tiled_adapt_slot_bytes(B), s) != cudaSuccess) return BURGERS_ERR_CUDA;
    for (int64_t k = 0; k < n_outer; ++k) {
        const ExplicitTiledAdapt<T> ta{slots, k == 0 ? -1 : (int)((k - 1) % 3), (int)(k % 3), (int)((k + 1) % 3), C, t_out,
                                       dt_scratch};
        st = launch_explicit<T>(u, B, N, grid_dx(N, L, bc), nu, dt_scratch, m_steps, bc, scheme, g, (T *)ws, nullptr, 0, s,
                                nullptr, &ta);
        if (st != BURGERS_OK) return st;
    }
    return BURGERS_OK;
}

// Discrete adjoint of n_steps forward-Euler steps with CHECKPOINTING: the forward states are needed in
// reverse order.  The steps are cut into segments of m steps; a first forward sweep stores the state at
// every segment start (trajectory output with snap_every = m), then, last segment first, the segment
// is recomputed from its checkpoint with one snapshot per step and swept backwards.  m = n_steps (one
// segment, nothing recomputed) while all states fit kAdjointFullBytes, else ceil(sqrt(n_steps)), which
// minimises the memory (n_steps/m + m states) at the cost of a second forward sweep.
// ws layout: [lam ping-pong B*N][u work B*N][checkpoints (K-1)*B*N][segment states (m-1)*B*N][explicit ws].
constexpr size_t kAdjointFullBytes = (size_t)8 << 30;

inline int64_t adjoint_segment(size_t esz, int64_t B, int64_t N, int64_t n_steps, int64_t segment) {
    if (segment > 0) return segment < n_steps ? segment : (n_steps > 0 ? n_steps : 1);
    if (n_steps <= 1 || (size_t)n_steps * (size_t)B * (size_t)N * esz <= kAdjointFullBytes) return n_steps > 0 ? n_steps : 1;
    int64_t m = (int64_t)std::ceil(std::sqrt((double)n_steps));
    return m < 1 ? 1 : m;
}

// (RK4: + the stage values and transposed-Jacobian products of the backward sweep, adjoint_rk4.cu)
template <typename T>
size_t adjoint_ws_bytes(int64_t B, int64_t N, int bc, int64_t n_steps, int64_t segment, int scheme) {
    const int64_t m = adjoint_segment(sizeof(T), B, N, n_steps, segment);
    const int64_t K = (n_steps + m - 1) / m;
    const size_t bn = align_up((size_t)B * (size_t)N * sizeof(T), 256);
    const size_t ck = align_up((size_t)(K > 1 ? K - 1 : 0) * (size_t)B * (size_t)N * sizeof(T), 256);
    const size_t st = align_up((size_t)(m > 1 ? m - 1 : 0) * (size_t)B * (size_t)N * sizeof(T), 256);
    const size_t rk = scheme == BURGERS_SCHEME_RK4 ? align_up(adjoint_rk4_ws_elems(B, N) * sizeof(T), 256) : 0;
    return 2 * bn + ck + st + rk + burgers_workspace_bytes(BURGERS_OP_EXPLICIT, sizeof(T) == 8, B, N, bc, scheme,
                                                           BURGERS_PLAN_AUTO);
}

template <typename T>
int adjoint_call(const T *u0, T *lam, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps,
                 int bc, int64_t segment, void *ws, size_t ws_bytes, void *stream, int scheme = BURGERS_SCHEME_EULER) {
    if (!lam) return BURGERS_ERR_NULL;
    int st = check_common(u0, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (!scheme_ok(scheme)) return BURGERS_ERR_ENUM;
    if (segment < 0) return BURGERS_ERR_SHAPE;
    if (n_steps == 0) return BURGERS_OK;
    if (!ws || ws_bytes < adjoint_ws_bytes<T>(B, N, bc, n_steps, segment, scheme)) return BURGERS_ERR_WORKSPACE;
    const bool rk4 = (scheme == BURGERS_SCHEME_RK4);
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t m = adjoint_segment(sizeof(T), B, N, n_steps, segment);
    const int64_t K = (n_steps + m - 1) / m;
    const size_t BN = (size_t)B * (size_t)N;
    const size_t bn = align_up(BN * sizeof(T), 256);
    const size_t ckb = align_up((size_t)(K > 1 ? K - 1 : 0) * BN * sizeof(T), 256);
    const size_t stb = align_up((size_t)(m > 1 ? m - 1 : 0) * BN * sizeof(T), 256);
    unsigned char *base = static_cast<unsigned char *>(ws);
    T *pong = reinterpret_cast<T *>(base);
    T *work = reinterpret_cast<T *>(base + bn);
    T *ckpt = reinterpret_cast<T *>(base + 2 * bn);
    T *seg = reinterpret_cast<T *>(base + 2 * bn + ckb);
    const size_t rkb = rk4 ? align_up(adjoint_rk4_ws_elems(B, N) * sizeof(T), 256) : 0;
    T *rkws = reinterpret_cast<T *>(base + 2 * bn + ckb + stb);
    void *ews = base + 2 * bn + ckb + stb + rkb;
    const size_t ews_bytes = ws_bytes - (2 * bn + ckb + stb + rkb);
    const double dx = grid_dx(N, L, bc);
    auto forward = [&](const T *from, int64_t steps, T *snaps, int64_t every) {
        if (cudaMemcpyAsync(work, from, BN * sizeof(T), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
            return (int)BURGERS_ERR_CUDA;
        // A snapshot after EVERY step makes the resident kernel HBM-write-bound: 8 points per thread (four
        // times the warps of the compute-optimal 32) keep more stores in flight -- measured, B = 256,
        // N = 4096, 1 000 steps: forward + backward 2.02 -> 1.85 ms.  Same arithmetic per point, same bits.
        int plan_x = BURGERS_PLAN_AUTO, ppt_x = 0;
        ExplicitGeom g8;
        if (every == 1 && explicit_geometry(sizeof(T) == 8, B, N, bc, scheme, BURGERS_PLAN_RESIDENT, 0, 8, &g8) == BURGERS_OK) {
            plan_x = BURGERS_PLAN_RESIDENT;
            ppt_x = 8;
        }
        return explicit_call<T>(work, B, N, L, nu, dt, steps, bc, scheme, plan_x, 0, ppt_x, ews, ews_bytes, stream, snaps,
                                every);
    };
    if (K > 1) {            // checkpoints u^{m}, u^{2m}, ..., u^{(K-1)m}
        st = forward(u0, (K - 1) * m, ckpt, m);
        if (st != BURGERS_OK) return st;
    }
    for (int64_t k = K - 1; k >= 0; --k) {
        const T *start = (k == 0) ? u0 : ckpt + (size_t)(k - 1) * BN;
        const int64_t len = (k == K - 1) ? n_steps - k * m : m;
        if (len > 1) {      // states u^{km+1} .. u^{km+len-1} of this segment
            st = forward(start, len - 1, seg, 1);
            if (st != BURGERS_OK) return st;
        }
        st = rk4 ? launch_adjoint_rk4_steps<T>(start, seg, lam, rkws, B, N, dx, nu, dt, len, bc, s)
                 : launch_adjoint_steps<T>(start, seg, lam, pong, B, N, dx, nu, dt, len, bc, s);
        if (st != BURGERS_OK) return st;
    }
    return BURGERS_OK;
}

// BTCS with trajectory output: one call of the plan per snapshot interval (the state is stored once
// per interval anyway), then a device copy of u into snaps[k].
template <typename T>
int btcs_traj_call(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc,
                   int64_t snap_every, T *snaps, void *ws, size_t ws_bytes, void *stream) {
    if (!snaps) return BURGERS_ERR_NULL;
    if (snap_every < 1) return BURGERS_ERR_SHAPE;
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (btcs_auto_plan(sizeof(T) == 8, B, N, bc) == BURGERS_PLAN_HYBRID)       // snapshots written by the kernel: one launch
        return launch_btcs_hybrid_traj<T>(u, B, N, grid_dx(N, L, bc), nu, dt, n_steps, bc, snap_every, snaps,
                                          (cudaStream_t)stream);
    int64_t done = 0, k = 0;
    while (done < n_steps) {
        const int64_t chunk = (n_steps - done < snap_every) ? n_steps - done : snap_every;
        st = btcs_call<T>(u, B, N, L, nu, dt, chunk, bc, BURGERS_PLAN_AUTO, ws, ws_bytes, stream);
        if (st != BURGERS_OK) return st;
        done += chunk;
        if (chunk == snap_every) {
            if (cudaMemcpyAsync(snaps + k * B * N, u, (size_t)B * (size_t)N * sizeof(T), cudaMemcpyDeviceToDevice,
                                (cudaStream_t)stream) != cudaSuccess)
                return BURGERS_ERR_CUDA;
            ++k;
        }
    }
    return BURGERS_OK;
}

// ---- checkpointed reverse sweeps of the two implicit schemes (D15, D16) -----------------------------------
// As adjoint_call above: segments of m steps (adjoint_segment: one segment while all states fit 8 GiB, else
// ceil(sqrt(n_steps)), or the caller's), checkpoints at the segment starts from a first forward sweep, each
// segment recomputed with one snapshot per step and swept backwards.  Unlike the explicit schemes the backward step
// needs the state at BOTH ends of a step (D_i of D15 and the Jacobian of D16 are taken at u^{n+1}), so a segment
// stores its len states u^{km+1} .. u^{km+len}.
// ws layout: [u work B*N][checkpoints (K-1)*B*N][segment states m*B*N][backward scratch][workspace of the forward op].
template <typename T>
size_t implicit_adjoint_ws_bytes(int64_t B, int64_t N, int bc, int64_t n_steps, int64_t segment, int op) {
    const int64_t m = adjoint_segment(sizeof(T), B, N, n_steps, segment);
    const int64_t K = (n_steps + m - 1) / m;
    const size_t BN = (size_t)B * (size_t)N;
    const size_t bn = align_up(BN * sizeof(T), 256);
    const size_t ck = align_up((size_t)(K > 1 ? K - 1 : 0) * BN * sizeof(T), 256);
    const size_t st = align_up((size_t)m * BN * sizeof(T), 256);
    const size_t sc = align_up((op == BURGERS_OP_BTCS ? adjoint_btcs_ws_elems(sizeof(T) == 8, B, N)
                                                      : adjoint_newton_ws_elems(sizeof(T) == 8, B, N)) * sizeof(T), 256);
    return bn + ck + st + sc + burgers_workspace_bytes(op, sizeof(T) == 8, B, N, bc, 0, BURGERS_PLAN_AUTO);
}

// forward(work, steps, snaps, every): `steps` steps from the state in `work`, snapshots as the *_traj_* calls;
// backward(start, states, scratch, len): lam through the len steps that start at `start` (states: the len states after it)
template <typename T, typename Fwd, typename Bwd>
int implicit_adjoint_sweep(const T *u0, int64_t B, int64_t N, int bc, int64_t n_steps, int64_t segment, int op, void *ws,
                           size_t ws_bytes, cudaStream_t s, Fwd forward, Bwd backward) {
    if (segment < 0) return BURGERS_ERR_SHAPE;
    if (n_steps == 0) return BURGERS_OK;
    if (!ws || ws_bytes < implicit_adjoint_ws_bytes<T>(B, N, bc, n_steps, segment, op)) return BURGERS_ERR_WORKSPACE;
    const int64_t m = adjoint_segment(sizeof(T), B, N, n_steps, segment);
    const int64_t K = (n_steps + m - 1) / m;
    const size_t BN = (size_t)B * (size_t)N;
    const size_t bn = align_up(BN * sizeof(T), 256);
    const size_t ckb = align_up((size_t)(K > 1 ? K - 1 : 0) * BN * sizeof(T), 256);
    const size_t stb = align_up((size_t)m * BN * sizeof(T), 256);
    const size_t scb = align_up((op == BURGERS_OP_BTCS ? adjoint_btcs_ws_elems(sizeof(T) == 8, B, N)
                                                       : adjoint_newton_ws_elems(sizeof(T) == 8, B, N)) * sizeof(T), 256);
    unsigned char *base = static_cast<unsigned char *>(ws);
    T *work = reinterpret_cast<T *>(base);
    T *ckpt = reinterpret_cast<T *>(base + bn);
    T *seg = reinterpret_cast<T *>(base + bn + ckb);
    T *scratch = reinterpret_cast<T *>(base + bn + ckb + stb);
    void *ows = base + bn + ckb + stb + scb;
    const size_t ows_bytes = ws_bytes - (bn + ckb + stb + scb);
    auto run_forward = [&](const T *from, int64_t steps, T *snaps, int64_t every) {
        if (cudaMemcpyAsync(work, from, BN * sizeof(T), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
            return (int)BURGERS_ERR_CUDA;
        return forward(work, steps, snaps, every, ows, ows_bytes);
    };
    int st = BURGERS_OK;
    if (K > 1) {            // checkpoints u^{m}, u^{2m}, ..., u^{(K-1)m}
        st = run_forward(u0, (K - 1) * m, ckpt, m);
        if (st != BURGERS_OK) return st;
    }
    for (int64_t k = K - 1; k >= 0; --k) {
        const T *start = (k == 0) ? u0 : ckpt + (size_t)(k - 1) * BN;
        const int64_t len = (k == K - 1) ? n_steps - k * m : m;
        st = run_forward(start, len, seg, 1);
        if (st != BURGERS_OK) return st;
        st = backward(start, seg, scratch, len);
        if (st != BURGERS_OK) return st;
    }
    return BURGERS_OK;
}

template <typename T>
int btcs_adjoint_call(const T *u0, T *lam, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc,
                      int64_t segment, void *ws, size_t ws_bytes, void *stream) {
    if (!lam) return BURGERS_ERR_NULL;
    int st = check_common(u0, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    const double dx = grid_dx(N, L, bc);
    return implicit_adjoint_sweep<T>(
        u0, B, N, bc, n_steps, segment, BURGERS_OP_BTCS, ws, ws_bytes, s,
        [&](T *work, int64_t steps, T *snaps, int64_t every, void *ows, size_t ows_bytes) {
            return btcs_traj_call<T>(work, B, N, L, nu, dt, steps, bc, every, snaps, ows, ows_bytes, stream);
        },
        [&](const T *start, const T *states, T *scratch, int64_t len) {
            return launch_adjoint_btcs_steps<T>(start, states, lam, scratch, B, N, dx, nu, dt, len, bc, s);
        });
}

template <typename T>
int gs_call(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc, double tol,
            int max_iter, int64_t *iters_out, void *ws, size_t ws_bytes, void *stream) {
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (!(tol >= 0.0) || max_iter < 0) return BURGERS_ERR_VALUE;
    const size_t need = btcs_gs_ws_elems(B, N) * sizeof(T);
    if (need && (!ws || ws_bytes < need)) return BURGERS_ERR_WORKSPACE;
    return launch_btcs_gs<T>(u, B, N, grid_dx(N, L, bc), nu, dt, n_steps, bc, tol, max_iter,
                             reinterpret_cast<long long *>(iters_out), (T *)ws, (cudaStream_t)stream);
}

template <typename T>
int newton_call(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc,
                double theta, double tol, int max_iter, int64_t *iters_out, int plan, void *ws, size_t ws_bytes,
                void *stream, bool accumulate = false) {
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (!(tol >= 0.0) || max_iter < 0 || !(theta >= 0.0 && theta <= 1.0)) return BURGERS_ERR_VALUE;
    const int is_f64 = sizeof(T) == 8;
    if (plan == BURGERS_PLAN_AUTO) plan = newton_hybrid_fits(is_f64, N) ? BURGERS_PLAN_HYBRID : BURGERS_PLAN_THOMAS;
    if (plan != BURGERS_PLAN_HYBRID && plan != BURGERS_PLAN_THOMAS) return BURGERS_ERR_ENUM;
    if (plan == BURGERS_PLAN_HYBRID && !newton_hybrid_fits(is_f64, N)) return BURGERS_ERR_PLAN;
    if (plan == BURGERS_PLAN_THOMAS) {
        const size_t need = newton_thomas_ws_elems(B, N, bc) * sizeof(T);
        if (!ws || ws_bytes < need) return BURGERS_ERR_WORKSPACE;
    }
    static_assert(sizeof(long long) == sizeof(int64_t), "iters_out is int64");
    return launch_newton<T>(u, B, N, grid_dx(N, L, bc), nu, dt, n_steps, bc, theta, tol, max_iter,
                            reinterpret_cast<long long *>(iters_out), plan, (T *)ws, (cudaStream_t)stream, accumulate);
}

// Newton / theta-scheme with trajectory output: shapes of the HYBRID plan write the snapshots from inside the kernel
// (one launch); otherwise one run of the plan per snapshot interval and a device copy of u into snaps[k], the
// iteration totals accumulating over the intervals.
template <typename T>
int newton_traj_call(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc, double theta,
                     double tol, int max_iter, int64_t *iters_out, int64_t snap_every, T *snaps, void *ws, size_t ws_bytes,
                     void *stream) {
    if (!snaps) return BURGERS_ERR_NULL;
    if (snap_every < 1) return BURGERS_ERR_SHAPE;
    int st = newton_call<T>(u, B, N, L, nu, dt, 0, bc, theta, tol, max_iter, iters_out, BURGERS_PLAN_AUTO, ws, ws_bytes,
                            stream);                       // validates everything, zeroes iters_out
    if (st != BURGERS_OK) return st;
    if (newton_hybrid_fits(sizeof(T) == 8, N))       // snapshots written by the kernel: one launch
        return launch_newton<T>(u, B, N, grid_dx(N, L, bc), nu, dt, n_steps, bc, theta, tol, max_iter,
                                reinterpret_cast<long long *>(iters_out), BURGERS_PLAN_HYBRID, (T *)ws, (cudaStream_t)stream,
                                true, snaps, snap_every);
    int64_t done = 0, k = 0;
    while (done < n_steps) {
        const int64_t chunk = (n_steps - done < snap_every) ? n_steps - done : snap_every;
        st = newton_call<T>(u, B, N, L, nu, dt, chunk, bc, theta, tol, max_iter, iters_out, BURGERS_PLAN_AUTO, ws, ws_bytes,
                            stream, true);
        if (st != BURGERS_OK) return st;
        done += chunk;
        if (chunk == snap_every) {
            if (cudaMemcpyAsync(snaps + k * B * N, u, (size_t)B * (size_t)N * sizeof(T), cudaMemcpyDeviceToDevice,
                                (cudaStream_t)stream) != cudaSuccess)
                return BURGERS_ERR_CUDA;
            ++k;
        }
    }
    return BURGERS_OK;
}

// Reverse mode of the Newton / theta-scheme (D16): the checkpointed sweep above with newton_traj_call forward and the
// backward kernels of adjoint_newton.cu.
template <typename T>
int newton_adjoint_call(const T *u0, T *lam, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps,
                        int bc, double theta, double tol, int max_iter, int64_t segment, void *ws, size_t ws_bytes,
                        void *stream) {
    if (!lam) return BURGERS_ERR_NULL;
    int st = check_common(u0, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (!(tol >= 0.0) || max_iter < 0 || !(theta >= 0.0 && theta <= 1.0)) return BURGERS_ERR_VALUE;
    cudaStream_t s = (cudaStream_t)stream;
    const double dx = grid_dx(N, L, bc);
    return implicit_adjoint_sweep<T>(
        u0, B, N, bc, n_steps, segment, BURGERS_OP_NEWTON, ws, ws_bytes, s,
        [&](T *work, int64_t steps, T *snaps, int64_t every, void *ows, size_t ows_bytes) {
            return newton_traj_call<T>(work, B, N, L, nu, dt, steps, bc, theta, tol, max_iter, nullptr, every, snaps, ows,
                                       ows_bytes, stream);
        },
        [&](const T *start, const T *states, T *scratch, int64_t len) {
            return launch_adjoint_newton_steps<T>(start, states, lam, scratch, B, N, dx, nu, dt, len, bc, theta, s);
        });
}

template <typename T>
int cfl_call(const T *u, int64_t B, int64_t N, double L, const T *nu, double C, int bc, T *dt_out,
             void *stream) {
    if (!u || !nu || !dt_out) return BURGERS_ERR_NULL;
    if (B < 1 || N < 3) return BURGERS_ERR_SHAPE;
    if (bc != BURGERS_BC_PERIODIC && bc != BURGERS_BC_DIRICHLET) return BURGERS_ERR_ENUM;
    if (!(L > 0.0) || !std::isfinite(L) || !(C > 0.0) || !std::isfinite(C)) return BURGERS_ERR_VALUE;
    return launch_cfl<T>(u, B, N, grid_dx(N, L, bc), nu, C, dt_out, (cudaStream_t)stream);
}

// ---- host-buffer path: allocate, copy in, run the device path, copy out, free ---------------
// Stream-ordered allocations from a memory pool the library owns (one per device, created by the first
// host-buffer call).  Freed blocks stay in that pool up to kHostPoolKeepBytes, so that a sequence of host
// calls does not map and unmap device memory every time: with the device's default pool, whose release
// threshold is 0, everything goes back to the driver at the next synchronisation and C2 fp32 end to end
// took 11.9 to 19.8 ms from call to call; now 11.6 to 12.0.  The default pool is not touched.
constexpr uint64_t kHostPoolKeepBytes = (uint64_t)1 << 30;

cudaMemPool_t host_pool() {
    static std::mutex mu;
    static cudaMemPool_t pools[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lk(mu);
    if (!pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        uint64_t keep = kHostPoolKeepBytes;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        pools[dev] = pool;
    }
    return pools[dev];
}

struct DevBuf {
    void *p = nullptr;
    ~DevBuf() { if (p) cudaFreeAsync(p, nullptr); }
    bool alloc(size_t bytes) {
        if (bytes == 0) return true;
        cudaMemPool_t pool = host_pool();
        const cudaError_t e = pool ? cudaMallocFromPoolAsync(&p, bytes, pool, nullptr) : cudaMallocAsync(&p, bytes, nullptr);
        if (e != cudaSuccess) { cudaGetLastError(); p = nullptr; return false; }
        return true;
    }
};

template <typename T, typename F>
int host_step(T *u, int64_t B, int64_t N, const T *nu, const T *dt, size_t ws_bytes, F run) {
    const size_t ub = (size_t)B * (size_t)N * sizeof(T), vb = (size_t)B * sizeof(T);
    DevBuf du, dnu, ddt, dws;
    if (!du.alloc(ub) || !dnu.alloc(vb) || !ddt.alloc(vb) || !dws.alloc(ws_bytes)) return BURGERS_ERR_CUDA;
    cudaStream_t s = nullptr;
    if (cudaMemcpyAsync(du.p, u, ub, cudaMemcpyHostToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    if (cudaMemcpyAsync(dnu.p, nu, vb, cudaMemcpyHostToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    if (cudaMemcpyAsync(ddt.p, dt, vb, cudaMemcpyHostToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    int st = run((T *)du.p, (const T *)dnu.p, (const T *)ddt.p, dws.p);
    if (st != BURGERS_OK) { cudaStreamSynchronize(s); return st; }
    if (cudaMemcpyAsync(u, du.p, ub, cudaMemcpyDeviceToHost, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    return cuda_status(cudaStreamSynchronize(s));
}

template <typename T>
int explicit_host(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps,
                  int bc, int scheme) {
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (!scheme_ok(scheme)) return BURGERS_ERR_ENUM;
    const size_t wsb = burgers_workspace_bytes(BURGERS_OP_EXPLICIT, sizeof(T) == 8, B, N, bc, scheme,
                                               BURGERS_PLAN_AUTO);
    return host_step<T>(u, B, N, nu, dt, wsb, [&](T *du, const T *dnu, const T *ddt, void *ws) {
        return explicit_call<T>(du, B, N, L, dnu, ddt, n_steps, bc, scheme, BURGERS_PLAN_AUTO, 0, 0, ws,
                                wsb, nullptr);
    });
}

template <typename T>
int btcs_host(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc) {
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    const size_t wsb = burgers_workspace_bytes(BURGERS_OP_BTCS, sizeof(T) == 8, B, N, bc, 0,
                                               BURGERS_PLAN_AUTO);
    return host_step<T>(u, B, N, nu, dt, wsb, [&](T *du, const T *dnu, const T *ddt, void *ws) {
        return btcs_call<T>(du, B, N, L, dnu, ddt, n_steps, bc, BURGERS_PLAN_AUTO, ws, wsb, nullptr);
    });
}

template <typename T>
int newton_host(T *u, int64_t B, int64_t N, double L, const T *nu, const T *dt, int64_t n_steps, int bc,
                double theta, double tol, int max_iter, int64_t *iters_out) {
    int st = check_common(u, nu, dt, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (!(tol >= 0.0) || max_iter < 0 || !(theta >= 0.0 && theta <= 1.0)) return BURGERS_ERR_VALUE;
    const size_t wsb = burgers_workspace_bytes(BURGERS_OP_NEWTON, sizeof(T) == 8, B, N, bc, 0, BURGERS_PLAN_AUTO);
    DevBuf dit;
    if (iters_out && !dit.alloc((size_t)B * sizeof(int64_t))) return BURGERS_ERR_CUDA;
    st = host_step<T>(u, B, N, nu, dt, wsb, [&](T *du, const T *dnu, const T *ddt, void *ws) {
        return newton_call<T>(du, B, N, L, dnu, ddt, n_steps, bc, theta, tol, max_iter, (int64_t *)dit.p, BURGERS_PLAN_AUTO,
                              ws, wsb, nullptr);
    });
    if (st != BURGERS_OK || !iters_out) return st;
    return cuda_status(cudaMemcpy(iters_out, dit.p, (size_t)B * sizeof(int64_t), cudaMemcpyDeviceToHost));
}

template <typename T>
int cfl_host(const T *u, int64_t B, int64_t N, double L, const T *nu, double C, int bc, T *dt_out) {
    if (!u || !nu || !dt_out) return BURGERS_ERR_NULL;
    if (B < 1 || N < 3) return BURGERS_ERR_SHAPE;
    const size_t ub = (size_t)B * (size_t)N * sizeof(T), vb = (size_t)B * sizeof(T);
    DevBuf du, dnu, ddt;
    if (!du.alloc(ub) || !dnu.alloc(vb) || !ddt.alloc(vb)) return BURGERS_ERR_CUDA;
    cudaStream_t s = nullptr;
    if (cudaMemcpyAsync(du.p, u, ub, cudaMemcpyHostToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    if (cudaMemcpyAsync(dnu.p, nu, vb, cudaMemcpyHostToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    int st = cfl_call<T>((const T *)du.p, B, N, L, (const T *)dnu.p, C, bc, (T *)ddt.p, nullptr);
    if (st != BURGERS_OK) { cudaStreamSynchronize(s); return st; }
    if (cudaMemcpyAsync(dt_out, ddt.p, vb, cudaMemcpyDeviceToHost, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    return cuda_status(cudaStreamSynchronize(s));
}

// Streams of the pipelined host path: one pair per device, created by the first call that uses them.
// Blocking streams: they are ordered against the legacy default stream, on which the stream-ordered
// allocations above are made and freed.
struct HostPipe {
    static constexpr int K = 2;
    cudaStream_t s[K] = {};
    bool ok = false;
};
HostPipe &host_pipe() {
    static std::mutex mu;
    static HostPipe pipes[64];
    static HostPipe none;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return none;
    std::lock_guard<std::mutex> lk(mu);
    HostPipe &p = pipes[dev];
    if (!p.ok) {
        bool ok = true;
        for (int i = 0; i < HostPipe::K; ++i) ok = ok && (cudaStreamCreate(&p.s[i]) == cudaSuccess);
        if (!ok) { cudaGetLastError(); return none; }
        p.ok = true;
    }
    return p;
}

// The whole hot path on host buffers with ONE upload of the state: dt_from_cfl on the device, the
// time-stepping call with that dt, one download (8(a): CFL step + time stepping).  Batches whose plan
// needs no workspace (RESIDENT, HYBRID: trajectories independent, one CTA each) go through as
// HostPipe::K = 2 halves, each on its own stream: the upload of the second half overlaps the kernels of
// the first, the download of the first those of the second, and the CTAs of the two launches fill the SMs
// as those of one launch would.  The plan is resolved once for the whole shape, so halving cannot change a
// bit.  Measured, C2 fp32: 11.73 -> 11.15 ms (10.29 ms of kernels; 3 or 4 chunks, or uneven ones: the
// same; 8 chunks: 12.5).
template <typename T>
int solve_host(T *u, int64_t B, int64_t N, double L, const T *nu, double C, int64_t n_steps, int bc, int op,
               int scheme, T *dt_out) {
    int st = check_common(u, nu, u, B, N, L, n_steps, bc);
    if (st != BURGERS_OK) return st;
    if (op != BURGERS_OP_EXPLICIT && op != BURGERS_OP_BTCS) return BURGERS_ERR_ENUM;
    if (op == BURGERS_OP_EXPLICIT && !scheme_ok(scheme)) return BURGERS_ERR_ENUM;
    if (!(C > 0.0) || !std::isfinite(C)) return BURGERS_ERR_VALUE;
    const int is_f64 = sizeof(T) == 8;
    const int plan = burgers_plan_query(op, is_f64, B, N, bc, scheme);
    if (plan < 0) return plan;
    const size_t wsb = burgers_workspace_bytes(op, is_f64, B, N, bc, scheme, plan);
    const size_t ub = (size_t)B * (size_t)N * sizeof(T), vb = (size_t)B * sizeof(T);
    DevBuf du, dnu, ddt, dws;
    if (!du.alloc(ub) || !dnu.alloc(vb) || !ddt.alloc(vb) || !dws.alloc(wsb)) return BURGERS_ERR_CUDA;
    T *const pu = (T *)du.p, *const pnu = (T *)dnu.p, *const pdt = (T *)ddt.p;
    // rows [b0, b0 + nb) on stream s: upload, CFL step, time stepping, download
    auto run = [&](int64_t b0, int64_t nb, cudaStream_t s) -> int {
        const size_t cu = (size_t)nb * (size_t)N * sizeof(T), cv = (size_t)nb * sizeof(T);
        T *const cu_d = pu + b0 * N;
        if (cudaMemcpyAsync(cu_d, u + b0 * N, cu, cudaMemcpyHostToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
        if (cudaMemcpyAsync(pnu + b0, nu + b0, cv, cudaMemcpyHostToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
        int r = cfl_call<T>(cu_d, nb, N, L, pnu + b0, C, bc, pdt + b0, s);
        if (r != BURGERS_OK) return r;
        r = (op == BURGERS_OP_EXPLICIT)
                ? explicit_call<T>(cu_d, nb, N, L, pnu + b0, pdt + b0, n_steps, bc, scheme, plan, 0, 0, dws.p, wsb, s)
                : btcs_call<T>(cu_d, nb, N, L, pnu + b0, pdt + b0, n_steps, bc, plan, dws.p, wsb, s);
        if (r != BURGERS_OK) return r;
        if (cudaMemcpyAsync(u + b0 * N, cu_d, cu, cudaMemcpyDeviceToHost, s) != cudaSuccess) return BURGERS_ERR_CUDA;
        if (dt_out && cudaMemcpyAsync(dt_out + b0, pdt + b0, cv, cudaMemcpyDeviceToHost, s) != cudaSuccess)
            return BURGERS_ERR_CUDA;
        return BURGERS_OK;
    };
    const bool chunked = wsb == 0 && B >= 2 * HostPipe::K && ub >= ((size_t)8 << 20) &&
                         (plan == BURGERS_PLAN_RESIDENT || plan == BURGERS_PLAN_HYBRID) && host_pipe().ok;
    if (!chunked) {
        st = run(0, B, nullptr);
        const int sy = cuda_status(cudaStreamSynchronize(nullptr));
        return st != BURGERS_OK ? st : sy;
    }
    HostPipe &hp = host_pipe();
    for (int i = 0; i < HostPipe::K && st == BURGERS_OK; ++i) {
        const int64_t b0 = B * i / HostPipe::K, b1 = B * (i + 1) / HostPipe::K;
        st = run(b0, b1 - b0, hp.s[i]);
    }
    int sy = BURGERS_OK;
    for (int i = 0; i < HostPipe::K; ++i) {
        const int r = cuda_status(cudaStreamSynchronize(hp.s[i]));
        if (r != BURGERS_OK) sy = r;
    }
    return st != BURGERS_OK ? st : sy;
}

}  // namespace

extern "C" {

int burgers_explicit_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                         int64_t n_steps, int bc, int scheme, void *ws, size_t ws_bytes, void *stream) {
    return explicit_call<float>(u, B, N, L, nu, dt, n_steps, bc, scheme, BURGERS_PLAN_AUTO, 0, 0, ws, ws_bytes, stream);
}
int burgers_explicit_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                         int64_t n_steps, int bc, int scheme, void *ws, size_t ws_bytes, void *stream) {
    return explicit_call<double>(u, B, N, L, nu, dt, n_steps, bc, scheme, BURGERS_PLAN_AUTO, 0, 0, ws, ws_bytes, stream);
}
int burgers_explicit_plan_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                              int64_t n_steps, int bc, int scheme, int plan, int tblock, int ppt,
                              void *ws, size_t ws_bytes, void *stream) {
    return explicit_call<float>(u, B, N, L, nu, dt, n_steps, bc, scheme, plan, tblock, ppt, ws, ws_bytes, stream);
}
int burgers_explicit_plan_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                              const double *dt, int64_t n_steps, int bc, int scheme, int plan,
                              int tblock, int ppt, void *ws, size_t ws_bytes, void *stream) {
    return explicit_call<double>(u, B, N, L, nu, dt, n_steps, bc, scheme, plan, tblock, ppt, ws, ws_bytes, stream);
}

int burgers_explicit_traj_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                              int64_t n_steps, int bc, int scheme, int64_t snap_every, float *snaps,
                              void *ws, size_t ws_bytes, void *stream) {
    if (!snaps) return BURGERS_ERR_NULL;
    if (snap_every < 1) return BURGERS_ERR_SHAPE;
    return explicit_call<float>(u, B, N, L, nu, dt, n_steps, bc, scheme, BURGERS_PLAN_AUTO, 0, 0, ws, ws_bytes, stream,
                                snaps, snap_every);
}
int burgers_explicit_traj_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                              int64_t n_steps, int bc, int scheme, int64_t snap_every, double *snaps,
                              void *ws, size_t ws_bytes, void *stream) {
    if (!snaps) return BURGERS_ERR_NULL;
    if (snap_every < 1) return BURGERS_ERR_SHAPE;
    return explicit_call<double>(u, B, N, L, nu, dt, n_steps, bc, scheme, BURGERS_PLAN_AUTO, 0, 0, ws, ws_bytes, stream,
                                 snaps, snap_every);
}

int burgers_explicit_adaptive_f32(float *u, int64_t B, int64_t N, double L, const float *nu, double C,
                                  int64_t n_outer, int64_t m_steps, int bc, int scheme, float *dt_scratch,
                                  double *t_out, void *ws, size_t ws_bytes, void *stream) {
    return adaptive_call<float>(u, B, N, L, nu, C, n_outer, m_steps, bc, scheme, dt_scratch, t_out, ws, ws_bytes, stream);
}
int burgers_explicit_adaptive_f64(double *u, int64_t B, int64_t N, double L, const double *nu, double C,
                                  int64_t n_outer, int64_t m_steps, int bc, int scheme, double *dt_scratch,
                                  double *t_out, void *ws, size_t ws_bytes, void *stream) {
    return adaptive_call<double>(u, B, N, L, nu, C, n_outer, m_steps, bc, scheme, dt_scratch, t_out, ws, ws_bytes, stream);
}

int burgers_explicit_adjoint_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                                 const float *dt, int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream) {
    return adjoint_call<float>(u0, lam, B, N, L, nu, dt, n_steps, bc, 0, ws, ws_bytes, stream);
}
int burgers_explicit_adjoint_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                                 const double *dt, int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream) {
    return adjoint_call<double>(u0, lam, B, N, L, nu, dt, n_steps, bc, 0, ws, ws_bytes, stream);
}
int burgers_explicit_adjoint_ckpt_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                                      const float *dt, int64_t n_steps, int bc, int64_t segment, void *ws,
                                      size_t ws_bytes, void *stream) {
    return adjoint_call<float>(u0, lam, B, N, L, nu, dt, n_steps, bc, segment, ws, ws_bytes, stream);
}
int burgers_explicit_adjoint_ckpt_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                                      const double *dt, int64_t n_steps, int bc, int64_t segment, void *ws,
                                      size_t ws_bytes, void *stream) {
    return adjoint_call<double>(u0, lam, B, N, L, nu, dt, n_steps, bc, segment, ws, ws_bytes, stream);
}
size_t burgers_adjoint_ckpt_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps,
                                            int64_t segment) {
    return burgers_adjoint_scheme_workspace_bytes(dtype_is_f64, B, N, bc, BURGERS_SCHEME_EULER, n_steps, segment);
}
size_t burgers_adjoint_scheme_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int scheme, int64_t n_steps,
                                              int64_t segment) {
    if (B < 1 || N < 3 || n_steps < 0 || segment < 0 || !scheme_ok(scheme)) return 0;
    return dtype_is_f64 ? adjoint_ws_bytes<double>(B, N, bc, n_steps, segment, scheme)
                        : adjoint_ws_bytes<float>(B, N, bc, n_steps, segment, scheme);
}
int burgers_explicit_adjoint_scheme_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                                        const float *dt, int64_t n_steps, int bc, int scheme, int64_t segment, void *ws,
                                        size_t ws_bytes, void *stream) {
    return adjoint_call<float>(u0, lam, B, N, L, nu, dt, n_steps, bc, segment, ws, ws_bytes, stream, scheme);
}
int burgers_explicit_adjoint_scheme_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                                        const double *dt, int64_t n_steps, int bc, int scheme, int64_t segment, void *ws,
                                        size_t ws_bytes, void *stream) {
    return adjoint_call<double>(u0, lam, B, N, L, nu, dt, n_steps, bc, segment, ws, ws_bytes, stream, scheme);
}
size_t burgers_adjoint_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps) {
    return burgers_adjoint_ckpt_workspace_bytes(dtype_is_f64, B, N, bc, n_steps, 0);
}

int burgers_btcs_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                     int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream) {
    return btcs_call<float>(u, B, N, L, nu, dt, n_steps, bc, BURGERS_PLAN_AUTO, ws, ws_bytes, stream);
}
int burgers_btcs_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                     int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream) {
    return btcs_call<double>(u, B, N, L, nu, dt, n_steps, bc, BURGERS_PLAN_AUTO, ws, ws_bytes, stream);
}
int burgers_btcs_plan_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                          int64_t n_steps, int bc, int plan, void *ws, size_t ws_bytes, void *stream) {
    return btcs_call<float>(u, B, N, L, nu, dt, n_steps, bc, plan, ws, ws_bytes, stream);
}
int burgers_btcs_plan_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                          int64_t n_steps, int bc, int plan, void *ws, size_t ws_bytes, void *stream) {
    return btcs_call<double>(u, B, N, L, nu, dt, n_steps, bc, plan, ws, ws_bytes, stream);
}

int burgers_btcs_traj_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                          int64_t n_steps, int bc, int64_t snap_every, float *snaps, void *ws, size_t ws_bytes,
                          void *stream) {
    return btcs_traj_call<float>(u, B, N, L, nu, dt, n_steps, bc, snap_every, snaps, ws, ws_bytes, stream);
}
int burgers_btcs_traj_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                          int64_t n_steps, int bc, int64_t snap_every, double *snaps, void *ws, size_t ws_bytes,
                          void *stream) {
    return btcs_traj_call<double>(u, B, N, L, nu, dt, n_steps, bc, snap_every, snaps, ws, ws_bytes, stream);
}

int burgers_btcs_adjoint_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                             int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream) {
    return btcs_adjoint_call<float>(u0, lam, B, N, L, nu, dt, n_steps, bc, 0, ws, ws_bytes, stream);
}
int burgers_btcs_adjoint_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                             const double *dt, int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream) {
    return btcs_adjoint_call<double>(u0, lam, B, N, L, nu, dt, n_steps, bc, 0, ws, ws_bytes, stream);
}
size_t burgers_btcs_adjoint_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps) {
    return burgers_implicit_adjoint_ckpt_workspace_bytes(BURGERS_OP_BTCS, dtype_is_f64, B, N, bc, n_steps, 0);
}
int burgers_btcs_adjoint_ckpt_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                                  const float *dt, int64_t n_steps, int bc, int64_t segment, void *ws, size_t ws_bytes,
                                  void *stream) {
    return btcs_adjoint_call<float>(u0, lam, B, N, L, nu, dt, n_steps, bc, segment, ws, ws_bytes, stream);
}
int burgers_btcs_adjoint_ckpt_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                                  const double *dt, int64_t n_steps, int bc, int64_t segment, void *ws, size_t ws_bytes,
                                  void *stream) {
    return btcs_adjoint_call<double>(u0, lam, B, N, L, nu, dt, n_steps, bc, segment, ws, ws_bytes, stream);
}
size_t burgers_implicit_adjoint_ckpt_workspace_bytes(int op, int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps,
                                                     int64_t segment) {
    if (B < 1 || N < 3 || n_steps < 0 || segment < 0) return 0;
    if (op != BURGERS_OP_BTCS && op != BURGERS_OP_NEWTON) return 0;
    return dtype_is_f64 ? implicit_adjoint_ws_bytes<double>(B, N, bc, n_steps, segment, op)
                        : implicit_adjoint_ws_bytes<float>(B, N, bc, n_steps, segment, op);
}

int burgers_newton_adjoint_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                               int64_t n_steps, int bc, double theta, double tol, int max_iter, void *ws, size_t ws_bytes,
                               void *stream) {
    return newton_adjoint_call<float>(u0, lam, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, 0, ws, ws_bytes, stream);
}
int burgers_newton_adjoint_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                               const double *dt, int64_t n_steps, int bc, double theta, double tol, int max_iter, void *ws,
                               size_t ws_bytes, void *stream) {
    return newton_adjoint_call<double>(u0, lam, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, 0, ws, ws_bytes, stream);
}
size_t burgers_newton_adjoint_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps) {
    return burgers_implicit_adjoint_ckpt_workspace_bytes(BURGERS_OP_NEWTON, dtype_is_f64, B, N, bc, n_steps, 0);
}
int burgers_newton_adjoint_ckpt_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                                    const float *dt, int64_t n_steps, int bc, double theta, double tol, int max_iter,
                                    int64_t segment, void *ws, size_t ws_bytes, void *stream) {
    return newton_adjoint_call<float>(u0, lam, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, segment, ws, ws_bytes,
                                      stream);
}
int burgers_newton_adjoint_ckpt_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                                    const double *dt, int64_t n_steps, int bc, double theta, double tol, int max_iter,
                                    int64_t segment, void *ws, size_t ws_bytes, void *stream) {
    return newton_adjoint_call<double>(u0, lam, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, segment, ws, ws_bytes,
                                       stream);
}

int burgers_btcs_gs_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                        int64_t n_steps, int bc, double tol, int max_iter, int64_t *iters_out, void *ws,
                        size_t ws_bytes, void *stream) {
    return gs_call<float>(u, B, N, L, nu, dt, n_steps, bc, tol, max_iter, iters_out, ws, ws_bytes, stream);
}
int burgers_btcs_gs_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                        int64_t n_steps, int bc, double tol, int max_iter, int64_t *iters_out, void *ws,
                        size_t ws_bytes, void *stream) {
    return gs_call<double>(u, B, N, L, nu, dt, n_steps, bc, tol, max_iter, iters_out, ws, ws_bytes, stream);
}

int burgers_newton_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                       int64_t n_steps, int bc, double theta, double tol, int max_iter, int64_t *iters_out,
                       int plan, void *ws, size_t ws_bytes, void *stream) {
    return newton_call<float>(u, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, iters_out, plan, ws, ws_bytes, stream);
}
int burgers_newton_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                       int64_t n_steps, int bc, double theta, double tol, int max_iter, int64_t *iters_out,
                       int plan, void *ws, size_t ws_bytes, void *stream) {
    return newton_call<double>(u, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, iters_out, plan, ws, ws_bytes, stream);
}

int burgers_newton_traj_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt, int64_t n_steps,
                            int bc, double theta, double tol, int max_iter, int64_t *iters_out, int64_t snap_every,
                            float *snaps, void *ws, size_t ws_bytes, void *stream) {
    return newton_traj_call<float>(u, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, iters_out, snap_every, snaps, ws,
                                   ws_bytes, stream);
}
int burgers_newton_traj_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt, int64_t n_steps,
                            int bc, double theta, double tol, int max_iter, int64_t *iters_out, int64_t snap_every,
                            double *snaps, void *ws, size_t ws_bytes, void *stream) {
    return newton_traj_call<double>(u, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, iters_out, snap_every, snaps, ws,
                                    ws_bytes, stream);
}

int dt_from_cfl_f32(const float *u, int64_t B, int64_t N, double L, const float *nu, double C, int bc,
                    float *dt_out, void *stream) {
    return cfl_call<float>(u, B, N, L, nu, C, bc, dt_out, stream);
}
int dt_from_cfl_f64(const double *u, int64_t B, int64_t N, double L, const double *nu, double C, int bc,
                    double *dt_out, void *stream) {
    return cfl_call<double>(u, B, N, L, nu, C, bc, dt_out, stream);
}

int burgers_explicit_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                              int64_t n_steps, int bc, int scheme) {
    return explicit_host<float>(u, B, N, L, nu, dt, n_steps, bc, scheme);
}
int burgers_explicit_host_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                              const double *dt, int64_t n_steps, int bc, int scheme) {
    return explicit_host<double>(u, B, N, L, nu, dt, n_steps, bc, scheme);
}
int burgers_btcs_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                          int64_t n_steps, int bc) {
    return btcs_host<float>(u, B, N, L, nu, dt, n_steps, bc);
}
int burgers_btcs_host_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                          int64_t n_steps, int bc) {
    return btcs_host<double>(u, B, N, L, nu, dt, n_steps, bc);
}
int burgers_newton_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                            int64_t n_steps, int bc, double theta, double tol, int max_iter, int64_t *iters_out) {
    return newton_host<float>(u, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, iters_out);
}
int burgers_newton_host_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                            int64_t n_steps, int bc, double theta, double tol, int max_iter, int64_t *iters_out) {
    return newton_host<double>(u, B, N, L, nu, dt, n_steps, bc, theta, tol, max_iter, iters_out);
}
int burgers_solve_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu, double C, int64_t n_steps,
                           int bc, int op, int scheme, float *dt_out) {
    return solve_host<float>(u, B, N, L, nu, C, n_steps, bc, op, scheme, dt_out);
}
int burgers_solve_host_f64(double *u, int64_t B, int64_t N, double L, const double *nu, double C, int64_t n_steps,
                           int bc, int op, int scheme, double *dt_out) {
    return solve_host<double>(u, B, N, L, nu, C, n_steps, bc, op, scheme, dt_out);
}
int dt_from_cfl_host_f32(const float *u, int64_t B, int64_t N, double L, const float *nu, double C,
                         int bc, float *dt_out) {
    if (bc != BURGERS_BC_PERIODIC && bc != BURGERS_BC_DIRICHLET) return BURGERS_ERR_ENUM;
    if (!(L > 0.0) || !std::isfinite(L) || !(C > 0.0) || !std::isfinite(C)) return BURGERS_ERR_VALUE;
    return cfl_host<float>(u, B, N, L, nu, C, bc, dt_out);
}
int dt_from_cfl_host_f64(const double *u, int64_t B, int64_t N, double L, const double *nu, double C,
                         int bc, double *dt_out) {
    if (bc != BURGERS_BC_PERIODIC && bc != BURGERS_BC_DIRICHLET) return BURGERS_ERR_ENUM;
    if (!(L > 0.0) || !std::isfinite(L) || !(C > 0.0) || !std::isfinite(C)) return BURGERS_ERR_VALUE;
    return cfl_host<double>(u, B, N, L, nu, C, bc, dt_out);
}

size_t burgers_workspace_bytes(int op, int dtype_is_f64, int64_t B, int64_t N, int bc, int scheme,
                               int plan) {
    if (B < 1 || N < 3) return 0;
    const size_t esz = dtype_is_f64 ? 8 : 4;
    if (op == BURGERS_OP_EXPLICIT) {
        ExplicitGeom g;
        if (explicit_geometry(dtype_is_f64, B, N, bc, scheme, plan, 0, 0, &g) != BURGERS_OK) return 0;
        // TILED: the ping-pong buffer, + the three maximum slots of the adaptive call (a few bytes per trajectory)
        return g.plan == BURGERS_PLAN_TILED ? align_up((size_t)B * (size_t)N * esz, 256) + tiled_adapt_slot_bytes(B) : 0;
    }
    if (op == BURGERS_OP_NEWTON) {
        if (plan == BURGERS_PLAN_AUTO) plan = newton_hybrid_fits(dtype_is_f64, N) ? BURGERS_PLAN_HYBRID : BURGERS_PLAN_THOMAS;
        return plan == BURGERS_PLAN_THOMAS ? align_up(newton_thomas_ws_elems(B, N, bc) * esz, 256) : 0;
    }
    if (op == BURGERS_OP_GS) return align_up(btcs_gs_ws_elems(B, N) * esz, 256);
    if (op == BURGERS_OP_BTCS) {
        if (plan == BURGERS_PLAN_AUTO) plan = btcs_auto_plan(dtype_is_f64, B, N, bc);
        if (plan == BURGERS_PLAN_THOMAS) return align_up(btcs_thomas_ws_elems(B, N, bc) * esz, 256);
        if (plan == BURGERS_PLAN_LONG || plan == BURGERS_PLAN_LONG_GENERAL)
            return btcs_long_fits(dtype_is_f64, B, N, bc) ? align_up(btcs_long_ws_bytes((int)esz, B, N), 256) : 0;
        return 0;
    }
    return 0;
}

int burgers_plan_query(int op, int dtype_is_f64, int64_t B, int64_t N, int bc, int scheme) {
    if (B < 1 || N < 3) return BURGERS_ERR_SHAPE;
    if (op == BURGERS_OP_EXPLICIT) {
        ExplicitGeom g;
        int st = explicit_geometry(dtype_is_f64, B, N, bc, scheme, BURGERS_PLAN_AUTO, 0, 0, &g);
        return st == BURGERS_OK ? g.plan : st;
    }
    if (op == BURGERS_OP_BTCS) return btcs_auto_plan(dtype_is_f64, B, N, bc);
    if (op == BURGERS_OP_NEWTON) return newton_hybrid_fits(dtype_is_f64, N) ? BURGERS_PLAN_HYBRID : BURGERS_PLAN_THOMAS;
    if (op == BURGERS_OP_GS) return BURGERS_PLAN_THOMAS;
    if (op == BURGERS_OP_CFL) return BURGERS_PLAN_AUTO;
    return BURGERS_ERR_ENUM;
}

int64_t burgers_launch_count(int op, int dtype_is_f64, int64_t B, int64_t N, int bc, int scheme,
                             int plan, int tblock, int64_t n_steps) {
    if (B < 1 || N < 3 || n_steps < 0) return 0;
    if (op == BURGERS_OP_CFL) return cfl_launch_count(dtype_is_f64, B, N);
    if (n_steps == 0) return 0;
    if (op == BURGERS_OP_EXPLICIT) {
        ExplicitGeom g;
        if (explicit_geometry(dtype_is_f64, B, N, bc, scheme, plan, tblock, 0, &g) != BURGERS_OK) return 0;
        return g.plan == BURGERS_PLAN_RESIDENT ? 1 : (n_steps + g.tblock - 1) / g.tblock;
    }
    if (op == BURGERS_OP_NEWTON) {
        if (plan == BURGERS_PLAN_AUTO) plan = newton_hybrid_fits(dtype_is_f64, N) ? BURGERS_PLAN_HYBRID : BURGERS_PLAN_THOMAS;
        return plan == BURGERS_PLAN_HYBRID ? 1 : 3;
    }
    if (op == BURGERS_OP_GS) return 3;
    if (op == BURGERS_OP_BTCS) {
        if (plan == BURGERS_PLAN_AUTO) plan = btcs_auto_plan(dtype_is_f64, B, N, bc);
        if (plan == BURGERS_PLAN_THOMAS) return btcs_thomas_launch_count(n_steps);
        if (plan == BURGERS_PLAN_HYBRID) return 1;
        if (plan == BURGERS_PLAN_LONG || plan == BURGERS_PLAN_LONG_GENERAL)
            return btcs_long_launch_count(B, N, n_steps, plan == BURGERS_PLAN_LONG_GENERAL);
    }
    return 0;
}

const char *burgers_strerror(int status) {
    switch (status) {
        case BURGERS_OK: return "ok";
        case BURGERS_ERR_NULL: return "null pointer argument";
        case BURGERS_ERR_SHAPE: return "bad shape (need B>=1, N>=3, n_steps>=0, grid within limits)";
        case BURGERS_ERR_ENUM: return "unknown bc / scheme / plan / op";
        case BURGERS_ERR_VALUE: return "bad value (need finite L>0, C>0, tol>=0, max_iter>=0, 0<=theta<=1)";
        case BURGERS_ERR_WORKSPACE: return "workspace missing or too small (see burgers_workspace_bytes)";
        case BURGERS_ERR_CUDA: return "CUDA runtime / launch failure";
        case BURGERS_ERR_PLAN: return "requested plan cannot run this shape";
        case BURGERS_ERR_LIMIT: return "problem needs more scratch than the no-allocation entry point holds (see burgers_noalloc_scratch_bytes)";
    }
    return "unknown status";
}

int burgers_version(void) { return BURGERS_VERSION; }

}  // extern "C"
