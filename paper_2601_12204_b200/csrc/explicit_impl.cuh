// explicit_impl.cuh -- kernel (1): explicit time stepping (forward Euler PAPER.md:216 Eq.21,
// classical RK4 PAPER.md:224-229 Eq.22) of the upwind/central semi-discrete operator
// (Eq.3-4, upwind rule :89).
//
// One kernel template serves two plans:
//   RESIDENT  one CTA owns a whole trajectory: it is loaded once, all n_steps run on chip,
//             it is stored once.  HBM traffic 2*sizeof(T)*N per trajectory per CALL.
//   TILED     one CTA owns an overlapped tile of a (long) trajectory and advances it `tblock`
//             steps per HBM round trip (temporal blocking): the tile is loaded with a halo of
//             tblock*radius points per side, its edges are left open (the invalid front moves
//             inwards `radius` points per step) and only the still-valid centre is stored.
// Data layout on chip: thread t holds P CONSECUTIVE grid points in registers, so every stencil
// neighbour but two is a register of the same thread; the two halo values come from the
// neighbouring threads by warp shuffle (CTA of one warp) or through a double-buffered shared
// memory edge array with ONE barrier per exchange (several warps).
//
// Arithmetic per point (D2, scaled by dt): with hcx = dt/(2 dx), rr = nu dt/dx^2 and l/c/r the
// left, centre and right values, the sign-switched upwind difference of PAPER.md:89 is written in
// its branch-free "central difference + numerical diffusion" form
//   u_i g_i = u_i (u_{i+1} - u_{i-1})/2 - |u_i| (u_{i+1} - 2u_i + u_{i-1})/2     (either sign of u_i)
// so that
//   dt*F = (rr + hcx*|c|) * (l + r - 2c) - hcx*c*(r - l)
// which is 7 FMA-pipe instructions and no compare/select (the select form costs 7 + 2): the
// kernels are issue-bound, so instructions per update are what matters.
// It equals D2 up to rounding, keeps constants exactly fixed and keeps odd symmetry exact.
// fp32 Euler carries the state as base + s (two fp32 terms; increments are accumulated into the
// small term s, so they are not lost against ulp(u)) -- the stencil reads the
// rounded sum v = fl(base + s).
#pragma once
#include "common.cuh"

namespace burgers {
namespace expl {

template <typename T>
struct Params {
    const T *src;     // [B][N]
    T *dst;           // [B][N]   (== src for RESIDENT)
    const T *nu;      // [B]
    const T *dt;      // [B]
    int64_t N;
    double inv_dx;
    int64_t steps;    // steps in this launch
    int nth;          // active threads per CTA
    int bc;
    int halo;         // TILED: halo points per side
    int64_t W;        // TILED: valid outputs per tile
    int64_t tiles;    // TILED: tiles per trajectory
};

template <typename T> __device__ __forceinline__ T t_abs(T x);
template <> __device__ __forceinline__ float t_abs<float>(float x) { return fabsf(x); }
template <> __device__ __forceinline__ double t_abs<double>(double x) { return fabs(x); }
template <typename T> __device__ __forceinline__ T t_fma(T a, T b, T c);
template <> __device__ __forceinline__ float t_fma<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <> __device__ __forceinline__ double t_fma<double>(double a, double b, double c) { return fma(a, b, c); }

// dt*F at one point (D2) added to `acc`:  acc + (rr + hcx|c|) lap - hcx c (r - l).  7 FP instructions.
template <typename T>
__device__ __forceinline__ T add_dtF(T acc, T l, T c, T r, T hcx, T rr) {
    const T lap = t_fma(T(-2), c, l + r);        // u_{i+1} - 2u_i + u_{i-1}   (Eq.4)
    const T k = t_fma(hcx, t_abs(c), rr);        // diffusion number + upwind numerical diffusion
    const T e = hcx * c;
    return t_fma(-e, r - l, t_fma(k, lap, acc));
}
template <typename T>
__device__ __forceinline__ T dtF(T l, T c, T r, T hcx, T rr) {
    const T lap = t_fma(T(-2), c, l + r);
    const T k = t_fma(hcx, t_abs(c), rr);
    const T e = hcx * c;
    return t_fma(-e, r - l, k * lap);
}

// Halo exchange: every thread publishes its first and last point and receives the last point
// of its left neighbour (tl) and the first point of its right neighbour (tr).
template <typename T, bool WARP>
__device__ __forceinline__ void exchange(T first, T last, T &left, T &right, int tl, int tr,
                                         T *edge, int &buf) {
    if (WARP) {
        left = __shfl_sync(0xffffffffu, last, tl);
        right = __shfl_sync(0xffffffffu, first, tr);
    } else {
        T *e = edge + buf * 2 * blockDim.x;
        e[threadIdx.x] = first;
        e[blockDim.x + threadIdx.x] = last;
        __syncthreads();
        left = e[blockDim.x + tl];
        right = e[tr];
        buf ^= 1;
    }
}

// Register budget -> launch bound.  State registers per thread: P points x words x arrays
// (fp32 Euler: base, s, v; other Euler: v; RK4: v, y, acc) plus ~40 for addressing/temporaries.
constexpr int max_threads_for(int bytes, int P, int scheme) {
    int arrays = (scheme == BURGERS_SCHEME_RK4) ? 3 : (bytes == 4 ? 3 : 1);
    int regs = P * (bytes / 4) * arrays + 40;
    int t = 1024;
    while (t > 32 && t * regs > 65536) t /= 2;
    return t;
}

template <typename T, int P, int SCHEME, bool TILED, bool WARP>
__global__ void __launch_bounds__(WARP ? 32 : max_threads_for(sizeof(T), P, SCHEME))
explicit_kernel(const Params<T> p) {
    constexpr bool SPLIT = (sizeof(T) == 4) && (SCHEME == BURGERS_SCHEME_EULER);
    constexpr int V = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *edge = reinterpret_cast<T *>(smem_raw);

    const int t = threadIdx.x;
    const int nth = p.nth;
    const int64_t N = p.N;
    const int64_t b = TILED ? (int64_t)(blockIdx.x / p.tiles) : (int64_t)blockIdx.x;
    const int64_t tile = TILED ? (int64_t)(blockIdx.x % p.tiles) : 0;
    const bool active = t < nth;
    const bool dirichlet = (p.bc == BURGERS_BC_DIRICHLET);
    // global index of this thread's first point (may be <0 or >=N in TILED halos)
    const int64_t g0 = (TILED ? tile * p.W - p.halo : 0) + (int64_t)t * P;
    const T *srow = p.src + b * N;
    T *drow = p.dst + b * N;

    // per-trajectory constants, evaluated in fp64 and rounded once
    const double dtb = (double)p.dt[b];
    const T hcx = (T)(0.5 * dtb * p.inv_dx);
    const T rr = (T)((double)p.nu[b] * dtb * p.inv_dx * p.inv_dx);

    // ---------------- load
    T v[P];
#pragma unroll
    for (int j = 0; j < P; ++j) v[j] = T(0);
    const bool vec_ok = (P % V == 0) && (N % V == 0) && (!TILED || (p.halo % V == 0 && p.W % V == 0));
    if (active) {
        if (vec_ok) {
#pragma unroll
            for (int c = 0; c < P / V; ++c) {
                int64_t g = g0 + c * V;
                bool inside = true;
                if (TILED) {
                    if (dirichlet) inside = (g >= 0 && g < N);
                    else { g %= N; if (g < 0) g += N; }
                }
                if (inside) {
                    int4 q = *reinterpret_cast<const int4 *>(srow + g);
                    const T *e = reinterpret_cast<const T *>(&q);
#pragma unroll
                    for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < P; ++j) {
                int64_t g = g0 + j;
                bool inside = true;
                if (TILED) {
                    if (dirichlet) inside = (g >= 0 && g < N);
                    else { g %= N; if (g < 0) g += N; }
                }
                if (inside) v[j] = srow[g];
            }
        }
    }

    // neighbours for the halo exchange; open edges (TILED) read their own value: garbage that
    // never reaches the stored centre.
    const int last_t = nth - 1;
    int tl = (t == 0) ? (TILED ? 0 : last_t) : t - 1;
    int tr = (t >= last_t) ? (TILED ? last_t : 0) : t + 1;
    if (!active) { tl = 0; tr = 0; }
    // Dirichlet: node 0 and node N-1 never move.  The host guarantees they sit at j = 0 and
    // j = P-1 of their thread (N % P == 0, tile origin % P == 0).
    const bool fixL = dirichlet && (g0 == 0);
    const bool fixR = dirichlet && (g0 + P - 1 == N - 1);
    int buf = 0;
    T left, right;

    if (SCHEME == BURGERS_SCHEME_EULER) {
        T base[SPLIT ? P : 1], s[SPLIT ? P : 1];
        if (SPLIT) {
#pragma unroll
            for (int j = 0; j < P; ++j) { base[j] = v[j]; s[j] = T(0); }
        }
        for (int64_t n = 0; n < p.steps; ++n) {
            exchange<T, WARP>(v[0], v[P - 1], left, right, tl, tr, edge, buf);
            T l = left;
#pragma unroll
            for (int j = 0; j < P; ++j) {
                const T c = v[j];
                const T r = (j + 1 < P) ? v[j + 1] : right;
                const bool frozen = (j == 0 && fixL) || (j == P - 1 && fixR);
                if (SPLIT) {
                    const T sn = add_dtF<T>(s[j], l, c, r, hcx, rr);
                    s[j] = frozen ? s[j] : sn;
                    v[j] = base[j] + s[j];
                } else {
                    const T vn = add_dtF<T>(c, l, c, r, hcx, rr);
                    v[j] = frozen ? c : vn;
                }
                l = c;
            }
            if (SPLIT && (n & 63) == 63) {  // renormalise: base <- fl(base+s), s <- exact remainder
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    const T nb = v[j];
                    s[j] = (base[j] - nb) + s[j];
                    base[j] = nb;
                }
            }
        }
    } else {  // classical RK4; K_s = dt*F(y_s)
        T y[P], acc[P];
        for (int64_t n = 0; n < p.steps; ++n) {
#pragma unroll
            for (int stage = 0; stage < 4; ++stage) {
                if (stage == 0) exchange<T, WARP>(v[0], v[P - 1], left, right, tl, tr, edge, buf);
                else exchange<T, WARP>(y[0], y[P - 1], left, right, tl, tr, edge, buf);
                T l = left;
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    const T c = (stage == 0) ? v[j] : y[j];
                    const T r = (j + 1 < P) ? ((stage == 0) ? v[j + 1] : y[j + 1]) : right;
                    const bool frozen = (j == 0 && fixL) || (j == P - 1 && fixR);
                    T K = dtF<T>(l, c, r, hcx, rr);
                    K = frozen ? T(0) : K;
                    if (stage == 0) { acc[j] = K; y[j] = t_fma(T(0.5), K, v[j]); }
                    else if (stage == 1) { acc[j] = t_fma(T(2), K, acc[j]); y[j] = t_fma(T(0.5), K, v[j]); }
                    else if (stage == 2) { acc[j] = t_fma(T(2), K, acc[j]); y[j] = v[j] + K; }
                    else { acc[j] += K; v[j] = t_fma(acc[j], T(1.0 / 6.0), v[j]); }
                    l = c;
                }
            }
        }
    }

    // ---------------- store
    if (active) {
        if (vec_ok) {
#pragma unroll
            for (int c = 0; c < P / V; ++c) {
                int64_t g = g0 + c * V;
                bool ok = true;
                if (TILED) {
                    const int64_t li = (int64_t)t * P + c * V;  // local index in the tile
                    ok = (li >= p.halo) && (li < p.halo + p.W) && (g < N);
                }
                if (ok) {
                    int4 q;
                    T *e = reinterpret_cast<T *>(&q);
#pragma unroll
                    for (int k = 0; k < V; ++k) e[k] = v[c * V + k];
                    *reinterpret_cast<int4 *>(drow + g) = q;
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < P; ++j) {
                int64_t g = g0 + j;
                bool ok = true;
                if (TILED) {
                    const int64_t li = (int64_t)t * P + j;
                    ok = (li >= p.halo) && (li < p.halo + p.W) && (g < N);
                }
                if (ok) drow[g] = v[j];
            }
        }
    }
}

// ------------------------------------------------------------------ host side
template <typename T, int P, int SCHEME>
int launch_P(const Params<T> &p, const ExplicitGeom &g, int64_t B, cudaStream_t s) {
    const bool tiled = (g.plan == BURGERS_PLAN_TILED);
    const int64_t grid = tiled ? B * g.tiles : B;
    if (grid > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    const size_t smem = (size_t)4 * g.block * sizeof(T);
    if (tiled) {
        explicit_kernel<T, P, SCHEME, true, false><<<(unsigned)grid, g.block, smem, s>>>(p);
    } else if (g.block == 32) {
        explicit_kernel<T, P, SCHEME, false, true><<<(unsigned)grid, 32, 0, s>>>(p);
    } else {
        explicit_kernel<T, P, SCHEME, false, false><<<(unsigned)grid, g.block, smem, s>>>(p);
    }
    return last_launch_status();
}

template <typename T, int SCHEME>
int launch_scheme(const Params<T> &p, const ExplicitGeom &g, int64_t B, cudaStream_t s) {
    switch (g.P) {
        case 1: return launch_P<T, 1, SCHEME>(p, g, B, s);
        case 2: return launch_P<T, 2, SCHEME>(p, g, B, s);
        case 4: return launch_P<T, 4, SCHEME>(p, g, B, s);
        case 8: return launch_P<T, 8, SCHEME>(p, g, B, s);
        case 16: return launch_P<T, 16, SCHEME>(p, g, B, s);
        case 32: return launch_P<T, 32, SCHEME>(p, g, B, s);
    }
    return BURGERS_ERR_PLAN;
}

template <typename T>
int launch_explicit_impl(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                         int64_t n_steps, int bc, int scheme, const ExplicitGeom &g, T *ws,
                         cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    Params<T> p;
    p.nu = nu; p.dt = dt; p.N = N; p.inv_dx = 1.0 / dx; p.nth = g.nth; p.bc = bc;
    p.halo = g.halo; p.W = g.W; p.tiles = g.tiles;
    if (g.plan == BURGERS_PLAN_RESIDENT) {
        p.src = u; p.dst = u; p.steps = n_steps;
        return scheme == BURGERS_SCHEME_EULER ? launch_scheme<T, BURGERS_SCHEME_EULER>(p, g, B, s)
                                              : launch_scheme<T, BURGERS_SCHEME_RK4>(p, g, B, s);
    }
    // TILED: ping-pong between u and ws, tblock steps per launch; arrange the parity so that the
    // last launch writes u when possible, else copy back once.
    T *cur = u, *nxt = ws;
    int64_t done = 0;
    while (done < n_steps) {
        const int64_t k = (n_steps - done < g.tblock) ? n_steps - done : g.tblock;
        p.src = cur; p.dst = nxt; p.steps = k;
        int st = scheme == BURGERS_SCHEME_EULER ? launch_scheme<T, BURGERS_SCHEME_EULER>(p, g, B, s)
                                                : launch_scheme<T, BURGERS_SCHEME_RK4>(p, g, B, s);
        if (st != BURGERS_OK) return st;
        T *tmp = cur; cur = nxt; nxt = tmp;
        done += k;
    }
    if (cur != u) {
        if (cudaMemcpyAsync(u, cur, (size_t)B * N * sizeof(T), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
            return BURGERS_ERR_CUDA;
    }
    return BURGERS_OK;
}

}  // namespace expl
}  // namespace burgers
