// newton.cu -- SURVEY 8(f) NEXT-1: fully implicit BTCS with CENTRAL convection solved by
// Newton-Raphson, the implicit scheme the paper writes out (Eq.10-15).
//
// Per time step (D11), w = iterate for u^{n+1}, h = dt/(2 dx), r = nu dt/dx^2:
//   residual (Eq.11)   F_i = w_i - u_i^n + h w_i (w_{i+1} - w_{i-1}) - r (w_{i+1} - 2 w_i + w_{i-1})
//   Jacobian (Eq.14; Eq.15 is garbled -- reading Q5: the derivative of Eq.11)
//                      J_{i,i-1} = -h w_i - r,  J_{i,i} = 1 + h (w_{i+1} - w_{i-1}) + 2r,  J_{i,i+1} = h w_i - r
//   Newton (Eq.12-13)  w^0 = u^n;  while max_i |F_i(w^k)| >= tol and k < max_iter:
//                      solve J(w^k) delta = -F(w^k),  w^{k+1} = w^k + delta
// (stopping rule: "maximum residual falling below 1e-6"; tol is an argument).
// Dirichlet end nodes are identity rows with zero right-hand side; periodic systems are cyclic.
// Residual and Jacobian are fused into the solver: nothing but u touches HBM.
// theta-scheme ("Crank-Nicolson"): with G(v) = dt times the central
// operator, F(w) = w - u^n + theta G(w) + (1-theta) G(u^n) and J = I + theta dG/dw; theta = 1 is Eq.11.
// The kernels keep k_i = (1-theta) G_i(u^n) - u_i^n per step, so F_i = (w_i + k_i) + theta G_i(w).
//
// Two plans:
//   HYBRID  one CTA per system, w and u^n resident in registers for all n_steps; per Newton iteration
//           one halo exchange, the residual with a block-wide convergence vote, then the same partition
//           elimination + cyclic-reduction + PCR interface solve as btcs_hybrid.cu (btcs_common.cuh)
//           on the Jacobian rows.  No pivoting: J is diagonally dominant when the cell Peclet number
//           |w| dx / nu <= 2 and h (w_{i+1} - w_{i-1}) > -1.
//   THOMAS  one thread per system on the interleaved [N][B] workspace layout of btcs_thomas.cu (any
//           N >= 3), Sherman-Morrison for periodic systems; the general-shape fallback and cross-check.
#include "btcs_common.cuh"

namespace burgers {
namespace {

using namespace btcs;

constexpr int newton_max_threads(int bytes, int P) {
    int regs = P * (bytes / 4) * 5 + 56;
    int t = 1024;
    while (t > 32 && t * regs > 65536) t /= 2;
    return t;
}

// SMALL: the instance for CTAs of at most 128 threads of the fp64, P = 16 kernel (C3's shape).  Asking for
// 3 CTAs per SM makes ptxas fit it into 168 registers (116 bytes spilled) instead of 216: 12 instead of 8
// warps per SM, measured 11 % faster.  Everything else keeps the budget newton_max_threads() assumes.
// RAGGED: any N on a power-of-two number of threads, thread t owning the q or q + 1 rows partition_of() deals
// it (btcs_common.cuh) in the first n of its P register slots; otherwise N == P * blockDim.x.
// TN: the thread count as a compile-time constant for the SMALL instances (PCR levels unrolled), else 0.
// PERIODIC: the boundary type is known to be periodic (no identity-row selects); false: decided by `bc`.
// SNAP: trajectory output from inside the time loop: after every snap_every-th step the state goes to
// snaps[k][b][:] (BN = B N elements per snapshot) -- burgers_newton_traj_* and the forward sweep of the reverse
// mode are then one launch (the three trailing parameters are unused otherwise).
template <typename T, int P, bool SMALL = false, bool RAGGED = false, int TN = 0, bool PERIODIC = false, bool SNAP = false>
__global__ void __launch_bounds__(SMALL ? 128 : newton_max_threads(sizeof(T), P), SMALL ? 3 : 1)
newton_hybrid_kernel(T *__restrict__ u, const T *__restrict__ nu, const T *__restrict__ dt, int N,
                     double inv_dx, int64_t n_steps, int bc, T theta, T tol, int max_iter,
                     long long *__restrict__ iters_out, T *__restrict__ snaps, int64_t snap_every, int64_t BN) {
    constexpr int V = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int t = threadIdx.x, Tn = TN ? TN : (int)blockDim.x, mask = Tn - 1;
    T *sR = reinterpret_cast<T *>(smem_raw);  // [2][Tn] reduced rows (A, C, D): PCR ping-pong
    T *sF = sR + 6 * Tn;                      // [Tn] first interface rows (A, C, D)
    T *sE = sF + 3 * Tn;                      // [2][Tn] partition edge values of w
    Part part;
    part.r0 = t * P; part.n = P;
    if (RAGGED) part = partition_of(t, N, Tn);
    const int n = part.n;                     // rows of this thread (== P unless RAGGED)
    __builtin_assume(n >= P - 1 && n <= P);   // P = ceil(N / Tn): only the last slot is conditional
    T *row = u + (int64_t)blockIdx.x * N + part.r0;

    const double dtb = (double)dt[blockIdx.x];
    const T h = (T)(0.5 * dtb * inv_dx);
    const T r = (T)((double)nu[blockIdx.x] * dtb * inv_dx * inv_dx);
    const T th = theta * h, tr = theta * r, omt = T(1) - theta;     // Jacobian: I + theta dG/dw
    const T b0 = T(1) + T(2) * tr;
    const bool fixL = !PERIODIC && (bc == BURGERS_BC_DIRICHLET) && t == 0;
    const bool fixR = !PERIODIC && (bc == BURGERS_BC_DIRICHLET) && t == Tn - 1;

    T w[P], un[P];       // un holds k_i = (1-theta) G_i(u^n) - u_i^n once the first residual of a step is done
    if (RAGGED) {
#pragma unroll
        for (int j = 0; j < P; ++j) w[j] = (j < n) ? row[j] : T(0);
    } else {
#pragma unroll
        for (int c = 0; c < P / V; ++c) {
            int4 q4 = *reinterpret_cast<const int4 *>(row + c * V);
            const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
            for (int k = 0; k < V; ++k) w[c * V + k] = e[k];
        }
    }
    long long iters = 0;
    int64_t until_snap = snap_every;
    T *snap_row = SNAP ? snaps + (int64_t)blockIdx.x * N + part.r0 : nullptr;
    for (int64_t step = 0; step < n_steps; ++step) {
#pragma unroll
        for (int j = 0; j < P; ++j) un[j] = w[j];
        for (int k = 0;; ++k) {
            // ---- halo exchange of the partition edges
            T wlast = w[P - 1];
            if (RAGGED) {                 // w[n - 1] without a run-time register index
                wlast = w[0];
#pragma unroll
                for (int j = 1; j < P; ++j)
                    if (j < n) wlast = w[j];
            }
            sE[t] = w[0]; sE[Tn + t] = wlast;
            __syncthreads();
            const T wl = sE[Tn + ((t - 1) & mask)], wr = sE[(t + 1) & mask];
            // ---- residual (Eq.11); q = -F is the right-hand side of Eq.12
            T q[P];
            int big = 0;
#pragma unroll
            for (int j = 0; j < P; ++j) {
                if (RAGGED && j >= n) { q[j] = T(0); continue; }
                const bool lastrow = RAGGED ? (j >= n - 1) : (j == P - 1);
                const T wm = (j == 0) ? wl : w[j - 1], wp = lastrow ? wr : w[(j + 1 < P) ? j + 1 : j];
                const T dc = wp - wm;
                const T lap = (wp - w[j]) - (w[j] - wm);
                const T g = t_fma(h * w[j], dc, -r * lap);              // G_i(w)
                if (k == 0) un[j] = t_fma(omt, g, -un[j]);              // w = u^n here
                T F = t_fma(theta, g, w[j] + un[j]);
                if ((j == 0 && fixL) || (lastrow && fixR)) F = T(0);
                q[j] = -F;
                big |= !(t_abs(F) < tol);          // NaN counts as not converged
            }
            const int any = __syncthreads_or(big);  // also orders the sE reads before the next writes
            if (!any || k >= max_iter) break;       // uniform over the CTA
            // ---- Jacobian rows (Eq.14), partition elimination, interface solve, back substitution
            T f[P], c[P];
            Row<T> first, last;
            auto jac = [&](int j, T &a, T &b, T &e) {
                const bool lastrow = RAGGED ? (j >= n - 1) : (j == P - 1);
                if ((j == 0 && fixL) || (lastrow && fixR)) { a = T(0); b = T(1); e = T(0); return; }
                const T wm = (j == 0) ? wl : w[j - 1], wp = lastrow ? wr : w[(j + 1 < P) ? j + 1 : j];
                const T hw = th * w[j];
                a = -hw - tr;
                b = t_fma(th, wp - wm, b0);
                e = hw - tr;
            };
            if (RAGGED) eliminate_general_ragged<T, P>(jac, n, q, f, c, first, last);
            else eliminate_general<T, P>(jac, q, f, c, first, last);
            T x0, xL;
            solve_interface<T, TN>(first, last, sR, sF, x0, xL, t, Tn);
            T d[P];
#pragma unroll
            for (int j = 0; j < P; ++j) d[j] = T(0);
            if (RAGGED) back_substitute_ragged<T, P>(d, n, f, c, q, x0, xL);
            else back_substitute<T, P>(d, f, c, q, x0, xL);
#pragma unroll
            for (int j = 0; j < P; ++j)
                if (!RAGGED || j < n) w[j] += d[j];      // Eq.13
            ++iters;
        }
        if (SNAP) {
            if (--until_snap == 0) {
                until_snap = snap_every;
                T *srow = snap_row;
                snap_row += BN;
#pragma unroll
                for (int j = 0; j < P; ++j)
                    if (!RAGGED || j < n) srow[j] = w[j];
            }
        }
    }
    if (iters_out && t == 0) iters_out[blockIdx.x] += iters;     // (zeroed by launch_newton unless it accumulates)

    if (RAGGED) {
#pragma unroll
        for (int j = 0; j < P; ++j)
            if (j < n) row[j] = w[j];
    } else {
#pragma unroll
        for (int c = 0; c < P / V; ++c) {
            int4 q4;
            T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
            for (int k = 0; k < V; ++k) e[k] = w[c * V + k];
            *reinterpret_cast<int4 *>(row + c * V) = q4;
        }
    }
}

bool newton_geometry(int is_f64, int64_t N, int *P_out, int *T_out, bool *ragged) {
    const int bytes = is_f64 ? 8 : 4;
    return pick_partition(N, [bytes](int P) { return newton_max_threads(bytes, P); }, P_out, T_out, ragged);
}

template <typename T, int P>
int launch_hybrid_P(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                    double theta, double tol, int max_iter, long long *iters_out, int Tn, bool ragged, cudaStream_t s,
                    T *snaps, int64_t snap_every) {
    const size_t smem = (size_t)11 * Tn * sizeof(T);
    const int64_t BN = B * N;
#define BURGERS_NEWTON_ARGS u, nu, dt, (int)N, 1.0 / dx, n_steps, bc, (T)theta, (T)tol, max_iter, iters_out, snaps, snap_every, BN
    if (snaps) {            // trajectory output: the generic instances, snapshots written by the kernel
        if (ragged) {
            newton_hybrid_kernel<T, P, false, true, 0, false, true><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
            return last_launch_status();
        }
        if constexpr (P == 4 || P == 8 || P == 16) {
            if (sizeof(T) == 8 && P == 16 && Tn == 128 && bc == BURGERS_BC_PERIODIC)      // C3's shape
                newton_hybrid_kernel<T, P, true, false, 128, true, true><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
            else if (sizeof(T) == 8 && P == 16 && Tn <= 128)
                newton_hybrid_kernel<T, P, true, false, 0, false, true><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
            else
                newton_hybrid_kernel<T, P, false, false, 0, false, true><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
            return last_launch_status();
        }
        return BURGERS_ERR_PLAN;
    }
    if (ragged) {
        newton_hybrid_kernel<T, P, false, true><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
        return last_launch_status();
    }
    if constexpr (P == 4 || P == 8 || P == 16) {
        if (sizeof(T) == 8 && P == 16 && Tn == 128 && bc == BURGERS_BC_PERIODIC)
            newton_hybrid_kernel<T, P, true, false, 128, true><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
        else if (sizeof(T) == 8 && P == 16 && Tn == 128)
            newton_hybrid_kernel<T, P, true, false, 128><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
        else if (sizeof(T) == 8 && P == 16 && Tn <= 128)
            newton_hybrid_kernel<T, P, true><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
        else
            newton_hybrid_kernel<T, P><<<(unsigned)B, Tn, smem, s>>>(BURGERS_NEWTON_ARGS);
        return last_launch_status();
    }
#undef BURGERS_NEWTON_ARGS
    return BURGERS_ERR_PLAN;
}

// ------------------------------------------------------------------ thread-per-system plan
// ws arrays (each [N][B], batch index fastest): un, w, cp, dp (= rhs, then solution), kn (the per-step
// constant k_i = (1-theta) G_i(u^n) - u_i^n), and for periodic systems wp (second right-hand side of
// Sherman-Morrison).
template <typename T>
__global__ void __launch_bounds__(128)
newton_thomas_kernel(T *__restrict__ un, T *__restrict__ w, T *__restrict__ cp, T *__restrict__ dp,
                     T *__restrict__ kn, T *__restrict__ wp, const T *__restrict__ nu, const T *__restrict__ dt,
                     int64_t B, int64_t N, double inv_dx, int64_t n_steps, int bc, T theta, T tol, int max_iter,
                     long long *__restrict__ iters_out) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const double dtb = (double)dt[b];
    const T h = (T)(0.5 * dtb * inv_dx);
    const T r = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    const T th = theta * h, tr = theta * r, omt = T(1) - theta;
    const T b0 = T(1) + T(2) * tr;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    long long iters = 0;
#define AT(arr, i) arr[(int64_t)(i) * B + b]
    for (int64_t n = 0; n < n_steps; ++n) {
        for (int64_t i = 0; i < N; ++i) AT(w, i) = AT(un, i);
        for (int k = 0;; ++k) {
            // residual; dp <- -F
            bool big = false;
            {
                T wm = dirichlet ? T(0) : AT(w, N - 1), wi = AT(w, 0);
                const T w0 = wi;
                for (int64_t i = 0; i < N; ++i) {
                    const T wpv = (i + 1 < N) ? AT(w, i + 1) : w0;
                    const T g = t_fma(h * wi, wpv - wm, -r * ((wpv - wi) - (wi - wm)));     // G_i(w)
                    if (k == 0) AT(kn, i) = t_fma(omt, g, -AT(un, i));                      // w = u^n here
                    T F = t_fma(theta, g, wi + AT(kn, i));
                    if (dirichlet && (i == 0 || i == N - 1)) F = T(0);
                    AT(dp, i) = -F;
                    big |= !(t_abs(F) < tol);
                    wm = wi; wi = wpv;
                }
            }
            if (!big || k >= max_iter) break;
            // J delta = -F
            if (dirichlet) {      // identity rows at both ends: delta_0 = delta_{N-1} = 0
                T cprev = T(0), dprev = T(0);
                AT(cp, 0) = T(0); AT(dp, 0) = T(0);
                T wm = AT(w, 0), wi = AT(w, 1);
                for (int64_t i = 1; i <= N - 2; ++i) {
                    const T wpv = AT(w, i + 1);
                    const T hw = th * wi;
                    const T a = -hw - tr, bb = t_fma(th, wpv - wm, b0), e = hw - tr;
                    const T inv = T(1) / (bb - a * cprev);
                    cprev = e * inv;
                    dprev = (AT(dp, i) - a * dprev) * inv;
                    AT(cp, i) = cprev; AT(dp, i) = dprev;
                    wm = wi; wi = wpv;
                }
                T x = T(0);      // delta_{N-1}
                for (int64_t i = N - 2; i >= 1; --i) {
                    x = AT(dp, i) - AT(cp, i) * x;
                    AT(w, i) += x;
                }
            } else {              // cyclic: Sherman-Morrison (D6) with gamma = -diag_0
                const T w0 = AT(w, 0), w1 = AT(w, 1), wN1 = AT(w, N - 1);
                const T a0 = -th * w0 - tr, d0 = t_fma(th, w1 - wN1, b0), e0 = th * w0 - tr;
                const T eN = th * wN1 - tr;
                const T gamma = -d0, alpha = a0, beta = eN;
                const T ag = alpha / gamma;
                T inv = T(1) / (d0 - gamma);
                T cprev = e0 * inv, dprev = AT(dp, 0) * inv, wprev = gamma * inv;
                AT(cp, 0) = cprev; AT(dp, 0) = dprev; AT(wp, 0) = wprev;
                T wm = w0, wi = w1;
                for (int64_t i = 1; i < N; ++i) {
                    const T wpv = (i + 1 < N) ? AT(w, i + 1) : w0;
                    const T hw = th * wi;
                    const T a = -hw - tr, e = hw - tr;
                    T bb = t_fma(th, wpv - wm, b0);
                    T ws2 = T(0);
                    if (i == N - 1) { bb = bb - alpha * beta / gamma; ws2 = beta; }
                    inv = T(1) / (bb - a * cprev);
                    cprev = e * inv;
                    dprev = (AT(dp, i) - a * dprev) * inv;
                    wprev = (ws2 - a * wprev) * inv;
                    AT(cp, i) = cprev; AT(dp, i) = dprev; AT(wp, i) = wprev;
                    wm = wi; wi = wpv;
                }
                T y = dprev, qq = wprev;
                const T yN = y, qN = qq;
                for (int64_t i = N - 2; i >= 0; --i) {
                    const T c = AT(cp, i);
                    y = AT(dp, i) - c * y;
                    qq = AT(wp, i) - c * qq;
                    AT(dp, i) = y; AT(wp, i) = qq;
                }
                const T fact = (y + ag * yN) / (T(1) + qq + ag * qN);
                for (int64_t i = 0; i < N; ++i) AT(w, i) += AT(dp, i) - fact * AT(wp, i);
            }
            ++iters;
        }
        for (int64_t i = 0; i < N; ++i) AT(un, i) = AT(w, i);
    }
#undef AT
    if (iters_out) iters_out[b] += iters;
}

}  // namespace

bool newton_hybrid_fits(int is_f64, int64_t N) {
    int P, Tn;
    bool ragged;
    return newton_geometry(is_f64, N, &P, &Tn, &ragged);
}
size_t newton_thomas_ws_elems(int64_t B, int64_t N, int bc) {
    return (size_t)B * (size_t)N * (bc == BURGERS_BC_PERIODIC ? 6 : 5);
}

template <typename T>
int launch_newton(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                  double theta, double tol, int max_iter, long long *iters_out, int plan, T *ws, cudaStream_t s,
                  bool accumulate, T *snaps, int64_t snap_every) {
    // the kernels ADD their iteration totals to iters_out (trajectory output calls this once per interval)
    if (iters_out && !accumulate && cudaMemsetAsync(iters_out, 0, (size_t)B * sizeof(long long), s) != cudaSuccess)
        return BURGERS_ERR_CUDA;
    if (n_steps == 0) return BURGERS_OK;
    if (plan == BURGERS_PLAN_HYBRID) {
        int P, Tn;
        bool ragged;
        if (!newton_geometry(sizeof(T) == 8, N, &P, &Tn, &ragged)) return BURGERS_ERR_PLAN;
        if (B > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
        switch (P) {
#define BURGERS_CASE(PP) \
    case PP: \
        return launch_hybrid_P<T, PP>(u, B, N, dx, nu, dt, n_steps, bc, theta, tol, max_iter, iters_out, Tn, ragged, s, snaps, \
                                      snap_every);
            BURGERS_CASE(4) BURGERS_CASE(5) BURGERS_CASE(6) BURGERS_CASE(7) BURGERS_CASE(8) BURGERS_CASE(9)
            BURGERS_CASE(10) BURGERS_CASE(11) BURGERS_CASE(12) BURGERS_CASE(13) BURGERS_CASE(14) BURGERS_CASE(15)
            BURGERS_CASE(16)
#undef BURGERS_CASE
        }
        return BURGERS_ERR_PLAN;
    }
    // THOMAS
    if (snaps) return BURGERS_ERR_PLAN;          // (trajectory output through this plan: one call per interval, api.cu)
    const size_t BN = (size_t)B * (size_t)N;
    T *un = ws, *w = ws + BN, *cp = ws + 2 * BN, *dp = ws + 3 * BN, *kn = ws + 4 * BN;
    T *wp = (bc == BURGERS_BC_PERIODIC) ? ws + 5 * BN : nullptr;
    int st = launch_transpose<T>(u, un, B, N, s);
    if (st != BURGERS_OK) return st;
    const int threads = thread_per_system_block(B);
    newton_thomas_kernel<T><<<(unsigned)((B + threads - 1) / threads), threads, 0, s>>>(
        un, w, cp, dp, kn, wp, nu, dt, B, N, 1.0 / dx, n_steps, bc, (T)theta, (T)tol, max_iter, iters_out);
    st = last_launch_status();
    if (st != BURGERS_OK) return st;
    return launch_transpose<T>(un, u, N, B, s);
}

template int launch_newton<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, double, double, int, long long *, int, float *, cudaStream_t, bool, float *, int64_t);
template int launch_newton<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, double, double, int, long long *, int, double *, cudaStream_t, bool, double *, int64_t);

}  // namespace burgers
