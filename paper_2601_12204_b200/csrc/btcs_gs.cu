// btcs_gs.cu -- SURVEY 8(f) NEXT-3: BTCS with the linear system of D4/D5 solved by lexicographic
// GAUSS-SEIDEL sweeps, the paper's iterative variant ("maximum residual falling
// below 1e-6", :339 "5-7 iterations per step"); D12.
//
// Per step: rows (a, b, e) from u^n as in D4, rhs = u^n, x^0 = u^n; repeat { if max_i |rhs_i -
// (a_i x_{i-1} + b_i x_i + e_i x_{i+1})| < tol or k >= max_iter: stop;  sweep i ascending:
// x_i <- (rhs_i - a_i x_{i-1} - e_i x_{i+1}) / b_i with the newest values }.  Dirichlet: unknowns
// 1..N-2; periodic neighbours wrap (row 0 sees the OLD x_{N-1}, row N-1 the NEW x_0).
//
// Two plans:
//  * CTA PER SYSTEM (64 <= N <= 4096).  With the right neighbour taken from the old
//    iterate, a lexicographic sweep is the first-order linear recurrence
//        x_i = p_i + q_i x_{i-1},   p_i = (rhs_i - e_i x_{i+1}^old) / b_i,   q_i = -a_i / b_i,  |q_i| < 1
//    (diagonal dominance), i.e. a composition of affine maps, which is associative: each thread
//    composes the maps of its P consecutive rows, the CTA scans the thread maps (warp shuffles, then
//    the warp totals serially), and a second pass over the P rows applies them.  The result is the
//    sequential sweep up to rounding order.  The state stays in registers for all n_steps: one load
//    and one store of u per call; per step rhs/b, e/b, q and b are computed once; the residual test
//    of iteration k shares p_i with sweep k (scaled by 1/b_i; b_i |.| is compared with tol).
//  * THREAD PER SYSTEM on the interleaved batch-minor layout of btcs_thomas.cu for the other
//    shapes (tiny systems, or systems too long for one CTA's registers): the literal loop.
#include "btcs_common.cuh"

namespace burgers {
namespace {

using namespace btcs;

template <typename T>
__global__ void __launch_bounds__(128)
btcs_gs_kernel(T *__restrict__ un, T *__restrict__ x, const T *__restrict__ nu, const T *__restrict__ dt,
               int64_t B, int64_t N, double inv_dx, int64_t n_steps, int bc, T tol, int max_iter,
               long long *__restrict__ iters_out) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    Coef<T> co;
    co.init(nu[b], dt[b], inv_dx);
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t lo = dirichlet ? 1 : 0, hi = dirichlet ? N - 1 : N;
    long long iters = 0;
#define AT(arr, i) arr[(int64_t)(i) * B + b]
    for (int64_t n = 0; n < n_steps; ++n) {
        for (int64_t i = 0; i < N; ++i) AT(x, i) = AT(un, i);
        for (int k = 0;; ++k) {
            // residual of the current iterate
            bool big = false;
            {
                T xm = AT(x, lo == 0 ? N - 1 : lo - 1), xi = AT(x, lo);
                const T x0 = AT(x, 0);
                for (int64_t i = lo; i < hi; ++i) {
                    const T xp = (i + 1 < N) ? AT(x, i + 1) : x0;
                    const T d = AT(un, i);
                    T a, bb, e;
                    co.at(d, a, bb, e);
                    const T res = d - t_fma(a, xm, t_fma(bb, xi, e * xp));
                    big |= !(t_abs(res) < tol);
                    xm = xi; xi = xp;
                }
            }
            if (!big || k >= max_iter) break;
            // one lexicographic sweep
            {
                T xm = AT(x, lo == 0 ? N - 1 : lo - 1);       // old x_{N-1} for i = 0 (periodic)
                for (int64_t i = lo; i < hi; ++i) {
                    const T xp = (i + 1 < N) ? AT(x, i + 1) : AT(x, 0);   // x_0 is already new at i = N-1
                    const T d = AT(un, i);
                    T a, bb, e;
                    co.at(d, a, bb, e);
                    const T xn = (d - a * xm - e * xp) / bb;
                    AT(x, i) = xn;
                    xm = xn;
                }
            }
            ++iters;
        }
        for (int64_t i = lo; i < hi; ++i) AT(un, i) = AT(x, i);
    }
#undef AT
    if (iters_out) iters_out[b] = iters;
}


template <typename T> __device__ __forceinline__ T shfl_up_t(T v, int off) { return __shfl_up_sync(0xffffffffu, v, off); }

// Six P-element arrays live across an iteration (x, rhs/b, e/b, q, tol/b, p): P = 16 in fp64 needs the
// full register budget (241 when ptxas is left alone, which is 5 % faster than asking for 2 CTAs per SM), so 2 CTAs of
// 128 threads per SM; measured on C3's shape (N = 2048, fp64), P = 16
// x 128 threads beats 8 x 256 (6.1 against 7.7 ms per 100 steps) and 4 x 512 (13.3): the scan over the
// threads, not the row arithmetic, is the expensive part, so few threads with many rows each.
constexpr int gs_min_ctas(int P, int NT) { return NT > 128 ? 1 : (P >= 16 ? 0 : P >= 8 ? 3 : 4); }   // 0 = unspecified

// CTA per system.  Thread t owns rows t*P .. t*P+P-1; rows >= N and the Dirichlet end nodes are
// identity rows (q = 0, e/b = 0, rhs/b = x, b = 1).  blockDim.x = ceil(N / P) rounded up to a warp.
// ALIGNED: N is a multiple of P, so row N-1 is the last row of thread N/P - 1 and the periodic wrap
// is a per-thread scalar choice of the right neighbour; otherwise row N-1 sits at a run-time position
// inside its thread and every row pays a compare + select for it.
template <typename T, int P, int NT, bool ALIGNED>
__global__ void __launch_bounds__(NT, gs_min_ctas(P, NT))
btcs_gs_cta_kernel(T *__restrict__ u, const T *__restrict__ nu, const T *__restrict__ dt, int N,
                   double inv_dx, int64_t n_steps, int bc, T tol, int max_iter,
                   long long *__restrict__ iters_out) {
    constexpr int NW = NT / 32;
    __shared__ T sFirst[NT], sLast[NT];
    __shared__ T sWP[NW], sWQ[NW];
    __shared__ T sP0, sQ0, sXl;
    const int t = threadIdx.x, lane = t & 31, w = t >> 5, nthr = blockDim.x;
    const int64_t b = blockIdx.x;
    T *__restrict__ row = u + b * (int64_t)N;
    Coef<T> co;
    co.init(nu[b], dt[b], inv_dx);
    const bool periodic = (bc == BURGERS_BC_PERIODIC);
    const int g0 = t * P;
    const int jl = (N - 1) - g0;            // local index of global row N-1 (outside 0..P-1 for most threads)
    const bool wrap_thread = periodic && (jl == P - 1);          // ALIGNED: the thread whose last row is N-1

    T x[P];
#pragma unroll
    for (int j = 0; j < P; ++j) x[j] = (g0 + j < N) ? row[g0 + j] : T(0);

    long long iters = 0;
    for (int64_t n = 0; n < n_steps; ++n) {
        T db[P], eb[P], q[P], tb[P];        // rhs/b, e/b, -a/b, tol/b
#pragma unroll
        for (int j = 0; j < P; ++j) {
            T a, bq, e;
            co.at(x[j], a, bq, e);
            const int g = g0 + j;
            if (g >= N || (!periodic && (g == 0 || g == N - 1))) { a = T(0); bq = T(1); e = T(0); }
            const T ib = rcp(bq);
            db[j] = x[j] * ib;
            eb[j] = e * ib;
            q[j] = -a * ib;
            tb[j] = tol * ib;
        }
        for (int k = 0;; ++k) {
            sFirst[t] = x[0];
            sLast[t] = x[P - 1];
            if (t == 0) { sP0 = t_fma(-eb[0], x[1], db[0]); sQ0 = q[0]; }
            if (!ALIGNED) {
#pragma unroll
                for (int j = 0; j < P; ++j)
                    if (j == jl) sXl = x[j];
            }
            __syncthreads();
            const T xl = ALIGNED ? sLast[N / P - 1] : sXl;      // old x_{N-1}
            const T x0old = sFirst[0];
            const T x0new = t_fma(sQ0, xl, sP0);                // the value thread 0 gives row 0 below, bitwise
            const T nextFirst = (t + 1 < nthr) ? sFirst[t + 1] : T(0);
            const T nf_res = (ALIGNED && wrap_thread) ? x0old : nextFirst;   // right neighbour of the thread's
            const T nf_swp = (ALIGNED && wrap_thread) ? x0new : nextFirst;   // last row: residual / sweep
            // pass 1: residual of the current iterate, and the thread's composed map x_out = Pt + Qt x_in
            bool big = false;
            T Pt = T(0), Qt = T(1);
            T xm = (t > 0) ? sLast[t - 1] : xl;
            T pp[P];
#pragma unroll
            for (int j = 0; j < P; ++j) {
                T xp = (j < P - 1) ? x[j + 1] : nf_res;
                if (!ALIGNED && periodic && j == jl) xp = x0old;
                T p = t_fma(-eb[j], xp, db[j]);
                const T s = t_fma(q[j], xm, p) - x[j];          // residual_j / b_j
                big |= !(t_abs(s) < tb[j]);
                if (ALIGNED) {
                    if (j == P - 1) p = t_fma(-eb[j], nf_swp, db[j]);
                } else if (periodic && j == jl) {
                    p = t_fma(-eb[j], x0new, db[j]);
                }
                pp[j] = p;
                Pt = t_fma(q[j], Pt, p);
                Qt = q[j] * Qt;
                xm = x[j];
            }
            // inclusive scan of the thread maps inside the warp
            T Pi = Pt, Qi = Qt;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const T Pu = shfl_up_t(Pi, off), Qu = shfl_up_t(Qi, off);
                if (lane >= off) { Pi = t_fma(Qi, Pu, Pi); Qi = Qi * Qu; }
            }
            if (lane == 31) { sWP[w] = Pi; sWQ[w] = Qi; }
            const int anybig = __syncthreads_or(big ? 1 : 0);
            if (!anybig || k >= max_iter) break;
            // value entering this warp's first row (the warp totals applied in order), then this thread's
            T v = xl;
#pragma unroll
            for (int ww = 0; ww < NW - 1; ++ww) {
                const T wq = sWQ[ww], wp = sWP[ww];
                if (ww < w) v = t_fma(wq, v, wp);
            }
            const T Pe = shfl_up_t(Pi, 1), Qe = shfl_up_t(Qi, 1);
            T xprev = (lane == 0) ? v : t_fma(Qe, v, Pe);
            // pass 2: the sweep
#pragma unroll
            for (int j = 0; j < P; ++j) {
                x[j] = t_fma(q[j], xprev, pp[j]);
                xprev = x[j];
            }
            ++iters;
        }
    }
#pragma unroll
    for (int j = 0; j < P; ++j)
        if (g0 + j < N) row[g0 + j] = x[j];
    if (iters_out && t == 0) iters_out[b] = iters;
}

template <typename T, int P, int NT>
int launch_gs_cta(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                  double tol, int max_iter, long long *iters_out, cudaStream_t s) {
    const int threads = (int)(((N + P - 1) / P + 31) / 32 * 32);
    if (N % P == 0)
        btcs_gs_cta_kernel<T, P, NT, true><<<(unsigned)B, threads, 0, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc,
                                                                           (T)tol, max_iter, iters_out);
    else
        btcs_gs_cta_kernel<T, P, NT, false><<<(unsigned)B, threads, 0, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc,
                                                                            (T)tol, max_iter, iters_out);
    return last_launch_status();
}

}  // namespace

bool btcs_gs_cta_plan(int64_t B, int64_t N) { return N >= 64 && N <= 4096 && B <= 0x7fffffffLL; }

size_t btcs_gs_ws_elems(int64_t B, int64_t N) { return btcs_gs_cta_plan(B, N) ? 0 : (size_t)2 * (size_t)B * (size_t)N; }

template <typename T>
int launch_btcs_gs(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                   double tol, int max_iter, long long *iters_out, T *ws, cudaStream_t s) {
    if (n_steps == 0) {
        if (iters_out && cudaMemsetAsync(iters_out, 0, (size_t)B * sizeof(long long), s) != cudaSuccess)
            return BURGERS_ERR_CUDA;
        return BURGERS_OK;
    }
    if (btcs_gs_cta_plan(B, N)) {
        if (N <= 512) return launch_gs_cta<T, 4, 128>(u, B, N, dx, nu, dt, n_steps, bc, tol, max_iter, iters_out, s);
        if (N <= 1024) return launch_gs_cta<T, 8, 128>(u, B, N, dx, nu, dt, n_steps, bc, tol, max_iter, iters_out, s);
        if (N <= 2048) return launch_gs_cta<T, 16, 128>(u, B, N, dx, nu, dt, n_steps, bc, tol, max_iter, iters_out, s);
        return launch_gs_cta<T, 16, 256>(u, B, N, dx, nu, dt, n_steps, bc, tol, max_iter, iters_out, s);
    }
    const size_t BN = (size_t)B * (size_t)N;
    T *un = ws, *x = ws + BN;
    int st = launch_transpose<T>(u, un, B, N, s);
    if (st != BURGERS_OK) return st;
    const int threads = thread_per_system_block(B);
    btcs_gs_kernel<T><<<(unsigned)((B + threads - 1) / threads), threads, 0, s>>>(
        un, x, nu, dt, B, N, 1.0 / dx, n_steps, bc, (T)tol, max_iter, iters_out);
    st = last_launch_status();
    if (st != BURGERS_OK) return st;
    return launch_transpose<T>(un, u, N, B, s);
}

template int launch_btcs_gs<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, double, int, long long *, float *, cudaStream_t);
template int launch_btcs_gs<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, double, int, long long *, double *, cudaStream_t);

}  // namespace burgers
