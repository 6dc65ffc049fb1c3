// btcs_gs.cu -- SURVEY 8(f) NEXT-3: BTCS with the linear system of D4/D5 solved by lexicographic
// GAUSS-SEIDEL sweeps, the paper's iterative variant ("maximum residual falling
// below 1e-6", :339 "5-7 iterations per step"); D12.
//
// Per step: rows (a, b, e) from u^n as in D4 (recomputed from the one loaded value, never stored),
// rhs = u^n, x^0 = u^n; repeat { if max_i |rhs_i - (a_i x_{i-1} + b_i x_i + e_i x_{i+1})| < tol or
// k >= max_iter: stop;  sweep i ascending: x_i <- (rhs_i - a_i x_{i-1} - e_i x_{i+1}) / b_i with the
// newest values }.  Dirichlet: unknowns 1..N-2; periodic neighbours wrap.
//
// A lexicographic sweep is a sequential recurrence, so the plan is ONE THREAD PER SYSTEM on the
// interleaved batch-minor layout of btcs_thomas.cu (coalesced across the batch).  It exists to
// reproduce the paper's iteration counts and for comparison with the direct solvers, which are
// exact and far cheaper (bench: DESIGN.md 6.5); it is not a tuned path.
#include "btcs_common.cuh"

namespace burgers {
namespace {

using namespace btcs;

template <typename T>
__global__ void gs_transpose_kernel(const T *__restrict__ in, T *__restrict__ out, int64_t rows, int64_t cols) {
    __shared__ T tile[32][33];
    const int64_t gx = (cols + 31) / 32;
    const int64_t c0 = ((int64_t)blockIdx.x % gx) * 32, r0 = ((int64_t)blockIdx.x / gx) * 32;
    for (int k = threadIdx.y; k < 32; k += blockDim.y) {
        int64_t r = r0 + k, c = c0 + threadIdx.x;
        if (r < rows && c < cols) tile[k][threadIdx.x] = in[r * cols + c];
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += blockDim.y) {
        int64_t c = c0 + k, r = r0 + threadIdx.x;
        if (r < rows && c < cols) out[c * rows + r] = tile[threadIdx.x][k];
    }
}

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

}  // namespace

size_t btcs_gs_ws_elems(int64_t B, int64_t N) { return (size_t)2 * (size_t)B * (size_t)N; }

template <typename T>
int launch_btcs_gs(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                   double tol, int max_iter, long long *iters_out, T *ws, cudaStream_t s) {
    if (n_steps == 0) {
        if (iters_out && cudaMemsetAsync(iters_out, 0, (size_t)B * sizeof(long long), s) != cudaSuccess)
            return BURGERS_ERR_CUDA;
        return BURGERS_OK;
    }
    const size_t BN = (size_t)B * (size_t)N;
    T *un = ws, *x = ws + BN;
    const int64_t nblk = ((N + 31) / 32) * ((B + 31) / 32);
    if (nblk > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    dim3 tb(32, 8);
    gs_transpose_kernel<T><<<(unsigned)nblk, tb, 0, s>>>(u, un, B, N);
    int st = last_launch_status();
    if (st != BURGERS_OK) return st;
    const int threads = (B <= 148 * 32 * 4) ? 32 : 128;
    btcs_gs_kernel<T><<<(unsigned)((B + threads - 1) / threads), threads, 0, s>>>(
        un, x, nu, dt, B, N, 1.0 / dx, n_steps, bc, (T)tol, max_iter, iters_out);
    st = last_launch_status();
    if (st != BURGERS_OK) return st;
    gs_transpose_kernel<T><<<(unsigned)nblk, tb, 0, s>>>(un, u, N, B);
    return last_launch_status();
}

template int launch_btcs_gs<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, double, int, long long *, float *, cudaStream_t);
template int launch_btcs_gs<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, double, int, long long *, double *, cudaStream_t);

}  // namespace burgers
