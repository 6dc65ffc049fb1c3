// btcs_thomas.cu -- kernels (2)+(3): fused BTCS assembly + batched Thomas solver, ONE THREAD PER
// SYSTEM on an interleaved batch-minor layout.
//
// BTCS rows (D4; Eq.23 with the coefficient lagged at u^n):
//   c_i = u_i^n dt/dx, r = nu dt/dx^2,
//   sub_i = -r - max(c_i,0), diag_i = 1 + 2r + |c_i|, sup_i = -r + min(c_i,0), rhs_i = u_i^n.
// The three coefficients are functions of the one loaded value u_i^n: they are recomputed on the
// fly and never touch memory.  Dirichlet (D5): unknowns 1..N-2 with the end values moved to the
// right-hand side.  Periodic (D6): Sherman-Morrison with gamma = -diag_0, two right-hand sides
// through one elimination, rank-one combine.  Thomas recurrences as in D7.
//
// Layout: the caller's [B][N] state is transposed once into ws as ut[N][B] (batch index fastest),
// so that at every sweep position i the 32 threads of a warp touch 32 consecutive elements
// (coalesced); cp/dp(/wp) sweeps use the same layout.  All n_steps run inside one launch; the
// result is transposed back once.  With B of a few thousand this plan is latency-bound (one
// dependent divide chain of length N per thread): it is the right plan only for B >~ 1e5 or as
// the general-shape fallback, and serves as the cross-check of the HYBRID plan.
#include "common.cuh"

namespace burgers {
namespace {

template <typename T>
struct Rows {
    T r, cx;
    __device__ __forceinline__ void at(T u, T &a, T &b, T &e) const {
        const T c = u * cx;
        const T cpos = (c > T(0)) ? c : T(0);
        const T cneg = (c > T(0)) ? T(0) : c;
        a = -r - cpos;
        b = T(1) + T(2) * r + (cpos - cneg);
        e = -r + cneg;
    }
};

template <typename T>
__global__ void __launch_bounds__(128)
btcs_thomas_kernel(T *__restrict__ ut, T *__restrict__ cp, T *__restrict__ dp, T *__restrict__ wp,
                   const T *__restrict__ nu, const T *__restrict__ dt, int64_t B, int64_t N,
                   double inv_dx, int64_t n_steps, int bc) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const double dtb = (double)dt[b];
    Rows<T> rows;
    rows.cx = (T)(dtb * inv_dx);
    rows.r = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
#define AT(arr, i) arr[(int64_t)(i) * B + b]
    if (bc == BURGERS_BC_DIRICHLET) {
        const T uL = AT(ut, 0), uR = AT(ut, N - 1);
        const int64_t last = N - 2;
        for (int64_t n = 0; n < n_steps; ++n) {
            T a, d, e, bb;
            T u = AT(ut, 1);
            rows.at(u, a, bb, e);
            d = u - a * uL;
            if (last == 1) d -= e * uR;
            T inv = T(1) / bb;
            T cprev = e * inv, dprev = d * inv;
            AT(cp, 1) = cprev; AT(dp, 1) = dprev;
            for (int64_t i = 2; i <= last; ++i) {
                u = AT(ut, i);
                rows.at(u, a, bb, e);
                d = u;
                if (i == last) d -= e * uR;
                inv = T(1) / (bb - a * cprev);
                cprev = e * inv;
                dprev = (d - a * dprev) * inv;
                AT(cp, i) = cprev; AT(dp, i) = dprev;
            }
            T x = dprev;
            AT(ut, last) = x;
            for (int64_t i = last - 1; i >= 1; --i) {
                x = AT(dp, i) - AT(cp, i) * x;
                AT(ut, i) = x;
            }
        }
    } else {
        for (int64_t n = 0; n < n_steps; ++n) {
            T a, bb, e;
            const T u0 = AT(ut, 0), uN = AT(ut, N - 1);
            T a0, b0, e0, aN, bN, eN;
            rows.at(u0, a0, b0, e0);
            rows.at(uN, aN, bN, eN);
            const T gamma = -b0, alpha = a0, beta = eN;  // corners M[0][N-1]=alpha, M[N-1][0]=beta
            const T ag = alpha / gamma;
            // row 0 of T: diag' = b0 - gamma
            T inv = T(1) / (b0 - gamma);
            T cprev = e0 * inv, dprev = u0 * inv, wprev = gamma * inv;
            AT(cp, 0) = cprev; AT(dp, 0) = dprev; AT(wp, 0) = wprev;
            for (int64_t i = 1; i < N; ++i) {
                const T u = (i == N - 1) ? uN : AT(ut, i);
                rows.at(u, a, bb, e);
                T w = T(0);
                if (i == N - 1) { bb = bb - alpha * beta / gamma; w = beta; }
                inv = T(1) / (bb - a * cprev);
                cprev = e * inv;
                dprev = (u - a * dprev) * inv;
                wprev = (w - a * wprev) * inv;
                AT(cp, i) = cprev; AT(dp, i) = dprev; AT(wp, i) = wprev;
            }
            T y = dprev, q = wprev;  // back substitution of both right-hand sides, in place
            const T yN = y, qN = q;
            for (int64_t i = N - 2; i >= 0; --i) {
                const T c = AT(cp, i);
                y = AT(dp, i) - c * y;
                q = AT(wp, i) - c * q;
                AT(dp, i) = y; AT(wp, i) = q;
            }
            const T fact = (y + ag * yN) / (T(1) + q + ag * qN);
            for (int64_t i = 0; i < N; ++i) AT(ut, i) = AT(dp, i) - fact * AT(wp, i);
        }
    }
#undef AT
}

}  // namespace

size_t btcs_thomas_ws_elems(int64_t B, int64_t N, int bc) {
    return (size_t)B * (size_t)N * (bc == BURGERS_BC_PERIODIC ? 4 : 3);
}
int64_t btcs_thomas_launch_count(int64_t n_steps) { return n_steps > 0 ? 3 : 0; }

template <typename T>
int launch_btcs_thomas(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                       int64_t n_steps, int bc, T *ws, cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    const size_t BN = (size_t)B * (size_t)N;
    T *ut = ws, *cp = ws + BN, *dp = ws + 2 * BN, *wp = (bc == BURGERS_BC_PERIODIC) ? ws + 3 * BN : nullptr;
    int st = launch_transpose<T>(u, ut, B, N, s);
    if (st != BURGERS_OK) return st;
    const int threads = thread_per_system_block(B);
    btcs_thomas_kernel<T><<<(unsigned)((B + threads - 1) / threads), threads, 0, s>>>(
        ut, cp, dp, wp, nu, dt, B, N, 1.0 / dx, n_steps, bc);
    st = last_launch_status();
    if (st != BURGERS_OK) return st;
    return launch_transpose<T>(ut, u, N, B, s);
}

template int launch_btcs_thomas<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, float *, cudaStream_t);
template int launch_btcs_thomas<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, double *, cudaStream_t);

}  // namespace burgers
