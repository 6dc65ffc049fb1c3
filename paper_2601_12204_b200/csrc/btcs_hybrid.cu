// btcs_hybrid.cu -- kernels (2)+(4): fused BTCS assembly + hybrid partition / parallel-cyclic-
// reduction solver, ONE CTA PER SYSTEM, state resident in registers for all n_steps.
//
// Per time step (D4-D6; Eq.23):
//  1. assembly: thread t owns rows t*P .. t*P+P-1; sub/diag/sup are recomputed from its u values
//     (never stored):  c = u dt/dx, r = nu dt/dx^2, a = -r - max(c,0), b = 1 + 2r + |c|,
//     e = -r + min(c,0), d = u.   Dirichlet: rows 0 and N-1 become identity rows (x = u), which is
//     D5's "known end values moved to the right-hand side" written as part of the system.
//  2. local elimination (one sequential sweep of P rows per thread, all threads in parallel):
//     forward  (rows 1..P-1):  f_j x_0 + x_j + c_j x_{j+1} = q_j        [normalised]
//     backward (rows P-3..1, scalars only) gives row 1 as  F x_0 + x_1 + G x_{P-1} = R, and
//     with it the thread's two INTERFACE rows
//        first:  A x_{-1} + x_0 + C x_{P-1} = D          last:  f x_0 + x_{P-1} + c x_P = q
//     (x_{-1} / x_P = last / first unknown of the neighbouring threads; periodic wrap between the
//     last and the first thread -- the cyclic corner terms need no special treatment here).
//  3. the 2T interface rows form a CYCLIC tridiagonal system, solved by parallel cyclic reduction
//     in shared memory (rows kept normalised, diag = 1).  The matrix is strictly diagonally
//     dominant (D4), so the off-diagonals of the reduced rows shrink quadratically per PCR level;
//     once every |A|,|C| is below 2^-70 (fp64; 2^-40 fp32) the remaining levels cannot change a
//     bit of the answer and the loop exits early (block-wide vote).  If it runs to the end, the
//     last level is the exact 2x2 solve of rows k and k+T.
//  4. back substitution inside each thread: x_j = q_j - f_j x_0 - c_j x_{j+1}, j = P-2..1.
// Periodic systems are solved directly as cyclic systems (no Sherman-Morrison second right-hand
// side); the result equals D6's up to rounding.
#include "btcs_common.cuh"

namespace burgers {
namespace {

using namespace btcs;

constexpr int hybrid_max_threads(int bytes, int P) {
    int regs = P * (bytes / 4) * 4 + 48;
    int t = 1024;
    while (t > 32 && t * regs > 65536) t /= 2;
    return t;
}

template <typename T, int P>
__global__ void __launch_bounds__(hybrid_max_threads(sizeof(T), P))
btcs_hybrid_kernel(T *__restrict__ u, const T *__restrict__ nu, const T *__restrict__ dt, int N,
                   double inv_dx, int64_t n_steps, int bc) {
    constexpr int V = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int t = threadIdx.x, Tn = blockDim.x, M = 2 * Tn;
    T *sA = reinterpret_cast<T *>(smem_raw);  // [2][M]
    T *sC = sA + 2 * M;
    T *sD = sC + 2 * M;
    T *row = u + (int64_t)blockIdx.x * N + (int64_t)t * P;

    Coef<T> co;
    co.init(nu[blockIdx.x], dt[blockIdx.x], inv_dx);
    const bool fixL = (bc == BURGERS_BC_DIRICHLET) && t == 0;
    const bool fixR = (bc == BURGERS_BC_DIRICHLET) && t == Tn - 1;

    T v[P];
#pragma unroll
    for (int c = 0; c < P / V; ++c) {
        int4 q4 = *reinterpret_cast<const int4 *>(row + c * V);
        const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
        for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
    }

    int cur = 0;
    for (int64_t n = 0; n < n_steps; ++n) {
        T f[P], c[P], q[P];
        // ---- assembly + partition elimination; interface rows -> shared memory, buffer cur^1
        {
            Row<T> first, last;
            eliminate<T, P>(v, co, [&](int j) { return (j == 0 && fixL) || (j == P - 1 && fixR); },
                            f, c, q, first, last);
            const int o = (cur ^ 1) * M + 2 * t;
            sA[o] = first.A; sA[o + 1] = last.A;
            sC[o] = first.C; sC[o + 1] = last.C;
            sD[o] = first.D; sD[o + 1] = last.D;
        }
        __syncthreads();
        cur ^= 1;
        // ---- parallel cyclic reduction over the M interface rows
        bool finished = false;
        for (int s = 1; s < Tn; s <<= 1) {
            int flag = 0;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int k = t + h * Tn;
                const int km = (k - s) & (M - 1), kp = (k + s) & (M - 1);
                const T *pA = sA + cur * M, *pC = sC + cur * M, *pD = sD + cur * M;
                const T A = pA[k], C = pC[k], D = pD[k];
                const T m = rcp(t_fma(-A, pC[km], t_fma(-C, pA[kp], T(1))));
                const T An = -A * pA[km] * m;
                const T Cn = -C * pC[kp] * m;
                const T Dn = t_fma(-A, pD[km], t_fma(-C, pD[kp], D)) * m;
                const int o = (cur ^ 1) * M + k;
                sA[o] = An; sC[o] = Cn; sD[o] = Dn;
                flag |= (t_abs(An) > Lim<T>::tiny()) | (t_abs(Cn) > Lim<T>::tiny());
            }
            const int any = __syncthreads_or(flag);
            cur ^= 1;
            if (!any) { finished = true; break; }
        }
        if (!finished) {  // rows k and k+Tn couple only to each other: exact 2x2 solve
            const T *pA = sA + cur * M, *pC = sC + cur * M, *pD = sD + cur * M;
            const int k = t, k2 = t + Tn;
            const T p1 = pA[k] + pC[k], p2 = pA[k2] + pC[k2];
            const T D1 = pD[k], D2 = pD[k2];
            const T m = rcp(t_fma(-p1, p2, T(1)));
            sD[(cur ^ 1) * M + k] = t_fma(-p1, D2, D1) * m;
            sD[(cur ^ 1) * M + k2] = t_fma(-p2, D1, D2) * m;
            __syncthreads();
            cur ^= 1;
        }
        // ---- back substitution
        back_substitute<T, P>(v, f, c, q, sD[cur * M + 2 * t], sD[cur * M + 2 * t + 1]);
    }

#pragma unroll
    for (int c = 0; c < P / V; ++c) {
        int4 q4;
        T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
        for (int k = 0; k < V; ++k) e[k] = v[c * V + k];
        *reinterpret_cast<int4 *>(row + c * V) = q4;
    }
}

bool pow2(int64_t x) { return x > 0 && (x & (x - 1)) == 0; }

// P rows per thread, Tn = N/P threads (a power of two >= 2)
bool hybrid_geometry(int is_f64, int64_t N, int *P_out, int *T_out) {
    const int bytes = is_f64 ? 8 : 4;
    const int cand[3] = {16, 8, 4};
    int bestP = 0;
    for (int i = 0; i < 3; ++i) {
        const int P = cand[i];
        if (N % P) continue;
        const int64_t Tn = N / P;
        if (!pow2(Tn) || Tn < 2 || Tn > hybrid_max_threads(bytes, P)) continue;
        if (Tn >= 32) { bestP = P; break; }   // largest P that still fills a warp
        bestP = P;                            // otherwise keep shrinking P (more threads)
    }
    if (!bestP) return false;
    *P_out = bestP; *T_out = (int)(N / bestP);
    return true;
}

template <typename T, int P>
int launch_P(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
             int Tn, cudaStream_t s) {
    const size_t smem = (size_t)12 * Tn * sizeof(T);
    btcs_hybrid_kernel<T, P><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc);
    return last_launch_status();
}

}  // namespace

bool btcs_hybrid_fits(int is_f64, int64_t N, int bc) {
    (void)bc;
    int P, Tn;
    return hybrid_geometry(is_f64, N, &P, &Tn);
}

template <typename T>
int launch_btcs_hybrid(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                       int64_t n_steps, int bc, cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    int P, Tn;
    if (!hybrid_geometry(sizeof(T) == 8, N, &P, &Tn)) return BURGERS_ERR_PLAN;
    if (B > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    switch (P) {
        case 4: return launch_P<T, 4>(u, B, N, dx, nu, dt, n_steps, bc, Tn, s);
        case 8: return launch_P<T, 8>(u, B, N, dx, nu, dt, n_steps, bc, Tn, s);
        case 16: return launch_P<T, 16>(u, B, N, dx, nu, dt, n_steps, bc, Tn, s);
    }
    return BURGERS_ERR_PLAN;
}

template int launch_btcs_hybrid<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, cudaStream_t);
template int launch_btcs_hybrid<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, cudaStream_t);

}  // namespace burgers
