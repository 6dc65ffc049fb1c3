// adjoint.cu -- SURVEY 8(f) NEXT-4c: discrete adjoint of the forward-Euler scheme, i.e. the
// reverse-mode derivative dJ/du^0 = (du^N/du^0)^T dJ/du^N that the paper gets from JAX autodiff
// (PAPER.md:231, :261, :409); D13.
//
// One forward step is u^{n+1} = Phi(u^n), Phi_i = u_i + dt F_i(u) (D2/D3).  With cx = dt/dx,
// rr = nu dt/dx^2 and the upwind switch held fixed, row i of dPhi/du is
//   u_i > 0 :  (cx u_i + rr,  1 - cx (2u_i - u_{i-1}) - 2rr,  rr)
//   u_i <= 0:  (rr,  1 - cx (u_{i+1} - 2u_i) - 2rr,  rr - cx u_i)          on columns (i-1, i, i+1)
// and the identity row for Dirichlet end nodes.  One adjoint step gathers column j:
//   lam^n_j = dPhi_{j-1}/du_j lam_{j-1} + dPhi_j/du_j lam_j + dPhi_{j+1}/du_j lam_{j+1}   at u^n.
// The forward states u^0..u^{N-1} come from the trajectory output of the explicit kernel (one
// snapshot per step, written by the RESIDENT kernel from its on-chip state).  Backward sweep, two plans:
//   RESIDENT  one CTA per trajectory keeps lam in registers for all steps (P consecutive points per
//             thread, edge values of u^n and lam exchanged through shared memory, one barrier per step)
//             and STREAMS the stored states two steps ahead; the column is evaluated in the scaled
//             variable w = cx u with every upwind coefficient formed once and applied as lam_j + increment
//             (see the kernel).  sizeof(T) bytes of HBM traffic per point and step.  Needs N = P * threads
//             with threads <= 512.
//   STREAMING one launch per step over all points (any N): reads u^n and lam, writes lam.
#include "common.cuh"

namespace burgers {
namespace {

template <typename T>
__global__ void __launch_bounds__(256)
adjoint_step_kernel(const T *__restrict__ u, const T *__restrict__ lam, T *__restrict__ out,
                    const T *__restrict__ nu, const T *__restrict__ dt, int64_t N, double inv_dx, int bc) {
    const int64_t b = blockIdx.y;
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const double dtb = (double)dt[b];
    const T cx = (T)(dtb * inv_dx);
    const T rr = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    const T *ur = u + b * N, *lr = lam + b * N;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t jm = (j == 0) ? N - 1 : j - 1, jp = (j == N - 1) ? 0 : j + 1;
    const T um = ur[jm], uj = ur[j], up = ur[jp];
    T acc;
    // row j (its diagonal entry)
    if (dirichlet && (j == 0 || j == N - 1)) {
        acc = lr[j];
    } else {
        const T g = (uj > T(0)) ? (uj - um) : (up - uj);
        const T d0 = T(1) - cx * ((uj > T(0)) ? uj : -uj) - cx * g - T(2) * rr;
        acc = d0 * lr[j];
    }
    // row j-1, column j: its "right" entry
    if (!(dirichlet && (j == 0 || jm == 0))) {
        const T dp = (um > T(0)) ? rr : rr - cx * um;
        acc += dp * lr[jm];
    }
    // row j+1, column j: its "left" entry
    if (!(dirichlet && (j == N - 1 || jp == N - 1))) {
        const T dm = (up > T(0)) ? cx * up + rr : rr;
        acc += dm * lr[jp];
    }
    out[b * N + j] = acc;
}

// ---- RESIDENT backward sweep
template <typename T, int P>
__global__ void __launch_bounds__(512)
adjoint_resident_kernel(const T *__restrict__ u0, const T *__restrict__ states, T *__restrict__ lam,
                        const T *__restrict__ nu, const T *__restrict__ dt, int64_t B, int64_t N, double inv_dx,
                        int64_t n_steps, int bc) {
    constexpr int V = 16 / sizeof(T);
    static_assert(P % V == 0, "a thread row must be a whole number of 16-byte vectors");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *edge = reinterpret_cast<T *>(smem_raw);          // [2][4][nth]
    const int t = threadIdx.x, nth = blockDim.x;
    const int64_t b = blockIdx.x;
    const double dtb = (double)dt[b];
    const T cx = (T)(dtb * inv_dx);
    const T rr = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t off = b * N + (int64_t)t * P, BN = B * N;
    auto load = [&](const T *src, T (&dst)[P]) {
#pragma unroll
        for (int c = 0; c < P / V; ++c) {
            const int4 q = *reinterpret_cast<const int4 *>(src + off + c * V);
            const T *e = reinterpret_cast<const T *>(&q);
#pragma unroll
            for (int k = 0; k < V; ++k) dst[c * V + k] = e[k];
        }
    };
    auto state = [&](int64_t n) { return (n == 0) ? u0 : states + (size_t)(n - 1) * (size_t)BN; };
    // the states are streamed TWO steps ahead (un1: step n-1, un2: step n-2): with one step in flight the
    // kernel kept only ~32 KB per SM outstanding and reached 0.61 of the HBM bandwidth
    T l[P], uc[P], un1[P], un2[P];
    load(lam, l);
    load(state(n_steps - 1), uc);
    if (n_steps >= 2) load(state(n_steps - 2), un1);
    const int tl = (t == 0) ? nth - 1 : t - 1, tr = (t == nth - 1) ? 0 : t + 1;
    const bool firstT = (t == 0), lastT = (t == nth - 1);
    int buf = 0;
    for (int64_t n = n_steps - 1; n >= 0; --n) {
        if (n > 1) load(state(n - 2), un2);             // prefetch the state of the step after next
        // Row j of the transposed step Jacobian in the scaled variable w = cx u (D13):
        //   (M^T l)_j = d0_j l_j + A_{j-1} l_{j-1} + C_{j+1} l_{j+1},
        //   A_i = rr - min(w_i, 0)   (dPhi_i/du_{i+1}),      C_i = rr + max(w_i, 0)   (dPhi_i/du_{i-1}),
        //   d0_j = 1 - 2 rr - |w_j| - (w_j > 0 ? w_j - w_{j-1} : w_{j+1} - w_j)   (applied as l_j + (d0_j - 1) l_j).
        // A frozen Dirichlet end node i has Phi_i = u_i: d0_i = 1, A_i = C_i = 0 -- which also removes the
        // periodic wrap terms, so the formula holds for every j.  Each A_i, C_i is formed once.
        T w[P];
#pragma unroll
        for (int j = 0; j < P; ++j) w[j] = cx * uc[j];
        const bool fixF = dirichlet && firstT, fixL = dirichlet && lastT;
        const T Cfirst = fixF ? T(0) : rr + fmax(w[0], T(0));
        const T Alast = fixL ? T(0) : rr - fmin(w[P - 1], T(0));
        T *e = edge + buf * 4 * nth;
        e[t] = w[0]; e[nth + t] = w[P - 1]; e[2 * nth + t] = Cfirst * l[0]; e[3 * nth + t] = Alast * l[P - 1];
        __syncthreads();
        const T wL = e[nth + tl], wR = e[tr], pL = e[3 * nth + tl], pR = e[2 * nth + tr];
        buf ^= 1;
        const T two_rr = T(2) * rr;
        T ln[P];
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const T wm = j ? w[j - 1] : wL, wj = w[j], wp = (j < P - 1) ? w[j + 1] : wR;
            const T gw = (wj > T(0)) ? (wj - wm) : (wp - wj);
            // l_j + increment: the increment is formed on its own and added once, so that a step costs
            // l_j one rounding (10 000 fp32 steps of C2 stay inside the 1e-4 bar)
            T inc = -((fabs(wj) + gw) + two_rr) * l[j];                  // (d0_j - 1) l_j
            if ((j == 0 && fixF) || (j == P - 1 && fixL)) inc = T(0);
            // left neighbour's Phi depends on u_j through A_{j-1}
            if (j == 0) inc += pL;
            else {
                T A = rr - fmin(wm, T(0));
                if (j == 1 && fixF) A = T(0);
                inc = fma(A, l[j - 1], inc);
            }
            // right neighbour's Phi depends on u_j through C_{j+1}
            if (j == P - 1) inc += pR;
            else {
                T C = rr + fmax(wp, T(0));
                if (j == P - 2 && fixL) C = T(0);
                inc = fma(C, l[j + 1], inc);
            }
            ln[j] = l[j] + inc;
        }
#pragma unroll
        for (int j = 0; j < P; ++j) { l[j] = ln[j]; uc[j] = un1[j]; un1[j] = un2[j]; }
    }
#pragma unroll
    for (int c = 0; c < P / V; ++c) {
        int4 q;
        T *e = reinterpret_cast<T *>(&q);
#pragma unroll
        for (int k = 0; k < V; ++k) e[k] = l[c * V + k];
        *reinterpret_cast<int4 *>(lam + off + c * V) = q;
    }
}

// P consecutive points per thread, N/P threads (<= 512): the smallest P that fits
int adjoint_resident_P(int64_t N, int esz) {
    const int V = 16 / esz;
    for (int P = (V > 4 ? V : 4); P * esz <= 128; P *= 2)      // four P-value arrays live in registers
        if (N % P == 0 && N / P <= 512 && N >= 2 * P) return P;
    return 0;
}

template <typename T, int P>
int launch_resident(const T *u0, const T *states, T *lam, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                    int64_t n_steps, int bc, cudaStream_t s) {
    const int nth = (int)(N / P);
    adjoint_resident_kernel<T, P><<<(unsigned)B, nth, (size_t)8 * nth * sizeof(T), s>>>(u0, states, lam, nu, dt, B, N,
                                                                                      1.0 / dx, n_steps, bc);
    return last_launch_status();
}

}  // namespace

template <typename T>
int launch_adjoint_steps(const T *u0, const T *states, T *lam, T *pong, int64_t B, int64_t N, double dx,
                         const T *nu, const T *dt, int64_t n_steps, int bc, cudaStream_t s) {
    switch (adjoint_resident_P(N, (int)sizeof(T))) {
        case 4: return launch_resident<T, 4>(u0, states, lam, B, N, dx, nu, dt, n_steps, bc, s);
        case 8: return launch_resident<T, 8>(u0, states, lam, B, N, dx, nu, dt, n_steps, bc, s);
        case 16: return launch_resident<T, 16>(u0, states, lam, B, N, dx, nu, dt, n_steps, bc, s);
        case 32:
            if (sizeof(T) == 4) return launch_resident<float, 32>((const float *)u0, (const float *)states, (float *)lam, B,
                                                                  N, dx, (const float *)nu, (const float *)dt, n_steps, bc, s);
            break;
    }
    if (B > 65535) return BURGERS_ERR_SHAPE;
    dim3 grid((unsigned)((N + 255) / 256), (unsigned)B);
    T *cur = lam, *nxt = pong;
    for (int64_t n = n_steps - 1; n >= 0; --n) {
        const T *un = (n == 0) ? u0 : states + (size_t)(n - 1) * (size_t)B * (size_t)N;
        adjoint_step_kernel<T><<<grid, 256, 0, s>>>(un, cur, nxt, nu, dt, N, 1.0 / dx, bc);
        T *tmp = cur; cur = nxt; nxt = tmp;
    }
    int st = last_launch_status();
    if (st != BURGERS_OK) return st;
    if (cur != lam &&
        cudaMemcpyAsync(lam, cur, (size_t)B * N * sizeof(T), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
        return BURGERS_ERR_CUDA;
    return BURGERS_OK;
}

template int launch_adjoint_steps<float>(const float *, const float *, float *, float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, cudaStream_t);
template int launch_adjoint_steps<double>(const double *, const double *, double *, double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, cudaStream_t);

}  // namespace burgers
