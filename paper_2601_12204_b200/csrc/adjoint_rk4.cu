// adjoint_rk4.cu -- discrete adjoint of the classical RK4 scheme (D14, VERDICT r01
// item 8; PAPER.md:224-229 Eq.22, gradients of "the numerical solution" PAPER.md:231, :261).
//
// One forward step, K_s = dt F(y_s):  y1 = u, y2 = u + K1/2, y3 = u + K2/2, y4 = u + K3,
// u' = u + (K1 + 2 K2 + 2 K3 + K4)/6.  With G_s = dt dF/dy(y_s) (upwind switch held fixed) reverse mode gives,
// for lam' = dJ/du',
//     t4 = G4^T (lam'/6),  t3 = G3^T (lam'/3 + t4),  t2 = G2^T (lam'/3 + t3/2),  t1 = G1^T (lam'/6 + t2/2),
//     lam = lam' + t4 + t3 + t2 + t1.
// Rows of G (cx = dt/dx, rr = nu dt/dx^2; D2), on columns (i-1, i, i+1):
//     C_i = rr + cx max(y_i, 0),   D_i = -cx (|y_i| + g_i) - 2 rr,   A_i = rr - cx min(y_i, 0),
//     g_i = y_i - y_{i-1} if y_i > 0 else y_{i+1} - y_i;   Dirichlet end nodes: zero rows (K = 0 there).
// Column j, gathered:  (G^T v)_j = A_{j-1} v_{j-1} + D_j v_j + C_{j+1} v_{j+1}.
//
// The forward states u^0 .. u^{n-1} come from the trajectory output of the explicit RK4 kernel (one snapshot per
// step, checkpointed like the Euler adjoint, api.cu).  Backward sweep, two plans: RESIDENT (N = P x threads, below)
// and STREAMING (any N): per step three launches rebuild the stage
// values y2, y3, y4 from the stored u^n (the same arithmetic the forward kernel uses, unscaled) and four launches
// apply the transposed stage Jacobians; every launch is one pass over [B][N] (any N), the stage values and the two
// t arrays live in the workspace (5 B N elements), which stays L2-resident for the batch sizes this is used at.
#include "common.cuh"

namespace burgers {
namespace {

template <typename T>
struct Consts {
    T cx, rr;
    __device__ __forceinline__ Consts(const T *nu, const T *dt, int64_t b, double inv_dx) {
        const double dtb = (double)dt[b];
        cx = (T)(dtb * inv_dx);
        rr = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    }
};

// yout = u + coef * dt F(yin)   (Dirichlet end nodes: K = 0)
template <typename T>
__global__ void __launch_bounds__(256)
rk4_stage_kernel(const T *__restrict__ u, const T *__restrict__ yin, T *__restrict__ yout, const T *__restrict__ nu,
                 const T *__restrict__ dt, int64_t N, double inv_dx, int bc, T coef) {
    const int64_t b = blockIdx.y, j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const Consts<T> k(nu, dt, b, inv_dx);
    const T *y = yin + b * N;
    const bool fixed = (bc == BURGERS_BC_DIRICHLET) && (j == 0 || j == N - 1);
    const int64_t jm = (j == 0) ? N - 1 : j - 1, jp = (j == N - 1) ? 0 : j + 1;
    const T ym = y[jm], yj = y[j], yp = y[jp];
    const T dm = yj - ym, dp = yp - yj;
    const T g = (yj > T(0)) ? dm : dp;
    const T K = fixed ? T(0) : fma(-k.cx, yj * g, k.rr * (dp - dm));
    yout[b * N + j] = fma(coef, K, u[b * N + j]);
}

// v = ca * lam + cb * tprev (tprev may be null: cb ignored);  tout = G(y)^T v;  acc (+)= tout, acc = lam + tout when first
template <typename T>
__global__ void __launch_bounds__(256)
rk4_jacT_kernel(const T *__restrict__ ys, const T *__restrict__ lam, const T *__restrict__ tprev, T *__restrict__ tout,
                T *__restrict__ acc, const T *__restrict__ nu, const T *__restrict__ dt, int64_t N, double inv_dx, int bc,
                T ca, T cb, int first) {
    const int64_t b = blockIdx.y, j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const Consts<T> k(nu, dt, b, inv_dx);
    const T *y = ys + b * N, *l = lam + b * N;
    const T *tp = tprev ? tprev + b * N : nullptr;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t jm = (j == 0) ? N - 1 : j - 1, jp = (j == N - 1) ? 0 : j + 1;
    auto v = [&](int64_t i) { return tp ? fma(cb, tp[i], ca * l[i]) : ca * l[i]; };
    auto frozen = [&](int64_t i) { return dirichlet && (i == 0 || i == N - 1); };
    const T ym = y[jm], yj = y[j], yp = y[jp];
    T out = T(0);
    if (!frozen(j)) {                            // row j, diagonal entry D_j
        const T g = (yj > T(0)) ? (yj - ym) : (yp - yj);
        out = -(k.cx * (fabs(yj) + g) + T(2) * k.rr) * v(j);
    }
    if (!frozen(jm)) out = fma(k.rr - k.cx * fmin(ym, T(0)), v(jm), out);      // row j-1, entry A_{j-1}
    if (!frozen(jp)) out = fma(k.rr + k.cx * fmax(yp, T(0)), v(jp), out);      // row j+1, entry C_{j+1}
    // (periodic N >= 3: jm, j, jp are distinct rows.  Dirichlet: the wrap neighbours of the end nodes are frozen rows.)
    tout[b * N + j] = out;
    acc[b * N + j] = (first ? l[j] : acc[b * N + j]) + out;
}


// ---- RESIDENT backward sweep: one CTA per trajectory, P consecutive points per thread, lam in registers for all
// steps; per step the stored u^n is streamed in (one step ahead), the stage values are rebuilt on chip and the four
// transposed stage Jacobians applied, with eight halo exchanges (first / last values of y_s resp. v_s of every thread
// through a double-buffered shared edge array, one barrier each).  HBM traffic: sizeof(T) per point and step.
template <typename T, int P>
__global__ void __launch_bounds__(512)
adjoint_rk4_resident_kernel(const T *__restrict__ start, const T *__restrict__ states, T *__restrict__ lam,
                            const T *__restrict__ nu, const T *__restrict__ dt, int64_t B, int64_t N, double inv_dx,
                            int64_t len, int bc) {
    constexpr int V = 16 / sizeof(T);
    static_assert(P % V == 0, "a thread row must be a whole number of 16-byte vectors");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *edge = reinterpret_cast<T *>(smem_raw);          // [2][4][nth]
    const int t = threadIdx.x, nth = blockDim.x;
    const int64_t b = blockIdx.x;
    const Consts<T> k(nu, dt, b, inv_dx);
    const T cx = k.cx, rr = k.rr, two_rr = T(2) * k.rr;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const bool fixF = dirichlet && t == 0, fixL = dirichlet && t == nth - 1;
    const int64_t off = b * N + (int64_t)t * P, BN = B * N;
    const int tl = (t == 0) ? nth - 1 : t - 1, tr = (t == nth - 1) ? 0 : t + 1;
    auto load = [&](const T *src, T (&dst)[P]) {
#pragma unroll
        for (int c = 0; c < P / V; ++c) {
            const int4 q = *reinterpret_cast<const int4 *>(src + off + c * V);
            const T *e = reinterpret_cast<const T *>(&q);
#pragma unroll
            for (int kk = 0; kk < V; ++kk) dst[c * V + kk] = e[kk];
        }
    };
    auto state = [&](int64_t n) { return (n == 0) ? start : states + (size_t)(n - 1) * (size_t)BN; };
    int buf = 0;
    // neighbours' values: aL = last `a` of the left thread, aR = first `a` of the right thread (same for b)
    auto exchange = [&](T a0, T a1, T b0, T b1, T &aL, T &aR, T &bL, T &bR) {
        T *e = edge + buf * 4 * nth;
        e[t] = a0; e[nth + t] = a1; e[2 * nth + t] = b0; e[3 * nth + t] = b1;
        __syncthreads();
        aL = e[nth + tl]; aR = e[tr]; bL = e[3 * nth + tl]; bR = e[2 * nth + tr];
        buf ^= 1;
    };
    auto frozen = [&](int j) { return (j == 0 && fixF) || (j == P - 1 && fixL); };
    // yout = u + coef * dt F(y) with the halo (yL, yR) of y
    auto stage = [&](const T (&u)[P], const T (&y)[P], T yL, T yR, T coef, T (&yout)[P]) {
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const T ym = j ? y[j - 1] : yL, yj = y[j], yp = (j < P - 1) ? y[j + 1] : yR;
            const T dm = yj - ym, dp = yp - yj;
            const T g = (yj > T(0)) ? dm : dp;
            const T K = frozen(j) ? T(0) : fma(-cx, yj * g, rr * (dp - dm));
            yout[j] = fma(coef, K, u[j]);
        }
    };
    // tt = G(y)^T v with the halos of y and v; rows of frozen nodes are zero
    auto jacT = [&](const T (&y)[P], T yL, T yR, const T (&v)[P], T vL, T vR, T (&tt)[P]) {
        // the halo rows belong to the neighbouring threads: frozen iff that thread holds a Dirichlet end there
        const bool frozL = dirichlet && (t == 0);           // left neighbour of row 0 is row N-1 (frozen) when t == 0
        const bool frozR = dirichlet && (t == nth - 1);     // right neighbour of row P-1 is row 0 (frozen) when t == nth-1
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const T ym = j ? y[j - 1] : yL, yj = y[j], yp = (j < P - 1) ? y[j + 1] : yR;
            const T vm = j ? v[j - 1] : vL, vp = (j < P - 1) ? v[j + 1] : vR;
            T out = T(0);
            if (!frozen(j)) {
                const T g = (yj > T(0)) ? (yj - ym) : (yp - yj);
                out = -(cx * (fabs(yj) + g) + two_rr) * v[j];
            }
            const bool fm = j ? frozen(j - 1) : frozL, fp = (j < P - 1) ? frozen(j + 1) : frozR;
            if (!fm) out = fma(rr - cx * fmin(ym, T(0)), vm, out);       // A_{j-1}
            if (!fp) out = fma(rr + cx * fmax(yp, T(0)), vp, out);       // C_{j+1}
            tt[j] = out;
        }
    };
    const T sixth = T(1) / T(6), third = T(1) / T(3), half = T(0.5);
    T l[P], u[P], un1[P];
    load(lam, l);
    load(state(len - 1), u);
    for (int64_t n = len - 1; n >= 0; --n) {
        if (n > 0) load(state(n - 1), un1);               // prefetch the state of the next (earlier) step
        T y2[P], y3[P], y4[P], v[P], tt[P], acc[P];
        T uL, uR, y2L, y2R, y3L, y3R, y4L, y4R, vL, vR, d0, d1;
        exchange(u[0], u[P - 1], T(0), T(0), uL, uR, d0, d1);
        stage(u, u, uL, uR, half, y2);
        exchange(y2[0], y2[P - 1], T(0), T(0), y2L, y2R, d0, d1);
        stage(u, y2, y2L, y2R, half, y3);
        exchange(y3[0], y3[P - 1], T(0), T(0), y3L, y3R, d0, d1);
        stage(u, y3, y3L, y3R, T(1), y4);
#pragma unroll
        for (int j = 0; j < P; ++j) v[j] = sixth * l[j];
        exchange(y4[0], y4[P - 1], v[0], v[P - 1], y4L, y4R, vL, vR);
        jacT(y4, y4L, y4R, v, vL, vR, tt);                                  // t4
#pragma unroll
        for (int j = 0; j < P; ++j) { acc[j] = l[j] + tt[j]; v[j] = fma(T(1), tt[j], third * l[j]); }
        exchange(v[0], v[P - 1], T(0), T(0), vL, vR, d0, d1);
        jacT(y3, y3L, y3R, v, vL, vR, tt);                                  // t3
#pragma unroll
        for (int j = 0; j < P; ++j) { acc[j] += tt[j]; v[j] = fma(half, tt[j], third * l[j]); }
        exchange(v[0], v[P - 1], T(0), T(0), vL, vR, d0, d1);
        jacT(y2, y2L, y2R, v, vL, vR, tt);                                  // t2
#pragma unroll
        for (int j = 0; j < P; ++j) { acc[j] += tt[j]; v[j] = fma(half, tt[j], sixth * l[j]); }
        exchange(v[0], v[P - 1], T(0), T(0), vL, vR, d0, d1);
        jacT(u, uL, uR, v, vL, vR, tt);                                     // t1
#pragma unroll
        for (int j = 0; j < P; ++j) { l[j] = acc[j] + tt[j]; u[j] = un1[j]; }
    }
#pragma unroll
    for (int c = 0; c < P / V; ++c) {
        int4 q;
        T *e = reinterpret_cast<T *>(&q);
#pragma unroll
        for (int kk = 0; kk < V; ++kk) e[kk] = l[c * V + kk];
        *reinterpret_cast<int4 *>(lam + off + c * V) = q;
    }
}

// resident when N = P * threads with P = 8 (fp32) / 4 (fp64) and at most 512 threads
template <typename T> constexpr int rk4_resident_P() { return sizeof(T) == 4 ? 8 : 4; }
template <typename T>
bool rk4_resident_fits(int64_t N) {
    constexpr int P = rk4_resident_P<T>();
    return N % P == 0 && N / P <= 512 && N / P >= 2;
}

}  // namespace

size_t adjoint_rk4_ws_elems(int64_t B, int64_t N) { return (size_t)6 * (size_t)B * (size_t)N; }

// lam <- (du^{n0+len}/du^{n0})^T lam over `len` RK4 steps whose start states are start (step 0) and states[k-1]
// (step k).  ws: 6 B N elements.
template <typename T>
int launch_adjoint_rk4_steps(const T *start, const T *states, T *lam, T *ws, int64_t B, int64_t N, double dx, const T *nu,
                             const T *dt, int64_t len, int bc, cudaStream_t s) {
    if (len > 0 && rk4_resident_fits<T>(N) && B <= 0x7fffffffLL) {
        constexpr int P = rk4_resident_P<T>();
        const int nth = (int)(N / P);
        adjoint_rk4_resident_kernel<T, P><<<(unsigned)B, nth, (size_t)8 * nth * sizeof(T), s>>>(start, states, lam, nu, dt, B,
                                                                                             N, 1.0 / dx, len, bc);
        return last_launch_status();
    }
    if (B > 65535) return BURGERS_ERR_SHAPE;
    const size_t BN = (size_t)B * (size_t)N;
    T *y2 = ws, *y3 = ws + BN, *y4 = ws + 2 * BN, *ta = ws + 3 * BN, *tb = ws + 4 * BN, *acc = ws + 5 * BN;
    const dim3 grid((unsigned)((N + 255) / 256), (unsigned)B);
    const double inv_dx = 1.0 / dx;
    const T sixth = T(1) / T(6), third = T(1) / T(3), half = T(0.5);
    for (int64_t n = len - 1; n >= 0; --n) {
        const T *u = (n == 0) ? start : states + (size_t)(n - 1) * BN;
        rk4_stage_kernel<T><<<grid, 256, 0, s>>>(u, u, y2, nu, dt, N, inv_dx, bc, half);
        rk4_stage_kernel<T><<<grid, 256, 0, s>>>(u, y2, y3, nu, dt, N, inv_dx, bc, half);
        rk4_stage_kernel<T><<<grid, 256, 0, s>>>(u, y3, y4, nu, dt, N, inv_dx, bc, T(1));
        rk4_jacT_kernel<T><<<grid, 256, 0, s>>>(y4, lam, (const T *)nullptr, ta, acc, nu, dt, N, inv_dx, bc, sixth, T(0), 1);
        rk4_jacT_kernel<T><<<grid, 256, 0, s>>>(y3, lam, ta, tb, acc, nu, dt, N, inv_dx, bc, third, T(1), 0);
        rk4_jacT_kernel<T><<<grid, 256, 0, s>>>(y2, lam, tb, ta, acc, nu, dt, N, inv_dx, bc, third, half, 0);
        rk4_jacT_kernel<T><<<grid, 256, 0, s>>>(u, lam, ta, tb, acc, nu, dt, N, inv_dx, bc, sixth, half, 0);
        int st = last_launch_status();
        if (st != BURGERS_OK) return st;
        if (cudaMemcpyAsync(lam, acc, BN * sizeof(T), cudaMemcpyDeviceToDevice, s) != cudaSuccess) return BURGERS_ERR_CUDA;
    }
    return BURGERS_OK;
}

template int launch_adjoint_rk4_steps<float>(const float *, const float *, float *, float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, cudaStream_t);
template int launch_adjoint_rk4_steps<double>(const double *, const double *, double *, double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, cudaStream_t);

}  // namespace burgers
