// btcs_common.cuh -- device helpers shared by the BTCS kernels (btcs_hybrid.cu, btcs_long.cu):
// kernel (2) "fused BTCS assembly" and the per-thread partition elimination of kernel (4).
//
// BTCS rows (D4; Eq.23 with the convective coefficient lagged
// at u^n): with c = u dt/dx, r = nu dt/dx^2,
//     sub a = -r - max(c,0),   diag b = 1 + 2r + |c|,   sup e = -r + min(c,0),   rhs d = u.
// All three coefficients are functions of the ONE loaded value u_i^n: they are recomputed in
// registers and never stored.  b - |a| - |e| = 1 for every dt, nu >= 0 and u (strict diagonal
// dominance), so no elimination below needs pivoting.
//
// Partition elimination (one thread owns P consecutive rows 0..P-1 of its system):
//   forward  (rows 1..P-1):  f_j x_0 + x_j + c_j x_{j+1} = q_j          [normalised, diag = 1]
//   backward (rows P-3..1, scalars only):  row 1 as  F x_0 + x_1 + G x_{P-1} = R, which turns the
//   thread's row 0 into an equation in (x_{-1}, x_0, x_{P-1}).  The thread's two INTERFACE rows
//       first:  A x_{-1} + x_0 + C x_{P-1} = D         last:  f x_0 + x_{P-1} + c x_P = q
//   (x_{-1} / x_P = last / first unknown of the neighbouring threads) form, over all threads, a
//   tridiagonal system of 2 rows per thread that the callers solve by parallel cyclic reduction.
//   Back substitution, once x_0 and x_{P-1} are known:  x_j = q_j - f_j x_0 - c_j x_{j+1}.
#pragma once
#include "common.cuh"

namespace burgers {
namespace btcs {

// PCR early-exit threshold: once every off-diagonal of the (normalised) reduced rows is below
// this, the remaining levels cannot change a bit of the answer.
template <typename T> struct Lim;
template <> struct Lim<double> { static __device__ __forceinline__ double tiny() { return 8.470329472543003e-22; } };  // 2^-70
template <> struct Lim<float> { static __device__ __forceinline__ float tiny() { return 9.094947e-13f; } };          // 2^-40

template <typename T> __device__ __forceinline__ T t_abs(T x);
template <> __device__ __forceinline__ float t_abs<float>(float x) { return fabsf(x); }
template <> __device__ __forceinline__ double t_abs<double>(double x) { return fabs(x); }
template <typename T> __device__ __forceinline__ T t_fma(T a, T b, T c);
template <> __device__ __forceinline__ float t_fma<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <> __device__ __forceinline__ double t_fma<double>(double a, double b, double c) { return fma(a, b, c); }

// Reciprocal of a pivot.  Every pivot of the eliminations here lies in a benign range (partition
// pivots are >= 1 by diagonal dominance, PCR pivots in (0, 1]), so the IEEE division's special-case
// handling (denormals, overflow: ~25 SASS instructions with a slow-path branch in fp64) buys
// nothing.  fp64: MUFU.RCP64H (measured on B200: relative error <= 2^-19.9) + ONE cubic Newton step
// y (1 + e + e^2), e = 1 - x y: error e^3 ~ 2^-60 before rounding, measured <= 1 ulp against the
// IEEE quotient over 2^28 arguments.  fp32: MUFU.RCP + one linear step.  NaN / Inf still propagate.
template <typename T> __device__ __forceinline__ T rcp(T x);
template <> __device__ __forceinline__ double rcp<double>(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    e = fma(e, e, e);
    return fma(y, e, y);
}
template <> __device__ __forceinline__ float rcp<float>(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    const float e = fmaf(-x, y, 1.0f);
    return fmaf(y, e, y);
}

// Rows of D4 from the one loaded value u, without compare/select: with ch = u dt/(2 dx),
//   max(c,0) = |ch| + ch,  min(c,0) = ch - |ch|,  |c| = 2|ch|     (c = 2 ch)
// so  a = (-r - |ch|) - ch,  e = (-r - |ch|) + ch,  b = (1 + 2r) + 2|ch|:  5 FP instructions (|.| is
// a free operand modifier).
template <typename T>
struct Coef {
    T nr, hcx, b0;  // nr = -r, hcx = dt/(2dx), b0 = 1 + 2r
    __device__ __forceinline__ void init(T nu, T dt, double inv_dx) {
        const double dtb = (double)dt;
        hcx = (T)(0.5 * dtb * inv_dx);
        const T r = (T)((double)nu * dtb * inv_dx * inv_dx);
        nr = -r;
        b0 = T(1) + T(2) * r;
    }
    __device__ __forceinline__ void at(T u, T &a, T &b, T &e) const {
        const T ch = u * hcx;
        const T t = nr - t_abs(ch);
        a = t - ch;
        e = t + ch;
        b = t_fma(T(2), t_abs(ch), b0);
    }
};

// One interface row  A x_prev + x + C x_next = D  (normalised).
template <typename T> struct Row { T A, C, D; };

// Assembly + partition elimination of P rows held in v[].  ident(j) == true makes row j the
// identity row x_j = v_j (Dirichlet end nodes, D5 written as part of the system; out-of-domain
// padding).  Outputs the forward-elimination coefficients f, c, q (entries 1..P-1) and the two
// interface rows.
template <typename T, int P, typename Ident>
__device__ __forceinline__ void eliminate(const T (&v)[P], const Coef<T> &co, Ident ident,
                                          T (&f)[P], T (&c)[P], T (&q)[P], Row<T> &first,
                                          Row<T> &last) {
    static_assert(P >= 3, "a partition needs at least 3 rows");
    T a0, b0, e0;
    co.at(v[0], a0, b0, e0);
    if (ident(0)) { a0 = T(0); b0 = T(1); e0 = T(0); }
    {
        T a, b, e;
        co.at(v[1], a, b, e);
        if (ident(1)) { a = T(0); b = T(1); e = T(0); }
        const T m = rcp(b);
        f[1] = a * m; c[1] = e * m; q[1] = v[1] * m;
    }
#pragma unroll
    for (int j = 2; j < P; ++j) {
        T a, b, e;
        co.at(v[j], a, b, e);
        if (ident(j)) { a = T(0); b = T(1); e = T(0); }
        const T m = rcp(t_fma(-a, c[j - 1], b));
        const T am = a * m;
        f[j] = -am * f[j - 1];
        c[j] = e * m;
        q[j] = t_fma(-am, q[j - 1], v[j] * m);
    }
    // backward recurrence (scalars): row 1 as F x_0 + x_1 + G x_{P-1} = R
    T F = f[P - 2], G = c[P - 2], R = q[P - 2];
#pragma unroll
    for (int j = P - 3; j >= 1; --j) {
        F = t_fma(-c[j], F, f[j]);
        G = -c[j] * G;
        R = t_fma(-c[j], R, q[j]);
    }
    const T m = rcp(t_fma(-e0, F, b0));
    first.A = a0 * m;
    first.C = -e0 * G * m;
    first.D = t_fma(-e0, R, v[0]) * m;
    last.A = f[P - 1];
    last.C = c[P - 1];
    last.D = q[P - 1];
}

// The same partition elimination for GENERAL rows (newton.cu): rowfn(j, a, b, e) yields sub / diag /
// sup of row j; q[] holds the right-hand sides on entry and the eliminated ones on exit.
template <typename T, int P, typename RowFn>
__device__ __forceinline__ void eliminate_general(RowFn rowfn, T (&q)[P], T (&f)[P], T (&c)[P],
                                                  Row<T> &first, Row<T> &last) {
    static_assert(P >= 3, "a partition needs at least 3 rows");
    T a0, b0, e0;
    rowfn(0, a0, b0, e0);
    const T d0 = q[0];
    {
        T a, b, e;
        rowfn(1, a, b, e);
        const T m = rcp(b);
        f[1] = a * m; c[1] = e * m; q[1] = q[1] * m;
    }
#pragma unroll
    for (int j = 2; j < P; ++j) {
        T a, b, e;
        rowfn(j, a, b, e);
        const T m = rcp(t_fma(-a, c[j - 1], b));
        const T am = a * m;
        f[j] = -am * f[j - 1];
        c[j] = e * m;
        q[j] = t_fma(-am, q[j - 1], q[j] * m);
    }
    T F = f[P - 2], G = c[P - 2], R = q[P - 2];
#pragma unroll
    for (int j = P - 3; j >= 1; --j) {
        F = t_fma(-c[j], F, f[j]);
        G = -c[j] * G;
        R = t_fma(-c[j], R, q[j]);
    }
    const T m = rcp(t_fma(-e0, F, b0));
    first.A = a0 * m;
    first.C = -e0 * G * m;
    first.D = t_fma(-e0, R, d0) * m;
    last.A = f[P - 1];
    last.C = c[P - 1];
    last.D = q[P - 1];
}

// ---- RAGGED partitions: any N on a power-of-two number of threads ---------------------------------
// The interface solve needs a power-of-two ring of threads, the grid length N is whatever the caller
// has ("any N >= 3 must work"; the paper's own grid is N = 201).  Padding
// the chain with identity rows would cut a periodic ring open, so instead the N rows are dealt out
// UNEVENLY: with q = N / Tn and rem = N - q Tn, thread t owns the n = q + (t < rem) consecutive rows
// starting at r0 = t q + min(t, rem), held in the first n of its P register slots (3 <= n <= P).  Every
// row is a real row, the ring of interface rows stays cyclic, and the per-slot work of the unrolled
// loops is skipped by early exits (n differs by at most one inside a warp).
struct Part { int r0, n; };
__device__ __forceinline__ Part partition_of(int t, int N, int Tn) {
    const int q = N / Tn, rem = N - q * Tn;
    Part p;
    p.n = q + (t < rem ? 1 : 0);
    p.r0 = t * q + (t < rem ? t : rem);
    return p;
}

// eliminate_general for a partition of n <= P rows (slots n..P-1 unused).
template <typename T, int P, typename RowFn>
__device__ __forceinline__ void eliminate_general_ragged(RowFn rowfn, int n, T (&q)[P], T (&f)[P], T (&c)[P],
                                                         Row<T> &first, Row<T> &last) {
    static_assert(P >= 3, "a partition needs at least 3 rows");
    T a0, b0, e0;
    rowfn(0, a0, b0, e0);
    const T d0 = q[0];
    {
        T a, b, e;
        rowfn(1, a, b, e);
        const T m = rcp(b);
        f[1] = a * m; c[1] = e * m; q[1] = q[1] * m;
    }
#pragma unroll
    for (int j = 2; j < P; ++j) {
        if (j < n) {
            T a, b, e;
            rowfn(j, a, b, e);
            const T m = rcp(t_fma(-a, c[j - 1], b));
            const T am = a * m;
            f[j] = -am * f[j - 1];
            c[j] = e * m;
            q[j] = t_fma(-am, q[j - 1], q[j] * m);
            // (every executed iteration overwrites `last`; the one that sticks is j = n - 1.  No test
            // "j == n - 1" here or below: the compiler would turn f[j] into f[n - 1], a run-time index
            // that sends the arrays to local memory)
            last.A = f[j]; last.C = c[j]; last.D = q[j];
        }
    }
    // backward recurrence from j = n - 2: started from (0, -1, 0), its first executed step yields
    // (f_j, c_j, q_j) exactly
    T F = T(0), G = T(-1), R = T(0);
#pragma unroll
    for (int j = P - 2; j >= 1; --j) {
        if (j <= n - 2) {
            F = t_fma(-c[j], F, f[j]);
            G = -c[j] * G;
            R = t_fma(-c[j], R, q[j]);
        }
    }
    const T m = rcp(t_fma(-e0, F, b0));
    first.A = a0 * m;
    first.C = -e0 * G * m;
    first.D = t_fma(-e0, R, d0) * m;
}

// back_substitute for a partition of n <= P rows: x0 = x_0, xl = x_{n-1}.
template <typename T, int P>
__device__ __forceinline__ void back_substitute_ragged(T (&v)[P], int n, const T (&f)[P], const T (&c)[P],
                                                       const T (&q)[P], T x0, T xl) {
    T xn = xl;
#pragma unroll
    for (int j = P - 1; j >= 1; --j) {
        if (j < n - 1) {
            xn = t_fma(-c[j], xn, t_fma(-f[j], x0, q[j]));
            v[j] = xn;
        } else {
            v[j] = xl;         // slot n - 1 (and the unused slots behind it)
        }
    }
    v[0] = x0;
}

// Host side: geometry of one CTA per system for N rows: Tn threads (a power of two >= 2) and P register slots
// per thread, given max_threads(P), the thread limit of the kernel's P-slot instance.
//   exact  (N == P Tn, P in {16, 8, 4}): every slot used, 128-bit loads; the largest P that still fills a warp,
//          otherwise the most threads;
//   ragged (any other N): P = ceil(N / Tn) in [4, 16], so that every thread owns P - 1 or P rows (the kernels
//          tell the compiler so, and only the last slot is conditional); the fewest threads (largest P) that
//          still fill a warp, otherwise the most threads with P >= 4.
template <typename MaxThreads>
inline bool pick_partition(int64_t N, MaxThreads max_threads, int *P_out, int *T_out, bool *ragged) {
    const int cand[3] = {16, 8, 4};
    int bestP = 0, bestT = 0;
    for (int i = 0; i < 3; ++i) {
        const int P = cand[i];
        if (N % P) continue;
        const int64_t Tn = N / P;
        if (Tn < 2 || (Tn & (Tn - 1)) || Tn > max_threads(P)) continue;
        if (Tn >= 32) { bestP = P; bestT = (int)Tn; break; }
        bestP = P; bestT = (int)Tn;
    }
    if (bestP) { *P_out = bestP; *T_out = bestT; *ragged = false; return true; }
    for (int64_t Tn = 2; Tn <= 1024; Tn *= 2) {
        const int64_t P = (N + Tn - 1) / Tn;
        if (P > 16) continue;                 // too few threads for 16 slots
        if (P < 4) break;                     // (and every larger Tn) partitions shorter than 3 rows
        if (Tn > max_threads((int)P)) break;
        bestP = (int)P; bestT = (int)Tn;
        if (Tn >= 32) break;
    }
    if (!bestP) return false;
    *P_out = bestP; *T_out = bestT; *ragged = true;
    return true;
}

// Solve the cyclic interface system of one CTA (Tn = blockDim.x threads, a power of two >= 2) given
// every thread's two interface rows: one cyclic-reduction step (one reduced row per thread in the
// unknowns x_L), parallel cyclic reduction with early exit, exact 2x2 ending; returns this thread's
// x_0 and x_L.  smem: sR = two buffers of Tn rows (A, C, D) each (PCR ping-pong), sF = Tn rows.  The rows
// are stored as (A, C, D) triples -- ONE address per neighbour row, its three values at immediate offsets,
// and 24-byte (fp64) / 12-byte strides are conflict-free for 64- / 32-bit shared loads: with a run-time Tn
// the three-array layout spent 50 of the 64 instructions of a PCR level on address arithmetic, and these
// kernels are bound by issue slots (c3_newton 54.0 -> 49.6 ms).
// Contains CTA barriers: call from uniform control flow.
// TN: the thread count when it is known at compile time (the PCR levels are unrolled), else 0.
template <typename T, int TN = 0>
__device__ __forceinline__ void solve_interface(const Row<T> &first, const Row<T> &last, T *sR, T *sF,
                                                T &x0, T &xL, const int t, const int Tn_rt) {
    const int Tn = TN ? TN : Tn_rt;
    const int mask = Tn - 1;
    {
        T *mine = sF + 3 * t;
        mine[0] = first.A; mine[1] = first.C; mine[2] = first.D;
    }
    __syncthreads();
    Row<T> r;
    {
        const T *nx = sF + 3 * ((t + 1) & mask);
        const T nA = nx[0], nC = nx[1], nD = nx[2];
        const T m = rcp(t_fma(-last.A, first.C, t_fma(-last.C, nA, T(1))));
        r.A = -last.A * first.A * m;
        r.C = -last.C * nC * m;
        r.D = t_fma(-last.A, first.D, t_fma(-last.C, nD, last.D)) * m;
    }
    T *rd = sR, *wr = sR + 3 * Tn;          // the buffer the next level reads / writes
    {
        T *mine = rd + 3 * t;
        mine[0] = r.A; mine[1] = r.C; mine[2] = r.D;
    }
    __syncthreads();
    bool finished = false;
#pragma unroll
    for (int s = 1; s < Tn / 2; s <<= 1) {
        const T *pm = rd + 3 * ((t - s) & mask), *pp = rd + 3 * ((t + s) & mask);
        Row<T> rm, rp;
        rm.A = pm[0]; rm.C = pm[1]; rm.D = pm[2];
        rp.A = pp[0]; rp.C = pp[1]; rp.D = pp[2];
        r = pcr_combine(r, rm, rp);
        T *mine = wr + 3 * t;
        mine[0] = r.A; mine[1] = r.C; mine[2] = r.D;
        T *tmp = rd; rd = wr; wr = tmp;
        if (s >= 4) {       // the vote starts at the third level (see btcs_hybrid.cu)
            const int flag = !((t_abs(r.A) <= Lim<T>::tiny()) & (t_abs(r.C) <= Lim<T>::tiny()));
            if (!__syncthreads_or(flag)) { finished = true; break; }
        } else {
            __syncthreads();
        }
    }
    T xLprev;
    xL = r.D;
    if (finished) {
        xLprev = rd[3 * ((t - 1) & mask) + 2];
    } else {  // rows t and t + Tn/2 couple only to each other: exact 2x2 solve
        const T *po = rd + 3 * ((t + Tn / 2) & mask);
        const T p1 = r.A + r.C, p2 = po[0] + po[1];
        const T D2 = po[2];
        xL = t_fma(-p1, D2, r.D) * rcp(t_fma(-p1, p2, T(1)));
        wr[3 * t + 2] = xL;                 // the other PCR buffer is free; the next write to it follows a barrier
        __syncthreads();
        xLprev = wr[3 * ((t - 1) & mask) + 2];
    }
    x0 = t_fma(-first.A, xLprev, t_fma(-first.C, xL, first.D));
}

// Back substitution into v[] given the partition's end unknowns x0 = x_0, xl = x_{P-1}.
template <typename T, int P>
__device__ __forceinline__ void back_substitute(T (&v)[P], const T (&f)[P], const T (&c)[P],
                                                const T (&q)[P], T x0, T xl) {
    v[0] = x0; v[P - 1] = xl;
    T xn = xl;
#pragma unroll
    for (int j = P - 2; j >= 1; --j) {
        xn = t_fma(-c[j], xn, t_fma(-f[j], x0, q[j]));
        v[j] = xn;
    }
}

// One PCR combination: row k with its neighbours km (k - s) and kp (k + s), all normalised.
template <typename T>
__device__ __forceinline__ Row<T> pcr_combine(const Row<T> &k, const Row<T> &km, const Row<T> &kp) {
    const T m = rcp(t_fma(-k.A, km.C, t_fma(-k.C, kp.A, T(1))));
    Row<T> n;
    n.A = -k.A * km.A * m;
    n.C = -k.C * kp.C * m;
    n.D = t_fma(-k.A, km.D, t_fma(-k.C, kp.D, k.D)) * m;
    return n;
}

constexpr int max_threads_for_regs(int regs) {
    int t = 1024;
    while (t > 32 && t * regs > 65536) t /= 2;
    return t;
}

}  // namespace btcs
}  // namespace burgers
