// btcs_long.cu -- kernels (2)+(4) for LONG systems: one (cyclic) tridiagonal system spread over
// many CTAs (BASELINE config 4b: N = 2^22, fp64, periodic).
//
// Per time step the system  A(u^n) u^{n+1} = u^n  (D4-D6; Eq.23)
// is solved exactly (to rounding) by partition elimination + parallel cyclic reduction, as in
// btcs_hybrid.cu, with the interface system now spanning CTAs.  Two device paths:
//
//  TILED (fast path, one launch per time step, ping-pong u <-> ws): every CTA owns W consecutive
//    points of one system and loads them with a halo of Hp points per side.  Its threads eliminate
//    their P-row partitions, and the CTA runs PCR on its 2*Tn interface rows as an OPEN chain (the
//    couplings leaving the tile are dropped).  The wrong rows at the two tile ends contaminate,
//    after j PCR levels, only the 2^j outermost rows; the matrix is strictly diagonally dominant,
//    so the off-diagonals of the reduced rows decay (quadratically per level) and the owned rows
//    are normally finished (all |A|,|C| < 2^-70 fp64 / 2^-40 fp32: x_k = D_k to the last bit)
//    before the contamination has crossed the halo.  The CTA CHECKS this: if after the J levels
//    the halo allows some owned row is not finished, it records the failing step in the status
//    word and every later TILED launch returns at once, leaving u^n of the failing step intact.
//  GENERAL (cooperative persistent kernel, exact for any coefficients): partitions eliminated by
//    all threads of the grid, interface rows in global memory (L2 resident), global PCR with one
//    grid-wide barrier per level and early exit as soon as every off-diagonal is below the
//    threshold (full depth ends in the exact 2x2 solve), then back substitution in place.  It is
//    enqueued after the TILED launches, reads the status word, and continues from the failing
//    step (or returns immediately when there was none) -- no host synchronisation anywhere.
#include <cooperative_groups.h>

#include "btcs_common.cuh"

namespace cg = cooperative_groups;

namespace burgers {
namespace {

using namespace btcs;

// ---- geometry (host + device agree through these constants) ---------------------------------
constexpr int kP = 8;          // rows per thread partition
constexpr int kTn = 256;       // threads per CTA of the TILED kernel (tile = kTn*kP points)
constexpr int kHaloT = 16;     // halo threads per side  (halo = kHaloT*kP = 128 points)
constexpr int kLevels = 5;     // PCR levels the halo allows: 2^kLevels == 2*kHaloT rows
constexpr int kW = (kTn - 2 * kHaloT) * kP;   // owned points per tile
constexpr int kGenThreads = 256;
constexpr int kStatusBytes = 1024;            // status word + 2 x 64 level flags
static_assert((1 << kLevels) == 2 * kHaloT, "levels must match the halo");

__device__ __forceinline__ int64_t wrap(int64_t g, int64_t N) {
    g %= N;
    return g < 0 ? g + N : g;
}

// ------------------------------------------------------------------------ TILED step kernel
template <typename T>
__global__ void __launch_bounds__(kTn, 2)
btcs_long_tiled_kernel(const T *__restrict__ src, T *__restrict__ dst, const T *__restrict__ nu,
                       const T *__restrict__ dt, int64_t N, int64_t tiles, double inv_dx, int bc,
                       int step, int *__restrict__ status) {
    constexpr int P = kP, Tn = kTn, M = 2 * kTn;
    constexpr int V = 16 / sizeof(T);
    __shared__ T sA[2][M], sC[2][M], sD[2][M];
    __shared__ int s_failed;
    const int t = threadIdx.x;
    if (t == 0) s_failed = *reinterpret_cast<volatile int *>(status);
    __syncthreads();
    if (s_failed != 0) return;            // an earlier step failed (uniform over the CTA)

    const int64_t b = blockIdx.x / tiles, tile = blockIdx.x % tiles;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t g0 = tile * kW + (int64_t)(t - kHaloT) * P;     // unwrapped index of row 0
    const T *srow = src + b * N;
    Coef<T> co;
    co.init(nu[b], dt[b], inv_dx);

    // ---- load the partition (periodic: wrap; Dirichlet: out-of-domain rows are x = 0)
    T v[P];
    const bool inside = (g0 >= 0 && g0 + P <= N);
    if ((N % V) == 0) {
#pragma unroll
        for (int c = 0; c < P / V; ++c) {
            int64_t g = g0 + c * V;
            bool ok = true;
            if (!inside) {
                if (dirichlet) ok = (g >= 0 && g < N);
                else g = wrap(g, N);
            }
            int4 q4 = make_int4(0, 0, 0, 0);
            if (ok) q4 = *reinterpret_cast<const int4 *>(srow + g);
            const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
            for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
        }
    } else {
#pragma unroll
        for (int j = 0; j < P; ++j) {
            int64_t g = g0 + j;
            bool ok = true;
            if (!inside) {
                if (dirichlet) ok = (g >= 0 && g < N);
                else g = wrap(g, N);
            }
            v[j] = ok ? srow[g] : T(0);
        }
    }

    // ---- assembly + partition elimination
    T f[P], c[P], q[P];
    Row<T> first, last;
    if (dirichlet && (g0 <= 0 || g0 + P >= N)) {
        eliminate<T, P>(v, co, [&](int j) { return g0 + j <= 0 || g0 + j >= N - 1; }, f, c, q, first, last);
    } else {
        eliminate<T, P>(v, co, [](int) { return false; }, f, c, q, first, last);
    }
    if (t == 0) first.A = T(0);          // open chain: drop the couplings leaving the tile
    if (t == Tn - 1) last.C = T(0);
    sA[0][2 * t] = first.A; sA[0][2 * t + 1] = last.A;
    sC[0][2 * t] = first.C; sC[0][2 * t + 1] = last.C;
    sD[0][2 * t] = first.D; sD[0][2 * t + 1] = last.D;
    __syncthreads();

    // ---- PCR on the open chain of M interface rows, at most kLevels levels
    int cur = 0;
    bool finished = false;
#pragma unroll 1
    for (int l = 0; l < kLevels; ++l) {
        const int s = 1 << l;
        int flag = 0;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int k = t + h * Tn;
            const int km = k - s, kp = k + s;
            Row<T> rk, rm, rp;
            rk.A = sA[cur][k]; rk.C = sC[cur][k]; rk.D = sD[cur][k];
            if (km >= 0) { rm.A = sA[cur][km]; rm.C = sC[cur][km]; rm.D = sD[cur][km]; }
            else { rm.A = T(0); rm.C = T(0); rm.D = T(0); }
            if (kp < M) { rp.A = sA[cur][kp]; rp.C = sC[cur][kp]; rp.D = sD[cur][kp]; }
            else { rp.A = T(0); rp.C = T(0); rp.D = T(0); }
            const Row<T> n = pcr_combine(rk, rm, rp);
            sA[cur ^ 1][k] = n.A; sC[cur ^ 1][k] = n.C; sD[cur ^ 1][k] = n.D;
            const bool owned = (k >= 2 * kHaloT) && (k < M - 2 * kHaloT);
            flag |= owned & ((t_abs(n.A) > Lim<T>::tiny()) | (t_abs(n.C) > Lim<T>::tiny()));
        }
        const int any = __syncthreads_or(flag);
        cur ^= 1;
        if (!any) { finished = true; break; }
    }
    if (!finished) {                       // the halo was too short for these coefficients
        if (t == 0) atomicCAS(status, 0, step + 1);
        return;
    }

    // ---- back substitution and store of the owned partitions
    const bool owned = (t >= kHaloT) && (t < Tn - kHaloT) && (g0 < N);
    if (!owned) return;
    back_substitute<T, P>(v, f, c, q, sD[cur][2 * t], sD[cur][2 * t + 1]);
    T *drow = dst + b * N;
    if ((N % V) == 0) {
#pragma unroll
        for (int cc = 0; cc < P / V; ++cc) {
            int4 q4;
            T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
            for (int k = 0; k < V; ++k) e[k] = v[cc * V + k];
            *reinterpret_cast<int4 *>(drow + g0 + cc * V) = q4;
        }
    } else {
#pragma unroll
        for (int j = 0; j < P; ++j) drow[g0 + j] = v[j];
    }
}

// After the TILED launches: move the newest valid state into u when it sits in ws.
//   no failure: u^{n_steps} is in ws iff n_steps is odd;  failure at step n: u^n is in ws iff n odd.
template <typename T>
__global__ void btcs_long_fixup_kernel(T *__restrict__ u, const T *__restrict__ ws, int64_t elems,
                                       int64_t n_steps, const int *__restrict__ status) {
    const int fail = *status;
    const int64_t n = fail ? (int64_t)(fail - 1) : n_steps;
    if ((n & 1) == 0) return;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < elems; i += stride) u[i] = ws[i];
}

// ------------------------------------------------------------------------ GENERAL kernel
template <typename T>
struct GenRows {   // interface rows in global memory, two buffers (PCR ping-pong)
    T *A[2], *C[2], *D[2];
};

template <typename T>
__device__ __forceinline__ void gen_load_partition(const T *__restrict__ u, int64_t N, int64_t part,
                                                   int64_t parts_per_sys, T (&v)[kP], int64_t &b,
                                                   int64_t &tt) {
    constexpr int V = 16 / sizeof(T);
    b = part / parts_per_sys;
    tt = part % parts_per_sys;
    const T *p = u + b * N + tt * kP;     // N % kP == 0: 16-byte aligned
#pragma unroll
    for (int c = 0; c < kP / V; ++c) {
        int4 q4 = __ldcg(reinterpret_cast<const int4 *>(p) + c);
        const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
        for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
    }
}

template <typename T>
__global__ void __launch_bounds__(kGenThreads)
btcs_long_general_kernel(T *__restrict__ u, const T *__restrict__ nu, const T *__restrict__ dt,
                         int64_t B, int64_t N, double inv_dx, int64_t n_steps, int bc, GenRows<T> R,
                         int *__restrict__ status, int force) {
    constexpr int P = kP;
    constexpr int V = 16 / sizeof(T);
    cg::grid_group grid = cg::this_grid();
    const int fail = force ? 1 : *reinterpret_cast<volatile int *>(status);
    if (fail == 0) return;                              // uniform over the grid
    int *flags = status + 64;                           // [2][32]
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t pps = N / P;                          // partitions per system
    const int64_t parts = B * pps;
    const int64_t M = 2 * pps;                          // interface rows per system (power of two)
    const int64_t rows = B * M;
    const int64_t gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t gthreads = (int64_t)gridDim.x * blockDim.x;

    for (int64_t step = fail - 1; step < n_steps; ++step) {
        const int par = (int)(step & 1);
        // ---- phase A: assembly + partition elimination, interface rows -> buffer 0
        for (int64_t part = gtid; part < parts; part += gthreads) {
            T v[P], f[P], c[P], q[P];
            int64_t b, tt;
            gen_load_partition<T>(u, N, part, pps, v, b, tt);
            Coef<T> co;
            co.init(nu[b], dt[b], inv_dx);
            const bool fixL = dirichlet && tt == 0, fixR = dirichlet && tt == pps - 1;
            Row<T> first, last;
            eliminate<T, P>(v, co, [&](int j) { return (j == 0 && fixL) || (j == P - 1 && fixR); },
                            f, c, q, first, last);
            const int64_t o = 2 * part;
            R.A[0][o] = first.A; R.A[0][o + 1] = last.A;
            R.C[0][o] = first.C; R.C[0][o + 1] = last.C;
            R.D[0][o] = first.D; R.D[0][o + 1] = last.D;
        }
        grid.sync();
        // every CTA has left step-1: its level flags (other parity) can be cleared for step+1
        if (blockIdx.x == 0 && threadIdx.x < 32) flags[(par ^ 1) * 32 + threadIdx.x] = 0;
        // ---- global PCR, one grid barrier per level, early exit
        int cur = 0;
        bool finished = false;
        int l = 0;
        for (int64_t s = 1; s < M / 2; s <<= 1, ++l) {
            int flag = 0;
            for (int64_t k = gtid; k < rows; k += gthreads) {
                const int64_t base = k & ~(M - 1), kk = k & (M - 1);
                const int64_t km = base + ((kk - s) & (M - 1)), kp = base + ((kk + s) & (M - 1));
                Row<T> rk, rm, rp;
                rk.A = __ldcg(R.A[cur] + k); rk.C = __ldcg(R.C[cur] + k); rk.D = __ldcg(R.D[cur] + k);
                rm.A = __ldcg(R.A[cur] + km); rm.C = __ldcg(R.C[cur] + km); rm.D = __ldcg(R.D[cur] + km);
                rp.A = __ldcg(R.A[cur] + kp); rp.C = __ldcg(R.C[cur] + kp); rp.D = __ldcg(R.D[cur] + kp);
                const Row<T> n = pcr_combine(rk, rm, rp);
                R.A[cur ^ 1][k] = n.A; R.C[cur ^ 1][k] = n.C; R.D[cur ^ 1][k] = n.D;
                flag |= (t_abs(n.A) > Lim<T>::tiny()) | (t_abs(n.C) > Lim<T>::tiny());
            }
            if (__syncthreads_or(flag) && threadIdx.x == 0) atomicOr(&flags[par * 32 + l], 1);
            grid.sync();
            cur ^= 1;
            if (*reinterpret_cast<volatile int *>(&flags[par * 32 + l]) == 0) { finished = true; break; }
        }
        if (!finished) {  // rows k and k + M/2 couple only to each other: exact 2x2 solve
            const int64_t half = M / 2;
            for (int64_t i = gtid; i < B * half; i += gthreads) {
                const int64_t k = (i / half) * M + (i % half), k2 = k + half;
                const T p1 = __ldcg(R.A[cur] + k) + __ldcg(R.C[cur] + k);
                const T p2 = __ldcg(R.A[cur] + k2) + __ldcg(R.C[cur] + k2);
                const T D1 = __ldcg(R.D[cur] + k), D2 = __ldcg(R.D[cur] + k2);
                const T m = rcp(t_fma(-p1, p2, T(1)));
                R.D[cur ^ 1][k] = t_fma(-p1, D2, D1) * m;
                R.D[cur ^ 1][k2] = t_fma(-p2, D1, D2) * m;
            }
            grid.sync();
            cur ^= 1;
        }
        // ---- phase C: redo the partition elimination, back substitution in place.  The next
        // step's phase A touches only this thread's own partitions and rows: no barrier needed.
        for (int64_t part = gtid; part < parts; part += gthreads) {
            T v[P], f[P], c[P], q[P];
            int64_t b, tt;
            gen_load_partition<T>(u, N, part, pps, v, b, tt);
            Coef<T> co;
            co.init(nu[b], dt[b], inv_dx);
            const bool fixL = dirichlet && tt == 0, fixR = dirichlet && tt == pps - 1;
            Row<T> first, last;
            eliminate<T, P>(v, co, [&](int j) { return (j == 0 && fixL) || (j == P - 1 && fixR); },
                            f, c, q, first, last);
            back_substitute<T, P>(v, f, c, q, __ldcg(R.D[cur] + 2 * part), __ldcg(R.D[cur] + 2 * part + 1));
            T *p = u + b * N + tt * P;
#pragma unroll
            for (int cc = 0; cc < P / V; ++cc) {
                int4 q4;
                T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
                for (int k = 0; k < V; ++k) e[k] = v[cc * V + k];
                *reinterpret_cast<int4 *>(p + cc * V) = q4;
            }
        }
    }
}

bool pow2(int64_t x) { return x > 0 && (x & (x - 1)) == 0; }

size_t row_elems(int64_t B, int64_t N) { return (size_t)B * (size_t)(2 * (N / kP)); }

}  // namespace

// LONG runs power-of-two grids of at least four tiles (shorter systems fit one CTA: HYBRID).
bool btcs_long_fits(int64_t N, int bc) {
    (void)bc;
    return pow2(N) && N >= 4 * (int64_t)kTn * kP;
}

// ws layout (elements of T): [B*N ping-pong state][6 x B*M interface rows] then kStatusBytes.
size_t btcs_long_ws_bytes(int esz, int64_t B, int64_t N) {
    const size_t state = ((size_t)B * (size_t)N * esz + 255) / 256 * 256;
    const size_t rows = (6 * row_elems(B, N) * esz + 255) / 256 * 256;
    return state + rows + kStatusBytes;
}

// memset + n_steps TILED + fixup + GENERAL (PLAN_LONG); GENERAL alone for PLAN_LONG_GENERAL
int64_t btcs_long_launch_count(int64_t n_steps, int general_only) {
    if (n_steps <= 0) return 0;
    return general_only ? 1 : n_steps + 2;
}

template <typename T>
int launch_btcs_long(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                     int64_t n_steps, int bc, void *ws, int general_only, cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    if (!btcs_long_fits(N, bc)) return BURGERS_ERR_PLAN;
    if (n_steps > 0x7ffffff0LL) return BURGERS_ERR_SHAPE;
    const size_t esz = sizeof(T);
    const size_t state_b = ((size_t)B * (size_t)N * esz + 255) / 256 * 256;
    const size_t rows_b = (6 * row_elems(B, N) * esz + 255) / 256 * 256;
    unsigned char *base = static_cast<unsigned char *>(ws);
    T *pong = reinterpret_cast<T *>(base);
    T *rows = reinterpret_cast<T *>(base + state_b);
    int *status = reinterpret_cast<int *>(base + state_b + rows_b);
    const double inv_dx = 1.0 / dx;
    if (cudaMemsetAsync(status, 0, kStatusBytes, s) != cudaSuccess) return BURGERS_ERR_CUDA;

    if (!general_only) {
        const int64_t tiles = (N + kW - 1) / kW;
        if (B * tiles > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
        T *cur = u, *nxt = pong;
        for (int64_t n = 0; n < n_steps; ++n) {
            btcs_long_tiled_kernel<T><<<(unsigned)(B * tiles), kTn, 0, s>>>(cur, nxt, nu, dt, N, tiles, inv_dx,
                                                                          bc, (int)n, status);
            T *tmp = cur; cur = nxt; nxt = tmp;
        }
        int st = last_launch_status();
        if (st != BURGERS_OK) return st;
        btcs_long_fixup_kernel<T><<<148 * 4, 256, 0, s>>>(u, pong, B * N, n_steps, status);
        st = last_launch_status();
        if (st != BURGERS_OK) return st;
    }

    // cooperative launch of the general kernel: the grid must be co-resident
    int dev = 0, sms = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, btcs_long_general_kernel<T>, kGenThreads, 0) !=
            cudaSuccess ||
        per_sm < 1)
        return BURGERS_ERR_CUDA;
    const int64_t want = (B * (N / kP) + kGenThreads - 1) / kGenThreads;
    int64_t grid = (int64_t)sms * per_sm;
    if (grid > want) grid = want;
    const size_t re = row_elems(B, N);
    GenRows<T> R;
    R.A[0] = rows;          R.C[0] = rows + re;     R.D[0] = rows + 2 * re;
    R.A[1] = rows + 3 * re; R.C[1] = rows + 4 * re; R.D[1] = rows + 5 * re;
    int force = general_only ? 1 : 0;
    void *args[] = {&u, &nu, &dt, &B, &N, (void *)&inv_dx, &n_steps, &bc, &R, &status, &force};
    if (cudaLaunchCooperativeKernel((const void *)btcs_long_general_kernel<T>, dim3((unsigned)grid),
                                    dim3(kGenThreads), args, 0, s) != cudaSuccess)
        return BURGERS_ERR_CUDA;
    return last_launch_status();
}

template int launch_btcs_long<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, void *, int, cudaStream_t);
template int launch_btcs_long<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, void *, int, cudaStream_t);

}  // namespace burgers
