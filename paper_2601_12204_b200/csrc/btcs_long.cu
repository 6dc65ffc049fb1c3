// btcs_long.cu -- kernels (2)+(4) for LONG systems: one (cyclic) tridiagonal system spread over
// many CTAs (BASELINE config 4b: N = 2^22, fp64, periodic).
//
// Per time step the system  A(u^n) u^{n+1} = u^n  (D4-D6; Eq.23)
// is solved exactly (to rounding) by partition elimination + parallel cyclic reduction, as in
// btcs_hybrid.cu, with the interface system now spanning CTAs.  Two device paths:
//
//  TILED (fast path, S = 1..6 time steps per launch, ping-pong u <-> ws): every tile of consecutive points of
//    one system is loaded with a halo of 8 S + 1 / 8 S threads (x kTP points) per side.
//    Its threads eliminate their kTP-row partitions, one in-CTA cyclic-reduction step leaves ONE
//    reduced row per thread, and the CTA runs PCR on these rows as an OPEN chain (the couplings
//    leaving the tile are dropped).  The wrong rows at the two tile ends contaminate, after j PCR
//    levels, only the 2^j outermost threads; the matrix is strictly diagonally dominant, so the
//    off-diagonals of the reduced rows decay (quadratically per level) and the needed rows are
//    normally finished (all |A|,|C| < 2^-70 fp64 / 2^-40 fp32) before the contamination has
//    crossed the halo.  The CTA CHECKS this: if after the kLevels levels the halo allows some
//    needed row is not finished, it records the first step of its launch in the status word and every
//    later TILED launch returns at once, leaving the state that launch started from intact.  The row
//    coefficients depend on the row's own u only, so the next step is solved from the registers: S solves
//    per tile, the band of wrong threads growing by 2^kLevels per step, then one store.  The kernel is
//    persistent within a launch (grid = SMs x resident CTAs) and software-pipelined with cp.async.
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
constexpr int kP = 8;          // rows per thread partition of the GENERAL kernel
// TILED kernel: kTP rows per thread, kTn threads per CTA (tile = kTn*kTP points).  After the in-CTA
// cyclic-reduction step every thread holds ONE reduced row (coupling ~ lambda^kTP between
// neighbours); kLevels PCR levels follow, which contaminate 2^kLevels threads from each open tile
// end.  The left halo is one thread wider because x_0 of a partition is recovered from the
// reduced unknown of its LEFT neighbour.
constexpr int kTP = 16;
constexpr int kTn = 128;
constexpr int kLevels = 3;
// Contaminated threads at the open ends of a tile after s steps in registers: one step spoils 2^kLevels reduced
// rows per end; the next step starts from partitions that are wrong there, so the band grows by 2^kLevels per
// step, plus one thread on the left (x_0 of a partition needs the reduced unknown of its left neighbour).
__host__ __device__ constexpr int tile_halo_r(int s) { return s << kLevels; }
__host__ __device__ constexpr int tile_halo_l(int s) { return (s << kLevels) + 1; }
__host__ __device__ constexpr int tile_width(int tn, int s) { return (tn - tile_halo_l(s) - tile_halo_r(s)) * kTP; }   // owned points
constexpr int kHaloR = tile_halo_r(1);        // threads; the one-step tile of kTn threads
constexpr int kHaloL = tile_halo_l(1);
constexpr int kW = tile_width(kTn, 1);
constexpr int kGenThreads = 256;
constexpr int kStatusBytes = 1024;            // status word + 2 x 64 level flags

__device__ __forceinline__ int64_t wrap(int64_t g, int64_t N) {
    g %= N;
    return g < 0 ? g + N : g;
}

// ------------------------------------------------------------------------ TILED step kernel
// Per thread: P-row partition elimination -> two interface rows
//     first:  A x_L(t-1) + x_0(t) + C x_L(t) = D          last:  f x_0(t) + x_L(t) + c x_0(t+1) = q
// One cyclic-reduction step removes every x_0 (substituting first(t) and first(t+1) into last(t)):
//     [-f A] x_L(t-1) + [1 - f C - c A'] x_L(t) + [-c C'] x_L(t+1) = q - f D - c D'     (' = thread t+1)
// leaving one row per thread in the unknowns x_L, solved by truncated PCR on the open chain; then
// x_0(t) = D - A x_L(t-1) - C x_L(t) and the partition is back-substituted.
//
// The kernel is PERSISTENT within a step: gridDim.x CTAs (a multiple of the SM count) walk over
// the tiles, and the next tile's points are fetched into a second shared-memory stage with
// cp.async (LDGSTS, 16 B per thread per request, fully coalesced) while the current tile is being
// eliminated, so that the global-load latency is hidden behind FP64 work.  The stage is written
// with an XOR swizzle of the 16-byte chunk index so that thread t can read its own P consecutive
// points (a 128-byte row in fp64) with conflict-free LDS.128.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(unsigned dst, const void *src, unsigned bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
// one element of T (4 or 8 bytes; src-size 0 zero-fills): the ragged wrap of a grid whose length is not a
// multiple of the 16-byte vector
template <int BYTES>
__device__ __forceinline__ void cp_async_elem(unsigned dst, const void *src, unsigned bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(dst), "l"(src), "n"(BYTES), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }

// TN threads per CTA, S time steps per launch (S = 2: the tile is solved twice in registers before it is stored;
// the contaminated band at each open end grows by 2^kLevels threads per step, tile_halo_l/r below).
template <typename T, int TN, int S, bool DIRI>
__global__ void __launch_bounds__(TN, 512 / TN)
btcs_long_tiled_kernel(const T *__restrict__ src, T *__restrict__ dst, const T *__restrict__ nu,
                       const T *__restrict__ dt, int64_t N, int tiles, int B, double inv_dx,
                       int bc, int step, int *__restrict__ status) {
    constexpr int P = kTP, Tn = TN;
    constexpr int kHaloL = tile_halo_l(S), kHaloR = tile_halo_r(S), kW = tile_width(TN, S);
    constexpr int V = 16 / sizeof(T);
    constexpr int CR = P / V;                 // 16-byte chunks per thread row (8 fp64, 4 fp32)
    constexpr int SW = 8 / CR;                // rows sharing one 128-byte line
    constexpr int RB = CR * 16;               // bytes per thread row
    constexpr int WB = 32 * RB;               // bytes per warp region of a stage
    extern __shared__ __align__(128) unsigned char stage_dyn[];    // [2][Tn * P] of T
    __shared__ T sA[2][Tn], sC[2][Tn], sD[2][Tn];
    __shared__ T sFA[Tn], sFC[Tn], sFD[Tn];   // first interface rows (own arrays: the PCR buffers of the
                                              // previous tile may still be read when these are written)
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    // Programmatic dependent launch: let the next step's grid be scheduled while this one runs
    // (its CTAs become resident as ours retire), and wait here for the previous step's grid to
    // have completed and flushed before reading anything it wrote.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (*reinterpret_cast<volatile int *>(status) != 0) return;   // an earlier step failed (uniform)
    const bool dirichlet = DIRI;                 // (bc == BURGERS_BC_DIRICHLET; the periodic instances carry no
    (void)bc;                                    // identity-row code: a third less to fetch per solve)
    const bool aligned = (N % V == 0);

    // Warp-private staging: warp w of the CTA owns rows 32w..32w+31 of a tile = WB contiguous bytes
    // of global memory.  It copies them with CR requests of 512 contiguous bytes each (lane l moves
    // chunk k*32+l), and every lane later reads / writes its OWN row: only __syncwarp() in between.
    // Chunk c of row r lives at r*RB + ((c ^ ((r/SW) % CR)) * 16); request k of lane l moves chunk
    // c = l % CR of row r = k*(32/CR) + l/CR of the warp region.
    const int fr = lane / CR, fc = lane % CR;                        // row / chunk of request 0
    auto f_off = [&](int k) {
        const int r = k * (32 / CR) + fr;
        return (unsigned)(warp * WB + r * RB + ((fc ^ ((r / SW) % CR)) * 16));
    };
    const unsigned r_off = (unsigned)(t * RB) | (unsigned)((((t / SW) % CR)) * 16);   // XOR with c*16 per chunk
    const unsigned stage0 = smem_u32(stage_dyn);
    constexpr unsigned kStageBytes = Tn * P * sizeof(T);

    auto fetch = [&](int b, int tile, int st) {
        const int64_t wg0 = (int64_t)tile * kW + (int64_t)(warp * 32 - kHaloL) * P;   // first point of the warp region
        const bool edge = (wg0 < 0) || (wg0 + 32 * P > N);
        const T *srow = src + (int64_t)b * N;
        const unsigned d0 = stage0 + st * kStageBytes;
        if (!edge) {
            const T *g = srow + wg0 + lane * V;
#pragma unroll
            for (int k = 0; k < CR; ++k) cp_async16(d0 + f_off(k), g + k * 32 * V, 16);
        } else if (aligned) {
#pragma unroll
            for (int k = 0; k < CR; ++k) {
                int64_t g = wg0 + (int64_t)(k * 32 + lane) * V;
                unsigned bytes = 16;
                if (dirichlet) { if (g < 0 || g >= N) { bytes = 0; g = 0; } }
                else { if (g < 0) g += N; else if (g >= N) g -= N; }
                cp_async16(d0 + f_off(k), srow + g, bytes);
            }
        } else {          // N % V != 0: the wrapped (or cut) chunks are not 16-byte pieces of the row any more
#pragma unroll
            for (int k = 0; k < CR; ++k) {
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    int64_t g = wg0 + (int64_t)(k * 32 + lane) * V + e;
                    unsigned bytes = sizeof(T);
                    if (dirichlet) { if (g < 0 || g >= N) { bytes = 0; g = 0; } }
                    else { if (g < 0) g += N; else if (g >= N) g -= N; }
                    cp_async_elem<sizeof(T)>(d0 + f_off(k) + e * sizeof(T), srow + g, bytes);
                }
            }
        }
        cp_async_commit();
    };

    // work items (system b, tile) in order; this CTA takes every gridDim.x-th one
    int b = (int)(blockIdx.x / (unsigned)tiles), tile = (int)(blockIdx.x % (unsigned)tiles);
    const int db = (int)(gridDim.x / (unsigned)tiles), dtile = (int)(gridDim.x % (unsigned)tiles);
    if (b < B) fetch(b, tile, 0);
    for (int st = 0; b < B; st ^= 1) {
        int bn = b + db, tn_ = tile + dtile;
        if (tn_ >= tiles) { tn_ -= tiles; ++bn; }
        if (bn < B) { fetch(bn, tn_, st ^ 1); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncwarp();

        const int64_t g0 = (int64_t)tile * kW + (int64_t)(t - kHaloL) * P;     // unwrapped index of row 0
        Coef<T> co;
        co.init(nu[b], dt[b], inv_dx);

        // ---- this thread's partition from the swizzled stage
        T v[P];
        const unsigned rbase = stage0 + st * kStageBytes + r_off;
#pragma unroll
        for (int c = 0; c < CR; ++c) {
            int4 q4;
            asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(q4.x), "=r"(q4.y), "=r"(q4.z), "=r"(q4.w) : "r"(rbase ^ (unsigned)(c * 16)));
            const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
            for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
        }

        bool failed = false;
#pragma unroll
        for (int sub = 0; sub < S; ++sub) {
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

        // ---- cyclic-reduction step: one row per thread in x_L
        sFA[t] = first.A; sFC[t] = first.C; sFD[t] = first.D;
        __syncthreads();
        Row<T> row;
        {
            const int tn = (t + 1 < Tn) ? t + 1 : t;       // t = Tn-1: last.C == 0, values unused
            const T nA = sFA[tn], nC = sFC[tn], nD = sFD[tn];
            const T m = rcp(t_fma(-last.A, first.C, t_fma(-last.C, nA, T(1))));
            row.A = -last.A * first.A * m;
            row.C = -last.C * nC * m;
            row.D = t_fma(-last.A, first.D, t_fma(-last.C, nD, last.D)) * m;
        }
        sA[0][t] = row.A; sC[0][t] = row.C; sD[0][t] = row.D;
        __syncthreads();

        // ---- PCR on the open chain of Tn rows, at most kLevels levels.  Rows that must be
        // finished: the threads still valid after this step and the left neighbour of the first of them.
        const bool needed = (t >= tile_halo_l(sub + 1) - 1) && (t < Tn - tile_halo_r(sub + 1));
        int cur = 0;
        bool finished = false;
#pragma unroll
        for (int l = 0; l < kLevels; ++l) {
            const int s = 1 << l;
            const int km = t - s, kp = t + s;
            Row<T> rm, rp;
            if (km >= 0) { rm.A = sA[cur][km]; rm.C = sC[cur][km]; rm.D = sD[cur][km]; }
            else { rm.A = T(0); rm.C = T(0); rm.D = T(0); }
            if (kp < Tn) { rp.A = sA[cur][kp]; rp.C = sC[cur][kp]; rp.D = sD[cur][kp]; }
            else { rp.A = T(0); rp.C = T(0); rp.D = T(0); }
            row = pcr_combine(row, rm, rp);
            sA[cur ^ 1][t] = row.A; sC[cur ^ 1][t] = row.C; sD[cur ^ 1][t] = row.D;
            cur ^= 1;
            // The check is made once, after the last level the halo allows (a vote per level costs the read-back
            // of the barrier's result and a dependent branch; levels past the decoupling change nothing that is
            // stored).  NaN-safe: a row that is not provably finished counts as unfinished.
            if (l == kLevels - 1) {
                const int flag = needed & !((t_abs(row.A) <= Lim<T>::tiny()) & (t_abs(row.C) <= Lim<T>::tiny()));
                finished = !__syncthreads_or(flag);
            } else {
                __syncthreads();
            }
        }
        if (!finished) {                       // the halo was too short for these coefficients
            if (t == 0) atomicCAS(status, 0, step + 1);
            failed = true;
            break;                             // uniform over the CTA
        }

        // ---- recover x_0, back substitution
        if (sub + 1 < S) {
            // another step follows in registers: every thread advances (the threads of the contaminated band
            // compute values nobody uses; what they touch is bounded by the reach of the PCR levels)
            const T xL = row.D;
            const T xLprev = sD[cur][t > 0 ? t - 1 : 0];
            const T x0 = t_fma(-first.A, xLprev, t_fma(-first.C, xL, first.D));
            back_substitute<T, P>(v, f, c, q, x0, xL);
        } else {
        // the warp's rows go back through its stage region so that the global stores are 512 contiguous
        // bytes per request
        const bool owned = (t >= kHaloL) && (t < Tn - kHaloR);
        if (owned) {
            const T xL = row.D;
            const T xLprev = sD[cur][t - 1];
            const T x0 = t_fma(-first.A, xLprev, t_fma(-first.C, xL, first.D));
            back_substitute<T, P>(v, f, c, q, x0, xL);
#pragma unroll
            for (int cc = 0; cc < CR; ++cc) {
                int4 q4;
                T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
                for (int k = 0; k < V; ++k) e[k] = v[cc * V + k];
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(rbase ^ (unsigned)(cc * 16)), "r"(q4.x), "r"(q4.y), "r"(q4.z), "r"(q4.w) : "memory");
            }
        }
        }
        }
        if (failed) break;
        __syncwarp();
        {
            const int64_t wg0 = (int64_t)tile * kW + (int64_t)(warp * 32 - kHaloL) * P;
            T *drow = dst + (int64_t)b * N;
            const unsigned s0 = stage0 + st * kStageBytes;
#pragma unroll
            for (int k = 0; k < CR; ++k) {
                const int rt = warp * 32 + (k * 32 + lane) / CR;            // thread that owns this chunk's row
                const int64_t g = wg0 + (int64_t)(k * 32 + lane) * V;
                if (rt >= kHaloL && rt < Tn - kHaloR && g < N) {
                    int4 q4;
                    asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(q4.x), "=r"(q4.y), "=r"(q4.z), "=r"(q4.w) : "r"(s0 + f_off(k)));
                    if (g + V <= N) {
                        *reinterpret_cast<int4 *>(drow + g) = q4;
                    } else {                   // the chunk that straddles the end of a grid with N % V != 0
                        const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
                        for (int k2 = 0; k2 < V; ++k2)
                            if (g + k2 < N) drow[g + k2] = e[k2];
                    }
                }
            }
        }
        __syncwarp();      // the stage region is re-filled by this warp's next-but-one fetch
        b = bn; tile = tn_;
    }
    cp_async_wait<0>();
}

// After the TILED launches: move the newest valid state into u when it sits in ws.  The first n_multi launches made
// S steps each, the others one; the state after L launches is in ws iff L is odd.  No failure: the final state;
// failure in the launch that starts at step n: u^n.
template <typename T>
__global__ void btcs_long_fixup_kernel(T *__restrict__ u, const T *__restrict__ ws, int64_t elems,
                                       int64_t n_steps, int64_t n_multi, int S, const int *__restrict__ status) {
    const int fail = *status;
    const int64_t n = fail ? (int64_t)(fail - 1) : n_steps;
    const int64_t launches = (n < S * n_multi) ? n / S : n_multi + (n - S * n_multi);
    if ((launches & 1) == 0) return;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < elems; i += stride) u[i] = ws[i];
}

// ------------------------------------------------------------------------ GENERAL kernel
template <typename T>
struct GenRows {   // interface rows in global memory, two buffers (PCR ping-pong)
    T *A[2], *C[2], *D[2];
};

// Partition `part` of the grid-wide list: system b, partition tt of its pps (a power of two).  RAGGED = false:
// N == kP * pps, rows tt*kP .. tt*kP + kP - 1 (16-byte aligned vector loads); RAGGED = true: any N, the rows
// btcs::partition_of() deals partition tt (n = N/pps or N/pps + 1 of them, in the first n slots).
template <typename T, bool RAGGED>
__device__ __forceinline__ void gen_load_partition(const T *__restrict__ u, int64_t N, int64_t part,
                                                   int64_t parts_per_sys, T (&v)[kP], int64_t &b,
                                                   int64_t &tt, Part &pt) {
    constexpr int V = 16 / sizeof(T);
    b = part / parts_per_sys;
    tt = part % parts_per_sys;
    if (RAGGED) {
        pt = partition_of((int)tt, (int)N, (int)parts_per_sys);
        const T *p = u + b * N + pt.r0;
#pragma unroll
        for (int j = 0; j < kP; ++j) v[j] = (j < pt.n) ? __ldcg(p + j) : T(0);
        return;
    }
    pt.r0 = (int)(tt * kP); pt.n = kP;
    const T *p = u + b * N + tt * kP;     // N % kP == 0: 16-byte aligned
#pragma unroll
    for (int c = 0; c < kP / V; ++c) {
        int4 q4 = __ldcg(reinterpret_cast<const int4 *>(p) + c);
        const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
        for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
    }
}

// assembly + elimination of one partition of the GENERAL kernel (both phases use it)
template <typename T, bool RAGGED>
__device__ __forceinline__ void gen_eliminate(const T (&v)[kP], const Coef<T> &co, const Part &pt, bool fixL, bool fixR,
                                              T (&f)[kP], T (&c)[kP], T (&q)[kP], Row<T> &first, Row<T> &last) {
    if (RAGGED) {
#pragma unroll
        for (int j = 0; j < kP; ++j) q[j] = v[j];
        eliminate_general_ragged<T, kP>(
            [&](int j, T &a, T &b, T &e) {
                co.at(v[j], a, b, e);
                if ((j == 0 && fixL) || (j >= pt.n - 1 && fixR)) { a = T(0); b = T(1); e = T(0); }
            },
            pt.n, q, f, c, first, last);
    } else {
        eliminate<T, kP>(v, co, [&](int j) { return (j == 0 && fixL) || (j == kP - 1 && fixR); }, f, c, q, first, last);
    }
}

template <typename T, bool RAGGED>
__global__ void __launch_bounds__(kGenThreads)
btcs_long_general_kernel(T *__restrict__ u, const T *__restrict__ nu, const T *__restrict__ dt,
                         int64_t B, int64_t N, int64_t pps, double inv_dx, int64_t n_steps, int bc, GenRows<T> R,
                         int *__restrict__ status, int force) {
    constexpr int P = kP;
    constexpr int V = 16 / sizeof(T);
    cg::grid_group grid = cg::this_grid();
    const int fail = force ? 1 : *reinterpret_cast<volatile int *>(status);
    if (fail == 0) return;                              // uniform over the grid
    int *flags = status + 64;                           // [2][32]
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t parts = B * pps;                      // pps partitions per system (a power of two)
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
            Part pt;
            gen_load_partition<T, RAGGED>(u, N, part, pps, v, b, tt, pt);
            Coef<T> co;
            co.init(nu[b], dt[b], inv_dx);
            const bool fixL = dirichlet && tt == 0, fixR = dirichlet && tt == pps - 1;
            Row<T> first, last;
            gen_eliminate<T, RAGGED>(v, co, pt, fixL, fixR, f, c, q, first, last);
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
            Part pt;
            gen_load_partition<T, RAGGED>(u, N, part, pps, v, b, tt, pt);
            Coef<T> co;
            co.init(nu[b], dt[b], inv_dx);
            const bool fixL = dirichlet && tt == 0, fixR = dirichlet && tt == pps - 1;
            Row<T> first, last;
            gen_eliminate<T, RAGGED>(v, co, pt, fixL, fixR, f, c, q, first, last);
            const T x0 = __ldcg(R.D[cur] + 2 * part), xl = __ldcg(R.D[cur] + 2 * part + 1);
            T *p = u + b * N + pt.r0;
            if (RAGGED) {
                back_substitute_ragged<T, P>(v, pt.n, f, c, q, x0, xl);
#pragma unroll
                for (int j = 0; j < P; ++j)
                    if (j < pt.n) p[j] = v[j];
                continue;
            }
            back_substitute<T, P>(v, f, c, q, x0, xl);
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

// partitions per system of the GENERAL kernel: the smallest power of two with pps * kP >= N (so that the
// 2 pps interface rows form a power-of-two ring); every partition then has N/pps >= kP/2 rows
int64_t gen_pps(int64_t N) {
    int64_t pps = 2;
    while (pps * kP < N) pps *= 2;
    return pps;
}

size_t row_elems(int64_t B, int64_t N) { return (size_t)B * (size_t)(2 * gen_pps(N)); }

}  // namespace

// LONG runs any grid longer than two tiles (shorter systems fit one CTA: HYBRID).  Rows must start on a
// 16-byte boundary: any N for a single system, N a multiple of the 16-byte vector for a batch.
bool btcs_long_fits(int is_f64, int64_t B, int64_t N, int bc) {
    (void)bc;
    const int V = is_f64 ? 2 : 4;
    return N > 2 * (int64_t)kTn * kTP && N < ((int64_t)1 << 31) - 4096 && (B == 1 || N % V == 0);
}

// ws layout (elements of T): [B*N ping-pong state][6 x B*M interface rows] then kStatusBytes.
size_t btcs_long_ws_bytes(int esz, int64_t B, int64_t N) {
    const size_t state = ((size_t)B * (size_t)N * esz + 255) / 256 * 256;
    const size_t rows = (6 * row_elems(B, N) * esz + 255) / 256 * 256;
    return state + rows + kStatusBytes;
}

namespace {

// TILED shapes: threads per CTA, steps per launch, and the measured time of one tile round of the persistent grid
// (us, fp64, B200, C4b's coefficients).  More steps per launch amortise the launch, the stage fill
// and the store over S solves in registers, wider tiles keep the growing halo (16 S + 1 threads) a small part of
// the tile; what decides between them for a given grid is how evenly its tiles fill the rounds.
struct TileShape { int tn, S; double round_us; };
constexpr TileShape kTileShapes[] = {{128, 1, 3.3}, {256, 2, 5.9}, {256, 4, 10.4}, {512, 4, 11.3}, {512, 5, 13.7}, {512, 6, 16.0}};
constexpr double kLaunchUs = 2.2;

int sm_count() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        (void)cudaGetLastError();
        return 148;                      // plan queries without a device: B200
    }
    return sms;
}

// The shape with the lowest modelled time per step: (launch + rounds x round time) / S, rounds = tiles of the
// call / CTAs of the persistent grid (512 / tn per SM), rounded up.
TileShape long_tile_shape(int64_t B, int64_t N, int64_t n_steps) {
    const int sms = sm_count();
    TileShape best = kTileShapes[0];
    double best_cost = 0;
    for (const TileShape &c : kTileShapes) {
        if (c.S > n_steps || N <= 2 * (int64_t)c.tn * kTP) continue;
        const int64_t width = tile_width(c.tn, c.S);
        const int64_t items = B * ((N + width - 1) / width);
        const int64_t grid = (int64_t)sms * (512 / c.tn);
        const double cost = (kLaunchUs + (double)((items + grid - 1) / grid) * c.round_us) / c.S;
        if (best_cost == 0 || cost < best_cost) { best = c; best_cost = cost; }
    }
    return best;
}

}  // namespace

// memset + TILED launches + fixup + GENERAL (PLAN_LONG); GENERAL alone for PLAN_LONG_GENERAL
int64_t btcs_long_launch_count(int64_t B, int64_t N, int64_t n_steps, int general_only) {
    if (n_steps <= 0) return 0;
    if (general_only) return 1;
    const int S = long_tile_shape(B, N, n_steps).S;
    return n_steps / S + n_steps % S + 2;
}

template <typename T>
int launch_btcs_long(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                     int64_t n_steps, int bc, void *ws, int general_only, cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    if (!btcs_long_fits(sizeof(T) == 8, B, N, bc)) return BURGERS_ERR_PLAN;
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
        int dev0 = 0, sms0 = 0;
        if (cudaGetDevice(&dev0) != cudaSuccess ||
            cudaDeviceGetAttribute(&sms0, cudaDevAttrMultiProcessorCount, dev0) != cudaSuccess)
            return BURGERS_ERR_CUDA;
        const TileShape shape = long_tile_shape(B, N, n_steps);
        const int64_t n_multi = n_steps / shape.S;                 // launches of shape.S steps, then single steps
        T *cur = u, *nxt = pong;
        // one persistent grid per launch: every SM gets the same number of CTAs, every CTA about the same number
        // of tiles; programmatic dependent launch lets the next grid become resident as this one retires
        auto run = [&](auto kernel, int tn, int width, int64_t first_step, int64_t launches, int steps_each) -> int {
            if (launches <= 0) return BURGERS_OK;
            const size_t dyn = 2 * (size_t)tn * kTP * sizeof(T);
            int occ0 = 0;
            if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn) != cudaSuccess ||
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ0, kernel, tn, dyn) != cudaSuccess || occ0 < 1)
                return BURGERS_ERR_CUDA;
            const int64_t tiles = (N + width - 1) / width;
            const int64_t items = B * tiles;
            int64_t grid_t = (int64_t)sms0 * occ0;
            if (grid_t > items) grid_t = items;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)grid_t); cfg.blockDim = dim3(tn); cfg.dynamicSmemBytes = dyn; cfg.stream = s;
            cfg.attrs = attr; cfg.numAttrs = 1;
            for (int64_t l = 0; l < launches; ++l) {
                if (cudaLaunchKernelEx(&cfg, kernel, (const T *)cur, nxt, nu, dt, N, (int)tiles, (int)B, inv_dx, bc,
                                       (int)(first_step + l * steps_each), status) != cudaSuccess)
                    return BURGERS_ERR_CUDA;
                T *tmp = cur; cur = nxt; nxt = tmp;
            }
            return last_launch_status();
        };
        int st = BURGERS_OK;
        const bool diri = (bc == BURGERS_BC_DIRICHLET);
        switch (shape.tn * 16 + shape.S) {
#define BURGERS_CASE(TN, S_) \
    case TN * 16 + S_: \
        st = diri ? run(btcs_long_tiled_kernel<T, TN, S_, true>, TN, tile_width(TN, S_), 0, n_multi, S_) \
                  : run(btcs_long_tiled_kernel<T, TN, S_, false>, TN, tile_width(TN, S_), 0, n_multi, S_); \
        break;
            BURGERS_CASE(256, 2) BURGERS_CASE(256, 4) BURGERS_CASE(512, 4) BURGERS_CASE(512, 5) BURGERS_CASE(512, 6)
#undef BURGERS_CASE
            default: break;                                        // (128, 1): everything goes to the loop below
        }
        if (st != BURGERS_OK) return st;
        const int64_t done = (shape.S > 1) ? shape.S * n_multi : 0;
        st = diri ? run(btcs_long_tiled_kernel<T, kTn, 1, true>, kTn, kW, done, n_steps - done, 1)
                  : run(btcs_long_tiled_kernel<T, kTn, 1, false>, kTn, kW, done, n_steps - done, 1);
        if (st != BURGERS_OK) return st;
        btcs_long_fixup_kernel<T><<<(unsigned)(sms0 * 4), 256, 0, s>>>(u, pong, B * N, n_steps,
                                                                      shape.S > 1 ? n_multi : 0, shape.S, status);
        st = last_launch_status();
        if (st != BURGERS_OK) return st;
    }

    // cooperative launch of the general kernel: the grid must be co-resident
    int64_t pps = gen_pps(N);
    const bool ragged = (pps * kP != N);
    const void *gen_fn = ragged ? (const void *)btcs_long_general_kernel<T, true>
                                : (const void *)btcs_long_general_kernel<T, false>;
    int dev = 0, sms = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gen_fn, kGenThreads, 0) != cudaSuccess ||
        per_sm < 1)
        return BURGERS_ERR_CUDA;
    const int64_t want = (B * pps + kGenThreads - 1) / kGenThreads;
    int64_t grid = (int64_t)sms * per_sm;
    if (grid > want) grid = want;
    const size_t re = row_elems(B, N);
    GenRows<T> R;
    R.A[0] = rows;          R.C[0] = rows + re;     R.D[0] = rows + 2 * re;
    R.A[1] = rows + 3 * re; R.C[1] = rows + 4 * re; R.D[1] = rows + 5 * re;
    int force = general_only ? 1 : 0;
    void *args[] = {&u, &nu, &dt, &B, &N, &pps, (void *)&inv_dx, &n_steps, &bc, &R, &status, &force};
    if (cudaLaunchCooperativeKernel(gen_fn, dim3((unsigned)grid),
                                    dim3(kGenThreads), args, 0, s) != cudaSuccess)
        return BURGERS_ERR_CUDA;
    return last_launch_status();
}

template int launch_btcs_long<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, void *, int, cudaStream_t);
template int launch_btcs_long<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, void *, int, cudaStream_t);

}  // namespace burgers
