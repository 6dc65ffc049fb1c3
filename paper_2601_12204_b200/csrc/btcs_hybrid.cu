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
//  3. one cyclic-reduction step substitutes the x_0 rows of threads t and t+1 into the last row of
//     thread t, leaving ONE reduced row per thread in the unknowns x_{P-1}(t); these T rows form a
//     CYCLIC tridiagonal system, solved by parallel cyclic reduction in shared memory (rows kept
//     normalised, diag = 1).  The matrix is strictly diagonally dominant (D4), so the off-diagonals
//     of the reduced rows shrink quadratically per PCR level; once every |A|,|C| is below 2^-70
//     (fp64; 2^-40 fp32) the remaining levels cannot change a bit of the answer and the loop exits
//     early (block-wide vote, NaN-safe).  If it runs to the end, the last level is the exact 2x2
//     solve of rows t and t+T/2.
//  4. x_0(t) = D - A x_{P-1}(t-1) - C x_{P-1}(t) from the thread's first interface row, then back
//     substitution inside each thread: x_j = q_j - f_j x_0 - c_j x_{j+1}, j = P-2..1.
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

// N == P * blockDim.x: every thread owns P rows, 128-bit loads.  The interface solve is written out here although
// btcs::solve_interface is the same code: this instance is C3's kernel and the schedule ptxas finds for the
// shared-helper form is 3 % slower (measured, C3: 15.70 ms inline, 16.16 ms through solve_interface, same 128
// registers, 608 / 616 instructions; DESIGN.md 6.1 "Instruction schedule").
// Two entry points for the same kernel text: ptxas keeps the 128-thread instances at 128 registers unprompted, and ANY
// second launch-bound argument (even 0), or the body moved into an inlined device function, changes the schedule
// it picks for them (measured, C3: 13.45 ms as it is, 14.08 - 14.38 ms otherwise; DESIGN.md 6.1 "Instruction
// schedule"); the other thread counts need the cap (N = 4096, 256 threads: 148 registers, one CTA per SM and
// 7.84 ms per 200 steps of 4096 systems without it, 6.08 ms with it).
#define BURGERS_HYBRID_NAME btcs_hybrid_kernel
#define BURGERS_HYBRID_BOUNDS __launch_bounds__(TN ? TN : hybrid_max_threads(sizeof(T), P))
#include "btcs_hybrid_kernel.cuh"
#undef BURGERS_HYBRID_NAME
#undef BURGERS_HYBRID_BOUNDS
#define BURGERS_HYBRID_NAME btcs_hybrid_kernel_capped
#define BURGERS_HYBRID_BOUNDS __launch_bounds__(TN, 512 / TN)        /* 512 threads per SM: 128 registers */
#include "btcs_hybrid_kernel.cuh"
#undef BURGERS_HYBRID_NAME
#undef BURGERS_HYBRID_BOUNDS

// Any N: thread t owns the P - 1 or P rows partition_of() deals it (btcs_common.cuh), scalar loads -- the state
// is loaded and stored once per CALL, so the load width does not matter.  Same steps as the kernel above, through
// the shared helpers (eliminate_general_ragged, solve_interface, back_substitute_ragged).
// SNAP: trajectory output from inside the time loop -- after every snap_every-th step the state goes to
// snaps[k][b][:] (k = 0, 1, ...; BN = B N elements per snapshot), so that burgers_btcs_traj_* and the forward sweep
// of the BTCS adjoint are ONE launch instead of one launch + one copy per snapshot (RAGGED = false: the exact
// partitions of the kernel above, through the helpers).
template <typename T, int P, bool RAGGED, bool SNAP>
__global__ void __launch_bounds__(hybrid_max_threads(sizeof(T), P))
btcs_hybrid_general_kernel(T *__restrict__ u, const T *__restrict__ nu, const T *__restrict__ dt, int N,
                           double inv_dx, int64_t n_steps, int bc, T *__restrict__ snaps, int64_t snap_every,
                           int64_t BN) {
    constexpr int V = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int t = threadIdx.x, Tn = blockDim.x;
    T *sR = reinterpret_cast<T *>(smem_raw);  // [2][Tn] reduced rows (A, C, D): PCR ping-pong
    T *sF = sR + 6 * Tn;                      // [Tn] first interface rows (A, C, D)
    T *sS = sF + 3 * Tn;                      // SNAP, exact partitions: [Tn * P] staging of a snapshot
    Part part;
    part.r0 = t * P; part.n = P;
    if (RAGGED) part = partition_of(t, N, Tn);
    const int n = part.n;
    __builtin_assume(n >= P - 1 && n <= P);     // P = ceil(N / Tn): only the last slot is conditional
    T *row = u + (int64_t)blockIdx.x * N + part.r0;

    Coef<T> co;
    co.init(nu[blockIdx.x], dt[blockIdx.x], inv_dx);
    const bool fixL = (bc == BURGERS_BC_DIRICHLET) && t == 0;
    const bool fixR = (bc == BURGERS_BC_DIRICHLET) && t == Tn - 1;

    T v[P];
    if (RAGGED) {
#pragma unroll
        for (int j = 0; j < P; ++j) v[j] = (j < n) ? row[j] : T(0);
    } else {
#pragma unroll
        for (int c = 0; c < P / V; ++c) {
            int4 q4 = *reinterpret_cast<const int4 *>(row + c * V);
            const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
            for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
        }
    }

    int64_t until_snap = snap_every;
    T *snap_row = SNAP ? snaps + (int64_t)blockIdx.x * N + part.r0 : nullptr;
    for (int64_t step = 0; step < n_steps; ++step) {
        T f[P], c[P], q[P];
        // ---- assembly + partition elimination
        Row<T> first, last;
        if (RAGGED) {
#pragma unroll
            for (int j = 0; j < P; ++j) q[j] = v[j];
            eliminate_general_ragged<T, P>(
                [&](int j, T &a, T &b, T &e) {
                    co.at(v[j], a, b, e);
                    if ((j == 0 && fixL) || (j == n - 1 && fixR)) { a = T(0); b = T(1); e = T(0); }
                },
                n, q, f, c, first, last);
        } else {
            eliminate<T, P>(v, co, [&](int j) { return (j == 0 && fixL) || (j == P - 1 && fixR); },
                            f, c, q, first, last);
        }
        // ---- cyclic-reduction step + parallel cyclic reduction over the ring of Tn reduced rows
        T x0, xL;
        solve_interface<T>(first, last, sR, sF, x0, xL, t, Tn);
        // ---- back substitution
        if (RAGGED) back_substitute_ragged<T, P>(v, n, f, c, q, x0, xL);
        else back_substitute<T, P>(v, f, c, q, x0, xL);
        if (SNAP) {
            if (--until_snap == 0) {
                until_snap = snap_every;
                T *srow = snap_row;
                snap_row += BN;
                if (RAGGED) {
#pragma unroll
                    for (int j = 0; j < P; ++j)
                        if (j < n) srow[j] = v[j];
                } else if (Tn < 32) {                  // (a partial warp: straight from the registers)
#pragma unroll
                    for (int c2 = 0; c2 < P / V; ++c2) {
                        int4 q4;
                        T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
                        for (int k = 0; k < V; ++k) e[k] = v[c2 * V + k];
                        *reinterpret_cast<int4 *>(srow + c2 * V) = q4;
                    }
                } else {
                    // Coalesced stores through a warp-private stage: the 32 rows of a warp are 32 * P contiguous
                    // elements of the snapshot.  Every lane puts its row into shared memory (16-byte chunk c of row
                    // r at r * CR + (c ^ ((r / SW) % CR)): conflict-free for the row-wise stores and for the
                    // chunk-wise loads), then the warp writes CR requests of 512 contiguous bytes.  Straight from
                    // the registers a store instruction touches 32 different 128-byte lines (27 -> 17 us per step
                    // of C3 with a snapshot after every step).
                    constexpr int CR = P / V;             // 16-byte chunks per row
                    constexpr int SW = (CR >= 8) ? 1 : 8 / CR;
                    const int lane = t & 31;
                    int4 *wst = reinterpret_cast<int4 *>(sS) + (t - lane) * CR;      // this warp's 32 * CR chunks
#pragma unroll
                    for (int c2 = 0; c2 < CR; ++c2) {
                        int4 q4;
                        T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
                        for (int k = 0; k < V; ++k) e[k] = v[c2 * V + k];
                        wst[lane * CR + (c2 ^ ((lane / SW) % CR))] = q4;
                    }
                    __syncwarp();
                    int4 *wdst = reinterpret_cast<int4 *>(srow - lane * P);          // first element of the warp's rows
#pragma unroll
                    for (int k = 0; k < CR; ++k) {
                        const int g = k * 32 + lane, r = g / CR, c2 = g % CR;
                        wdst[g] = wst[r * CR + (c2 ^ ((r / SW) % CR))];
                    }
                    __syncwarp();
                }
            }
        }
    }

    if (RAGGED) {
#pragma unroll
        for (int j = 0; j < P; ++j)
            if (j < n) row[j] = v[j];
    } else {
#pragma unroll
        for (int c = 0; c < P / V; ++c) {
            int4 q4;
            T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
            for (int k = 0; k < V; ++k) e[k] = v[c * V + k];
            *reinterpret_cast<int4 *>(row + c * V) = q4;
        }
    }
}

// P register slots per thread, Tn threads (a power of two >= 2): btcs::pick_partition
bool hybrid_geometry(int is_f64, int64_t N, int *P_out, int *T_out, bool *ragged) {
    const int bytes = is_f64 ? 8 : 4;
    return pick_partition(N, [bytes](int P) { return hybrid_max_threads(bytes, P); }, P_out, T_out, ragged);
}

template <typename T, int P>
int launch_P(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
             int Tn, bool ragged, cudaStream_t s) {
    const size_t smem = (size_t)9 * Tn * sizeof(T);
    if (ragged) {
        btcs_hybrid_general_kernel<T, P, true, false><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc,
                                                                                  nullptr, 0, 0);
        return last_launch_status();
    }
    if constexpr (P == 4 || P == 8 || P == 16) {
        switch (Tn) {
#define BURGERS_TN(TN_) \
    case TN_: \
        if constexpr (TN_ <= hybrid_max_threads(sizeof(T), P)) { \
            if constexpr (TN_ == 128) { \
                if (bc == BURGERS_BC_DIRICHLET) \
                    btcs_hybrid_kernel<T, P, TN_, true><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc); \
                else \
                    btcs_hybrid_kernel<T, P, TN_, false><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc); \
            } else { \
                if (bc == BURGERS_BC_DIRICHLET) \
                    btcs_hybrid_kernel_capped<T, P, TN_, true><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc); \
                else \
                    btcs_hybrid_kernel_capped<T, P, TN_, false><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc); \
            } \
            return last_launch_status(); \
        } \
        break;
            BURGERS_TN(32) BURGERS_TN(64) BURGERS_TN(128) BURGERS_TN(256) BURGERS_TN(512)
#undef BURGERS_TN
            default: break;
        }
        if (bc == BURGERS_BC_DIRICHLET)
            btcs_hybrid_kernel<T, P, 0, true><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc);
        else
            btcs_hybrid_kernel<T, P, 0, false><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc);
        return last_launch_status();
    }
    return BURGERS_ERR_PLAN;
}

template <typename T, int P>
int launch_traj_P(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                  int64_t snap_every, T *snaps, int Tn, bool ragged, cudaStream_t s) {
    const size_t smem = (size_t)9 * Tn * sizeof(T);
    if (ragged) {
        btcs_hybrid_general_kernel<T, P, true, true><<<(unsigned)B, Tn, smem, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc,
                                                                                 snaps, snap_every, B * N);
        return last_launch_status();
    }
    if constexpr (P == 4 || P == 8 || P == 16) {
        const size_t smem_s = smem + (size_t)Tn * P * sizeof(T);                  // + the snapshot stage
        if (smem_s > 48 * 1024 &&
            cudaFuncSetAttribute(btcs_hybrid_general_kernel<T, P, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)smem_s) != cudaSuccess)
            return BURGERS_ERR_CUDA;
        btcs_hybrid_general_kernel<T, P, false, true><<<(unsigned)B, Tn, smem_s, s>>>(u, nu, dt, (int)N, 1.0 / dx, n_steps, bc,
                                                                                    snaps, snap_every, B * N);
        return last_launch_status();
    }
    return BURGERS_ERR_PLAN;
}

}  // namespace

bool btcs_hybrid_fits(int is_f64, int64_t N, int bc) {
    (void)bc;
    int P, Tn;
    bool ragged;
    return hybrid_geometry(is_f64, N, &P, &Tn, &ragged);
}

template <typename T>
int launch_btcs_hybrid(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                       int64_t n_steps, int bc, cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    int P, Tn;
    bool ragged;
    if (!hybrid_geometry(sizeof(T) == 8, N, &P, &Tn, &ragged)) return BURGERS_ERR_PLAN;
    if (B > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    switch (P) {
#define BURGERS_CASE(PP) case PP: return launch_P<T, PP>(u, B, N, dx, nu, dt, n_steps, bc, Tn, ragged, s);
        BURGERS_CASE(4) BURGERS_CASE(5) BURGERS_CASE(6) BURGERS_CASE(7) BURGERS_CASE(8) BURGERS_CASE(9) BURGERS_CASE(10)
        BURGERS_CASE(11) BURGERS_CASE(12) BURGERS_CASE(13) BURGERS_CASE(14) BURGERS_CASE(15) BURGERS_CASE(16)
#undef BURGERS_CASE
    }
    return BURGERS_ERR_PLAN;
}

// n_steps steps with a snapshot after every snap_every-th one (snaps: [n_steps / snap_every][B][N]); one launch.
template <typename T>
int launch_btcs_hybrid_traj(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                            int64_t snap_every, T *snaps, cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    int P, Tn;
    bool ragged;
    if (!hybrid_geometry(sizeof(T) == 8, N, &P, &Tn, &ragged)) return BURGERS_ERR_PLAN;
    if (B > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    switch (P) {
#define BURGERS_CASE(PP) \
    case PP: return launch_traj_P<T, PP>(u, B, N, dx, nu, dt, n_steps, bc, snap_every, snaps, Tn, ragged, s);
        BURGERS_CASE(4) BURGERS_CASE(5) BURGERS_CASE(6) BURGERS_CASE(7) BURGERS_CASE(8) BURGERS_CASE(9) BURGERS_CASE(10)
        BURGERS_CASE(11) BURGERS_CASE(12) BURGERS_CASE(13) BURGERS_CASE(14) BURGERS_CASE(15) BURGERS_CASE(16)
#undef BURGERS_CASE
    }
    return BURGERS_ERR_PLAN;
}

template int launch_btcs_hybrid_traj<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, int64_t, float *, cudaStream_t);
template int launch_btcs_hybrid_traj<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, int64_t, double *, cudaStream_t);
template int launch_btcs_hybrid<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, cudaStream_t);
template int launch_btcs_hybrid<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, cudaStream_t);

}  // namespace burgers
