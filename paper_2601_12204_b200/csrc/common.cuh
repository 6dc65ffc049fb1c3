// common.cuh -- internal declarations shared by the translation units of libburgers.
// (Product code only; the CPU oracle under oracle/ shares nothing with this.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/burgers.h"

namespace burgers {

constexpr int kWarp = 32;

// Grid spacing (D1): periodic dx = L/N (node N == node 0),
// Dirichlet dx = L/(N-1).
inline double grid_dx(int64_t N, double L, int bc) {
    return bc == BURGERS_BC_PERIODIC ? L / (double)N : L / (double)(N - 1);
}

inline int cuda_status(cudaError_t e) { return e == cudaSuccess ? BURGERS_OK : BURGERS_ERR_CUDA; }
inline int last_launch_status() { return cuda_status(cudaGetLastError()); }

// ---------------------------------------------------------------- re-layout (layout.cu)
// in[rows][cols] -> out[cols][rows]; the thread-per-system plans work on the batch-minor layout [N][B].
template <typename T>
int launch_transpose(const T *in, T *out, int64_t rows, int64_t cols, cudaStream_t s);
// CTA size of the thread-per-system kernels: one warp per CTA until every SM has four of them
inline int thread_per_system_block(int64_t B) { return (B <= 148 * 32 * 4) ? 32 : 128; }

// ---------------------------------------------------------------- CFL (cfl.cu)
template <typename T>
int launch_cfl(const T *u, int64_t B, int64_t N, double dx, const T *nu, double C, T *dt_out,
               cudaStream_t s);
int64_t cfl_launch_count(int is_f64, int64_t B, int64_t N);

// ---------------------------------------------------------------- explicit (explicit_*.cu)
// dt from the CFL condition (D8) for one trajectory whose max |u| is m: evaluated in
// fp64 on the (already T-rounded) inputs, rounded to T once.  x/0 = +inf.  Shared by cfl.cu and the adaptive
// explicit kernel so that both give the same bits.
template <typename T>
__device__ __forceinline__ T cfl_dt(T m, T nu, double dx, double C) {
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double conv = (m > T(0)) ? dx / (double)m : inf;
    double diff = ((double)nu > 0.0) ? dx * dx / (2.0 * (double)nu) : inf;
    return (T)(C * ((conv < diff) ? conv : diff));
}

// Geometry of one explicit launch plan, decided on the host (explicit_plan.cu).
struct ExplicitGeom {
    int plan;        // BURGERS_PLAN_RESIDENT / BURGERS_PLAN_TILED
    int P;           // grid points per thread
    int nth;         // active threads per CTA (CTA holds nth*P points)
    int block;       // launched threads per CTA (nth rounded up to a warp multiple)
    int tblock;      // steps per launch (TILED), unused for RESIDENT
    int halo;        // halo points per side (TILED) = tblock*radius rounded up
    int64_t W;       // valid outputs per tile (TILED)
    int64_t tiles;   // tiles per trajectory (TILED)
};
// Fills `g` for (dtype, N, bc, scheme) under `plan` (AUTO allowed) with optional overrides
// (tblock/ppt = 0 -> defaults).  Returns BURGERS_OK or BURGERS_ERR_PLAN.
int explicit_geometry(int is_f64, int64_t B, int64_t N, int bc, int scheme, int plan, int tblock,
                      int ppt, ExplicitGeom *g);
// Adaptive time step fused into the RESIDENT kernel (SURVEY 8(f) NEXT-4a): dt is re-evaluated from the
// CFL condition every `every` steps inside the kernel; `dt` of launch_explicit is then not read.
template <typename T>
struct ExplicitAdapt {
    int64_t every;   // m: steps per CFL evaluation (>= 1)
    double C;        // CFL number
    double *t_out;   // [B] simulated time, sum of m*dt (may be nullptr)
    T *dt_out;       // [B] the last dt used
};
// The same for TILED grids, one call per segment of n_steps steps (explicit_impl.cuh, Params::umax): the last
// launch of the segment leaves max |u| in slot seg_write of umax[3][B], the launches of the next segment compute
// their dt from slot seg_read (< 0: from `dt`), its first launch clears slot seg_zero and records dt / time.
template <typename T>
struct ExplicitTiledAdapt {
    unsigned long long *umax;
    int seg_read, seg_write, seg_zero;
    double C;
    double *t_out;
    T *dt_out;
};
template <typename T>
int launch_explicit(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                    int64_t n_steps, int bc, int scheme, const ExplicitGeom &g, T *ws,
                    T *snaps, int64_t snap_every, cudaStream_t s, const ExplicitAdapt<T> *adapt = nullptr,
                    const ExplicitTiledAdapt<T> *tadapt = nullptr);
// Register budget -> launch bound of explicit_kernel<T, P, scheme> (the one definition: the kernel's
// __launch_bounds__ and the host-side geometry both use it).  State registers per thread: P points x
// words x arrays (fp32 Euler: base, s, v; other Euler: v; RK4: v, y, acc) plus ~40 for addressing and
// temporaries; 64 K registers per SM.
constexpr int explicit_max_threads_for(int bytes, int P, int scheme) {
    int arrays = (scheme == BURGERS_SCHEME_RK4) ? 3 : (bytes == 4 ? 3 : 1);
    int regs = P * (bytes / 4) * arrays + 40;
    int t = 1024;
    while (t > 32 && t * regs > 65536) t /= 2;
    return t;
}
inline int explicit_max_threads(int is_f64, int P, int scheme) {
    return explicit_max_threads_for(is_f64 ? 8 : 4, P, scheme);
}

// ---------------------------------------------------------------- BTCS (btcs_*.cu)
template <typename T>
int launch_btcs_thomas(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                       int64_t n_steps, int bc, T *ws, cudaStream_t s);
size_t btcs_thomas_ws_elems(int64_t B, int64_t N, int bc);
int64_t btcs_thomas_launch_count(int64_t n_steps);

template <typename T>
int launch_btcs_hybrid(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                       int64_t n_steps, int bc, cudaStream_t s);
bool btcs_hybrid_fits(int is_f64, int64_t N, int bc);
// the same with trajectory output from inside the kernel (one launch): snaps[k] after every snap_every-th step
template <typename T>
int launch_btcs_hybrid_traj(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                            int64_t snap_every, T *snaps, cudaStream_t s);

// LONG: one system across many CTAs.  `ws` holds the ping-pong state, the global interface rows
// and the status word (btcs_long_ws_bytes).  general_only != 0 runs the cooperative GENERAL
// kernel alone (BURGERS_PLAN_LONG_GENERAL).
template <typename T>
int launch_btcs_long(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                     int64_t n_steps, int bc, void *ws, int general_only, cudaStream_t s);
size_t btcs_long_ws_bytes(int esz, int64_t B, int64_t N);
int64_t btcs_long_launch_count(int64_t B, int64_t N, int64_t n_steps, int general_only);
bool btcs_long_fits(int is_f64, int64_t B, int64_t N, int bc);

// ---------------------------------------------------------------- adjoint of explicit Euler (adjoint.cu)
template <typename T>
int launch_adjoint_steps(const T *u0, const T *states, T *lam, T *pong, int64_t B, int64_t N, double dx,
                         const T *nu, const T *dt, int64_t n_steps, int bc, cudaStream_t s);

// ---------------------------------------------------------------- adjoint of RK4 (adjoint_rk4.cu)
template <typename T>
int launch_adjoint_rk4_steps(const T *start, const T *states, T *lam, T *ws, int64_t B, int64_t N, double dx, const T *nu,
                             const T *dt, int64_t len, int bc, cudaStream_t s);
size_t adjoint_rk4_ws_elems(int64_t B, int64_t N);

// ---------------------------------------------------------------- reverse mode of the Newton / theta-scheme (adjoint_newton.cu)
// states: u^1 .. u^{n_steps} ([n_steps][B][N]); ws: adjoint_newton_ws_elems elements (0 when the resident plan runs)
template <typename T>
int launch_adjoint_newton_steps(const T *u0, const T *states, T *lam, T *ws, int64_t B, int64_t N, double dx,
                                const T *nu, const T *dt, int64_t n_steps, int bc, double theta, cudaStream_t s);
size_t adjoint_newton_ws_elems(int is_f64, int64_t B, int64_t N);

// ---------------------------------------------------------------- adjoint of BTCS (adjoint_btcs.cu)
// states: u^1 .. u^{n_steps} ([n_steps][B][N]); ws: adjoint_btcs_ws_elems elements (0 when the resident plan runs)
template <typename T>
int launch_adjoint_btcs_steps(const T *u0, const T *states, T *lam, T *ws, int64_t B, int64_t N, double dx, const T *nu,
                              const T *dt, int64_t n_steps, int bc, cudaStream_t s);
size_t adjoint_btcs_ws_elems(int is_f64, int64_t B, int64_t N);

// ---------------------------------------------------------------- Gauss-Seidel BTCS (btcs_gs.cu)
template <typename T>
int launch_btcs_gs(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                   double tol, int max_iter, long long *iters_out, T *ws, cudaStream_t s);
size_t btcs_gs_ws_elems(int64_t B, int64_t N);

// ---------------------------------------------------------------- Newton BTCS (newton.cu)
template <typename T>
int launch_newton(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt, int64_t n_steps, int bc,
                  double theta, double tol, int max_iter, long long *iters_out, int plan, T *ws, cudaStream_t s,
                  bool accumulate = false, T *snaps = nullptr, int64_t snap_every = 0);   // snaps: HYBRID plan only
bool newton_hybrid_fits(int is_f64, int64_t N);
size_t newton_thomas_ws_elems(int64_t B, int64_t N, int bc);

}  // namespace burgers
