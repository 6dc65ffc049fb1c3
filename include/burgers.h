/*
 * burgers.h -- C ABI of libburgers: time stepping of the 1D viscous Burgers
 * equation  u_t + u u_x = nu u_xx  (Eq.1) on B200 (sm_100a).
 *
 * Spatial discretisation (Eq.3-4; upwind rule PAPER.md:89):
 * first-order upwind convection, second-order central diffusion.
 * Time discretisation: forward Euler (Eq.21), classical RK4 of the
 * same semi-discrete operator (Eq.22), and BTCS
 * (Eq.23) in the lagged-coefficient reading of
 * DESIGN.md (Q4): per step one (cyclic) tridiagonal solve.
 * Time-step limit (PAPER.md:116-118 Eq.7-8, :287 Eq.24).
 *
 * Conventions common to every call
 * --------------------------------
 *  - Status: 0 = BURGERS_OK, <0 = error.  Nothing throws, nothing aborts.
 *    Argument errors are returned synchronously BEFORE anything is enqueued.
 *  - Device entry points (no `_host` suffix): `u`, `nu`, `dt`, `dt_out`, `ws` are
 *    CUDA DEVICE pointers owned by the caller; `stream` is a cudaStream_t passed
 *    as void* (NULL = default stream).  Calls only enqueue work on `stream` and
 *    return; no device synchronisation inside.  The DEVICE entry points allocate
 *    nothing and keep no global mutable state (re-entrant; concurrent calls on
 *    different streams with disjoint buffers are legal, from one or several host
 *    threads).
 *  - `_host` entry points: every pointer is a HOST pointer (pinned or pageable);
 *    the call takes device buffers from a memory pool the LIBRARY owns (one per
 *    device, created by the first `_host` call, freed blocks kept up to 1 GiB, never
 *    destroyed) and, for large batches, two library-owned streams per device; it
 *    copies in, runs the same device path, copies out, and returns after the result
 *    is in host memory.  This per-device pool and stream pair is the only state
 *    the library keeps.  `_host` calls work on the legacy default stream: calls from
 *    several host threads are legal but serialise on the device.
 *  - Layout: `u` is [B][N] row-major (trajectory-contiguous), base 16-byte
 *    aligned; `nu`, `dt`, `dt_out` have length B (one value per trajectory).
 *    `u` is updated IN PLACE: after the call (stream-ordered) it holds the state
 *    after `n_steps` steps.  n_steps = 0 is a valid no-op.
 *  - Grid (readings Q6/Q8 of DESIGN.md).  Periodic: N distinct nodes,
 *    dx = L/N, node i at i dx, neighbours wrap mod N (Eq.18).
 *    Dirichlet: N nodes including both ends, dx = L/(N-1); the boundary values
 *    are u[b][0] and u[b][N-1] AS FOUND IN THE INPUT and are never modified
 *    (Eq.16-17).
 *  - Errors: NULL pointer -> BURGERS_ERR_NULL; B<1, N<3, n_steps<0 ->
 *    BURGERS_ERR_SHAPE; unknown bc/scheme/plan/op -> BURGERS_ERR_ENUM; L<=0, C<=0
 *    or non-finite, tol < 0 or NaN, max_iter < 0, theta outside [0,1] -> BURGERS_ERR_VALUE; workspace too small (or NULL when a
 *    non-zero size is required) -> BURGERS_ERR_WORKSPACE; a CUDA launch/runtime
 *    failure -> BURGERS_ERR_CUDA; a plan that cannot run this shape ->
 *    BURGERS_ERR_PLAN.  Device-side values (nu<0, dt<=0, NaN in u) are not
 *    checked; NaN/Inf propagate per IEEE.
 *  - Scratch comes from `ws` (size from burgers_workspace_bytes, 256-byte aligned
 *    base recommended, 16-byte required).  Its content is undefined on return.
 */
#ifndef BURGERS_H
#define BURGERS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BURGERS_VERSION 100 /* 0.1.0 */

enum {
    BURGERS_OK = 0,
    BURGERS_ERR_NULL = -1,
    BURGERS_ERR_SHAPE = -2,
    BURGERS_ERR_ENUM = -3,
    BURGERS_ERR_VALUE = -4,
    BURGERS_ERR_WORKSPACE = -5,
    BURGERS_ERR_CUDA = -6,
    BURGERS_ERR_PLAN = -7,
    BURGERS_ERR_LIMIT = -8     /* burgers_btcs_noalloc: the problem needs more than the built-in scratch */
};
enum { BURGERS_BC_PERIODIC = 0, BURGERS_BC_DIRICHLET = 1 };
enum { BURGERS_SCHEME_EULER = 0, BURGERS_SCHEME_RK4 = 1 };
enum { BURGERS_OP_EXPLICIT = 0, BURGERS_OP_BTCS = 1, BURGERS_OP_CFL = 2, BURGERS_OP_NEWTON = 3,
       BURGERS_OP_GS = 4 };

/* Kernel plans.  AUTO picks by shape; the others force one
 * plan (tests use this for cross-plan agreement, G10) and return
 * BURGERS_ERR_PLAN when the shape does not fit it. */
enum {
    BURGERS_PLAN_AUTO = 0,
    /* explicit: */
    BURGERS_PLAN_RESIDENT = 1, /* whole trajectory on chip for all n_steps      */
    BURGERS_PLAN_TILED = 2,    /* overlapped tiles, k steps per HBM round trip  */
    /* BTCS: */
    BURGERS_PLAN_THOMAS = 3,   /* one thread per system, interleaved [N][B] ws  */
    BURGERS_PLAN_HYBRID = 4,   /* one CTA per system: partitions + PCR, resident*/
    BURGERS_PLAN_LONG = 5,     /* one system across many CTAs: overlapped tiles (1-6 steps per launch) with a
                                  checked truncated PCR, cooperative fallback     */
    BURGERS_PLAN_LONG_GENERAL = 6 /* the cooperative global-PCR kernel alone       */
};

/* ---- explicit time stepping (PAPER.md:216 Eq.21; :224-229 Eq.22) --------------
 * n_steps steps of  u^{n+1} = u^n + dt F(u^n)  (Euler) or classical RK4 of F,
 * F_i = -u_i g_i/dx + nu (u_{i+1} - 2u_i + u_{i-1})/dx^2,
 * g_i = u_i - u_{i-1} if u_i > 0 else u_{i+1} - u_i.
 * dt[b] is held fixed over the call.  RK4: the upwind direction is re-decided from
 * each stage value; Dirichlet end nodes have k = 0 in every stage.
 * fp32: on chip the state is carried scaled by dt/dx and (Euler) as a two-term sum
 * (compensated accumulation); it is unscaled and rounded to fp32 once
 * when written back, so p then q steps agree with p+q steps to rounding, not bitwise
 * (fp64 is bitwise).  dt[b] = 0 leaves trajectory b untouched; dt[b] < 0 is not supported. */
int burgers_explicit_f32(float *u, int64_t B, int64_t N, double L, const float *nu,
                         const float *dt, int64_t n_steps, int bc, int scheme,
                         void *ws, size_t ws_bytes, void *stream);
int burgers_explicit_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                         const double *dt, int64_t n_steps, int bc, int scheme,
                         void *ws, size_t ws_bytes, void *stream);
/* Same, forcing a plan.  `tblock` = steps per HBM round trip of the TILED plan
 * (0 = library default; ignored by RESIDENT); `ppt` = grid points held per thread
 * (0 = library default; else one of 1,2,4,8,16,32 -- BURGERS_ERR_PLAN if the shape
 * does not fit it). */
int burgers_explicit_plan_f32(float *u, int64_t B, int64_t N, double L, const float *nu,
                              const float *dt, int64_t n_steps, int bc, int scheme,
                              int plan, int tblock, int ppt, void *ws, size_t ws_bytes,
                              void *stream);
int burgers_explicit_plan_f64(double *u, int64_t B, int64_t N, double L,
                              const double *nu, const double *dt, int64_t n_steps,
                              int bc, int scheme, int plan, int tblock, int ppt,
                              void *ws, size_t ws_bytes, void *stream);

/* Same time stepping with TRAJECTORY output (SURVEY.md 8(f) NEXT-4b; the paper's stated purpose is data
 * generation): after every snap_every-th step (steps snap_every, 2 snap_every, ...)
 * the state is also written to snaps[k][B][N], k = 0 .. n_steps/snap_every - 1 (DEVICE pointer, room
 * for floor(n_steps/snap_every) * B * N elements); u holds the final state as usual.  The RESIDENT
 * plan writes the snapshots from the resident state inside the one kernel; the TILED plan runs one
 * launch sequence per snapshot interval.  snap_every < 1 -> BURGERS_ERR_SHAPE. */
int burgers_explicit_traj_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                              int64_t n_steps, int bc, int scheme, int64_t snap_every, float *snaps,
                              void *ws, size_t ws_bytes, void *stream);
int burgers_explicit_traj_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                              const double *dt, int64_t n_steps, int bc, int scheme,
                              int64_t snap_every, double *snaps, void *ws, size_t ws_bytes,
                              void *stream);

/* Explicit stepping with an ADAPTIVE time step (SURVEY.md 8(f) NEXT-4a; "timesteps chosen to
 * satisfy the CFL criteria"): n_outer times { dt_b = C min(dx/max|u_b|, dx^2/(2 nu_b)) from the current
 * state (dt_from_cfl_*); m_steps steps of the scheme with it }.  Shapes of the RESIDENT plan run as ONE
 * kernel with the CFL evaluation inside its time loop (fp64: the bits of the separate calls; fp32: the
 * state is not rounded to fp32 between the segments); longer grids (TILED) as the launches of the time stepping
 * alone, the last launch of a segment leaving max|u| for the next segment's dt (the bits of the separate calls);
 * their workspace is that of burgers_workspace_bytes(BURGERS_OP_EXPLICIT, ...).  Everything is
 * enqueued on the stream; nothing synchronises with the host.  dt_scratch: DEVICE [B] (holds the last dt on return);
 * t_out: DEVICE double [B] receiving the simulated time sum m_steps*dt_b, or NULL. */
int burgers_explicit_adaptive_f32(float *u, int64_t B, int64_t N, double L, const float *nu, double C,
                                  int64_t n_outer, int64_t m_steps, int bc, int scheme,
                                  float *dt_scratch, double *t_out, void *ws, size_t ws_bytes,
                                  void *stream);
int burgers_explicit_adaptive_f64(double *u, int64_t B, int64_t N, double L, const double *nu, double C,
                                  int64_t n_outer, int64_t m_steps, int bc, int scheme,
                                  double *dt_scratch, double *t_out, void *ws, size_t ws_bytes,
                                  void *stream);

/* Discrete ADJOINT of n_steps forward-Euler steps (SURVEY.md 8(f) NEXT-4c; the reverse-mode derivative
 * the paper takes from JAX; D13).  u0: the initial state (not
 * modified); lam: in dJ/du^N, out dJ/du^0 = (du^N/du^0)^T lam, with dt and nu held fixed and the upwind
 * switch locally constant.  The forward states are recomputed into the workspace
 * (burgers_adjoint_workspace_bytes; checkpointed when they would not fit, see below). */
int burgers_explicit_adjoint_f32(const float *u0, float *lam, int64_t B, int64_t N, double L,
                                 const float *nu, const float *dt, int64_t n_steps, int bc, void *ws,
                                 size_t ws_bytes, void *stream);
int burgers_explicit_adjoint_f64(const double *u0, double *lam, int64_t B, int64_t N, double L,
                                 const double *nu, const double *dt, int64_t n_steps, int bc, void *ws,
                                 size_t ws_bytes, void *stream);
size_t burgers_adjoint_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps);
/* Same with an explicit checkpoint segment: the steps are cut into segments of `segment` steps, the
 * state at every segment start is stored by a first forward sweep, and each segment is recomputed (one
 * snapshot per step) just before it is swept backwards: memory (n_steps/segment + segment) states, one
 * extra forward sweep.  segment = 0: automatic (one segment while all states fit 8 GiB, else
 * ceil(sqrt(n_steps))) -- this is what burgers_explicit_adjoint_* use.  segment < 0 -> BURGERS_ERR_SHAPE. */
int burgers_explicit_adjoint_ckpt_f32(const float *u0, float *lam, int64_t B, int64_t N, double L,
                                      const float *nu, const float *dt, int64_t n_steps, int bc,
                                      int64_t segment, void *ws, size_t ws_bytes, void *stream);
int burgers_explicit_adjoint_ckpt_f64(const double *u0, double *lam, int64_t B, int64_t N, double L,
                                      const double *nu, const double *dt, int64_t n_steps, int bc,
                                      int64_t segment, void *ws, size_t ws_bytes, void *stream);
size_t burgers_adjoint_ckpt_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc,
                                            int64_t n_steps, int64_t segment);

/* The same for either explicit scheme: scheme = BURGERS_SCHEME_EULER (D13) or BURGERS_SCHEME_RK4 -- the discrete
 * adjoint of the classical RK4 step (D14; PAPER.md:224-229 Eq.22, :231): with G_s = dt dF/dy at the
 * stage value y_s,  t4 = G4^T lam/6, t3 = G3^T (lam/3 + t4), t2 = G2^T (lam/3 + t3/2), t1 = G1^T (lam/6 + t2/2),
 * lam <- lam + t4 + t3 + t2 + t1 per step, the stage values rebuilt from the stored (checkpointed) u^n.
 * segment as above (0 = automatic). */
int burgers_explicit_adjoint_scheme_f32(const float *u0, float *lam, int64_t B, int64_t N, double L,
                                        const float *nu, const float *dt, int64_t n_steps, int bc,
                                        int scheme, int64_t segment, void *ws, size_t ws_bytes, void *stream);
int burgers_explicit_adjoint_scheme_f64(const double *u0, double *lam, int64_t B, int64_t N, double L,
                                        const double *nu, const double *dt, int64_t n_steps, int bc,
                                        int scheme, int64_t segment, void *ws, size_t ws_bytes, void *stream);
size_t burgers_adjoint_scheme_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int scheme,
                                              int64_t n_steps, int64_t segment);

/* ---- BTCS (Eq.23; D4-D7) ----------------------
 * Per step solve  A(u^n) u^{n+1} = u^n  with, c_i = u_i^n dt/dx, r = nu dt/dx^2:
 *   sub_i = -r - max(c_i,0),  diag_i = 1 + 2r + |c_i|,  sup_i = -r + min(c_i,0).
 * Dirichlet: unknowns i = 1..N-2, known end values moved to the right-hand side.
 * Periodic: cyclic system (corner terms; Sherman-Morrison in the THOMAS plan,
 * cyclic reduction of the interface system in HYBRID/LONG -- same solution up to
 * rounding).  The matrix is strictly diagonally dominant: no pivoting. */
int burgers_btcs_f32(float *u, int64_t B, int64_t N, double L, const float *nu,
                     const float *dt, int64_t n_steps, int bc, void *ws,
                     size_t ws_bytes, void *stream);
int burgers_btcs_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                     const double *dt, int64_t n_steps, int bc, void *ws,
                     size_t ws_bytes, void *stream);
int burgers_btcs_plan_f32(float *u, int64_t B, int64_t N, double L, const float *nu,
                          const float *dt, int64_t n_steps, int bc, int plan, void *ws,
                          size_t ws_bytes, void *stream);
int burgers_btcs_plan_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                          const double *dt, int64_t n_steps, int bc, int plan, void *ws,
                          size_t ws_bytes, void *stream);

/* BTCS with trajectory output, semantics as burgers_explicit_traj_*.  Systems that fit one CTA (plan HYBRID):
 * ONE launch, the kernel stores the state after every snap_every-th step; longer grids: one run of the AUTO
 * plan per snapshot interval followed by a device copy (workspace as for burgers_btcs_*). */
int burgers_btcs_traj_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                          int64_t n_steps, int bc, int64_t snap_every, float *snaps, void *ws,
                          size_t ws_bytes, void *stream);
int burgers_btcs_traj_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                          int64_t n_steps, int bc, int64_t snap_every, double *snaps, void *ws,
                          size_t ws_bytes, void *stream);

/* Discrete ADJOINT of n_steps BTCS steps (D15; gradients of the numerical solution).
 * One step solves A(u) u' = u; reverse mode:  mu = A(u^n)^{-T} lam,  lam_i <- (1 - D_i) mu_i,
 * D_i = (dt/dx) (u'_i - u'_{i-1}) if u_i > 0 else (dt/dx) (u'_{i+1} - u'_i)  (identity rows, D = 0 at Dirichlet ends).
 * u0: initial state (not modified); lam: in dJ/du^N, out dJ/du^0.  The forward sweep stores every state in the
 * workspace (burgers_btcs_adjoint_workspace_bytes: (n_steps + 1) B N elements + the BTCS workspace while that is
 * below 8 GiB, checkpointed beyond -- see burgers_btcs_adjoint_ckpt_*); the backward sweep keeps lam resident per CTA for every N that fits one CTA (thread per system
 * otherwise). */
int burgers_btcs_adjoint_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                             const float *dt, int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream);
int burgers_btcs_adjoint_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                             const double *dt, int64_t n_steps, int bc, void *ws, size_t ws_bytes, void *stream);
size_t burgers_btcs_adjoint_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps);
/* The same with an explicit checkpoint segment, as burgers_explicit_adjoint_ckpt_*: checkpoints every `segment`
 * steps from a first forward sweep, each segment recomputed (one state per step, written by the forward kernel) and
 * swept backwards; memory (n_steps/segment + segment + 1) states.  segment = 0: automatic (one segment while all
 * states fit 8 GiB, else ceil(sqrt(n_steps))) -- what burgers_btcs_adjoint_* / burgers_newton_adjoint_* use, so the
 * reverse sweep of a full-size config (C3: 1000 steps of 4096 x 2048 = 67 GB of states) fits in 4.5 GB.
 * op: BURGERS_OP_BTCS or BURGERS_OP_NEWTON (the workspace query serves both schemes). */
int burgers_btcs_adjoint_ckpt_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                                  const float *dt, int64_t n_steps, int bc, int64_t segment, void *ws,
                                  size_t ws_bytes, void *stream);
int burgers_btcs_adjoint_ckpt_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                                  const double *dt, int64_t n_steps, int bc, int64_t segment, void *ws,
                                  size_t ws_bytes, void *stream);
size_t burgers_implicit_adjoint_ckpt_workspace_bytes(int op, int dtype_is_f64, int64_t B, int64_t N, int bc,
                                                     int64_t n_steps, int64_t segment);

/* ---- BTCS with a Gauss-Seidel inner solver -----------
 * The system of burgers_btcs_* solved per step by lexicographic Gauss-Seidel sweeps from x = u^n until
 * max_i |rhs_i - (A x)_i| < tol or max_iter sweeps were done (D12) -- the paper's iterative
 * variant, kept for its iteration counts and for comparison; the direct solvers are exact and cheaper.
 * 64 <= N <= 4096: one CTA per system, the sweep evaluated as a scan of the affine maps x_i = p_i + q_i x_{i-1}
 * (the sequential sweep up to rounding order), no workspace; other N: one thread per system, needs workspace.
 * burgers_workspace_bytes(BURGERS_OP_GS, ...) says which (0 = none; ws may then be NULL).
 * iters_out: DEVICE pointer to B int64 (sweeps summed over the steps), or NULL. */
int burgers_btcs_gs_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                        int64_t n_steps, int bc, double tol, int max_iter, int64_t *iters_out,
                        void *ws, size_t ws_bytes, void *stream);
int burgers_btcs_gs_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                        int64_t n_steps, int bc, double tol, int max_iter, int64_t *iters_out,
                        void *ws, size_t ws_bytes, void *stream);

/* ---- fully implicit BTCS with central convection, Newton-Raphson (Eq.10-15) ----
 * (D11.)  Per step solve F(w) = 0 for w = u^{n+1},
 *   F_i = w_i - u_i^n + dt [ w_i (w_{i+1} - w_{i-1})/(2 dx) - nu (w_{i+1} - 2 w_i + w_{i-1})/dx^2 ]   (Eq.11)
 * by Newton's method from w = u^n:  J(w) delta = -F(w), w += delta (Eq.12-13), with the tridiagonal
 * Jacobian J_{i,i-1} = -dt w_i/(2dx) - r, J_{i,i} = 1 + dt (w_{i+1} - w_{i-1})/(2dx) + 2r,
 * J_{i,i+1} = dt w_i/(2dx) - r, r = nu dt/dx^2 (Eq.14; Eq.15 of the paper is garbled, Q5),
 * until max_i |F_i| < tol or max_iter iterations were done (PAPER.md:245 uses tol = 1e-6).
 * theta in [0,1] ("Crank-Nicolson"): with G(v) = dt times the
 * bracket of Eq.11, F(w) = w - u^n + theta G(w) + (1-theta) G(u^n); theta = 1 is Eq.11 itself,
 * theta = 1/2 Crank-Nicolson (second order in time), theta = 0 forward Euler with central convection.
 * Dirichlet end nodes stay fixed; periodic systems are cyclic.  No pivoting: J is diagonally
 * dominant when |w| dx / nu <= 2 and dt (w_{i+1} - w_{i-1})/(2dx) > -1.
 * iters_out: DEVICE pointer to B int64 (Newton iterations summed over the steps), or NULL.
 * plan: BURGERS_PLAN_AUTO, BURGERS_PLAN_HYBRID (one CTA per system, N = P 2^k that fits one CTA, no
 * workspace) or BURGERS_PLAN_THOMAS (one thread per system, any N, needs workspace). */
int burgers_newton_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                       int64_t n_steps, int bc, double theta, double tol, int max_iter,
                       int64_t *iters_out, int plan, void *ws, size_t ws_bytes, void *stream);
int burgers_newton_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                       int64_t n_steps, int bc, double theta, double tol, int max_iter,
                       int64_t *iters_out, int plan, void *ws, size_t ws_bytes, void *stream);

/* The same with TRAJECTORY output, semantics as burgers_explicit_traj_* / burgers_btcs_traj_*: one launch that
 * stores snaps[k][B][N] from inside the kernel when the system fits one CTA, else one run of the AUTO plan per
 * snapshot interval followed by a device copy (room for floor(n_steps/snap_every) snapshots); iters_out receives
 * the totals over all intervals.  Workspace as for burgers_newton_* (AUTO plan). */
int burgers_newton_traj_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                            int64_t n_steps, int bc, double theta, double tol, int max_iter,
                            int64_t *iters_out, int64_t snap_every, float *snaps, void *ws, size_t ws_bytes,
                            void *stream);
int burgers_newton_traj_f64(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                            int64_t n_steps, int bc, double theta, double tol, int max_iter,
                            int64_t *iters_out, int64_t snap_every, double *snaps, void *ws, size_t ws_bytes,
                            void *stream);

/* REVERSE MODE of n_steps Newton / theta-scheme steps (D16; the scheme: Eq.10-15; the
 * purpose: PAPER.md:231, :261).  One step maps u = u^n to the root w = u^{n+1} of
 *   F(w; u) = w - u + theta G(w) + (1 - theta) G(u),   G_i(v) = h v_i (v_{i+1} - v_{i-1}) - r (v_{i+1} - 2 v_i + v_{i-1}),
 * h = dt/(2 dx), r = nu dt/dx^2 (identity rows at Dirichlet end nodes).  Implicit-function theorem:
 *   J(u^{n+1})^T mu = lam,   lam <- mu - (1 - theta) G'(u^n)^T M mu     (J: the Newton Jacobian, Eq.14; M: zero rows at
 * Dirichlet ends) -- the derivative of the map the CONVERGED iteration defines: pass a tol near rounding
 * (e.g. 1e-13 in fp64); tol and max_iter drive the forward sweep exactly as in burgers_newton_*.
 * u0: initial state (not modified); lam: in dJ/du^N, out dJ/du^0.  The forward sweep stores every state in the
 * workspace (burgers_newton_adjoint_workspace_bytes: (n_steps + 1) B N elements + the Newton workspace while that
 * is below 8 GiB, checkpointed beyond); the backward sweep keeps lam resident per CTA for every N that fits one CTA (thread per system
 * otherwise).  Errors as burgers_newton_*. */
int burgers_newton_adjoint_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                               const float *dt, int64_t n_steps, int bc, double theta, double tol, int max_iter,
                               void *ws, size_t ws_bytes, void *stream);
int burgers_newton_adjoint_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                               const double *dt, int64_t n_steps, int bc, double theta, double tol, int max_iter,
                               void *ws, size_t ws_bytes, void *stream);
size_t burgers_newton_adjoint_workspace_bytes(int dtype_is_f64, int64_t B, int64_t N, int bc, int64_t n_steps);
/* With an explicit checkpoint segment (see burgers_btcs_adjoint_ckpt_*; workspace:
 * burgers_implicit_adjoint_ckpt_workspace_bytes(BURGERS_OP_NEWTON, ...)). */
int burgers_newton_adjoint_ckpt_f32(const float *u0, float *lam, int64_t B, int64_t N, double L, const float *nu,
                                    const float *dt, int64_t n_steps, int bc, double theta, double tol, int max_iter,
                                    int64_t segment, void *ws, size_t ws_bytes, void *stream);
int burgers_newton_adjoint_ckpt_f64(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                                    const double *dt, int64_t n_steps, int bc, double theta, double tol, int max_iter,
                                    int64_t segment, void *ws, size_t ws_bytes, void *stream);

/* ---- CFL time step (PAPER.md:116-118 Eq.7-8, :287 Eq.24) -----------------------
 * dt_out[b] = C * min(dx / max_i |u[b][i]|, dx^2 / (2 nu[b])), with x/0 = +inf
 * (u == 0 gives the diffusive bound, nu == 0 the convective one, both: +inf).
 * The max runs over all N stored nodes (Dirichlet: end nodes included).
 * dt_out doubles as the reduction scratch (no workspace). */
int dt_from_cfl_f32(const float *u, int64_t B, int64_t N, double L, const float *nu,
                    double C, int bc, float *dt_out, void *stream);
int dt_from_cfl_f64(const double *u, int64_t B, int64_t N, double L, const double *nu,
                    double C, int bc, double *dt_out, void *stream);

/* ---- host-buffer variants (end-to-end path; all pointers HOST) -----------------
 * Device buffers come from a stream-ordered memory pool owned by the library (per device, created by the
 * first host-buffer call; freed blocks are kept up to 1 GiB so that repeated calls do not remap memory).
 * The calls return when the result is in the host buffers. */
int burgers_explicit_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu,
                              const float *dt, int64_t n_steps, int bc, int scheme);
int burgers_explicit_host_f64(double *u, int64_t B, int64_t N, double L,
                              const double *nu, const double *dt, int64_t n_steps,
                              int bc, int scheme);
int burgers_btcs_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu,
                          const float *dt, int64_t n_steps, int bc);
int burgers_btcs_host_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                          const double *dt, int64_t n_steps, int bc);
int burgers_newton_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu, const float *dt,
                            int64_t n_steps, int bc, double theta, double tol, int max_iter,
                            int64_t *iters_out);
int burgers_newton_host_f64(double *u, int64_t B, int64_t N, double L, const double *nu,
                            const double *dt, int64_t n_steps, int bc, double theta, double tol,
                            int max_iter, int64_t *iters_out);
int dt_from_cfl_host_f32(const float *u, int64_t B, int64_t N, double L, const float *nu,
                         double C, int bc, float *dt_out);
int dt_from_cfl_host_f64(const double *u, int64_t B, int64_t N, double L,
                         const double *nu, double C, int bc, double *dt_out);
/* The whole hot path of SURVEY.md 8(a) on HOST buffers in one call: u and nu are uploaded once,
 * dt = dt_from_cfl(u0, C) is computed on the device and used for all n_steps
 * of op = BURGERS_OP_EXPLICIT (`scheme` = BURGERS_SCHEME_*) or BURGERS_OP_BTCS (`scheme` ignored), AUTO
 * plan; u is overwritten with the result; dt_out (B values, may be NULL) receives the step used.
 * Same kernels, hence bitwise the same result, as dt_from_cfl_host_* followed by burgers_*_host_*, with
 * one upload of the state instead of two (large batches go through as two halves on two streams so that
 * copies overlap kernels).  Errors as for the separate calls. */
int burgers_solve_host_f32(float *u, int64_t B, int64_t N, double L, const float *nu, double C,
                           int64_t n_steps, int bc, int op, int scheme, float *dt_out);
int burgers_solve_host_f64(double *u, int64_t B, int64_t N, double L, const double *nu, double C,
                           int64_t n_steps, int bc, int op, int scheme, double *dt_out);

/* ---- queries (pure functions of the shape; no device work) -------------------- */
/* Scratch bytes needed by op (BURGERS_OP_*) with `plan` (BURGERS_PLAN_AUTO allowed).
 * `scheme` is ignored for BTCS/CFL.  Returns 0 when none is needed or when the
 * arguments are invalid (the op call itself reports the error). */
size_t burgers_workspace_bytes(int op, int dtype_is_f64, int64_t B, int64_t N, int bc,
                               int scheme, int plan);
/* The plan AUTO resolves to for this shape (BURGERS_PLAN_*), or <0 on bad args.
 * Needs a CUDA device only for the resident-fit check of the explicit op. */
int burgers_plan_query(int op, int dtype_is_f64, int64_t B, int64_t N, int bc,
                       int scheme);
/* ---- BTCS without any allocation ----------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): burgers_btcs_f32 / _f64 (above; plan AUTO, same kernels, same bits) with the workspace
 * taken from a device array built into the library instead of from the caller.  u, nu, dt: DEVICE pointers
 * of the element type dtype_is_f64 selects, caller-owned as in burgers_btcs_*; stream: cudaStream_t.
 * The call, like burgers_btcs_*, is asynchronous and calls no cudaMalloc / cudaFree / allocating routine.
 *  - Limit: burgers_noalloc_scratch_bytes() = 32 MiB per GPU, held by every GPU that loads the library from
 *    module load until the process exits.  A problem whose burgers_workspace_bytes(BURGERS_OP_BTCS, ...,
 *    BURGERS_PLAN_AUTO) exceeds it (a single fp64 grid of more than 2^20 points, say) is rejected with
 *    BURGERS_ERR_LIMIT before anything is launched; the other errors are those of burgers_btcs_*.
 *  - Set-up: the array's device address is looked up once per device, on the first call made with that
 *    device current (or by burgers_noalloc_init(), which does only that: call it before a graph capture).
 *  - Sharing: every call on a device uses the same array, which keeps the last call's contents; what must
 *    start at zero is cleared on `stream` by the call itself.  Calls that OVERLAP on the GPU (two streams,
 *    two host threads, two graphs replayed concurrently) race on it: serialise them. */
size_t burgers_noalloc_scratch_bytes(void);
int burgers_noalloc_init(void);
int burgers_btcs_noalloc(int dtype_is_f64, void *u, int64_t B, int64_t N, double L, const void *nu,
                         const void *dt, int64_t n_steps, int bc, void *stream);

/* Number of kernel launches (memset/memcpy nodes excluded) the op enqueues. */
int64_t burgers_launch_count(int op, int dtype_is_f64, int64_t B, int64_t N, int bc,
                             int scheme, int plan, int tblock, int64_t n_steps);
/* ---- measurement aid (bench.py) -------------------------------------------------------
 * One launch of a register-only micro-benchmark of the FP pipe the "alu" rooflines are quoted against:
 * every SM at full occupancy, every thread `iters` rounds of 64 independent instructions of one kind:
 *   BURGERS_PEAK_FFMA_CHAIN  a = fma(a, x, y), shared constant operands (operand-reuse cache): issue rate
 *   BURGERS_PEAK_FFMA_3REG   a = fma(a, b, c), three distinct registers: register-operand bandwidth
 *   BURGERS_PEAK_FADD_2REG   a = a + b
 *   BURGERS_PEAK_DFMA_CHAIN / _DFMA_3REG / _DADD_2REG: the same in fp64;
 *   BURGERS_PEAK_DFMA_SELECT_MIX  5 DFMA chains and one FSETP + 2 FSEL per round (the mix of the fp64
 *                            upwind stencil); only the DFMAs are counted.
 * The caller times the launch (CUDA events on `stream`); *lane_instr_out (HOST pointer, may be NULL)
 * receives the lane-instructions executed = threads x 64 x iters.  sink: DEVICE pointer to 8 writable
 * bytes (never written in practice).  Computes nothing of the method. */
enum {
    BURGERS_PEAK_FFMA_CHAIN = 0, BURGERS_PEAK_FFMA_3REG = 1, BURGERS_PEAK_FADD_2REG = 2,
    BURGERS_PEAK_DFMA_CHAIN = 3, BURGERS_PEAK_DFMA_3REG = 4, BURGERS_PEAK_DADD_2REG = 5,
    BURGERS_PEAK_DFMA_SELECT_MIX = 6, BURGERS_PEAK_KINDS = 7
};
int burgers_pipe_peak(int kind, int64_t iters, void *sink, void *stream, double *lane_instr_out);

const char *burgers_strerror(int status); /* static strings */
int burgers_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BURGERS_H */
