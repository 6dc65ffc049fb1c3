/*
 * burgers_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, scalar fp64 restatement of what the hot path of
 * arxiv 2601.12204 computes: time-stepping the 1D viscous Burgers equation
 *     u_t + u u_x = nu u_xx                              (Eq.1)
 * with first-order upwind convection (Eq.3 + upwind rule) and
 * second-order central diffusion (Eq.4), explicit (forward Euler,
 * PAPER.md:216 Eq.21; classical RK4, Eq.22) and implicit
 * (BTCS, Eq.23, in the lagged-coefficient reading of
 * DESIGN.md "Readings" Q4), plus the CFL time step (Eq.7-8,
 * :287 Eq.24).
 *
 * Rules this file obeys:
 *   - only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *     --impl reference leg may load it; the product path never does;
 *   - it shares no code, header, table or helper with the CUDA path;
 *   - always fp64, compiled -O2 -ffp-contract=off (no FMA contraction), no
 *     blocking, fusion or reordering beyond what each definition states;
 *   - OpenMP only over independent trajectories (and over space for the
 *     Jacobi-style explicit update of a single long grid, which is
 *     order-independent by definition: all of u^{n+1} comes from u^n).
 *
 * Parity pins (tests/test_oracle_*.py): worked 4-node example done in exact
 * rational arithmetic (G1,G4), Cole-Hopf closed form (R1/G2), exact Fourier
 * amplification factors (R2/G3), dense Gaussian elimination for N<=16 (R3),
 * CFL limit closed form (R4/G5), invariants (G6), textbook special cases (G7),
 * travelling viscous shock (G8); the adjoints (D13-D16): exact transpose in the linear case, dense one-step
 * formulas in numpy, central finite differences of the pinned forward functions.  No function here is
 * "parity unpinned".
 *
 * Notation follows the paper / SURVEY.md 8(c): c_i = u_i dt/dx, r = nu dt/dx^2.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { BC_PERIODIC = 0, BC_DIRICHLET = 1 };
enum { SCHEME_EULER = 0, SCHEME_RK4 = 1 };

/* D1: grid spacing.  Periodic: N distinct nodes, dx = L/N (node N == node 0,
 * PAPER.md:181 Eq.18).  Dirichlet: N nodes including both ends, dx = L/(N-1)
 * (Eq.16-17). */
static double grid_dx(int64_t N, double L, int bc)
{
    return (bc == BC_PERIODIC) ? L / (double)N : L / (double)(N - 1);
}

/* D2: semi-discrete operator F(u) (Eq.3-4, upwind rule :89,
 * assembled form :216 Eq.21).  Dirichlet end nodes get F = 0 (they never move).
 * Test hook: if use_adv, the constant `adv` replaces the multiplying u_i and the
 * sign test (linear advection-diffusion, used only by the Fourier pin R2). */
static void rhs_F(const double *u, double *F, int64_t N, double dx, double nu,
                  int bc, int use_adv, double adv)
{
    int64_t lo = 0, hi = N;
    if (bc == BC_DIRICHLET) {
        F[0] = 0.0;
        F[N - 1] = 0.0;
        lo = 1;
        hi = N - 1;
    }
    for (int64_t i = lo; i < hi; ++i) {
        int64_t im = (i == 0) ? N - 1 : i - 1;     /* periodic wrap, D1 */
        int64_t ip = (i == N - 1) ? 0 : i + 1;
        double ui = u[i];
        double dm = ui - u[im];                    /* backward difference, Eq.3 */
        double dp = u[ip] - ui;                    /* forward difference, :89   */
        double a = use_adv ? adv : ui;
        double g = (a > 0.0) ? dm : dp;            /* upwind rule, :89 (Q3: 0 -> dp) */
        double conv = a * g / dx;
        double diff = nu * (dp - dm) / (dx * dx);  /* Eq.4 */
        F[i] = -conv + diff;
    }
}

/* Exposed for the worked-example pin G1. */
void oracle_rhs(const double *u, double *F, int64_t N, double L, double nu,
                int bc, int use_adv, double adv)
{
    rhs_F(u, F, N, grid_dx(N, L, bc), nu, bc, use_adv, adv);
}

/* D3: one trajectory, n_steps explicit steps with fixed dt.
 * Euler: u^{n+1} = u^n + dt F(u^n)                               (Eq.21)
 * RK4 : k1=F(u), k2=F(u+dt/2 k1), k3=F(u+dt/2 k2), k4=F(u+dt k3),
 *       u^{n+1} = u + dt/6 (k1+2k2+2k3+k4)                       (Eq.22)
 * Jacobi-style: all of u^{n+1} from u^n. */
static void explicit_one(double *u, int64_t N, double dx, double nu, double dt,
                         int64_t n_steps, int bc, int scheme, int use_adv,
                         double adv, double *wk /* 5N doubles */)
{
    double *k1 = wk, *k2 = wk + N, *k3 = wk + 2 * N, *k4 = wk + 3 * N,
           *y = wk + 4 * N;
    for (int64_t n = 0; n < n_steps; ++n) {
        if (scheme == SCHEME_EULER) {
            rhs_F(u, k1, N, dx, nu, bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) u[i] = u[i] + dt * k1[i];
        } else {
            rhs_F(u, k1, N, dx, nu, bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) y[i] = u[i] + 0.5 * dt * k1[i];
            rhs_F(y, k2, N, dx, nu, bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) y[i] = u[i] + 0.5 * dt * k2[i];
            rhs_F(y, k3, N, dx, nu, bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) y[i] = u[i] + dt * k3[i];
            rhs_F(y, k4, N, dx, nu, bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i)
                u[i] = u[i] + dt / 6.0 * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
        }
    }
}

/* Explicit time stepping of B independent trajectories, u is [B][N] row-major,
 * updated in place; nu[b], dt[b] per trajectory.  Returns 0, or -1 on bad args /
 * allocation failure. */
int oracle_explicit(double *u, int64_t B, int64_t N, double L, const double *nu,
                    const double *dt, int64_t n_steps, int bc, int scheme,
                    int use_adv, double adv, int nthreads)
{
    if (!u || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    if (scheme != SCHEME_EULER && scheme != SCHEME_RK4) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel num_threads(nthreads)
    {
        double *wk = (double *)malloc((size_t)5 * (size_t)N * sizeof(double));
        if (!wk) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t b = 0; b < B; ++b)
                explicit_one(u + b * N, N, dx, nu[b], dt[b], n_steps, bc, scheme,
                             use_adv, adv, wk);
            free(wk);
        }
    }
    return fail ? -1 : 0;
}

/* Single long grid (B = 1), forward Euler only: same arithmetic as
 * explicit_one, the spatial loop split over threads (the update is Jacobi-style,
 * so the result does not depend on the split).  Used for timing/parity of the
 * long-grid config; results are bitwise equal to oracle_explicit. */
int oracle_explicit_long(double *u, int64_t N, double L, double nu, double dt,
                         int64_t n_steps, int bc, int nthreads)
{
    if (!u || N < 3 || n_steps < 0 || !(L > 0.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    double *v = (double *)malloc((size_t)N * sizeof(double));
    if (!v) return -1;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
    double *src = u, *dst = v;
    for (int64_t n = 0; n < n_steps; ++n) {
#pragma omp parallel for num_threads(nthreads) schedule(static)
        for (int64_t i = 0; i < N; ++i) {
            if (bc == BC_DIRICHLET && (i == 0 || i == N - 1)) {
                dst[i] = src[i];
                continue;
            }
            int64_t im = (i == 0) ? N - 1 : i - 1;
            int64_t ip = (i == N - 1) ? 0 : i + 1;
            double ui = src[i];
            double dm = ui - src[im];
            double dp = src[ip] - ui;
            double g = (ui > 0.0) ? dm : dp;
            double conv = ui * g / dx;
            double diff = nu * (dp - dm) / (dx * dx);
            double Fi = -conv + diff;
            dst[i] = ui + dt * Fi;
        }
        double *t = src; src = dst; dst = t;
    }
    if (src != u) memcpy(u, src, (size_t)N * sizeof(double));
    free(v);
    return 0;
}

/* D4: BTCS rows from the lagged state u^n (Q4).  With c_i = a_i dt/dx
 * (a_i = u_i^n, or the constant adv under the test hook), r = nu dt/dx^2:
 *   sub_i  = -r - max(c_i,0)   (multiplies u_{i-1}^{n+1})
 *   diag_i = 1 + 2r + |c_i|
 *   sup_i  = -r + min(c_i,0)   (multiplies u_{i+1}^{n+1})
 *   rhs_i  = u_i^n
 * i.e. (u_i^{n+1}-u_i^n)/dt + u_i^n * upwind_x(u^{n+1}) = nu * central_xx(u^{n+1}).
 */
static void btcs_rows(const double *u, int64_t N, double dx, double nu, double dt,
                      int use_adv, double adv, double *sub, double *diag,
                      double *sup, double *rhs)
{
    double r = nu * dt / (dx * dx);
    for (int64_t i = 0; i < N; ++i) {
        double a = use_adv ? adv : u[i];
        double c = a * dt / dx;
        double cpos = (c > 0.0) ? c : 0.0;
        double cneg = (c > 0.0) ? 0.0 : c;
        sub[i] = -r - cpos;
        diag[i] = 1.0 + 2.0 * r + fabs(c);
        sup[i] = -r + cneg;
        rhs[i] = u[i];
    }
}

/* Exposed for the row-value pin G4. */
void oracle_btcs_rows(const double *u, int64_t N, double L, double nu, double dt,
                      int bc, int use_adv, double adv, double *sub, double *diag,
                      double *sup, double *rhs)
{
    btcs_rows(u, N, grid_dx(N, L, bc), nu, dt, use_adv, adv, sub, diag, sup, rhs);
}

/* D7: Thomas algorithm, rows 0..n-1 (sub[0] and sup[n-1] are not referenced).
 * cp, dp: scratch of n doubles each.  No pivoting (D4: strictly diagonally
 * dominant). */
static void thomas(int64_t n, const double *sub, const double *diag,
                   const double *sup, const double *rhs, double *x, double *cp,
                   double *dp)
{
    cp[0] = sup[0] / diag[0];
    dp[0] = rhs[0] / diag[0];
    for (int64_t i = 1; i < n; ++i) {
        double m = diag[i] - sub[i] * cp[i - 1];
        cp[i] = sup[i] / m;
        dp[i] = (rhs[i] - sub[i] * dp[i - 1]) / m;
    }
    x[n - 1] = dp[n - 1];
    for (int64_t i = n - 2; i >= 0; --i) x[i] = dp[i] - cp[i] * x[i + 1];
}

/* Exposed for the dense-elimination pin R3.  Returns -1 on allocation failure. */
int oracle_thomas(int64_t n, const double *sub, const double *diag,
                  const double *sup, const double *rhs, double *x)
{
    double *wk = (double *)malloc((size_t)2 * (size_t)n * sizeof(double));
    if (!wk) return -1;
    thomas(n, sub, diag, sup, rhs, x, wk, wk + n);
    free(wk);
    return 0;
}

/* D6: cyclic tridiagonal solve by Sherman-Morrison.  M = tridiag(sub,diag,sup)
 * plus corners M[0][n-1] = sub[0], M[n-1][0] = sup[n-1].  gamma = -diag[0];
 * T = tridiagonal part with diag'[0] = diag[0]-gamma,
 * diag'[n-1] = diag[n-1] - sub[0]*sup[n-1]/gamma; w = (gamma,0,..,0,sup[n-1])^T,
 * v = (1,0,..,0,sub[0]/gamma)^T, M = T + w v^T.  Solve T y = rhs, T q = w;
 * x = y - q (v.y)/(1 + v.q).   wk: 6n doubles. */
static void cyclic_sm(int64_t n, const double *sub, const double *diag,
                      const double *sup, const double *rhs, double *x, double *wk)
{
    double *dmod = wk, *w = wk + n, *y = wk + 2 * n, *q = wk + 3 * n,
           *cp = wk + 4 * n, *dp = wk + 5 * n;
    double gamma = -diag[0];
    double alpha = sub[0];      /* corner M[0][n-1]   */
    double beta = sup[n - 1];   /* corner M[n-1][0]   */
    for (int64_t i = 0; i < n; ++i) {
        dmod[i] = diag[i];
        w[i] = 0.0;
    }
    dmod[0] = diag[0] - gamma;
    dmod[n - 1] = diag[n - 1] - alpha * beta / gamma;
    w[0] = gamma;
    w[n - 1] = beta;
    thomas(n, sub, dmod, sup, rhs, y, cp, dp);
    thomas(n, sub, dmod, sup, w, q, cp, dp);
    double vy = y[0] + alpha / gamma * y[n - 1];
    double vq = q[0] + alpha / gamma * q[n - 1];
    double fact = vy / (1.0 + vq);
    for (int64_t i = 0; i < n; ++i) x[i] = y[i] - fact * q[i];
}

/* Exposed for the dense-elimination pin R3. */
int oracle_cyclic(int64_t n, const double *sub, const double *diag,
                  const double *sup, const double *rhs, double *x)
{
    double *wk = (double *)malloc((size_t)6 * (size_t)n * sizeof(double));
    if (!wk) return -1;
    cyclic_sm(n, sub, diag, sup, rhs, x, wk);
    free(wk);
    return 0;
}

/* One trajectory, n_steps BTCS steps.  Periodic: D6 on all N rows.  Dirichlet
 * (D5): unknowns i = 1..N-2, rhs_1 -= sub_1 u_0, rhs_{N-2} -= sup_{N-2} u_{N-1},
 * end nodes untouched.  wk: 10N doubles + N for the new state. */
static void btcs_one(double *u, int64_t N, double dx, double nu, double dt,
                     int64_t n_steps, int bc, int use_adv, double adv, double *wk)
{
    double *sub = wk, *diag = wk + N, *sup = wk + 2 * N, *rhs = wk + 3 * N,
           *x = wk + 4 * N, *wk2 = wk + 5 * N; /* 6N */
    for (int64_t n = 0; n < n_steps; ++n) {
        btcs_rows(u, N, dx, nu, dt, use_adv, adv, sub, diag, sup, rhs);
        if (bc == BC_PERIODIC) {
            cyclic_sm(N, sub, diag, sup, rhs, x, wk2);
            for (int64_t i = 0; i < N; ++i) u[i] = x[i];
        } else {
            int64_t m = N - 2;
            rhs[1] = rhs[1] - sub[1] * u[0];
            rhs[N - 2] = rhs[N - 2] - sup[N - 2] * u[N - 1];
            thomas(m, sub + 1, diag + 1, sup + 1, rhs + 1, x + 1, wk2, wk2 + N);
            for (int64_t i = 1; i <= N - 2; ++i) u[i] = x[i];
        }
    }
}

int oracle_btcs(double *u, int64_t B, int64_t N, double L, const double *nu,
                const double *dt, int64_t n_steps, int bc, int use_adv, double adv,
                int nthreads)
{
    if (!u || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel num_threads(nthreads)
    {
        double *wk = (double *)malloc((size_t)11 * (size_t)N * sizeof(double));
        if (!wk) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t b = 0; b < B; ++b)
                btcs_one(u + b * N, N, dx, nu[b], dt[b], n_steps, bc, use_adv, adv, wk);
            free(wk);
        }
    }
    return fail ? -1 : 0;
}

/* D8: dt_b = C * min(dx / max_i |u_b,i|, dx^2 / (2 nu_b)), x/0 = +inf
 * (PAPER.md:116-118 Eq.7-8, :287 Eq.24).  Max over all N stored nodes. */
int oracle_dt_from_cfl(const double *u, int64_t B, int64_t N, double L,
                       const double *nu, double C, int bc, double *dt_out)
{
    if (!u || !nu || !dt_out || B < 1 || N < 3 || !(L > 0.0) || !(C > 0.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    for (int64_t b = 0; b < B; ++b) {
        double m = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            double a = fabs(u[b * N + i]);
            if (a > m) m = a;
        }
        double conv = (m > 0.0) ? dx / m : INFINITY;
        double diff = (nu[b] > 0.0) ? dx * dx / (2.0 * nu[b]) : INFINITY;
        dt_out[b] = C * ((conv < diff) ? conv : diff);
    }
    return 0;
}

/* ---------------------------------------------------------------------------
 * D11: fully implicit BTCS with CENTRAL convection solved
 * by Newton-Raphson, as the paper writes it out (Eq.10-15).
 * Residual (Eq.11), w = iterate for u^{n+1}, h = dt/(2 dx), r = nu dt/dx^2:
 *   F_i(w) = w_i - u_i^n + h w_i (w_{i+1} - w_{i-1}) - r (w_{i+1} - 2 w_i + w_{i-1})
 * Jacobian (Eq.14; Eq.15 is garbled in the paper -- reading Q5: differentiate Eq.11):
 *   J_{i,i-1} = -h w_i - r,  J_{i,i} = 1 + h (w_{i+1} - w_{i-1}) + 2 r,  J_{i,i+1} = h w_i - r
 * Newton (Eq.12-13): w^0 = u^n; while max_i |F_i(w^k)| >= tol and k < max_iter:
 *   solve J(w^k) delta = -F(w^k), w^{k+1} = w^k + delta.   (criterion: PAPER.md:245)
 * Dirichlet: end nodes fixed (F = 0, delta = 0 there); periodic: cyclic system.
 * theta-scheme ("Crank-Nicolson"): with
 *   G_i(v) = h v_i (v_{i+1} - v_{i-1}) - r (v_{i+1} - 2 v_i + v_{i-1})     (dt times the central operator)
 * the residual is  F_i(w) = w_i - u_i^n + theta G_i(w) + (1 - theta) G_i(u^n)  and the Jacobian
 * I + theta dG/dw;  theta = 1 is Eq.11 (BTCS), theta = 1/2 Crank-Nicolson (second order in time),
 * theta = 0 forward Euler with central convection (residual zero after one trivial iteration).
 * Test hook use_adv: the multiplying w_i is replaced by the constant adv (linear
 * advection-diffusion: J does not depend on w, one iteration is exact).
 * No pivoting: J is diagonally dominant when the cell Peclet number
 * |w| dx / nu <= 2 and h (w_{i+1} - w_{i-1}) > -1 (D11).
 */
static double newton_G(const double *v, int64_t i, int64_t N, double h, double r,
                       int use_adv, double adv)
{
    int64_t im = (i == 0) ? N - 1 : i - 1;
    int64_t ip = (i == N - 1) ? 0 : i + 1;
    double a = use_adv ? adv : v[i];
    return h * a * (v[ip] - v[im]) - r * (v[ip] - 2.0 * v[i] + v[im]);
}

static void newton_residual(const double *w, const double *un, int64_t N, double h,
                            double r, double theta, int bc, int use_adv, double adv, double *F)
{
    for (int64_t i = 0; i < N; ++i) {
        if (bc == BC_DIRICHLET && (i == 0 || i == N - 1)) { F[i] = 0.0; continue; }
        double Gw = newton_G(w, i, N, h, r, use_adv, adv);
        if (theta == 1.0) { F[i] = w[i] - un[i] + Gw; continue; }     /* Eq.11 as printed */
        double Gu = newton_G(un, i, N, h, r, use_adv, adv);
        F[i] = w[i] - un[i] + theta * Gw + (1.0 - theta) * Gu;
    }
}

static void newton_jacobian(const double *w, int64_t N, double h, double r, double theta, int bc,
                            int use_adv, double adv, double *sub, double *diag, double *sup)
{
    for (int64_t i = 0; i < N; ++i) {
        if (bc == BC_DIRICHLET && (i == 0 || i == N - 1)) { sub[i] = 0.0; diag[i] = 1.0; sup[i] = 0.0; continue; }
        int64_t im = (i == 0) ? N - 1 : i - 1;
        int64_t ip = (i == N - 1) ? 0 : i + 1;
        double a = use_adv ? adv : w[i];
        sub[i] = theta * (-h * a - r);
        diag[i] = 1.0 + theta * ((use_adv ? 0.0 : h * (w[ip] - w[im])) + 2.0 * r);
        sup[i] = theta * (h * a - r);
    }
}

/* Exposed for the pins (worked example, finite-difference Jacobian check). */
void oracle_newton_residual(const double *w, const double *un, int64_t N, double L, double nu,
                            double dt, double theta, int bc, int use_adv, double adv, double *F)
{
    double dx = grid_dx(N, L, bc);
    newton_residual(w, un, N, dt / (2.0 * dx), nu * dt / (dx * dx), theta, bc, use_adv, adv, F);
}
void oracle_newton_jacobian(const double *w, int64_t N, double L, double nu, double dt, double theta,
                            int bc, int use_adv, double adv, double *sub, double *diag, double *sup)
{
    double dx = grid_dx(N, L, bc);
    newton_jacobian(w, N, dt / (2.0 * dx), nu * dt / (dx * dx), theta, bc, use_adv, adv, sub, diag, sup);
}

/* One trajectory; returns the total number of Newton iterations (linear solves).
 * wk: 13N doubles. */
static int64_t newton_one(double *u, int64_t N, double dx, double nu, double dt, double theta,
                          int64_t n_steps, int bc, double tol, int max_iter, int use_adv, double adv,
                          double *wk)
{
    double *w = wk, *F = wk + N, *sub = wk + 2 * N, *diag = wk + 3 * N, *sup = wk + 4 * N,
           *rhs = wk + 5 * N, *x = wk + 6 * N, *wk2 = wk + 7 * N; /* 6N */
    double h = dt / (2.0 * dx), r = nu * dt / (dx * dx);
    int64_t total = 0;
    for (int64_t n = 0; n < n_steps; ++n) {
        for (int64_t i = 0; i < N; ++i) w[i] = u[i];
        for (int k = 0;; ++k) {
            newton_residual(w, u, N, h, r, theta, bc, use_adv, adv, F);
            double m = 0.0;
            for (int64_t i = 0; i < N; ++i) { double a = fabs(F[i]); if (!(a <= m)) m = a; }
            if (m < tol || k >= max_iter) break;
            newton_jacobian(w, N, h, r, theta, bc, use_adv, adv, sub, diag, sup);
            for (int64_t i = 0; i < N; ++i) rhs[i] = -F[i];
            if (bc == BC_PERIODIC) cyclic_sm(N, sub, diag, sup, rhs, x, wk2);
            else thomas(N, sub, diag, sup, rhs, x, wk2, wk2 + N);   /* identity rows at the ends */
            for (int64_t i = 0; i < N; ++i) w[i] = w[i] + x[i];
            ++total;
        }
        for (int64_t i = 0; i < N; ++i) u[i] = w[i];
    }
    return total;
}

/* B trajectories, in place; iters_out[b] (may be NULL) = Newton iterations summed over the steps. */
int oracle_newton_btcs(double *u, int64_t B, int64_t N, double L, const double *nu,
                       const double *dt, double theta, int64_t n_steps, int bc, double tol,
                       int max_iter, int use_adv, double adv, int64_t *iters_out, int nthreads)
{
    if (!u || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0) || max_iter < 0) return -1;
    if (!(theta >= 0.0 && theta <= 1.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel num_threads(nthreads)
    {
        double *wk = (double *)malloc((size_t)13 * (size_t)N * sizeof(double));
        if (!wk) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t b = 0; b < B; ++b) {
                int64_t it = newton_one(u + b * N, N, dx, nu[b], dt[b], theta, n_steps, bc, tol, max_iter,
                                        use_adv, adv, wk);
                if (iters_out) iters_out[b] = it;
            }
            free(wk);
        }
    }
    return fail ? -1 : 0;
}

/* ---------------------------------------------------------------------------
 * D12: the BTCS system of D4/D5 solved by GAUSS-SEIDEL sweeps
 * instead of the direct solve -- the paper's iterative variant (PAPER.md:129,
 * :245 "iterative Gauss-Seidel ... maximum residual falling below 1e-6", :339
 * "5-7 iterations per step").  Per step, rows (sub, diag, sup, rhs) from u^n as
 * in D4; x^0 = u^n; repeat: if max_i |rhs_i - (sub_i x_{i-1} + diag_i x_i +
 * sup_i x_{i+1})| < tol or k >= max_iter stop; else one lexicographic sweep
 * i = 0..N-1 (Dirichlet: 1..N-2), x_i <- (rhs_i - sub_i x_{i-1} - sup_i x_{i+1})
 * / diag_i with the newest values (periodic neighbours wrap).
 */
static int64_t gs_one(double *u, int64_t N, double dx, double nu, double dt, int64_t n_steps,
                      int bc, double tol, int max_iter, int use_adv, double adv, double *wk)
{
    double *sub = wk, *diag = wk + N, *sup = wk + 2 * N, *rhs = wk + 3 * N, *x = wk + 4 * N;
    int64_t lo = (bc == BC_DIRICHLET) ? 1 : 0, hi = (bc == BC_DIRICHLET) ? N - 1 : N;
    int64_t total = 0;
    for (int64_t n = 0; n < n_steps; ++n) {
        btcs_rows(u, N, dx, nu, dt, use_adv, adv, sub, diag, sup, rhs);
        for (int64_t i = 0; i < N; ++i) x[i] = u[i];
        for (int k = 0;; ++k) {
            double m = 0.0;
            for (int64_t i = lo; i < hi; ++i) {
                int64_t im = (i == 0) ? N - 1 : i - 1;
                int64_t ip = (i == N - 1) ? 0 : i + 1;
                double res = rhs[i] - (sub[i] * x[im] + diag[i] * x[i] + sup[i] * x[ip]);
                double a = fabs(res);
                if (!(a <= m)) m = a;
            }
            if (m < tol || k >= max_iter) break;
            for (int64_t i = lo; i < hi; ++i) {
                int64_t im = (i == 0) ? N - 1 : i - 1;
                int64_t ip = (i == N - 1) ? 0 : i + 1;
                x[i] = (rhs[i] - sub[i] * x[im] - sup[i] * x[ip]) / diag[i];
            }
            ++total;
        }
        for (int64_t i = lo; i < hi; ++i) u[i] = x[i];
    }
    return total;
}

int oracle_btcs_gs(double *u, int64_t B, int64_t N, double L, const double *nu, const double *dt,
                   int64_t n_steps, int bc, double tol, int max_iter, int use_adv, double adv,
                   int64_t *iters_out, int nthreads)
{
    if (!u || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0) || max_iter < 0) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel num_threads(nthreads)
    {
        double *wk = (double *)malloc((size_t)5 * (size_t)N * sizeof(double));
        if (!wk) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t b = 0; b < B; ++b) {
                int64_t it = gs_one(u + b * N, N, dx, nu[b], dt[b], n_steps, bc, tol, max_iter,
                                    use_adv, adv, wk);
                if (iters_out) iters_out[b] = it;
            }
            free(wk);
        }
    }
    return fail ? -1 : 0;
}

/* ---------------------------------------------------------------------------
 * D13 (SURVEY 8(f) NEXT-4c): DISCRETE ADJOINT of the forward-Euler scheme (D3), the
 * reverse-mode derivative the paper obtains from JAX.
 * One step is u^{n+1} = Phi(u^n), Phi_i = u_i + dt F_i(u) (D2).  With cx = dt/dx,
 * rr = nu dt/dx^2 and the upwind switch held fixed (it is locally constant):
 *   u_i > 0 :  dPhi_i/du_{i-1} = cx u_i + rr,  dPhi_i/du_i = 1 - cx (2u_i - u_{i-1}) - 2rr,  dPhi_i/du_{i+1} = rr
 *   u_i <= 0:  dPhi_i/du_{i-1} = rr,  dPhi_i/du_i = 1 - cx (u_{i+1} - 2u_i) - 2rr,  dPhi_i/du_{i+1} = rr - cx u_i
 * Dirichlet end nodes: Phi_i = u_i (row of the identity).  Given lam^N = dJ/du^N, the adjoint
 * recursion is lam^n = (dPhi/du (u^n))^T lam^{n+1}, n = N-1..0, and lam^0 = dJ/du^0 (dt, nu fixed).
 * The forward states are recomputed and stored (N * n_steps doubles per trajectory).
 * Test hook use_adv as in D2 (the map is then linear and the adjoint its exact transpose).
 */
static void adjoint_step(const double *u, const double *lam, double *out, int64_t N, double cx,
                         double rr, int bc, int use_adv, double adv)
{
    /* out_j = sum_i dPhi_i/du_j lam_i: scatter row i of the Jacobian into columns */
    for (int64_t j = 0; j < N; ++j) out[j] = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        if (bc == BC_DIRICHLET && (i == 0 || i == N - 1)) { out[i] += lam[i]; continue; }
        int64_t im = (i == 0) ? N - 1 : i - 1;
        int64_t ip = (i == N - 1) ? 0 : i + 1;
        double a = use_adv ? adv : u[i];
        double dm, d0, dp;
        if (a > 0.0) {
            dm = cx * a + rr;
            d0 = 1.0 - cx * a - (use_adv ? 0.0 : cx * (u[i] - u[im])) - 2.0 * rr;
            dp = rr;
        } else {
            dm = rr;
            d0 = 1.0 + cx * a - (use_adv ? 0.0 : cx * (u[ip] - u[i])) - 2.0 * rr;
            dp = rr - cx * a;
        }
        out[im] += dm * lam[i];
        out[i] += d0 * lam[i];
        out[ip] += dp * lam[i];
    }
}

int oracle_explicit_adjoint(const double *u0, double *lam, int64_t B, int64_t N, double L,
                            const double *nu, const double *dt, int64_t n_steps, int bc, int use_adv,
                            double adv, int nthreads)
{
    if (!u0 || !lam || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 1)
    for (int64_t b = 0; b < B; ++b) {
        double *st = (double *)malloc((size_t)(n_steps + 7) * (size_t)N * sizeof(double));
        if (!st) {
#pragma omp atomic write
            fail = 1;
            continue;
        }
        double *wk = st + (size_t)(n_steps + 1) * N; /* 5N + N */
        for (int64_t i = 0; i < N; ++i) st[i] = u0[b * N + i];
        for (int64_t n = 0; n < n_steps; ++n) {      /* forward, storing u^0..u^{n_steps} */
            double *cur = st + (size_t)(n + 1) * N;
            for (int64_t i = 0; i < N; ++i) cur[i] = st[(size_t)n * N + i];
            explicit_one(cur, N, dx, nu[b], dt[b], 1, bc, SCHEME_EULER, use_adv, adv, wk);
        }
        double cx = dt[b] / dx, rr = nu[b] * dt[b] / (dx * dx);
        double *tmp = wk + 5 * N;
        for (int64_t n = n_steps - 1; n >= 0; --n) {
            adjoint_step(st + (size_t)n * N, lam + b * N, tmp, N, cx, rr, bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) lam[b * N + i] = tmp[i];
        }
        free(st);
    }
    return fail ? -1 : 0;
}

/* ---------------------------------------------------------------------------
 * D14: DISCRETE ADJOINT of the classical RK4 scheme of D3
 * (Eq.22; gradients of "the numerical solution").
 * One step:  y1 = u, k_s = F(y_s), y2 = u + dt/2 k1, y3 = u + dt/2 k2, y4 = u + dt k3,
 *            u' = u + dt/6 (k1 + 2 k2 + 2 k3 + k4).
 * Reverse mode, given lam' = dJ/du' (J_s = dF/dy at y_s, the upwind switch held fixed):
 *   kb4 = dt/6 lam', kb3 = dt/3 lam', kb2 = dt/3 lam', kb1 = dt/6 lam', ub = lam';
 *   yb4 = J4^T kb4:  ub += yb4, kb3 += dt   yb4;
 *   yb3 = J3^T kb3:  ub += yb3, kb2 += dt/2 yb3;
 *   yb2 = J2^T kb2:  ub += yb2, kb1 += dt/2 yb2;
 *   yb1 = J1^T kb1:  ub += yb1;                         lam = ub.
 * Rows of J = dF/dy (D2: F_i = -y_i g_i/dx + nu (y_{i+1} - 2 y_i + y_{i-1})/dx^2):
 *   y_i > 0 :  dF_i/dy_{i-1} =  y_i/dx + nu/dx^2,  dF_i/dy_i = -(2 y_i - y_{i-1})/dx - 2 nu/dx^2,  dF_i/dy_{i+1} = nu/dx^2
 *   y_i <= 0:  dF_i/dy_{i-1} =  nu/dx^2,  dF_i/dy_i = -(y_{i+1} - 2 y_i)/dx - 2 nu/dx^2,  dF_i/dy_{i+1} = -y_i/dx + nu/dx^2
 * Dirichlet end nodes: F = 0, zero rows (and u' = u there, which `ub = lam'` carries).
 * Test hook use_adv as in D2 (constant speed a: the rows are (a/dx + nu/dx^2, -a/dx - 2 nu/dx^2,
 * nu/dx^2) for a > 0, mirrored otherwise; the step is then linear and the adjoint its transpose).
 */
static void rhs_jacT(const double *y, const double *v, double *out, int64_t N, double dx, double nu,
                     int bc, int use_adv, double adv)
{
    /* out_j = sum_i dF_i/dy_j v_i: scatter row i of J into columns */
    double d2 = nu / (dx * dx);
    for (int64_t j = 0; j < N; ++j) out[j] = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        if (bc == BC_DIRICHLET && (i == 0 || i == N - 1)) continue;
        int64_t im = (i == 0) ? N - 1 : i - 1;
        int64_t ip = (i == N - 1) ? 0 : i + 1;
        double a = use_adv ? adv : y[i];
        double jm, j0, jp;
        if (a > 0.0) {
            jm = a / dx + d2;
            j0 = -a / dx - (use_adv ? 0.0 : (y[i] - y[im]) / dx) - 2.0 * d2;
            jp = d2;
        } else {
            jm = d2;
            j0 = a / dx - (use_adv ? 0.0 : (y[ip] - y[i]) / dx) - 2.0 * d2;
            jp = -a / dx + d2;
        }
        out[im] += jm * v[i];
        out[i] += j0 * v[i];
        out[ip] += jp * v[i];
    }
}

int oracle_rk4_adjoint(const double *u0, double *lam, int64_t B, int64_t N, double L,
                       const double *nu, const double *dt, int64_t n_steps, int bc, int use_adv,
                       double adv, int nthreads)
{
    if (!u0 || !lam || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 1)
    for (int64_t b = 0; b < B; ++b) {
        /* states u^0..u^{n_steps-1}, then 5N (explicit_one) + 3 stage values + 4 kb + ub + yb */
        double *st = (double *)malloc((size_t)(n_steps + 15) * (size_t)N * sizeof(double));
        if (!st) {
#pragma omp atomic write
            fail = 1;
            continue;
        }
        double *wk = st + (size_t)(n_steps + 1) * N;
        double *y2 = wk + 5 * N, *y3 = wk + 6 * N, *y4 = wk + 7 * N, *kk = wk + 8 * N;
        double *kb1 = wk + 9 * N, *kb2 = wk + 10 * N, *kb3 = wk + 11 * N, *kb4 = wk + 12 * N, *yb = wk + 13 * N;
        double h = dt[b];
        for (int64_t i = 0; i < N; ++i) st[i] = u0[b * N + i];
        for (int64_t n = 0; n + 1 < n_steps; ++n) {  /* forward, storing u^0..u^{n_steps-1} */
            double *cur = st + (size_t)(n + 1) * N;
            for (int64_t i = 0; i < N; ++i) cur[i] = st[(size_t)n * N + i];
            explicit_one(cur, N, dx, nu[b], h, 1, bc, SCHEME_RK4, use_adv, adv, wk);
        }
        double *ub = lam + b * N;
        for (int64_t n = n_steps - 1; n >= 0; --n) {
            const double *u = st + (size_t)n * N;
            /* the stage values of step n again, exactly as explicit_one forms them */
            rhs_F(u, kk, N, dx, nu[b], bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) y2[i] = u[i] + 0.5 * h * kk[i];
            rhs_F(y2, kk, N, dx, nu[b], bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) y3[i] = u[i] + 0.5 * h * kk[i];
            rhs_F(y3, kk, N, dx, nu[b], bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) y4[i] = u[i] + h * kk[i];
            for (int64_t i = 0; i < N; ++i) {
                kb4[i] = h / 6.0 * ub[i];
                kb3[i] = h / 3.0 * ub[i];
                kb2[i] = h / 3.0 * ub[i];
                kb1[i] = h / 6.0 * ub[i];
            }
            rhs_jacT(y4, kb4, yb, N, dx, nu[b], bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) { ub[i] += yb[i]; kb3[i] += h * yb[i]; }
            rhs_jacT(y3, kb3, yb, N, dx, nu[b], bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) { ub[i] += yb[i]; kb2[i] += 0.5 * h * yb[i]; }
            rhs_jacT(y2, kb2, yb, N, dx, nu[b], bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) { ub[i] += yb[i]; kb1[i] += 0.5 * h * yb[i]; }
            rhs_jacT(u, kb1, yb, N, dx, nu[b], bc, use_adv, adv);
            for (int64_t i = 0; i < N; ++i) ub[i] += yb[i];
        }
        free(st);
    }
    return fail ? -1 : 0;
}

/* ---------------------------------------------------------------------------
 * D15: DISCRETE ADJOINT of the lagged upwind BTCS scheme of D4-D6 ("gradients of the
 * numerical solution"; VERDICT r01 "missing" item 6).  One step solves A(u) u' = u, where row i of A depends on
 * u_i alone (D4).  Differentiating,  A du' + diag(D) du = du  with
 *   D_i = d/du_i [ sub_i(u_i) u'_{i-1} + diag_i(u_i) u'_i + sup_i(u_i) u'_{i+1} ]
 *       = (dt/dx) (u'_i - u'_{i-1})   if u_i > 0,      (dt/dx) (u'_{i+1} - u'_i)   otherwise
 * (sub' = -dt/dx [u>0], diag' = dt/dx sign(u), sup' = dt/dx [u<=0]; the upwind switch held fixed), so
 * du' = A^{-1} (I - D) du and the reverse step is   mu = A^{-T} lam',   lam_i = (1 - D_i) mu_i.
 * Dirichlet: the system is written on all N nodes with identity rows at the two end nodes (x_0 = u_0), D = 0
 * there; A^T mu = lam' then reads: interior j:  sup_{j-1} mu_{j-1} + diag_j mu_j + sub_{j+1} mu_{j+1} = lam'_j
 * (neighbours that are end nodes drop out), and mu_0 = lam'_0 - sub_1 mu_1, mu_{N-1} = lam'_{N-1} - sup_{N-2} mu_{N-2}.
 * Periodic: the transposed cyclic system (Sherman-Morrison, D6, on the transposed rows).
 * Test hook use_adv: A is then constant, D = 0, and the adjoint is the exact transpose of the linear step.
 */
int oracle_btcs_adjoint(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                        const double *dt, int64_t n_steps, int bc, int use_adv, double adv, int nthreads)
{
    if (!u0 || !lam || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 1)
    for (int64_t b = 0; b < B; ++b) {
        /* states u^0..u^{n_steps}, 11N for btcs_one, then 4N rows + 3N transposed + N mu + 6N cyclic scratch */
        double *st = (double *)malloc((size_t)(n_steps + 1 + 11 + 14) * (size_t)N * sizeof(double));
        if (!st) {
#pragma omp atomic write
            fail = 1;
            continue;
        }
        double *wk = st + (size_t)(n_steps + 1) * N;
        double *sub = wk + 11 * N, *diag = sub + N, *sup = diag + N, *rhs = sup + N;
        double *subT = rhs + N, *supT = subT + N, *mu = supT + N, *wk2 = mu + N; /* wk2: 6N */
        for (int64_t i = 0; i < N; ++i) st[i] = u0[b * N + i];
        for (int64_t n = 0; n < n_steps; ++n) {      /* forward, storing u^0..u^{n_steps} */
            double *cur = st + (size_t)(n + 1) * N;
            for (int64_t i = 0; i < N; ++i) cur[i] = st[(size_t)n * N + i];
            btcs_one(cur, N, dx, nu[b], dt[b], 1, bc, use_adv, adv, wk);
        }
        double cx = dt[b] / dx;
        double *l = lam + b * N;
        for (int64_t n = n_steps - 1; n >= 0; --n) {
            const double *u = st + (size_t)n * N, *up = st + (size_t)(n + 1) * N;
            btcs_rows(u, N, dx, nu[b], dt[b], use_adv, adv, sub, diag, sup, rhs);
            if (bc == BC_PERIODIC) {
                for (int64_t j = 0; j < N; ++j) {      /* rows of A^T, cyclic indexing */
                    subT[j] = sup[(j == 0) ? N - 1 : j - 1];
                    supT[j] = sub[(j == N - 1) ? 0 : j + 1];
                }
                cyclic_sm(N, subT, diag, supT, l, mu, wk2);
            } else {
                int64_t m = N - 2;                      /* interior unknowns 1..N-2 */
                for (int64_t j = 1; j <= N - 2; ++j) {
                    subT[j] = sup[j - 1];               /* not referenced for j = 1 */
                    supT[j] = sub[j + 1];               /* not referenced for j = N-2 */
                }
                thomas(m, subT + 1, diag + 1, supT + 1, l + 1, mu + 1, wk2, wk2 + N);
                mu[0] = l[0] - sub[1] * mu[1];
                mu[N - 1] = l[N - 1] - sup[N - 2] * mu[N - 2];
            }
            for (int64_t i = 0; i < N; ++i) {
                double D = 0.0;
                if (!use_adv && !(bc == BC_DIRICHLET && (i == 0 || i == N - 1))) {
                    int64_t im = (i == 0) ? N - 1 : i - 1;
                    int64_t ip = (i == N - 1) ? 0 : i + 1;
                    D = (u[i] > 0.0) ? cx * (up[i] - up[im]) : cx * (up[ip] - up[i]);
                }
                l[i] = (1.0 - D) * mu[i];
            }
        }
        free(st);
    }
    return fail ? -1 : 0;
}

/* ---------------------------------------------------------------------------
 * D16: reverse mode of the Newton / theta-scheme of D11 (PAPER.md:137-159 Eq.10-15 for the scheme; :231, :261 for
 * the purpose: "gradients of the numerical solution").  One step maps u = u^n to the root w = u^{n+1} of
 *   F_i(w; u) = w_i - u_i + theta G_i(w) + (1 - theta) G_i(u)   (interior / periodic rows; F_i = w_i - u_i at
 * Dirichlet end nodes), so by the implicit-function theorem dw/du = -(dF/dw)^{-1} dF/du with
 *   dF/dw = J(w)                                   (newton_jacobian at the root: identity rows at Dirichlet ends),
 *   dF/du = -I + (1 - theta) M G'(u)               (M: zero rows at Dirichlet end nodes),
 *   G'(v) row i = (-h v_i - r,  h (v_{i+1} - v_{i-1}) + 2 r,  h v_i - r)   on columns (i-1, i, i+1), cyclic.
 * Reverse mode, given lam' = dJ/du^{n+1}:
 *   J(u^{n+1})^T mu = lam',        lam_i = mu_i - (1 - theta) (G'(u^n)^T M mu)_i,
 *   (G'(v)^T x)_i = (h v_{i-1} - r) x_{i-1} + (h (v_{i+1} - v_{i-1}) + 2 r) x_i + (-h v_{i+1} - r) x_{i+1}.
 * This differentiates the map the CONVERGED iteration defines; the forward sweep below is newton_one with the
 * caller's tol and max_iter (use a tol near rounding for gradients), all states stored.
 * J^T: row j = (sup_{j-1}, diag_j, sub_{j+1}); with identity rows at Dirichlet ends sub_0 = sup_{N-1} = 0, so the
 * wrap entries vanish and the plain Thomas solve of all N rows applies; periodic: Sherman-Morrison (D6).
 * Test hook use_adv: G is linear (multiplier adv), the step is u' = S u and the adjoint is S^T.
 */
int oracle_newton_adjoint(const double *u0, double *lam, int64_t B, int64_t N, double L, const double *nu,
                          const double *dt, double theta, int64_t n_steps, int bc, double tol, int max_iter,
                          int use_adv, double adv, int nthreads)
{
    if (!u0 || !lam || !nu || !dt || B < 1 || N < 3 || n_steps < 0 || !(L > 0.0) || max_iter < 0) return -1;
    if (!(theta >= 0.0 && theta <= 1.0)) return -1;
    if (bc != BC_PERIODIC && bc != BC_DIRICHLET) return -1;
    double dx = grid_dx(N, L, bc);
    int fail = 0;
    if (nthreads < 1) nthreads = 1;
    (void)nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 1)
    for (int64_t b = 0; b < B; ++b) {
        /* states u^0..u^{n_steps}, 13N for newton_one, 3N rows, 2N transposed, 2N mu / masked mu, 6N cyclic scratch */
        double *st = (double *)malloc((size_t)(n_steps + 1 + 13 + 13) * (size_t)N * sizeof(double));
        if (!st) {
#pragma omp atomic write
            fail = 1;
            continue;
        }
        double *wk = st + (size_t)(n_steps + 1) * N;
        double *sub = wk + 13 * N, *diag = sub + N, *sup = diag + N;
        double *subT = sup + N, *supT = subT + N, *mu = supT + N, *mm = mu + N, *wk2 = mm + N; /* wk2: 6N */
        double h = dt[b] / (2.0 * dx), r = nu[b] * dt[b] / (dx * dx);
        for (int64_t i = 0; i < N; ++i) st[i] = u0[b * N + i];
        for (int64_t n = 0; n < n_steps; ++n) {      /* forward, storing u^0..u^{n_steps} */
            double *cur = st + (size_t)(n + 1) * N;
            for (int64_t i = 0; i < N; ++i) cur[i] = st[(size_t)n * N + i];
            newton_one(cur, N, dx, nu[b], dt[b], theta, 1, bc, tol, max_iter, use_adv, adv, wk);
        }
        double *l = lam + b * N;
        for (int64_t n = n_steps - 1; n >= 0; --n) {
            const double *u = st + (size_t)n * N, *up = st + (size_t)(n + 1) * N;
            newton_jacobian(up, N, h, r, theta, bc, use_adv, adv, sub, diag, sup);
            for (int64_t j = 0; j < N; ++j) {        /* rows of J^T, cyclic indexing (zero wrap for Dirichlet) */
                subT[j] = sup[(j == 0) ? N - 1 : j - 1];
                supT[j] = sub[(j == N - 1) ? 0 : j + 1];
            }
            if (bc == BC_PERIODIC) cyclic_sm(N, subT, diag, supT, l, mu, wk2);
            else thomas(N, subT, diag, supT, l, mu, wk2, wk2 + N);
            for (int64_t i = 0; i < N; ++i)
                mm[i] = (bc == BC_DIRICHLET && (i == 0 || i == N - 1)) ? 0.0 : mu[i];     /* M mu */
            for (int64_t i = 0; i < N; ++i) {
                int64_t im = (i == 0) ? N - 1 : i - 1;
                int64_t ip = (i == N - 1) ? 0 : i + 1;
                double am = use_adv ? adv : u[im], ap = use_adv ? adv : u[ip];
                double dg = use_adv ? 0.0 : h * (u[ip] - u[im]);
                double gt = (h * am - r) * mm[im] + (dg + 2.0 * r) * mm[i] + (-h * ap - r) * mm[ip];
                l[i] = mu[i] - (1.0 - theta) * gt;
            }
        }
        free(st);
    }
    return fail ? -1 : 0;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
