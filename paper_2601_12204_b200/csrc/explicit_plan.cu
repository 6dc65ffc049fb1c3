// explicit_plan.cu -- host-side geometry of the explicit plans (no device code).
#include "common.cuh"

namespace burgers {

static bool valid_ppt(int p) { return p == 1 || p == 2 || p == 4 || p == 8 || p == 16 || p == 32; }

static bool resident_fit(int is_f64, int64_t N, int scheme, int P, ExplicitGeom *g) {
    if (N % P) return false;
    const int64_t nth = N / P;
    if (nth > explicit_max_threads(is_f64, P, scheme)) return false;
    g->plan = BURGERS_PLAN_RESIDENT;
    g->P = P;
    g->nth = (int)nth;
    g->block = (int)((nth + 31) / 32 * 32);
    g->tblock = 0; g->halo = 0; g->W = N; g->tiles = 1;
    return true;
}

static bool resident_geometry(int is_f64, int64_t N, int scheme, int ppt, ExplicitGeom *g) {
    if (ppt) return resident_fit(is_f64, N, scheme, ppt, g);
    // Prefer many points per thread (few halo exchanges per update) while a CTA still has a full warp.
    // Measured on B200 (ms, 8192-16384 trajectories; P = 8 / 16 / 32):
    //   fp32 Euler  N=512: 1.34 / 1.07 / 2.48   N=1024: 5.14 / 4.38 / 4.93   N=2048: 10.3 / 8.67 / 8.21
    //   fp32 RK4    N=512: 1.42 / 1.29 / 2.53   N=1024: 5.50 / 5.19 / 5.00   N=4096: 11.2 / 10.6 / 9.93
    //   fp64 Euler  N=512: 1.85 / 1.66 / 3.31   N=2048: 14.3 / 12.8 / 13.1   N=4096: 14.8 / 13.0 / 13.1
    //   fp64 RK4    N=512: 2.63 / 2.53 / 4.84   N=2048: 20.6 / 18.6 / 19.5   N=4096: 22.3 / 18.8 / 19.5
    // hence: P = 32 needs two warps for Euler, one for fp32 RK4, and comes after P = 16 for fp64 RK4 (254
    // registers); the smaller P need one full warp.
    const bool rk4 = (scheme == BURGERS_SCHEME_RK4);
    const int order_default[6] = {32, 16, 8, 4, 2, 1}, order_f64_rk4[6] = {16, 32, 8, 4, 2, 1};
    const int *order = (rk4 && is_f64) ? order_f64_rk4 : order_default;
    for (int i = 0; i < 6; ++i) {
        const int P = order[i];
        const int min_threads = (P == 32 && !rk4) ? 64 : 32;
        if (N / P >= min_threads && resident_fit(is_f64, N, scheme, P, g)) return true;
    }
    for (int P = 1; P <= 32; P *= 2)
        if (resident_fit(is_f64, N, scheme, P, g)) return true;
    return false;
}

static bool tiled_geometry(int is_f64, int64_t N, int bc, int scheme, int tblock, int ppt,
                           ExplicitGeom *g) {
    const int V = is_f64 ? 2 : 4;
    const int radius = (scheme == BURGERS_SCHEME_RK4) ? 4 : 1;
    // Defaults measured on C4a's grid (N = 2^24; ms, P = 16 -> P = 32 at the tblock below):
    //   fp32 Euler (2 000 steps) tblock  64 / 128 / 256 / 400:  9.43 -> 9.56 / 9.10 / 8.87 / 9.39
    //   fp64 Euler (1 000 steps) tblock  64 / 128 / 256:        7.85 -> 7.55 / 7.35 / 7.25
    //   fp32 RK4   (  400 steps) tblock  16 /  32 /  64:        8.00 -> 7.89 / 7.58 / 7.46
    //   fp64 RK4   (  200 steps) tblock  16 /  32 /  64:        7.59 -> 8.19 / 7.68 / 7.37
    // hence 32 points per thread, 256 (Euler) / 64 (RK4) steps per launch.
    int P = ppt ? ppt : 32;
    // Dirichlet: the frozen end nodes must be the first / last point of a thread
    if (bc == BURGERS_BC_DIRICHLET) {
        if (ppt && N % P) return false;
        while (N % P) P /= 2;
    }
    int nth = 256;
    const int maxt = explicit_max_threads(is_f64, P, scheme);
    if (nth > maxt) nth = maxt;
    if (tblock <= 0) tblock = (scheme == BURGERS_SCHEME_RK4) ? (P == 32 ? 64 : 16) : (P == 32 ? 256 : 64);
    const int64_t Wt = (int64_t)nth * P;
    const int q = P > V ? P : V;
    int halo = 0;
    for (;;) {
        halo = (tblock * radius + q - 1) / q * q;
        if (Wt - 2 * halo >= Wt / 4 && Wt - 2 * halo >= 1) break;
        if (tblock == 1) return false;
        tblock /= 2;
    }
    g->plan = BURGERS_PLAN_TILED;
    g->P = P; g->nth = nth; g->block = nth;
    g->tblock = tblock; g->halo = halo; g->W = Wt - 2 * halo;
    g->tiles = (N + g->W - 1) / g->W;
    return true;
}

int explicit_geometry(int is_f64, int64_t B, int64_t N, int bc, int scheme, int plan, int tblock,
                      int ppt, ExplicitGeom *g) {
    (void)B;
    if (ppt && !valid_ppt(ppt)) return BURGERS_ERR_PLAN;
    if (tblock < 0) return BURGERS_ERR_PLAN;
    if (plan == BURGERS_PLAN_AUTO || plan == BURGERS_PLAN_RESIDENT) {
        if (resident_geometry(is_f64, N, scheme, ppt, g)) return BURGERS_OK;
        if (plan == BURGERS_PLAN_RESIDENT) return BURGERS_ERR_PLAN;
    }
    if (plan == BURGERS_PLAN_AUTO || plan == BURGERS_PLAN_TILED)
        return tiled_geometry(is_f64, N, bc, scheme, tblock, ppt, g) ? BURGERS_OK : BURGERS_ERR_PLAN;
    return BURGERS_ERR_ENUM;
}

}  // namespace burgers
