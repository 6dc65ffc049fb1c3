/* A plain C99 consumer of include/burgers.h (compiled and run by tests/test_abi_cpu.py): the header must be
 * valid C, the library must link without any C++ or torch symbol on the caller's side, and argument errors
 * must come back as status codes before any device work (so this runs on a box without a GPU).
 * `c_abi_client run` (tests/test_gpu_parity.py, needs a device) drives the kernels from C: the whole hot path
 * on host buffers (burgers_solve_host_f64: CFL step + 50 Euler steps, then 7 BTCS steps) on a 1 x 64 periodic
 * grid, results printed for the test to compare with the oracle. */
#include <math.h>
#include <stdio.h>
#include <string.h>

#include "burgers.h"

static int run(void) {
    double u[64], v[64], nu[1] = {0.05}, dt[1];
    const double two_pi = 6.283185307179586;
    int i, st;
    for (i = 0; i < 64; ++i) u[i] = v[i] = sin(two_pi * i / 64.0) + 0.25;
    st = burgers_solve_host_f64(u, 1, 64, two_pi, nu, 0.4, 50, BURGERS_BC_PERIODIC, BURGERS_OP_EXPLICIT,
                                BURGERS_SCHEME_EULER, dt);
    if (st != BURGERS_OK) { printf("status %d %s\n", st, burgers_strerror(st)); return 1; }
    printf("dt %.17g\neuler", dt[0]);
    for (i = 0; i < 64; ++i) printf(" %.17g", u[i]);
    st = burgers_solve_host_f64(v, 1, 64, two_pi, nu, 4.0, 7, BURGERS_BC_PERIODIC, BURGERS_OP_BTCS, 0, dt);
    if (st != BURGERS_OK) { printf("status %d %s\n", st, burgers_strerror(st)); return 1; }
    printf("\ndt %.17g\nbtcs", dt[0]);
    for (i = 0; i < 64; ++i) printf(" %.17g", v[i]);
    printf("\n");
    return 0;
}

int main(int argc, char **argv) {
    double u[8] = {0}, nu[1] = {0.1}, dt[1] = {0.1};
    float uf[8] = {0}, nuf[1] = {0.1f};
    int bad = 0;
    if (argc > 1 && strcmp(argv[1], "run") == 0) return run();
    bad += burgers_explicit_f64(u, 1, 8, -1.0, nu, dt, 1, BURGERS_BC_PERIODIC, BURGERS_SCHEME_EULER, NULL, 0, NULL) != BURGERS_ERR_VALUE;
    bad += burgers_btcs_f64(NULL, 1, 8, 1.0, nu, dt, 1, BURGERS_BC_PERIODIC, NULL, 0, NULL) != BURGERS_ERR_NULL;
    bad += burgers_btcs_f64(u, 1, 2, 1.0, nu, dt, 1, BURGERS_BC_PERIODIC, NULL, 0, NULL) != BURGERS_ERR_SHAPE;
    bad += dt_from_cfl_f32(uf, 1, 8, 1.0, nuf, 0.4, 7, nuf, NULL) != BURGERS_ERR_ENUM;
    bad += burgers_solve_host_f32(uf, 1, 8, 1.0, nuf, 0.4, 1, BURGERS_BC_DIRICHLET, BURGERS_OP_CFL, 0, NULL) != BURGERS_ERR_ENUM;
    bad += burgers_workspace_bytes(BURGERS_OP_BTCS, 1, 1, (int64_t)1 << 22, BURGERS_BC_PERIODIC, 0, BURGERS_PLAN_AUTO) == 0;
    bad += burgers_plan_query(BURGERS_OP_BTCS, 1, 4096, 2048, BURGERS_BC_PERIODIC, 0) != BURGERS_PLAN_HYBRID;
    bad += strlen(burgers_strerror(BURGERS_ERR_WORKSPACE)) == 0;
    printf("version %d bad %d\n", burgers_version(), bad);
    return bad;
}
