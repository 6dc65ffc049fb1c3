// adjoint.cu -- SURVEY 8(f) NEXT-4c: discrete adjoint of the forward-Euler scheme, i.e. the
// reverse-mode derivative dJ/du^0 = (du^N/du^0)^T dJ/du^N that the paper gets from JAX autodiff
// (PAPER.md:231, :261, :409); D13.
//
// One forward step is u^{n+1} = Phi(u^n), Phi_i = u_i + dt F_i(u) (D2/D3).  With cx = dt/dx,
// rr = nu dt/dx^2 and the upwind switch held fixed, row i of dPhi/du is
//   u_i > 0 :  (cx u_i + rr,  1 - cx (2u_i - u_{i-1}) - 2rr,  rr)
//   u_i <= 0:  (rr,  1 - cx (u_{i+1} - 2u_i) - 2rr,  rr - cx u_i)          on columns (i-1, i, i+1)
// and the identity row for Dirichlet end nodes.  One adjoint step gathers column j:
//   lam^n_j = dPhi_{j-1}/du_j lam_{j-1} + dPhi_j/du_j lam_j + dPhi_{j+1}/du_j lam_{j+1}   at u^n.
// The forward states u^0..u^{N-1} come from the trajectory output of the explicit kernel (one
// snapshot per step, written by the RESIDENT kernel from its on-chip state); the backward sweep is one
// streaming launch per step (HBM-bound: reads u^n and lam, writes lam).
#include "common.cuh"

namespace burgers {
namespace {

template <typename T>
__global__ void __launch_bounds__(256)
adjoint_step_kernel(const T *__restrict__ u, const T *__restrict__ lam, T *__restrict__ out,
                    const T *__restrict__ nu, const T *__restrict__ dt, int64_t N, double inv_dx, int bc) {
    const int64_t b = blockIdx.y;
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const double dtb = (double)dt[b];
    const T cx = (T)(dtb * inv_dx);
    const T rr = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    const T *ur = u + b * N, *lr = lam + b * N;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const int64_t jm = (j == 0) ? N - 1 : j - 1, jp = (j == N - 1) ? 0 : j + 1;
    const T um = ur[jm], uj = ur[j], up = ur[jp];
    T acc;
    // row j (its diagonal entry)
    if (dirichlet && (j == 0 || j == N - 1)) {
        acc = lr[j];
    } else {
        const T g = (uj > T(0)) ? (uj - um) : (up - uj);
        const T d0 = T(1) - cx * ((uj > T(0)) ? uj : -uj) - cx * g - T(2) * rr;
        acc = d0 * lr[j];
    }
    // row j-1, column j: its "right" entry
    if (!(dirichlet && (j == 0 || jm == 0))) {
        const T dp = (um > T(0)) ? rr : rr - cx * um;
        acc += dp * lr[jm];
    }
    // row j+1, column j: its "left" entry
    if (!(dirichlet && (j == N - 1 || jp == N - 1))) {
        const T dm = (up > T(0)) ? cx * up + rr : rr;
        acc += dm * lr[jp];
    }
    out[b * N + j] = acc;
}

}  // namespace

template <typename T>
int launch_adjoint_steps(const T *u0, const T *states, T *lam, T *pong, int64_t B, int64_t N, double dx,
                         const T *nu, const T *dt, int64_t n_steps, int bc, cudaStream_t s) {
    if (B > 65535) return BURGERS_ERR_SHAPE;
    dim3 grid((unsigned)((N + 255) / 256), (unsigned)B);
    T *cur = lam, *nxt = pong;
    for (int64_t n = n_steps - 1; n >= 0; --n) {
        const T *un = (n == 0) ? u0 : states + (size_t)(n - 1) * (size_t)B * (size_t)N;
        adjoint_step_kernel<T><<<grid, 256, 0, s>>>(un, cur, nxt, nu, dt, N, 1.0 / dx, bc);
        T *tmp = cur; cur = nxt; nxt = tmp;
    }
    int st = last_launch_status();
    if (st != BURGERS_OK) return st;
    if (cur != lam &&
        cudaMemcpyAsync(lam, cur, (size_t)B * N * sizeof(T), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
        return BURGERS_ERR_CUDA;
    return BURGERS_OK;
}

template int launch_adjoint_steps<float>(const float *, const float *, float *, float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, cudaStream_t);
template int launch_adjoint_steps<double>(const double *, const double *, double *, double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, cudaStream_t);

}  // namespace burgers
