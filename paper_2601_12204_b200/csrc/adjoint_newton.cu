// adjoint_newton.cu -- reverse mode of the Newton / theta-scheme of newton.cu (D16; the scheme:
// PAPER.md:137-159 Eq.10-15; the purpose: "gradients of the numerical solution").
//
// One forward step maps u = u^n to the root w = u^{n+1} of F(w; u) = w - u + theta G(w) + (1 - theta) G(u) (identity
// rows at Dirichlet end nodes), G_i(v) = h v_i (v_{i+1} - v_{i-1}) - r (v_{i+1} - 2 v_i + v_{i-1}), h = dt/(2 dx),
// r = nu dt/dx^2.  By the implicit-function theorem (dF/dw = J(w), dF/du = -I + (1 - theta) M G'(u), M = zero rows at
// Dirichlet ends) the reverse step is
//     J(u^{n+1})^T mu = lam^{n+1},
//     lam^n_i = mu_i - (1 - theta) [ (h u_{i-1} - r) m_{i-1} + (h (u_{i+1} - u_{i-1}) + 2 r) m_i + (-h u_{i+1} - r) m_{i+1} ],
// m = M mu, u = u^n, neighbours cyclic.  Row j of J^T is (sup_{j-1}, diag_j, sub_{j+1}) with J's rows
//     sub_i = theta (-h w_i - r),  diag_i = 1 + theta (h (w_{i+1} - w_{i-1}) + 2 r),  sup_i = theta (h w_i - r)
// (Eq.14 / reading Q5) at w = u^{n+1}; identity rows of J at Dirichlet ends make the wrap entries of J^T zero, so
// the cyclic form serves both boundary types.  Like J itself, J^T is eliminated without pivoting (cell Peclet
// number <= 2, D11) with the machinery of the forward solver (btcs_common.cuh).
//
// This is the derivative of the map the CONVERGED iteration defines: run the forward sweep with a tolerance
// near rounding.  The forward states u^1 .. u^n come from burgers_newton_traj_* (one snapshot per step).  Plans:
//   RESIDENT  one CTA per system, lam in registers across the steps, any N that fits one CTA.  Exact partitions
//             (N == P * threads): the STAGED kernel (states through a ring of three shared-memory stages); ragged
//             partitions: u^{n+1} in registers, u^n streamed in one step ahead;
//   THOMAS    one thread per system on [B][N] as it lies (the general-shape fallback), Sherman-Morrison for
//             periodic systems; scratch 3 B N.
#include "btcs_common.cuh"

namespace burgers {
namespace {

using namespace btcs;

constexpr int adjn_max_threads(int bytes, int P) {
    int regs = P * (bytes / 4) * 6 + 56;
    int t = 1024;
    while (t > 32 && t * regs > 65536) t /= 2;
    return t;
}

template <typename T, int P, bool RAGGED>
__global__ void __launch_bounds__(adjn_max_threads(sizeof(T), P))
adjoint_newton_resident_kernel(const T *__restrict__ u0, const T *__restrict__ states, T *__restrict__ lam,
                               const T *__restrict__ nu, const T *__restrict__ dt, int64_t B, int N, double inv_dx,
                               int64_t n_steps, int bc, T theta) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int t = threadIdx.x, Tn = blockDim.x, mask = Tn - 1;
    T *sR = reinterpret_cast<T *>(smem_raw);  // [2][Tn] reduced rows (A, C, D): PCR ping-pong
    T *sF = sR + 6 * Tn;                      // [Tn] first interface rows (A, C, D)
    T *sE = sF + 3 * Tn;                      // [6][Tn] partition edge values of u^n, u^{n+1} and M mu
    Part part;
    part.r0 = t * P; part.n = P;
    if (RAGGED) part = partition_of(t, N, Tn);
    const int n = part.n;
    __builtin_assume(n >= P - 1 && n <= P);
    const int64_t b = blockIdx.x, BN = B * (int64_t)N, off = b * N + part.r0;

    const double dtb = (double)dt[b];
    const T h = (T)(0.5 * dtb * inv_dx);
    const T r = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    const T th = theta * h, tr = theta * r, omt = T(1) - theta;
    const T b0 = T(1) + T(2) * tr;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const bool fixL = dirichlet && t == 0, fixR = dirichlet && t == Tn - 1;
    auto state = [&](int64_t k) { return (k == 0) ? u0 : states + (size_t)(k - 1) * (size_t)BN; };
    auto load = [&](const T *src, T (&dst)[P]) {
#pragma unroll
        for (int j = 0; j < P; ++j) dst[j] = (j < n) ? src[off + j] : T(0);
    };
    auto last_of = [&](const T (&a)[P]) {          // value of slot n - 1 without a run-time register index
        T x = a[0];
#pragma unroll
        for (int j = 1; j < P; ++j)
            if (j < n) x = a[j];
        return x;
    };
    auto frozen_at = [&](int j) { return (j == 0 && fixL) || (j >= n - 1 && fixR); };
    const bool frozL = dirichlet && t == 0;        // the row left of this partition (wrap: row N-1) is an end node
    const bool frozR = dirichlet && t == Tn - 1;   // the row right of it (wrap: row 0)

    T l[P], u[P], up[P];
    load(lam, l);
    load(state(n_steps), up);
    load(state(n_steps - 1), u);
    for (int64_t k = n_steps - 1; k >= 0; --k) {
        // the state of the NEXT backward step is fetched now and consumed at the end of this one: its DRAM latency
        // (the states are read once, in reverse order, nothing is in cache) hides behind the solve
        T nx[P];
        if (k > 0) load(state(k - 1), nx);
        sE[t] = u[0]; sE[Tn + t] = last_of(u); sE[2 * Tn + t] = up[0]; sE[3 * Tn + t] = last_of(up);
        __syncthreads();
        const int tl = (t - 1) & mask, tr_ = (t + 1) & mask;
        const T uL = sE[Tn + tl], uR = sE[tr_], upL = sE[3 * Tn + tl], upR = sE[2 * Tn + tr_];
        // ---- J(u^{n+1})^T mu = lam
        T f[P], c[P];
        Row<T> first, last;
        auto rowT = [&](int j, T &a, T &bb, T &e) {        // row j of J^T: (sup_{j-1}, diag_j, sub_{j+1})
            const bool lastrow = (j >= n - 1);
            const T wm = j ? up[j - 1] : upL, wp = lastrow ? upR : up[(j + 1 < P) ? j + 1 : j];
            const bool fm = j ? frozen_at(j - 1) : frozL, fp = lastrow ? frozR : frozen_at(j + 1);
            a = fm ? T(0) : t_fma(th, wm, -tr);             // sup_{j-1} = theta (h w_{j-1} - r)
            e = fp ? T(0) : t_fma(-th, wp, -tr);            // sub_{j+1} = theta (-h w_{j+1} - r)
            bb = frozen_at(j) ? T(1) : t_fma(th, wp - wm, b0);
        };
        if (RAGGED) eliminate_general_ragged<T, P>(rowT, n, l, f, c, first, last);
        else eliminate_general<T, P>(rowT, l, f, c, first, last);
        T x0, xL;
        solve_interface<T>(first, last, sR, sF, x0, xL, t, Tn);
        // (mu overwrites lam in place: slot j of the right-hand side is read before slot j of the solution is written)
        T (&mu)[P] = l;
        if (RAGGED) back_substitute_ragged<T, P>(mu, n, f, c, l, x0, xL);
        else back_substitute<T, P>(mu, f, c, l, x0, xL);
        // ---- lam^n = mu - (1 - theta) G'(u^n)^T (M mu)
        T m[P];
#pragma unroll
        for (int j = 0; j < P; ++j) m[j] = (frozen_at(j) || j >= n) ? T(0) : mu[j];
        sE[4 * Tn + t] = m[0]; sE[5 * Tn + t] = last_of(m);
        __syncthreads();
        const T mL = sE[5 * Tn + tl], mR = sE[4 * Tn + tr_];
#pragma unroll
        for (int j = 0; j < P; ++j) {
            if (j < n) {
                const bool lastrow = (j >= n - 1);
                const T vm = j ? u[j - 1] : uL, vp = lastrow ? uR : u[(j + 1 < P) ? j + 1 : j];
                const T mm = j ? m[j - 1] : mL, mp = lastrow ? mR : m[(j + 1 < P) ? j + 1 : j];
                T g = t_fma(h, vm, -r) * mm;
                g = t_fma(t_fma(h, vp - vm, T(2) * r), m[j], g);
                g = t_fma(t_fma(-h, vp, -r), mp, g);
                l[j] = t_fma(-omt, g, mu[j]);
            } else {
                l[j] = T(0);                               // (the unused slot of a ragged partition stays zero)
            }
        }
#pragma unroll
        for (int j = 0; j < P; ++j) { up[j] = u[j]; u[j] = nx[j]; }
        __syncthreads();                                   // sE is rewritten by the next step
    }
#pragma unroll
    for (int j = 0; j < P; ++j)
        if (j < n) lam[off + j] = l[j];
}

// ---- STAGED variant of the resident kernel for exact partitions (N == P * threads, at least one warp): as
// adjoint_btcs_staged_kernel (adjoint_btcs.cu) -- the stored states go through a ring of three shared-memory stages
// (cp.async, warp-private, swizzled) instead of through registers; lam, u^{k+1} (the Jacobian's state) and the two
// coefficient arrays are what the registers hold, u^k is read back from its stage for the G'(u^k)^T product.
__device__ __forceinline__ unsigned adjn_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

template <typename T, int P, bool SMALL>
__global__ void __launch_bounds__(SMALL ? 128 : adjn_max_threads(sizeof(T), P), SMALL ? 3 : 1)
adjoint_newton_staged_kernel(const T *__restrict__ u0, const T *__restrict__ states, T *__restrict__ lam,
                             const T *__restrict__ nu, const T *__restrict__ dt, int64_t B, int N, double inv_dx,
                             int64_t n_steps, int bc, T theta) {
    constexpr int V = 16 / sizeof(T);
    constexpr int CR = P / V;
    constexpr int SW = (CR >= 8) ? 1 : 8 / CR;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int t = threadIdx.x, Tn = blockDim.x, mask = Tn - 1, lane = t & 31, warp0 = t - lane;
    T *sR = reinterpret_cast<T *>(smem_raw);  // [2][Tn] reduced rows (A, C, D): PCR ping-pong
    T *sF = sR + 6 * Tn;                      // [Tn] first interface rows (A, C, D)
    T *sE = sF + 3 * Tn;                      // [2][Tn] partition edge values of M mu
    int4 *sS = reinterpret_cast<int4 *>(sE + 2 * Tn + (Tn & 1));   // [3][Tn * CR] chunks: ring of stages (Tn is even)
    const int64_t b = blockIdx.x, BN = B * (int64_t)N;
    const int64_t off = b * N + (int64_t)t * P, woff = b * N + (int64_t)warp0 * P;

    const double dtb = (double)dt[b];
    const T h = (T)(0.5 * dtb * inv_dx);
    const T r = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    const T th = theta * h, tr = theta * r, omt = T(1) - theta;
    const T b0 = T(1) + T(2) * tr;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    const bool fixL = dirichlet && t == 0, fixR = dirichlet && t == Tn - 1;
    auto state = [&](int64_t k) { return (k == 0) ? u0 : states + (size_t)(k - 1) * (size_t)BN; };
    auto chunk_of = [&](int rr, int c) { return rr * CR + (c ^ ((rr / SW) % CR)); };
    auto fetch = [&](int64_t k) {              // this warp's rows of u^k -> stage k % 3
        const int4 *src = reinterpret_cast<const int4 *>(state(k) + woff);
        int4 *dst = sS + (int)(k % 3) * Tn * CR;
#pragma unroll
        for (int i = 0; i < CR; ++i) {
            const int g = i * 32 + lane, rr = warp0 + g / CR, c = g % CR;
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(adjn_smem_u32(dst + chunk_of(rr, c))), "l"(src + g)
                         : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    auto own_row = [&](int64_t k, T (&dst)[P]) {
        const int4 *st = sS + (int)(k % 3) * Tn * CR;
#pragma unroll
        for (int c = 0; c < CR; ++c) {
            const int4 q4 = st[chunk_of(t, c)];
            const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
            for (int i = 0; i < V; ++i) dst[c * V + i] = e[i];
        }
    };
    auto elem = [&](int64_t k, int rr, int j) {  // element j of row rr of u^k
        const T *st = reinterpret_cast<const T *>(sS + (int)(k % 3) * Tn * CR);
        return st[chunk_of(rr, j / V) * V + (j % V)];
    };
    const bool frozL = dirichlet && t == 0;        // the row left of this partition (wrap: row N-1) is an end node
    const bool frozR = dirichlet && t == Tn - 1;   // the row right of it (wrap: row 0)
    auto frozen_at = [&](int j) { return (j == 0 && fixL) || (j == P - 1 && fixR); };

    T l[P], w[P];
#pragma unroll
    for (int c = 0; c < CR; ++c) {
        const int4 q4 = *reinterpret_cast<const int4 *>(lam + off + c * V);
        const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
        for (int i = 0; i < V; ++i) l[c * V + i] = e[i];
    }
    fetch(n_steps);
    fetch(n_steps - 1);
    for (int64_t k = n_steps - 1; k >= 0; --k) {
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                       // u^k and u^{k+1} staged by every warp; the reads of step k + 1 are done
        if (k > 0) fetch(k - 1);               // into the stage that held u^{k+2}
        own_row(k + 1, w);                     // the Jacobian is taken at w = u^{k+1}
        const int tl = (t - 1) & mask, tr_ = (t + 1) & mask;
        const T wL = elem(k + 1, tl, P - 1), wR = elem(k + 1, tr_, 0);
        // ---- J(u^{k+1})^T mu = lam
        T f[P], c[P];
        Row<T> first, last;
        auto rowT = [&](int j, T &a, T &bb, T &e) {        // row j of J^T: (sup_{j-1}, diag_j, sub_{j+1})
            const T wm = j ? w[j - 1] : wL, wp = (j == P - 1) ? wR : w[(j + 1 < P) ? j + 1 : j];
            const bool fm = j ? frozen_at(j - 1) : frozL, fp = (j == P - 1) ? frozR : frozen_at(j + 1);
            a = fm ? T(0) : t_fma(th, wm, -tr);
            e = fp ? T(0) : t_fma(-th, wp, -tr);
            bb = frozen_at(j) ? T(1) : t_fma(th, wp - wm, b0);
        };
        eliminate_general<T, P>(rowT, l, f, c, first, last);
        T x0, xL;
        solve_interface<T>(first, last, sR, sF, x0, xL, t, Tn);
        T (&mu)[P] = l;                                     // in place
        back_substitute<T, P>(mu, f, c, l, x0, xL);
        // ---- lam^k = mu - (1 - theta) G'(u^k)^T (M mu), u^k from its stage
        const T m0 = frozen_at(0) ? T(0) : mu[0], mP = frozen_at(P - 1) ? T(0) : mu[P - 1];
        sE[t] = m0; sE[Tn + t] = mP;
        __syncthreads();
        const T mL = sE[Tn + tl], mR = sE[tr_];
        T u[P];
        own_row(k, u);
        const T uL = elem(k, tl, P - 1), uR = elem(k, tr_, 0);
        T mprev = mL;
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const T vm = j ? u[j - 1] : uL, vp = (j == P - 1) ? uR : u[(j + 1 < P) ? j + 1 : j];
            const T mj = frozen_at(j) ? T(0) : mu[j];
            const T mp = (j == P - 1) ? mR : (frozen_at(j + 1) ? T(0) : mu[(j + 1 < P) ? j + 1 : j]);
            T g = t_fma(h, vm, -r) * mprev;
            g = t_fma(t_fma(h, vp - vm, T(2) * r), mj, g);
            g = t_fma(t_fma(-h, vp, -r), mp, g);
            l[j] = t_fma(-omt, g, mu[j]);                   // (mu[j] is l[j]: read, then written; mu[j + 1] is still mu)
            mprev = mj;
        }
    }
#pragma unroll
    for (int c = 0; c < CR; ++c) {
        int4 q4;
        T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
        for (int i = 0; i < V; ++i) e[i] = l[c * V + i];
        *reinterpret_cast<int4 *>(lam + off + c * V) = q4;
    }
}

// ---- thread-per-system fallback on the caller's [B][N] layout.  ws: cp, dp, wp ([B][N] each).
template <typename T>
__global__ void __launch_bounds__(64)
adjoint_newton_thomas_kernel(const T *__restrict__ u0, const T *__restrict__ states, T *__restrict__ lam,
                             T *__restrict__ ws, const T *__restrict__ nu, const T *__restrict__ dt, int64_t B, int64_t N,
                             double inv_dx, int64_t n_steps, int bc, T theta) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const int64_t BN = B * N;
    const double dtb = (double)dt[b];
    const T h = (T)(0.5 * dtb * inv_dx);
    const T r = (T)((double)nu[b] * dtb * inv_dx * inv_dx);
    const T th = theta * h, tr = theta * r, omt = T(1) - theta;
    const T b0 = T(1) + T(2) * tr;
    const bool dirichlet = (bc == BURGERS_BC_DIRICHLET);
    T *cp = ws + b * N, *dp = ws + BN + b * N, *wp = ws + 2 * BN + b * N, *l = lam + b * N;
    auto frozen = [&](int64_t i) { return dirichlet && (i == 0 || i == N - 1); };
    auto rowT = [&](const T *w, int64_t j, T &a, T &bb, T &e) {      // row j of J(w)^T, cyclic neighbours
        const int64_t jm = (j == 0) ? N - 1 : j - 1, jp = (j == N - 1) ? 0 : j + 1;
        a = frozen(jm) ? T(0) : t_fma(th, w[jm], -tr);
        e = frozen(jp) ? T(0) : t_fma(-th, w[jp], -tr);
        bb = frozen(j) ? T(1) : t_fma(th, w[jp] - w[jm], b0);
    };
    for (int64_t k = n_steps - 1; k >= 0; --k) {
        const T *u = ((k == 0) ? u0 : states + (size_t)(k - 1) * (size_t)BN) + b * N;
        const T *up = states + (size_t)k * (size_t)BN + b * N;
        // cyclic Thomas by Sherman-Morrison (D6) on the transposed rows; for Dirichlet the corner entries are zero,
        // the correction term vanishes and the plain solve remains
        T a, bb, e;
        rowT(up, 0, a, bb, e);
        const T alpha = a;                       // corner (0, N-1)
        T aN, bN, eN;
        rowT(up, N - 1, aN, bN, eN);
        const T beta = eN;                       // corner (N-1, 0)
        const T gamma = -bb;
        T m = bb - gamma;
        cp[0] = e / m; dp[0] = l[0] / m; wp[0] = gamma / m;
        for (int64_t j = 1; j < N; ++j) {
            rowT(up, j, a, bb, e);
            if (j == N - 1) bb = bb - alpha * beta / gamma;
            m = bb - a * cp[j - 1];
            cp[j] = e / m;
            dp[j] = (l[j] - a * dp[j - 1]) / m;
            wp[j] = (((j == N - 1) ? beta : T(0)) - a * wp[j - 1]) / m;
        }
        for (int64_t j = N - 2; j >= 0; --j) {
            dp[j] = dp[j] - cp[j] * dp[j + 1];
            wp[j] = wp[j] - cp[j] * wp[j + 1];
        }
        const T fact = (dp[0] + alpha / gamma * dp[N - 1]) / (T(1) + wp[0] + alpha / gamma * wp[N - 1]);
        for (int64_t j = 0; j < N; ++j) dp[j] = dp[j] - fact * wp[j];            // mu
        auto masked = [&](int64_t i) { return frozen(i) ? T(0) : dp[i]; };
        for (int64_t j = 0; j < N; ++j) {
            const int64_t jm = (j == 0) ? N - 1 : j - 1, jp = (j == N - 1) ? 0 : j + 1;
            T g = t_fma(h, u[jm], -r) * masked(jm);
            g = t_fma(t_fma(h, u[jp] - u[jm], T(2) * r), masked(j), g);
            g = t_fma(t_fma(-h, u[jp], -r), masked(jp), g);
            l[j] = t_fma(-omt, g, dp[j]);
        }
    }
}

bool adjn_geometry(int is_f64, int64_t N, int *P_out, int *T_out, bool *ragged) {
    const int bytes = is_f64 ? 8 : 4;
    return pick_partition(N, [bytes](int P) { return adjn_max_threads(bytes, P); }, P_out, T_out, ragged);
}

template <typename T, int P>
int launch_resident_P(const T *u0, const T *states, T *lam, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                      int64_t n_steps, int bc, double theta, int Tn, bool ragged, cudaStream_t s) {
    const size_t smem = (size_t)15 * Tn * sizeof(T);
    if (ragged) {
        adjoint_newton_resident_kernel<T, P, true><<<(unsigned)B, Tn, smem, s>>>(u0, states, lam, nu, dt, B, (int)N,
                                                                               1.0 / dx, n_steps, bc, (T)theta);
        return last_launch_status();
    }
    if constexpr (P == 4 || P == 8 || P == 16) {
        if (Tn >= 32) {                                     // states through the shared-memory ring
            const size_t smem_s = (size_t)(11 + 3 * P) * Tn * sizeof(T) + 16;
            auto go = [&](auto kernel) {
                if (smem_s > 48 * 1024 &&
                    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_s) != cudaSuccess)
                    return (int)BURGERS_ERR_CUDA;
                kernel<<<(unsigned)B, Tn, smem_s, s>>>(u0, states, lam, nu, dt, B, (int)N, 1.0 / dx, n_steps, bc, (T)theta);
                return last_launch_status();
            };
            return Tn <= 128 ? go(adjoint_newton_staged_kernel<T, P, true>) : go(adjoint_newton_staged_kernel<T, P, false>);
        }
        adjoint_newton_resident_kernel<T, P, false><<<(unsigned)B, Tn, smem, s>>>(u0, states, lam, nu, dt, B, (int)N,
                                                                                1.0 / dx, n_steps, bc, (T)theta);
        return last_launch_status();
    }
    return BURGERS_ERR_PLAN;
}

}  // namespace

size_t adjoint_newton_ws_elems(int is_f64, int64_t B, int64_t N) {
    int P, Tn;
    bool ragged;
    return adjn_geometry(is_f64, N, &P, &Tn, &ragged) ? 0 : (size_t)3 * (size_t)B * (size_t)N;
}

template <typename T>
int launch_adjoint_newton_steps(const T *u0, const T *states, T *lam, T *ws, int64_t B, int64_t N, double dx,
                                const T *nu, const T *dt, int64_t n_steps, int bc, double theta, cudaStream_t s) {
    if (n_steps == 0) return BURGERS_OK;
    if (B > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    int P, Tn;
    bool ragged;
    if (adjn_geometry(sizeof(T) == 8, N, &P, &Tn, &ragged)) {
        switch (P) {
#define BURGERS_CASE(PP) \
    case PP: return launch_resident_P<T, PP>(u0, states, lam, B, N, dx, nu, dt, n_steps, bc, theta, Tn, ragged, s);
            BURGERS_CASE(4) BURGERS_CASE(5) BURGERS_CASE(6) BURGERS_CASE(7) BURGERS_CASE(8) BURGERS_CASE(9)
            BURGERS_CASE(10) BURGERS_CASE(11) BURGERS_CASE(12) BURGERS_CASE(13) BURGERS_CASE(14) BURGERS_CASE(15)
            BURGERS_CASE(16)
#undef BURGERS_CASE
        }
        return BURGERS_ERR_PLAN;
    }
    adjoint_newton_thomas_kernel<T><<<(unsigned)((B + 63) / 64), 64, 0, s>>>(u0, states, lam, ws, nu, dt, B, N, 1.0 / dx,
                                                                           n_steps, bc, (T)theta);
    return last_launch_status();
}

template int launch_adjoint_newton_steps<float>(const float *, const float *, float *, float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, double, cudaStream_t);
template int launch_adjoint_newton_steps<double>(const double *, const double *, double *, double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, double, cudaStream_t);

}  // namespace burgers
