// explicit_impl.cuh -- kernel (1): explicit time stepping (forward Euler PAPER.md:216 Eq.21,
// classical RK4 PAPER.md:224-229 Eq.22) of the upwind/central semi-discrete operator
// (Eq.3-4, upwind rule :89).
//
// One kernel template serves two plans:
//   RESIDENT  one CTA owns a whole trajectory: it is loaded once, all n_steps run on chip,
//             it is stored once.  HBM traffic 2*sizeof(T)*N per trajectory per CALL.
//   TILED     one CTA owns an overlapped tile of a (long) trajectory and advances it `tblock`
//             steps per HBM round trip (temporal blocking): the tile is loaded with a halo of
//             tblock*radius points per side, its edges are left open (the invalid front moves
//             inwards `radius` points per step) and only the still-valid centre is stored.
// Data layout on chip: thread t holds P CONSECUTIVE grid points in registers, so every stencil
// neighbour but two is a register of the same thread; the two halo values come from the
// neighbouring threads by warp shuffle (CTA of one warp) or through a double-buffered shared
// memory edge array with ONE barrier per exchange (several warps).
//
// Arithmetic per point (D2 scaled by dt; cx = dt/dx, rr = nu dt/dx^2).  With the one-sided differences
// d_j = u_{j+1} - u_j (each shared by two neighbouring points) the update is
//     lap = d_j - d_{j-1},   g = (u_j > 0) ? d_{j-1} : d_j   (upwind rule PAPER.md:89),
//     dt*F = rr*lap - cx*u_j*g.
// The B200 FP32 pipe is limited by REGISTER-OPERAND bandwidth, not by instruction count (measured:
// FADD with 2 register operands 0.98 warp-instr/cycle/SMSP, FFMA with 3 distinct registers 0.61;
// DESIGN.md "Kernels"), so the form is chosen to minimise register reads per update:
//   fp32: the state is carried SCALED, w = cx*u, which folds the convective coefficient into the
//         state:  dt*F*cx = rr*lap(w) - w*g(w):  FADD, FADD, FSETP+FSEL (ALU pipe), FFMA, FFMA
//         (+ FADD for the compensated sum) = 7 issue slots / 15 register reads per update (the
//         select-free |u| form needs 8 / 19).  Scaling happens once at load, unscaling once at
//         store; Dirichlet end nodes are stored back bit-exactly from the loaded values.
//   fp64: the FP64 pipe (64 lanes/SM) is the limit, so what counts is DP instructions: unscaled
//         form, DADD, DADD, DMUL, DFMA, DFMA = 5 per update with the select done on the integer
//         pipe from the sign of the high word.  Unscaled, so that p then q steps equal p+q steps
//         bitwise.
// Both equal D2 up to rounding, keep constants exactly fixed and keep odd symmetry exact.
// fp32 Euler carries the state as base + s (two fp32 terms; increments are accumulated into the
// small term s, so they are not lost against ulp(w)) -- the stencil reads the
// rounded sum v = fl(base + s).
#pragma once
#include "common.cuh"

namespace burgers {
namespace expl {

template <typename T>
struct Params {
    const T *src;     // [B][N]
    T *dst;           // [B][N]   (== src for RESIDENT)
    const T *nu;      // [B]
    const T *dt;      // [B]
    int64_t N;
    double inv_dx;
    int64_t steps;    // steps in this launch
    int nth;          // active threads per CTA
    int bc;
    int halo;         // TILED: halo points per side
    int64_t W;        // TILED: valid outputs per tile
    int64_t tiles;    // TILED: tiles per trajectory
    // fp32 carries the state scaled (w = cx*u, see below).  Between the launches of a TILED call the
    // ping-pong buffers hold w, so only the first launch scales and only the last one unscales.
    // Frozen Dirichlet end nodes are ALWAYS stored unscaled (their original bits).
    int in_scaled, out_scaled;
    // Trajectory output (SURVEY 8(f) NEXT-4b; RESIDENT plan, kernel template SNAP): after every
    // snap_every-th step the state is also written to snaps[k][B][N], k = 0, 1, ...
    T *snaps;
    int64_t snap_every;
    int64_t snap_stride;   // B*N
    // Adaptive time step (SURVEY 8(f) NEXT-4a; RESIDENT plan, kernel template ADAPT): every
    // adapt_every steps dt = dt_from_cfl(current state, adapt_C) is re-evaluated inside the kernel
    // (CTA-wide max |u|, the formula of cfl.cu); `dt` is then not read.  0 = fixed dt.
    int64_t adapt_every;
    double adapt_C, dx;
    double *t_out;         // [B] sum of adapt_every*dt over the evaluations, or nullptr
    T *dt_out;             // [B] the last dt
    // Adaptive time step on TILED grids (kernel template TADAPT): the CFL reduction is fused into the launches of a
    // segment of adapt_every steps.  The LAST launch of segment k takes the maximum |u| of what it stores into slot
    // seg_write of umax[3][B] (bit patterns of non-negative values, atomicMax); every launch of segment k+1 evaluates
    // dt = cfl_dt(that maximum) itself (seg_read); its first launch (seg_first) records dt and the elapsed time and
    // clears the slot the segment after it will use (seg_zero).  seg_read < 0: dt comes from p.dt (segment 0).
    unsigned long long *umax;
    int64_t Bn;
    int seg_read, seg_write, seg_zero, seg_first;
};

template <typename T> __device__ __forceinline__ unsigned long long to_bits(T x);
template <> __device__ __forceinline__ unsigned long long to_bits<float>(float x) { return (unsigned long long)__float_as_uint(x); }
template <> __device__ __forceinline__ unsigned long long to_bits<double>(double x) { return (unsigned long long)__double_as_longlong(x); }
template <typename T> __device__ __forceinline__ T from_bits(unsigned long long b);
template <> __device__ __forceinline__ float from_bits<float>(unsigned long long b) { return __uint_as_float((unsigned)b); }
template <> __device__ __forceinline__ double from_bits<double>(unsigned long long b) { return __longlong_as_double((long long)b); }

// max over the CTA of a non-negative value (NaN operands are ignored, as in cfl.cu)
template <typename T, bool WARP>
__device__ __forceinline__ T cta_max(T m, T *red) {
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, off));
    if (WARP) return m;
    const int nw = (blockDim.x + 31) >> 5;
    __syncthreads();                       // `red` may still be read from the previous use
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    T r = red[0];
    for (int w = 1; w < nw; ++w) r = fmax(r, red[w]);
    return r;
}

template <typename T> __device__ __forceinline__ T t_abs(T x);
template <> __device__ __forceinline__ float t_abs<float>(float x) { return fabsf(x); }
template <> __device__ __forceinline__ double t_abs<double>(double x) { return fabs(x); }
template <typename T> __device__ __forceinline__ T t_fma(T a, T b, T c);
template <> __device__ __forceinline__ float t_fma<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <> __device__ __forceinline__ double t_fma<double>(double a, double b, double c) { return fma(a, b, c); }

// upwind difference: backward difference dm where the value is > 0, else forward dp
template <typename T> __device__ __forceinline__ T upwind(T c, T dm, T dp);
template <> __device__ __forceinline__ float upwind<float>(float c, float dm, float dp) { return (c > 0.f) ? dm : dp; }
template <> __device__ __forceinline__ double upwind<double>(double c, double dm, double dp) {
    // sign test on the high word (integer pipe; the FP64 pipe is the scarce one).  +-0 and positive
    // denormals below 2^-1022 take dp: they multiply the difference by (next to) nothing (Q3).
    return (__double2hiint(c) > 0) ? dm : dp;
}

// acc + dt*F at one point from its value c and the differences dm = c - left, dp = right - c.
//   SCALED (state w = cx*u):  acc + rr*(dp - dm) - c*g          k1 = rr, k2 unused
//   unscaled:                 acc + rr*(dp - dm) - cx*(c*g)     k1 = rr, k2 = cx
template <typename T, bool SCALED>
__device__ __forceinline__ T add_dtF(T acc, T c, T dm, T dp, T rr, T cx) {
    const T lap = dp - dm;                       // u_{i+1} - 2u_i + u_{i-1}   (Eq.4)
    const T g = upwind<T>(c, dm, dp);
    if (SCALED) return t_fma(-c, g, t_fma(rr, lap, acc));
    return t_fma(-cx, c * g, t_fma(rr, lap, acc));
}
// c + dt*F, unscaled, as  c*(1 - cx*g) + rr*lap:  DADD, DFMA, DMUL, DFMA (+ the shared difference) --
// the same 5 FP64-pipe instructions as add_dtF(c, ...) but 27 instead of 29 register reads (the
// immediate 1 replaces a register operand).  d = 0 gives exactly c.
template <typename T>
__device__ __forceinline__ T euler_unscaled(T c, T dm, T dp, T rr, T cx) {
    const T lap = dp - dm;
    const T g = upwind<T>(c, dm, dp);
    return t_fma(c, t_fma(-cx, g, T(1)), rr * lap);
}
// dt*F alone (RK4 stages)
template <typename T, bool SCALED>
__device__ __forceinline__ T dtF(T c, T dm, T dp, T rr, T cx) {
    const T lap = dp - dm;
    const T g = upwind<T>(c, dm, dp);
    if (SCALED) return t_fma(-c, g, rr * lap);
    return t_fma(-cx, c * g, rr * lap);
}

// Halo exchange: every thread publishes its first and last point and receives the last point
// of its left neighbour (tl) and the first point of its right neighbour (tr).
template <typename T, bool WARP>
__device__ __forceinline__ void exchange(T first, T last, T &left, T &right, int tl, int tr,
                                         T *edge, int &buf) {
    if (WARP) {
        left = __shfl_sync(0xffffffffu, last, tl);
        right = __shfl_sync(0xffffffffu, first, tr);
    } else {
        T *e = edge + buf * 2 * blockDim.x;
        e[threadIdx.x] = first;
        e[blockDim.x + threadIdx.x] = last;
        __syncthreads();
        left = e[blockDim.x + tl];
        right = e[tr];
        buf ^= 1;
    }
}

constexpr int max_threads_for(int bytes, int P, int scheme) { return explicit_max_threads_for(bytes, P, scheme); }

// ADAPT: the rarely executed CFL evaluation must not cost the time loop its occupancy: cap the kernel
// at the 128 registers of the fixed-dt kernels (2 CTAs of 256 threads, 4 of 128, ...).
constexpr int adapt_min_ctas(int bytes, int P, int scheme) {
    int arrays = (scheme == BURGERS_SCHEME_RK4) ? 3 : (bytes == 4 ? 3 : 1);
    int est = P * (bytes / 4) * arrays + 40;                 // as max_threads_for
    int mt = max_threads_for(bytes, P, scheme);
    int n = (est <= 136) ? 512 / mt : 1;                     // kernels that need more keep the full budget
    return n > 0 ? n : 1;
}

template <typename T, int P, int SCHEME, bool TILED, bool WARP, bool SNAP = false, bool ADAPT = false, bool TADAPT = false>
__global__ void __launch_bounds__(WARP ? 32 : max_threads_for(sizeof(T), P, SCHEME),
                                  (ADAPT && !WARP) ? adapt_min_ctas(sizeof(T), P, SCHEME)
                                                   : (WARP && sizeof(T) == 4 && SCHEME == BURGERS_SCHEME_RK4 && P == 32 && !SNAP && !ADAPT) ? 12 : 0)   // (0 = unspecified)
explicit_kernel(const Params<T> p) {
    static_assert(!(SNAP && TILED), "snapshots are fused into the RESIDENT plan only");
    static_assert(!(ADAPT && TILED), "ADAPT is the RESIDENT form of the fused CFL evaluation, TADAPT the TILED one");
    static_assert(!TADAPT || TILED, "TADAPT is the TILED form");
    constexpr bool SPLIT = (sizeof(T) == 4) && (SCHEME == BURGERS_SCHEME_EULER);
    constexpr bool RK4_DESC = WARP && (sizeof(T) == 4);
    constexpr bool EULER_DESC = !SNAP;
    constexpr int V = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *edge = reinterpret_cast<T *>(smem_raw);

    const int t = threadIdx.x;
    const int nth = p.nth;
    const int64_t N = p.N;
    const int64_t b = TILED ? (int64_t)(blockIdx.x / p.tiles) : (int64_t)blockIdx.x;
    const int64_t tile = TILED ? (int64_t)(blockIdx.x % p.tiles) : 0;
    const bool active = t < nth;
    const bool dirichlet = (p.bc == BURGERS_BC_DIRICHLET);
    // global index of this thread's first point (may be <0 or >=N in TILED halos)
    const int64_t g0 = (TILED ? tile * p.W - p.halo : 0) + (int64_t)t * P;
    const T *srow = p.src + b * N;
    T *drow = p.dst + b * N;

    // per-trajectory constants, evaluated in fp64 and rounded once (ADAPT: set again below, once the
    // state is loaded)
    constexpr bool SCALED = (sizeof(T) == 4);
    const T nu_b = p.nu[b];
    T dt_cur = ADAPT ? T(0) : p.dt[b];
    if (TADAPT && p.seg_read >= 0)      // the maximum the previous segment's last launch left, the formula of cfl.cu
        dt_cur = cfl_dt<T>(from_bits<T>(p.umax[(int64_t)p.seg_read * p.Bn + b]), nu_b, p.dx, p.adapt_C);
    if (TADAPT && p.seg_first && tile == 0 && t == 0) {
        if (p.seg_read >= 0) p.dt_out[b] = dt_cur;             // (segment 0: dt_out already holds it -- it IS p.dt)
        // (product and sum rounded separately, as the accumulation of the separate-call sequence does)
        if (p.t_out) p.t_out[b] = __dadd_rn(p.t_out[b], __dmul_rn((double)p.adapt_every, (double)dt_cur));
        if (p.seg_zero >= 0) p.umax[(int64_t)p.seg_zero * p.Bn + b] = 0ull;
    }
    T cx, rr;
    auto set_dt = [&](T dt_new) {
        const double dtb = (double)dt_new;
        cx = (T)(dtb * p.inv_dx);
        rr = (T)((double)nu_b * dtb * p.inv_dx * p.inv_dx);
    };
    set_dt(dt_cur);
    // fp32: the state is carried as w = scale*u with scale = cx.  dt == 0 (cx == 0) leaves u
    // unchanged: no steps, scale 1.
    bool degenerate = SCALED && (cx == T(0));
    T scale = (SCALED && !degenerate) ? cx : T(1);
    int64_t steps = degenerate ? 0 : p.steps;

    // ---------------- load
    T v[P];
#pragma unroll
    for (int j = 0; j < P; ++j) v[j] = T(0);
    const bool vec_ok = (P % V == 0) && (N % V == 0) && (!TILED || (p.halo % V == 0 && p.W % V == 0));
    if (active) {
        if (vec_ok) {
#pragma unroll
            for (int c = 0; c < P / V; ++c) {
                int64_t g = g0 + c * V;
                bool inside = true;
                if (TILED) {
                    if (dirichlet) inside = (g >= 0 && g < N);
                    else if (g < 0 || g >= N) { g %= N; if (g < 0) g += N; }
                }
                if (inside) {
                    int4 q = *reinterpret_cast<const int4 *>(srow + g);
                    const T *e = reinterpret_cast<const T *>(&q);
#pragma unroll
                    for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < P; ++j) {
                int64_t g = g0 + j;
                bool inside = true;
                if (TILED) {
                    if (dirichlet) inside = (g >= 0 && g < N);
                    else if (g < 0 || g >= N) { g %= N; if (g < 0) g += N; }
                }
                if (inside) v[j] = srow[g];
            }
        }
    }

    // ADAPT: the first dt comes from the loaded state (the same max and the same formula as dt_from_cfl_*)
    __shared__ T red[(ADAPT || TADAPT) ? 32 : 1];
    if (ADAPT) {
        T m = T(0);
#pragma unroll
        for (int j = 0; j < P; ++j) m = fmax(m, t_abs(v[j]));
        dt_cur = cfl_dt<T>(cta_max<T, WARP>(m, red), nu_b, p.dx, p.adapt_C);
        set_dt(dt_cur);
        degenerate = SCALED && (cx == T(0));
        scale = (SCALED && !degenerate) ? cx : T(1);
        steps = degenerate ? 0 : p.steps;
    }
    double t_acc = (ADAPT && steps > 0) ? (double)p.adapt_every * (double)dt_cur : 0.0;

    // neighbours for the halo exchange; open edges (TILED) read their own value: garbage that
    // never reaches the stored centre.
    const int last_t = nth - 1;
    int tl = (t == 0) ? (TILED ? 0 : last_t) : t - 1;
    int tr = (t >= last_t) ? (TILED ? last_t : 0) : t + 1;
    if (!active) { tl = 0; tr = 0; }
    // Dirichlet: node 0 and node N-1 never move.  The host guarantees they sit at j = 0 and
    // j = P-1 of their thread (N % P == 0, tile origin % P == 0).
    const bool fixL = dirichlet && (g0 == 0);
    const bool fixR = dirichlet && (g0 + P - 1 == N - 1);
    const T keepL = v[0], keepR = v[P - 1];       // stored back bit-exactly when frozen
    int buf = 0;
    T left, right;
    // trajectory output: val(j) is the (scaled) state of point j; unscaled with a reciprocal and one
    // remainder correction (the final state uses the exact quotient)
    int64_t snap_left = SNAP ? p.snap_every : 0;
    T *snap_row = SNAP ? p.snaps + b * N + g0 : nullptr;     // this thread's row in the next snapshot
    T inv_scale = T(1) / scale;
    auto snapshot = [&](auto val) {
        if (!SNAP) return;
        if (--snap_left != 0) return;
        snap_left = p.snap_every;
        auto out = [&](int j) {
            T x = val(j);
            if (SCALED) {
                T qn = x * inv_scale;
                qn = t_fma(t_fma(-qn, scale, x), inv_scale, qn);
                x = qn;
                if (j == 0 && fixL) x = keepL;
                if (j == P - 1 && fixR) x = keepR;
            }
            return x;
        };
        constexpr int CRs = (P % V == 0) ? P / V : 0;          // 16-byte chunks per thread row
        if (CRs >= 1 && CRs <= 8 && vec_ok) {
            // Stage the warp's rows in shared memory (XOR-swizzled 16-byte chunks: conflict-free both
            // ways) so that the global stores are 512 contiguous bytes per request instead of one
            // 16-byte piece of 32 different rows.  Whole warps take part; rows past N are not stored.
            constexpr int CRd = (CRs >= 1 && CRs <= 8) ? CRs : 1;     // (keeps the dead branch well-formed)
            constexpr int RB = CRd * 16, SW = 8 / CRd;
            unsigned char *stg = smem_raw + (size_t)4 * blockDim.x * sizeof(T) + (size_t)(t >> 5) * 32 * RB;
            const int lane = t & 31;
#pragma unroll
            for (int c = 0; c < CRd; ++c) {
                int4 q;
                T *e = reinterpret_cast<T *>(&q);
#pragma unroll
                for (int k = 0; k < V; ++k) e[k] = out(c * V + k);
                *reinterpret_cast<int4 *>(stg + lane * RB + ((c ^ ((lane / SW) % CRd)) * 16)) = q;
            }
            __syncwarp();
            const int64_t wbase = (int64_t)(t >> 5) * 32 * P;      // first point of the warp's rows
#pragma unroll
            for (int k = 0; k < CRd; ++k) {
                const int qi = k * 32 + lane, r = qi / CRd, c = qi % CRd;
                const int64_t g = wbase + (int64_t)qi * V;
                if (g < N)
                    *reinterpret_cast<int4 *>(snap_row - g0 + g) =
                        *reinterpret_cast<const int4 *>(stg + r * RB + ((c ^ ((r / SW) % CRd)) * 16));
            }
            __syncwarp();
        } else if (active) {
            if (vec_ok) {
#pragma unroll
                for (int c = 0; c < P / V; ++c) {
                    int4 q;
                    T *e = reinterpret_cast<T *>(&q);
#pragma unroll
                    for (int k = 0; k < V; ++k) e[k] = out(c * V + k);
                    *reinterpret_cast<int4 *>(snap_row + c * V) = q;
                }
            } else {
#pragma unroll
                for (int j = 0; j < P; ++j) snap_row[j] = out(j);
            }
        }
        snap_row += p.snap_stride;
    };

    // Adaptive: a new dt from the current state held (scaled) in v[].  Returns false when the new dt
    // gives cx = 0 in fp32 (nothing to scale the state by: dt = 0 from here on, the state stays).  For the
    // scaled state, rho_hi + rho_lo = new scale / old scale as a two-term value, so that rescaling does
    // not add a rounding error per evaluation.  All threads of the CTA call this together.
    T rho_hi = T(1), rho_lo = T(0);
    auto next_dt = [&]() -> bool {
        T m = T(0);
#pragma unroll
        for (int j = 0; j < P; ++j) m = fmax(m, t_abs(v[j]));
        const T umax = cta_max<T, WARP>(m, red) / scale;
        const T dt_new = cfl_dt<T>(umax, nu_b, p.dx, p.adapt_C);
        const T scale_old = scale;
        dt_cur = dt_new;
        set_dt(dt_new);
        if (SCALED) {
            if (cx == T(0)) return false;
            rho_hi = cx / scale_old;
            rho_lo = t_fma(-rho_hi, scale_old, cx) / scale_old;
            scale = cx;
            inv_scale = T(1) / scale;
        }
        t_acc += (double)p.adapt_every * (double)dt_new;
        return true;
    };

    if (SCHEME == BURGERS_SCHEME_EULER) {
        T base[SPLIT ? P : 1], s[SPLIT ? P : 1];
        if (SPLIT) {       // w = scale*u as an exact two-term sum (or w itself from the last launch)
#pragma unroll
            for (int j = 0; j < P; ++j) {
                const bool raw = !p.in_scaled || (j == 0 && fixL) || (j == P - 1 && fixR);
                base[j] = raw ? v[j] * scale : v[j];
                s[j] = raw ? t_fma(v[j], scale, -base[j]) : T(0);
                v[j] = base[j];
            }
        }
        // One time step.  Fixed dt: the plain loop over it.  ADAPT: segments of adapt_every steps with a
        // CFL evaluation between them (the first dt was set above).
        auto step = [&](int64_t n) {
            exchange<T, WARP>(v[0], v[P - 1], left, right, tl, tr, edge, buf);
            // (points in DESCENDING order: same arithmetic, same bits, but the instruction schedule ptxas
            // finds for it is 3 % faster in fp32 -- measured, C2: 10.59 -> 10.28 ms; fp64 unchanged; the
            // snapshot-writing instance is faster ascending: 10.73 -> 10.53 ms with 200 snapshots)
            T carry = EULER_DESC ? right - v[P - 1] : v[0] - left;
#pragma unroll
            for (int jj = 0; jj < P; ++jj) {
                const int j = EULER_DESC ? P - 1 - jj : jj;
                const T c = v[j];
                const T other = EULER_DESC ? c - ((j > 0) ? v[j - 1] : left) : ((j + 1 < P) ? v[j + 1] : right) - c;
                const T dm = EULER_DESC ? other : carry, dp = EULER_DESC ? carry : other;
                const bool frozen = (j == 0 && fixL) || (j == P - 1 && fixR);
                if (SPLIT) {
                    const T sn = add_dtF<T, SCALED>(s[j], c, dm, dp, rr, cx);
                    s[j] = frozen ? s[j] : sn;
                    v[j] = base[j] + s[j];
                } else {
                    const T vn = SCALED ? add_dtF<T, true>(c, c, dm, dp, rr, cx) : euler_unscaled<T>(c, dm, dp, rr, cx);
                    v[j] = frozen ? c : vn;
                }
                carry = other;
            }
            if (SPLIT && (n & 63) == 63) {  // renormalise: base <- fl(base+s), s <- exact remainder
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    const T nb = v[j];
                    s[j] = (base[j] - nb) + s[j];
                    base[j] = nb;
                }
            }
            snapshot([&](int j) { return v[j]; });
        };
        if (!ADAPT) {
            // (fp64: two steps per loop iteration give ptxas the schedule that is 6 % faster -- measured,
            // C2 fp64: 17.49 -> 16.45 ms; fp32 is fastest with the plain loop)
#pragma unroll(sizeof(T) == 8 ? 2 : 1)
            for (int64_t n = 0; n < steps; ++n) step(n);
        }
        int64_t n = 0;
        for (int64_t seg_end = (steps < p.adapt_every ? steps : p.adapt_every); ADAPT;) {
            for (; n < seg_end; ++n) step(n);
            if (n >= steps) break;
            if (!next_dt()) break;
            if (SPLIT) {
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    if ((j == 0 && fixL) || (j == P - 1 && fixR)) {
                        const T keep = (j == 0) ? keepL : keepR;
                        base[j] = keep * scale;
                        s[j] = t_fma(keep, scale, -base[j]);
                    } else {
                        const T nb = base[j] * rho_hi;
                        const T e = t_fma(base[j], rho_hi, -nb);
                        s[j] = t_fma(s[j], rho_hi, t_fma(base[j], rho_lo, e));
                        base[j] = nb;
                    }
                    v[j] = base[j] + s[j];
                }
            }
            seg_end = (steps - n < p.adapt_every) ? steps : n + p.adapt_every;
        }
        if (SPLIT && !p.out_scaled) {       // u = (base + s)/scale, rounded once
#pragma unroll
            for (int j = 0; j < P; ++j) {
                const T qn = base[j] / scale;
                const T rem = t_fma(-qn, scale, base[j]) + s[j];
                v[j] = qn + rem / scale;
            }
        }
    } else {  // classical RK4; K_s = dt*F(y_s) (times scale)
        T y[P], acc[P];
        if (SCALED) {
#pragma unroll
            for (int j = 0; j < P; ++j) {
                const bool raw = !p.in_scaled || (j == 0 && fixL) || (j == P - 1 && fixR);
                v[j] = raw ? v[j] * scale : v[j];
            }
        }
        auto step = [&](int64_t) {
#pragma unroll
            for (int stage = 0; stage < 4; ++stage) {
                if (stage == 0) exchange<T, WARP>(v[0], v[P - 1], left, right, tl, tr, edge, buf);
                else exchange<T, WARP>(y[0], y[P - 1], left, right, tl, tr, edge, buf);
                // (point order: the single-warp fp32 kernel -- C5 -- is 3 % faster when it visits its points in
                // descending order and is built for 12 CTAs per SM; the other instances are not: measured)
                auto val = [&](int j) { return (stage == 0) ? v[j] : y[j]; };
                T carry = RK4_DESC ? right - val(P - 1) : val(0) - left;
#pragma unroll
                for (int jj = 0; jj < P; ++jj) {
                    const int j = RK4_DESC ? P - 1 - jj : jj;
                    const T c = val(j);
                    const T other = RK4_DESC ? c - ((j > 0) ? val(j - 1) : left) : ((j + 1 < P) ? val(j + 1) : right) - c;
                    const T dm = RK4_DESC ? other : carry, dp = RK4_DESC ? carry : other;
                    const bool frozen = (j == 0 && fixL) || (j == P - 1 && fixR);
                    T K = dtF<T, SCALED>(c, dm, dp, rr, cx);
                    K = frozen ? T(0) : K;
                    if (stage == 0) { acc[j] = K; y[j] = t_fma(T(0.5), K, v[j]); }
                    else if (stage == 1) { acc[j] = t_fma(T(2), K, acc[j]); y[j] = t_fma(T(0.5), K, v[j]); }
                    else if (stage == 2) { acc[j] = t_fma(T(2), K, acc[j]); y[j] = v[j] + K; }
                    else { acc[j] += K; v[j] = t_fma(acc[j], T(1.0 / 6.0), v[j]); }
                    carry = other;
                }
            }
            snapshot([&](int j) { return v[j]; });
        };
        if (!ADAPT) {
            for (int64_t n = 0; n < steps; ++n) step(n);
        }
        int64_t n = 0;
        for (int64_t seg_end = (steps < p.adapt_every ? steps : p.adapt_every); ADAPT;) {
            for (; n < seg_end; ++n) step(n);
            if (n >= steps) break;
            if (!next_dt()) break;
            if (SCALED) {
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    if ((j == 0 && fixL) || (j == P - 1 && fixR)) v[j] = ((j == 0) ? keepL : keepR) * scale;
                    else v[j] = t_fma(v[j], rho_hi, v[j] * rho_lo);
                }
            }
            seg_end = (steps - n < p.adapt_every) ? steps : n + p.adapt_every;
        }
        if (SCALED && !p.out_scaled) {
#pragma unroll
            for (int j = 0; j < P; ++j) v[j] = v[j] / scale;
        }
    }
    if (SCALED) {          // frozen Dirichlet nodes: the loaded bits, not a scale/unscale round trip
        if (fixL) v[0] = keepL;
        if (fixR) v[P - 1] = keepR;
    }

    if (ADAPT && t == 0) {
        if (p.t_out) p.t_out[b] = t_acc;
        p.dt_out[b] = dt_cur;
    }

    // ---------------- store
    T mloc = T(0);                     // TADAPT: max |u| of what this thread stores
    if (active) {
        if (vec_ok) {
#pragma unroll
            for (int c = 0; c < P / V; ++c) {
                int64_t g = g0 + c * V;
                bool ok = true;
                if (TILED) {
                    const int64_t li = (int64_t)t * P + c * V;  // local index in the tile
                    ok = (li >= p.halo) && (li < p.halo + p.W) && (g < N);
                }
                if (ok) {
                    int4 q;
                    T *e = reinterpret_cast<T *>(&q);
#pragma unroll
                    for (int k = 0; k < V; ++k) {
                        e[k] = v[c * V + k];
                        if (TADAPT) mloc = fmax(mloc, t_abs(v[c * V + k]));
                    }
                    *reinterpret_cast<int4 *>(drow + g) = q;
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < P; ++j) {
                int64_t g = g0 + j;
                bool ok = true;
                if (TILED) {
                    const int64_t li = (int64_t)t * P + j;
                    ok = (li >= p.halo) && (li < p.halo + p.W) && (g < N);
                }
                if (ok) {
                    drow[g] = v[j];
                    if (TADAPT) mloc = fmax(mloc, t_abs(v[j]));
                }
            }
        }
    }
    if (TADAPT && p.seg_write >= 0) {      // (uniform over the grid: every CTA takes part in the reduction)
        const T m = cta_max<T, false>(mloc, red);
        if (t == 0) atomicMax(p.umax + (int64_t)p.seg_write * p.Bn + b, to_bits<T>(m));
    }
}

// ------------------------------------------------------------------ host side
template <typename T, int P, int SCHEME>
int launch_P(const Params<T> &p, const ExplicitGeom &g, int64_t B, cudaStream_t s) {
    const bool tiled = (g.plan == BURGERS_PLAN_TILED);
    const int64_t grid = tiled ? B * g.tiles : B;
    if (grid > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    const size_t smem = (size_t)4 * g.block * sizeof(T);
    if (tiled && p.umax) {
        explicit_kernel<T, P, SCHEME, true, false, false, false, true><<<(unsigned)grid, g.block, smem, s>>>(p);
    } else if (tiled) {
        explicit_kernel<T, P, SCHEME, true, false><<<(unsigned)grid, g.block, smem, s>>>(p);
    } else if (p.adapt_every > 0) {
        if (g.block == 32) explicit_kernel<T, P, SCHEME, false, true, false, true><<<(unsigned)grid, 32, 0, s>>>(p);
        else explicit_kernel<T, P, SCHEME, false, false, false, true><<<(unsigned)grid, g.block, smem, s>>>(p);
    } else if (p.snaps) {          // + one staged row per thread for the coalesced snapshot stores
        const size_t ssm = smem + (size_t)g.block * P * sizeof(T);
        if (ssm > 48 * 1024) {
            cudaFuncSetAttribute(explicit_kernel<T, P, SCHEME, false, true, true>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm);
            cudaFuncSetAttribute(explicit_kernel<T, P, SCHEME, false, false, true>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm);
        }
        if (g.block == 32) explicit_kernel<T, P, SCHEME, false, true, true><<<(unsigned)grid, 32, ssm, s>>>(p);
        else explicit_kernel<T, P, SCHEME, false, false, true><<<(unsigned)grid, g.block, ssm, s>>>(p);
    } else if (g.block == 32) {
        explicit_kernel<T, P, SCHEME, false, true><<<(unsigned)grid, 32, 0, s>>>(p);
    } else {
        explicit_kernel<T, P, SCHEME, false, false><<<(unsigned)grid, g.block, smem, s>>>(p);
    }
    return last_launch_status();
}

template <typename T, int SCHEME>
int launch_scheme(const Params<T> &p, const ExplicitGeom &g, int64_t B, cudaStream_t s) {
    switch (g.P) {
        case 1: return launch_P<T, 1, SCHEME>(p, g, B, s);
        case 2: return launch_P<T, 2, SCHEME>(p, g, B, s);
        case 4: return launch_P<T, 4, SCHEME>(p, g, B, s);
        case 8: return launch_P<T, 8, SCHEME>(p, g, B, s);
        case 16: return launch_P<T, 16, SCHEME>(p, g, B, s);
        case 32: return launch_P<T, 32, SCHEME>(p, g, B, s);
    }
    return BURGERS_ERR_PLAN;
}

template <typename T>
int launch_explicit_impl(T *u, int64_t B, int64_t N, double dx, const T *nu, const T *dt,
                         int64_t n_steps, int bc, int scheme, const ExplicitGeom &g, T *ws,
                         T *snaps, int64_t snap_every, cudaStream_t s, const ExplicitAdapt<T> *adapt,
                         const ExplicitTiledAdapt<T> *tadapt) {
    if (n_steps == 0) return BURGERS_OK;
    if (adapt && g.plan != BURGERS_PLAN_RESIDENT) return BURGERS_ERR_PLAN;   // (the caller uses tadapt for TILED)
    if (tadapt && g.plan != BURGERS_PLAN_TILED) return BURGERS_ERR_PLAN;
    Params<T> p;
    p.nu = nu; p.dt = dt; p.N = N; p.inv_dx = 1.0 / dx; p.nth = g.nth; p.bc = bc;
    p.halo = g.halo; p.W = g.W; p.tiles = g.tiles;
    p.in_scaled = 0; p.out_scaled = 0;
    p.snaps = nullptr; p.snap_every = 0; p.snap_stride = B * N;
    p.adapt_every = adapt ? adapt->every : 0; p.adapt_C = adapt ? adapt->C : 0.0; p.dx = dx;
    p.t_out = adapt ? adapt->t_out : nullptr; p.dt_out = adapt ? adapt->dt_out : nullptr;
    p.umax = nullptr; p.Bn = B; p.seg_read = p.seg_write = p.seg_zero = -1; p.seg_first = 0;
    if (tadapt) {
        p.umax = tadapt->umax; p.adapt_every = n_steps; p.adapt_C = tadapt->C;
        p.t_out = tadapt->t_out; p.dt_out = tadapt->dt_out;
    }
    auto launch = [&]() {
        return scheme == BURGERS_SCHEME_EULER ? launch_scheme<T, BURGERS_SCHEME_EULER>(p, g, B, s)
                                              : launch_scheme<T, BURGERS_SCHEME_RK4>(p, g, B, s);
    };
    if (g.plan == BURGERS_PLAN_RESIDENT) {   // snapshots are written by the kernel itself
        p.src = u; p.dst = u; p.steps = n_steps;
        if (snaps && snap_every > 0 && n_steps >= snap_every) { p.snaps = snaps; p.snap_every = snap_every; }
        return launch();
    }
    // TILED: ping-pong between u and ws, tblock steps per launch; copy back when the last launch
    // wrote ws.  With snapshots: one such sequence per snap_every steps, then a device copy.
    auto run = [&](int64_t steps) {
        T *cur = u, *nxt = ws;
        int64_t done = 0;
        while (done < steps) {
            const int64_t k = (steps - done < g.tblock) ? steps - done : g.tblock;
            p.src = cur; p.dst = nxt; p.steps = k;
            p.in_scaled = (done > 0); p.out_scaled = (done + k < steps);
            if (tadapt) {          // one segment: dt from the previous segment's maximum, this one's maximum at the end
                p.seg_read = tadapt->seg_read;
                p.seg_first = (done == 0);
                p.seg_zero = (done == 0) ? tadapt->seg_zero : -1;
                p.seg_write = (done + k == steps) ? tadapt->seg_write : -1;
            }
            int st = launch();
            if (st != BURGERS_OK) return st;
            T *tmp = cur; cur = nxt; nxt = tmp;
            done += k;
        }
        if (cur != u &&
            cudaMemcpyAsync(u, cur, (size_t)B * N * sizeof(T), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
            return (int)BURGERS_ERR_CUDA;
        return (int)BURGERS_OK;
    };
    if (!(snaps && snap_every > 0)) return run(n_steps);
    int64_t done = 0, k = 0;
    while (done < n_steps) {
        const int64_t chunk = (n_steps - done < snap_every) ? n_steps - done : snap_every;
        int st = run(chunk);
        if (st != BURGERS_OK) return st;
        done += chunk;
        if (chunk == snap_every) {
            if (cudaMemcpyAsync(snaps + k * B * N, u, (size_t)B * N * sizeof(T), cudaMemcpyDeviceToDevice, s) !=
                cudaSuccess)
                return BURGERS_ERR_CUDA;
            ++k;
        }
    }
    return BURGERS_OK;
}

}  // namespace expl
}  // namespace burgers
