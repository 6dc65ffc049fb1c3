// cfl.cu -- kernel (5): per-trajectory max|u| reduction and the CFL time step
//   dt_b = C * min(dx / max_i |u_b,i|, dx^2 / (2 nu_b))     (PAPER.md:116-118 Eq.7-8, :287 Eq.24)
// One pass over u: B*N*sizeof(T) bytes read.  Thread-level max over 128-bit loads, warp
// shuffle max, one smem hop per warp, then either the CTA owns the whole trajectory and
// writes dt directly, or (long trajectories split over several CTAs) an atomicMax on the
// bit pattern of the non-negative maximum in dt_out[b] followed by a finalize kernel.
#include "common.cuh"

namespace burgers {
namespace {

constexpr int kCflThreads = 256;
constexpr int kCflItems = 32;  // elements per thread per CTA chunk

template <typename T> struct Bits;
template <> struct Bits<float> {
    using U = unsigned int;
    static __device__ __forceinline__ U to(float x) { return __float_as_uint(x); }
    static __device__ __forceinline__ float from(U b) { return __uint_as_float(b); }
};
template <> struct Bits<double> {
    using U = unsigned long long;
    static __device__ __forceinline__ U to(double x) { return (U)__double_as_longlong(x); }
    static __device__ __forceinline__ double from(U b) { return __longlong_as_double((long long)b); }
};

template <typename T> __device__ __forceinline__ T absmax(T m, T x) { return fmax(m, fabs(x)); }
template <> __device__ __forceinline__ float absmax<float>(float m, float x) { return fmaxf(m, fabsf(x)); }

template <typename T>
__global__ void __launch_bounds__(kCflThreads)
cfl_reduce_kernel(const T *__restrict__ u, const T *__restrict__ nu, T *__restrict__ dt_out,
                  int64_t N, int chunks, double dx, double C) {
    constexpr int V = 16 / sizeof(T);
    using U = typename Bits<T>::U;
    const int64_t b = blockIdx.x / chunks;
    const int chunk = blockIdx.x % chunks;
    const int64_t span = (int64_t)blockDim.x * kCflItems;
    const int64_t lo = (int64_t)chunk * span;
    const int64_t hi = (lo + span < N) ? lo + span : N;
    const T *row = u + b * N;
    T m = T(0);
    if ((N % V) == 0) {  // every row start is 16-byte aligned: 128-bit loads
        const int4 *row4 = reinterpret_cast<const int4 *>(row);
        for (int64_t i = lo / V + threadIdx.x; i < hi / V; i += blockDim.x) {
            int4 q = __ldg(row4 + i);
            const T *e = reinterpret_cast<const T *>(&q);
#pragma unroll
            for (int k = 0; k < V; ++k) m = absmax(m, e[k]);
        }
    } else {
        for (int64_t i = lo + threadIdx.x; i < hi; i += blockDim.x) m = absmax(m, __ldg(row + i));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        T other = __shfl_xor_sync(0xffffffffu, m, o);
        m = (other > m) ? other : m;
    }
    __shared__ T wmax[kCflThreads / kWarp];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wmax[w] = m;
    __syncthreads();
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        m = (lane < nw) ? wmax[lane] : T(0);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            T other = __shfl_xor_sync(0xffffffffu, m, o);
            m = (other > m) ? other : m;
        }
        if (lane == 0) {
            if (chunks == 1) dt_out[b] = cfl_dt<T>(m, nu[b], dx, C);
            else atomicMax(reinterpret_cast<U *>(dt_out) + b, Bits<T>::to(m));
        }
    }
}

// Short rows (at most kWarpRowVecs 16-byte vectors): ONE WARP PER TRAJECTORY, several trajectories
// per CTA, no shared memory and no CTA barrier; every lane keeps up to 8 independent 128-bit loads
// in flight.  (One CTA per 4 KB row, as the chunked kernel would do for config 5, is latency-bound:
// measured 2.5 TB/s.)
constexpr int kWarpRowVecs = 1024;   // rows up to 16 KB
constexpr int kWarpRowWarps = 8;

template <typename T>
__global__ void __launch_bounds__(kWarpRowWarps * 32)
cfl_warp_row_kernel(const T *__restrict__ u, const T *__restrict__ nu, T *__restrict__ dt_out,
                    int64_t B, int64_t N, double dx, double C) {
    constexpr int V = 16 / sizeof(T);
    const int lane = threadIdx.x & 31;
    const int64_t b = (int64_t)blockIdx.x * kWarpRowWarps + (threadIdx.x >> 5);
    if (b >= B) return;
    const int4 *row4 = reinterpret_cast<const int4 *>(u + b * N);   // N % V == 0: 16-byte aligned rows
    const int nv = (int)(N / V);
    T m = T(0);
    int i = lane;
    for (; i + 7 * 32 < nv; i += 8 * 32) {
        int4 q[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) q[k] = __ldg(row4 + i + k * 32);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const T *e = reinterpret_cast<const T *>(&q[k]);
#pragma unroll
            for (int j = 0; j < V; ++j) m = absmax(m, e[j]);
        }
    }
    for (; i < nv; i += 32) {
        int4 q = __ldg(row4 + i);
        const T *e = reinterpret_cast<const T *>(&q);
#pragma unroll
        for (int j = 0; j < V; ++j) m = absmax(m, e[j]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        T other = __shfl_xor_sync(0xffffffffu, m, o);
        m = (other > m) ? other : m;
    }
    if (lane == 0) dt_out[b] = cfl_dt<T>(m, nu[b], dx, C);
}

template <typename T>
__global__ void cfl_finalize_kernel(const T *__restrict__ nu, T *__restrict__ dt_out, int64_t B,
                                    double dx, double C) {
    using U = typename Bits<T>::U;
    int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    T m = Bits<T>::from(reinterpret_cast<const U *>(dt_out)[b]);
    dt_out[b] = cfl_dt<T>(m, nu[b], dx, C);
}

inline int cfl_threads(int64_t N, int V) {
    int64_t want = (N + V - 1) / V;  // one vector per thread is enough for short rows
    int t = kCflThreads;
    while (t > 32 && t / 2 >= want) t /= 2;
    return t;
}

}  // namespace

template <typename T>
int launch_cfl(const T *u, int64_t B, int64_t N, double dx, const T *nu, double C, T *dt_out,
               cudaStream_t s) {
    const int V = 16 / (int)sizeof(T);
    if (N % V == 0 && N / V <= kWarpRowVecs && B >= 4 * 148) {    // many short rows: warp per trajectory
        const int64_t grid = (B + kWarpRowWarps - 1) / kWarpRowWarps;
        if (grid > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
        cfl_warp_row_kernel<T><<<(unsigned)grid, kWarpRowWarps * 32, 0, s>>>(u, nu, dt_out, B, N, dx, C);
        return last_launch_status();
    }
    const int threads = cfl_threads(N, V);
    const int64_t span = (int64_t)threads * kCflItems;
    const int64_t chunks = (N + span - 1) / span;
    if (B * chunks > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    if (chunks > 1) {
        if (cudaMemsetAsync(dt_out, 0, (size_t)B * sizeof(T), s) != cudaSuccess) return BURGERS_ERR_CUDA;
    }
    cfl_reduce_kernel<T><<<(unsigned)(B * chunks), threads, 0, s>>>(u, nu, dt_out, N, (int)chunks, dx, C);
    int st = last_launch_status();
    if (st != BURGERS_OK) return st;
    if (chunks > 1) {
        cfl_finalize_kernel<T><<<(unsigned)((B + 255) / 256), 256, 0, s>>>(nu, dt_out, B, dx, C);
        st = last_launch_status();
    }
    return st;
}

int64_t cfl_launch_count(int is_f64, int64_t B, int64_t N) {
    const int V = is_f64 ? 2 : 4;
    if (N % V == 0 && N / V <= kWarpRowVecs && B >= 4 * 148) return 1;
    const int64_t span = (int64_t)cfl_threads(N, V) * kCflItems;
    return ((N + span - 1) / span > 1) ? 2 : 1;
}

template int launch_cfl<float>(const float *, int64_t, int64_t, double, const float *, double, float *, cudaStream_t);
template int launch_cfl<double>(const double *, int64_t, int64_t, double, const double *, double, double *, cudaStream_t);

}  // namespace burgers
