// peak.cu -- micro-benchmarks of the FP pipes the "alu" rooflines of bench.py are quoted against
// ("lane counts and sustained clock to be measured on the box with an FMA-chain
// micro-benchmark").  No arithmetic of the method lives here.
//
// Every thread carries ACC independent dependency chains in registers and executes `iters` rounds
// of one instruction per chain; the grid fills every SM to full occupancy.  The caller times the
// launch with CUDA events; the lane-instructions executed are returned so that
// lane-instr/s = grid * block * ACC * UNROLL * iters / time.  Kinds:
//   FFMA_CHAIN   a = fma(a, x, y), x and y the same two registers for every chain: the constants sit in
//                the operand-reuse cache, one register-file read per instruction -- the pure issue rate
//   FFMA_3REG    a_k = fma(a_k, b_k, c_k) with b_k, c_k distinct registers per chain: three register
//                reads per instruction -- what register-operand bandwidth allows
//   FADD_2REG    a_k = a_k + b_k: two register reads per instruction
//   DFMA_CHAIN / DFMA_3REG / DADD_2REG: the same on the FP64 pipe
//   DFMA_SELECT_MIX  per round 5 independent DFMA chains and one "64-bit select" (FSETP + 2 FSEL), the instruction
//                mix of the fp64 upwind stencil per update: how much of the FP64 rate is left when ALU-pipe
//                instructions are issued in between (only the DFMAs are counted)
#include "common.cuh"

namespace burgers {
namespace {

constexpr int kAcc = 8, kUnroll = 8, kBlock = 256;

template <typename T, int KIND>
__global__ void __launch_bounds__(kBlock) pipe_peak_kernel(T *sink, long long iters, T x, T y) {
    T a[kAcc], b[kAcc], c[kAcc];
#pragma unroll
    for (int k = 0; k < kAcc; ++k) {
        a[k] = x + T(threadIdx.x + k);
        b[k] = x + T(k) * y;           // values near 1 and small: chains stay finite for any iters
        c[k] = y * T(k + 1);
    }
    for (long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < kUnroll; ++r) {
#pragma unroll
            for (int k = 0; k < kAcc; ++k) {
                if (KIND == 0) a[k] = fma(a[k], x, y);
                else if (KIND == 1) a[k] = fma(a[k], b[k], c[k]);
                else a[k] = a[k] + b[k];
            }
        }
    }
    T s = T(0);
#pragma unroll
    for (int k = 0; k < kAcc; ++k) s += a[k];
    if (s == T(-123.456)) *sink = s;       // never true for the finite chains above; keeps the loop alive
}

__global__ void __launch_bounds__(kBlock) pipe_mix_kernel(double *sink, long long iters, double x, double y, float fx) {
    double a[5];
    float f[4], g[3];
#pragma unroll
    for (int k = 0; k < 5; ++k) a[k] = x + double(threadIdx.x + k);
#pragma unroll
    for (int k = 0; k < 4; ++k) f[k] = fx + float(k);
#pragma unroll
    for (int k = 0; k < 3; ++k) g[k] = fx - float(threadIdx.x + k);
    for (long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < kUnroll; ++r) {
#pragma unroll
            for (int k = 0; k < 5; ++k) a[k] = fma(a[k], x, y);
            // one "64-bit select": a predicate from the sign test and the two 32-bit halves (FSETP + 2 FSEL)
            const bool p = f[0] > fx;
            const float lo = p ? f[1] : g[0], hi = p ? f[2] : g[1];
            f[0] = lo; f[1] = hi;
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 5; ++k) s += a[k];
    s += f[0] + f[1] + f[2];
    if (s == -123.456) *sink = s;
}

template <typename T>
int launch_kind(int kind, T *sink, long long iters, int grid, cudaStream_t s) {
    // x slightly below 1 and y tiny: |a| decays towards y/(1-x), no overflow, no denormals
    const T x = T(0.999), y = T(1e-3);
    switch (kind) {
        case 0: pipe_peak_kernel<T, 0><<<grid, kBlock, 0, s>>>(sink, iters, x, y); break;
        case 1: pipe_peak_kernel<T, 1><<<grid, kBlock, 0, s>>>(sink, iters, x, y); break;
        case 2: pipe_peak_kernel<T, 2><<<grid, kBlock, 0, s>>>(sink, iters, x, y); break;
        default: return BURGERS_ERR_ENUM;
    }
    return last_launch_status();
}

}  // namespace
}  // namespace burgers

extern "C" int burgers_pipe_peak(int kind, int64_t iters, void *sink, void *stream, double *lane_instr_out) {
    using namespace burgers;
    if (!sink) return BURGERS_ERR_NULL;
    if (iters < 1) return BURGERS_ERR_SHAPE;
    if (kind < 0 || kind >= BURGERS_PEAK_KINDS) return BURGERS_ERR_ENUM;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return BURGERS_ERR_CUDA;
    const int grid = sms * (2048 / kBlock);            // every SM at full occupancy, one wave
    cudaStream_t s = (cudaStream_t)stream;
    if (kind == BURGERS_PEAK_DFMA_SELECT_MIX) {
        if (lane_instr_out) *lane_instr_out = (double)grid * kBlock * 5 * kUnroll * (double)iters;
        pipe_mix_kernel<<<grid, kBlock, 0, s>>>((double *)sink, iters, 0.999, 1e-3, 1.0001f);
        return last_launch_status();
    }
    if (lane_instr_out) *lane_instr_out = (double)grid * kBlock * kAcc * kUnroll * (double)iters;
    return kind < 3 ? launch_kind<float>(kind, (float *)sink, iters, grid, s)
                    : launch_kind<double>(kind - 3, (double *)sink, iters, grid, s);
}
