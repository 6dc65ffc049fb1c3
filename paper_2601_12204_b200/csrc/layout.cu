// layout.cu -- the one re-layout the thread-per-system plans need: [B][N] (trajectory-contiguous, as the
// caller owns it) <-> [N][B] (batch index fastest), so that at every sweep position the 32 threads of a
// warp touch 32 consecutive elements (north_star kernel (3)).  32 x 33 shared tile.
#include "common.cuh"

namespace burgers {
namespace {

template <typename T>
__global__ void transpose_kernel(const T *__restrict__ in, T *__restrict__ out, int64_t rows, int64_t cols) {
    // in[rows][cols] -> out[cols][rows]
    __shared__ T tile[32][33];
    const int64_t gx = (cols + 31) / 32;
    const int64_t c0 = ((int64_t)blockIdx.x % gx) * 32, r0 = ((int64_t)blockIdx.x / gx) * 32;
    for (int k = threadIdx.y; k < 32; k += blockDim.y) {
        int64_t r = r0 + k, c = c0 + threadIdx.x;
        if (r < rows && c < cols) tile[k][threadIdx.x] = in[r * cols + c];
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += blockDim.y) {
        int64_t c = c0 + k, r = r0 + threadIdx.x;
        if (r < rows && c < cols) out[c * rows + r] = tile[threadIdx.x][k];
    }
}

}  // namespace

template <typename T>
int launch_transpose(const T *in, T *out, int64_t rows, int64_t cols, cudaStream_t s) {
    const int64_t nblk = ((cols + 31) / 32) * ((rows + 31) / 32);
    if (nblk > 0x7fffffffLL) return BURGERS_ERR_SHAPE;
    transpose_kernel<T><<<(unsigned)nblk, dim3(32, 8), 0, s>>>(in, out, rows, cols);
    return last_launch_status();
}

template int launch_transpose<float>(const float *, float *, int64_t, int64_t, cudaStream_t);
template int launch_transpose<double>(const double *, double *, int64_t, int64_t, cudaStream_t);

}  // namespace burgers
