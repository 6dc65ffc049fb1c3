// noalloc.cu -- burgers_btcs_noalloc: BTCS time stepping for callers that cannot allocate (code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The BTCS plans that need scratch memory (LONG: ping-pong state, interface rows of the cooperative fallback,
// status words; THOMAS: the batch-minor copies) normally take it from the caller (`ws`, burgers_workspace_bytes).
// Here the scratch is a file-scope device array of kScratchBytes: every GPU that loads the library holds it from
// module load until the process exits, and nothing is allocated or freed by any call.  What runs is the stock
// path (burgers_btcs_f32 / _f64, plan AUTO) with `ws` pointing at that array -- same kernels, same bits.
//
// In HOST code the array's name is a host-side stand-in for the symbol, not a device address: a kernel handed
// `g_noalloc_scratch` directly would fault (or, where the GPU can reach host memory, scribble over the wrong
// memory).  The device address is looked up once per device with cudaGetSymbolAddress, with that device current,
// and cached (scratch_address below); that pointer is what goes to the kernels.
//
// Sharing: ALL calls on a device use the same array, and it keeps the last call's contents.  Nothing in it has
// to start at zero except the LONG plan's status words, which launch_btcs_long clears on the call's stream at
// the start of every call (cudaMemsetAsync, not an allocation); every other region is written before it is
// read.  Calls that overlap on the GPU (two streams, two host threads, two captured graphs replayed
// concurrently) RACE on the array: serialise them (one stream, or events between them).
#include <cmath>
#include <mutex>

#include "common.cuh"

namespace burgers {
namespace {

constexpr size_t kScratchBytes = (size_t)32 << 20;      // 32 MiB: one fp64 periodic grid of up to 2^20 points
                                                        // (LONG: 8 MiB state + 12 MiB rows), or its equivalent
static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mutex;
void *g_scratch_on[kMaxDevices];                        // device address of the array on device d (0: not looked up)

// Set-up, once per device: the address of g_noalloc_scratch on the CURRENT device.
int scratch_address(void **out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return BURGERS_ERR_CUDA; }
    if (dev < 0 || dev >= kMaxDevices) return BURGERS_ERR_CUDA;
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch_on[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return BURGERS_ERR_CUDA;
        }
        g_scratch_on[dev] = p;
    }
    *out = g_scratch_on[dev];
    return BURGERS_OK;
}

}  // namespace
}  // namespace burgers

extern "C" {

size_t burgers_noalloc_scratch_bytes(void) { return burgers::kScratchBytes; }

int burgers_noalloc_init(void) {
    void *p = nullptr;
    return burgers::scratch_address(&p);
}

int burgers_btcs_noalloc(int dtype_is_f64, void *u, int64_t B, int64_t N, double L, const void *nu, const void *dt,
                         int64_t n_steps, int bc, void *stream) {
    // the argument rules of burgers_btcs_* (include/burgers.h "Errors"), in its order, before anything touches
    // the device
    if (!u || !nu || !dt) return BURGERS_ERR_NULL;
    if (B < 1 || N < 3 || n_steps < 0) return BURGERS_ERR_SHAPE;
    if (bc != BURGERS_BC_PERIODIC && bc != BURGERS_BC_DIRICHLET) return BURGERS_ERR_ENUM;
    if (!(L > 0.0) || !std::isfinite(L)) return BURGERS_ERR_VALUE;
    const size_t need = burgers_workspace_bytes(BURGERS_OP_BTCS, dtype_is_f64 ? 1 : 0, B, N, bc, 0, BURGERS_PLAN_AUTO);
    if (need > burgers::kScratchBytes) return BURGERS_ERR_LIMIT;
    void *ws = nullptr;
    if (need) {
        const int st = burgers::scratch_address(&ws);
        if (st != BURGERS_OK) return st;
    }
    if (dtype_is_f64)
        return burgers_btcs_f64(static_cast<double *>(u), B, N, L, static_cast<const double *>(nu),
                                static_cast<const double *>(dt), n_steps, bc, ws, need, stream);
    return burgers_btcs_f32(static_cast<float *>(u), B, N, L, static_cast<const float *>(nu),
                            static_cast<const float *>(dt), n_steps, bc, ws, need, stream);
}

}  // extern "C"
