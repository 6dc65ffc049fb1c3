// btcs_hybrid.cu -- placeholder until the resident partition+PCR solver lands.
#include "common.cuh"
namespace burgers {
bool btcs_hybrid_fits(int, int64_t, int) { return false; }
template <typename T>
int launch_btcs_hybrid(T *, int64_t, int64_t, double, const T *, const T *, int64_t, int, cudaStream_t) {
    return BURGERS_ERR_PLAN;
}
template int launch_btcs_hybrid<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, cudaStream_t);
template int launch_btcs_hybrid<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, cudaStream_t);
}  // namespace burgers
