// btcs_long.cu -- placeholder until the multi-CTA partitioned solver lands.
#include "common.cuh"
namespace burgers {
bool btcs_long_fits(int64_t, int) { return false; }
size_t btcs_long_ws_elems(int64_t, int64_t, int) { return 0; }
int64_t btcs_long_launch_count(int64_t, int64_t, int64_t) { return 0; }
template <typename T>
int launch_btcs_long(T *, int64_t, int64_t, double, const T *, const T *, int64_t, int, T *, cudaStream_t) {
    return BURGERS_ERR_PLAN;
}
template int launch_btcs_long<float>(float *, int64_t, int64_t, double, const float *, const float *, int64_t, int, float *, cudaStream_t);
template int launch_btcs_long<double>(double *, int64_t, int64_t, double, const double *, const double *, int64_t, int, double *, cudaStream_t);
}  // namespace burgers
