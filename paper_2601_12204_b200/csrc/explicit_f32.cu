// explicit_f32.cu -- fp32 instantiation of the explicit kernels (see explicit_impl.cuh).
#include "explicit_impl.cuh"

namespace burgers {
template <>
int launch_explicit<float>(float *u, int64_t B, int64_t N, double dx, const float *nu, const float *dt,
                           int64_t n_steps, int bc, int scheme, const ExplicitGeom &g, float *ws,
                           float *snaps, int64_t snap_every, cudaStream_t s,
                           const ExplicitAdapt<float> *adapt, const ExplicitTiledAdapt<float> *tadapt) {
    return expl::launch_explicit_impl<float>(u, B, N, dx, nu, dt, n_steps, bc, scheme, g, ws, snaps, snap_every, s, adapt, tadapt);
}
}  // namespace burgers
