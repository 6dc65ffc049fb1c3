// explicit_f64.cu -- fp64 instantiation of the explicit kernels (see explicit_impl.cuh).
#include "explicit_impl.cuh"

namespace burgers {
template <>
int launch_explicit<double>(double *u, int64_t B, int64_t N, double dx, const double *nu,
                            const double *dt, int64_t n_steps, int bc, int scheme,
                            const ExplicitGeom &g, double *ws, double *snaps,
                            int64_t snap_every, cudaStream_t s,
                           const ExplicitAdapt<double> *adapt, const ExplicitTiledAdapt<double> *tadapt) {
    return expl::launch_explicit_impl<double>(u, B, N, dx, nu, dt, n_steps, bc, scheme, g, ws, snaps, snap_every, s, adapt, tadapt);
}
}  // namespace burgers
