// transport_f64_box.cu -- double transport kernels for geometries of unrotated boxes (gn_geometry::coherent)
#include "transport.cuh"
namespace gn {
template int transport_impl<double, false>(const gn_geometry*, const SourceDev<double>&, uint64_t, int64_t, int64_t, double*, gn_run_stats*, uint64_t*, uint32_t*, double*, cudaStream_t);
}
