// transport_f64_gen.cu -- double transport kernels for general geometries (any solid, rotations)
#include "transport.cuh"
namespace gn {
template int transport_impl<double, true>(const gn_geometry*, const SourceDev<double>&, uint64_t, int64_t, int64_t, double*, gn_run_stats*, uint64_t*, uint32_t*, double*, cudaStream_t);
}
