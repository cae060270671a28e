// transport_f32_gen.cu -- float transport kernels for general geometries (any solid, rotations)
#include "transport.cuh"
namespace gn {
template int transport_impl<float, true>(const gn_geometry*, const SourceDev<float>&, uint64_t, int64_t, int64_t, double*, gn_run_stats*, uint64_t*, uint32_t*, double*, cudaStream_t);
}
