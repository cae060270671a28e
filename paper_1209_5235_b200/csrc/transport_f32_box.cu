// transport_f32_box.cu -- float transport kernels for geometries of unrotated boxes (gn_geometry::coherent)
#include "transport.cuh"
namespace gn {
template int transport_impl<float, false>(const gn_geometry*, const SourceDev<float>&, uint64_t, int64_t, int64_t, double*, gn_run_stats*, uint64_t*, uint32_t*, double*, cudaStream_t);
}
