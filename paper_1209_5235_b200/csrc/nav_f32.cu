// nav_f32.cu -- fp32 instantiations of the navigation launchers (nav_kernels.cuh)
#include "nav_kernels.cuh"
namespace gn {
template int locate_impl<float>(const gn_geometry*, const void*, const void*, int64_t, int32_t*, cudaStream_t);
template int step_impl<float>(const gn_geometry*, const void*, const void*, const int32_t*, const void*, int64_t, void*, int32_t*, cudaStream_t);
template int step_normal_impl<float>(const gn_geometry*, const void*, const void*, const int32_t*, const void*, int64_t, void*, int32_t*, void*, cudaStream_t);
template int safety_impl<float>(const gn_geometry*, const void*, const int32_t*, int64_t, void*, cudaStream_t);
template int free_path_impl<float>(const gn_geometry*, const void*, const void*, const void*, int64_t, double, void*, uint32_t*, cudaStream_t);
}
