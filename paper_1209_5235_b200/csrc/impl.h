// impl.h -- declarations of the per-precision launchers.  Each is a template defined in nav_kernels.cuh / transport.cuh and
// explicitly instantiated in ONE translation unit (nav_f32.cu, nav_f64.cu, transport_f{32,64}_{box,gen}.cu), so that the
// kernels compile in parallel; api.cu (the extern "C" entry points) sees only these declarations.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "geometry.h"

namespace gn {

template <class R> struct SourceDev;

template <class R> int locate_impl(const gn_geometry* geo, const void* pos, const void* dir, int64_t n, int32_t* out, cudaStream_t s);
template <class R> int step_impl(const gn_geometry* geo, const void* pos, const void* dir, const int32_t* vol, const void* max_step,
                                 int64_t n, void* step, int32_t* next, cudaStream_t s);
template <class R> int step_normal_impl(const gn_geometry* geo, const void* pos, const void* dir, const int32_t* vol, const void* max_step,
                                        int64_t n, void* step, int32_t* next, void* normal, cudaStream_t s);
template <class R> int safety_impl(const gn_geometry* geo, const void* pos, const int32_t* vol, int64_t n, void* out, cudaStream_t s);
template <class R> int free_path_impl(const gn_geometry* geo, const void* pos, const void* dir, const void* Y, int64_t n, double mu_mass,
                                      void* T, uint32_t* nsteps, cudaStream_t s);
// FLAT = true: any solid, rotations, several candidates per voxel cell; FLAT = false: unrotated boxes only (gn_geometry::coherent)
template <class R, bool FLAT> int transport_impl(const gn_geometry* geo, const SourceDev<R>& src, uint64_t seed, int64_t first_id, int64_t n_photons,
                                                 double* d_edep, gn_run_stats* h_stats, uint64_t* d_hash, uint32_t* d_nsteps, double* d_efinal,
                                                 cudaStream_t s);

}  // namespace gn
