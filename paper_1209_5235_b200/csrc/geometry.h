// geometry.h -- the opaque gn_geometry handle (host side) shared by geometry.cu and kernels.cu
#pragma once
#include <mutex>
#include <string>
#include <vector>
#include "store.h"
#include "../../include/gammanav.h"

#define GN_TIMED_PASSES 64      // lean step passes of a batch that are timed one by one

struct gn_geometry {
    gn::GeoView<float> v32{};
    gn::GeoView<double> v64{};
    std::vector<void*> allocations;      // every cudaMalloc owned by the handle
    int32_t n_places = 0, n_solids = 0, n_mats = 0;
    double tol32 = 0, tol64 = 0;
    gn_opts opts{};
    int64_t n_grids = 0, n_cells = 0, n_cand = 0, device_bytes = 0;
    int device = 0;
    float world_c[3] = {0, 0, 0}, world_h[3] = {1, 1, 1};      // bounding box of the world solid (centre, half extents): cells of the ray-coherent work order (coherent.cuh)
    bool voxel_sched = false;            // coherent and mostly regular voxels: lean passes are voxel_pass + slow_pass (voxel_pass.cuh)
    bool has_slabs = false;              // some leaf boxes are regular slabs (NODE_SLAB): the regular-voxel step kernel is built with the slab rule
    bool coherent = false;               // boxes only, no rotations, at most one candidate per voxel cell: lanes of a warp do the same thing per node visit
    // transport workspace (photon queues, counters, pinned read-back, events): grown on demand, reused by every
    // gn_transport_run on this handle, released by gn_geometry_destroy; runs on one handle are serialised
    mutable std::mutex ws_mutex;
    mutable std::mutex host_mutex;            // held across a whole gn_transport_run_host call (its staging buffer is shared)
    mutable char* ws_scratch = nullptr;
    mutable size_t ws_bytes = 0;
    mutable void* ws_pinned = nullptr;
    mutable double* ws_host_edep = nullptr;   // device staging of the tally for gn_transport_run_host (n_places doubles)
    mutable cudaEvent_t ws_events[8 + 2 * GN_TIMED_PASSES] = {};
    mutable bool ws_events_ok = false;
    // host-buffer entry points: two streams and a two-slot device staging area, so that the copies of one chunk overlap
    // the kernels of the other
    mutable cudaStream_t hp_stream[2] = {};
    mutable bool hp_streams_ok = false;
    mutable char* hp_buf = nullptr;
    mutable size_t hp_bytes = 0;
    cudaMemPool_t pool = nullptr;             // stream-ordered scratch (query sort) of this handle
};

namespace gn {
void set_error(const std::string& msg);
int fail(int code, const std::string& msg);
}
