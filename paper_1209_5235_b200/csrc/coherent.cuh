// coherent.cuh -- ray-coherent work order ("compacts and sorts live photons by volume and interaction type
// between stages to reduce SIMT divergence"; divergence is what the paper's GPU version loses to).
//
// Rays arrive in arbitrary order, so the 32 lanes of a warp stand in different volumes, look in different directions and
// take different branches of the distance and relocation code.  The remedy is the ray tracer's: order the work so that
// neighbours in the order are neighbours in phase space.  Key of one ray =
//     kind of its current volume (solid type x has daughters; 0 when there is none yet)
//   | cell of its position in a C^3 grid over the world's bounding box
//   | bin of its direction in a D^3 grid over [-1, 1]^3
// and the work order is the counting sort of the ray indices by that key:
//   1. whoever produces the rays computes the key, takes rank = atomicAdd(&hist[key], 1) and stores (key, rank);
//   2. three small kernels turn hist into exclusive prefix sums (tile sums, scan of the tile sums, scan inside the tiles);
//   3. coh_scatter_kernel writes perm[hist[key] + rank] = ray index.
// A kernel then runs through perm and writes its results to the rays' own slots, so the order changes the schedule only --
// which ray shares a warp with which -- never a result (ranks inside a bucket depend on the timing of the atomics).
// It pays where a ray costs much more than the gather of its record: the free-path walks (Algorithm 2 phase 5) and the
// transport passes; for plain locate / ComputeStep queries the gather of 28-byte queries through the order costs more than
// the coherence saves (measured), they keep the 9-key sort by volume kind.
#pragma once
#include <algorithm>
#include <cstdint>
#include <cuda_runtime.h>

namespace gn {

struct CohGrid {
    float lo[3], scale[3];      // cell_k = clamp((int)((x_k - lo_k) * scale_k), 0, C - 1)
    int C, D, nk;               // cells per axis, direction bins per axis, number of volume kinds
    __host__ __device__ uint32_t buckets() const { return (uint32_t)nk * (uint32_t)(C * C * C) * (uint32_t)(D * D * D); }
};
// c, h: centre and half extents of the world's bounding box
inline CohGrid coh_grid(const float c[3], const float h[3], int C, int D, int nk) {
    CohGrid g;
    g.C = C; g.D = D; g.nk = nk;
    for (int k = 0; k < 3; ++k) { const float hk = h[k] > 0 ? h[k] : 1.0f; g.lo[k] = c[k] - hk; g.scale[k] = (float)C / (2.0f * hk); }
    return g;
}
__device__ __forceinline__ uint32_t coh_key(const CohGrid& g, float x, float y, float z, float wx, float wy, float wz, int kind) {
    const int top = g.C - 1, dt = g.D - 1;
    const int cx = min(max((int)((x - g.lo[0]) * g.scale[0]), 0), top);
    const int cy = min(max((int)((y - g.lo[1]) * g.scale[1]), 0), top);
    const int cz = min(max((int)((z - g.lo[2]) * g.scale[2]), 0), top);
    const float hd = 0.5f * (float)g.D;
    const int dx = min(max((int)((wx + 1.0f) * hd), 0), dt), dy = min(max((int)((wy + 1.0f) * hd), 0), dt), dz = min(max((int)((wz + 1.0f) * hd), 0), dt);
    const uint32_t cell = (uint32_t)(cx + g.C * (cy + g.C * cz)), dir = (uint32_t)(dx + g.D * (dy + g.D * dz));
    return ((uint32_t)kind * (uint32_t)(g.C * g.C * g.C) + cell) * (uint32_t)(g.D * g.D * g.D) + dir;
}

constexpr int COH_THREADS = 256;
constexpr int COH_TILE = 2048;            // histogram entries per block of the scan kernels

// exclusive prefix of v over the block (COH_THREADS threads); total = sum over the block
__device__ __forceinline__ unsigned coh_block_exclusive(unsigned v, unsigned* sh_warp, unsigned& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) sh_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const unsigned w = lane < COH_THREADS / 32 ? sh_warp[lane] : 0u;
        unsigned wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += t; }
        if (lane < COH_THREADS / 32) sh_warp[lane] = wi - w;
        if (lane == 31) sh_warp[COH_THREADS / 32] = wi;
    }
    __syncthreads();
    total = sh_warp[COH_THREADS / 32];
    const unsigned r = sh_warp[warp] + inc - v;
    __syncthreads();
    return r;
}
static __global__ void __launch_bounds__(COH_THREADS) coh_tile_sums_kernel(const unsigned* __restrict__ hist, unsigned nb, unsigned* __restrict__ tile_sums) {
    __shared__ unsigned sh[COH_THREADS / 32 + 1];
    const unsigned base = blockIdx.x * COH_TILE;
    unsigned s = 0;
#pragma unroll
    for (int q = 0; q < COH_TILE / COH_THREADS; ++q) { const unsigned i = base + q * COH_THREADS + threadIdx.x; s += i < nb ? hist[i] : 0u; }
    unsigned total;
    coh_block_exclusive(s, sh, total);
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}
static __global__ void __launch_bounds__(COH_THREADS) coh_scan_tiles_kernel(unsigned* __restrict__ tile_sums, unsigned n_tiles) {      // one block
    __shared__ unsigned sh[COH_THREADS / 32 + 1];
    const unsigned per = (n_tiles + COH_THREADS - 1) / COH_THREADS;
    const unsigned lo = min(threadIdx.x * per, n_tiles), hi = min(lo + per, n_tiles);
    unsigned s = 0;
    for (unsigned i = lo; i < hi; ++i) s += tile_sums[i];
    unsigned total;
    unsigned run = coh_block_exclusive(s, sh, total);
    for (unsigned i = lo; i < hi; ++i) { const unsigned v = tile_sums[i]; tile_sums[i] = run; run += v; }
}
// in place: hist[key] becomes the first position of bucket `key` in the order
static __global__ void __launch_bounds__(COH_THREADS) coh_scan_kernel(unsigned* __restrict__ hist, unsigned nb, const unsigned* __restrict__ tile_sums) {
    __shared__ unsigned sh[COH_THREADS / 32 + 1];
    constexpr int PER = COH_TILE / COH_THREADS;
    const unsigned base = blockIdx.x * COH_TILE + threadIdx.x * PER;      // each thread owns PER consecutive entries
    unsigned v[PER], s = 0;
#pragma unroll
    for (int q = 0; q < PER; ++q) { v[q] = base + q < nb ? hist[base + q] : 0u; s += v[q]; }
    unsigned total;
    unsigned run = coh_block_exclusive(s, sh, total) + tile_sums[blockIdx.x];
#pragma unroll
    for (int q = 0; q < PER; ++q) { if (base + q < nb) hist[base + q] = run; run += v[q]; }
}
// kr[i] = (key, rank) of ray i; a key of 0xffffffff marks a slot that holds no ray
static __global__ void __launch_bounds__(COH_THREADS) coh_scatter_kernel(const uint2* __restrict__ kr, int64_t n, const unsigned* __restrict__ n_ptr,
                                                                         const unsigned* __restrict__ hist, uint32_t* __restrict__ perm) {
    if (n_ptr) n = (int64_t)*n_ptr;                                        // count known only on the device (transport passes)
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const uint2 e = kr[i];
        if (e.x != 0xffffffffu) perm[__ldg(&hist[e.x]) + e.y] = (uint32_t)i;
    }
}
inline size_t coh_tiles(unsigned nb) { return ((size_t)nb + COH_TILE - 1) / COH_TILE; }
// hist (counts) -> bucket starts -> perm; everything on stream s.  tile_sums: coh_tiles(nb) words.
inline void coh_build_order(unsigned* hist, unsigned nb, unsigned* tile_sums, const uint2* kr, int64_t n_upper, const unsigned* n_ptr, uint32_t* perm, cudaStream_t s) {
    const unsigned n_tiles = (unsigned)coh_tiles(nb);
    coh_tile_sums_kernel<<<n_tiles, COH_THREADS, 0, s>>>(hist, nb, tile_sums);
    coh_scan_tiles_kernel<<<1, COH_THREADS, 0, s>>>(tile_sums, n_tiles);
    coh_scan_kernel<<<n_tiles, COH_THREADS, 0, s>>>(hist, nb, tile_sums);
    const int64_t blocks = std::max<int64_t>(1, std::min<int64_t>((n_upper + COH_THREADS - 1) / COH_THREADS, 148 * 16));
    coh_scatter_kernel<<<(unsigned)blocks, COH_THREADS, 0, s>>>(kr, n_upper, n_ptr, hist, perm);
}

}  // namespace gn
