// common.cuh -- what every kernel translation unit shares: launch constants, the per-block shared-memory copies of the
// small geometry tables, and the host-side helpers of the launchers.
#pragma once
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include "geometry.h"
#include "nav.cuh"

namespace gn {

constexpr int NAV_THREADS = 256;
#ifndef NAV_LOCATE_MIN_BLOCKS
#define NAV_LOCATE_MIN_BLOCKS 8
#endif
#ifndef NAV_STEP_MIN_BLOCKS
#define NAV_STEP_MIN_BLOCKS 8      // ComputeStep kernels are latency-bound at ~10 of 32 lanes: full occupancy (32 registers, spills) wins
#endif
#ifndef NAV_LOCATE_MIN_BLOCKS_F64
#define NAV_LOCATE_MIN_BLOCKS_F64 4
#endif
#ifndef NAV_STEP_MIN_BLOCKS_F64
#define NAV_STEP_MIN_BLOCKS_F64 4      // 64 registers: +14 % on config 5 fp64 over 3 blocks
#endif
constexpr int MAX_SMEM_SOLIDS = 32;
constexpr int MAX_SMEM_GRIDS = 8;
constexpr int MAX_SMEM_MATS = 32;

// per-block copies of the small tables + the pointer block the out-of-line navigation helpers read
template <class R> struct BlockTables {
    SolidRec<R> solids[MAX_SMEM_SOLIDS];
    GridRec<R> grids[MAX_SMEM_GRIDS];
    NavCtx<R> ctx;
};
template <class R> __device__ __forceinline__ void stage_tables(const GeoView<R>& g, BlockTables<R>& t) {
    const bool ss = g.n_solids <= MAX_SMEM_SOLIDS, sg = g.n_grids <= MAX_SMEM_GRIDS;
    if (ss) for (int i = threadIdx.x; i < g.n_solids; i += blockDim.x) t.solids[i] = g.solids[i];
    if (sg) for (int i = threadIdx.x; i < g.n_grids; i += blockDim.x) t.grids[i] = g.grids[i];
    if (threadIdx.x == 0) {
        t.ctx.node = g.node; t.ctx.rot = g.rot; t.ctx.dlist = g.dlist; t.ctx.cells = g.cells; t.ctx.cand = g.cand;
        t.ctx.solids = ss ? t.solids : g.solids; t.ctx.grids = sg ? t.grids : g.grids; t.ctx.delta = g.delta;
    }
}

// Sort of the navigation queries by volume key (SURVEY 8(a) A10 applied to A11): queries arrive in arbitrary order, so in
// a geometry with mixed solids the lanes of a warp would do different things (world: box exit + scan of the barrels;
// sector: tube exit; ...).  Two small kernels build a work order -- a counting sort of the query indices by key = (solid
// type of the current volume, has daughters) -- and step_kernel runs through it; outputs go back to the original slots.
// Which query lands where inside its key's segment depends on block scheduling; the results do not.
constexpr int SORT_KEYS = 9;              // 4 solid types x {leaf, mother} + "no volume"
constexpr int SORT_TILE = 1024;
template <class R>
__global__ void __launch_bounds__(NAV_THREADS) sort_keys_kernel(GeoView<R> g, const int32_t* __restrict__ vol_in, int64_t n,
                                                                uint8_t* __restrict__ keys, unsigned long long* __restrict__ totals) {
    __shared__ unsigned sh[SORT_KEYS];
    if (threadIdx.x < SORT_KEYS) sh[threadIdx.x] = 0;
    __syncthreads();
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int v = vol_in[i];
        int key = SORT_KEYS - 1;
        if (v >= 0 && v < g.n_nodes) {
            const int4 h = __ldg(reinterpret_cast<const int4*>(g.node + v));          // {parent, info, mat, ndau}
            key = 2 * __ldg(&g.solids[h.y & NODE_SOLID_MASK].type) + (h.w > 0 ? 1 : 0);
        }
        keys[i] = (uint8_t)key;
        atomicAdd(&sh[key], 1u);
    }
    __syncthreads();
    if (threadIdx.x < SORT_KEYS && sh[threadIdx.x]) atomicAdd(&totals[threadIdx.x], (unsigned long long)sh[threadIdx.x]);
}
constexpr int SORT_KEYS_MAX = 32;         // the scatter kernel takes the number of keys as an argument (<= this)
constexpr int SORT_KEYS2 = 2 * SORT_KEYS; // relocation order of ComputeStep queries: volume kind x (boundary is the volume's own / a daughter's)
static __global__ void __launch_bounds__(NAV_THREADS) sort_scatter_kernel(const uint8_t* __restrict__ keys, int64_t n, const unsigned long long* __restrict__ totals,
                                                                   unsigned long long* __restrict__ cursors, uint32_t* __restrict__ perm,
                                                                   const unsigned* __restrict__ n_ptr, int nkeys = SORT_KEYS) {
    __shared__ unsigned sh_cnt[SORT_KEYS_MAX];
    __shared__ unsigned long long sh_base[SORT_KEYS_MAX];
    if (n_ptr) n = (int64_t)*n_ptr;                                          // count known only on the device (transport passes)
    const int64_t n_tiles = (n + SORT_TILE - 1) / SORT_TILE;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        if (threadIdx.x < nkeys) sh_cnt[threadIdx.x] = 0;
        __syncthreads();
        int key[SORT_TILE / NAV_THREADS]; unsigned rank[SORT_TILE / NAV_THREADS];
#pragma unroll
        for (int q = 0; q < SORT_TILE / NAV_THREADS; ++q) {
            const int64_t i = tile * SORT_TILE + q * NAV_THREADS + threadIdx.x;
            key[q] = i < n ? keys[i] : -1;
            // rank inside the tile: one shared atomic per warp and distinct key (most of a warp shares one or two keys)
            const unsigned peers = __match_any_sync(0xffffffffu, key[q]);
            const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
            unsigned base = 0;
            if (lane == leader && key[q] >= 0) base = atomicAdd(&sh_cnt[key[q]], (unsigned)__popc(peers));
            rank[q] = __shfl_sync(0xffffffffu, base, leader) + __popc(peers & ((1u << lane) - 1u));
        }
        __syncthreads();
        if (threadIdx.x < nkeys) {
            unsigned long long seg = 0;                                        // start of this key's segment
            for (int k = 0; k < (int)threadIdx.x; ++k) seg += totals[k];
            sh_base[threadIdx.x] = seg + (sh_cnt[threadIdx.x] ? atomicAdd(&cursors[threadIdx.x], (unsigned long long)sh_cnt[threadIdx.x]) : 0ull);
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < SORT_TILE / NAV_THREADS; ++q)
            if (key[q] >= 0) perm[sh_base[key[q]] + rank[q]] = (uint32_t)(tile * SORT_TILE + q * NAV_THREADS + threadIdx.x);
        __syncthreads();
    }
}


// ---- host side ---------------------------------------------------------------------------------------------------
inline int cuda_fail(cudaError_t e, const char* where) {
    return fail(GN_CUDA_ERROR, std::string(where) + ": " + cudaGetErrorString(e));
}
#define GN_CUDA(call, where) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(e__, where); } while (0)

inline int nav_grid(int64_t n) {
    int64_t blocks = (n + NAV_THREADS - 1) / NAV_THREADS;
    const int64_t cap = 148 * 64;                 // grid-stride beyond this; multiple of the SM count
    return (int)std::max<int64_t>(1, std::min(blocks, cap));
}

template <class R> inline const GeoView<R>& view(const gn_geometry* g);
template <> inline const GeoView<float>& view<float>(const gn_geometry* g) { return g->v32; }
template <> inline const GeoView<double>& view<double>(const gn_geometry* g) { return g->v64; }

}  // namespace gn
