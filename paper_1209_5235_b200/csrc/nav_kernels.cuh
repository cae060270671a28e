// nav_kernels.cuh -- navigation kernels (locate, ComputeStep, surface normal, safety, the paper's free-path benchmark) and
// their launchers, templated on the precision; instantiated in nav_f32.cu / nav_f64.cu.
#pragma once
#include <cstdlib>
#include "common.cuh"
#include "coherent.cuh"
#include "impl.h"

namespace gn {

// -------------------------------------------------------------------------------------------------------
// navigation kernels: pure maps over queries
// -------------------------------------------------------------------------------------------------------
template <class R, bool HAS_DIR, bool FLAT>
__global__ void __launch_bounds__(NAV_THREADS, sizeof(R) == 4 ? NAV_LOCATE_MIN_BLOCKS : NAV_LOCATE_MIN_BLOCKS_F64) locate_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir,
                                                             int64_t n, int32_t* __restrict__ vol_out) {
    __shared__ BlockTables<R> tab;
    stage_tables(g, tab);
    __syncthreads();
    Navigator<R, HAS_DIR, FLAT> nav(g, &tab.ctx);
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        V3<R> w{0, 0, 0};
        if (HAS_DIR) { w.x = dir[3 * i]; w.y = dir[3 * i + 1]; w.z = dir[3 * i + 2]; }
        NodeRec<R> nd;
        vol_out[i] = nav.locate(x, w, nd);
    }
}

// locate on general geometries (tubes, rotations, nested placements) as a level-synchronous wavefront inside each warp.
// In locate_kernel every lane runs its whole descent; lanes of a warp sit at different depths of the placement tree (config 5:
// 70 % of the points are in the world volume, the others three to five levels down), so the voxel-cell lookups of a mother run
// at 2.6 of 32 lanes and the kernel at 14.4 (profiles/r2_compute_step_split.md).  Here a warp owns a tile of up to
// LOCATE_WTILE consecutive queries and walks the tree one level per round: the queries still descending are kept as a packed
// list in shared memory (slot in the tile, volume reached); 32 entries at a time, each lane runs Navigator::descend_level on
// one entry and puts it back (in place: a round writes no further than it has read) if it has further to go.  The lanes of a
// round all do the same thing -- cell lookup or list walk of one kind of mother, then occupancy tests of candidates -- and a
// query that is done leaves the list instead of idling in a warp.  No block barrier: a first version with one list per block
// ran at 24.7 lanes but waited at __syncthreads (10 warps per issue) and gained 5 %.  Same visits, same arithmetic, same
// answers as locate_kernel (tests/test_gpu_parity.py compares with the oracle bit for bit).  Queries are re-read from global
// memory at every level (the tile is 7 KB: L1), answers are written as they are found.
constexpr int LOCATE_WTILE = 256;
// blocks per SM, measured on config 5 (6 / 3: 40 / 80 registers; 8 / 4 spill, fp32 11.70 -> 11.62 ms, fp64 19.59 -> 19.36 ms; fp64 at 5, 6, 8: 20.0, 21.0, 22.1 ms)
#ifndef NAV_LEVELS_MIN_BLOCKS
#define NAV_LEVELS_MIN_BLOCKS 6
#endif
#ifndef NAV_LEVELS_MIN_BLOCKS_F64
#define NAV_LEVELS_MIN_BLOCKS_F64 3
#endif
template <class R, bool HAS_DIR>
__global__ void __launch_bounds__(NAV_THREADS, sizeof(R) == 4 ? NAV_LEVELS_MIN_BLOCKS : NAV_LEVELS_MIN_BLOCKS_F64)
locate_levels_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir, int64_t n, int32_t* __restrict__ vol_out, int wtile) {
    constexpr int WARPS = NAV_THREADS / 32;
    __shared__ BlockTables<R> tab;
    __shared__ int32_t sh_vol[WARPS][LOCATE_WTILE];      // per warp: the queries still descending -- volume reached ...
    __shared__ uint8_t sh_slot[WARPS][LOCATE_WTILE];     // ... and slot in the warp's tile
    static_assert(LOCATE_WTILE <= 256, "tile slots are stored in a byte");
    stage_tables(g, tab);
    __syncthreads();
    Navigator<R, HAS_DIR, true> nav(g, &tab.ctx);
    const unsigned lane = threadIdx.x & 31u, below = (1u << lane) - 1u;
    int32_t* const lv = sh_vol[threadIdx.x >> 5];
    uint8_t* const ls = sh_slot[threadIdx.x >> 5];
    const int64_t n_tiles = (n + wtile - 1) / wtile;
    for (int64_t wt = (int64_t)blockIdx.x * WARPS + (threadIdx.x >> 5); wt < n_tiles; wt += (int64_t)gridDim.x * WARPS) {
        const int64_t base = wt * wtile;
        unsigned count = 0;                               // entries in the list (warp-uniform)
        // the world volume and its own daughters: every query of the tile
        for (int s = 0; s < wtile; s += 32) {
            const int64_t i = base + s + lane;
            bool more = false; int vol = -1;
            if (i < n) {
                const V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
                V3<R> w{0, 0, 0};
                if (HAS_DIR) { w.x = dir[3 * i]; w.y = dir[3 * i + 1]; w.z = dir[3 * i + 2]; }
                NodeRec<R> nd = nav.node(0);
                V3<R> p, v;
                to_local<R, true>(g.rot, 0, nd, x, w, p, v);
                if (nav.occupied(nd, p, v)) { vol = 0; if (nd.ndau > 0) more = nav.descend_level(vol, nd, x, w); }
                if (!more) vol_out[i] = vol;
            }
            const unsigned bal = __ballot_sync(0xffffffffu, more);
            if (more) { const unsigned o = count + __popc(bal & below); lv[o] = vol; ls[o] = (uint8_t)(s + lane); }
            count += __popc(bal);
        }
        __syncwarp();
        while (count > 0) {                               // one level of the tree per turn
            unsigned kept = 0;
            for (unsigned t0 = 0; t0 < count; t0 += 32) {
                const unsigned t = t0 + lane;
                bool more = false; int vol = 0, slot = 0;
                if (t < count) {
                    vol = lv[t]; slot = ls[t];
                    const int64_t i = base + slot;
                    const V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
                    V3<R> w{0, 0, 0};
                    if (HAS_DIR) { w.x = dir[3 * i]; w.y = dir[3 * i + 1]; w.z = dir[3 * i + 2]; }
                    NodeRec<R> nd = nav.node(vol);
                    more = nav.descend_level(vol, nd, x, w);
                    if (!more) vol_out[i] = vol;
                }
                __syncwarp();                             // entries t0 .. t0 + 31 are read; kept <= t0: the writes below stay behind
                const unsigned bal = __ballot_sync(0xffffffffu, more);
                if (more) { const unsigned o = kept + __popc(bal & below); lv[o] = vol; ls[o] = (uint8_t)slot; }
                kept += __popc(bal);
            }
            __syncwarp();
            count = kept;
        }
    }
}
// queries per warp tile: LOCATE_WTILE when the batch fills the chip that way, fewer (a multiple of 32) for small batches
inline int locate_wtile(int64_t n) {
    const int64_t warps = 148 * 64;
    const int64_t per = (n + warps - 1) / warps;
    return (int)std::min<int64_t>(LOCATE_WTILE, std::max<int64_t>(32, (per + 31) / 32 * 32));
}
inline int locate_grid(int64_t n, int wtile) {
    const int64_t per_block = (int64_t)wtile * (NAV_THREADS / 32);
    return (int)std::max<int64_t>(1, std::min<int64_t>((n + per_block - 1) / per_block, 148 * 64));
}

template <class R, bool FLAT>
__global__ void __launch_bounds__(NAV_THREADS, sizeof(R) == 4 ? NAV_STEP_MIN_BLOCKS : NAV_STEP_MIN_BLOCKS_F64) step_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir,
                                                           const int32_t* __restrict__ vol_in, const R* __restrict__ max_step,
                                                           int64_t n, R* __restrict__ step_out, int32_t* __restrict__ next_out,
                                                           const uint32_t* __restrict__ perm) {
    __shared__ BlockTables<R> tab;
    stage_tables(g, tab);
    __syncthreads();
    Navigator<R, true, FLAT> nav(g, &tab.ctx);
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = perm ? (int64_t)perm[t] : t;                     // work order: queries grouped by volume key (sort_queries)
        V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        V3<R> w{dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        int vol = vol_in[i];
        R step = rinf<R>(); int next = -1;
        if (vol >= 0 && vol < g.n_nodes) {
            NodeRec<R> nd = nav.node(vol);
            V3<R> xn;
            nav.compute_step(vol, nd, x, w, max_step ? max_step[i] : rinf<R>(), step, xn);
            next = vol;
        }
        step_out[i] = step; next_out[i] = next;
    }
}

// Isotropic safety (reading 17): min of SafetyToOut of the volume's own solid and SafetyToIn of
// each of its daughters, SafetyToOut / In = max(-D, 0) / max(D, 0) with D the outsideness of C2.  Scan of the daughter list in
// index order, one thread per query (lanes of a warp in the same mother read the same daughters: broadcast loads from L1 /
// L2), ended as soon as the minimum is 0.
template <class R>
__global__ void __launch_bounds__(NAV_THREADS) safety_kernel(GeoView<R> g, const R* __restrict__ pos, const int32_t* __restrict__ vol_in,
                                                             int64_t n, R* __restrict__ safety_out) {
    __shared__ BlockTables<R> tab;
    stage_tables(g, tab);
    __syncthreads();
    const NavCtx<R>* c = &tab.ctx;
    const V3<R> w0{0, 0, 1};
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        const int vol = vol_in[i];
        R best = 0;
        if (vol >= 0 && vol < g.n_nodes) {
            const NodeRec<R> nd = load_node(g.node, vol);
            V3<R> p, v;
            to_local<R, true>(c->rot, vol, nd, x, w0, p, v);
            best = rmax(-outsideness(c->solids[nd.info & NODE_SOLID_MASK], p), (R)0);
            // Every term is >= +0, so the minimum is final once it is 0 (same bits as the full scan).  A voxelised mother
            // (10^5 daughters in a phantom's container) first looks at the daughters listed in the cells around the point:
            // a point of the mother that is not deep inside it usually lies in or on one of them, and the scan is skipped.
            if (nd.link < 0 && best > 0) {
                const V3<R> pm = p;
                int cursor = 0;
                for (int it = 0; it < 16 && best > 0; ++it) {
                    const int d = grid_candidate<R, true>(c->grids[~nd.link], c->cells, c->cand, pm, cursor, -1);
                    if (d == 0x7fffffff) break;
                    cursor = d + 1;
                    const NodeRec<R> dn = load_node(g.node, d);
                    to_local<R, true>(c->rot, d, dn, x, w0, p, v);
                    best = rmin(best, rmax(outsideness(c->solids[dn.info & NODE_SOLID_MASK], p), (R)0));
                }
            }
            const int first = __ldg(&g.dfirst[vol]);
            for (int k = 0; k < nd.ndau && best > 0; ++k) {
                const int d = __ldg(&g.dlist[first + k]);
                const NodeRec<R> dn = load_node(g.node, d);
                to_local<R, true>(c->rot, d, dn, x, w0, p, v);
                best = rmin(best, rmax(outsideness(c->solids[dn.info & NODE_SOLID_MASK], p), (R)0));
            }
        }
        safety_out[i] = best;
    }
}

// ComputeStep + surface normal of the boundary crossed
// ComputeStep of a general geometry as two wavefronts: the distance kernel and the relocation kernel each hold half of the
// navigator's code (the single kernel stalls on instruction fetch) and each runs through the work order by volume kind;
// the step lengths go through step_out, which the caller gets anyway.  Same arithmetic, same results.
template <class R>
__global__ void __launch_bounds__(NAV_THREADS, sizeof(R) == 4 ? NAV_STEP_MIN_BLOCKS : NAV_STEP_MIN_BLOCKS_F64)
step_distance_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir, const int32_t* __restrict__ vol_in, const R* __restrict__ max_step,
                     int64_t n, R* __restrict__ step_out, const uint32_t* __restrict__ perm, uint8_t* __restrict__ keys2, unsigned long long* __restrict__ totals2) {
    __shared__ BlockTables<R> tab;
    __shared__ unsigned sh_k2[SORT_KEYS2];
    stage_tables(g, tab);
    if (threadIdx.x < SORT_KEYS2) sh_k2[threadIdx.x] = 0;
    __syncthreads();
    Navigator<R, true, true> nav(g, &tab.ctx);
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = perm ? (int64_t)perm[t] : t;
        const V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        const V3<R> w{dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        const int vol = vol_in[i];
        R step = rinf<R>();
        int key2 = 2 * (SORT_KEYS - 1);
        if (vol >= 0 && vol < g.n_nodes) {
            const NodeRec<R> nd = nav.node(vol);
            bool entered = false;
            step = nav.step_distance(vol, nd, x, w, max_step ? max_step[i] : rinf<R>(), &entered);
            // key of the relocation to come: what the lanes of a warp will do there depends on the kind of volume they start in
            // and on whether they leave it or enter one of its daughters (a world query that leaves is done after one visit)
            key2 = 2 * (2 * nav.solid_of(nd).type + (nd.ndau > 0 ? 1 : 0)) + (entered ? 1 : 0);
        }
        step_out[i] = step;
        if (keys2) { keys2[i] = (uint8_t)key2; atomicAdd(&sh_k2[key2], 1u); }
    }
    __syncthreads();
    if (keys2 && threadIdx.x < SORT_KEYS2 && sh_k2[threadIdx.x]) atomicAdd(&totals2[threadIdx.x], (unsigned long long)sh_k2[threadIdx.x]);
}
template <class R>
__global__ void __launch_bounds__(NAV_THREADS, sizeof(R) == 4 ? NAV_STEP_MIN_BLOCKS : NAV_STEP_MIN_BLOCKS_F64)
step_relocate_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir, const int32_t* __restrict__ vol_in, const R* __restrict__ step_in,
                     int64_t n, int32_t* __restrict__ next_out, const uint32_t* __restrict__ perm) {
    __shared__ BlockTables<R> tab;
    stage_tables(g, tab);
    __syncthreads();
    Navigator<R, true, true> nav(g, &tab.ctx);
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = perm ? (int64_t)perm[t] : t;
        int vol = vol_in[i];
        int next = -1;
        if (vol >= 0 && vol < g.n_nodes) {
            const R step = step_in[i];
            if (step < rinf<R>()) {
                const V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
                const V3<R> w{dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
                NodeRec<R> nd = nav.node(vol);
                nav.relocate(vol, nd, advance(x, w, step), w);
            }
            next = vol;
        }
        next_out[i] = next;
    }
}

template <class R, bool FLAT>
__global__ void __launch_bounds__(NAV_THREADS) step_normal_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir,
                                                                  const int32_t* __restrict__ vol_in, const R* __restrict__ max_step, int64_t n,
                                                                  R* __restrict__ step_out, int32_t* __restrict__ next_out, R* __restrict__ normal_out) {
    __shared__ BlockTables<R> tab;
    stage_tables(g, tab);
    __syncthreads();
    Navigator<R, true, FLAT> nav(g, &tab.ctx);
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        V3<R> w{dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        int vol = vol_in[i];
        R step = rinf<R>(); int next = -1; V3<R> ng{0, 0, 0};
        if (vol >= 0 && vol < g.n_nodes) {
            NodeRec<R> nd = nav.node(vol);
            nav.compute_step_normal(vol, nd, x, w, max_step ? max_step[i] : rinf<R>(), step, ng);
            next = vol;
        }
        step_out[i] = step; next_out[i] = next;
        normal_out[3 * i] = ng.x; normal_out[3 * i + 1] = ng.y; normal_out[3 * i + 2] = ng.z;
    }
}

// -------------------------------------------------------------------------------------------------------
// the paper's own benchmark: Algorithm 1 with attenuation only, one thread per particle
// -------------------------------------------------------------------------------------------------------
template <class R, bool FLAT>
__global__ void __launch_bounds__(NAV_THREADS) free_path_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir,
                                                                const R* __restrict__ Yin, int64_t n, double mu_mass,
                                                                R* __restrict__ T_out, uint32_t* __restrict__ nsteps_out, const uint32_t* __restrict__ perm) {
    __shared__ BlockTables<R> tab;
    __shared__ R sh_mu[MAX_SMEM_MATS];
    stage_tables(g, tab);
    // Eq. 9: mu = rho mu_mass, here in 1/mm; fp64, rounded once to Real
    for (int i = threadIdx.x; i < g.n_mats && i < MAX_SMEM_MATS; i += blockDim.x) sh_mu[i] = (R)(g.rho[i] * mu_mass / 10.0);
    __syncthreads();
    Navigator<R, true, FLAT> nav(g, &tab.ctx);
    for (int64_t t_ = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t_ < n; t_ += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = perm ? (int64_t)perm[t_] : t_;                   // ray-coherent work order (coherent.cuh)
        V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        const V3<R> w{dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        NodeRec<R> nd;
        int vol = nav.locate(x, w, nd);
        R t = 0, Yrem = Yin[i], T = rinf<R>();
        uint32_t ns = 0; int zero_steps = 0;
        while (vol >= 0) {
            const R mu = nd.mat < MAX_SMEM_MATS ? sh_mu[nd.mat] : (R)(g.rho[nd.mat] * mu_mass / 10.0);
            const R s_int = mu > 0 ? rdiv(Yrem, mu) : rinf<R>();        // remaining part of Eq. 7
            R step; V3<R> xn;
            nav.compute_step(vol, nd, x, w, s_int, step, xn);             // "next intersection"
            ++ns;
            if (step == rinf<R>()) { T = t + s_int; break; }               // S_j >= Y inside this volume (L76)
            x = xn;
            t = t + step;
            Yrem = rmax(Yrem - step * mu, (R)0);                           // S_j update (L71)
            zero_steps = (step <= g.delta) ? zero_steps + 1 : 0;
            if (vol >= 0 && zero_steps >= g.stuck_limit) break;
        }
        T_out[i] = T;
        if (nsteps_out) nsteps_out[i] = ns;
    }
}

// (key, rank) of every ray of a batch for the ray-coherent work order: cell of the position, bin of the direction
template <class R>
__global__ void __launch_bounds__(NAV_THREADS) coh_ray_keys_kernel(CohGrid cg, const R* __restrict__ pos, const R* __restrict__ dir, int64_t n,
                                                                   unsigned* __restrict__ hist, uint2* __restrict__ kr) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t key = coh_key(cg, (float)pos[3 * i], (float)pos[3 * i + 1], (float)pos[3 * i + 2],
                                     (float)dir[3 * i], (float)dir[3 * i + 1], (float)dir[3 * i + 2], 0);
        kr[i] = make_uint2(key, atomicAdd(&hist[key], 1u));
    }
}
// Work order of a batch of rays (stream-ordered scratch from the handle's pool).  nullptr = arrival order: small batches, or
// no scratch to be had.  The caller frees *scratch_out with cudaFreeAsync once its kernel is enqueued.
constexpr int64_t COH_MIN_RAYS = 1 << 12;
template <class R>
static const uint32_t* ray_order(const gn_geometry* geo, const void* pos, const void* dir, int64_t n, cudaStream_t s, char** scratch_out) {
    *scratch_out = nullptr;
    if (n < COH_MIN_RAYS || n >= (1ll << 32) || !geo->pool) return nullptr;
    const CohGrid cg = coh_grid(geo->world_c, geo->world_h, 4, 16, 1);            // 64 cells x 4096 direction bins
    const unsigned nb = cg.buckets();
    const size_t b_hist = ((size_t)nb * 4 + 255) & ~(size_t)255, b_tiles = (coh_tiles(nb) * 4 + 255) & ~(size_t)255, b_kr = ((size_t)n * 8 + 255) & ~(size_t)255;
    char* scratch = nullptr;
    if (cudaMallocFromPoolAsync((void**)&scratch, b_hist + b_tiles + b_kr + (size_t)n * 4, geo->pool, s) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    unsigned* hist = (unsigned*)scratch; unsigned* tiles = (unsigned*)(scratch + b_hist);
    uint2* kr = (uint2*)(scratch + b_hist + b_tiles);
    uint32_t* perm = (uint32_t*)(scratch + b_hist + b_tiles + b_kr);
    cudaMemsetAsync(hist, 0, (size_t)nb * 4, s);
    coh_ray_keys_kernel<R><<<nav_grid(n), NAV_THREADS, 0, s>>>(cg, (const R*)pos, (const R*)dir, n, hist, kr);
    coh_build_order(hist, nb, tiles, kr, n, nullptr, perm, s);
    *scratch_out = scratch;
    return perm;
}

template <class R> int locate_impl(const gn_geometry* geo, const void* pos, const void* dir, int64_t n, int32_t* out, cudaStream_t s) {
    if (n == 0) return GN_OK;
    // geometries whose lanes do different things per node visit (tubes, rotations, long candidate lists) use the flat
    // one-visit-per-iteration search, coherent ones (voxel phantoms) the nested climb / descend loops
    if (geo->coherent) {
        if (dir) locate_kernel<R, true, false><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, n, out);
        else locate_kernel<R, false, false><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, nullptr, n, out);
    } else {
#ifdef GN_LOCATE_FLAT
        if (dir) locate_kernel<R, true, true><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, n, out);
        else locate_kernel<R, false, true><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, nullptr, n, out);
#else
        const int wtile = locate_wtile(n);
        if (dir) locate_levels_kernel<R, true><<<locate_grid(n, wtile), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, n, out, wtile);
        else locate_levels_kernel<R, false><<<locate_grid(n, wtile), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, nullptr, n, out, wtile);
#endif
    }
    GN_CUDA(cudaGetLastError(), "gn_nav_locate launch");
    return GN_OK;
}
// scratch head of the ComputeStep sorts: totals and cursors of the first order, totals and cursors of the second (u64 each)
constexpr size_t STEP_SORT_HEAD = 4 * SORT_KEYS_MAX * sizeof(unsigned long long);
// distance wavefront through `perm`, then -- with sort scratch -- the relocation order from the keys it wrote, then the relocation
// wavefront (keys and perm are reused: each is dead by the time it is overwritten, in stream order)
template <class R>
static void step_two_wavefronts(const gn_geometry* geo, const void* pos, const void* dir, const int32_t* vol, const void* ms, int64_t n, void* step,
                                int32_t* next, uint32_t* perm, uint8_t* keys, unsigned long long* totals2, cudaStream_t s) {
    step_distance_kernel<R><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, vol, (const R*)ms, n, (R*)step, perm, keys, totals2);
    if (perm && keys && totals2)
        sort_scatter_kernel<<<nav_grid((n + 3) / 4), NAV_THREADS, 0, s>>>(keys, n, totals2, totals2 + SORT_KEYS_MAX, perm, nullptr, SORT_KEYS2);
    step_relocate_kernel<R><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, vol, (const R*)step, n, next, perm);
}

template <class R> int step_impl(const gn_geometry* geo, const void* pos, const void* dir, const int32_t* vol, const void* ms,
                                 int64_t n, void* step, int32_t* next, cudaStream_t s) {
    if (n == 0) return GN_OK;
    if (geo->coherent) {
        step_kernel<R, false><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, vol, (const R*)ms, n, (R*)step, next, nullptr);
        GN_CUDA(cudaGetLastError(), "gn_nav_compute_step launch");
        return GN_OK;
    }
    // general geometry: group the queries by volume key first (large batches only; stream-ordered scratch).  Two wavefronts,
    // each through a work order of its own: the distances by the kind of the current volume, the relocations by that kind
    // and by whether the boundary found is the volume's own or a daughter's (the distance kernel writes those keys).
    // Measured on config 5 against the single step_kernel<R, true>: 16.25 -> 14.92 ms with one order, see DESIGN.md.
    uint32_t* perm = nullptr;
    uint8_t* keys = nullptr;
    unsigned long long* totals2 = nullptr;
    char* scratch = nullptr;
    if (n >= (1 << 16) && n < (1ll << 32)) {
        const size_t bytes = STEP_SORT_HEAD + (size_t)n + 4 * (size_t)n + 64;
        if (geo->pool && cudaMallocFromPoolAsync((void**)&scratch, bytes, geo->pool, s) == cudaSuccess) {
            unsigned long long* totals = (unsigned long long*)scratch; unsigned long long* cursors = totals + SORT_KEYS_MAX;
            totals2 = cursors + SORT_KEYS_MAX;
            keys = (uint8_t*)(scratch + STEP_SORT_HEAD);
            perm = (uint32_t*)(scratch + STEP_SORT_HEAD + (((size_t)n + 63) & ~(size_t)63));
            cudaMemsetAsync(scratch, 0, STEP_SORT_HEAD, s);
            sort_keys_kernel<R><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), vol, n, keys, totals);
            sort_scatter_kernel<<<nav_grid((n + 3) / 4), NAV_THREADS, 0, s>>>(keys, n, totals, cursors, perm, nullptr);
        } else { cudaGetLastError(); scratch = nullptr; }                     // no scratch: run in arrival order
    }
    step_two_wavefronts<R>(geo, pos, dir, vol, ms, n, step, next, perm, keys, totals2, s);
    cudaError_t e = cudaGetLastError();
    if (scratch) cudaFreeAsync(scratch, s);
    GN_CUDA(e, "gn_nav_compute_step launch");
    return GN_OK;
}

template <class R> int step_normal_impl(const gn_geometry* geo, const void* pos, const void* dir, const int32_t* vol, const void* ms,
                                        int64_t n, void* step, int32_t* next, void* normal, cudaStream_t s) {
    if (n == 0) return GN_OK;
    if (geo->coherent) step_normal_kernel<R, false><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, vol, (const R*)ms, n, (R*)step, next, (R*)normal);
    else step_normal_kernel<R, true><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, vol, (const R*)ms, n, (R*)step, next, (R*)normal);
    GN_CUDA(cudaGetLastError(), "gn_nav_compute_step_normal launch");
    return GN_OK;
}

template <class R> int safety_impl(const gn_geometry* geo, const void* pos, const int32_t* vol, int64_t n, void* out, cudaStream_t s) {
    if (n == 0) return GN_OK;
    safety_kernel<R><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, vol, n, (R*)out);
    GN_CUDA(cudaGetLastError(), "gn_nav_compute_safety launch");
    return GN_OK;
}

template <class R> int free_path_impl(const gn_geometry* geo, const void* pos, const void* dir, const void* Y, int64_t n, double mu_mass,
                                      void* T, uint32_t* ns, cudaStream_t s) {
    if (n == 0) return GN_OK;
    const int64_t blocks = (n + NAV_THREADS - 1) / NAV_THREADS;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(blocks, 148 * 64));
    // one thread walks one particle to the end: lanes that start close together and look the same way visit the same
    // cells and daughters, so the particles are walked in ray-coherent order (Random set, N = 1e5: 1.4x; 1e6: 2.4x)
    char* scratch = nullptr;
    const uint32_t* perm = ray_order<R>(geo, pos, dir, n, s, &scratch);
    if (geo->coherent) free_path_kernel<R, false><<<grid, NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, (const R*)Y, n, mu_mass, (R*)T, ns, perm);
    else free_path_kernel<R, true><<<grid, NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, (const R*)Y, n, mu_mass, (R*)T, ns, perm);
    const cudaError_t e = cudaGetLastError();
    if (scratch) cudaFreeAsync(scratch, s);
    GN_CUDA(e, "gn_free_path_run launch");
    return GN_OK;
}

}  // namespace gn
