// voxel_pass.cuh -- the wavefront schedule of geometries that are mostly regular voxels (voxel phantoms; box-only kernels).
//
// The lean step pass of transport.cuh keeps the general ComputeStep in line, which costs it registers (80, 24 warps / SM)
// while ~94 % of a phantom's steps are "leave a regular voxel through one face into the next one".  Here that step gets a
// kernel of its own:
//   * voxel_pass: every thread loads one travelling photon and takes up to K regular_steps (nav.cuh); a photon that reaches
//     its interaction point parks (as before), one whose next step is anything else -- it stands in the world or the
//     container, leaves through an edge or out of the phantom -- goes to the slow buffer S; parked photons go to the back of
//     the output queue, the rest to the front.  No general navigation code, no physics: few registers, many warps per SM
//     to hide the latency of the dependent node loads.
//   * general_pass: one thread per flagged photon takes general ComputeSteps until the photon stands in a regular voxel
//     again (at most SLOW_STEPS) and appends it to the input queue of the coming voxel_pass; interact_pass (transport.cuh)
//     then handles the parked photons as in the other schedules.  Three populations, three kernels: full, uniform warps.
// Per photon the arithmetic and its order are those of the other schedules; only which kernel takes which step differs.
#pragma once

namespace gn {

enum : uint32_t { REC_ABOVE = 1u, REC_PENDING = 2u, REC_MAT_SHIFT = 8u };      // PhotonRec::tail[0]: flags, material of vol from bit 8
#ifndef VOX_MIN_BLOCKS
#define VOX_MIN_BLOCKS 8            // 64 registers: 32 warps / SM (10 blocks = 48 registers spill)
#endif
#ifndef GENERAL_MIN_BLOCKS
#define GENERAL_MIN_BLOCKS 6        // general_pass, fp32: 80 registers, 24 warps / SM
#endif
#ifndef VOX_MIN_BLOCKS_F64
#define VOX_MIN_BLOCKS_F64 6        // voxel_pass, fp64: 80 registers, 24 warps / SM (4 / 5 / 6 / 8 blocks measured on config 2: 2.55 / 2.44 / 2.42 / 2.47 ms)
#endif
#ifndef GENERAL_MIN_BLOCKS_F64
#define GENERAL_MIN_BLOCKS_F64 2
#endif
constexpr int SLOW_STEPS = 8;       // general steps a flagged photon may take in one slow_pass

template <class R> __device__ __forceinline__ bool direction_cacheable(const V3<R>& w, R delta) {
    VoxLane<R> c; lane_direction(w, delta, c);
    return c.ok;
}

template <class R, bool TRACK, bool SLABS>
__global__ void __launch_bounds__(TR_THREADS, TR_PER_128 * (sizeof(R) == 4 ? VOX_MIN_BLOCKS : VOX_MIN_BLOCKS_F64))
voxel_pass(GeoView<R> g, const PassCounters* __restrict__ cin, PassCounters* __restrict__ cout, const PhotonRec<R>* __restrict__ qin,
           PhotonRec<R>* __restrict__ qout, PhotonRec<R>* __restrict__ S, uint32_t cap, DevStats* __restrict__ stats, PerPhotonOut pp, SecIO<R> sec,
           int K, int regroup_pct, int timed) {
    const unsigned n_front = cin->front, n_in = n_front + cin->back;
    if (blockIdx.x * TR_THREADS >= n_in) return;
    __shared__ SolidRec<R> sh_solids[MAX_SMEM_SOLIDS];
    __shared__ GridRec<R> sh_grids[MAX_SMEM_GRIDS];
    __shared__ MatRec<R> sh_mats[MAX_SMEM_MATS];
    __shared__ unsigned sh_wcount[3][TR_WARPS];
    __shared__ unsigned sh_base[3];
    __shared__ unsigned long long sh_steps, sh_stuck;
    __shared__ double sh_estuck;
    // the tables fit (a condition of the voxel schedule, gn_geometry::voxel_sched): shared-memory addresses, no generic loads
    for (int i = threadIdx.x; i < g.n_solids; i += blockDim.x) sh_solids[i] = g.solids[i];
    for (int i = threadIdx.x; i < g.n_grids; i += blockDim.x) sh_grids[i] = g.grids[i];
    for (int i = threadIdx.x; i < g.n_mats; i += blockDim.x) sh_mats[i] = g.mats[i];
    const SolidRec<R>* solids = sh_solids; const GridRec<R>* grids = sh_grids; const MatRec<R>* mats = sh_mats;
    if (threadIdx.x == 0) { sh_steps = 0; sh_stuck = 0; sh_estuck = 0.0; }
    __syncthreads();
    const unsigned i = blockIdx.x * TR_THREADS + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    bool alive = i < n_in, pending = false, needgen = false, stuck = false;
    V3<R> x{0, 0, 0}, w{0, 0, 1}; R E = 1, Y = 0, gPE = 0, gKN = 0, L2k = 0;
    uint32_t idx = 0, misc = 0, ctr = 0, above = 0;
    uint64_t h = 0;
    int vol = -1; NodeRec<R> nd = {};
    VoxLane<R> vl; vl.hx = vl.hy = vl.hz = 0; vl.r0 = vl.r1 = vl.r2 = 0; vl.solid = -1; vl.ok = false;
    unsigned c_steps = 0;
    if (alive) {
        GN_CHECK(n_in <= cap, CHK_LOAD_SLOT);
        PhotonRec<R> r; load_rec(qin, i < n_front ? i : cap - 1u - (i - n_front), r);
        GN_CHECK(r.vol < g.n_nodes, CHK_VOLUME);
        if (r.vol < 0) alive = false;                        // absorbed by interact_pass
        x.x = r.x; x.y = r.y; x.z = r.z; w.x = r.wx; w.y = r.wy; w.z = r.wz; E = r.E; Y = r.Y;
        gPE = r.gPE; gKN = r.gKN; L2k = r.L2k; above = r.tail[0] & REC_ABOVE;
        pending = (r.tail[0] & REC_PENDING) != 0;
        idx = r.idx; misc = r.misc; ctr = r.ctr; vol = r.vol;
        if (alive) {
            nd = load_node(g.node, vol);
            lane_direction(w, g.delta, vl);
            lane_solid(solids, nd.info, vl);
            if (!(nd.info & (NODE_REGULAR | (SLABS ? NODE_SLAB : 0))) || !vl.ok) needgen = true;
            if (TRACK && !pending && !needgen) h = hash_state(pp, sec, idx);
        }
    }
    int act0 = 32;
#pragma unroll 1
    for (int k = 0; k < K; ++k) {
        const bool go = alive && !pending && !needgen;
        const unsigned act = __ballot_sync(0xffffffffu, go);
        if (act == 0) break;
        if (k == 0) act0 = __popc(act);
        else if (__popc(act) * 100 < act0 * regroup_pct) break;        // regroup: let the compaction refill this warp
        if (go) {
            const MatRec<R> m = mats[nd.mat];
            const R muPE = m.aPE * gPE, muC = m.aC * gKN;
            const R P = rmin((R)(28.0 / 9.0) * L2k - (R)(218.0 / 27.0), m.capZ);
            const R muP = (above && P > 0) ? m.aP * P : (R)0;
            const R mu = (muPE + muC) + muP;
            R step = 0; V3<R> xn{0, 0, 0};
            const int vol_before = vol;
            const int rc = regular_step<R, SLABS>(g, grids, solids, x, w, vl, mu, Y, vol, nd, step, xn);
            if (rc == REG_BAIL) needgen = true;
            else {
                ++c_steps; misc += 0x100u;
                uint32_t zs = misc & 0xffu;
                zs = (step <= g.delta) ? min(zs + 1u, 255u) : 0u;      // step = s_int for an interaction step
                misc = (misc & ~0xffu) | zs;
                if (rc == REG_INTERACT) {
                    x = advance(x, w, step);
                    pending = true;                                     // the event word of this step is written by the interaction
                } else {
                    x = xn;
                    Y = rmax(Y - step * mu, (R)0);                      // S_j update
                    int ev = EV_BOUNDARY;
                    if (zs >= (uint32_t)g.stuck_limit) { ev = EV_STUCK; stuck = true; alive = false; }      // stuck guard (C9)
                    if (TRACK) {
                        fnv_word(h, (uint32_t)vol_before); fnv_word(h, (uint32_t)ev);
                        if (stuck) history_out(pp, sec, idx, h, misc >> 8, E);
                    }
                }
            }
        }
    }
    // ---- compaction: travelling photons to the front, parked ones to the back of the other queue, flagged ones to S ------
    const bool key1 = alive && pending, key2 = alive && !pending && needgen;
    const unsigned bal0 = __ballot_sync(0xffffffffu, alive && !key1 && !key2), bal1 = __ballot_sync(0xffffffffu, key1), bal2 = __ballot_sync(0xffffffffu, key2);
    if (lane == 0) { sh_wcount[0][warp] = __popc(bal0); sh_wcount[1][warp] = __popc(bal1); sh_wcount[2][warp] = __popc(bal2); }
    __syncthreads();
    if (threadIdx.x < 3) {
        unsigned tot = 0;
        for (int q = 0; q < TR_WARPS; ++q) { unsigned c = sh_wcount[threadIdx.x][q]; sh_wcount[threadIdx.x][q] = tot; tot += c; }
        sh_base[threadIdx.x] = tot ? atomicAdd(threadIdx.x == 0 ? &cout->front : (threadIdx.x == 1 ? &cout->back : &cout->slow), tot) : 0u;
    }
    __syncthreads();
    if (alive) {
        const unsigned below = (1u << lane) - 1u;
        PhotonRec<R> r;
        r.x = x.x; r.y = x.y; r.z = x.z; r.wx = w.x; r.wy = w.y; r.wz = w.z; r.E = E; r.Y = Y;
        r.gPE = gPE; r.gKN = gKN; r.L2k = L2k; r.vol = vol; r.idx = idx; r.ctr = ctr; r.misc = misc;
#pragma unroll
        for (int q = 0; q < (int)(sizeof(r.tail) / 4); ++q) r.tail[q] = 0;
        r.tail[0] = above | (pending ? REC_PENDING : 0u) | ((uint32_t)nd.mat << REC_MAT_SHIFT);
        GN_CHECK(vol >= 0 && vol < g.n_nodes && nd.mat < g.n_mats, CHK_VOLUME);
        GN_CHECK(!key2 || sh_base[2] + sh_wcount[2][warp] + __popc(bal2 & below) < cap, CHK_SLOW_SLOT);
        GN_CHECK(key2 || (key1 ? sh_base[1] + sh_wcount[1][warp] + __popc(bal1 & below) : sh_base[0] + sh_wcount[0][warp] + __popc(bal0 & below)) < cap, CHK_STORE_SLOT);
        if (key2) store_rec(S, sh_base[2] + sh_wcount[2][warp] + __popc(bal2 & below), r);
        else store_rec(qout, key1 ? cap - 1u - (sh_base[1] + sh_wcount[1][warp] + __popc(bal1 & below)) : sh_base[0] + sh_wcount[0][warp] + __popc(bal0 & below), r);
        if (TRACK && c_steps) hash_state(pp, sec, idx) = h;
    }
    {
        const unsigned s = warp_sum(c_steps);
        const unsigned ns = warp_sum(stuck ? 1u : 0u);
        if (lane == 0 && s) atomicAdd(&sh_steps, (unsigned long long)s);
        if (ns) {
            const double es = warp_sum(stuck ? (double)E : 0.0);
            if (lane == 0) { atomicAdd(&sh_stuck, (unsigned long long)ns); atomicAdd(&sh_estuck, es); }
        }
    }
    __syncthreads();
    GN_CHECK(cout->front + cout->back + cout->slow <= cap, CHK_SEGMENTS);
    if (threadIdx.x == 0) {
        if (sh_steps) { atomicAdd(&stats->cnt[ST_STEPS], sh_steps); if (timed) atomicAdd(&stats->lean_steps, sh_steps); }
        if (sh_stuck) { atomicAdd(&stats->cnt[ST_STUCK], sh_stuck); atomicAdd(&stats->en[EN_STUCK], sh_estuck); }
    }
}

// The general wavefront of the voxel schedule: one thread per flagged photon (slow buffer S, filled by the previous
// voxel_pass) takes general ComputeSteps until the photon stands in a regular voxel again (at most SLOW_STEPS; typically one:
// an exit through an edge, or two: out of the phantom and out of the world).  Survivors are appended to the input queue of the
// coming voxel_pass -- travelling ones behind its front segment, those that reached their interaction point to its back
// segment, where interact_pass finds them; there is room, because front + back + flagged never exceeds the photons alive.
template <class R, bool TRACK>
__global__ void __launch_bounds__(TR_THREADS, TR_PER_128 * (sizeof(R) == 4 ? GENERAL_MIN_BLOCKS : GENERAL_MIN_BLOCKS_F64))
general_pass(GeoView<R> g, PassCounters* __restrict__ ctr, const PhotonRec<R>* __restrict__ S, PhotonRec<R>* __restrict__ q, uint32_t cap,
             DevStats* __restrict__ stats, PerPhotonOut pp, SecIO<R> sec) {
    const unsigned n = ctr->slow;
    if (blockIdx.x * TR_THREADS >= n) return;
    __shared__ BlockTables<R> tab;
    __shared__ MatRec<R> sh_mats[MAX_SMEM_MATS];
    __shared__ unsigned long long sh_cnt[ST_COUNT];
    __shared__ double sh_en[4];
    stage_tables(g, tab);
    const MatRec<R>* mats = g.mats;
    if (g.n_mats <= MAX_SMEM_MATS) { for (int i = threadIdx.x; i < g.n_mats; i += blockDim.x) sh_mats[i] = g.mats[i]; mats = sh_mats; }
    if (threadIdx.x < ST_COUNT) sh_cnt[threadIdx.x] = 0;
    if (threadIdx.x < 4) sh_en[threadIdx.x] = 0.0;
    __syncthreads();
    Navigator<R, true, false> nav(g, &tab.ctx);
    const unsigned i = blockIdx.x * TR_THREADS + threadIdx.x;
    const int lane = threadIdx.x & 31;
    bool alive = i < n, pending = false;
    PhotonRec<R> r;
    unsigned c_steps = 0, c_esc = 0, c_stuck = 0; double e_esc = 0.0, e_stuck = 0.0;
    if (alive) {
        GN_CHECK(n <= cap, CHK_SLOW_SLOT);
        load_rec(S, i, r);
        GN_CHECK(r.vol >= 0 && r.vol < g.n_nodes, CHK_VOLUME);
        V3<R> x{r.x, r.y, r.z};
        const V3<R> w{r.wx, r.wy, r.wz};
        R Y = r.Y;
        uint32_t misc = r.misc;
        const int above = (int)(r.tail[0] & REC_ABOVE);
        int vol = r.vol;
        uint64_t h = 0;
        if (TRACK) h = hash_state(pp, sec, r.idx);
        NodeRec<R> nd = nav.node(vol);
        const bool cacheable = direction_cacheable(w, g.delta);
        for (int it = 0; it < SLOW_STEPS; ++it) {
            const R mu = photon_mu(g, mats[nd.mat], nd.mat, r.E, r.gPE, r.gKN, r.L2k, above).tot;
            const R s_int = mu > 0 ? rdiv(Y, mu) : rinf<R>();              // remaining part of Eq. 7
            const int vol_before = vol;
            R step; V3<R> xn;
            nav.compute_step(vol, nd, x, w, s_int, step, xn);              // "next intersection"
            ++c_steps; misc += 0x100u;
            const bool inter = step == rinf<R>();
            const R len = inter ? s_int : step;
            uint32_t zs = misc & 0xffu;
            zs = (len <= g.delta) ? min(zs + 1u, 255u) : 0u;
            misc = (misc & ~0xffu) | zs;
            if (inter) { x = advance(x, w, s_int); pending = true; break; } // the interaction writes this step's event word
            x = xn;
            Y = rmax(Y - step * mu, (R)0);                                 // S_j update
            int ev = EV_BOUNDARY;
            if (vol < 0) { ev = EV_ESCAPE; alive = false; ++c_esc; e_esc += (double)r.E; }
            else if (zs >= (uint32_t)g.stuck_limit) { ev = EV_STUCK; alive = false; ++c_stuck; e_stuck += (double)r.E; }      // stuck guard (C9)
            if (TRACK) { fnv_word(h, (uint32_t)vol_before); fnv_word(h, (uint32_t)ev); if (!alive) history_out(pp, sec, r.idx, h, misc >> 8, r.E); }
            if (!alive || ((nd.info & (NODE_REGULAR | NODE_SLAB)) && cacheable)) break;  // gone, or voxel_pass takes over
        }
        if (TRACK && alive) hash_state(pp, sec, r.idx) = h;
        r.x = x.x; r.y = x.y; r.z = x.z; r.Y = Y; r.misc = misc; r.vol = vol;
        r.tail[0] = (uint32_t)above | (pending ? REC_PENDING : 0u) | ((uint32_t)nd.mat << REC_MAT_SHIFT);
    }
    // ---- append the survivors to the queue: warp-aggregated cursors ------------------------------------------------------
    {
        const unsigned b0 = __ballot_sync(0xffffffffu, alive && !pending), b1 = __ballot_sync(0xffffffffu, alive && pending);
        unsigned base0 = 0, base1 = 0;
        if (lane == 0) { if (b0) base0 = atomicAdd(&ctr->front, (unsigned)__popc(b0)); if (b1) base1 = atomicAdd(&ctr->back, (unsigned)__popc(b1)); }
        base0 = __shfl_sync(0xffffffffu, base0, 0); base1 = __shfl_sync(0xffffffffu, base1, 0);
        const unsigned below = (1u << lane) - 1u;
        GN_CHECK(!alive || (pending ? base1 + __popc(b1 & below) : base0 + __popc(b0 & below)) < cap, CHK_STORE_SLOT);
        if (alive) store_rec(q, pending ? cap - 1u - (base1 + __popc(b1 & below)) : base0 + __popc(b0 & below), r);
    }
    {
        const unsigned s = warp_sum(c_steps), ne = warp_sum(c_esc), ns = warp_sum(c_stuck);
        if (lane == 0 && s) atomicAdd(&sh_cnt[ST_STEPS], (unsigned long long)s);
        if (ne) { const double ee = warp_sum(e_esc); if (lane == 0) { atomicAdd(&sh_cnt[ST_ESCAPED], (unsigned long long)ne); atomicAdd(&sh_en[EN_ESCAPED], ee); } }
        if (ns) { const double es = warp_sum(e_stuck); if (lane == 0) { atomicAdd(&sh_cnt[ST_STUCK], (unsigned long long)ns); atomicAdd(&sh_en[EN_STUCK], es); } }
    }
    __syncthreads();
    GN_CHECK(ctr->front + ctr->back <= cap, CHK_SEGMENTS);
    if (threadIdx.x < ST_COUNT && sh_cnt[threadIdx.x]) atomicAdd(&stats->cnt[threadIdx.x], sh_cnt[threadIdx.x]);
    if (threadIdx.x >= 16 && threadIdx.x < 20 && sh_en[threadIdx.x - 16] != 0.0) atomicAdd(&stats->en[threadIdx.x - 16], sh_en[threadIdx.x - 16]);
}

}  // namespace gn
