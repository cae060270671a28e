// voxel_pass.cuh -- the wavefront schedule of geometries that are mostly regular voxels (voxel phantoms; box-only kernels).
//
// The lean step pass of transport.cuh keeps the general ComputeStep in line, which costs it registers (80, 24 warps / SM)
// while ~94 % of a phantom's steps are "leave a regular voxel through one face into the next one".  Here that step gets a
// kernel of its own:
//   * voxel_pass: every thread loads one travelling photon and takes up to K regular_steps (nav.cuh); a photon that reaches
//     its interaction point parks (as before), one whose next step is anything else -- it stands in the world or the
//     container, leaves through an edge or out of the phantom -- is flagged NEED_GENERAL; both kinds go to the BACK of the
//     output queue, the rest to the front.  No general navigation code, no physics: few registers, many warps per SM to hide
//     the latency of the dependent cell -> node loads.
//   * slow_pass (instead of interact_pass): one thread per photon of the back segment; flagged photons take general
//     ComputeSteps until they stand in a regular voxel again (at most SLOW_STEPS), parked ones interact.  In place.
// Per photon the arithmetic and its order are those of the other schedules; only which kernel takes which step differs.
#pragma once

namespace gn {

enum : uint32_t { REC_ABOVE = 1u, REC_PENDING = 2u, REC_NEED_GENERAL = 4u };      // PhotonRec::tail[0]
#ifndef VOX_MIN_BLOCKS
#define VOX_MIN_BLOCKS 8            // 64 registers: 32 warps / SM (10 blocks = 48 registers spill)
#endif
constexpr int SLOW_STEPS = 8;       // general steps a flagged photon may take in one slow_pass

template <class R> __device__ __forceinline__ bool direction_cacheable(const V3<R>& w, R delta) {
    VoxLane<R> c; lane_direction(w, delta, c);
    return c.ok;
}

template <class R, bool TRACK>
__global__ void __launch_bounds__(TR_THREADS, sizeof(R) == 4 ? VOX_MIN_BLOCKS : 4)
voxel_pass(GeoView<R> g, const PassCounters* __restrict__ cin, PassCounters* __restrict__ cout, const PhotonRec<R>* __restrict__ qin,
           PhotonRec<R>* __restrict__ qout, uint32_t cap, DevStats* __restrict__ stats, PerPhotonOut pp, SecIO<R> sec, int K, int regroup_pct, int timed) {
    const unsigned n_front = cin->front, n_in = n_front + cin->back;
    if (blockIdx.x * TR_THREADS >= n_in) return;
    __shared__ SolidRec<R> sh_solids[MAX_SMEM_SOLIDS];
    __shared__ GridRec<R> sh_grids[MAX_SMEM_GRIDS];
    __shared__ MatRec<R> sh_mats[MAX_SMEM_MATS];
    __shared__ unsigned sh_wcount[2][TR_WARPS];
    __shared__ unsigned sh_base[2];
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
        PhotonRec<R> r; load_rec(qin, i < n_front ? i : cap - 1u - (i - n_front), r);
        if (r.vol < 0) alive = false;                        // ended in slow_pass
        x.x = r.x; x.y = r.y; x.z = r.z; w.x = r.wx; w.y = r.wy; w.z = r.wz; E = r.E; Y = r.Y;
        gPE = r.gPE; gKN = r.gKN; L2k = r.L2k; above = r.tail[0] & REC_ABOVE;
        pending = (r.tail[0] & REC_PENDING) != 0; needgen = (r.tail[0] & REC_NEED_GENERAL) != 0;
        idx = r.idx; misc = r.misc; ctr = r.ctr; vol = r.vol;
        if (alive) {
            nd = load_node(g.node, vol);
            lane_direction(w, g.delta, vl);
            lane_solid(solids, nd.info, vl);
            if (!(nd.info & NODE_REGULAR) || !vl.ok) needgen = true;
            if (TRACK && !pending && !needgen) h = pp.hash[idx];
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
            const int rc = regular_step(g, grids, x, w, vl, mu, Y, vol, nd, step, xn);
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
    // ---- compaction: travelling photons to the front, parked / flagged ones to the back of the other queue -----------
    const bool key1 = alive && (pending || needgen);
    const unsigned bal0 = __ballot_sync(0xffffffffu, alive && !key1), bal1 = __ballot_sync(0xffffffffu, key1);
    if (lane == 0) { sh_wcount[0][warp] = __popc(bal0); sh_wcount[1][warp] = __popc(bal1); }
    __syncthreads();
    if (threadIdx.x < 2) {
        unsigned tot = 0;
        for (int q = 0; q < TR_WARPS; ++q) { unsigned c = sh_wcount[threadIdx.x][q]; sh_wcount[threadIdx.x][q] = tot; tot += c; }
        sh_base[threadIdx.x] = tot ? atomicAdd(threadIdx.x == 0 ? &cout->front : &cout->back, tot) : 0u;
    }
    __syncthreads();
    if (alive) {
        const unsigned below = (1u << lane) - 1u;
        const unsigned o = key1 ? cap - 1u - (sh_base[1] + sh_wcount[1][warp] + __popc(bal1 & below))
                                : sh_base[0] + sh_wcount[0][warp] + __popc(bal0 & below);
        PhotonRec<R> r;
        r.x = x.x; r.y = x.y; r.z = x.z; r.wx = w.x; r.wy = w.y; r.wz = w.z; r.E = E; r.Y = Y;
        r.gPE = gPE; r.gKN = gKN; r.L2k = L2k; r.vol = vol; r.idx = idx; r.ctr = ctr; r.misc = misc;
#pragma unroll
        for (int q = 0; q < (int)(sizeof(r.tail) / 4); ++q) r.tail[q] = 0;
        r.tail[0] = above | (pending ? REC_PENDING : 0u) | (needgen ? REC_NEED_GENERAL : 0u);
        store_rec(qout, o, r);
        if (TRACK && c_steps) pp.hash[idx] = h;
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
    if (threadIdx.x == 0) {
        if (sh_steps) { atomicAdd(&stats->cnt[ST_STEPS], sh_steps); if (timed) atomicAdd(&stats->lean_steps, sh_steps); }
        if (sh_stuck) { atomicAdd(&stats->cnt[ST_STUCK], sh_stuck); atomicAdd(&stats->en[EN_STUCK], sh_estuck); }
    }
}

// The slow wavefront of the voxel schedule: general ComputeSteps for the flagged photons, interactions for the parked ones.
template <class R, bool TRACK>
__global__ void __launch_bounds__(TR_THREADS)
slow_pass(GeoView<R> g, uint64_t seed, uint64_t first_id, const PassCounters* __restrict__ cin, PhotonRec<R>* __restrict__ q, uint32_t cap,
          double* __restrict__ edep, DevStats* __restrict__ stats, PerPhotonOut pp, SecIO<R> sec) {
    const unsigned n = cin->back;
    if (blockIdx.x * TR_THREADS >= n) return;
    __shared__ BlockTables<R> tab;
    __shared__ MatRec<R> sh_mats[MAX_SMEM_MATS];
    __shared__ unsigned long long sh_cnt[8];
    __shared__ double sh_en[4];
    stage_tables(g, tab);
    const MatRec<R>* mats = g.mats;
    if (g.n_mats <= MAX_SMEM_MATS) { for (int i = threadIdx.x; i < g.n_mats; i += blockDim.x) sh_mats[i] = g.mats[i]; mats = sh_mats; }
    if (threadIdx.x < 8) sh_cnt[threadIdx.x] = 0;
    if (threadIdx.x < 4) sh_en[threadIdx.x] = 0.0;
    __syncthreads();
    Navigator<R, true, false> nav(g, &tab.ctx);
    const unsigned i = blockIdx.x * TR_THREADS + threadIdx.x;
    const bool active = i < n;
    double dep_d = 0.0; int dep_vol = 0; bool has_dep = false;
    if (active) {
        PhotonRec<R> r; load_rec(q, cap - 1u - i, r);
        V3<R> x{r.x, r.y, r.z}, w{r.wx, r.wy, r.wz};
        R E = r.E, Y = r.Y, gPE = r.gPE, gKN = r.gKN, L2k = r.L2k;
        uint32_t misc = r.misc, ctr = r.ctr; const uint32_t idx = r.idx;
        int above = (int)(r.tail[0] & REC_ABOVE), vol = r.vol;
        bool pending = (r.tail[0] & REC_PENDING) != 0, needgen = (r.tail[0] & REC_NEED_GENERAL) != 0, alive = vol >= 0;
        uint64_t h = 0;
        if (TRACK && alive) h = pp.hash[idx];
        NodeRec<R> nd = {};
        bool have_nd = false;
        unsigned c_steps = 0;
        auto mu_of = [&](int mat, R& muPE, R& muC, R& muP) -> R {
            const MatRec<R> m = mats[mat];
            muPE = m.aPE * gPE; muC = m.aC * gKN;
            const R P = rmin((R)(28.0 / 9.0) * L2k - (R)(218.0 / 27.0), m.capZ);
            muP = (above && P > 0) ? m.aP * P : (R)0;
            return (muPE + muC) + muP;
        };
        auto end_history = [&](int ev, int vol_before) {
            if (TRACK) { fnv_word(h, (uint32_t)vol_before); fnv_word(h, (uint32_t)ev); if (!alive) history_out(pp, sec, idx, h, misc >> 8, E); }
        };
        if (alive && needgen && !pending) {
            nd = nav.node(vol); have_nd = true;
            for (int it = 0; it < SLOW_STEPS; ++it) {
                R muPE, muC, muP;
                const R mu = mu_of(nd.mat, muPE, muC, muP);
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
                if (inter) { x = advance(x, w, s_int); pending = true; break; }
                x = xn;
                Y = rmax(Y - step * mu, (R)0);                                 // S_j update
                int ev = EV_BOUNDARY;
                if (vol < 0) { ev = EV_ESCAPE; alive = false; atomicAdd(&sh_cnt[ST_ESCAPED], 1ull); atomicAdd(&sh_en[EN_ESCAPED], (double)E); }
                else if (zs >= (uint32_t)g.stuck_limit) { ev = EV_STUCK; alive = false; atomicAdd(&sh_cnt[ST_STUCK], 1ull); atomicAdd(&sh_en[EN_STUCK], (double)E); }
                end_history(ev, vol_before);
                if (!alive) break;
                if ((nd.info & NODE_REGULAR) && direction_cacheable(w, g.delta)) break;      // voxel_pass takes over
            }
            needgen = alive && !pending && !((nd.info & NODE_REGULAR) && direction_cacheable(w, g.delta));
        }
        if (alive && pending) {
            const int mat = have_nd ? nd.mat : __ldg(&g.node[vol].mat);
            R muPE, muC, muP;
            const R mu = mu_of(mat, muPE, muC, muP);
            InteractIO<R> io;
            io.E = E; io.wx = w.x; io.wy = w.y; io.wz = w.z; io.Y = Y; io.gPE = gPE; io.gKN = gKN; io.L2k = L2k; io.j = ctr; io.above = above;
            interact(&io, muPE, muC, muP, mu, g.e_cut, seed, first_id + (sec.in ? sec.in[idx >> 1].idx : idx), sec.in ? 1u + (idx & 1u) : 0u, sec.out != nullptr);
            int ev = io.ev; ctr = io.j;
            if (ev == EV_PAIR && sec.out) { PairVtx<R> pv; pv.x = x.x; pv.y = x.y; pv.z = x.z; pv.idx = idx; sec.out[atomicAdd(sec.n_out, 1u)] = pv; }
            dep_d = (double)io.dep; dep_vol = vol; has_dep = true;
            alive = false;
            if (ev == EV_COMPTON || ev == EV_CUT) {
                E = io.E; w.x = io.wx; w.y = io.wy; w.z = io.wz;
                atomicAdd(&sh_cnt[ST_COMPTON], 1ull);
                if (ev == EV_CUT) atomicAdd(&sh_cnt[ST_CUT], 1ull);
                else { Y = io.Y; gPE = io.gPE; gKN = io.gKN; L2k = io.L2k; above = io.above; alive = true; }
            } else atomicAdd(&sh_cnt[ev == EV_PE ? ST_PE : ST_PAIR], 1ull);
            if (alive && (misc & 0xffu) >= (uint32_t)g.stuck_limit) {         // stuck guard (C9), after the step's event
                ev = EV_STUCK; alive = false;
                atomicAdd(&sh_cnt[ST_STUCK], 1ull); atomicAdd(&sh_en[EN_STUCK], (double)E);
            }
            end_history(ev, vol);
            pending = false;
            needgen = false;                                                  // voxel_pass looks at the volume and the new direction itself
        }
        if (TRACK && alive) pp.hash[idx] = h;
        if (c_steps) atomicAdd(&sh_cnt[ST_STEPS], (unsigned long long)c_steps);
        r.x = x.x; r.y = x.y; r.z = x.z; r.wx = w.x; r.wy = w.y; r.wz = w.z; r.E = E; r.Y = Y; r.gPE = gPE; r.gKN = gKN; r.L2k = L2k;
        r.vol = alive ? vol : -1; r.ctr = ctr; r.misc = misc;
        r.tail[0] = (uint32_t)above | (needgen ? REC_NEED_GENERAL : 0u);
        store_rec(q, cap - 1u - i, r);
    }
    warp_tally(edep, &sh_en[EN_DEPOSITED], dep_vol, dep_d, has_dep);
    __syncthreads();
    if (threadIdx.x < 8 && sh_cnt[threadIdx.x]) atomicAdd(&stats->cnt[threadIdx.x], sh_cnt[threadIdx.x]);
    if (threadIdx.x >= 8 && threadIdx.x < 12 && sh_en[threadIdx.x - 8] != 0.0) atomicAdd(&stats->en[threadIdx.x - 8], sh_en[threadIdx.x - 8]);
}

}  // namespace gn
