// kernels.cu -- navigation kernels, the wavefront transport kernel and the C entry points that launch them.
//
// transport_run design (B200-first; the paper's one-thread-runs-Algorithm-1-to-completion kernel, PAPER.md
// L143, and its CUDPP compaction experiment, L195, are the prior art):
//   * photon state lives in two queues in HBM, one 16-byte-aligned record per photon (64 B in fp32, 112 B in
//     fp64: position, direction, E, remaining optical depth Y, the three energy factors of mu, volume, photon
//     index, Philox draw counter, step counters), moved with 16-byte vector loads / stores;
//   * one wavefront pass = one launch of transport_pass: every thread loads one live photon, advances it by up
//     to K steps (Algorithm 1 loop body: mu, s_int, ComputeStep, move / interact) keeping the node record of the
//     current volume in registers, and survivors are compacted into the other queue with a ballot + block-
//     aggregated atomic cursor, partitioned by a 1-bit key (photon parked at an interaction point or not) to the
//     back / front of the queue; pass 0 generates the photons from the source and takes one step, so photons that miss
//     everything leave the warps at once;
//   * passes are chained on the device: a pass reads its input count from the counter its predecessor
//     incremented, so the host enqueues passes back to back and only looks at counts that are two passes old;
//     once few photons are left, one last pass runs them to completion;
//   * energy deposits are reduced across the warp per distinct volume (shuffle tree) before the fp64 atomic;
//   * rare physics (Philox rounds, Klein-Nishina sampling, energy factors in fp64) and bulky geometry (tube
//     distances, daughter scans, voxel walk) are out of line, one copy each, so that the hot navigation loop is
//     small in registers and instruction cache;
//   * solids, voxel-grid headers and material factors are staged in shared memory; node records and voxel
//     cells stay in L2.
#pragma once
#include <vector>
#include "common.cuh"
#include "impl.h"
#include "physics.cuh"

namespace gn {

// -------------------------------------------------------------------------------------------------------
// transport
// -------------------------------------------------------------------------------------------------------
#ifndef TR_THREADS_N
#define TR_THREADS_N 128          // threads per block of the transport kernels
#endif
constexpr int TR_THREADS = TR_THREADS_N;
constexpr int TR_WARPS = TR_THREADS / 32;
constexpr int TR_PER_128 = 128 / TR_THREADS;      // the min-blocks figures below are per 128 threads
#ifndef TR_MIN_BLOCKS
#define TR_MIN_BLOCKS 8          // general fp32 step pass: 64 registers, 32 warps / SM
#endif
#ifndef TR_MIN_BLOCKS_F64
#define TR_MIN_BLOCKS_F64 4      // fp64 step / source passes: 128 registers, 16 warps / SM (measured: +13 % on config 2 over 1 block's 162 registers)
#endif
#ifndef TR_MIN_BLOCKS_SRC
#define TR_MIN_BLOCKS_SRC 6      // source pass (birth + locate + first step)
#endif
#ifndef TR_MIN_BLOCKS_BOX
#define TR_MIN_BLOCKS_BOX 6      // box-only fp32 step pass: 80 registers (no spills), 24 warps / SM
#endif
constexpr int REFILL_BATCH = 8;       // empty lanes that trigger a warp's refill (persistent refill kernel)
constexpr int INTERACT_BATCH = 8;     // parked lanes that trigger a warp's interaction phase
#ifndef GENERAL_BATCH
#define GENERAL_BATCH 8            // box-only kernels: lanes waiting for the general ComputeStep that trigger it
#endif
enum : int { EV_BOUNDARY = 0, EV_PE = 1, EV_COMPTON = 2, EV_PAIR = 3, EV_CUT = 4, EV_ESCAPE = 5, EV_STUCK = 6, EV_RAYLEIGH = 7 };
enum : int { FATE_ALIVE = 0, FATE_ABSORBED = 1, FATE_ESCAPED = 2, FATE_STUCK = 3, FATE_NONE = 4 };
enum : int { ST_STEPS = 0, ST_COMPTON, ST_PE, ST_PAIR, ST_CUT, ST_ESCAPED, ST_STUCK, ST_PHOTONS, ST_RAYLEIGH, ST_COUNT };
enum : int { EN_ESCAPED = 0, EN_STUCK, EN_SOURCE, EN_DEPOSITED };

struct DevStats {
    unsigned long long cnt[16];      // ST_*
    unsigned long long lean_steps;   // steps taken inside the lean wavefront passes (the dominant kernel)
    double en[4];                    // EN_*
    unsigned long long dbg[8];       // GN_DEBUG_COUNTERS builds only: fast steps, bails, general phases, general lane-steps, iterations
};
#ifdef GN_DEBUG_COUNTERS
#define GN_DBG(i, v) atomicAdd(&stats->dbg[i], (unsigned long long)(v))
#else
#define GN_DBG(i, v) ((void)0)
#endif
// Checked builds (-DGN_CHECKED; compute-sanitizer is closed on the GPU pool): the invariants a memory checker would watch --
// every queue slot, node index and buffer index in range, the queue segments never overlapping -- are tested in the kernels;
// a violation sets bit `code` of stats->dbg[7] and gn_transport_run returns GN_CUDA_ERROR naming the bits.
#ifdef GN_CHECKED
#define GN_CHECK(cond, code) do { if (!(cond)) atomicOr(&stats->dbg[7], 1ull << (code)); } while (0)
#else
#define GN_CHECK(cond, code) ((void)0)
#endif
enum : int { CHK_LOAD_SLOT = 0, CHK_STORE_SLOT = 1, CHK_VOLUME = 2, CHK_SEGMENTS = 3, CHK_SLOW_SLOT = 4, CHK_PHOTON_INDEX = 5, CHK_PAIR_SLOT = 6, CHK_MATERIAL = 7 };
// survivors of a pass: key-0 photons fill the output queue from the front, key-1 photons from the back
struct PassCounters { unsigned front, back, slow, pad; };      // slow: photons flagged for the general step (voxel schedule: buffer S)
// general geometries: the travelling survivors of a pass are also counted by volume key, and a small kernel turns the
// keys into the work order of the next pass (sort_scatter_kernel), so that its warps are mostly of one kind
struct KeyCounters { unsigned long long tot[SORT_KEYS], cur[SORT_KEYS]; unsigned long long pad[2]; };
struct SortIO { KeyCounters* kout; uint8_t* keys_out; const uint32_t* perm_in; };

// one photon in the queue; sizeof = 64 (float) / 112 (double), moved as 16-byte words
template <class R> struct alignas(16) PhotonRec {
    R x, y, z, wx, wy, wz, E, Y, gPE, gKN, L2k;
    int32_t vol; uint32_t idx, ctr, misc;        // misc = zero_steps | nsteps << 8
    uint32_t tail[sizeof(R) == 4 ? 1 : 2];       // tail[0]: bit 0 = E above the pair threshold (k > 2), bit 1 = parked at an interaction point, bits 8.. = material of vol (written by the step passes for interact_pass); rest padding
};
static_assert(sizeof(PhotonRec<float>) == 64 && sizeof(PhotonRec<double>) == 112, "photon record layout");

template <class R> __device__ __forceinline__ void load_rec(const PhotonRec<R>* q, unsigned i, PhotonRec<R>& r) {
    const uint4* s = reinterpret_cast<const uint4*>(q + i);
    uint4* d = reinterpret_cast<uint4*>(&r);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(PhotonRec<R>) / 16); ++k) d[k] = __ldcs(s + k);      // streamed: read once
}
template <class R> __device__ __forceinline__ void store_rec(PhotonRec<R>* q, unsigned i, const PhotonRec<R>& r) {
    uint4* d = reinterpret_cast<uint4*>(q + i);
    const uint4* s = reinterpret_cast<const uint4*>(&r);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(PhotonRec<R>) / 16); ++k) __stcs(d + k, s[k]);
}

struct PerPhotonOut { uint64_t* hash; uint32_t* nsteps; double* efinal; };

// Secondary photons (reading 16).  A pair event of a primary appends its vertex to a list
// (out / n_out).  Annihilation photon k (k = 0, 1, ... over the whole list) belongs to pair k >> 1, runs on Philox stream
// tag 1 + (k & 1) of its parent's id, and adds its history hash and step count to the parent's (sums: the order in which
// they finish does not matter).  It travels through the same queues and kernels as the primaries -- a source pass with
// birth = 1 appends photons 2 birth_first ... to the queue of the pass that comes next -- and is told apart by SEC_BIT of
// its photon index: idx = SEC_BIT | k.
constexpr uint32_t SEC_BIT = 0x80000000u;
template <class R> struct alignas(16) PairVtx { R x, y, z; uint32_t idx; };
template <class R> struct SecIO {
    PairVtx<R>* out; unsigned* n_out;                          // where pair vertices go (nullptr = secondaries off)
    const PairVtx<R>* in;                                      // the list again, for the photons with SEC_BIT: their parents' vertices
    unsigned long long* parent_hash; uint32_t* parent_nsteps;  // per-photon outputs wanted: the parents' slots
    unsigned long long* state_hash;                            // hash state of annihilation photon k between passes (tracked runs)
    uint32_t birth_first; int birth;                           // source pass: birth = 1 -> it births photons 2 birth_first + i
};
template <class R> __host__ __device__ inline SecIO<R> no_secondaries() { SecIO<R> o; o.out = nullptr; o.n_out = nullptr; o.in = nullptr; o.parent_hash = nullptr; o.parent_nsteps = nullptr; o.state_hash = nullptr; o.birth_first = 0; o.birth = 0; return o; }
// id and Philox stream tag of photon idx; its hash state between passes
template <class R> __device__ __forceinline__ uint64_t photon_id(const SecIO<R>& sec, uint64_t first_id, uint32_t idx) {
    return first_id + ((idx & SEC_BIT) ? sec.in[(idx & ~SEC_BIT) >> 1].idx : idx);
}
__device__ __forceinline__ uint32_t photon_tag(uint32_t idx) { return (idx & SEC_BIT) ? 1u + (idx & 1u) : 0u; }
template <class R> __device__ __forceinline__ unsigned long long& hash_state(const PerPhotonOut& pp, const SecIO<R>& sec, uint32_t idx) {
    return (idx & SEC_BIT) ? sec.state_hash[idx & ~SEC_BIT] : *reinterpret_cast<unsigned long long*>(&pp.hash[idx]);
}
// per-photon outputs at the end of a history
template <class R> __device__ __forceinline__ void history_out(const PerPhotonOut& pp, const SecIO<R>& sec, uint32_t idx, uint64_t h, uint32_t ns, R E) {
    if (idx & SEC_BIT) {
        const uint32_t parent = sec.in[(idx & ~SEC_BIT) >> 1].idx;
        if (sec.parent_hash) atomicAdd(&sec.parent_hash[parent], (unsigned long long)h);
        if (sec.parent_nsteps) atomicAdd(&sec.parent_nsteps[parent], ns);
    } else {
        pp.hash[idx] = h; if (pp.nsteps) pp.nsteps[idx] = ns; if (pp.efinal) pp.efinal[idx] = (double)E;
    }
}

// history hash: FNV-1a-64, one 32-bit word = its four bytes, least significant first
__device__ __forceinline__ void fnv_word(uint64_t& h, uint32_t w) {
    const uint64_t prime = 0x100000001b3ull;
    h = (h ^ (uint64_t)(w & 0xffu)) * prime;
    h = (h ^ (uint64_t)((w >> 8) & 0xffu)) * prime;
    h = (h ^ (uint64_t)((w >> 16) & 0xffu)) * prime;
    h = (h ^ (uint64_t)(w >> 24)) * prime;
}

template <class T> __device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// warp-aggregated tally: one fp64 atomic per distinct volume per warp
static __device__ __noinline__ void warp_tally(double* __restrict__ edep, double* sh_dep_total, int vol, double dep, bool has) {
    const int lane = threadIdx.x & 31;
    {   // book-keeping total: one shared atomic per warp
        double tot = has ? dep : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
        if (lane == 0 && tot != 0.0) atomicAdd(sh_dep_total, tot);
    }
    // lanes whose volume no other lane of the warp deposits in add directly; the rest are summed per distinct volume
    const unsigned grp = __match_any_sync(0xffffffffu, has ? vol : ~lane);
    const bool alone = grp == (1u << lane);
    if (has && alone) atomicAdd(&edep[vol], dep);
    unsigned pending = __ballot_sync(0xffffffffu, has && !alone);
    while (pending) {
        int leader = __ffs(pending) - 1;
        int v = __shfl_sync(0xffffffffu, vol, leader);
        bool same = has && vol == v;
        unsigned g2 = __ballot_sync(0xffffffffu, same);
        double s = same ? dep : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == leader) atomicAdd(&edep[v], s);
        pending &= ~g2;
    }
}

// One interaction (C6 / C7), out of line: process choice, Klein-Nishina sampling, new direction, new energy
// factors, new optical depth.  State goes through a short-lived record so that the caller's registers never
// have their address taken.
template <class R> struct InteractIO {
    R E, wx, wy, wz, Y, gPE, gKN, L2k, dep;
    uint32_t j; int above, ev;
};
template <class R>
__device__ __noinline__ void interact(InteractIO<R>* io, R muPE, R muC, R muR, R muP, R mu, R e_cut, int pe_pd, uint64_t seed, uint64_t id, uint32_t tag, bool annihilate) {
    PhiloxStream rng; rng.init(seed, id, io->j, tag);
    R E = io->E;
    R t = draw<R>(rng) * mu;
    // cumulative thresholds PE | Compton | Rayleigh | pair; U = 1 falls to the last process with a non-zero coefficient (reading 2)
    const bool last_pair = muP > 0, last_rayleigh = !last_pair && muR > 0;
    if (t < muPE) { io->dep = E; io->ev = EV_PE; }
    else if (t < muPE + muC || (!last_pair && !last_rayleigh)) {
        R eps, cost, s2;
        kn_sample(E, rng, eps, cost, s2);
        R Ep = eps * E;
        R phi = (R)6.283185307179586 * draw<R>(rng);
        V3<R> w{io->wx, io->wy, io->wz};
        rotate_direction(w, cost, rsqrt_(rmax(s2, (R)0)), phi);
        io->wx = w.x; io->wy = w.y; io->wz = w.z;
        R dep = E - Ep;
        io->E = Ep; io->ev = EV_COMPTON;
        if (Ep < e_cut) { dep = dep + Ep; io->ev = EV_CUT; }
        else {
            EnergyFactors<R> ef = energy_factors(Ep, pe_pd);
            io->gPE = ef.gPE; io->gKN = ef.gKN; io->L2k = ef.L2k; io->above = ef.above_pair;
            io->Y = -rlog(draw<R>(rng));
        }
        io->dep = dep;
    } else if (t < (muPE + muC) + muR || last_rayleigh) {          // Rayleigh (reading 18): new direction, same energy, no deposit
        const R cost = rayleigh_sample<R>(rng);
        const R sint = rsqrt_(rmax(((R)1 - cost) * ((R)1 + cost), (R)0));
        R phi = (R)6.283185307179586 * draw<R>(rng);
        V3<R> w{io->wx, io->wy, io->wz};
        rotate_direction(w, cost, sint, phi);
        io->wx = w.x; io->wy = w.y; io->wz = w.z;
        io->Y = -rlog(draw<R>(rng));
        io->dep = 0; io->ev = EV_RAYLEIGH;
    } else { io->dep = annihilate ? E - (R)(2.0 * GN_ME_C2) : E; io->ev = EV_PAIR; }   // pair: all of E, or the pair's kinetic energy
    io->j = rng.j;
}

// photon birth (C8, Algorithm 1 steps 1-2), out of line: source sampling, energy factors, first optical depth
template <class R> struct BirthIO { R x, y, z, wx, wy, wz, E, Y, gPE, gKN, L2k; uint32_t j; int above; };
template <class R>
__device__ __forceinline__ void birth(BirthIO<R>* io, const SourceDev<R>* src, const EnergyFactors<R>* mono, int pe_pd, uint64_t seed, uint64_t id) {
    PhiloxStream rng; rng.init(seed, id, 0);
    V3<R> x, w; R E;
    sample_source(*src, rng, x, w, E);
    io->x = x.x; io->y = x.y; io->z = x.z; io->wx = w.x; io->wy = w.y; io->wz = w.z; io->E = E;
    io->Y = -rlog(draw<R>(rng));                       // Algorithm 1 steps 1-2
    // mono-energetic source: the factors of E0 were evaluated once per block (same function, same value)
    EnergyFactors<R> ef = mono ? *mono : energy_factors(E, pe_pd);
    io->gPE = ef.gPE; io->gKN = ef.gKN; io->L2k = ef.L2k; io->above = ef.above_pair;
    io->j = rng.j;
}

// birth of annihilation photon k (NEXT-3): isotropic direction from draws 0, 1 of stream tag 1 of the parent (cos theta =
// 1 - 2 u0, phi = 2 pi u1); photon 2 flies exactly the other way on stream tag 2; both have E = me c^2
template <class R>
__device__ __noinline__ void birth_secondary(BirthIO<R>* io, const PairVtx<R>* vtx, uint32_t k, int pe_pd, uint64_t seed, uint64_t first_id) {
    const PairVtx<R> pv = vtx[k >> 1];
    PhiloxStream rng; rng.init(seed, first_id + pv.idx, 0, 1);
    R u0 = draw<R>(rng), u1 = draw<R>(rng);
    R ct = (R)1 - (R)2 * u0;
    R st = rsqrt_(rmax(((R)1 - ct) * ((R)1 + ct), (R)0));
    R sp, cp; rsincos((R)6.283185307179586 * u1, &sp, &cp);
    R wx = st * cp, wy = st * sp, wz = ct;
    if (k & 1u) { wx = -wx; wy = -wy; wz = -wz; rng.init(seed, first_id + pv.idx, 0, 2); }
    io->x = pv.x; io->y = pv.y; io->z = pv.z; io->wx = wx; io->wy = wy; io->wz = wz; io->E = (R)GN_ME_C2;
    io->Y = -rlog(draw<R>(rng));
    EnergyFactors<R> ef = energy_factors(io->E, pe_pd);
    io->gPE = ef.gPE; io->gKN = ef.gKN; io->L2k = ef.L2k; io->above = ef.above_pair;
    io->j = rng.j;
}

// PHYS = false: the lean wavefront pass -- photons that reach an interaction point park there and are written to the
// back of the output queue; interact_pass handles them before the next pass.  PHYS = true: interactions happen inside
// the pass (batched per warp); used for the last pass, which runs the few remaining photons to completion.
template <class R, bool FROM_SOURCE, bool TRACK, bool PHYS, bool FLAT>
__global__ void __launch_bounds__(TR_THREADS, TR_PER_128 * (PHYS ? 1 : (sizeof(R) == 4 ? (FROM_SOURCE ? TR_MIN_BLOCKS_SRC : (FLAT ? TR_MIN_BLOCKS : TR_MIN_BLOCKS_BOX)) : TR_MIN_BLOCKS_F64)))
transport_pass(GeoView<R> g, SourceDev<R> src, uint64_t seed, uint64_t first_id, uint32_t n_src, const PassCounters* __restrict__ cin,
               PassCounters* __restrict__ cout, const PhotonRec<R>* __restrict__ qin, PhotonRec<R>* __restrict__ qout, uint32_t cap,
               double* __restrict__ edep, DevStats* __restrict__ stats, PerPhotonOut pp, int K, int regroup_pct, SortIO sio, SecIO<R> sec, int timed) {
    // input: pass 0 generates n_src photons; later passes read the survivors of the previous pass, whose count is
    // known only on the device (front + back of cin)
    unsigned n_front = n_src, n_in = n_src;
    if (!FROM_SOURCE) { n_front = cin->front; n_in = n_front + cin->back; }
    if (blockIdx.x * TR_THREADS >= n_in) return;

    __shared__ BlockTables<R> tab;
    __shared__ MatRec<R> sh_mats[MAX_SMEM_MATS];
    __shared__ SourceDev<R> sh_src;
    __shared__ EnergyFactors<R> sh_mono;
    __shared__ unsigned sh_wcount[2][TR_WARPS];
    __shared__ unsigned sh_base[2];
    __shared__ unsigned long long sh_cnt[ST_COUNT];
    __shared__ double sh_en[4];
    __shared__ unsigned sh_key[SORT_KEYS];
    if (threadIdx.x < SORT_KEYS) sh_key[threadIdx.x] = 0;
    stage_tables(g, tab);
    const MatRec<R>* mats = g.mats;
    if (g.n_mats <= MAX_SMEM_MATS) { for (int i = threadIdx.x; i < g.n_mats; i += blockDim.x) sh_mats[i] = g.mats[i]; mats = sh_mats; }
    if (FROM_SOURCE && threadIdx.x == 0) { sh_src = src; if (src.energy_kind == 0) sh_mono = energy_factors(src.e0, g.pe_per_decade); }
    if (threadIdx.x < ST_COUNT) sh_cnt[threadIdx.x] = 0;
    if (threadIdx.x < 4) sh_en[threadIdx.x] = 0.0;
    __syncthreads();
    Navigator<R, true, FLAT> nav(g, &tab.ctx);
    const unsigned i = blockIdx.x * TR_THREADS + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    int fate = i < n_in ? FATE_ALIVE : FATE_NONE;
    V3<R> x{0, 0, 0}, w{0, 0, 1}; R E = 1, Y = 0, gPE = 0, gKN = 0, L2k = 0;
    uint32_t idx = 0, misc = 0, ctr = 0; int above = 0;
    uint64_t h = 0xcbf29ce484222325ull;
    int vol = -1; NodeRec<R> nd = {};
    unsigned c_steps = 0;
    // events of this lane's photon inside the pass (tail pass only; a lane follows one photon): Compton scatters in bits 0-15,
    // Rayleigh scatters in 16-28, energy cut / photoelectric / pair (at most one each) in bits 29 / 30 / 31; summed per warp
    // at the end (a 64-bit shared-memory atomic per lane and event is a compare-and-swap loop under contention)
    unsigned c_ev = 0;
    bool pending = false;       // the photon sits at its interaction point, waiting for an interaction phase

    if (FROM_SOURCE) {
        unsigned c_phot = 0; double e_src = 0.0;
        if (fate == FATE_ALIVE) {
            BirthIO<R> b;
            if (sec.birth) { idx = SEC_BIT | (2u * sec.birth_first + i); birth_secondary(&b, sec.in, idx & ~SEC_BIT, g.pe_per_decade, seed, first_id); }
            else { idx = i; birth(&b, &sh_src, sh_src.energy_kind == 0 ? &sh_mono : nullptr, g.pe_per_decade, seed, first_id + i); }
            x.x = b.x; x.y = b.y; x.z = b.z; w.x = b.wx; w.y = b.wy; w.z = b.wz; E = b.E; Y = b.Y;
            gPE = b.gPE; gKN = b.gKN; L2k = b.L2k; above = b.above; ctr = b.j;
            if (!sec.birth) { c_phot = 1; e_src = (double)E; }            // annihilation photons are not source photons
            vol = nav.locate(x, w, nd);
            if (vol < 0) {
                fate = FATE_ESCAPED;
                if (TRACK) history_out(pp, sec, idx, h, 0u, E);
            }
        }
        c_phot = warp_sum(c_phot); e_src = warp_sum(e_src);
        if (lane == 0) { atomicAdd(&sh_cnt[ST_PHOTONS], (unsigned long long)c_phot); atomicAdd(&sh_en[EN_SOURCE], e_src); }
    } else if (fate == FATE_ALIVE) {
        const unsigned slot_in = i < n_front ? ((FLAT && sio.perm_in) ? sio.perm_in[i] : i) : cap - 1u - (i - n_front);
        GN_CHECK(slot_in < cap && n_in <= cap, CHK_LOAD_SLOT);
        PhotonRec<R> r; load_rec(qin, slot_in, r);
        GN_CHECK(r.vol < g.n_nodes && (r.vol < 0 || g.node[r.vol].mat < g.n_mats), CHK_VOLUME);
        if (r.vol < 0) fate = FATE_NONE;                 // absorbed by interact_pass
        x.x = r.x; x.y = r.y; x.z = r.z; w.x = r.wx; w.y = r.wy; w.z = r.wz; E = r.E; Y = r.Y;
        gPE = r.gPE; gKN = r.gKN; L2k = r.L2k; above = (int)(r.tail[0] & 1u); pending = (r.tail[0] & 2u) != 0;
        idx = r.idx; misc = r.misc; ctr = r.ctr; vol = r.vol;
        if (fate == FATE_ALIVE) { nd = nav.node(vol); if (TRACK) h = hash_state(pp, sec, idx); }
    }

    // A lane whose photon reaches its interaction point parks there (pending) instead of running the rare, long
    // physics alone with 31 lanes idle; the warp runs one interaction phase for all parked lanes once
    // INTERACT_BATCH of them wait, or when nothing else is left to do.  Photons still parked when the pass ends
    // are written to the BACK of the output queue (key = event type), so the next pass finds
    // them packed into full warps.
    auto finish_step = [&](int ev, int vol_before) {          // stuck guard (C9) + history hash; after the step's event
        if (fate == FATE_ALIVE && (misc & 0xffu) >= (uint32_t)g.stuck_limit) { ev = EV_STUCK; fate = FATE_STUCK; }
        if (TRACK) {
            fnv_word(h, (uint32_t)vol_before); fnv_word(h, (uint32_t)ev);
            if (fate != FATE_ALIVE) history_out(pp, sec, idx, h, misc >> 8, E);
        }
    };
    // what a ComputeStep does to the photon (Algorithm 1 loop body): (vol, nd) already hold the volume
    // after the boundary; inter = the interaction point s_int comes first (S_j >= Y inside vol_before)
    auto apply_step = [&](bool inter, R s_int, R step, const V3<R>& xn, R mu, int vol_before) {
        ++c_steps; misc += 0x100u;
        const R len = inter ? s_int : step;
        uint32_t zs = misc & 0xffu;
        zs = (len <= g.delta) ? min(zs + 1u, 255u) : 0u;                  // saturates: stuck_limit <= 255 is enforced at create time
        misc = (misc & ~0xffu) | zs;
        if (inter) {
            x = advance(x, w, s_int);
            pending = true;
        } else {                                                           // boundary: S_j update
            x = xn;
            Y = rmax(Y - step * mu, (R)0);
            int ev = EV_BOUNDARY;
            if (vol < 0) { ev = EV_ESCAPE; fate = FATE_ESCAPED; }
            finish_step(ev, vol_before);
        }
    };
    // Box-only kernels: photons inside regular voxels take regular_step (nav.cuh); whoever cannot (another kind of volume, an
    // exit through an edge or out of the mother, ...) waits for the general ComputeStep, which the warp runs once
    // GENERAL_BATCH lanes wait, when no lane could take the short step, or in the last iteration of the pass.
    constexpr bool FASTV = !FLAT;
    VoxLane<R> vl; vl.hx = vl.hy = vl.hz = 0; vl.r0 = vl.r1 = vl.r2 = 0; vl.solid = -1; vl.ok = false;
    if (FASTV && fate == FATE_ALIVE) lane_direction(w, g.delta, vl);
    bool bailed = false;                                                   // regular_step gave up on this photon's next step
    int act0 = 32;
#pragma unroll 1
    for (int k = 0;;) {
        const unsigned pen = PHYS ? __ballot_sync(0xffffffffu, pending) : 0u;
        const unsigned act = __ballot_sync(0xffffffffu, fate == FATE_ALIVE && !pending);
        const bool budget = k < K;
        if (PHYS && budget && pen && (act == 0 || __popc(pen) >= INTERACT_BATCH)) {
            // ---- interaction phase (A6-A9) ----------------------------------------------------------------------
            double dep_d = 0.0;
            if (pending) {
                const MuParts<R> mp = photon_mu(g, mats[nd.mat], nd.mat, E, gPE, gKN, L2k, above);
                InteractIO<R> io;
                io.E = E; io.wx = w.x; io.wy = w.y; io.wz = w.z; io.Y = Y; io.gPE = gPE; io.gKN = gKN; io.L2k = L2k; io.j = ctr; io.above = above;
                interact(&io, mp.pe, mp.c, mp.r, mp.p, mp.tot, g.e_cut, g.pe_per_decade, seed, photon_id(sec, first_id, idx), photon_tag(idx), sec.out != nullptr);
                const int ev = io.ev; ctr = io.j;
                if (ev == EV_PAIR && sec.out) { PairVtx<R> pv; pv.x = x.x; pv.y = x.y; pv.z = x.z; pv.idx = idx; sec.out[atomicAdd(sec.n_out, 1u)] = pv; }
                dep_d = (double)io.dep;
                if (ev == EV_RAYLEIGH) {
                    w.x = io.wx; w.y = io.wy; w.z = io.wz; Y = io.Y;
                    c_ev += 1u << 16;
                    if (((c_ev >> 16) & 0x1fffu) == 0x1fffu) { atomicAdd(&sh_cnt[ST_RAYLEIGH], 0x1fffull); c_ev &= ~(0x1fffu << 16); }      // field full: flush
                    if (FASTV) lane_direction(w, g.delta, vl);
                } else if (ev == EV_COMPTON || ev == EV_CUT) {
                    E = io.E; w.x = io.wx; w.y = io.wy; w.z = io.wz;
                    c_ev += 1u;
                    if ((c_ev & 0xffffu) == 0xffffu) { atomicAdd(&sh_cnt[ST_COMPTON], 0xffffull); c_ev &= ~0xffffu; }                        // field full: flush
                    if (ev == EV_CUT) { c_ev |= 1u << 29; fate = FATE_ABSORBED; }
                    else {
                        Y = io.Y; gPE = io.gPE; gKN = io.gKN; L2k = io.L2k; above = io.above;
                        if (FASTV) lane_direction(w, g.delta, vl);
                    }
                } else {
                    c_ev |= ev == EV_PE ? 1u << 30 : 1u << 31;
                    fate = FATE_ABSORBED;
                }
                finish_step(ev, vol);
            }
            warp_tally(edep, &sh_en[EN_DEPOSITED], vol, dep_d, pending);
            pending = false;
            continue;
        }
        if (act == 0 || !budget) break;
        // regroup early: once fewer than regroup_pct % of the lanes that entered the pass still travel, the warp stops
        // and lets the compaction refill it (only the lean passes; the tail pass has nobody to regroup with)
        if (!PHYS) {
            if (k == 0) act0 = __popc(act);
            else if (__popc(act) * 100 < act0 * regroup_pct) break;
        }
        ++k;
        bool todo = fate == FATE_ALIVE && !pending;                            // this lane wants a step
        R mu = 0;
        if (todo) mu = photon_mu(g, mats[nd.mat], nd.mat, E, gPE, gKN, L2k, above).tot;
        if (FASTV) {
            bool stepped = false;
            if (todo && !bailed && vl.ok && (nd.info & (NODE_REGULAR | NODE_SLAB))) {
                if ((nd.info & NODE_SOLID_MASK) != vl.solid) lane_solid(nav.solids, nd.info, vl);
                R step = 0; V3<R> xn{0, 0, 0};
                const int vol_before = vol;
                const int rc = regular_step<R, true>(g, nav.grids, nav.solids, x, w, vl, mu, Y, vol, nd, step, xn);
                if (rc == REG_BAIL) { bailed = true; GN_DBG(1, 1); }
                else {
                    GN_DBG(0, 1);
                    apply_step(rc == REG_INTERACT, step, step, xn, mu, vol_before);
                    stepped = true; todo = false;
                }
            }
            const unsigned waiting = __ballot_sync(0xffffffffu, todo);
            if (waiting && !(__popc(waiting) >= GENERAL_BATCH || !__any_sync(0xffffffffu, stepped) || k >= K)) todo = false;      // wait
        }
        if (lane == 0) GN_DBG(4, 1);
        if (todo) { GN_DBG(3, 1); }
        if (__any_sync(0xffffffffu, todo) && lane == 0) GN_DBG(2, 1);
        if (todo) {
            const R s_int = mu > 0 ? rdiv(Y, mu) : rinf<R>();                  // remaining part of Eq. 7
            const int vol_before = vol;
            R step; V3<R> xn;
            nav.compute_step(vol, nd, x, w, s_int, step, xn);                  // "next intersection"
            apply_step(step == rinf<R>(), s_int, step, xn, mu, vol_before);
            bailed = false;
        }
    }

    // ---- compaction of survivors into the other queue, partitioned by key -------------------
    const bool alive = fate == FATE_ALIVE;
    const bool key1 = alive && pending;
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
        unsigned o = key1 ? cap - 1u - (sh_base[1] + sh_wcount[1][warp] + __popc(bal1 & below))
                          : sh_base[0] + sh_wcount[0][warp] + __popc(bal0 & below);
        PhotonRec<R> r;
        r.x = x.x; r.y = x.y; r.z = x.z; r.wx = w.x; r.wy = w.y; r.wz = w.z; r.E = E; r.Y = Y;
        r.gPE = gPE; r.gKN = gKN; r.L2k = L2k; r.vol = vol; r.idx = idx; r.ctr = ctr; r.misc = misc;
#pragma unroll
        for (int q = 0; q < (int)(sizeof(r.tail) / 4); ++q) r.tail[q] = 0;
        r.tail[0] = (uint32_t)above | (pending ? 2u : 0u) | ((uint32_t)nd.mat << 8);      // material of vol: interact_pass needs no node load
        GN_CHECK(o < cap && vol >= 0 && vol < g.n_nodes, CHK_STORE_SLOT);
        store_rec(qout, o, r);
        if (TRACK) hash_state(pp, sec, idx) = h;
        if (FLAT && sio.keys_out && !key1) {                                 // volume key of a travelling survivor
            const int key = 2 * nav.solid_of(nd).type + (nd.ndau > 0 ? 1 : 0);
            sio.keys_out[o] = (uint8_t)key;
            atomicAdd(&sh_key[key], 1u);
        }
    }
    // ---- statistics: warp tree, shared atomics, one global atomic per counter per block -----------------------
    {
        unsigned s = warp_sum(c_steps);
        unsigned ne = warp_sum(fate == FATE_ESCAPED ? 1u : 0u), ns = warp_sum(fate == FATE_STUCK ? 1u : 0u);
        double ee = warp_sum(fate == FATE_ESCAPED ? (double)E : 0.0);
        if (lane == 0) {
            if (s) atomicAdd(&sh_cnt[ST_STEPS], (unsigned long long)s);
            if (ne) { atomicAdd(&sh_cnt[ST_ESCAPED], (unsigned long long)ne); atomicAdd(&sh_en[EN_ESCAPED], ee); }
        }
        if (ns) {                                                           // warp-uniform, rare
            double es = warp_sum(fate == FATE_STUCK ? (double)E : 0.0);
            if (lane == 0) { atomicAdd(&sh_cnt[ST_STUCK], (unsigned long long)ns); atomicAdd(&sh_en[EN_STUCK], es); }
        }
        if (PHYS) {
            const unsigned nc = warp_sum(c_ev & 0xffffu), nr = warp_sum((c_ev >> 16) & 0x1fffu), nx = warp_sum((c_ev >> 29) & 1u),
                           ne = warp_sum((c_ev >> 30) & 1u), np = warp_sum(c_ev >> 31);
            if (lane == 0) {
                if (nc) atomicAdd(&sh_cnt[ST_COMPTON], (unsigned long long)nc);
                if (nr) atomicAdd(&sh_cnt[ST_RAYLEIGH], (unsigned long long)nr);
                if (nx) atomicAdd(&sh_cnt[ST_CUT], (unsigned long long)nx);
                if (ne) atomicAdd(&sh_cnt[ST_PE], (unsigned long long)ne);
                if (np) atomicAdd(&sh_cnt[ST_PAIR], (unsigned long long)np);
            }
        }
    }
    __syncthreads();
    GN_CHECK(cout->front + cout->back <= cap, CHK_SEGMENTS);
    if (threadIdx.x < ST_COUNT && sh_cnt[threadIdx.x]) atomicAdd(&stats->cnt[threadIdx.x], sh_cnt[threadIdx.x]);
    if (threadIdx.x >= 16 && threadIdx.x < 20 && sh_en[threadIdx.x - 16] != 0.0) atomicAdd(&stats->en[threadIdx.x - 16], sh_en[threadIdx.x - 16]);
    if (!FROM_SOURCE && !PHYS && timed && threadIdx.x == 12 && sh_cnt[ST_STEPS]) atomicAdd(&stats->lean_steps, sh_cnt[ST_STEPS]);
    if (FLAT && sio.kout && threadIdx.x >= 32 && threadIdx.x < 32 + SORT_KEYS && sh_key[threadIdx.x - 32]) atomicAdd(&sio.kout->tot[threadIdx.x - 32], (unsigned long long)sh_key[threadIdx.x - 32]);
}

// The interaction wavefront (A6-A9): every photon parked at an interaction point by the previous pass sits in the
// back segment of the queue (slots cap-1, cap-2, ...); one thread per photon samples the process, updates the record
// in place (absorbed photons are marked vol = -1) and the warp tallies the deposits.
#ifndef INTERACT_THREADS
#define INTERACT_THREADS TR_THREADS     // threads per block of interact_pass (a block waits for its slowest warp)
#endif
#ifndef INTERACT_MIN_BLOCKS
#define INTERACT_MIN_BLOCKS 6      // 80 registers, 24 warps / SM (1 block: 82 registers -- the same code, but the occupancy is then promised)
#endif
#ifndef INTERACT_MIN_BLOCKS_F64
#define INTERACT_MIN_BLOCKS_F64 3
#endif
template <class R, bool TRACK>
__global__ void __launch_bounds__(INTERACT_THREADS, ((sizeof(R) == 4 ? INTERACT_MIN_BLOCKS : INTERACT_MIN_BLOCKS_F64) * TR_THREADS + INTERACT_THREADS - 1) / INTERACT_THREADS)
interact_pass(GeoView<R> g, uint64_t seed, uint64_t first_id, const PassCounters* __restrict__ cin, PhotonRec<R>* __restrict__ q, uint32_t cap,
              double* __restrict__ edep, DevStats* __restrict__ stats, PerPhotonOut pp, SecIO<R> sec) {
    const unsigned n = cin->back;
    if (blockIdx.x * INTERACT_THREADS >= n) return;
    __shared__ unsigned sh_cnt[ST_COUNT];            // a block counts at most TR_THREADS events: 32-bit shared atomics are single instructions,
    __shared__ double sh_en[4];                      // 64-bit ones compare-and-swap loops (5 % of this kernel's stall samples, profiles/r2_final.md)
    if (threadIdx.x < ST_COUNT) sh_cnt[threadIdx.x] = 0;
    if (threadIdx.x < 4) sh_en[threadIdx.x] = 0.0;
    __syncthreads();
    const unsigned i = blockIdx.x * INTERACT_THREADS + threadIdx.x;
    const bool active = i < n;
    double dep_d = 0.0; int vol = 0, ev_done = -1;
    if (active) {
        GN_CHECK(n <= cap, CHK_LOAD_SLOT);
        PhotonRec<R> r; load_rec(q, cap - 1u - i, r);
        vol = r.vol;
        GN_CHECK(vol >= 0 && vol < g.n_nodes && (int)(r.tail[0] >> 8) == g.node[vol].mat, CHK_VOLUME);
        const int above = (int)(r.tail[0] & 1u);
        const int mat = (int)(r.tail[0] >> 8);                                 // written with the record by the pass that parked the photon
        const MuParts<R> mp = photon_mu(g, g.mats[mat], mat, r.E, r.gPE, r.gKN, r.L2k, above);
        InteractIO<R> io;
        io.E = r.E; io.wx = r.wx; io.wy = r.wy; io.wz = r.wz; io.Y = r.Y; io.gPE = r.gPE; io.gKN = r.gKN; io.L2k = r.L2k; io.j = r.ctr; io.above = above;
        interact(&io, mp.pe, mp.c, mp.r, mp.p, mp.tot, g.e_cut, g.pe_per_decade, seed, photon_id(sec, first_id, r.idx), photon_tag(r.idx), sec.out != nullptr);
        int ev = io.ev;
        if (ev == EV_PAIR && sec.out) { PairVtx<R> pv; pv.x = r.x; pv.y = r.y; pv.z = r.z; pv.idx = r.idx; const unsigned ps = atomicAdd(sec.n_out, 1u); GN_CHECK(ps < cap, CHK_PAIR_SLOT); sec.out[ps] = pv; }
        dep_d = (double)io.dep;
        bool alive = false;
        ev_done = ev;                                                          // counted per warp below
        if (ev == EV_RAYLEIGH) {
            r.wx = io.wx; r.wy = io.wy; r.wz = io.wz; r.Y = io.Y; alive = true;
        } else if (ev == EV_COMPTON || ev == EV_CUT) {
            r.E = io.E; r.wx = io.wx; r.wy = io.wy; r.wz = io.wz;
            if (ev != EV_CUT) { r.Y = io.Y; r.gPE = io.gPE; r.gKN = io.gKN; r.L2k = io.L2k; r.tail[0] = (uint32_t)io.above; alive = true; }
        }
        r.ctr = io.j;
        if (alive && (r.misc & 0xffu) >= (uint32_t)g.stuck_limit) {           // stuck guard (C9), after the step's event
            ev = EV_STUCK; alive = false;
            atomicAdd(&sh_cnt[ST_STUCK], 1u); atomicAdd(&sh_en[EN_STUCK], (double)r.E);
        }
        if (TRACK) {
            uint64_t h = hash_state(pp, sec, r.idx);
            fnv_word(h, (uint32_t)vol); fnv_word(h, (uint32_t)ev);
            if (alive) hash_state(pp, sec, r.idx) = h;
            else history_out(pp, sec, r.idx, h, r.misc >> 8, r.E);
        }
        if (alive) r.tail[0] &= 1u; else r.vol = -1;
        store_rec(q, cap - 1u - i, r);
    }
    {   // event counters: one ballot per kind of event, one shared atomic per warp and counter that is not zero
        const unsigned nC = __popc(__ballot_sync(0xffffffffu, ev_done == EV_COMPTON || ev_done == EV_CUT)), nX = __popc(__ballot_sync(0xffffffffu, ev_done == EV_CUT));
        const unsigned nE = __popc(__ballot_sync(0xffffffffu, ev_done == EV_PE)), nP = __popc(__ballot_sync(0xffffffffu, ev_done == EV_PAIR));
        const unsigned nR = __popc(__ballot_sync(0xffffffffu, ev_done == EV_RAYLEIGH));
        if ((threadIdx.x & 31) == 0) {
            if (nC) atomicAdd(&sh_cnt[ST_COMPTON], nC);
            if (nX) atomicAdd(&sh_cnt[ST_CUT], nX);
            if (nE) atomicAdd(&sh_cnt[ST_PE], nE);
            if (nP) atomicAdd(&sh_cnt[ST_PAIR], nP);
            if (nR) atomicAdd(&sh_cnt[ST_RAYLEIGH], nR);
        }
    }
    warp_tally(edep, &sh_en[EN_DEPOSITED], vol, dep_d, active);
    __syncthreads();
    if (threadIdx.x < ST_COUNT && sh_cnt[threadIdx.x]) atomicAdd(&stats->cnt[threadIdx.x], (unsigned long long)sh_cnt[threadIdx.x]);
    if (threadIdx.x >= 16 && threadIdx.x < 20 && sh_en[threadIdx.x - 16] != 0.0) atomicAdd(&stats->en[threadIdx.x - 16], sh_en[threadIdx.x - 16]);
}

// The paper's own remedy for threads whose particle has finished (stream compaction "and filling the empty places
// with new particles ... some speedup"), as a persistent kernel (gn_opts.refill): every lane follows
// its photon to the end (interactions batched per warp, as in the tail pass), and a lane whose photon is gone takes the next photon id from a device
// counter (one warp-aggregated atomic per refill) until the batch is used up.  Same arithmetic per photon as the
// wavefront passes -- Philox streams are keyed by photon id, so which lane follows which photon changes nothing.
template <class R, bool TRACK, bool FLAT>
__global__ void __launch_bounds__(TR_THREADS)
transport_refill(GeoView<R> g, SourceDev<R> src, uint64_t seed, uint64_t first_id, uint32_t n_src, unsigned* __restrict__ next,
                 double* __restrict__ edep, DevStats* __restrict__ stats, PerPhotonOut pp) {
    __shared__ BlockTables<R> tab;
    __shared__ MatRec<R> sh_mats[MAX_SMEM_MATS];
    __shared__ SourceDev<R> sh_src;
    __shared__ EnergyFactors<R> sh_mono;
    __shared__ unsigned long long sh_cnt[ST_COUNT];
    __shared__ double sh_en[4];
    stage_tables(g, tab);
    const MatRec<R>* mats = g.mats;
    if (g.n_mats <= MAX_SMEM_MATS) { for (int i = threadIdx.x; i < g.n_mats; i += blockDim.x) sh_mats[i] = g.mats[i]; mats = sh_mats; }
    if (threadIdx.x == 0) { sh_src = src; if (src.energy_kind == 0) sh_mono = energy_factors(src.e0, g.pe_per_decade); }
    if (threadIdx.x < ST_COUNT) sh_cnt[threadIdx.x] = 0;
    if (threadIdx.x < 4) sh_en[threadIdx.x] = 0.0;
    __syncthreads();
    Navigator<R, true, FLAT> nav(g, &tab.ctx);
    const int lane = threadIdx.x & 31;
    const SecIO<R> nosec = no_secondaries<R>();

    bool alive = false, exhausted = false, pending = false;      // pending: parked at its interaction point
    V3<R> x{0, 0, 0}, w{0, 0, 1}; R E = 1, Y = 0, gPE = 0, gKN = 0, L2k = 0;
    uint32_t idx = 0, misc = 0, ctr = 0; int above = 0;
    uint64_t h = 0;
    int vol = -1; NodeRec<R> nd = {};
    unsigned c_steps = 0, c_phot = 0, c_esc = 0, c_stuck = 0, c_compton = 0, c_pe = 0, c_pair = 0, c_cut = 0, c_ray = 0;
    double e_src = 0.0, e_esc = 0.0, e_stuck = 0.0;
#pragma unroll 1
    for (;;) {
        // ---- refill: lanes without a photon take the next ids ---------------------------------------------------
        // (batched like the interactions: birth + locate of a few lanes stalls the rest of the warp)
        const unsigned want = __ballot_sync(0xffffffffu, !alive && !exhausted);
        if (want && (FLAT || __popc(want) >= REFILL_BATCH || !__any_sync(0xffffffffu, alive))) {      // general geometries: warps are thin anyway, refill at once
            const int leader = __ffs(want) - 1;
            unsigned base = 0;
            if (lane == leader) base = atomicAdd(next, (unsigned)__popc(want));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (!alive && !exhausted) {
                const unsigned i = base + __popc(want & ((1u << lane) - 1u));
                if (i >= n_src || base >= n_src) exhausted = true;
                else {
                    idx = i; misc = 0; h = 0xcbf29ce484222325ull;
                    BirthIO<R> b;
                    birth(&b, &sh_src, sh_src.energy_kind == 0 ? &sh_mono : nullptr, g.pe_per_decade, seed, first_id + i);
                    x.x = b.x; x.y = b.y; x.z = b.z; w.x = b.wx; w.y = b.wy; w.z = b.wz; E = b.E; Y = b.Y;
                    gPE = b.gPE; gKN = b.gKN; L2k = b.L2k; above = b.above; ctr = b.j;
                    ++c_phot; e_src += (double)E;
                    vol = nav.locate(x, w, nd);
                    if (vol < 0) { ++c_esc; e_esc += (double)E; if (TRACK) history_out(pp, nosec, idx, h, 0u, E); }
                    else alive = true;
                }
            }
        }
        if (!__any_sync(0xffffffffu, alive || !exhausted)) break;
        // ---- interaction phase (A6-A9): lanes parked at their interaction points, batched per warp as in the tail pass ----
        const unsigned pen = __ballot_sync(0xffffffffu, alive && pending);
        const unsigned act = __ballot_sync(0xffffffffu, alive && !pending);
        if (pen && (act == 0 || __popc(pen) >= INTERACT_BATCH)) {
            double dep_d = 0.0;
            const bool was = alive && pending;
            if (was) {
                const MuParts<R> mp = photon_mu(g, mats[nd.mat], nd.mat, E, gPE, gKN, L2k, above);
                InteractIO<R> io;
                io.E = E; io.wx = w.x; io.wy = w.y; io.wz = w.z; io.Y = Y; io.gPE = gPE; io.gKN = gKN; io.L2k = L2k; io.j = ctr; io.above = above;
                interact(&io, mp.pe, mp.c, mp.r, mp.p, mp.tot, g.e_cut, g.pe_per_decade, seed, first_id + idx, 0u, false);
                int ev = io.ev; ctr = io.j;
                dep_d = (double)io.dep;
                if (ev == EV_RAYLEIGH) { w.x = io.wx; w.y = io.wy; w.z = io.wz; Y = io.Y; ++c_ray; }
                else if (ev == EV_COMPTON || ev == EV_CUT) {
                    E = io.E; w.x = io.wx; w.y = io.wy; w.z = io.wz;
                    ++c_compton;
                    if (ev == EV_CUT) { ++c_cut; alive = false; }
                    else { Y = io.Y; gPE = io.gPE; gKN = io.gKN; L2k = io.L2k; above = io.above; }
                } else {
                    if (ev == EV_PE) ++c_pe; else ++c_pair;
                    alive = false;
                }
                if (alive && (misc & 0xffu) >= (uint32_t)g.stuck_limit) { ev = EV_STUCK; alive = false; ++c_stuck; e_stuck += (double)E; }
                if (TRACK) {
                    fnv_word(h, (uint32_t)vol); fnv_word(h, (uint32_t)ev);
                    if (!alive) history_out(pp, nosec, idx, h, misc >> 8, E);
                }
                pending = false;
            }
            warp_tally(edep, &sh_en[EN_DEPOSITED], vol, dep_d, was);
            continue;
        }
        // ---- one navigation step (A1-A5) for every travelling lane ----------------------------------------------------
        if (alive && !pending) {
            const R mu = photon_mu(g, mats[nd.mat], nd.mat, E, gPE, gKN, L2k, above).tot;
            const R s_int = mu > 0 ? rdiv(Y, mu) : rinf<R>();
            const int vol_before = vol;
            R step; V3<R> xn;
            nav.compute_step(vol, nd, x, w, s_int, step, xn);
            ++c_steps; misc += 0x100u;
            const bool inter = step == rinf<R>();
            const R len = inter ? s_int : step;
            uint32_t zs = misc & 0xffu;
            zs = (len <= g.delta) ? min(zs + 1u, 255u) : 0u;                  // saturates: stuck_limit <= 255 is enforced at create time
            misc = (misc & ~0xffu) | zs;
            if (inter) {
                x = advance(x, w, s_int);
                pending = true;
            } else {
                x = xn;
                Y = rmax(Y - step * mu, (R)0);
                int ev = EV_BOUNDARY;
                if (vol < 0) { ev = EV_ESCAPE; alive = false; ++c_esc; e_esc += (double)E; }
                if (alive && (misc & 0xffu) >= (uint32_t)g.stuck_limit) { ev = EV_STUCK; alive = false; ++c_stuck; e_stuck += (double)E; }
                if (TRACK) {
                    fnv_word(h, (uint32_t)vol_before); fnv_word(h, (uint32_t)ev);
                    if (!alive) history_out(pp, nosec, idx, h, misc >> 8, E);
                }
            }
        }
    }
    // ---- statistics -----------------------------------------------------------------------------------------------
    {
        const unsigned v[ST_COUNT] = {c_steps, c_compton, c_pe, c_pair, c_cut, c_esc, c_stuck, c_phot, c_ray};      // ST_* order
#pragma unroll
        for (int q = 0; q < ST_COUNT; ++q) { unsigned t = warp_sum(v[q]); if (lane == 0 && t) atomicAdd(&sh_cnt[q], (unsigned long long)t); }
        double a = warp_sum(e_esc), b2 = warp_sum(e_stuck), c2 = warp_sum(e_src);
        if (lane == 0) { if (a != 0.0) atomicAdd(&sh_en[EN_ESCAPED], a); if (b2 != 0.0) atomicAdd(&sh_en[EN_STUCK], b2); if (c2 != 0.0) atomicAdd(&sh_en[EN_SOURCE], c2); }
    }
    __syncthreads();
    if (threadIdx.x < ST_COUNT && sh_cnt[threadIdx.x]) atomicAdd(&stats->cnt[threadIdx.x], sh_cnt[threadIdx.x]);
    if (threadIdx.x >= 16 && threadIdx.x < 20 && sh_en[threadIdx.x - 16] != 0.0) atomicAdd(&stats->en[threadIdx.x - 16], sh_en[threadIdx.x - 16]);
}

}  // namespace gn
#include "voxel_pass.cuh"
namespace gn {

constexpr int64_t TR_BATCH = 1ll << 24;     // photons per batch (bounds scratch at 2 x 16.8 M x 64 B = 2.1 GB in fp32)
constexpr int TR_MAX_PASSES = 4096;         // device counters per batch; the last one always runs to completion
constexpr int TR_LAG = 2;                   // the host looks at survivor counts that are this many passes old
constexpr int K_UNLIMITED = 0x7fffffff;
constexpr int TR_TIMED = GN_TIMED_PASSES;   // lean step passes per batch timed one by one (CUDA events around the launch)

template <class R, bool SRC, bool PHYS, bool FLAT>
static void launch_pass(bool track, unsigned blocks, cudaStream_t s, const GeoView<R>& g, const SourceDev<R>& src, uint64_t seed, uint64_t first_id,
                        uint32_t n_src, const PassCounters* cin, PassCounters* cout, const PhotonRec<R>* qin, PhotonRec<R>* qout, uint32_t cap,
                        double* edep, DevStats* stats, PerPhotonOut pp, int K, int regroup_pct, SecIO<R> sec, SortIO sio = SortIO{nullptr, nullptr, nullptr},
                        int timed = 0) {
    if (track) transport_pass<R, SRC, true, PHYS, FLAT><<<blocks, TR_THREADS, 0, s>>>(g, src, seed, first_id, n_src, cin, cout, qin, qout, cap, edep, stats, pp, K, regroup_pct, sio, sec, timed);
    else transport_pass<R, SRC, false, PHYS, FLAT><<<blocks, TR_THREADS, 0, s>>>(g, src, seed, first_id, n_src, cin, cout, qin, qout, cap, edep, stats, pp, K, regroup_pct, sio, sec, timed);
}
template <class R>
static void launch_interact(bool track, unsigned blocks, cudaStream_t s, const GeoView<R>& g, uint64_t seed, uint64_t first_id, const PassCounters* cin,
                            PhotonRec<R>* q, uint32_t cap, double* edep, DevStats* stats, PerPhotonOut pp, SecIO<R> sec) {
    const unsigned ib = (unsigned)(((uint64_t)blocks * TR_THREADS + INTERACT_THREADS - 1) / INTERACT_THREADS);
    if (track) interact_pass<R, true><<<ib, INTERACT_THREADS, 0, s>>>(g, seed, first_id, cin, q, cap, edep, stats, pp, sec);
    else interact_pass<R, false><<<ib, INTERACT_THREADS, 0, s>>>(g, seed, first_id, cin, q, cap, edep, stats, pp, sec);
}

template <class R, bool FLAT>
int transport_impl(const gn_geometry* geo, const SourceDev<R>& src, uint64_t seed, int64_t first_id, int64_t n_photons,
                   double* d_edep, gn_run_stats* h_stats, uint64_t* d_hash, uint32_t* d_nsteps, double* d_efinal, cudaStream_t s) {
    const bool track = d_hash || d_nsteps || d_efinal;
    const int K = geo->opts.steps_per_pass;
    const int K0 = std::min(K, geo->opts.first_pass_steps);      // first pass: short, sheds photons that miss
    const bool secondaries = geo->opts.secondaries > 0;        // NEXT-3: pair events leave two annihilation photons
    const bool refill = geo->opts.refill > 0;                  // NEXT-4: persistent kernel, finished lanes take fresh photons
    if (refill && secondaries) return fail(GN_INVALID_ARGUMENT, "gn_transport_run: gn_opts.refill and gn_opts.secondaries cannot be combined");
    const size_t cap = (size_t)std::min<int64_t>(std::max<int64_t>(n_photons, 2), TR_BATCH);
    const size_t qb = cap * sizeof(PhotonRec<R>);
    const size_t hb = (track && !d_hash) ? cap * 8 : 0;       // the hash array doubles as per-photon state between passes
    const size_t cb = sizeof(PassCounters) * (TR_MAX_PASSES + 2);
    const bool sorted = FLAT;                                  // general geometries: work order of every pass sorted by volume key
    const size_t kb = sorted ? sizeof(KeyCounters) * (TR_MAX_PASSES + 2) : 0;
    const size_t sb = sorted ? ((cap + 255) & ~(size_t)255) + 4 * cap : 0;      // keys + perm
    const size_t pb = secondaries ? cap * sizeof(PairVtx<R>) + 16 : 0;          // pair vertices of a batch + their count
    const size_t hb2 = (secondaries && track) ? 2 * cap * 8 : 0;                // hash state of the annihilation photons (two per pair vertex)
    const size_t base = (2 * qb + hb + 512 + cb + kb + sb + 15) & ~(size_t)15;
    bool voxel_sched = false;
    if constexpr (!FLAT) voxel_sched = geo->voxel_sched;
    const size_t vb = voxel_sched ? qb : 0;                    // buffer S of the voxel schedule: photons flagged for the general step
    const size_t need = base + pb + hb2 + vb + 16;
    std::lock_guard<std::mutex> lock(geo->ws_mutex);          // one run at a time per handle: the workspace is shared
    GN_CUDA(cudaMemsetAsync(d_edep, 0, sizeof(double) * (size_t)geo->n_places, s), "gn_transport_run memset edep");
    if (geo->ws_bytes < need) {
        if (geo->ws_scratch) { cudaStreamSynchronize(s); cudaFree(geo->ws_scratch); geo->ws_scratch = nullptr; geo->ws_bytes = 0; }
        cudaError_t e = cudaMalloc((void**)&geo->ws_scratch, need);
        if (e != cudaSuccess) { cudaGetLastError(); geo->ws_scratch = nullptr; return fail(GN_OUT_OF_MEMORY, std::string("gn_transport_run scratch: ") + cudaGetErrorString(e)); }
        geo->ws_bytes = need;
    }
    const size_t npb = sizeof(unsigned) * (TR_MAX_PASSES + 2);     // pinned: the pair count seen after every pass
    if (!geo->ws_pinned && cudaMallocHost(&geo->ws_pinned, cb + npb) != cudaSuccess) { cudaGetLastError(); geo->ws_pinned = nullptr; return fail(GN_OUT_OF_MEMORY, "gn_transport_run: pinned alloc"); }
    if (!geo->ws_events_ok) {
        bool ok = cudaEventCreate(&geo->ws_events[0]) == cudaSuccess && cudaEventCreate(&geo->ws_events[1]) == cudaSuccess;
        for (int q = 0; q <= TR_LAG; ++q) ok = ok && cudaEventCreateWithFlags(&geo->ws_events[2 + q], cudaEventDisableTiming) == cudaSuccess;
        for (int q = 0; q < 2 * TR_TIMED; ++q) ok = ok && cudaEventCreate(&geo->ws_events[8 + q]) == cudaSuccess;
        if (!ok) { cudaGetLastError(); return fail(GN_CUDA_ERROR, "gn_transport_run: event create"); }
        geo->ws_events_ok = true;
    }
    char* scratch = geo->ws_scratch;
    PhotonRec<R>* qa = (PhotonRec<R>*)scratch; PhotonRec<R>* qb_ = (PhotonRec<R>*)(scratch + qb);
    uint64_t* tmp_hash = hb ? (uint64_t*)(scratch + 2 * qb) : nullptr;
    DevStats* d_stats = (DevStats*)(scratch + 2 * qb + hb);
    PassCounters* d_ctr = (PassCounters*)(scratch + 2 * qb + hb + 512);
    PassCounters* h_ctr = (PassCounters*)geo->ws_pinned;
    unsigned* h_np = (unsigned*)((char*)geo->ws_pinned + cb);
    KeyCounters* d_kctr = sorted ? (KeyCounters*)(scratch + 2 * qb + hb + 512 + cb) : nullptr;
    uint8_t* d_keys = sorted ? (uint8_t*)(scratch + 2 * qb + hb + 512 + cb + kb) : nullptr;
    uint32_t* d_perm = sorted ? (uint32_t*)(scratch + 2 * qb + hb + 512 + cb + kb + ((cap + 255) & ~(size_t)255)) : nullptr;
    unsigned* d_npairs = secondaries ? (unsigned*)(scratch + base) : nullptr;
    PairVtx<R>* d_pairs = secondaries ? (PairVtx<R>*)(scratch + base + 16) : nullptr;
    uint64_t* sec_hash = hb2 ? (uint64_t*)(scratch + base + pb) : nullptr;
    PhotonRec<R>* d_slow = vb ? (PhotonRec<R>*)(scratch + ((base + pb + hb2 + 15) & ~(size_t)15)) : nullptr;
    int rc = GN_OK;
    uint64_t passes = 0, launches = 0;
    cudaEvent_t ev0 = geo->ws_events[0], ev1 = geo->ws_events[1];
    cudaEvent_t* ring = &geo->ws_events[2];
    double kernel_ms = 0.0, step_pass_ms = 0.0;
    cudaEvent_t* tev = &geo->ws_events[8];
    cudaError_t e = cudaSuccess;
    const unsigned tail = (unsigned)geo->opts.tail_photons;
    const int regroup = geo->opts.regroup_percent;
    cudaMemsetAsync(d_stats, 0, 512, s);
    const GeoView<R>& g = view<R>(geo);
    // one batch of photons through the wavefront: n0 photons born in pass 0 (from the source, or -- sec.in -- at their
    // parents' pair vertices), passes until none is left; ends with a stream synchronise
    // `sec.birth`: a batch of annihilation photons (pair vertices sec.birth_first ...); otherwise a batch of primaries, into
    // whose queue the annihilation photons of the pair events seen so far are injected between passes (`injected` counts the
    // pair vertices used up): they then ride the primaries' passes and share their tail instead of paying their own.
    unsigned injected = 0;
    auto run_batch = [&](uint32_t n0, uint64_t fid, PerPhotonOut pp, SecIO<R> sec) {
        PhotonRec<R>* in = qb_; PhotonRec<R>* out = qa;
        const bool sec_batch = sec.birth != 0;
        const bool inject = secondaries && !sec_batch;
        const int k_first = sec_batch ? K : K0;                   // annihilation photons are born inside the detector: no short first pass
        cudaMemsetAsync(d_ctr, 0, cb, s);
        if (sorted) cudaMemsetAsync(d_kctr, 0, kb, s);
        cudaEventRecord(ev0, s);
        // pass p reads counter p and adds to counter p + 1; the host enqueues passes back to back and learns the
        // survivor counts TR_LAG passes late (upper bound for the grid; blocks past the true count return at once)
        unsigned ub = n0;
        bool finished = false;
        int n_timed = 0;
        std::vector<unsigned> inj(inject ? TR_MAX_PASSES + 2 : 0, 0u);       // photons injected into the input queue of pass p
        for (int p = 0; !finished; ++p) {
            if (p > TR_LAG) {
                e = cudaEventSynchronize(ring[(p - TR_LAG) % (TR_LAG + 1)]);
                if (e != cudaSuccess) { rc = cuda_fail(e, "gn_transport_run pass"); break; }
                ub = h_ctr[p - TR_LAG].front + h_ctr[p - TR_LAG].back + h_ctr[p - TR_LAG].slow;      // input count of pass p - TR_LAG >= that of pass p
                if (inject) for (int q = p - TR_LAG; q < p; ++q) ub += inj[q];     // ... plus what was injected since (the copy of counter q predates the injection at q)
                if (ub == 0) break;
            }
            if (inject && p > TR_LAG) {
                // annihilation photons of the pair vertices recorded so far join the input queue of this pass
                unsigned seen = h_np[p - TR_LAG];                                   // as the counters: TR_LAG passes old
                if (ub <= tail || p == TR_MAX_PASSES - 1) {                         // about to run to completion: the exact figures
                    PassCounters now{};
                    e = cudaMemcpyAsync(&now, d_ctr + p, sizeof now, cudaMemcpyDeviceToHost, s);
                    if (e == cudaSuccess) e = cudaMemcpyAsync(&seen, d_npairs, sizeof seen, cudaMemcpyDeviceToHost, s);
                    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
                    if (e != cudaSuccess) { rc = cuda_fail(e, "gn_transport_run pair count"); break; }
                    ub = now.front + now.back + now.slow;
                }
                unsigned avail = seen > injected ? seen - injected : 0u;
                const bool ending = ub <= tail || p == TR_MAX_PASSES - 1;
                avail = (unsigned)std::min<uint64_t>(avail, ((uint64_t)cap - std::min<uint64_t>(cap, ub)) / 2);      // as many as the queue has room for
                if (avail > 0 && (avail >= std::max(256u, ub >> 7) || ending)) {       // enough of them to be worth a source-pass launch of their own
                    SecIO<R> bs = sec; bs.birth = 1; bs.birth_first = injected;
                    const unsigned nb = 2u * avail;
                    launch_pass<R, true, false, FLAT>(track, (nb + TR_THREADS - 1) / TR_THREADS, s, g, src, seed, fid, nb, nullptr, d_ctr + p, nullptr, in, (uint32_t)cap, d_edep, d_stats, pp,
                                                      K, regroup, bs, sorted ? SortIO{d_kctr + p, d_keys, nullptr} : SortIO{nullptr, nullptr, nullptr});
                    ++launches;
                    if (sorted) {                                                    // the work order of this pass again, with the newcomers
                        cudaMemsetAsync(d_kctr[p].cur, 0, sizeof d_kctr[p].cur, s);
                        sort_scatter_kernel<<<nav_grid(((int64_t)ub + nb + 3) / 4), NAV_THREADS, 0, s>>>(d_keys, 0, d_kctr[p].tot, d_kctr[p].cur, d_perm, &d_ctr[p].front);
                        ++launches;
                    }
                    ub += nb; injected += avail; inj[p] = nb;
                }
                if (ub == 0) break;
            }
            const bool last = p > 0 && (ub <= tail || p == TR_MAX_PASSES - 1);
            const unsigned blocks = (ub + TR_THREADS - 1) / TR_THREADS;
            if (p == 0) {
                launch_pass<R, true, false, FLAT>(track, blocks, s, g, src, seed, fid, n0, nullptr, d_ctr + 1, in, out, (uint32_t)cap, d_edep, d_stats, pp, k_first, regroup, sec,
                                                  sorted ? SortIO{d_kctr + 1, d_keys, nullptr} : SortIO{nullptr, nullptr, nullptr});
            } else if (last) {
                if constexpr (!FLAT) if (geo->voxel_sched) {                 // the flagged photons of the last voxel_pass rejoin the queue
                    if (track) general_pass<R, true><<<blocks, TR_THREADS, 0, s>>>(g, d_ctr + p, d_slow, in, (uint32_t)cap, d_stats, pp, sec);
                    else general_pass<R, false><<<blocks, TR_THREADS, 0, s>>>(g, d_ctr + p, d_slow, in, (uint32_t)cap, d_stats, pp, sec);
                    ++launches;
                }
                launch_pass<R, false, true, FLAT>(track, blocks, s, g, src, seed, fid, 0u, d_ctr + p, d_ctr + p + 1, in, out, (uint32_t)cap, d_edep, d_stats, pp, K_UNLIMITED, regroup, sec,
                                                  sorted ? SortIO{nullptr, nullptr, d_perm} : SortIO{nullptr, nullptr, nullptr});
            } else {
                // interaction wavefront on the photons parked in the back of the input queue, then the lean step pass; the
                // first TR_TIMED lean passes of a batch are timed one by one, and only their steps count as lean_steps
                const bool timed = n_timed < TR_TIMED && h_stats != nullptr;      // per-pass event timing only for callers that ask for statistics
                bool voxel = false;
                if constexpr (!FLAT) voxel = geo->voxel_sched;
                if (voxel) {
                    // voxel phantoms: the slow wavefront (general steps of the flagged photons, interactions of the parked ones),
                    // then the regular-voxel step pass (voxel_pass.cuh)
                    if constexpr (!FLAT) {
                        if (track) general_pass<R, true><<<blocks, TR_THREADS, 0, s>>>(g, d_ctr + p, d_slow, in, (uint32_t)cap, d_stats, pp, sec);
                        else general_pass<R, false><<<blocks, TR_THREADS, 0, s>>>(g, d_ctr + p, d_slow, in, (uint32_t)cap, d_stats, pp, sec);
                        launch_interact<R>(track, blocks, s, g, seed, fid, d_ctr + p, in, (uint32_t)cap, d_edep, d_stats, pp, sec);
                        if (timed) cudaEventRecord(tev[2 * n_timed], s);
                        auto vp = geo->has_slabs ? (track ? voxel_pass<R, true, true> : voxel_pass<R, false, true>) : (track ? voxel_pass<R, true, false> : voxel_pass<R, false, false>);
                        vp<<<blocks, TR_THREADS, 0, s>>>(g, d_ctr + p, d_ctr + p + 1, in, out, d_slow, (uint32_t)cap, d_stats, pp, sec, K, regroup, timed ? 1 : 0);
                        ++launches;
                    }
                } else {
                    launch_interact<R>(track, blocks, s, g, seed, fid, d_ctr + p, in, (uint32_t)cap, d_edep, d_stats, pp, sec);
                    if (timed) cudaEventRecord(tev[2 * n_timed], s);
                    launch_pass<R, false, false, FLAT>(track, blocks, s, g, src, seed, fid, 0u, d_ctr + p, d_ctr + p + 1, in, out, (uint32_t)cap, d_edep, d_stats, pp, K, regroup, sec,
                                                       sorted ? SortIO{d_kctr + p + 1, d_keys, d_perm} : SortIO{nullptr, nullptr, nullptr}, timed ? 1 : 0);
                }
                if (timed) { cudaEventRecord(tev[2 * n_timed + 1], s); ++n_timed; }
                ++launches;
            }
            if (sorted && !last) {                                           // work order of the next pass: travelling survivors by volume key
                sort_scatter_kernel<<<nav_grid(((int64_t)ub + 3) / 4), NAV_THREADS, 0, s>>>(d_keys, 0, d_kctr[p + 1].tot, d_kctr[p + 1].cur, d_perm, &d_ctr[p + 1].front);
                ++launches;
            }
            ++passes; ++launches;
            e = cudaGetLastError();
            if (e == cudaSuccess && !last) {
                e = cudaMemcpyAsync(&h_ctr[p + 1], d_ctr + p + 1, sizeof(PassCounters), cudaMemcpyDeviceToHost, s);
                if (e == cudaSuccess && inject) e = cudaMemcpyAsync(&h_np[p + 1], d_npairs, sizeof(unsigned), cudaMemcpyDeviceToHost, s);
                if (e == cudaSuccess) e = cudaEventRecord(ring[(p + 1) % (TR_LAG + 1)], s);
            }
            if (e != cudaSuccess) { rc = cuda_fail(e, "gn_transport_run pass"); break; }
            finished = last;
            PhotonRec<R>* t = in; in = out; out = t;
        }
        cudaEventRecord(ev1, s);
        e = cudaStreamSynchronize(s);
        if (e != cudaSuccess && rc == GN_OK) rc = cuda_fail(e, "gn_transport_run batch");
        { float ms = 0.f; if (rc == GN_OK && cudaEventElapsedTime(&ms, ev0, ev1) == cudaSuccess) kernel_ms += ms; }
        for (int q = 0; q < n_timed && rc == GN_OK; ++q) { float ms = 0.f; if (cudaEventElapsedTime(&ms, tev[2 * q], tev[2 * q + 1]) == cudaSuccess) step_pass_ms += ms; }
    };
    for (int64_t done = 0; done < n_photons && rc == GN_OK; done += (int64_t)cap) {
        const uint32_t n0 = (uint32_t)std::min<int64_t>((int64_t)cap, n_photons - done);
        const uint64_t fid = (uint64_t)(first_id + done);
        PerPhotonOut pp{d_hash ? d_hash + done : tmp_hash, d_nsteps ? d_nsteps + done : nullptr, d_efinal ? d_efinal + done : nullptr};
        if (refill) {                                        // one persistent launch per batch: as many blocks as fit on the chip
            unsigned* d_next = (unsigned*)((char*)d_stats + 256);
            int per_sm = 0, sms = 0;
            auto kern = track ? transport_refill<R, true, FLAT> : transport_refill<R, false, FLAT>;
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, TR_THREADS, 0);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, geo->device);
            const unsigned blocks = std::min<unsigned>((n0 + TR_THREADS - 1) / TR_THREADS, (unsigned)std::max(1, per_sm * sms));
            cudaMemsetAsync(d_next, 0, sizeof(unsigned), s);
            cudaEventRecord(ev0, s);
            kern<<<blocks, TR_THREADS, 0, s>>>(g, src, seed, fid, n0, d_next, d_edep, d_stats, pp);
            cudaEventRecord(ev1, s);
            e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
            if (e != cudaSuccess) { rc = cuda_fail(e, "gn_transport_run refill"); break; }
            { float ms = 0.f; if (cudaEventElapsedTime(&ms, ev0, ev1) == cudaSuccess) kernel_ms += ms; }
            ++passes; ++launches;
            continue;
        }
        if (secondaries) cudaMemsetAsync(d_npairs, 0, sizeof(unsigned), s);
        SecIO<R> sec = no_secondaries<R>();
        if (secondaries) {
            sec.out = d_pairs; sec.n_out = d_npairs; sec.in = d_pairs; sec.state_hash = (unsigned long long*)sec_hash;
            sec.parent_hash = d_hash ? (unsigned long long*)(d_hash + done) : nullptr; sec.parent_nsteps = d_nsteps ? d_nsteps + done : nullptr;
        }
        injected = 0;
        run_batch(n0, fid, pp, sec);
        if (!secondaries || rc != GN_OK) continue;
        // the annihilation photons of the pair vertices that were not injected (pair events of the tail pass, or no room in the
        // queue), at most cap at a time (511 keV: they cannot pair again)
        unsigned n_pairs = 0;
        e = cudaMemcpyAsync(&n_pairs, d_npairs, sizeof(unsigned), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { rc = cuda_fail(e, "gn_transport_run pair count"); break; }
        const unsigned chunk = (unsigned)(cap / 2);
        for (unsigned off = injected; off < n_pairs && rc == GN_OK; off += chunk) {
            const unsigned np = std::min(chunk, n_pairs - off);
            SecIO<R> bs = sec; bs.birth = 1; bs.birth_first = off;
            run_batch(2u * np, fid, pp, bs);
        }
    }
    if (rc == GN_OK) {
        DevStats hs;
        e = cudaMemcpyAsync(&hs, d_stats, sizeof hs, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) rc = cuda_fail(e, "gn_transport_run stats");
#ifdef GN_CHECKED
        else if (hs.dbg[7]) { char msg[96]; snprintf(msg, sizeof msg, "gn_transport_run (checked build): invariant bits 0x%llx violated", hs.dbg[7]); rc = fail(GN_CUDA_ERROR, msg); }
#endif
        else if (h_stats) {
            h_stats->n_steps = hs.cnt[ST_STEPS]; h_stats->n_compton = hs.cnt[ST_COMPTON]; h_stats->n_pe = hs.cnt[ST_PE]; h_stats->n_pair = hs.cnt[ST_PAIR];
            h_stats->n_cut = hs.cnt[ST_CUT]; h_stats->n_escaped = hs.cnt[ST_ESCAPED]; h_stats->n_stuck = hs.cnt[ST_STUCK]; h_stats->n_photons = hs.cnt[ST_PHOTONS];
            h_stats->e_escaped = hs.en[EN_ESCAPED]; h_stats->e_stuck = hs.en[EN_STUCK]; h_stats->e_source = hs.en[EN_SOURCE]; h_stats->e_deposited = hs.en[EN_DEPOSITED];
            h_stats->n_passes = passes; h_stats->n_kernel_launches = launches; h_stats->kernel_ms = kernel_ms;
            h_stats->step_pass_ms = step_pass_ms; h_stats->n_steps_step_pass = hs.lean_steps; h_stats->n_rayleigh = hs.cnt[ST_RAYLEIGH];
#ifdef GN_DEBUG_COUNTERS
            fprintf(stderr, "[gn debug] fast steps %llu, bails %llu, general phases (warps) %llu, general lane-steps %llu, warp iterations %llu\n", hs.dbg[0], hs.dbg[1], hs.dbg[2], hs.dbg[3], hs.dbg[4]);
#endif
        }
    }
    return rc;
}

}  // namespace gn
