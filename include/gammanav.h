/*
 * gammanav.h -- C ABI of the B200-native gamma transport / Geant4-style navigation library
 * (libgammanav.so, hand-written CUDA for sm_100a; no CPU fallback).
 *
 * The four entry points follow the paper's statement of the problem:
 *   - "Load the geometry and transfer it to GPU memory"            PAPER.md L139 (Algorithm 2, phase 1)  -> gn_geometry_create
 *   - "If a particle is in point A, inside which ... volumes is it?" PAPER.md L124                        -> gn_nav_locate
 *   - "Will the particle hit a volume boundary ... on its way to point B? If so, where"  PAPER.md L125   -> gn_nav_compute_step
 *   - Algorithm 1 run for N particles in parallel (Algorithm 2 phase 5, L143),
 *     generalised to Compton / photoelectric / pair sampling with a per-volume energy tally
 *     (BASELINE.json north_star)                                                   -> gn_transport_run
 *
 * Conventions: lengths mm, energies MeV, densities g/cm3.  `precision` is 32 or 64 and selects the
 * element type (float / double) of every `void*` Real buffer and the arithmetic of the kernels.
 * Pointers named h_* are HOST memory, d_* are DEVICE memory (caller-owned, never retained).
 * Positions / directions at the ABI are row-major n x 3 (x0 y0 z0 x1 ...).
 * Every function returns GN_OK (0) or a negative gn_status; nothing throws or aborts, and outputs are
 * untouched on failure.  gn_last_error() gives a human-readable string for the calling thread's last failure.
 * All nav calls are asynchronous on `cuda_stream` (a cudaStream_t, NULL = default stream).  gn_transport_run is
 * host-synchronous: the stream only orders it against earlier work; the call waits for survivor counts while it
 * enqueues its passes, synchronises the stream at the end of every batch (with gn_opts.secondaries also before the last pass of a batch
 * and once per leftover batch of annihilation photons) and returns when the tally and the statistics are complete.
 * Every call runs on the device the geometry was created on; the caller's current device is restored on return.
 */
#ifndef GAMMANAV_H
#define GAMMANAV_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GN_OK = 0,
    GN_INVALID_ARGUMENT = -1,   /* NULL / negative sizes / bad precision / index out of range */
    GN_UNSUPPORTED_SOLID = -2,  /* unknown type, or tube with pi < dphi < 2 pi (non-convex sector) */
    GN_BAD_TREE = -3,           /* node 0 not the world, parent >= child, R not orthonormal (1e-9) */
    GN_OUT_OF_MEMORY = -4,
    GN_CUDA_ERROR = -5
} gn_status;

enum { GN_BOX = 0, GN_TUBE = 1, GN_ORB = 2, GN_CONE = 3 };
enum { GN_SRC_PENCIL = 0, GN_SRC_GAUSS_PENCIL = 1, GN_SRC_CONE = 2, GN_SRC_ISOTROPIC = 3 };
enum { GN_E_MONO = 0, GN_E_LOGUNIFORM = 1 };

typedef struct gn_geometry gn_geometry;   /* opaque; owns all device allocations of one geometry */

/* Options (all fields: <= 0 selects the default).  SURVEY 8(c) C0, C5, C6, C9. */
typedef struct {
    double tol64;              /* surface tolerance in fp64 mode [mm]; default 1e-9 */
    double tol32;              /* surface tolerance in fp32 mode [mm]; default (largest world half-extent) * 2^-18 */
    double sigma_pe0;          /* photoelectric cross-section of Z = 82 at 0.1 MeV [barn/atom]; default 1750 */
    double e_cut;              /* photons below this energy are absorbed locally [MeV]; default 0.010 */
    int32_t voxel_min_daughters; /* mothers with at least this many daughters get a voxel grid; default 8 */
    int32_t stuck_limit;       /* consecutive steps of length <= tol/2 before a photon is killed; default 8, at most 255
                                  (gn_geometry_create returns GN_INVALID_ARGUMENT above that: the per-photon counter has 8 bits;
                                  the per-photon step count has 24 bits and wraps at 2^24 steps of one photon) */
    int32_t steps_per_pass;    /* K: steps a photon takes per wavefront pass before it is re-queued; default 16 (24 with the
                                  regular-voxel schedule) */
    int32_t first_pass_steps;  /* K0: steps in the pass that also generates the photons (sheds photons that miss early); default 1 */
    int32_t tail_photons;      /* once at most this many photons are left, one last pass runs them to completion; default 148 * 1024 */
    int32_t regroup_percent;   /* a warp ends its pass early once fewer than this % of the lanes it started with still travel
                                  (the compaction then refills it); default 35 for box-only unrotated geometries, else 90 */
    int32_t secondaries;       /* 1: a pair event deposits E - 2 me c^2 locally and its two back-to-back annihilation photons
                                  (me c^2 each, isotropic axis, Philox stream tags 1 / 2 of the parent's id) are transported
                                  from the vertex; their steps, events, hashes and step counts are added to
                                  the parent's.  0 (default): a pair event deposits all of E locally (BASELINE.json config 1) */
    int32_t refill;            /* 1: the paper's own scheduling remedy ("filling the empty places with new
                                  particles") as one persistent kernel per batch: each lane follows its photon to the end and
                                  then takes the next photon id from a device counter.  Same per-photon results as the default
                                  wavefront passes (0); cannot be combined with secondaries */
    int32_t no_voxel_pass;     /* 1: keep the general lean step pass even when the geometry is mostly regular voxels (a voxel
                                  phantom of unrotated boxes), for which the default (0) schedules the regular-voxel step kernel
                                  plus a slow wavefront for every other step; same per-photon results either way */
    int32_t rayleigh;          /* 1: coherent (Rayleigh) scattering is a fourth process (reading 18):
                                  mu_R = n sigma_R0 (Z/13)^2 / E^2, angle from 1 + cos^2(theta) by rejection, energy unchanged, nothing
                                  deposited, event word 7; 0 (default): off (BASELINE.json config 1's physics) */
    double sigma_r0;           /* Rayleigh cross-section of Z = 13 at 1 MeV [barn/atom]; default 7.886e-3 (the model's mu / rho of
                                  aluminium at 1 MeV then equals PAPER.md L150's 0.06146 cm^2/g) */
    int32_t pe_table_per_decade; /* > 0: the photoelectric coefficient comes from a per-material table with this many points per
                                  decade over 10 keV .. 1 GeV, interpolated linearly in ln E (reading 19); 0 (default): the closed
                                  form; at most 4096 */
    int32_t pe_k_edge;         /* with the table: 1 = the tabulated cross-section drops by the K jump ratio 5 below
                                  E_K = 13.6 eV (Z - 1)^2; 0 = the table is the Z^5 / E^3.5 law itself.
                                  Either option switches the regular-voxel schedule off (the general passes handle them) */
} gn_opts;

/* Photon source.  axis need not be normalised. */
typedef struct {
    int32_t kind;              /* GN_SRC_* */
    int32_t energy_kind;       /* GN_E_*   */
    double origin[3];          /* mm */
    double axis[3];
    double sigma;              /* GN_SRC_GAUSS_PENCIL: lateral Gaussian sigma [mm] */
    double half_angle;         /* GN_SRC_CONE: half opening angle [rad], uniform in solid angle */
    double e0, e1;             /* MONO: e0; LOGUNIFORM: uniform in ln E over [e0, e1] */
} gn_source;

/* Run statistics (host).  n_steps = number of ComputeStep calls = the "photon steps" of BASELINE.json's metric. */
typedef struct {
    uint64_t n_steps, n_compton, n_pe, n_pair, n_cut, n_escaped, n_stuck, n_photons;
    double e_escaped, e_stuck, e_source, e_deposited;
    uint64_t n_passes;         /* wavefront passes (kernel launches of the step kernel) */
    uint64_t n_kernel_launches;/* all kernels launched by the call */
    double kernel_ms;          /* duration of the whole kernel sequence of the run (source pass, step passes, interaction
                                  passes, tail), CUDA events on the launching stream */
    double step_pass_ms;       /* sum of the launch durations of the lean wavefront step passes (the dominant kernel), one
                                  CUDA-event pair per launch; only the first 64 such passes of each batch are timed, and only when
                                  h_stats_out is not NULL (a caller that asks for no statistics gets no per-pass events) */
    uint64_t n_steps_step_pass;/* steps taken inside exactly those timed passes (later lean passes count in n_steps only) */
    uint64_t n_rayleigh;       /* Rayleigh scatters (gn_opts.rayleigh) */
} gn_run_stats;

/*
 * gn_geometry_create -- PAPER.md L139 / L127 (volumes hierarchy, solids, per-material density).
 *   h_materials    n_mats x 3 doubles: Z, A [g/mol], rho [g/cm3]
 *   h_solid_type   n_solids int32: GN_BOX | GN_TUBE | GN_ORB | GN_CONE (ORB: r,-,-,-,- ; CONE: solid frustum, r1 at -hz, r2 at +hz, hz,-,- ;
 *                  DESIGN.md "orb solid" / "cone solid"; the four solid types PAPER.md L160 names)
 *   h_solid_params n_solids x 5 doubles: BOX hx,hy,hz,-,- ; TUBE rmin,rmax,hz,sphi,dphi  (C2; dphi >= 2 pi
 *                  = full tube, 0 < dphi <= pi = convex sector)
 *   h_placements   n_places x 4 int32: parent (-1 for node 0 = world, parent < child), solid, material,
 *                  transform index.  Every node is its own touchable: volume index = node index (C1).
 *   h_transforms   n_transforms x 12 doubles: R row-major (local -> parent) then T [mm]   (C0)
 *   h_opts         NULL = defaults
 * All input arrays are host memory, copied during the call.  The handle owns its device memory
 * (structure-of-arrays store: node records, composed global->local affine transforms in fp32 and fp64,
 * solids, material factors, flattened voxel grids) until gn_geometry_destroy.
 * Overlapping / protruding daughters are not detected (Geant4 convention).
 */
int gn_geometry_create(const double* h_materials, int32_t n_mats,
                       const int32_t* h_solid_type, const double* h_solid_params, int32_t n_solids,
                       const int32_t* h_placements, int32_t n_places,
                       const double* h_transforms, int32_t n_transforms,
                       const gn_opts* h_opts, gn_geometry** out);
int gn_geometry_destroy(gn_geometry* geo);

/* geometry queries (host side, cheap) */
int32_t gn_geometry_num_places(const gn_geometry* geo);
double gn_geometry_tolerance(const gn_geometry* geo, int precision);
/* voxel store summary: info[0] = number of voxelised mothers, [1] = total cells, [2] = total candidate
 * references, [3] = bytes of device memory held by the geometry */
int gn_geometry_voxel_info(const gn_geometry* geo, int64_t info[4]);

/*
 * gn_nav_locate -- PAPER.md L124; SURVEY 8(c) C3.
 *   d_pos n x 3 Real, d_dir n x 3 Real or NULL (NULL: a point on a surface counts as inside),
 *   d_vol_out n int32: deepest volume occupied, -1 = outside the world.
 */
int gn_nav_locate(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir,
                  int64_t n, int32_t* d_vol_out, void* cuda_stream);

/*
 * gn_nav_compute_step -- PAPER.md L125; SURVEY 8(c) C4.
 *   d_vol_in n int32 (as returned by gn_nav_locate; -1 gives (+inf, -1)),
 *   d_max_step n Real or NULL (= +inf): if the nearest boundary is farther than max_step the result is
 *   (+inf, vol_in),
 *   d_step_out n Real: distance to the nearest boundary (DistanceToOut of the current solid, DistanceToIn of
 *   its daughters via the voxel grid), d_next_vol_out n int32: the volume occupied just after the boundary
 *   (-1 = left the world).
 */
int gn_nav_compute_step(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir,
                        const int32_t* d_vol_in, const void* d_max_step, int64_t n,
                        void* d_step_out, int32_t* d_next_vol_out, void* cuda_stream);

/*
 * gn_nav_compute_step_noalloc -- gn_nav_compute_step for callers that must not allocate:
 * code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same arguments, same results bit
 * for bit.  gn_nav_compute_step takes the scratch of its query sort (general geometries: queries grouped by the kind of
 * their current volume before ComputeStep) from the handle's stream-ordered memory pool; this entry point takes it from one
 * fixed array in device memory that belongs to the library, and calls no cudaMalloc, cudaFree or pool routine.
 *   Limit: n <= GN_NOALLOC_MAX_QUERIES (2^20); larger n returns GN_INVALID_ARGUMENT with outputs untouched -- split the
 *   batch.  Cost: every GPU that loads the library holds GN_NOALLOC_SCRATCH_BYTES (5.3 MB) until the process exits.
 *   All calls share the array, on every handle: two calls that overlap on the GPU (different streams) race on it --
 *   serialise them (same stream, or an event between them).  Asynchronous on cuda_stream like gn_nav_compute_step.
 */
#define GN_NOALLOC_MAX_QUERIES (1 << 20)
#define GN_NOALLOC_SCRATCH_BYTES (1024 + 5 * (1 << 20))
int gn_nav_compute_step_noalloc(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir,
                                const int32_t* d_vol_in, const void* d_max_step, int64_t n,
                                void* d_step_out, int32_t* d_next_vol_out, void* cuda_stream);

/*
 * gn_nav_compute_step_normal -- PAPER.md L125 in full: "... If so, where, and what is the normal of the boundary surface at
 * that point?"  As gn_nav_compute_step, plus d_normal_out n x 3 Real: the outward unit normal, in the global frame, of the
 * solid whose surface ends the step -- the current volume's own solid (the step leaves it), or the daughter entered (ties:
 * mother first, then the lowest daughter index).  The surface of that solid is the one with the largest signed outsideness
 * at the crossing point.  (0,0,0) when no boundary lies within max_step.
 */
int gn_nav_compute_step_normal(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir,
                               const int32_t* d_vol_in, const void* d_max_step, int64_t n,
                               void* d_step_out, int32_t* d_next_vol_out, void* d_normal_out, void* cuda_stream);

/*
 * gn_nav_compute_safety -- isotropic safety distance (the boundary problem of PAPER.md L124-125 without a
 * direction): a lower bound, valid in EVERY direction, of the distance from d_pos[i] to the nearest boundary of volume
 * d_vol_in[i]'s own solid or of one of its daughters -- no gn_nav_compute_step from that point is shorter.
 *   = min( max(-D_vol(p), 0), min over daughters d of max(D_d(p_d), 0) ),  D = the outsideness of SURVEY 8(c) C2 (the largest
 *   signed distance to one bounding plane / cylinder / sphere / cone of the solid, negative inside); from inside it is the exact
 *   distance to the nearest bounding surface for box, tube and orb (reading 17).
 *   d_pos n x 3 Real (device), d_vol_in n int32 (as returned by gn_nav_locate; -1 or out of range gives 0),
 *   d_safety_out n Real (device, caller-owned).  Asynchronous on cuda_stream.  Daughters are scanned linearly.
 */
int gn_nav_compute_safety(const gn_geometry* geo, int precision, const void* d_pos, const int32_t* d_vol_in, int64_t n,
                          void* d_safety_out, void* cuda_stream);

/*
 * gn_transport_run -- PAPER.md Algorithm 1 (L55-76) for photons first_photon_id .. first_photon_id + n - 1,
 * each with its own Philox4x32-10 stream keyed by (seed, photon id).
 *   d_edep_out    gn_geometry_num_places doubles [MeV]; ZEROED by the callee, then accumulated (fp64 atomics)
 *   h_stats_out   host, may be NULL
 *   d_hash_out    n uint64 history hashes (FNV-1a-64 over (volume, event) per step), or NULL
 *   d_nsteps_out  n uint32 steps per photon, or NULL
 *   d_efinal_out  n doubles: photon energy when it terminated, or NULL
 * With gn_opts.secondaries = 1 a photon's hash and step count are the sums (wrapping, order-independent) over itself and the
 * two annihilation photons of its pair event, d_efinal_out stays the primary's own energy at its end, and the counters of
 * h_stats_out count every photon followed except n_photons / e_source (primaries only); scratch grows by one pair-vertex
 * list (16 / 32 B per photon of a batch).  gn_opts.refill = 1 runs the same histories in one persistent kernel per batch
 * (no queues are used); combining it with secondaries returns GN_INVALID_ARGUMENT.
 * Scratch (two photon-state queues, 2 x min(n, 2^24) x 64 B in fp32 / 112 B in fp64, plus counters) belongs to
 * the geometry handle: grown on demand, reused by later runs, released by gn_geometry_destroy.  Runs on one
 * handle are serialised (internal mutex); use one handle per stream for concurrent runs.
 */
int gn_transport_run(const gn_geometry* geo, int precision, const gn_source* h_src, uint64_t seed,
                     int64_t first_photon_id, int64_t n_photons,
                     double* d_edep_out, gn_run_stats* h_stats_out,
                     uint64_t* d_hash_out, uint32_t* d_nsteps_out, double* d_efinal_out, void* cuda_stream);

/*
 * gn_free_path_run -- the paper's own benchmark, Algorithm 2 phase 5: the free path T_i of particle i
 * from (x0, w, Y)_i by Algorithm 1 (L55-76) with attenuation only, mu = rho(volume) * mu_mass (Eq. 9;
 * mu_mass in cm^2/g: 0.06146 for aluminium at 1 MeV, L150).  One thread walks one particle from boundary to boundary
 * carrying the remaining optical depth, as the paper's kernel did.
 *   d_pos, d_dir  n x 3 Real; d_Y n Real (the "lifetimes", generated by the caller as in Algorithm 2 steps 2-3)
 *   d_T_out       n Real: free path [mm]; +inf when the particle leaves the world first ("S_j may be infinite", L73)
 *   d_nsteps_out  n uint32 ComputeStep calls per particle, or NULL
 * Asynchronous on cuda_stream.
 */
int gn_free_path_run(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir, const void* d_Y,
                     int64_t n, double mu_mass_cm2_g, void* d_T_out, uint32_t* d_nsteps_out, void* cuda_stream);

/* Host-buffer wrappers (the "end to end" path: copies host<->device inside the call).  The query arrays are processed in
 * chunks of 2^22 on two internal streams with a device staging area owned by the handle, so that uploads, kernels and
 * downloads of neighbouring chunks overlap when the caller's buffers are page-locked (pageable buffers work, serially).
 * Synchronous: results are complete on return.  Calls on one handle are serialised. */
int gn_nav_query_host(const gn_geometry* geo, int precision, const void* h_pos, const void* h_dir, int64_t n,
                      int32_t* h_vol_out, void* h_step_out, int32_t* h_next_vol_out);
int gn_free_path_run_host(const gn_geometry* geo, int precision, const void* h_pos, const void* h_dir, const void* h_Y, int64_t n,
                          double mu_mass_cm2_g, void* h_T_out, uint32_t* h_nsteps_out /* or NULL */);   /* Algorithm 2 phases 4-6 */
int gn_transport_run_host(const gn_geometry* geo, int precision, const gn_source* h_src, uint64_t seed,
                          int64_t first_photon_id, int64_t n_photons, double* h_edep_out, gn_run_stats* h_stats_out);

/*
 * gn_selftest_arith -- device self-test of the library's in-line correctly rounded fp32 division and square root
 * (SURVEY 8(c) C0 "canonical arithmetic": navigation may only use correctly rounded + - x / sqrt) against the
 * toolchain's IEEE intrinsics, bit for bit: all 2^32 square-root arguments and n_div_pairs pseudo-random /
 * structured division pairs.  h_out[0] = sqrt mismatches, [1] = division mismatches, [2] / [3] = smallest failing
 * argument index of each (all ones when none).  Synchronous; default stream.
 */
int gn_selftest_arith(int64_t n_div_pairs, uint64_t h_out[4]);

/*
 * gn_selftest_pipe_peak -- FP32 (precision 32: FFMA) or FP64 (64: DFMA) pipe peak of the current device by a register-
 * resident fused-multiply-add kernel (8 independent chains per thread, one block of 1024 threads per SM): the flops leg of the
 * per-step roofline.  h_out[0] = TFLOP/s (fma = 2 flops), [1] = SM clock during the run [MHz],
 * [2] = kernel time [ms], [3] = number of SMs.  Synchronous; default stream.
 */
int gn_selftest_pipe_peak(int precision, double h_out[4]);

/*
 * Host-only hooks (no device needed): the fp64 set-up arithmetic of the library, exposed so that tests can compare it with
 * an independent implementation of the same definitions.
 *   gn_host_source_frame: frame_out = a (axis / |axis|), e1, e2, as rounded to `precision`
 *   gn_host_compose_transforms: for every placement the composed global -> local rotation M (row-major 9 doubles) and
 *   translation T (3 doubles) of SURVEY 8(c) C0 (M = R_global^T, p_local = M (x - T)); same validation and status codes as
 *   gn_geometry_create
 */
int gn_host_source_frame(const gn_source* h_src, int precision, double frame_out[9]);
/*
 *   gn_host_voxel_tables: the host tables gn_geometry_create would upload for this geometry (same arguments, same code, no
 *   device touched): counts = {voxel grids, voxel cells, candidate references}; per node its info word (solid index in bits
 *   0-15; bit 30 identity rotation, 29 regular voxel, 28 regular slab, 31 sibling hints) and link (first daughter / ~grid id
 *   of a voxelised mother / cell index of a regular voxel or slab); h_hint 4 per node (sibling across the lower / upper z face,
 *   the start / end phi plane; -1 none); h_grids 11 doubles per grid (mother node, gmin[3], cell width[3], cells[3], first
 *   cell); h_cell_start (cells + 1 offsets into h_cand) and h_cand (candidate daughters of every cell, ascending).  Any
 *   output pointer but counts may be NULL; call once for the counts, then with arrays of those sizes.
 */
int gn_host_voxel_tables(const double* h_materials, int32_t n_mats, const int32_t* h_solid_type, const double* h_solid_params,
                         int32_t n_solids, const int32_t* h_placements, int32_t n_places, const double* h_transforms,
                         int32_t n_transforms, const gn_opts* h_opts, int64_t counts[3], int32_t* h_node_info,
                         int32_t* h_node_link, int32_t* h_hint, double* h_grids, int32_t* h_cell_start, int32_t* h_cand);
int gn_host_compose_transforms(const int32_t* h_placements, int32_t n_places, const double* h_transforms, int32_t n_transforms,
                               double* h_M_out, double* h_T_out);

const char* gn_last_error(void);
const char* gn_version(void);

#ifdef __cplusplus
}
#endif
#endif
