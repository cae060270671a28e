/*
 * oracle.h -- C interface of the CPU ORACLE.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA library (include/gammanav.h,
 * paper_1209_5235_b200/csrc/): the structs below are the oracle's own.
 *
 * What it computes: the per-photon transport step loop of the paper's gamma Monte Carlo
 * (Algorithm 1, L55-76; Eq. 1-9) with Geant4-style navigation
 * (locate / step) as made precise in SURVEY.md section 8(c) C0-C10
 * and DESIGN.md "Readings".  Plain, scalar, single-threaded.
 *
 * All pointers are HOST pointers.  Lengths mm, energies MeV, densities g/cm3.
 * Return value: 0 = ok, negative = error (same meaning as the product's codes, but
 * defined independently here).
 */
#ifndef ORACLE_H
#define ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_OK = 0, ORACLE_INVALID_ARGUMENT = -1, ORACLE_UNSUPPORTED_SOLID = -2, ORACLE_BAD_TREE = -3 };
enum { ORACLE_BOX = 0, ORACLE_TUBE = 1, ORACLE_ORB = 2, ORACLE_CONE = 3 };
enum { ORACLE_SRC_PENCIL = 0, ORACLE_SRC_GAUSS_PENCIL = 1, ORACLE_SRC_CONE = 2, ORACLE_SRC_ISOTROPIC = 3 };
enum { ORACLE_E_MONO = 0, ORACLE_E_LOGUNIFORM = 1 };

typedef struct {
    double tol64;        /* surface tolerance, fp64 mode [mm]; <=0 -> 1e-9                      (C0) */
    double tol32;        /* surface tolerance, fp32 mode [mm]; <=0 -> world half-extent * 2^-18 (C0) */
    double sigma_pe0;    /* photoelectric normalisation [barn/atom] at 0.1 MeV for Z=82; <=0 -> 1750 (C6) */
    double e_cut;        /* photon cut [MeV]; <=0 -> 0.010                                      (C6) */
    int32_t grid_min_daughters; /* mothers with >= this many daughters get a locate grid; <=0 -> 8 */
    int32_t stuck_limit; /* consecutive steps of length <= delta before a photon is killed; <=0 -> 8 (C9) */
    int32_t secondaries; /* 1: a pair event deposits E - 2 me c^2 and two annihilation photons are followed (S:8(f) NEXT-3); 0: deposits E */
    int32_t rayleigh;    /* 1: coherent (Rayleigh) scattering is a fourth process (S:8(f) NEXT-3, D:reading 18); 0: off */
    double sigma_r0;     /* Rayleigh cross-section of Z = 13 at 1 MeV [barn/atom]; <=0 -> 7.886e-3 (D:reading 18) */
    int32_t pe_table_per_decade; /* > 0: the photoelectric coefficient comes from a per-material table with this many points per
                                    decade of energy, 10 keV .. 1 GeV (S:8(f) NEXT-3, D:reading 19); 0: the closed form of C6 */
    int32_t pe_k_edge;   /* with the table: 1 = the tabulated cross-section drops by the K jump ratio 5 below E_K = 13.6 eV (Z-1)^2 */
} oracle_opts_t;

typedef struct {
    int32_t kind;        /* ORACLE_SRC_* */
    int32_t energy_kind; /* ORACLE_E_*   */
    double origin[3];    /* mm */
    double axis[3];      /* need not be normalised */
    double sigma;        /* GAUSS_PENCIL lateral sigma [mm] */
    double half_angle;   /* CONE half angle [rad] */
    double e0, e1;       /* MONO: e0; LOGUNIFORM: [e0, e1] MeV */
} oracle_source_t;

typedef struct {
    uint64_t n_steps, n_compton, n_pe, n_pair, n_cut, n_escaped, n_stuck, n_photons;
    double e_escaped, e_stuck, e_source, e_deposited;
    uint64_t n_rayleigh; /* Rayleigh scatters (only with opts.rayleigh) */
} oracle_stats_t;

/* geometry ------------------------------------------------------------------------------ */
/* materials: n_mats x 3 doubles (Z, A, rho).  solid_type: n_solids int32; solid_params: n_solids x 5
 * doubles (BOX: hx,hy,hz,-,-; TUBE: rmin,rmax,hz,sphi,dphi; ORB: r,-,-,-,-; CONE: r1 (at -hz),r2 (at +hz),hz,-,-).  placements: n_places x 4 int32
 * (parent, solid, material, transform); node 0 is the world (parent -1), parent < child.
 * transforms: n_transforms x 12 doubles, R row-major (local->parent) then T.                      */
int oracle_geometry_create(const double* materials, int32_t n_mats,
                           const int32_t* solid_type, const double* solid_params, int32_t n_solids,
                           const int32_t* placements, int32_t n_places,
                           const double* transforms, int32_t n_transforms,
                           const oracle_opts_t* opts, void** out);
int oracle_geometry_destroy(void* geo);
double oracle_geometry_tolerance(const void* geo, int precision);

/* navigation.  precision = 32 | 64 selects float | double buffers.
 * use_grid = 0 forces the plain definition (linear scan over all daughters) everywhere.            */
int oracle_nav_locate(const void* geo, int precision, const void* pos, const void* dir /*or NULL*/,
                      int64_t n, int32_t* vol_out, int use_grid);
/* the pin for locate: linear scan over ALL nodes with hierarchical per-level fp64 transforms       */
int oracle_nav_locate_bruteforce(const void* geo, const double* pos, int64_t n, int32_t* vol_out);
int oracle_nav_compute_step(const void* geo, int precision, const void* pos, const void* dir,
                            const int32_t* vol_in, const void* max_step /*or NULL*/, int64_t n,
                            void* step_out, int32_t* next_vol_out, int use_grid);

/* ComputeStep with the surface normal ("what is the normal of the boundary surface at that point?"): as
 * oracle_nav_compute_step, plus normal_out n x 3 Real: outward unit normal, global frame, of the solid whose surface ends
 * the step (own solid on exit, the entered daughter otherwise); (0,0,0) when no boundary lies within max_step. */
/* isotropic safety (S:8(f) NEXT-4, D:reading 17): lower bound, valid in every direction, of the distance from pos[i] (a point
 * of volume vol_in[i]) to the nearest boundary of that volume's solid or of one of its daughters; linear scan; vol -1 -> 0 */
int oracle_nav_compute_safety(const void* geo, int precision, const void* pos, const int32_t* vol_in, int64_t n, void* safety_out);
int oracle_nav_compute_step_normal(const void* geo, int precision, const void* pos, const void* dir, const int32_t* vol_in,
                                   const void* max_step, int64_t n, void* step_out, int32_t* next_vol_out, void* normal_out, int use_grid);

/* transport (C6-C9).  Photons first_id .. first_id+n-1; edep_out has n_places doubles and is
 * ACCUMULATED INTO (caller zeroes); per-photon outputs may be NULL.                                */
int oracle_transport_run(const void* geo, int precision, const oracle_source_t* src, uint64_t seed,
                         int64_t first_id, int64_t n_photons, double* edep_out, oracle_stats_t* stats_out,
                         uint64_t* hash_out, uint32_t* nsteps_out, double* efinal_out, int use_grid);

/* as oracle_transport_run, plus per volume (n_places each, ACCUMULATED INTO, may be NULL): edep_sq_out = sum of the squares of
 * the deposits, n_dep_out = number of deposits -- the Monte Carlo error of a group of volumes for S:C10's "1e-3 + 3 sigma_MC" */
int oracle_transport_run_tally(const void* geo, int precision, const oracle_source_t* src, uint64_t seed, int64_t first_id,
                               int64_t n_photons, double* edep_out, double* edep_sq_out, uint32_t* n_dep_out, oracle_stats_t* stats_out,
                               uint64_t* hash_out, uint32_t* nsteps_out, double* efinal_out, int use_grid);

/* Operation counts of the algorithm on a real workload (S:8(d) "instrumented oracle"): the same templates run in a
 * counting type (fp64 values).  counts_out = {add/sub, mul, div, sqrt, compare/min/max/abs, fma, transcendental,
 * flops = sum with fma counted twice}.  Transport: photons first_id.. (the locate grid is used; ComputeStep is the plain
 * linear scan); nav: n config-5 queries (locate, then ComputeStep), pos / dir n x 3 doubles. */
int oracle_transport_count_ops(const void* geo, const oracle_source_t* src, uint64_t seed, int64_t first_id, int64_t n_photons,
                               uint64_t counts_out[8], oracle_stats_t* stats_out);
int oracle_nav_count_ops(const void* geo, const double* pos, const double* dir, int64_t n, uint64_t counts_out[8]);

/* test hooks: the history hash (S:C9) of a byte string / of a list of 32-bit words (vol_before, event, ...); the source
 * frame (a, e1, e2; D:reading 4) and the composed global->local transforms (M row-major 9, T 3 per node; S:C0) as rounded
 * to the given precision */
uint64_t oracle_fnv1a_bytes(const uint8_t* bytes, int64_t n);
uint64_t oracle_history_hash(const uint32_t* words, int64_t n_words);
int oracle_source_frame(const oracle_source_t* src, int precision, double frame_out[9]);
int oracle_composed_transforms(const void* geo, int precision, double* M_out, double* T_out);

/* The paper's own benchmark (Algorithm 2 phase 5): free path T_i of particle i from (x0, w, Y)_i by
 * Algorithm 1 with attenuation only, mu = rho * mu_mass (Eq. 9; mu_mass in cm^2/g, 0.06146 for Al at
 * 1 MeV).  pos/dir: n x 3 Real, Y: n Real, T_out: n Real (+inf: left the world), nsteps_out: n or NULL. */
int oracle_free_path_run(const void* geo, int precision, const void* pos, const void* dir, const void* Y, int64_t n,
                         double mu_mass_cm2_g, void* T_out, uint32_t* nsteps_out, int use_grid);

/* unit entry points used by the pins ------------------------------------------------------- */
/* one solid, many points.  what: 0 = Inside (out: int32 0 in / 1 surface / 2 out written as Real),
 * 1 = DistanceToIn, 2 = DistanceToOut, 3 = surface normal at pos (out: n x 3 Real).  pos/dir: n x 3 Real, out: n Real.                          */
int oracle_solid_eval(int32_t type, const double* params5, double tol, int precision, int what,
                      const void* pos, const void* dir, int64_t n, void* out);
double oracle_sigma_kn(double k);                       /* Klein-Nishina total, cm^2 per electron */
double oracle_sigma_pair(double k, double Z);           /* cm^2 per atom */
double oracle_sigma_pe(double E, double Z, double sigma_pe0_barn); /* cm^2 per atom */
/* mu[3] = (mu_PE, mu_C, mu_pair) in 1/mm for material m at energy E, in the given precision (mu_PE from the table when the
 * geometry was created with pe_table_per_decade > 0); oracle_mu_rayleigh: mu_R (0 unless created with rayleigh = 1) */
int oracle_mu(const void* geo, int precision, int32_t material, double E, double* mu3);
double oracle_mu_rayleigh(const void* geo, int precision, int32_t material, double E);
/* n cosines of the Rayleigh scattering angle, photon ids first_id.. (draws start at 0): rejection from p(c) ~ 1 + c^2 */
int oracle_rayleigh_sample(int precision, uint64_t seed, int64_t first_id, int64_t n, double* cost_out, int32_t* ntrials_out);
/* directions of the two annihilation photons of photon id's pair event (S:8(f) NEXT-3): n x 3 doubles each */
int oracle_pair_directions(int precision, uint64_t seed, int64_t first_id, int64_t n, double* w1_out, double* w2_out);
void oracle_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t* out4);
double oracle_uniform_from_lane(uint64_t lane, int precision);
/* draw j (0-based) of photon id under seed, as a uniform in (0,1] */
double oracle_draw(uint64_t seed, uint64_t id, uint32_t j, int precision);
/* n Klein-Nishina samples at energy E using photon ids first_id.. (draws start at 0):
 * eps_out = E'/E, cost_out = cos(theta), ntrials_out = rejection trials used */
int oracle_kn_sample(int precision, double E, uint64_t seed, int64_t first_id, int64_t n,
                     double* eps_out, double* cost_out, int32_t* ntrials_out);
/* direction update C7: rotates w (n x 3 doubles) by (cost, phi) */
int oracle_rotate(int precision, const double* w, const double* cost, const double* phi, int64_t n, double* w_out);
/* the canonical move C0: pos_out = fma(step, dir, pos), n x 3 Real */
int oracle_move(int precision, const void* pos, const void* dir, const void* step, int64_t n, void* pos_out);
/* source sampling C8: positions, directions, energies of photons first_id.., and draws consumed */
int oracle_source_sample(int precision, const oracle_source_t* src, uint64_t seed, int64_t first_id, int64_t n,
                         double* pos_out, double* dir_out, double* e_out, int32_t* ndraws_out);

#ifdef __cplusplus
}
#endif
#endif
