/* mcdc.h -- C-ABI of the B200-native event-based Monte Carlo neutron transport library.
 *
 * What it computes: the data-parallel hot path of the transport loop named in arxiv 2501.05440
 * ("continuous and multi-group energy neutron transport physics with constructive solid
 * geometry modeling using surface tracking ... k-eigenvalue and fully dynamic simulations ...
 * replicable random number generation"; PAPER.md:51 one "segment" = one event; PAPER.md:55 dual
 * particle banks; PAPER.md:57 per-event kernels; PAPER.md:124 inactive/active cycles
 * time-dependent fixed source).  The paper prints no formulas; every step follows the readings
 * R1..R40 of DESIGN.md section 3 (R1..R31 = SURVEY.md 8c).
 *
 * Conventions for every call
 *   - plain C: pointers + sizes only.  All INPUT pointers are HOST pointers; the library copies what
 *     it needs during the call (the caller may free them as soon as the call returns).  All OUTPUT
 *     pointers are HOST pointers to caller-allocated arrays of the documented length.
 *   - the only DEVICE pointer is mcdc_device.workspace: device memory owned by the caller (the Python
 *     binding allocates it with torch.empty); the library never calls cudaMalloc/cudaFree.  All kernels
 *     are launched on mcdc_device.stream (a cudaStream_t; NULL = the legacy default stream).
 *   - every call returns 0 or a negative MCDC_E* code; mcdc_last_error() gives a thread-local
 *     message.  Nothing throws or aborts across the ABI.  A failed run call leaves the results of the last
 *     successful call readable (mcdc_get_dims / mcdc_get_tallies keep reporting them) and the problem usable: the
 *     next run has to start again from cycle 0.
 *   - all floating point is float64.
 */
#ifndef MCDC_H
#define MCDC_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { MCDC_OK = 0, MCDC_EINVAL = -1, MCDC_EGEOM = -2, MCDC_EBANK = -3, MCDC_ELOST = -4, MCDC_ECUDA = -5,
       MCDC_ENOMEM = -6 };

/* surface types / boundary conditions (R11-R13) */
enum { MCDC_PLANE_X = 0, MCDC_PLANE_Y, MCDC_PLANE_Z, MCDC_PLANE, MCDC_CYL_X, MCDC_CYL_Y, MCDC_CYL_Z, MCDC_SPHERE };
enum { MCDC_BC_TRANSMIT = 0, MCDC_BC_REFLECT = 1, MCDC_BC_VACUUM = 2 };

/* event codes of the trace and of the event counters (one event per segment) */
enum { MCDC_EV_SCATTER = 1, MCDC_EV_FISSION, MCDC_EV_CAPTURE, MCDC_EV_TRANSMIT, MCDC_EV_REFLECT, MCDC_EV_LEAK,
       MCDC_EV_LATTICE, MCDC_EV_TIME_EDGE, MCDC_EV_CUTOFF, MCDC_EV_LOST };
/* counters[0] tracks started, [1..10] events by code, [11] children banked, [12] largest fission / secondary bank
 * of the run (sites), [13] kernel rounds (sweeps + persistent launches), [14] particles the persistent kernel took
 * from its work queue, [15] reserved */
#define MCDC_N_COUNTERS 16

/* CSG geometry: at most 3800 surfaces, conjunctive cells grouped by universe, one optional rectangular lattice whose
 * elements may themselves hold second-level lattices (R11-R16, R37).  surf_param[s][4]: PLANE_X/Y/Z (p,-,-,-); PLANE (a,b,c,d): a x+b y+c z = d; CYL_Z (x0,y0,r,-)
 * (CYL_X (y0,z0,r), CYL_Y (x0,z0,r)); SPHERE (x0,y0,z0,r).  Cells of universe u are
 * [univ_cell_off[u], univ_cell_off[u+1]); universe 0 is the root.  cell_fill_type 0: cell_fill = material
 * id; 1: the cell is filled by the lattice (at most one such cell, in the root universe).  lat_univ[iy][ix]
 * names the universe of element (ix,iy); its cells are written in element-centred coordinates.
 * Second-level lattices (a core of assemblies of pin lattices; R37): cell_fill_type 2 = the
 * cell, which must belong to a universe used by lattice elements, is filled by second-level lattice k = cell_fill:
 * lat2_nx[k] x lat2_ny[k] elements of pitch lat2_px[k], lat2_py[k], centred on the origin of that universe's
 * coordinates; element (ix,iy) holds universe lat2_univ[lat2_off[k] + iy lat2_nx[k] + ix], whose cells (material-
 * filled only) are written in coordinates centred on the element.  At most one such cell per universe.  The
 * first-level lattice has at most 2^20 elements, a second-level one at most 2047.
 * A location inside lattices is reported (traces, mcdc_test_geometry) as first-level element | (second-level element
 * + 1) << 20; lattice-wall hit codes are n_surf + 0..3 (first level: -x,+x,-y,+y) and n_surf + 4..7 (second level).
 * A lattice's outermost lines are never events: the enclosing cell's surfaces, or the first-level walls, bound it. */
typedef struct {
    int32_t n_surf;
    const int32_t *surf_type;
    const double *surf_param;
    const int32_t *surf_bc;
    int32_t n_cell;
    const int32_t *cell_surf_off;   /* [n_cell+1] */
    const int32_t *cell_surf_id;    /* [cell_surf_off[n_cell]] */
    const int32_t *cell_surf_sense; /* +1: f(x) > 0 side, -1: f(x) < 0 side */
    const int32_t *cell_fill_type;
    const int32_t *cell_fill;
    int32_t n_univ;
    const int32_t *univ_cell_off; /* [n_univ+1] */
    int32_t has_lattice;
    double lat_x0, lat_y0, lat_px, lat_py;
    int32_t lat_nx, lat_ny;
    const int32_t *lat_univ; /* [lat_ny][lat_nx] */
    int32_t n_lat2;          /* second-level lattices (0: none; the pointers below may then be NULL) */
    const int32_t *lat2_nx, *lat2_ny;
    const double *lat2_px, *lat2_py;
    const int32_t *lat2_off;  /* [n_lat2+1] */
    const int32_t *lat2_univ; /* [lat2_off[n_lat2]] */
} mcdc_geometry;

/* time-dependent multi-group data ("fully dynamic simulations"; R38-R40):
 * speed[G] cm/s; n_dgroup delayed-neutron precursor groups per material with yields nu_d[n_mat][n_dgroup][G] (the
 * materials' nu is then the PROMPT yield), decay constants decay[n_mat][n_dgroup] 1/s and emission spectra
 * chi_d[n_mat][n_dgroup][G].  The time edges are mcdc_tally_spec.t_edges; every edge is a census.  census_target > 0:
 * the population entering every census interval but the first is combed to that many particles (weight-conserving
 * population control). */
typedef struct {
    const double *speed;
    int32_t n_dgroup;
    int32_t pad;
    const double *nu_d, *decay, *chi_d;
    int64_t census_target;
} mcdc_kinetics;

/* multi-group materials (R3-R5, R30): arrays [n_mat][G]; S[n_mat][G][G], row = incident group.
 * Sigma_s = row sum of S; Sigma_c = Sigma_t - Sigma_s - Sigma_f.  Pass NULL for a continuous-energy problem.
 * kinetics != NULL makes the problem a time-dependent fixed-source one (mcdc_run_fixed_source / mcdc_run_cycle);
 * NULL: k-eigenvalue problem. */
typedef struct {
    int32_t n_mat, G;
    const double *sig_t, *sig_f, *nu, *chi, *S;
    const mcdc_kinetics *kinetics;
} mcdc_materials;

/* continuous-energy data (R19-R23): union grid [n_grid] (eV, strictly increasing), microscopic elastic /
 * capture / fission per nuclide [n_nuc][n_grid] (barns), materials as (nuclide, atom density 1/(b cm)) lists,
 * nu(E) = nu0 + nu1 E[MeV], Watt(a [MeV], b [1/MeV]).  Pass NULL for a multi-group problem.
 * search: 0 binary search on the grid, 1 hashed search (exponent/mantissa-keyed buckets, then bisection);
 * both return the same index. */
typedef struct {
    int32_t n_mat;
    int32_t n_grid;
    const double *grid;
    int32_t n_nuc;
    const double *nuc_A;
    const double *nuc_el, *nuc_c, *nuc_f;
    const int32_t *mat_nuc_off; /* [n_mat+1] */
    const int32_t *mat_nuc_id;
    const double *mat_nuc_dens;
    double nu0, nu1, watt_a, watt_b;
    int32_t search;
} mcdc_xs;

/* source: uniform in the box [lo,hi], isotropic or fixed direction; MG: group pdf [G]; CE: mono-energetic E
 * (eV) at time t (s).  Birth always consumes six draws (draw budget table of DESIGN.md). */
typedef struct {
    double lo[3], hi[3];
    int32_t isotropic;
    double dir[3];
    const double *group_pdf;
    double E, t;
} mcdc_source;

/* track-length flux tally (R17, R24): spatial bin of a particle = cell_bin[cell] (+ lat_bin[element] inside
 * the lattice, + lat2_bin[lat2_off[k] + element] inside second-level lattice k); MG: flux[bin][g]; CE: flux[bin][time
 * bin][energy bin] with explicit edges; time-dependent MG: flux[bin][time bin][g]. */
typedef struct {
    int32_t n_bins;
    const int32_t *cell_bin; /* [n_cell] */
    const int32_t *lat_bin;  /* [lat_ny][lat_nx] or NULL */
    int32_t n_t;
    const double *t_edges; /* [n_t+1], CE and time-dependent MG */
    int32_t n_e;
    const double *e_edges; /* [n_e+1], CE only */
    const int32_t *lat2_bin; /* [lat2_off[n_lat2]] or NULL */
} mcdc_tally_spec;

/* device resources handed in by the caller.
 * schedule: 0 (default) = event-based sweeps over dense particle queues regrouped by next event, one kernel per sweep
 *   (each particle's pending scatter / surface event is finished by the kernel that picks it up), and the persistent
 *   asynchronous kernel once at most persist_threshold particles are alive;
 *   1 = monolithic one-segment-per-launch kernel over every bank slot, no compaction (the paper's PAPER.md:51-55
 *   design, kept for the divergence comparison);
 *   2 = as 0, but the pending events are finished by two separate per-event kernels after every sweep (split
 *   per-event kernels).
 * persist_threshold: 0 = library default, negative = never use the persistent kernel, 2^31-1 = always. */
typedef struct {
    void *workspace; /* DEVICE pointer, 256-byte aligned */
    uint64_t workspace_bytes;
    void *stream; /* cudaStream_t */
    int32_t device;
    int32_t schedule;
    int32_t persist_threshold;
    int32_t reserved[3];
} mcdc_device;

typedef struct {
    int32_t mode; /* 0 MG, 1 CE */
    int32_t n_tally; /* length of flux_mean / flux_sdev */
    int32_t n_cycles; /* cycles run so far (fixed source: 1) */
    int32_t n_active;
    uint64_t bank_count; /* sites in the current source bank */
} mcdc_dims;

typedef struct {
    double *k_cycle;   /* [n_cycles] */
    double *flux_mean; /* [n_tally] */
    double *flux_sdev; /* [n_tally] */
    uint64_t *counters; /* [MCDC_N_COUNTERS] */
    double k_mean, k_sdev, leak_mean, leak_sdev;
} mcdc_tallies;

/* one record per event of a traced particle: location BEFORE the event (root cell c0, lattice element or -1,
 * local cell c1 or -1), surface hit (or -1; n_surf+k for lattice wall k), group / grid index, position and time
 * AFTER the move, flight distance d and flight energy E. */
typedef struct {
    uint64_t id;
    uint32_t cycle, seq;
    int32_t ev, c0, elem, c1, surf, gi;
    double x, y, z, d, E, t;
} mcdc_trace_rec;

/* fission-bank site (R5: the parent samples group and direction) */
typedef struct {
    double x, y, z, ux, uy, uz;
    int32_t g;
    int32_t pad;
} mcdc_site;

typedef struct mcdc_problem mcdc_problem;

/* bytes of device workspace needed for runs of up to n_particles nominal particles per cycle. */
int mcdc_workspace_bytes(const mcdc_geometry *geo, const mcdc_materials *mat, const mcdc_xs *xs,
                         const mcdc_tally_spec *tally, uint64_t n_particles, uint64_t *bytes);

/* validate + copy all inputs, build derived tables (cumulative scatter rows, chi CDF, macroscopic CE rows,
 * hash buckets, per-lattice-element boundary codes), upload them into the workspace.  Exactly one of mat / xs is
 * non-NULL.  Checked here: index ranges and monotone offset arrays, Sigma_s + Sigma_f <= Sigma_t, a strictly
 * increasing grid and edges, cell_bin + lat_bin < n_bins, the source time inside the time edges, and that the source
 * box lies inside the geometry (a 9 x 9 x 9 grid of its points must all be in a cell; MCDC_EGEOM otherwise). */
int mcdc_create(const mcdc_geometry *geo, const mcdc_materials *mat, const mcdc_xs *xs, const mcdc_source *src,
                const mcdc_tally_spec *tally, const mcdc_device *dev, uint64_t max_particles, mcdc_problem **out);

/* k-eigenvalue power iteration (R6, R7): n_inactive + n_active cycles of n_particles nominal
 * histories; cycle 0 samples the source, later cycles start from the fission bank with weight N/M. */
int mcdc_run_eigenvalue(mcdc_problem *p, uint64_t n_particles, int32_t n_inactive, int32_t n_active, uint64_t seed);

/* Eigenvalue problem: one power-iteration cycle (cycle 0 resets the run and samples the source); returns the cycle's
 * track-length k.  active != 0 accumulates the flux / leakage / k statistics.
 * Fixed-source problem (continuous energy or time-dependent multi-group): `cycle` = a census interval (time edge cycle
 * -> cycle + 1): the interval that holds the source time resets the run and samples the source; every later call must
 * name the next interval and starts from the census bank the previous call left (the particles that reached the time
 * edge, and delayed neutrons emitted in that interval), sorted by particle id and, with census_target > 0, combed.
 * Intervals called in order to the last one give the tallies of mcdc_run_fixed_source.  `active` is ignored. */
int mcdc_run_cycle(mcdc_problem *p, uint64_t n_particles, uint32_t cycle, int32_t active, uint64_t seed,
                   double *k_cycle);

/* host-buffer form of one cycle (the end-to-end path): uploads n_in source sites from HOST memory (NULL/0:
 * sample the source), transports them as cycle `cycle` with k_prev, downloads the produced fission bank
 * (at most max_out sites; *n_out = produced count) and this cycle's per-source-particle flux [n_tally]. */
int mcdc_run_cycle_host(mcdc_problem *p, uint64_t n_particles, uint32_t cycle, uint64_t seed, double k_prev,
                        const mcdc_site *sites_in, uint64_t n_in, mcdc_site *sites_out, uint64_t max_out,
                        uint64_t *n_out, double *flux_cycle, double *k_cycle, double *leak_cycle);

/* time-dependent fixed source (R24, R25): n_particles source particles and all their fission secondaries,
 * to the last time edge.  Continuous energy: one persistent launch (a census is a synchronisation point only).
 * Time-dependent multi-group: census interval by census interval (population control happens between them). */
int mcdc_run_fixed_source(mcdc_problem *p, uint64_t n_particles, uint64_t seed);

/* Physics options beyond the analog target-at-rest model ("free-gas scattering model
 * with constant cross-sections"; R35, R36).  Takes effect from the next run call; NULL restores the defaults.
 *   kT (eV): continuous-energy elastic collisions below 400 kT sample the target's thermal velocity (constant cross
 *     section free gas); 0 = every target at rest.  Ignored by multi-group problems.
 *   implicit_capture != 0: survival biasing.  Every particle carries its own weight; a collision removes the capture
 *     share (w <- w (Sigma_t - Sigma_c) / Sigma_t) and chooses among scatter / fission; a scattered particle whose weight
 *     fell below w_roulette survives with probability w / w_survive at weight w_survive (one extra draw).
 *     0 <= w_roulette <= w_survive is required (w_roulette = 0: no roulette). */
typedef struct {
    double kT;
    int32_t implicit_capture;
    int32_t pad;
    double w_roulette, w_survive;
} mcdc_physics;
int mcdc_set_physics(mcdc_problem *p, const mcdc_physics *phys);

/* weight balance of the last successful run, summed over its cycles (not normalised): out[0] weight started (source
 * particles and secondaries), [1] absorbed (capture, fission, and the capture share removed by implicit capture),
 * [2] leaked, [3] cut off at the last time edge, [4] killed by roulette, [5] gained by roulette survivors.
 * out[0] = out[1] + out[2] + out[3] + out[4] - out[5] up to rounding. */
int mcdc_get_balance(const mcdc_problem *p, double out[6]);

/* population entering each census interval of the last fixed-source run made interval by interval: counts[2k] particles
 * before and counts[2k+1] after the comb, weights[2k], [2k+1] their total weights; *n = intervals reported (<= max) */
int mcdc_get_census(const mcdc_problem *p, uint64_t *counts, double *weights, int32_t max, int32_t *n);

int mcdc_get_dims(const mcdc_problem *p, mcdc_dims *dims);
int mcdc_get_tallies(const mcdc_problem *p, mcdc_tallies *out);
/* current source bank (after a cycle: the sorted fission bank), at most max sites; returns the count via *n */
int mcdc_get_bank(const mcdc_problem *p, mcdc_site *out, uint64_t max, uint64_t *n);

/* record the events of particles first_id .. first_id+n_ids-1 (at most max_events each, per cycle) */
int mcdc_set_trace(mcdc_problem *p, uint64_t first_id, uint32_t n_ids, uint32_t max_events);
/* copies at most max records (ordered by cycle, id, seq); *n = records available */
int mcdc_get_trace(const mcdc_problem *p, mcdc_trace_rec *out, uint64_t max, uint64_t *n);

/* The per-particle random-number stream (R1, R2) evaluated on the GPU WITHOUT any device
 * memory from the caller: out[i] = draw number draw[i] of stream (seed, id[i], domain, cycle), bit for bit what
 * mcdc_test_draws (include/mcdc_test.h) returns, but no mcdc_problem and no workspace are needed.
 *
 * Who this is for.  Every other call of this library works inside a workspace the caller allocated on the device.  Some
 * callers have nothing to give and no way to get it: a checking tool that runs beside a simulation whose workspace was
 * sized to fill the GPU (cudaMalloc fails there); a plug-in running inside a host program whose memory pool owns all
 * device memory and whose rules keep plug-ins from allocating; code that runs at a point where allocating would stall
 * the whole device (cudaMalloc and cudaFree synchronise it).  Such a caller can still check that this GPU draws the same
 * numbers as the CPU: this call makes no cudaMalloc / cudaFree and calls no library routine that allocates device memory.
 *
 * How.  The device-side staging of id, draw and out (24 bytes per draw) lives in a fixed array inside the library's
 * device image, MCDC_NOALLOC_DRAWS_MAX entries long: 1.5 MiB that every GPU which loads the library holds until the
 * process exits, used or not.  n > MCDC_NOALLOC_DRAWS_MAX is refused with MCDC_EINVAL and a message (nothing is launched);
 * split larger requests into several calls.
 *
 * id, draw, out: HOST pointers, n entries each, owned by the caller (as everywhere in this header).  device: CUDA device
 * ordinal (0..63); it is made current for the duration of the call and the caller's current device is restored.
 * stream: a cudaStream_t of that device (NULL = the legacy default stream); the call returns after the stream has
 * finished the work, so out is ready on return.
 *
 * First call on a device: the library looks up the array's address on that device once and remembers it.  Make that
 * first call before starting any stream capture on the device.
 * Sharing: all calls, from all threads and streams, stage through the same array.  Calls into this entry point are
 * serialised by a lock inside the library, and each call overwrites every byte it later reads (nothing has to start at
 * zero, nothing is carried from one call to the next), so results never depend on earlier calls.  But the array is one
 * per GPU and process: if the work of two such calls could ever overlap on the GPU, they would race.
 * Errors: MCDC_EINVAL (device out of range, n too large, NULL pointer with n > 0), MCDC_ECUDA (any CUDA failure, text in
 * mcdc_last_error()).  n = 0 is a valid call that does nothing. */
#define MCDC_NOALLOC_DRAWS_MAX 65536
int mcdc_draws_noalloc(int32_t device, void *stream, uint64_t seed, uint32_t domain, uint32_t cycle, const uint64_t *id,
                       const uint32_t *draw, uint64_t n, double *out);

/* device time (ms, CUDA events on the library's stream) of the transport part of the last run call, and the
 * number of kernels it launched */
int mcdc_get_timing(const mcdc_problem *p, double *ms_transport, uint64_t *n_launches);

/* per-kernel-class device timing: when on, every launch is bracketed by a CUDA event pair on the library's
 * stream (costs a few microseconds per launch, so it is off for throughput runs).  mcdc_get_profile fills
 * ms[MCDC_N_PROFILE] and launches[MCDC_N_PROFILE] accumulated since mcdc_set_profile, and the number of segments
 * (= events) the sweep kernels ran in that time (the rest of the run's events ran in the persistent kernel). */
enum { MCDC_PROF_SWEEP = 0, MCDC_PROF_SCATTER, MCDC_PROF_SURFACE, MCDC_PROF_PERSIST, MCDC_PROF_SEGMENT, MCDC_PROF_BANK,
       MCDC_N_PROFILE };
int mcdc_set_profile(mcdc_problem *p, int32_t on);
int mcdc_get_profile(const mcdc_problem *p, double *ms, uint64_t *launches, uint64_t *sweep_events);

/* identity of the sources this library was compiled from: the first 16 hex digits of a sha256 over csrc/ and this header,
 * put in by the build (binding.build); "unknown" for a hand build without -DMCDC_BUILD_ID.  Measurement files that
 * describe a build (profiles/r03_counts.csv) carry the same string; static storage, never NULL. */
const char *mcdc_build_id(void);

void mcdc_destroy(mcdc_problem *p);
const char *mcdc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
