/* mcdc_oracle.h -- interface of the CPU ORACLE (test infrastructure, not the product).
 *
 * A plain, slow, history-based float64 implementation of the Monte Carlo neutron transport loop
 * named by arxiv 2501.05440 ("continuous and multi-group energy neutron transport
 * physics with constructive solid geometry modeling using surface tracking ... k-eigenvalue ...
 * fully dynamic simulations ... replicable random number generation"; PAPER.md:51 one "segment"
 * = one event; PAPER.md:124 inactive/active cycles; PAPER.md:134 time-dependent fixed source).
 * The paper gives no formulas; every step follows the readings listed in DESIGN.md section 3
 * (= SURVEY.md 8c).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this library.  It shares no code, header, table generator or helper
 * with the CUDA library under paper_2501_05440_b200/csrc.
 *
 * Parity pins: tests/test_oracle_*.py.  Unpinned in absolute terms (no closed form, the paper
 * prints no k or flux): heterogeneous C3/C4/C5 k and flux values -- "parity unpinned" for those
 * absolute values; they are pinned only through the reductions to closed forms listed in DESIGN.md.
 */
#ifndef MCDC_ORACLE_H
#define MCDC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t mode; /* 0 multi-group, 1 continuous energy */
    /* geometry */
    int32_t n_surf;
    const int32_t *surf_type;
    const double *surf_param; /* [n_surf][4] */
    const int32_t *surf_bc;
    int32_t n_cell;
    const int32_t *cell_surf_off, *cell_surf_id, *cell_surf_sense;
    const int32_t *cell_fill_type, *cell_fill, *cell_bin;
    int32_t n_univ;
    const int32_t *univ_cell_off;
    int32_t has_lat;
    double lat_x0, lat_y0, lat_px, lat_py;
    int32_t lat_nx, lat_ny;
    const int32_t *lat_univ, *lat_bin; /* [ny][nx] */
    /* second-level lattices (R37; "fully 3D C5G7": assemblies are lattices of pin lattices): a cell of a
     * lattice element's universe with cell_fill_type 2 is filled by inner lattice k = cell_fill, nx[k] x ny[k] elements
     * of pitch px[k], py[k], centred on the origin of that universe's coordinates; the universes and tally-bin offsets
     * of its elements are lat2_univ / lat2_bin [lat2_off[k] + iy nx[k] + ix].  At most one such cell per universe. */
    int32_t n_lat2;
    const int32_t *lat2_nx, *lat2_ny;
    const double *lat2_px, *lat2_py;
    const int32_t *lat2_off; /* [n_lat2+1] */
    const int32_t *lat2_univ, *lat2_bin;
    int32_t n_bins;
    int32_t n_mat;
    /* multi-group */
    int32_t G;
    const double *sig_t, *sig_f, *nu, *chi; /* [n_mat][G] */
    const double *S;                        /* [n_mat][G][G], row = incident group */
    /* continuous energy */
    int32_t n_grid;
    const double *grid;
    int32_t n_nuc;
    const double *nuc_A;
    const double *nuc_el, *nuc_c, *nuc_f; /* [n_nuc][n_grid] barns */
    const int32_t *mat_nuc_off, *mat_nuc_id;
    const double *mat_nuc_dens;
    double nu0, nu1, watt_a, watt_b;
    int32_t n_t;
    const double *t_edges; /* [n_t+1] */
    int32_t n_e;
    const double *e_edges; /* [n_e+1] */
    /* source */
    double src_lo[3], src_hi[3];
    int32_t src_iso;
    double src_dir[3];
    const double *src_group_pdf; /* [G] */
    double src_E, src_t;
    /* free-gas thermal scattering (R35): temperature kT in eV, 0 = target at rest */
    double kT;
    /* implicit capture / survival biasing with weight roulette (R36) */
    int32_t implicit_capture;
    double w_roulette, w_survive;
    /* time-dependent multi-group with delayed-neutron precursors and census population control (R38-R40;
     * PAPER.md:31 "fully dynamic simulations"): td != 0 switches it on for a multi-group problem.  speed[G] cm/s;
     * n_dgroup precursor groups per material: nu_d[n_mat][n_dgroup][G] delayed yields (nu above = the prompt yield),
     * decay[n_mat][n_dgroup] 1/s, chi_d[n_mat][n_dgroup][G] emission spectra; time edges t_edges[n_t+1] above (every
     * edge is a census); census_target > 0: the population entering each census interval but the first is combed to
     * that many particles. */
    int32_t td, n_dgroup;
    const double *speed, *nu_d, *decay, *chi_d;
    int64_t census_target;
} orc_input;

typedef struct {
    uint64_t id;
    uint32_t cycle, seq;
    int32_t ev, c0, elem, c1, surf, gi;
    double x, y, z, d, E, t;
} orc_trace_rec;

typedef struct {
    double x, y, z, ux, uy, uz;
    int32_t g;
    int32_t pad;
} orc_site;

typedef struct orc_problem orc_problem;

enum { ORC_EV_SCATTER = 1, ORC_EV_FISSION, ORC_EV_CAPTURE, ORC_EV_TRANSMIT, ORC_EV_REFLECT,
       ORC_EV_LEAK, ORC_EV_LATTICE, ORC_EV_TIME_EDGE, ORC_EV_CUTOFF, ORC_EV_LOST };
/* counters[0] tracks started, [1..10] events by type, [11] children banked, [12] bank high-water */
#define ORC_N_COUNTERS 16

orc_problem *orc_create(const orc_input *in);
void orc_destroy(orc_problem *p);
int orc_set_trace(orc_problem *p, uint64_t first_id, uint64_t n_ids, uint64_t max_records);
int orc_run_eigenvalue(orc_problem *p, uint64_t n_particles, int n_inactive, int n_active, uint64_t seed);
/* all-core timing variant (bench.py cpu_baseline): n_threads contiguous id ranges, joined in thread order */
int orc_run_eigenvalue_mt(orc_problem *p, uint64_t n_particles, int n_inactive, int n_active, uint64_t seed, int n_threads);
int orc_run_fixed_source(orc_problem *p, uint64_t n_particles, uint64_t seed);
/* time-dependent multi-group fixed source (td != 0), census interval by census interval (R38-R40) */
int orc_run_td(orc_problem *p, uint64_t n_particles, uint64_t seed);
/* population entering each census interval of the last orc_run_td: out[2k] = particles before, out[2k+1] after the
 * comb (equal without population control); weights[2k], [2k+1] = their total weights; returns the number of intervals */
int orc_get_census(const orc_problem *p, uint64_t *counts, double *weights, int max_intervals);
/* the comb itself (R40) on plain arrays: M weights in bank order, N teeth, offset draw xi in (0,1): copies[i] = number
 * of teeth that fall on particle i; returns the tooth spacing */
double orc_comb(const double *w, uint64_t M, uint64_t N, double xi, uint32_t *copies);
/* results; arrays sized by the caller: k_cycle[n_cycles], flux_*[n_tally], counters[ORC_N_COUNTERS] */
int64_t orc_n_tally(const orc_problem *p);
int orc_get_results(const orc_problem *p, double *k_cycle, double *k_mean, double *k_sdev, double *flux_mean,
                    double *flux_sdev, double *leak_mean, double *leak_sdev, uint64_t *counters);
/* weight balance of the last run, summed over all its cycles (not normalised): out[0] source weight started,
 * [1] absorbed (analog capture / fission: the particle's weight; implicit capture: the weight removed at each
 * collision), [2] leaked, [3] cut off at the last time edge, [4] killed by roulette, [5] gained by roulette survivors.
 * Identity (to rounding): out[0] = out[1] + out[2] + out[3] + out[4] - out[5]. */
void orc_get_balance(const orc_problem *p, double out[6]);
/* free-gas elastic collision (R35) with the draws taken from stream (seed, id, domain 0, cycle) starting at *ctr */
void orc_free_gas(double E, const double u[3], double A, double kT, uint64_t seed, uint64_t id, uint32_t cycle, uint32_t *ctr,
                  double *E_out, double u_out[3]);
uint64_t orc_get_trace(const orc_problem *p, orc_trace_rec *out, uint64_t max);
uint64_t orc_get_bank(const orc_problem *p, orc_site *out, uint64_t max);

/* unit-level entry points used by the pins */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_draw(uint64_t seed, uint64_t id, uint32_t domain, uint32_t cycle, uint32_t draw_index);
uint64_t orc_child_id(uint64_t seed, uint64_t parent_id, uint32_t parent_ctr, uint32_t j);
int32_t orc_grid_index(const orc_problem *p, double E);
/* out[0] = Sigma_t, out[1..] = cumulative thresholds [el_1..el_n, fission, capture] of material m */
int orc_ce_xs(const orc_problem *p, int32_t m, double E, double *out);
/* loc = {c0, elem, c1}; returns 0 or -1 (no cell) */
int orc_locate(const orc_problem *p, const double x[3], const double u[3], int32_t last_surf, int32_t loc[3]);
/* nearest boundary from a located point: returns distance, *surf = global surface id or n_surf+k for lattice wall k */
double orc_distance(const orc_problem *p, const double x[3], const double u[3], const int32_t loc[3],
                    int32_t last_surf, int32_t *surf);
void orc_iso_dir(double xi_mu, double xi_phi, double out[3]);
/* elastic target-at-rest: in E,u[3],A,xi1,xi2 -> out E', u'[3] (before energy clamping) */
void orc_elastic(double E, const double u[3], double A, double xi_mu, double xi_phi, double *E_out, double u_out[3]);
double orc_watt(double a, double b, double xi1, double xi2, double xi3, double xi4);
double orc_speed(double E_eV);

#ifdef __cplusplus
}
#endif
#endif
