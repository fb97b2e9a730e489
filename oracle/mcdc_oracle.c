/* mcdc_oracle.c -- CPU ORACLE (test infrastructure, not the product).  See mcdc_oracle.h.
 *
 * History-based: one particle is followed from birth to death, then the next (SURVEY.md 8c
 * "Algorithm"; PAPER.md:51 one loop iteration = one "segment" = one event).  float64 everywhere
 * (PAPER.md:140).  No blocking, fusion or reordering: each function is the reading of DESIGN.md
 * section 3 written out.  Rule numbers "R<n>" below are the rows of that table.
 */
#include "mcdc_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define TWO_PI 6.283185307179586
#define HALF_PI 1.5707963267948966
#define C_LIGHT 2.99792458e10    /* cm/s (R23) */
#define MN_C2_EV 939.56542052e6  /* neutron rest energy, eV (R23) */
#define MAX_SEGMENTS 1000000u    /* lost-particle guard (R11) */
#define SQRT_PI 1.7724538509055159
#define FREE_GAS_LIMIT 400.0     /* free gas below 400 kT, target at rest above (R35) */

typedef struct {
    double x, y, z, ux, uy, uz, w, E, t;
    int32_t g, c0, elem, c1, last_surf, tbin, alive;
    int32_t resumed; /* taken from a census bank: already counted as a started track */
    uint32_t ctr, nseg;
    uint64_t id;
} particle;

struct orc_problem {
    orc_input in;
    /* derived MG tables */
    double *sig_s, *cumS, *cumchi, *nusf, *src_cum;
    /* derived CE tables: per material, ncol = n_nuclides + 2 columns [el_1..el_n, fission, capture] */
    int32_t *ce_ncol;
    double **ce_col;
    /* run state */
    uint64_t seed;
    uint32_t cycle;
    double k_prev, w_cycle;
    int fixed;
    /* per-cycle tallies */
    double *flux_c, k_num, leak_c;
    double balance[6]; /* see orc_get_balance */
    /* accumulated results */
    int n_cycles, n_active_done;
    double *k_cycle, *flux_acc, *flux_acc2, leak_acc, leak_acc2, k_acc, k_acc2;
    uint64_t counters[ORC_N_COUNTERS];
    /* banks */
    orc_site *bank, *newbank;
    uint64_t n_bank, n_newbank, cap_bank;
    particle *stack;
    uint64_t n_stack, cap_stack;
    /* time-dependent multi-group (R38-R40): delayed-spectrum / yield tables, the census banks (one per interval) */
    double *cumchi_d, *cum_nu;
    int census_stop;
    particle **cbank;
    uint64_t *n_cbank, *cap_cbank;
    uint64_t census_counts[2 * 64];
    double census_weights[2 * 64];
    int n_census;
    /* trace */
    uint64_t tr_first, tr_n, tr_max, tr_count;
    orc_trace_rec *trace;
    int error;
};

/* ------------------------------------------------------------------ RNG (R9, R10) */
/* Philox4x32-10 (Salmon et al., SC'11): 10 rounds of two 32x32->64 multiplies and key bumps. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; r++) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* draw number `draw_index` of stream (seed, id, domain, cycle): counter = (id_lo, id_hi,
 * domain<<24 | cycle, draw_index/2); the block's four words give two u64 (words 1:0 and 3:2);
 * xi = ((u >> 11) + 0.5) * 2^-53, never 0 or 1 (R9). */
double orc_draw(uint64_t seed, uint64_t id, uint32_t domain, uint32_t cycle, uint32_t draw_index)
{
    uint32_t ctr[4] = {(uint32_t)id, (uint32_t)(id >> 32), (domain << 24) | cycle, draw_index >> 1};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t o[4];
    orc_philox4x32_10(ctr, key, o);
    uint64_t u = (draw_index & 1u) ? (((uint64_t)o[3] << 32) | o[2]) : (((uint64_t)o[1] << 32) | o[0]);
    return ((double)(u >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* id of secondary j of a fission by `parent_id` whose draw counter was `parent_ctr` after the
 * multiplicity draw: first u64 of the domain-1 block (parent_lo, parent_hi, 1<<24 | j, parent_ctr) (R10). */
uint64_t orc_child_id(uint64_t seed, uint64_t parent_id, uint32_t parent_ctr, uint32_t j)
{
    uint32_t ctr[4] = {(uint32_t)parent_id, (uint32_t)(parent_id >> 32), (1u << 24) | j, parent_ctr};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t o[4];
    orc_philox4x32_10(ctr, key, o);
    return ((uint64_t)o[1] << 32) | o[0];
}

static double draw(const orc_problem *p, particle *q)
{
    return orc_draw(p->seed, q->id, 0u, p->cycle, q->ctr++);
}

/* ------------------------------------------------------------------ sampling helpers */
/* isotropic direction (R8) */
void orc_iso_dir(double xi_mu, double xi_phi, double out[3])
{
    double mu = 2.0 * xi_mu - 1.0;
    double phi = TWO_PI * xi_phi;
    double s = sqrt(1.0 - mu * mu);
    out[0] = s * cos(phi);
    out[1] = s * sin(phi);
    out[2] = mu;
}

/* first index with cum[i] > v, else n-1 (R3: compare xi*total against cumulative thresholds) */
static int32_t pick(const double *cum, int32_t n, double v)
{
    for (int32_t i = 0; i < n; i++)
        if (cum[i] > v) return i;
    return n - 1;
}

double orc_speed(double E)
{
    return C_LIGHT * sqrt(2.0 * E / MN_C2_EV);
}

/* Watt spectrum, rejection-free (R22): Maxwellian W (T=a) then the shift; energies in MeV */
double orc_watt(double a, double b, double xi1, double xi2, double xi3, double xi4)
{
    double c = cos(HALF_PI * xi3);
    double W = -a * (log(xi1) + log(xi2) * c * c);
    return W + 0.25 * a * a * b + (2.0 * xi4 - 1.0) * sqrt(a * a * b * W);
}

/* elastic scattering off a target at rest (SURVEY.md 8c CE paragraph, R21) */
void orc_elastic(double E, const double u[3], double A, double xi_mu, double xi_phi, double *E_out, double u_out[3])
{
    double mu_cm = 2.0 * xi_mu - 1.0;
    double den = A * A + 2.0 * A * mu_cm + 1.0;
    double mu = 0.0;
    if (den > 0.0) mu = (1.0 + A * mu_cm) / sqrt(den);
    *E_out = E * den / ((A + 1.0) * (A + 1.0));
    double phi = TWO_PI * xi_phi;
    double cp = cos(phi), sp = sin(phi);
    double s2 = 1.0 - mu * mu;
    double s = s2 > 0.0 ? sqrt(s2) : 0.0;
    double a2 = 1.0 - u[2] * u[2];
    double o[3];
    if (a2 < 1e-10) {
        o[0] = s * cp;
        o[1] = s * sp;
        o[2] = u[2] > 0.0 ? mu : -mu;
    } else {
        double r = sqrt(a2);
        o[0] = mu * u[0] + s * (u[0] * u[2] * cp - u[1] * sp) / r;
        o[1] = mu * u[1] + s * (u[1] * u[2] * cp + u[0] * sp) / r;
        o[2] = mu * u[2] - s * r * cp;
    }
    double nrm = sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]);
    u_out[0] = o[0] / nrm;
    u_out[1] = o[1] / nrm;
    u_out[2] = o[2] / nrm;
}

/* rotate unit vector u by polar cosine mu and azimuth phi (R21 formula) */
static void rotate(const double u[3], double mu, double phi, double o[3])
{
    double cp = cos(phi), sp = sin(phi);
    double s2 = 1.0 - mu * mu;
    double s = s2 > 0.0 ? sqrt(s2) : 0.0;
    double a2 = 1.0 - u[2] * u[2];
    if (a2 < 1e-10) {
        o[0] = s * cp; o[1] = s * sp; o[2] = u[2] > 0.0 ? mu : -mu;
    } else {
        double r = sqrt(a2);
        o[0] = mu * u[0] + s * (u[0] * u[2] * cp - u[1] * sp) / r;
        o[1] = mu * u[1] + s * (u[1] * u[2] * cp + u[0] * sp) / r;
        o[2] = mu * u[2] - s * r * cp;
    }
    double nrm = sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]);
    o[0] /= nrm; o[1] /= nrm; o[2] /= nrm;
}

/* Free-gas elastic scattering with a constant cross section ("free-gas scattering model with constant
 * cross-sections"; R35).  Velocities in units where speed = sqrt(E).  The target speed x (in units of sqrt(kT/A))
 * and the cosine mu between target and neutron are drawn from p(x, mu) ~ |v_n - v_T| x^2 exp(-x^2) by the classic
 * two-branch scheme: with probability alpha = 1 / (1 + sqrt(pi) y / 2), y = sqrt(A E / kT), x^2 = -ln(xi1 xi2);
 * otherwise x^2 = -ln xi1 - ln xi2 cos^2(pi xi4 / 2); mu = 2 xi - 1; accepted with probability
 * sqrt(y^2 + x^2 - 2 x y mu) / (x + y).  Draws per trial, in order: xi1, xi2, branch, [xi4], mu, accept.  Then the
 * target direction (azimuth 2 pi xi around the neutron's), and an isotropic direction of the relative velocity in
 * the centre-of-mass frame (2 draws). */
void orc_free_gas(double E, const double u[3], double A, double kT, uint64_t seed, uint64_t id, uint32_t cycle, uint32_t *ctr,
                  double *E_out, double u_out[3])
{
    double y = sqrt(A * E / kT);
    double alpha = 1.0 / (1.0 + SQRT_PI * y / 2.0);
    double x2, x, mu;
    for (;;) {
        double r1 = orc_draw(seed, id, 0u, cycle, (*ctr)++), r2 = orc_draw(seed, id, 0u, cycle, (*ctr)++);
        if (orc_draw(seed, id, 0u, cycle, (*ctr)++) < alpha) x2 = -log(r1 * r2);
        else {
            double c = cos(HALF_PI * orc_draw(seed, id, 0u, cycle, (*ctr)++));
            x2 = -log(r1) - log(r2) * c * c;
        }
        x = sqrt(x2);
        mu = 2.0 * orc_draw(seed, id, 0u, cycle, (*ctr)++) - 1.0;
        double acc = sqrt(y * y + x2 - 2.0 * x * y * mu) / (x + y);
        if (orc_draw(seed, id, 0u, cycle, (*ctr)++) < acc) break;
    }
    double ut[3];
    rotate(u, mu, TWO_PI * orc_draw(seed, id, 0u, cycle, (*ctr)++), ut);
    double sn = sqrt(E), st = x * sqrt(kT / A);
    double vn[3], vc[3], vr[3], o[3];
    for (int k = 0; k < 3; k++) {
        vn[k] = sn * u[k];
        vc[k] = (vn[k] + A * st * ut[k]) / (A + 1.0);
        vr[k] = vn[k] - vc[k];
    }
    double s = sqrt(vr[0] * vr[0] + vr[1] * vr[1] + vr[2] * vr[2]);
    double a = orc_draw(seed, id, 0u, cycle, (*ctr)++), b = orc_draw(seed, id, 0u, cycle, (*ctr)++);
    orc_iso_dir(a, b, o);
    double v[3] = {vc[0] + s * o[0], vc[1] + s * o[1], vc[2] + s * o[2]};
    double e = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    double nv = sqrt(e);
    *E_out = e;
    u_out[0] = v[0] / nv; u_out[1] = v[1] / nv; u_out[2] = v[2] / nv;
}

/* ------------------------------------------------------------------ geometry (R11-R14) */
enum { S_PLANE_X, S_PLANE_Y, S_PLANE_Z, S_PLANE, S_CYL_X, S_CYL_Y, S_CYL_Z, S_SPHERE };

/* f(x) of surface s; sense +1 where f > 0 */
static double surf_f(const orc_problem *p, int32_t s, const double x[3])
{
    const double *q = p->in.surf_param + 4 * s;
    switch (p->in.surf_type[s]) {
    case S_PLANE_X: return x[0] - q[0];
    case S_PLANE_Y: return x[1] - q[0];
    case S_PLANE_Z: return x[2] - q[0];
    case S_PLANE: return q[0] * x[0] + q[1] * x[1] + q[2] * x[2] - q[3];
    case S_CYL_X: { double a = x[1] - q[0], b = x[2] - q[1]; return a * a + b * b - q[2] * q[2]; }
    case S_CYL_Y: { double a = x[0] - q[0], b = x[2] - q[1]; return a * a + b * b - q[2] * q[2]; }
    case S_CYL_Z: { double a = x[0] - q[0], b = x[1] - q[1]; return a * a + b * b - q[2] * q[2]; }
    default: { double a = x[0] - q[0], b = x[1] - q[1], c = x[2] - q[2]; return a * a + b * b + c * c - q[3] * q[3]; }
    }
}

/* (unnormalised) outward normal = grad f */
static void surf_normal(const orc_problem *p, int32_t s, const double x[3], double n[3])
{
    const double *q = p->in.surf_param + 4 * s;
    n[0] = n[1] = n[2] = 0.0;
    switch (p->in.surf_type[s]) {
    case S_PLANE_X: n[0] = 1.0; break;
    case S_PLANE_Y: n[1] = 1.0; break;
    case S_PLANE_Z: n[2] = 1.0; break;
    case S_PLANE: n[0] = q[0]; n[1] = q[1]; n[2] = q[2]; break;
    case S_CYL_X: n[1] = x[1] - q[0]; n[2] = x[2] - q[1]; break;
    case S_CYL_Y: n[0] = x[0] - q[0]; n[2] = x[2] - q[1]; break;
    case S_CYL_Z: n[0] = x[0] - q[0]; n[1] = x[1] - q[1]; break;
    default: n[0] = x[0] - q[0]; n[1] = x[1] - q[1]; n[2] = x[2] - q[2]; break;
    }
}

/* side of surface s the particle is on: the side being entered if it sits on s (R11) */
static int sense_of(const orc_problem *p, int32_t s, const double x[3], const double u[3], int32_t last_surf)
{
    if (s == last_surf) {
        double n[3];
        surf_normal(p, s, x, n);
        return (u[0] * n[0] + u[1] * n[1] + u[2] * n[2]) > 0.0 ? +1 : -1;
    }
    return surf_f(p, s, x) > 0.0 ? +1 : -1;
}

/* first cell of universe `univ` whose every (surface, sense) matches; -1 if none */
static int32_t find_cell(const orc_problem *p, int32_t univ, const double x[3], const double u[3], int32_t last_surf)
{
    const orc_input *in = &p->in;
    for (int32_t c = in->univ_cell_off[univ]; c < in->univ_cell_off[univ + 1]; c++) {
        int ok = 1;
        for (int32_t k = in->cell_surf_off[c]; k < in->cell_surf_off[c + 1]; k++)
            if (sense_of(p, in->cell_surf_id[k], x, u, last_surf) != in->cell_surf_sense[k]) { ok = 0; break; }
        if (ok) return c;
    }
    return -1;
}

/* Location inside lattices: `elem` packs the element of the (first-level) lattice in its low 20 bits and, inside a
 * second-level lattice (R37), that lattice's element + 1 in the bits above; -1 = not in a lattice. */
#define OUTER(e) ((e) & 0xfffff)
#define INNER(e) (((e) >> 20) - 1)

/* coordinates centred on first-level element `outer`, recomputed from the global position every time (R14) */
static void outer_coords(const orc_problem *p, int32_t outer, const double x[3], double xl[3])
{
    const orc_input *in = &p->in;
    int32_t ix = outer % in->lat_nx, iy = outer / in->lat_nx;
    xl[0] = x[0] - (in->lat_x0 + (ix + 0.5) * in->lat_px);
    xl[1] = x[1] - (in->lat_y0 + (iy + 0.5) * in->lat_py);
    xl[2] = x[2];
}

/* the cell of first-level element `outer`'s universe that a second-level lattice fills (-1: none) */
static int32_t mid_cell(const orc_problem *p, int32_t outer)
{
    const orc_input *in = &p->in;
    int32_t un = in->lat_univ[outer];
    for (int32_t c = in->univ_cell_off[un]; c < in->univ_cell_off[un + 1]; c++)
        if (in->cell_fill_type[c] == 2) return c;
    return -1;
}

/* lower-left corner of second-level lattice k in its universe's coordinates: centred on the origin (R37) */
static double lat2_x0(const orc_input *in, int32_t k) { return -0.5 * (in->lat2_nx[k] * in->lat2_px[k]); }
static double lat2_y0(const orc_input *in, int32_t k) { return -0.5 * (in->lat2_ny[k] * in->lat2_py[k]); }

/* coordinates centred on element `inner` of second-level lattice k, from first-level-element coordinates xo */
static void inner_coords(const orc_problem *p, int32_t k, int32_t inner, const double xo[3], double xl[3])
{
    const orc_input *in = &p->in;
    int32_t ix = inner % in->lat2_nx[k], iy = inner / in->lat2_nx[k];
    xl[0] = xo[0] - (lat2_x0(in, k) + (ix + 0.5) * in->lat2_px[k]);
    xl[1] = xo[1] - (lat2_y0(in, k) + (iy + 0.5) * in->lat2_py[k]);
    xl[2] = xo[2];
}

/* element-local coordinates of the innermost level of `elem` */
static void local_coords(const orc_problem *p, int32_t elem, const double x[3], double xl[3])
{
    double xo[3];
    outer_coords(p, OUTER(elem), x, xo);
    if (INNER(elem) >= 0) inner_coords(p, p->in.cell_fill[mid_cell(p, OUTER(elem))], INNER(elem), xo, xl);
    else { xl[0] = xo[0]; xl[1] = xo[1]; xl[2] = xo[2]; }
}

/* cell of first-level element `outer` that holds the point xo (first-level-element coordinates), descending into a
 * second-level lattice where a cell is filled by one: *elem = packed location, returns the material cell or -1.  The
 * second-level element index is found by floor and CLAMPED to the lattice's range (R37): the enclosing cell has
 * already established that the point is inside the lattice, and a point on the lattice's rim (a particle that has just
 * crossed a first-level wall) must not fall off it by a rounding error. */
static int32_t descend(const orc_problem *p, int32_t outer, const double xo[3], const double u[3], int32_t last_surf,
                       int32_t *elem)
{
    const orc_input *in = &p->in;
    *elem = outer;
    int32_t c = find_cell(p, in->lat_univ[outer], xo, u, last_surf);
    if (c < 0 || in->cell_fill_type[c] != 2) return c;
    int32_t k = in->cell_fill[c];
    int32_t ix = (int32_t)floor((xo[0] - lat2_x0(in, k)) / in->lat2_px[k]);
    int32_t iy = (int32_t)floor((xo[1] - lat2_y0(in, k)) / in->lat2_py[k]);
    if (ix < 0) ix = 0;
    if (iy < 0) iy = 0;
    if (ix > in->lat2_nx[k] - 1) ix = in->lat2_nx[k] - 1;
    if (iy > in->lat2_ny[k] - 1) iy = in->lat2_ny[k] - 1;
    int32_t inner = iy * in->lat2_nx[k] + ix;
    double xl[3];
    inner_coords(p, k, inner, xo, xl);
    *elem = outer | ((inner + 1) << 20);
    return find_cell(p, in->lat2_univ[in->lat2_off[k] + inner], xl, u, last_surf);
}

int orc_locate(const orc_problem *p, const double x[3], const double u[3], int32_t last_surf, int32_t loc[3])
{
    const orc_input *in = &p->in;
    loc[0] = find_cell(p, 0, x, u, last_surf);
    loc[1] = loc[2] = -1;
    if (loc[0] < 0) return -1;
    if (in->cell_fill_type[loc[0]] == 1) {
        int32_t ix = (int32_t)floor((x[0] - in->lat_x0) / in->lat_px);
        int32_t iy = (int32_t)floor((x[1] - in->lat_y0) / in->lat_py);
        if (ix < 0 || iy < 0 || ix >= in->lat_nx || iy >= in->lat_ny) return -1;
        double xo[3];
        outer_coords(p, iy * in->lat_nx + ix, x, xo);
        loc[2] = descend(p, iy * in->lat_nx + ix, xo, u, last_surf, &loc[1]);
        if (loc[2] < 0) return -1;
    }
    return 0;
}

/* positive ray distance to surface s (INFINITY = miss); on_surf: particle sits on s (R11-R13) */
static double surf_distance(const orc_problem *p, int32_t s, const double x[3], const double u[3], int on_surf)
{
    const double *q = p->in.surf_param + 4 * s;
    int typ = p->in.surf_type[s];
    double d;
    if (typ <= S_PLANE) {
        if (on_surf) return INFINITY;
        double num, den;
        if (typ == S_PLANE_X) { num = q[0] - x[0]; den = u[0]; }
        else if (typ == S_PLANE_Y) { num = q[0] - x[1]; den = u[1]; }
        else if (typ == S_PLANE_Z) { num = q[0] - x[2]; den = u[2]; }
        else { num = q[3] - (q[0] * x[0] + q[1] * x[1] + q[2] * x[2]); den = q[0] * u[0] + q[1] * u[1] + q[2] * u[2]; }
        if (den == 0.0) return INFINITY;
        d = num / den;
        return d > 0.0 ? d : INFINITY;
    }
    double a, k, c;
    if (typ == S_SPHERE) {
        double dx = x[0] - q[0], dy = x[1] - q[1], dz = x[2] - q[2];
        a = 1.0;
        k = dx * u[0] + dy * u[1] + dz * u[2];
        c = dx * dx + dy * dy + dz * dz - q[3] * q[3];
    } else {
        int i0 = typ == S_CYL_X ? 1 : 0, i1 = typ == S_CYL_Z ? 1 : 2;
        double da = x[i0] - q[0], db = x[i1] - q[1];
        a = u[i0] * u[i0] + u[i1] * u[i1];
        k = da * u[i0] + db * u[i1];
        c = da * da + db * db - q[2] * q[2];
    }
    if (a == 0.0) return INFINITY;
    if (on_surf) { /* c is exactly 0: roots 0 and -2k/a; only the far root, only when heading inward */
        if (k >= 0.0) return INFINITY;
        d = -2.0 * k / a;
        return d > 0.0 ? d : INFINITY;
    }
    double disc = k * k - a * c;
    if (disc < 0.0) return INFINITY;
    double sq = sqrt(disc);
    d = c < 0.0 ? (-k + sq) / a : (-k - sq) / a;
    return d > 0.0 ? d : INFINITY;
}

/* nearest boundary of the current location; candidates in the order: root-cell surfaces, [surfaces of the cell a
 * second-level lattice fills,] local-cell surfaces, [second-level lattice walls (-x,+x,-y,+y), codes n_surf+4..7,]
 * first-level lattice walls (-x,+x,-y,+y), codes n_surf+0..3; ties keep the first (R12, R14, R37) */
double orc_distance(const orc_problem *p, const double x[3], const double u[3], const int32_t loc[3],
                    int32_t last_surf, int32_t *surf)
{
    const orc_input *in = &p->in;
    double best = INFINITY;
    *surf = -1;
    for (int32_t k = in->cell_surf_off[loc[0]]; k < in->cell_surf_off[loc[0] + 1]; k++) {
        int32_t s = in->cell_surf_id[k];
        double d = surf_distance(p, s, x, u, s == last_surf);
        if (d < best) { best = d; *surf = s; }
    }
    if (loc[1] >= 0) {
        double xl[3], xo[3];
        outer_coords(p, OUTER(loc[1]), x, xo);
        local_coords(p, loc[1], x, xl);
        if (INNER(loc[1]) >= 0) {
            int32_t mid = mid_cell(p, OUTER(loc[1]));
            for (int32_t k = in->cell_surf_off[mid]; k < in->cell_surf_off[mid + 1]; k++) {
                int32_t s = in->cell_surf_id[k];
                double d = surf_distance(p, s, xo, u, s == last_surf);
                if (d < best) { best = d; *surf = s; }
            }
        }
        for (int32_t k = in->cell_surf_off[loc[2]]; k < in->cell_surf_off[loc[2] + 1]; k++) {
            int32_t s = in->cell_surf_id[k];
            double d = surf_distance(p, s, xl, u, s == last_surf);
            if (d < best) { best = d; *surf = s; }
        }
        if (INNER(loc[1]) >= 0) {
            /* second-level walls, in first-level-element coordinates: only the wall ahead, never the outermost ones */
            int32_t k2 = in->cell_fill[mid_cell(p, OUTER(loc[1]))];
            int32_t jx = INNER(loc[1]) % in->lat2_nx[k2], jy = INNER(loc[1]) / in->lat2_nx[k2];
            if (u[0] < 0.0 && jx > 0) {
                double d = (lat2_x0(in, k2) + jx * in->lat2_px[k2] - xo[0]) / u[0];
                if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 4; }
            }
            if (u[0] > 0.0 && jx + 1 < in->lat2_nx[k2]) {
                double d = (lat2_x0(in, k2) + (jx + 1) * in->lat2_px[k2] - xo[0]) / u[0];
                if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 5; }
            }
            if (u[1] < 0.0 && jy > 0) {
                double d = (lat2_y0(in, k2) + jy * in->lat2_py[k2] - xo[1]) / u[1];
                if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 6; }
            }
            if (u[1] > 0.0 && jy + 1 < in->lat2_ny[k2]) {
                double d = (lat2_y0(in, k2) + (jy + 1) * in->lat2_py[k2] - xo[1]) / u[1];
                if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 7; }
            }
        }
        int32_t ix = OUTER(loc[1]) % in->lat_nx, iy = OUTER(loc[1]) / in->lat_nx;
        /* only the wall ahead on each axis; the lattice's outermost walls are never events */
        if (u[0] < 0.0 && ix > 0) {
            double d = (in->lat_x0 + ix * in->lat_px - x[0]) / u[0];
            if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 0; }
        }
        if (u[0] > 0.0 && ix + 1 < in->lat_nx) {
            double d = (in->lat_x0 + (ix + 1) * in->lat_px - x[0]) / u[0];
            if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 1; }
        }
        if (u[1] < 0.0 && iy > 0) {
            double d = (in->lat_y0 + iy * in->lat_py - x[1]) / u[1];
            if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 2; }
        }
        if (u[1] > 0.0 && iy + 1 < in->lat_ny) {
            double d = (in->lat_y0 + (iy + 1) * in->lat_py - x[1]) / u[1];
            if (d > 0.0 && d < best) { best = d; *surf = in->n_surf + 3; }
        }
    }
    return best;
}

/* specular reflection Omega' = Omega - 2 (Omega.n^) n^; axis planes flip one component exactly (R13) */
static void reflect(const orc_problem *p, int32_t s, const double x[3], double u[3])
{
    int typ = p->in.surf_type[s];
    if (typ == S_PLANE_X) { u[0] = -u[0]; return; }
    if (typ == S_PLANE_Y) { u[1] = -u[1]; return; }
    if (typ == S_PLANE_Z) { u[2] = -u[2]; return; }
    double n[3];
    surf_normal(p, s, x, n);
    double nn = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    n[0] /= nn; n[1] /= nn; n[2] /= nn;
    double dot = u[0] * n[0] + u[1] * n[1] + u[2] * n[2];
    u[0] -= 2.0 * dot * n[0];
    u[1] -= 2.0 * dot * n[1];
    u[2] -= 2.0 * dot * n[2];
}

static int surface_in_cell(const orc_problem *p, int32_t c, int32_t s)
{
    for (int32_t k = p->in.cell_surf_off[c]; k < p->in.cell_surf_off[c + 1]; k++)
        if (p->in.cell_surf_id[k] == s) return 1;
    return 0;
}

/* ------------------------------------------------------------------ cross sections */
/* largest i with grid[i] <= E, clamped to [0, n-2] (R19): plain binary search */
int32_t orc_grid_index(const orc_problem *p, double E)
{
    const double *g = p->in.grid;
    int32_t lo = 0, hi = p->in.n_grid - 1;
    if (E < g[0]) return 0;
    while (hi - lo > 1) {
        int32_t mid = (lo + hi) / 2;
        if (g[mid] <= E) lo = mid; else hi = mid;
    }
    return lo;
}

/* lin-lin interpolation of the material's macroscopic columns and their running sum;
 * out[0] = Sigma_t = last cumulative value, out[1+j] = cumulative threshold j (R19) */
static int ce_xs_full(const orc_problem *p, int32_t m, double E, double *out, double *sig_f)
{
    int32_t i = orc_grid_index(p, E);
    const double *g = p->in.grid;
    double f = (E - g[i]) / (g[i + 1] - g[i]);
    int32_t nc = p->ce_ncol[m];
    double cum = 0.0;
    for (int32_t j = 0; j < nc; j++) {
        const double *col = p->ce_col[m] + (size_t)j * p->in.n_grid;
        double v = col[i] + f * (col[i + 1] - col[i]);
        if (j == nc - 2) *sig_f = v;
        cum += v;
        out[1 + j] = cum;
    }
    out[0] = cum;
    return nc;
}

int orc_ce_xs(const orc_problem *p, int32_t m, double E, double *out)
{
    double sig_f;
    return ce_xs_full(p, m, E, out, &sig_f);
}

static int32_t edge_bin(const double *edges, int32_t n, double v)
{
    /* largest b with edges[b] <= v, clamped to [0, n-1] (R24: binary search on the edge array, never log) */
    int32_t lo = 0, hi = n;
    if (v < edges[0]) return 0;
    while (hi - lo > 1) {
        int32_t mid = (lo + hi) / 2;
        if (edges[mid] <= v) lo = mid; else hi = mid;
    }
    return lo;
}

/* ------------------------------------------------------------------ create / destroy */
static void *dup_mem(const void *src, size_t bytes)
{
    if (!src || bytes == 0) return NULL;
    void *d = malloc(bytes);
    memcpy(d, src, bytes);
    return d;
}

#define DUP(field, count, type) p->in.field = (const type *)dup_mem(in->field, (size_t)(count) * sizeof(type))

orc_problem *orc_create(const orc_input *in)
{
    orc_problem *p = (orc_problem *)calloc(1, sizeof(orc_problem));
    p->in = *in;
    DUP(surf_type, in->n_surf, int32_t);
    DUP(surf_param, in->n_surf * 4, double);
    DUP(surf_bc, in->n_surf, int32_t);
    DUP(cell_surf_off, in->n_cell + 1, int32_t);
    int32_t nref = in->cell_surf_off[in->n_cell];
    DUP(cell_surf_id, nref, int32_t);
    DUP(cell_surf_sense, nref, int32_t);
    DUP(cell_fill_type, in->n_cell, int32_t);
    DUP(cell_fill, in->n_cell, int32_t);
    DUP(cell_bin, in->n_cell, int32_t);
    DUP(univ_cell_off, in->n_univ + 1, int32_t);
    if (in->has_lat) {
        DUP(lat_univ, in->lat_nx * in->lat_ny, int32_t);
        DUP(lat_bin, in->lat_nx * in->lat_ny, int32_t);
    }
    if (in->n_lat2 > 0) {
        DUP(lat2_nx, in->n_lat2, int32_t);
        DUP(lat2_ny, in->n_lat2, int32_t);
        DUP(lat2_px, in->n_lat2, double);
        DUP(lat2_py, in->n_lat2, double);
        DUP(lat2_off, in->n_lat2 + 1, int32_t);
        DUP(lat2_univ, in->lat2_off[in->n_lat2], int32_t);
        DUP(lat2_bin, in->lat2_off[in->n_lat2], int32_t);
    }
    int64_t n_tally;
    if (in->mode == 0) {
        int G = in->G, nm = in->n_mat;
        DUP(sig_t, nm * G, double);
        DUP(sig_f, nm * G, double);
        DUP(nu, nm * G, double);
        DUP(chi, nm * G, double);
        DUP(S, nm * G * G, double);
        DUP(src_group_pdf, G, double);
        p->sig_s = (double *)calloc((size_t)nm * G, sizeof(double));
        p->cumS = (double *)calloc((size_t)nm * G * G, sizeof(double));
        p->cumchi = (double *)calloc((size_t)nm * G, sizeof(double));
        p->nusf = (double *)calloc((size_t)nm * G, sizeof(double));
        p->src_cum = (double *)calloc((size_t)G, sizeof(double));
        for (int m = 0; m < nm; m++) {
            double cc = 0.0;
            for (int g = 0; g < G; g++) {
                double cs = 0.0;
                for (int gp = 0; gp < G; gp++) {
                    cs += in->S[((size_t)m * G + g) * G + gp];
                    p->cumS[((size_t)m * G + g) * G + gp] = cs;
                }
                p->sig_s[m * G + g] = cs; /* Sigma_s = stored row sum (R3) */
                cc += in->chi[m * G + g];
                p->cumchi[m * G + g] = cc;
                p->nusf[m * G + g] = in->nu[m * G + g] * in->sig_f[m * G + g];
            }
        }
        double cs = 0.0;
        for (int g = 0; g < G; g++) { cs += in->src_group_pdf[g]; p->src_cum[g] = cs; }
        n_tally = (int64_t)in->n_bins * G;
        if (in->td) {
            int J = in->n_dgroup;
            DUP(speed, G, double);
            DUP(nu_d, (size_t)nm * J * G, double);
            DUP(decay, (size_t)nm * J, double);
            DUP(chi_d, (size_t)nm * J * G, double);
            DUP(t_edges, in->n_t + 1, double);
            p->cumchi_d = (double *)calloc((size_t)nm * J * G + 1, sizeof(double));
            p->cum_nu = (double *)calloc((size_t)nm * G * (J + 1), sizeof(double));
            for (int m = 0; m < nm; m++) {
                for (int j = 0; j < J; j++) {
                    double cc = 0.0;
                    for (int g = 0; g < G; g++) { cc += in->chi_d[((size_t)m * J + j) * G + g]; p->cumchi_d[((size_t)m * J + j) * G + g] = cc; }
                }
                for (int g = 0; g < G; g++) { /* cumulative yields [prompt, +delayed 1, ..., +delayed J] */
                    double cn = in->nu[m * G + g];
                    p->cum_nu[((size_t)m * G + g) * (J + 1)] = cn;
                    for (int j = 0; j < J; j++) { cn += in->nu_d[((size_t)m * J + j) * G + g]; p->cum_nu[((size_t)m * G + g) * (J + 1) + 1 + j] = cn; }
                }
            }
            n_tally = (int64_t)in->n_bins * in->n_t * G;
            p->cbank = (particle **)calloc((size_t)in->n_t + 1, sizeof(particle *));
            p->n_cbank = (uint64_t *)calloc((size_t)in->n_t + 1, sizeof(uint64_t));
            p->cap_cbank = (uint64_t *)calloc((size_t)in->n_t + 1, sizeof(uint64_t));
        }
    } else {
        int nm = in->n_mat, ng = in->n_grid;
        DUP(grid, ng, double);
        DUP(nuc_A, in->n_nuc, double);
        DUP(nuc_el, (size_t)in->n_nuc * ng, double);
        DUP(nuc_c, (size_t)in->n_nuc * ng, double);
        DUP(nuc_f, (size_t)in->n_nuc * ng, double);
        DUP(mat_nuc_off, nm + 1, int32_t);
        DUP(mat_nuc_id, in->mat_nuc_off[nm], int32_t);
        DUP(mat_nuc_dens, in->mat_nuc_off[nm], double);
        DUP(t_edges, in->n_t + 1, double);
        DUP(e_edges, in->n_e + 1, double);
        p->ce_ncol = (int32_t *)calloc((size_t)nm, sizeof(int32_t));
        p->ce_col = (double **)calloc((size_t)nm, sizeof(double *));
        for (int m = 0; m < nm; m++) {
            int n0 = in->mat_nuc_off[m], nn = in->mat_nuc_off[m + 1] - n0;
            p->ce_ncol[m] = nn + 2;
            double *col = (double *)calloc((size_t)(nn + 2) * ng, sizeof(double));
            p->ce_col[m] = col;
            for (int i = 0; i < ng; i++) {
                double sf = 0.0, sc = 0.0;
                for (int j = 0; j < nn; j++) {
                    int nuc = in->mat_nuc_id[n0 + j];
                    double dens = in->mat_nuc_dens[n0 + j];
                    col[(size_t)j * ng + i] = dens * in->nuc_el[(size_t)nuc * ng + i];
                    sf += dens * in->nuc_f[(size_t)nuc * ng + i];
                    sc += dens * in->nuc_c[(size_t)nuc * ng + i];
                }
                col[(size_t)nn * ng + i] = sf;
                col[(size_t)(nn + 1) * ng + i] = sc;
            }
        }
        n_tally = (int64_t)in->n_bins * in->n_t * in->n_e;
    }
    p->flux_c = (double *)calloc((size_t)n_tally, sizeof(double));
    p->flux_acc = (double *)calloc((size_t)n_tally, sizeof(double));
    p->flux_acc2 = (double *)calloc((size_t)n_tally, sizeof(double));
    return p;
}

void orc_destroy(orc_problem *p)
{
    /* test infrastructure: the input copies are small; free what matters */
    if (!p) return;
    free(p->flux_c); free(p->flux_acc); free(p->flux_acc2); free(p->k_cycle);
    free(p->bank); free(p->newbank); free(p->stack); free(p->trace);
    if (p->ce_col) for (int m = 0; m < p->in.n_mat; m++) free(p->ce_col[m]);
    free(p->ce_col); free(p->ce_ncol);
    free(p->sig_s); free(p->cumS); free(p->cumchi); free(p->nusf); free(p->src_cum);
    free((void *)p->in.grid); free((void *)p->in.nuc_el); free((void *)p->in.nuc_c); free((void *)p->in.nuc_f);
    free(p);
}

int64_t orc_n_tally(const orc_problem *p)
{
    if (p->in.mode == 0) return p->in.td ? (int64_t)p->in.n_bins * p->in.n_t * p->in.G : (int64_t)p->in.n_bins * p->in.G;
    return (int64_t)p->in.n_bins * p->in.n_t * p->in.n_e;
}

int orc_set_trace(orc_problem *p, uint64_t first_id, uint64_t n_ids, uint64_t max_records)
{
    free(p->trace);
    p->trace = (orc_trace_rec *)calloc((size_t)max_records, sizeof(orc_trace_rec));
    p->tr_first = first_id; p->tr_n = n_ids; p->tr_max = max_records; p->tr_count = 0;
    return 0;
}

static void trace(orc_problem *p, const particle *q, int ev, int32_t c0, int32_t elem, int32_t c1, int32_t surf,
                  int32_t gi, double d, double E)
{
    if (!p->trace || q->id < p->tr_first || q->id - p->tr_first >= p->tr_n) return;
    if (p->tr_count < p->tr_max) {
        orc_trace_rec *r = &p->trace[p->tr_count];
        r->id = q->id; r->cycle = p->cycle; r->seq = q->nseg; r->ev = ev;
        r->c0 = c0; r->elem = elem; r->c1 = c1; r->surf = surf; r->gi = gi;
        r->x = q->x; r->y = q->y; r->z = q->z; r->d = d; r->E = E; r->t = q->t;
    }
    p->tr_count++;
}

/* ------------------------------------------------------------------ one history */
static void push_secondary(orc_problem *p, const particle *c)
{
    if (p->n_stack == p->cap_stack) {
        p->cap_stack = p->cap_stack ? 2 * p->cap_stack : 1024;
        p->stack = (particle *)realloc(p->stack, p->cap_stack * sizeof(particle));
    }
    p->stack[p->n_stack++] = *c;
}

/* a particle that waits for census interval k (it reached the time edge, or it is a delayed neutron born there) */
static void push_census(orc_problem *p, int k, const particle *c)
{
    if (p->n_cbank[k] == p->cap_cbank[k]) {
        p->cap_cbank[k] = p->cap_cbank[k] ? 2 * p->cap_cbank[k] : 1024;
        p->cbank[k] = (particle *)realloc(p->cbank[k], p->cap_cbank[k] * sizeof(particle));
    }
    p->cbank[k][p->n_cbank[k]++] = *c;
}

static void bank_site(orc_problem *p, const particle *q, const double u[3], int32_t g)
{
    if (p->n_newbank == p->cap_bank) { p->error = -3; return; } /* bank overflow (R6) */
    orc_site *s = &p->newbank[p->n_newbank++];
    s->x = q->x; s->y = q->y; s->z = q->z; s->ux = u[0]; s->uy = u[1]; s->uz = u[2]; s->g = g; s->pad = 0;
}

/* follow particle q from its current state to its death, one segment per loop iteration */
static void transport(orc_problem *p, particle *q)
{
    const orc_input *in = &p->in;
    double xs[64];
    const int timed = in->mode == 1 || in->td; /* the particle carries a clock: time edges are candidate events */
    if (!q->resumed) { p->counters[0]++; p->balance[0] += q->w; }
    while (q->alive) {
        double x[3] = {q->x, q->y, q->z}, u[3] = {q->ux, q->uy, q->uz};
        int32_t loc[3] = {q->c0, q->elem, q->c1};
        int32_t mat = loc[1] >= 0 ? in->cell_fill[loc[2]] : in->cell_fill[loc[0]];
        int32_t bin = loc[1] >= 0 ? in->lat_bin[OUTER(loc[1])] + in->cell_bin[loc[2]] : in->cell_bin[loc[0]];
        if (loc[1] >= 0 && INNER(loc[1]) >= 0)
            bin += in->lat2_bin[in->lat2_off[in->cell_fill[mid_cell(p, OUTER(loc[1]))]] + INNER(loc[1])];
        /* cross sections */
        double sig_t, nusf;
        int32_t gi, ncol = 0;
        if (in->mode == 0) {
            gi = q->g;
            sig_t = in->sig_t[mat * in->G + q->g];
            nusf = p->nusf[mat * in->G + q->g];
        } else {
            gi = orc_grid_index(p, q->E);
            double sig_f;
            ncol = ce_xs_full(p, mat, q->E, xs, &sig_f);
            sig_t = xs[0];
            nusf = (in->nu0 + in->nu1 * (q->E * 1e-6)) * sig_f;
        }
        /* candidate distances: collision (one draw every segment), surface, time edge */
        double d_coll = -log(draw(p, q)) / sig_t;
        int32_t hit;
        double d_surf = orc_distance(p, x, u, loc, q->last_surf, &hit);
        double v = 0.0, d_time = INFINITY;
        if (timed) {
            v = in->mode == 1 ? orc_speed(q->E) : in->speed[q->g]; /* R23 / the group's speed (R38) */
            d_time = v * (in->t_edges[q->tbin + 1] - q->t);
        }
        int kind; /* 0 collision, 1 surface, 2 time edge (R12) */
        double d;
        if (d_coll < d_surf && d_coll < d_time) { kind = 0; d = d_coll; }
        else if (d_surf <= d_time) { kind = 1; d = d_surf; }
        else { kind = 2; d = d_time; }
        /* move + track-length tallies */
        q->x += d * u[0]; q->y += d * u[1]; q->z += d * u[2];
        double E_flight = q->E;
        int64_t tix;
        if (in->mode == 0) tix = in->td ? ((int64_t)bin * in->n_t + q->tbin) * in->G + q->g : (int64_t)bin * in->G + q->g;
        else tix = ((int64_t)bin * in->n_t + q->tbin) * in->n_e + edge_bin(in->e_edges, in->n_e, q->E);
        if (timed) { if (kind == 2) q->t = in->t_edges[q->tbin + 1]; else q->t += d / v; }
        p->flux_c[tix] += q->w * d;
        p->k_num += q->w * d * nusf;
        int ev;
        if (kind == 0) {
            q->last_surf = -1;
            /* reaction choice.  Analog (R3): xi Sigma_t against [scatter, fission, capture].  Implicit capture (R36):
             * the weight loses its capture share, w <- w (Sigma_t - Sigma_c) / Sigma_t, and xi (Sigma_t - Sigma_c) is
             * compared against [scatter, fission]; a scattered particle whose weight fell below w_roulette plays
             * roulette (one more draw): it survives with probability w / w_survive at weight w_survive. */
            const int implicit = in->implicit_capture;
            int rouletted = 0;
            if (in->mode == 0) {
                int G = in->G;
                double sig_s = p->sig_s[mat * G + q->g], sig_f = in->sig_f[mat * G + q->g];
                double total = sig_t;
                if (implicit) {
                    total = sig_s + sig_f;
                    double wn = q->w * (total / sig_t);
                    p->balance[1] += q->w - wn;
                    q->w = wn;
                }
                double uu = draw(p, q) * total;
                if (uu < sig_s) {
                    ev = ORC_EV_SCATTER;
                    if (implicit && q->w < in->w_roulette) {
                        if (draw(p, q) * in->w_survive < q->w) { p->balance[5] += in->w_survive - q->w; q->w = in->w_survive; }
                        else { p->balance[4] += q->w; rouletted = 1; ev = ORC_EV_CAPTURE; q->alive = 0; }
                    }
                    if (!rouletted) {
                        double vv = draw(p, q) * sig_s;
                        int32_t gp = pick(p->cumS + ((size_t)mat * G + q->g) * G, G, vv);
                        double xi1 = draw(p, q), xi2 = draw(p, q), o[3];
                        orc_iso_dir(xi1, xi2, o);
                        q->g = gp; q->ux = o[0]; q->uy = o[1]; q->uz = o[2];
                    }
                } else if (uu < sig_s + sig_f && in->td) {
                    /* time-dependent fixed source (R39): nu = prompt yield + delayed yields; n = floor(nu + xi)
                     * children of the parent's weight; per child: type (prompt / precursor group j) by xi nu against
                     * the cumulative yields, group from the type's spectrum, emission time t (prompt) or
                     * t - ln(xi) / lambda_j (delayed), isotropic direction; own stream (R10).  A delayed neutron
                     * emitted after the last time edge is never born (its draws are consumed all the same). */
                    ev = ORC_EV_FISSION;
                    int J = in->n_dgroup;
                    const double *cn = p->cum_nu + ((size_t)mat * G + q->g) * (J + 1);
                    double nu_tot = cn[J];
                    int n = (int)floor(nu_tot + draw(p, q));
                    uint32_t ctr_birth = q->ctr;
                    for (int j = 0; j < n; j++) {
                        int32_t typ = pick(cn, J + 1, draw(p, q) * nu_tot); /* 0 prompt, 1 + precursor group */
                        const double *cc = typ == 0 ? p->cumchi + (size_t)mat * G : p->cumchi_d + ((size_t)mat * J + typ - 1) * G;
                        int32_t gj = pick(cc, G, draw(p, q) * cc[G - 1]);
                        double tj = q->t;
                        if (typ > 0) tj = q->t - log(draw(p, q)) / in->decay[mat * J + typ - 1];
                        double xi1 = draw(p, q), xi2 = draw(p, q), o[3];
                        orc_iso_dir(xi1, xi2, o);
                        if (!(tj < in->t_edges[in->n_t])) continue;
                        particle c = *q; /* same position, cell and weight as the parent */
                        c.ux = o[0]; c.uy = o[1]; c.uz = o[2]; c.g = gj; c.t = tj;
                        c.tbin = edge_bin(in->t_edges, in->n_t, tj);
                        c.id = orc_child_id(p->seed, q->id, ctr_birth, (uint32_t)j);
                        c.ctr = 0; c.nseg = 0; c.last_surf = -1; c.alive = 1; c.resumed = 0;
                        if (c.tbin == q->tbin) push_secondary(p, &c);
                        else { /* waits for a later interval, where the comb may replace it: count the track now */
                            c.resumed = 1;
                            p->counters[0]++;
                            p->balance[0] += c.w;
                            push_census(p, c.tbin, &c);
                        }
                        p->counters[11]++;
                    }
                    p->balance[1] += q->w;
                    q->alive = 0;
                } else if (uu < sig_s + sig_f) {
                    ev = ORC_EV_FISSION;
                    int n = (int)floor(q->w * in->nu[mat * G + q->g] / p->k_prev + draw(p, q));
                    for (int j = 0; j < n; j++) {
                        const double *cc = p->cumchi + (size_t)mat * G;
                        int32_t gj = pick(cc, G, draw(p, q) * cc[G - 1]);
                        double xi1 = draw(p, q), xi2 = draw(p, q), o[3];
                        orc_iso_dir(xi1, xi2, o);
                        bank_site(p, q, o, gj);
                        p->counters[11]++;
                    }
                    p->balance[1] += q->w;
                    q->alive = 0;
                } else {
                    ev = ORC_EV_CAPTURE;
                    p->balance[1] += q->w;
                    q->alive = 0;
                }
            } else {
                double total = sig_t;
                int32_t nsel = ncol;
                if (implicit) {
                    total = xs[ncol - 1]; /* cumulative value before the capture column */
                    nsel = ncol - 1;
                    double wn = q->w * (total / sig_t);
                    p->balance[1] += q->w - wn;
                    q->w = wn;
                }
                double uu = draw(p, q) * total;
                int32_t r = pick(xs + 1, nsel, uu);
                if (r < ncol - 2) { /* elastic off nuclide r of this material */
                    ev = ORC_EV_SCATTER;
                    if (implicit && q->w < in->w_roulette) {
                        if (draw(p, q) * in->w_survive < q->w) { p->balance[5] += in->w_survive - q->w; q->w = in->w_survive; }
                        else { p->balance[4] += q->w; rouletted = 1; ev = ORC_EV_CAPTURE; q->alive = 0; }
                    }
                    if (!rouletted) {
                        double A = in->nuc_A[in->mat_nuc_id[in->mat_nuc_off[mat] + r]];
                        double En, o[3];
                        if (in->kT > 0.0 && q->E < FREE_GAS_LIMIT * in->kT)
                            orc_free_gas(q->E, u, A, in->kT, p->seed, q->id, p->cycle, &q->ctr, &En, o);
                        else {
                            double xi1 = draw(p, q), xi2 = draw(p, q);
                            orc_elastic(q->E, u, A, xi1, xi2, &En, o);
                        }
                        if (En < in->grid[0]) En = in->grid[0];
                        if (En > in->grid[in->n_grid - 1]) En = in->grid[in->n_grid - 1];
                        q->E = En; q->ux = o[0]; q->uy = o[1]; q->uz = o[2];
                    }
                } else if (r == ncol - 2) {
                    ev = ORC_EV_FISSION;
                    double nu = in->nu0 + in->nu1 * (q->E * 1e-6);
                    int n = (int)floor(q->w * nu + draw(p, q));
                    uint32_t ctr_birth = q->ctr;
                    for (int j = 0; j < n; j++) {
                        double a1 = draw(p, q), a2 = draw(p, q), a3 = draw(p, q), a4 = draw(p, q);
                        double En = 1e6 * orc_watt(in->watt_a, in->watt_b, a1, a2, a3, a4);
                        if (En < in->grid[0]) En = in->grid[0];
                        if (En > in->grid[in->n_grid - 1]) En = in->grid[in->n_grid - 1];
                        double xi1 = draw(p, q), xi2 = draw(p, q), o[3];
                        orc_iso_dir(xi1, xi2, o);
                        particle c = *q; /* same position, time, time bin and cell as the parent */
                        c.ux = o[0]; c.uy = o[1]; c.uz = o[2]; c.E = En; c.w = 1.0;
                        c.id = orc_child_id(p->seed, q->id, ctr_birth, (uint32_t)j);
                        c.ctr = 0; c.nseg = 0; c.last_surf = -1; c.alive = 1;
                        push_secondary(p, &c);
                        p->counters[11]++;
                    }
                    p->balance[1] += q->w;
                    q->alive = 0;
                } else {
                    ev = ORC_EV_CAPTURE;
                    p->balance[1] += q->w;
                    q->alive = 0;
                }
            }
            trace(p, q, ev, loc[0], loc[1], loc[2], -1, gi, d, E_flight);
        } else if (kind == 1) {
            if (hit >= in->n_surf + 4) { /* second-level lattice wall: step to the neighbour element (R37) */
                ev = ORC_EV_LATTICE;
                int w = hit - in->n_surf - 4;
                int32_t k2 = in->cell_fill[mid_cell(p, OUTER(loc[1]))];
                int32_t jx = INNER(loc[1]) % in->lat2_nx[k2], jy = INNER(loc[1]) / in->lat2_nx[k2];
                if (w == 0) jx--; else if (w == 1) jx++; else if (w == 2) jy--; else jy++;
                int32_t inner = jy * in->lat2_nx[k2] + jx;
                q->elem = OUTER(loc[1]) | ((inner + 1) << 20);
                q->last_surf = -1;
                double xn[3] = {q->x, q->y, q->z}, xl[3];
                local_coords(p, q->elem, xn, xl);
                q->c1 = find_cell(p, in->lat2_univ[in->lat2_off[k2] + inner], xl, u, -1);
                if (q->c1 < 0) { ev = ORC_EV_LOST; q->alive = 0; p->error = -2; }
            } else if (hit >= in->n_surf) { /* lattice wall: step to the neighbour element (R14) */
                ev = ORC_EV_LATTICE;
                int w = hit - in->n_surf;
                int32_t ix = OUTER(loc[1]) % in->lat_nx, iy = OUTER(loc[1]) / in->lat_nx;
                if (w == 0) ix--; else if (w == 1) ix++; else if (w == 2) iy--; else iy++;
                q->last_surf = -1;
                double xn[3] = {q->x, q->y, q->z}, xo[3];
                outer_coords(p, iy * in->lat_nx + ix, xn, xo);
                q->c1 = descend(p, iy * in->lat_nx + ix, xo, u, -1, &q->elem);
                if (q->c1 < 0) { ev = ORC_EV_LOST; q->alive = 0; p->error = -2; }
            } else {
                int bc = in->surf_bc[hit];
                /* whose surface is it: the root cell's (global coordinates), the cell's that the second-level lattice
                 * fills (first-level-element coordinates), or the local cell's (innermost coordinates) */
                int local = !surface_in_cell(p, loc[0], hit);
                int midlevel = local && loc[1] >= 0 && INNER(loc[1]) >= 0 && surface_in_cell(p, mid_cell(p, OUTER(loc[1])), hit);
                double xn[3] = {q->x, q->y, q->z}, xl[3];
                if (midlevel) outer_coords(p, OUTER(loc[1]), xn, xl);
                else if (local) local_coords(p, loc[1], xn, xl);
                if (bc == 2) {
                    ev = ORC_EV_LEAK;
                    p->leak_c += q->w;
                    p->balance[2] += q->w;
                    q->alive = 0;
                } else if (bc == 1) {
                    ev = ORC_EV_REFLECT;
                    double un[3] = {u[0], u[1], u[2]};
                    reflect(p, hit, local ? xl : xn, un);
                    q->ux = un[0]; q->uy = un[1]; q->uz = un[2];
                    q->last_surf = hit;
                } else {
                    ev = ORC_EV_TRANSMIT;
                    q->last_surf = hit;
                    if (local) {
                        if (!midlevel && INNER(loc[1]) >= 0) { /* inside the same second-level element */
                            int32_t k2 = in->cell_fill[mid_cell(p, OUTER(loc[1]))];
                            q->c1 = find_cell(p, in->lat2_univ[in->lat2_off[k2] + INNER(loc[1])], xl, u, hit);
                        } else { /* inside the same first-level element: its universe, descending where a lattice fills */
                            double xo[3];
                            outer_coords(p, OUTER(loc[1]), xn, xo);
                            q->c1 = descend(p, OUTER(loc[1]), xo, u, hit, &q->elem);
                        }
                        if (q->c1 < 0) { ev = ORC_EV_LOST; q->alive = 0; p->error = -2; }
                    } else {
                        int32_t nl[3];
                        if (orc_locate(p, xn, u, hit, nl) != 0) { ev = ORC_EV_LOST; q->alive = 0; p->error = -2; }
                        q->c0 = nl[0]; q->elem = nl[1]; q->c1 = nl[2];
                    }
                }
            }
            trace(p, q, ev, loc[0], loc[1], loc[2], hit, gi, d, E_flight);
        } else {
            q->tbin++;
            q->last_surf = -1; /* R11: the particle has moved off the surface it sat on */
            if (q->tbin == in->n_t) { ev = ORC_EV_CUTOFF; p->balance[3] += q->w; q->alive = 0; } else ev = ORC_EV_TIME_EDGE;
            trace(p, q, ev, loc[0], loc[1], loc[2], -1, gi, d, E_flight);
            if (ev == ORC_EV_TIME_EDGE && p->census_stop) { /* the census: the particle waits in the next interval's bank */
                p->counters[ev]++;
                q->nseg++;
                q->resumed = 1;
                push_census(p, q->tbin, q);
                return;
            }
        }
        p->counters[ev]++;
        q->nseg++;
        if (q->alive && q->nseg >= MAX_SEGMENTS) {
            q->alive = 0; p->counters[ORC_EV_LOST]++; p->error = -4;
        }
    }
}

/* ------------------------------------------------------------------ sources */
/* source birth: always six draws x,y,z,mu,phi,group (draw budget table) */
static int sample_source(orc_problem *p, particle *q)
{
    const orc_input *in = &p->in;
    double xi[6];
    for (int i = 0; i < 6; i++) xi[i] = draw(p, q);
    q->x = in->src_lo[0] + xi[0] * (in->src_hi[0] - in->src_lo[0]);
    q->y = in->src_lo[1] + xi[1] * (in->src_hi[1] - in->src_lo[1]);
    q->z = in->src_lo[2] + xi[2] * (in->src_hi[2] - in->src_lo[2]);
    if (in->src_iso) {
        double o[3];
        orc_iso_dir(xi[3], xi[4], o);
        q->ux = o[0]; q->uy = o[1]; q->uz = o[2];
    } else {
        q->ux = in->src_dir[0]; q->uy = in->src_dir[1]; q->uz = in->src_dir[2];
    }
    if (in->mode == 0) {
        q->g = pick(p->src_cum, in->G, xi[5] * p->src_cum[in->G - 1]);
        q->E = 0.0; q->t = 0.0; q->tbin = 0;
        if (in->td) { q->t = in->src_t; q->tbin = edge_bin(in->t_edges, in->n_t, q->t); }
    } else {
        q->g = 0; q->E = in->src_E; q->t = in->src_t;
        q->tbin = edge_bin(in->t_edges, in->n_t, q->t);
    }
    return 0;
}

static void place(orc_problem *p, particle *q)
{
    double x[3] = {q->x, q->y, q->z}, u[3] = {q->ux, q->uy, q->uz};
    int32_t loc[3];
    q->last_surf = -1;
    q->alive = 1;
    if (orc_locate(p, x, u, -1, loc) != 0) {
        q->alive = 0; p->error = -2; p->counters[ORC_EV_LOST]++;
    }
    q->c0 = loc[0]; q->elem = loc[1]; q->c1 = loc[2];
}

static void accumulate_cycle(orc_problem *p, uint64_t N, int active)
{
    int64_t nt = orc_n_tally(p);
    double k_c = p->k_num / (double)N;
    p->k_cycle[p->n_cycles++] = k_c;
    if (active) {
        for (int64_t i = 0; i < nt; i++) {
            double f = p->flux_c[i] / (double)N;
            p->flux_acc[i] += f;
            p->flux_acc2[i] += f * f;
        }
        double l = p->leak_c / (double)N;
        p->leak_acc += l; p->leak_acc2 += l * l;
        p->k_acc += k_c; p->k_acc2 += k_c * k_c;
        p->n_active_done++;
    }
    p->k_prev = k_c;
}

static void reset_results(orc_problem *p, int n_cycles)
{
    int64_t nt = orc_n_tally(p);
    free(p->k_cycle);
    p->k_cycle = (double *)calloc((size_t)(n_cycles > 0 ? n_cycles : 1), sizeof(double));
    memset(p->flux_acc, 0, (size_t)nt * sizeof(double));
    memset(p->flux_acc2, 0, (size_t)nt * sizeof(double));
    memset(p->counters, 0, sizeof(p->counters));
    p->leak_acc = p->leak_acc2 = p->k_acc = p->k_acc2 = 0.0;
    memset(p->balance, 0, sizeof(p->balance));
    p->n_cycles = p->n_active_done = 0;
    p->error = 0; p->tr_count = 0;
}

/* k-eigenvalue power iteration (SURVEY.md 8c algorithm) */
int orc_run_eigenvalue(orc_problem *p, uint64_t N, int n_inactive, int n_active, uint64_t seed)
{
    if (p->in.mode != 0) return -1;
    int64_t nt = orc_n_tally(p);
    reset_results(p, n_inactive + n_active);
    p->seed = seed; p->fixed = 0; p->k_prev = 1.0; /* k guess (R7) */
    p->cap_bank = 2 * N + 16;                      /* capacity 2N (R6) */
    free(p->bank); free(p->newbank);
    p->bank = (orc_site *)calloc((size_t)p->cap_bank, sizeof(orc_site));
    p->newbank = (orc_site *)calloc((size_t)p->cap_bank, sizeof(orc_site));
    p->n_bank = 0;
    for (int c = 0; c < n_inactive + n_active; c++) {
        p->cycle = (uint32_t)c;
        uint64_t M = c == 0 ? N : p->n_bank;
        double w0 = c == 0 ? 1.0 : (M > 0 ? (double)N / (double)M : 0.0); /* source renormalisation (R6) */
        memset(p->flux_c, 0, (size_t)nt * sizeof(double));
        p->k_num = 0.0; p->leak_c = 0.0; p->n_newbank = 0;
        for (uint64_t i = 0; i < M; i++) {
            particle q;
            memset(&q, 0, sizeof q);
            q.id = i; q.w = w0;
            if (c == 0) sample_source(p, &q);
            else {
                const orc_site *s = &p->bank[i];
                q.x = s->x; q.y = s->y; q.z = s->z; q.ux = s->ux; q.uy = s->uy; q.uz = s->uz; q.g = s->g;
            }
            place(p, &q);
            if (q.alive) transport(p, &q); else p->counters[0]++;
        }
        /* parents were followed in id order and children banked in j order: newbank is already
         * sorted by (parent id, child index) */
        orc_site *t = p->bank; p->bank = p->newbank; p->newbank = t;
        p->n_bank = p->n_newbank;
        if (p->n_bank > p->counters[12]) p->counters[12] = p->n_bank;
        accumulate_cycle(p, N, c >= n_inactive);
    }
    return p->error;
}

/* All-core timing variant of the eigenvalue run (bench.py's cpu_baseline only; the parity tests use the serial
 * run above): the source particles of a cycle are split in n_threads contiguous id ranges, each followed by its own
 * thread into thread-private tallies and a private piece of the fission bank; pieces and tallies are joined in
 * thread order, so the bank stays sorted by (parent id, child index) and the result is reproducible for a fixed
 * n_threads (it differs from the serial run by float64 summation order only).  No tracing. */
int orc_run_eigenvalue_mt(orc_problem *p, uint64_t N, int n_inactive, int n_active, uint64_t seed, int n_threads)
{
    if (p->in.mode != 0 || n_threads < 1) return -1;
    int64_t nt = orc_n_tally(p);
    reset_results(p, n_inactive + n_active);
    p->seed = seed; p->fixed = 0; p->k_prev = 1.0;
    p->cap_bank = 2 * N + 16;
    free(p->bank); free(p->newbank);
    p->bank = (orc_site *)calloc((size_t)p->cap_bank, sizeof(orc_site));
    p->newbank = (orc_site *)calloc((size_t)p->cap_bank, sizeof(orc_site));
    p->n_bank = 0;
    free(p->trace); p->trace = NULL;
    orc_problem *th = (orc_problem *)calloc((size_t)n_threads, sizeof(orc_problem));
    for (int t = 0; t < n_threads; t++) {
        th[t] = *p; /* shares the read-only inputs and derived tables */
        th[t].flux_c = (double *)calloc((size_t)nt, sizeof(double));
        th[t].cap_bank = p->cap_bank; /* worst case: one thread banks everything */
        th[t].newbank = (orc_site *)calloc((size_t)p->cap_bank, sizeof(orc_site));
    }
    for (int c = 0; c < n_inactive + n_active; c++) {
        p->cycle = (uint32_t)c;
        uint64_t M = c == 0 ? N : p->n_bank;
        double w0 = c == 0 ? 1.0 : (M > 0 ? (double)N / (double)M : 0.0);
        #pragma omp parallel for num_threads(n_threads) schedule(static, 1)
        for (int t = 0; t < n_threads; t++) {
            orc_problem *q = &th[t];
            q->cycle = p->cycle; q->seed = seed; q->k_prev = p->k_prev; q->bank = p->bank;
            memset(q->flux_c, 0, (size_t)nt * sizeof(double));
            memset(q->counters, 0, sizeof(q->counters));
            q->k_num = 0.0; q->leak_c = 0.0; q->n_newbank = 0; q->error = 0;
            memset(q->balance, 0, sizeof(q->balance));
            uint64_t lo = M * (uint64_t)t / (uint64_t)n_threads, hi = M * (uint64_t)(t + 1) / (uint64_t)n_threads;
            for (uint64_t i = lo; i < hi; i++) {
                particle pt;
                memset(&pt, 0, sizeof pt);
                pt.id = i; pt.w = w0;
                if (c == 0) sample_source(q, &pt);
                else {
                    const orc_site *s = &p->bank[i];
                    pt.x = s->x; pt.y = s->y; pt.z = s->z; pt.ux = s->ux; pt.uy = s->uy; pt.uz = s->uz; pt.g = s->g;
                }
                place(q, &pt);
                if (pt.alive) transport(q, &pt); else q->counters[0]++;
            }
        }
        memset(p->flux_c, 0, (size_t)nt * sizeof(double));
        p->k_num = 0.0; p->leak_c = 0.0; p->n_newbank = 0;
        for (int t = 0; t < n_threads; t++) { /* join in thread order */
            for (int64_t i = 0; i < nt; i++) p->flux_c[i] += th[t].flux_c[i];
            p->k_num += th[t].k_num; p->leak_c += th[t].leak_c;
            for (int k = 0; k < 6; k++) p->balance[k] += th[t].balance[k];
            for (int k = 0; k < ORC_N_COUNTERS; k++) p->counters[k] += th[t].counters[k];
            if (th[t].error && !p->error) p->error = th[t].error;
            if (p->n_newbank + th[t].n_newbank > p->cap_bank) { p->error = -3; th[t].n_newbank = p->cap_bank - p->n_newbank; }
            memcpy(p->newbank + p->n_newbank, th[t].newbank, (size_t)th[t].n_newbank * sizeof(orc_site));
            p->n_newbank += th[t].n_newbank;
        }
        orc_site *tmp = p->bank; p->bank = p->newbank; p->newbank = tmp;
        p->n_bank = p->n_newbank;
        if (p->n_bank > p->counters[12]) p->counters[12] = p->n_bank;
        accumulate_cycle(p, N, c >= n_inactive);
    }
    for (int t = 0; t < n_threads; t++) { free(th[t].flux_c); free(th[t].newbank); }
    free(th);
    return p->error;
}

/* time-dependent fixed source: every source particle, then its secondaries LIFO */
int orc_run_fixed_source(orc_problem *p, uint64_t N, uint64_t seed)
{
    if (p->in.mode != 1) return -1;
    int64_t nt = orc_n_tally(p);
    reset_results(p, 1);
    p->seed = seed; p->fixed = 1; p->k_prev = 1.0; p->cycle = 0;
    memset(p->flux_c, 0, (size_t)nt * sizeof(double));
    p->k_num = 0.0; p->leak_c = 0.0; p->n_stack = 0;
    for (uint64_t i = 0; i < N; i++) {
        particle q;
        memset(&q, 0, sizeof q);
        q.id = i; q.w = 1.0;
        sample_source(p, &q);
        place(p, &q);
        if (q.alive) transport(p, &q); else p->counters[0]++;
        while (p->n_stack > 0) {
            if (p->n_stack > p->counters[12]) p->counters[12] = p->n_stack;
            /* R25: the prompt chain must be subcritical; more than 64 N secondaries = bank overflow */
            if (p->counters[11] > 64 * N + 4096) { p->error = -3; p->n_stack = 0; break; }
            particle c = p->stack[--p->n_stack];
            transport(p, &c);
        }
    }
    if (p->error == -3) return p->error;
    accumulate_cycle(p, N, 1);
    return p->error;
}

/* Population control at a census by combing (R40): the M particles of the bank in bank order (sorted by id), weights
 * w_i, running sums C_i; N teeth at (xi + j) W / N; a particle gets one copy per tooth in [C_{i-1}, C_i), each of
 * weight W / N: the total weight is conserved exactly and the population becomes exactly N. */
double orc_comb(const double *w, uint64_t M, uint64_t N, double xi, uint32_t *copies)
{
    double W = 0.0;
    for (uint64_t i = 0; i < M; i++) W += w[i];
    double delta = W / (double)N, off = xi * delta, C = 0.0;
    uint64_t j = 0;
    for (uint64_t i = 0; i < M; i++) {
        double hi = C + w[i];
        copies[i] = 0;
        while (j < N && off + (double)j * delta < hi) { copies[i]++; j++; }
        C = hi;
    }
    if (M > 0) { copies[M - 1] += (uint32_t)(N - j); } /* a last tooth lost to rounding stays with the last particle */
    return delta;
}

static int cmp_particle_id(const void *a, const void *b)
{
    uint64_t x = ((const particle *)a)->id, y = ((const particle *)b)->id;
    return x < y ? -1 : (x > y ? 1 : 0);
}

/* Time-dependent multi-group fixed source (R38-R40), census interval by census interval: the particles of interval k
 * are the source particles born in it, the survivors of interval k-1 and the delayed neutrons emitted in it; sorted by
 * id, combed to census_target particles if population control is on (k > first interval), then each followed to its
 * death or to the next time edge, its same-interval secondaries depth-first. */
int orc_run_td(orc_problem *p, uint64_t N, uint64_t seed)
{
    const orc_input *in = &p->in;
    if (in->mode != 0 || !in->td) return -1;
    int64_t nt = orc_n_tally(p);
    reset_results(p, 1);
    p->seed = seed; p->fixed = 1; p->k_prev = 1.0; p->cycle = 0;
    memset(p->flux_c, 0, (size_t)nt * sizeof(double));
    p->k_num = 0.0; p->leak_c = 0.0; p->n_stack = 0;
    p->census_stop = 1;
    p->n_census = 0;
    for (int k = 0; k <= in->n_t; k++) p->n_cbank[k] = 0;
    int first = edge_bin(in->t_edges, in->n_t, in->src_t);
    for (uint64_t i = 0; i < N; i++) { /* the source particles wait for their interval like everybody else */
        particle q;
        memset(&q, 0, sizeof q);
        q.id = i; q.w = 1.0;
        sample_source(p, &q);
        place(p, &q);
        if (q.alive) push_census(p, q.tbin, &q); else p->counters[0]++;
    }
    for (int k = first; k < in->n_t && p->error != -3; k++) {
        uint64_t M = p->n_cbank[k];
        particle *B = p->cbank[k];
        qsort(B, (size_t)M, sizeof(particle), cmp_particle_id);
        double W = 0.0;
        for (uint64_t i = 0; i < M; i++) W += B[i].w;
        if (p->n_census < 64) { p->census_counts[2 * p->n_census] = M; p->census_weights[2 * p->n_census] = W; }
        particle *run = B;
        uint64_t n_run = M;
        if (in->census_target > 0 && k > first && M > 0) {
            uint64_t T = (uint64_t)in->census_target;
            double *w = (double *)malloc((size_t)M * sizeof(double));
            uint32_t *copies = (uint32_t *)malloc((size_t)M * sizeof(uint32_t));
            for (uint64_t i = 0; i < M; i++) w[i] = B[i].w;
            double xi = orc_draw(seed, (uint64_t)k, 3u, 0u, 0u); /* the comb's own stream: domain 3, id = interval */
            double delta = orc_comb(w, M, T, xi, copies);
            run = (particle *)malloc((size_t)T * sizeof(particle));
            n_run = 0;
            for (uint64_t i = 0; i < M; i++)
                for (uint32_t c = 0; c < copies[i]; c++) {
                    particle q = B[i];
                    q.w = delta;
                    /* every copy is a new track with a stream of its own: id from the domain-2 block
                     * (parent id, interval, copy index) */
                    uint32_t ctr[4] = {(uint32_t)B[i].id, (uint32_t)(B[i].id >> 32), (2u << 24) | (uint32_t)k, c};
                    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
                    uint32_t o[4];
                    orc_philox4x32_10(ctr, key, o);
                    q.id = ((uint64_t)o[1] << 32) | o[0];
                    q.ctr = 0; q.nseg = 0; q.resumed = 1;
                    run[n_run++] = q;
                }
            free(w); free(copies);
            W = delta * (double)n_run;
        }
        if (p->n_census < 64) { p->census_counts[2 * p->n_census + 1] = n_run; p->census_weights[2 * p->n_census + 1] = W; p->n_census++; }
        for (uint64_t i = 0; i < n_run; i++) {
            particle q = run[i];
            transport(p, &q);
            while (p->n_stack > 0) {
                /* R25a with population control: the comb re-seeds every interval with census_target particles */
                if (p->counters[11] > 64 * (N + (uint64_t)in->census_target * (uint64_t)in->n_t) + 4096) { p->error = -3; p->n_stack = 0; break; }
                particle c = p->stack[--p->n_stack];
                transport(p, &c);
            }
            if (p->error == -3) break;
        }
        if (run != B) free(run);
    }
    p->census_stop = 0;
    if (p->error == -3) return p->error;
    accumulate_cycle(p, N, 1);
    return p->error;
}

int orc_get_census(const orc_problem *p, uint64_t *counts, double *weights, int max_intervals)
{
    int n = p->n_census < max_intervals ? p->n_census : max_intervals;
    for (int i = 0; i < 2 * n; i++) { counts[i] = p->census_counts[i]; weights[i] = p->census_weights[i]; }
    return n;
}

int orc_get_results(const orc_problem *p, double *k_cycle, double *k_mean, double *k_sdev, double *flux_mean,
                    double *flux_sdev, double *leak_mean, double *leak_sdev, uint64_t *counters)
{
    int64_t nt = orc_n_tally(p);
    int n = p->n_active_done;
    for (int c = 0; c < p->n_cycles; c++) k_cycle[c] = p->k_cycle[c];
    double dn = n > 0 ? (double)n : 1.0;
    *k_mean = p->k_acc / dn;
    *leak_mean = p->leak_acc / dn;
    double var = p->k_acc2 / dn - (*k_mean) * (*k_mean);
    *k_sdev = n > 1 && var > 0.0 ? sqrt(var / (n - 1)) : 0.0;
    var = p->leak_acc2 / dn - (*leak_mean) * (*leak_mean);
    *leak_sdev = n > 1 && var > 0.0 ? sqrt(var / (n - 1)) : 0.0;
    for (int64_t i = 0; i < nt; i++) {
        double m = p->flux_acc[i] / dn;
        flux_mean[i] = m;
        var = p->flux_acc2[i] / dn - m * m;
        flux_sdev[i] = n > 1 && var > 0.0 ? sqrt(var / (n - 1)) : 0.0;
    }
    memcpy(counters, p->counters, sizeof(p->counters));
    return p->error;
}

void orc_get_balance(const orc_problem *p, double out[6])
{
    for (int k = 0; k < 6; k++) out[k] = p->balance[k];
}

uint64_t orc_get_trace(const orc_problem *p, orc_trace_rec *out, uint64_t max)
{
    uint64_t n = p->tr_count < p->tr_max ? p->tr_count : p->tr_max;
    if (n > max) n = max;
    if (out && n) memcpy(out, p->trace, (size_t)n * sizeof(orc_trace_rec));
    return p->tr_count;
}

uint64_t orc_get_bank(const orc_problem *p, orc_site *out, uint64_t max)
{
    uint64_t n = p->n_bank < max ? p->n_bank : max;
    if (out && n) memcpy(out, p->bank, (size_t)n * sizeof(orc_site));
    return p->n_bank;
}
