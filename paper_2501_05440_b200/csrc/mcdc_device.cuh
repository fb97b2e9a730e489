// mcdc_device.cuh -- device-side data layout and per-particle device functions of the B200 transport
// library (include/mcdc.h).  Written from the readings R1..R40 of DESIGN.md section 3 (= SURVEY.md 8c);
// shares no code with oracle/.  float64 everywhere.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mcdc {

constexpr int CE_ROW = 8;          // doubles per (material, grid point) row of the macroscopic CE table
constexpr int MAX_CE_COL = 6;      // cumulative columns kept per row: [el_1..el_n, fission, capture], n <= 4
constexpr int RING = 8;            // per-sweep queue-counter sets kept alive for the lagging host read-back
constexpr unsigned int MAX_SEGMENTS = 1000000u;  // lost-particle guard (R11): segments per history

// Pending event of a banked particle (low 12 bits of Bank::ev; the high 20 bits count the history's segments):
// a surface / lattice-wall hit code (< PEND_SCATTER), an elastic / group-transfer scatter (PEND_SCATTER | column),
// a time edge, or nothing.  The event is FINISHED by whichever kernel picks the particle up next.
constexpr unsigned int PEND_SCATTER = 0xF00u, PEND_TIME = 0xFFEu, PEND_NONE = 0xFFFu, PEND_MASK = 0xFFFu;
constexpr int MAX_SURFACES = 3800;  // hit codes 0 .. n_surf+3 must stay below PEND_SCATTER

// ------------------------------------------------------------------ layout in HBM
// Geometry: small read-only tables in the workspace (L1/L2 resident).
// Straight-line geometry path: where the boundaries of the current location are axis planes (at most one per
// direction of flight), lattice walls and at most one z-cylinder, the nearest boundary is found without loops:
//   lat_info[e] (lattice element e; one 16-byte load per segment): x = universe of the element | LAT_FAST, y = tally
//     bin of the element, z = boundary code per direction -x,+x,-y,+y (8 bits each), w = codes for -z,+z.
//   cell_info[c] (cell c outside a lattice): x = CELL_FAST | the cell across the cylinder (or CELL_NO_NEIGHBOUR),
//     y = the cell's z-cylinder (or -1), z / w = boundary codes as above.
//   Code 0: nothing can be hit that way; 1: a lattice wall that is an event (R14); 2+j: axis plane j of the problem
//   (ap_pos, ap_sid).  The cylinder of a lattice element is its universe's (ufast).
// Locations without the flag use the generic loops; for lattice elements with lat_rmask (bit j = surface j of the
// enclosing cell's list can be the nearest boundary; built at create).
struct Geo {
    int n_surf, n_cell, n_univ, has_lat, lat_nx, lat_ny, lat_cell, n_ap;
    unsigned int lat_magic;  // floor(2^32 / lat_nx) + 1: elem / lat_nx == umulhi(elem, lat_magic) (lat_nx >= 2)
    double lat_x0, lat_y0, lat_px, lat_py;
    const int *surf_type, *surf_bc;
    const double *surf_param;  // [n_surf][4]
    const int *cso, *csi, *css, *cft, *cfill, *cbin, *uco;
    const int4 *lat_info, *cell_info;
    const unsigned int *lat_rmask;
    const int4 *ufast;      // per universe: x bit 0 = it is one cell, or two cells split by one CYL_Z (bit 1: which lies
                            // strictly inside every lattice element that can hold the universe); y = that
                            // cylinder (or -1); z = cell inside it (or the only cell); w = cell outside it
    const double *ap_pos;   // [n_ap] position of axis plane j
    const int *ap_sid;      // [n_ap] its surface id
    // Second-level lattices (R37): lattice k fills the cell umid[u] (fill type 2, cfill = k) of universe u, centred on
    // the origin of u's coordinates.  A location packs (first-level element | (second-level element + 1) << 20); a
    // first-level element that holds a second-level lattice is never LAT_FAST (generic geometry path).
    int n_lat2;
    const int *l2_nx, *l2_ny, *l2_off, *l2_univ, *l2_bin, *umid;
    const int4 *l2_info;
    const double *l2_px, *l2_py;
};
constexpr int INNER_SHIFT = 20;
constexpr int HIT_BITS = 12;  // hit codes (surfaces, lattice walls) are below PEND_SCATTER < 2^12
__device__ __forceinline__ int outer_of(const Geo &, int elem) { return elem & ((1 << INNER_SHIFT) - 1); }
__device__ __forceinline__ int inner_of(const Geo &, int elem) { return (elem >> INNER_SHIFT) - 1; }
constexpr int LAT_FAST = 1 << 30, CELL_FAST = 1 << 30, CELL_NO_NEIGHBOUR = (1 << 30) - 1;
// LAT_FAST2 (lat_info[e].x): the element's universe is ONE cell without surfaces filled by second-level lattice k
// (k in the high 16 bits of lat_info[e].w; for the other elements those bits hold the universe's z-cylinder + 1)
// and the enclosing cell's surfaces fit the boundary-code pattern: elements
// of that lattice whose own universe is simple (l2_info[..].x & LAT_FAST) take the two-level straight-line path.
// l2_info[l2_off[k] + i]: x = universe | LAT_FAST, y = tally-bin offset, z = codes for -x,+x,-y,+y: 1 = second-level
// wall (an event), 3 = the lattice's rim (the first-level element's code for that direction applies).
constexpr int LAT_FAST2 = 1 << 29, UNIV_MASK = (1 << 29) - 1;

struct MGTab {  // [n_mat][G] each; cumS [n_mat][G][G] running row sums; cumchi running chi sums.  One contiguous
    int G, n_mat, blob_doubles;  // blob: the transport kernels copy it to shared memory when it fits
    const double *blob;
    int o_sig_t, o_sig_s, o_sig_f, o_nu, o_nusf, o_cumS, o_cumchi, o_src_cum;  // offsets (doubles) into the blob
    int half;     // largest power of two <= G - 1 (0 for one group): first step of the group-transfer bisection
    int o_inv_t;  // 1 / Sigma_t: the distance to collision is -ln(xi) * (1 / Sigma_t), one multiply instead of a division
};

struct CETab {
    int n_grid, n_mat, n_t, n_e, search;
    const double *grid;
    const double *tab;    // [n_mat][n_grid][CE_ROW]: cumulative macroscopic columns, the grid energy in slot 6, Sigma_f in 7
    const int *ncol;      // [n_mat] number of cumulative columns (= n_nuclides + 2)
    const double *colA;   // [n_mat][CE_ROW] mass ratio A of the nuclide behind elastic column j
    const double *t_edges, *e_edges;
    const int *hash;      // [n_hash+1] bucket b -> last grid index <= lower edge of the bucket
    int hash_shift, hash_lo, n_hash;
    const int *ehash;     // the same for the energy-bin edges of the tally: bucket -> last edge index <= its lower edge
    int ehash_shift, ehash_lo, n_ehash;
    double nu0, nu1, watt_a, watt_b, E_min, E_max;
};

// Particle banks ("dual particle banks"): two dense structure-of-arrays banks.  A sweep reads the
// live particles of bank[s&1] (scatter-pending ones packed at the FRONT, surface-pending ones at the BACK) and
// writes every survivor, whole, to the front or the back of bank[(s+1)&1]: the queues hold the particles
// themselves, so every load and store is coalesced.
// gl packs the group (low 16 bits) and last_surf+1 (high 16 bits); ev = pending event | segments << 12;
// slot = index of the particle inside its cycle / wave (= its id in eigenvalue mode, R6).
struct Bank {
    double *x, *y, *z, *ux, *uy, *uz, *E, *t;
    double *w;  // statistical weight (implicit capture, R36); the analog path never touches it (R2: w = w0)
    int *cell, *elem, *gl, *tbin;
    uint32_t *ev, *ctr, *slot;
    uint64_t *id;
};

// What a fission leaves behind, indexed by the parent's slot: number of children, the site, the parent's
// location and draw counter (the parent's stream continues in k_emit, R5).
struct FisRec {
    int *n, *cell, *elem, *tbin;
    double *x, *y, *z, *t;
    uint32_t *ctr;
    uint64_t *id;
};

// Time-dependent multi-group (R38-R40): group speeds, cumulative fission yields [prompt, +delayed 1 .. +delayed J] per
// (material, group), delayed emission spectra (running sums) and decay constants per (material, precursor group).
// The time edges are CETab::t_edges / n_t for both energy treatments.
struct TDTab {
    int on, J;
    const double *speed, *cum_nu, *cumchi_d, *decay;
};

struct QCount {  // one set per sweep (ring of RING)
    unsigned int n_scat, n_surf, n_alive, err;
};

struct Trace {
    unsigned long long first, n_ids;
    unsigned int max_events, cap_slots;  // cap_slots = (cycle, id) slots available
    void *rec;                           // mcdc_trace_rec[cap_slots][max_events]
    unsigned int *count;                 // [cap_slots]
};

struct Ctx {
    Geo geo;
    MGTab mg;
    CETab ce;
    Bank bank[2];
    Bank cbank;          // census bank (R40): particles that wait for a later census interval; count in work[4]
    int census_stop;     // a particle that reaches a time edge (not the last) goes to the census bank instead of going on
    TDTab td;
    FisRec fis;
    unsigned int cap;   // slots per bank
    int mode;           // 0 MG, 1 CE
    int n_tally, n_bins;
    int mg_stage;        // doubles of the multi-group table blob staged in shared memory by every transport kernel (0: none)
    int flux_aggregate;  // global tally flavour: 1 = warp-aggregate equal bins before the atomic
    int flux_copy_mask;  // R - 1: the per-cycle tally is kept in R copies, copy = block index & mask
    double *flux;       // [R][n_tally] per-cycle track-length tally
    double *scal;       // [0] k numerator, [1] leakage weight
    unsigned long long *counters;  // [16]
    int *err;           // device error flag
    QCount *qc;          // [RING] per-sweep counts of the front / back regions
    unsigned int *work;  // persistent kernel: queue head, secondaries pushed, histories ended, secondaries born
    unsigned long long max_secondaries;  // R25a: more prompt secondaries than this = bank overflow
    Trace tr;
    const Trace *tr_g;   // copy of tr in global memory for the out-of-line trace_event (see Acc::geo)
    unsigned long long seed;
    uint32_t rk[20];     // the ten Philox round keys of the seed (rk[2r], rk[2r+1]): launch constants read straight from the
                         // kernel-parameter bank by the XORs of the rounds (no key-bump additions in the draw path)
    unsigned int cycle;
    double w0, k_prev;
    // options set by mcdc_set_physics: free-gas thermal scattering below 400 kT (R35; kT in eV, 0 = target at rest),
    // implicit capture with weight roulette (R36)
    double kT, w_roulette, w_survive;
    int implicit;
    int src_iso;
    double src_lo[3], src_hi[3], src_dir[3], src_E, src_t;
};

// ------------------------------------------------------------------ RNG (R9, R10)
// Philox4x32-10: 10 rounds of two 32x32->64 multiplies, xors with the counter words and key, key bumps.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

#ifndef MCDC_INV_SIGT
#define MCDC_INV_SIGT 1
#endif
#ifndef MCDC_NEXT_PRE
#define MCDC_NEXT_PRE 1
#endif
#ifndef MCDC_NEXT3
#define MCDC_NEXT3 1
#endif
#ifndef MCDC_GROUP_COUNT
#define MCDC_GROUP_COUNT 2
#endif
// the same with the round keys precomputed (Ctx::rk)
__device__ __forceinline__ void philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t (&rk)[20],
                                                 uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ rk[2 * r];
        c1 = l1;
        c2 = h0 ^ c3 ^ rk[2 * r + 1];
        c3 = l0;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

// Stream (seed, id, domain 0, cycle): counter = (id_lo, id_hi, cycle, draw/2); one block yields the draws 2b
// (words 1:0) and 2b+1 (words 3:2); xi = ((u >> 11) + 0.5) 2^-53.  The block is kept in registers so that two
// consecutive draws cost one Philox evaluation; seed and cycle are launch constants read from the Ctx at use.
// (A buffer of the segment's 5 draws filled at one code site was measured: 3 instead of ~5 Philox evaluations per
// warp and segment, but 8 more live registers and the selects to read it: 31.0 instead of 29.9 ms per C4 cycle.)
// (One out-of-line copy of the ten rounds called from every draw site -- 5 % less code -- was measured as well:
// 31.5 instead of 29.8 ms per C4 cycle, C5 unchanged; profiles/r02_experiments.md.)
struct Rng {
    unsigned long long id;
    uint32_t ctr, blk;
    uint64_t u0, u1;
    __device__ __forceinline__ void init(unsigned long long id_, uint32_t ctr_)
    {
        id = id_; ctr = ctr_; blk = 0xFFFFFFFFu;
    }
    __device__ __forceinline__ double next(const Ctx &c)
    {
        uint32_t b = ctr >> 1;
        if (b != blk) {
            uint32_t o0, o1, o2, o3;
            philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), c.cycle, b, c.rk, o0, o1, o2, o3);
            u0 = ((uint64_t)o1 << 32) | o0;
            u1 = ((uint64_t)o3 << 32) | o2;
            blk = b;
        }
        uint64_t u = (ctr & 1u) ? u1 : u0;
        ctr++;
        return ((double)(u >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    }
    // The first draw of a segment (distance to collision), leaving the block of the draw AFTER it in the cache: a lane
    // at an even draw index evaluates its block (both draws in it), a lane at an odd index takes its cached word and
    // evaluates the NEXT block -- one evaluation site reached by every lane of the warp together, and the reaction draw
    // (or the next segment's first draw) finds its block cached whatever the parity.
    __device__ __forceinline__ double next_pre(const Ctx &c)
    {
        const uint32_t b = ctr >> 1;
        const bool odd = (ctr & 1u) != 0u;
        uint32_t o0, o1, o2, o3;
        if (odd && b != blk) {  // no cached block to take the odd word from (a particle just loaded): rare
            philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), c.cycle, b, c.rk, o0, o1, o2, o3);
            u1 = ((uint64_t)o3 << 32) | o2;
            blk = b;
        }
        const uint64_t old1 = u1;
        if (odd || b != blk) {
            const uint32_t bb = odd ? b + 1u : b;
            philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), c.cycle, bb, c.rk, o0, o1, o2, o3);
            u0 = ((uint64_t)o1 << 32) | o0;
            u1 = ((uint64_t)o3 << 32) | o2;
            blk = bb;
        }
        const uint64_t u = odd ? old1 : u0;
        ctr++;
        return ((double)(u >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    }
    // The next TWO draws at once (a continuous-energy elastic scatter: mu_cm, azimuth): one evaluation site for every
    // lane -- an even draw index evaluates its own block (both draws), an odd one takes its cached word and evaluates
    // the next block for the second draw.
    __device__ __forceinline__ void next2(const Ctx &c, double &x0, double &x1)
    {
        const uint32_t b = ctr >> 1;
        const bool odd = (ctr & 1u) != 0u;
        uint32_t o0, o1, o2, o3;
        if (odd && b != blk) {
            philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), c.cycle, b, c.rk, o0, o1, o2, o3);
            u1 = ((uint64_t)o3 << 32) | o2;
            blk = b;
        }
        const uint64_t old1 = u1;
        if (odd || b != blk) {
            const uint32_t bb = odd ? b + 1u : b;
            philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), c.cycle, bb, c.rk, o0, o1, o2, o3);
            u0 = ((uint64_t)o1 << 32) | o0;
            u1 = ((uint64_t)o3 << 32) | o2;
            blk = bb;
        }
        const uint64_t a0 = odd ? old1 : u0, a1 = odd ? u0 : u1;
        ctr += 2u;
        const double sc = 1.0 / 9007199254740992.0;
        x0 = ((double)(a0 >> 11) + 0.5) * sc;
        x1 = ((double)(a1 >> 11) + 0.5) * sc;
    }
    // The next THREE draws at once (a multi-group scatter: group, mu, phi).  They span the blocks b = ctr / 2 and b + 1
    // whatever the parity: block b + 1 is evaluated by every lane together, block b only by the lanes that do not hold
    // it -- two evaluations per warp where three separate next() calls make three (each reached by half the lanes).
    __device__ __forceinline__ void next3(const Ctx &c, double &x0, double &x1, double &x2)
    {
        const uint32_t b = ctr >> 1;
        uint32_t o0, o1, o2, o3;
        if (b != blk) {
            philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), c.cycle, b, c.rk, o0, o1, o2, o3);
            u0 = ((uint64_t)o1 << 32) | o0;
            u1 = ((uint64_t)o3 << 32) | o2;
        }
        philox4x32_10_rk((uint32_t)id, (uint32_t)(id >> 32), c.cycle, b + 1u, c.rk, o0, o1, o2, o3);
        const uint64_t v0 = ((uint64_t)o1 << 32) | o0, v1 = ((uint64_t)o3 << 32) | o2;
        const bool odd = (ctr & 1u) != 0u;
        const uint64_t a0 = odd ? u1 : u0, a1 = odd ? v0 : u1, a2 = odd ? v1 : v0;
        u0 = v0; u1 = v1; blk = b + 1u;
        ctr += 3u;
        const double sc = 1.0 / 9007199254740992.0;
        x0 = ((double)(a0 >> 11) + 0.5) * sc;
        x1 = ((double)(a1 >> 11) + 0.5) * sc;
        x2 = ((double)(a2 >> 11) + 0.5) * sc;
    }
};

// one draw of an arbitrary stream (unit-level entry point)
__device__ __forceinline__ double draw_at(unsigned long long seed, unsigned long long id, uint32_t domain, uint32_t cycle,
                                          uint32_t index)
{
    uint32_t o0, o1, o2, o3;
    philox4x32_10((uint32_t)id, (uint32_t)(id >> 32), (domain << 24) | cycle, index >> 1, (uint32_t)seed,
                  (uint32_t)(seed >> 32), o0, o1, o2, o3);
    uint64_t u = (index & 1u) ? (((uint64_t)o3 << 32) | o2) : (((uint64_t)o1 << 32) | o0);
    return ((double)(u >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

__device__ __forceinline__ unsigned long long child_id(unsigned long long seed, unsigned long long parent, uint32_t parent_ctr,
                                                       uint32_t j)
{
    uint32_t o0, o1, o2, o3;
    philox4x32_10((uint32_t)parent, (uint32_t)(parent >> 32), (1u << 24) | j, parent_ctr, (uint32_t)seed,
                  (uint32_t)(seed >> 32), o0, o1, o2, o3);
    return ((unsigned long long)o1 << 32) | o0;
}

// ------------------------------------------------------------------ sampling helpers
// isotropic direction (R8): mu = 2 xi1 - 1, phi = 2 pi xi2
__device__ __forceinline__ void iso_dir(double xi_mu, double xi_phi, double &ux, double &uy, double &uz)
{
    double mu = 2.0 * xi_mu - 1.0;
    double s = sqrt(1.0 - mu * mu);
    double sp, cp;
    sincospi(2.0 * xi_phi, &sp, &cp);
    ux = s * cp; uy = s * sp; uz = mu;
}

// first index with cum[i] > v, else n-1 (R3); cum in global memory
__device__ __forceinline__ int pick(const double *__restrict__ cum, int n, double v)
{
    int i = 0;
    while (i < n - 1 && !(__ldg(cum + i) > v)) i++;
    return i;
}

// largest b with edges[b] <= v, clamped to [0, n-1] (R24: bisection on the edge array, never a log)
__device__ __forceinline__ int edge_bin(const double *__restrict__ edges, int n, double v)
{
    int lo = 0, hi = n;
    if (v < __ldg(edges)) return 0;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(edges + mid) <= v) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ double speed_of(double E)  // R23
{
    return 2.99792458e10 * sqrt(2.0 * E / 939.56542052e6);
}

// ------------------------------------------------------------------ union-grid search (R19, R20)
__device__ __forceinline__ int grid_bisect(const double *__restrict__ g, int lo, int hi, double E)
{
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(g + mid) <= E) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ int grid_index_binary(const CETab &ce, double E)
{
    if (E < ce.E_min) return 0;
    return grid_bisect(ce.grid, 0, ce.n_grid - 1, E);
}

// Hashed search: the bucket key is the top bits of the IEEE-754 representation of E (exponent plus
// (52 - hash_shift) mantissa bits), an exact monotone function of E, so the bucket brackets the answer
// without any floating-point logarithm and the result equals the bisection index bit for bit.
__device__ __forceinline__ int grid_index_hash(const CETab &ce, double E)
{
    if (E < ce.E_min) return 0;
    if (E >= ce.E_max) return ce.n_grid - 2;
    int b = (int)(__double_as_longlong(E) >> ce.hash_shift) - ce.hash_lo;
    int lo = __ldg(ce.hash + b), hi = __ldg(ce.hash + b + 1) + 1;
    if (hi > ce.n_grid - 1) hi = ce.n_grid - 1;
    if (hi <= lo) return lo < ce.n_grid - 2 ? lo : ce.n_grid - 2;
    return grid_bisect(ce.grid, lo, hi, E);
}

__device__ __forceinline__ int grid_index(const CETab &ce, double E)
{
    return ce.search ? grid_index_hash(ce, E) : grid_index_binary(ce, E);
}

// tally energy bin (R24: the largest b with e_edges[b] <= E, clamped): the same exact bucket key narrows the
// bisection to the one or two edges that can fall in the bucket; equals edge_bin(e_edges, n_e, E) bit for bit
__device__ __forceinline__ int energy_bin(const CETab &ce, double E)
{
    if (E < __ldg(ce.e_edges)) return 0;
    if (E >= __ldg(ce.e_edges + ce.n_e)) return ce.n_e - 1;
    int b = (int)(__double_as_longlong(E) >> ce.ehash_shift) - ce.ehash_lo;
    int lo = __ldg(ce.ehash + b), hi = __ldg(ce.ehash + b + 1) + 1;
    if (hi > ce.n_e) hi = ce.n_e;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(ce.e_edges + mid) <= E) lo = mid; else hi = mid;
    }
    return lo < ce.n_e - 1 ? lo : ce.n_e - 1;
}

// ------------------------------------------------------------------ geometry (R11-R14)
struct Particle;
__device__ __forceinline__ double surf_f(const Geo &G, int s, double x, double y, double z)
{
    const double *q = G.surf_param + 4 * s;
    int t = __ldg(G.surf_type + s);
    double q0 = __ldg(q), q1 = __ldg(q + 1), q2 = __ldg(q + 2), q3 = __ldg(q + 3);
    switch (t) {
    case 0: return x - q0;
    case 1: return y - q0;
    case 2: return z - q0;
    case 3: return q0 * x + q1 * y + q2 * z - q3;
    case 4: { double a = y - q0, b = z - q1; return a * a + b * b - q2 * q2; }
    case 5: { double a = x - q0, b = z - q1; return a * a + b * b - q2 * q2; }
    case 6: { double a = x - q0, b = y - q1; return a * a + b * b - q2 * q2; }
    default: { double a = x - q0, b = y - q1, c = z - q2; return a * a + b * b + c * c - q3 * q3; }
    }
}

// grad f (unnormalised outward normal)
__device__ __forceinline__ void surf_normal(const Geo &G, int s, double x, double y, double z, double &nx, double &ny,
                                            double &nz)
{
    const double *q = G.surf_param + 4 * s;
    int t = __ldg(G.surf_type + s);
    double q0 = __ldg(q), q1 = __ldg(q + 1), q2 = __ldg(q + 2);
    nx = ny = nz = 0.0;
    switch (t) {
    case 0: nx = 1.0; break;
    case 1: ny = 1.0; break;
    case 2: nz = 1.0; break;
    case 3: nx = q0; ny = q1; nz = q2; break;
    case 4: ny = y - q0; nz = z - q1; break;
    case 5: nx = x - q0; nz = z - q1; break;
    case 6: nx = x - q0; ny = y - q1; break;
    default: nx = x - q0; ny = y - q1; nz = z - q2; break;
    }
}

// side of s the particle is on; if it sits on s (s == last) the side it is heading into (R11)
__device__ __forceinline__ int sense_of(const Geo &G, int s, double x, double y, double z, double ux, double uy, double uz,
                                        int last)
{
    if (s == last) {
        double nx, ny, nz;
        surf_normal(G, s, x, y, z, nx, ny, nz);
        return (ux * nx + uy * ny + uz * nz) > 0.0 ? 1 : -1;
    }
    return surf_f(G, s, x, y, z) > 0.0 ? 1 : -1;
}

// first cell of universe `univ` all of whose (surface, sense) pairs match; -1 if none
__device__ __forceinline__ int find_cell(const Geo &G, int univ, double x, double y, double z, double ux, double uy,
                                         double uz, int last)
{
    int c1 = __ldg(G.uco + univ + 1);
    for (int c = __ldg(G.uco + univ); c < c1; c++) {
        bool ok = true;
        int k1 = __ldg(G.cso + c + 1);
        for (int k = __ldg(G.cso + c); k < k1; k++)
            if (sense_of(G, __ldg(G.csi + k), x, y, z, ux, uy, uz, last) != __ldg(G.css + k)) { ok = false; break; }
        if (ok) return c;
    }
    return -1;
}

// lattice element -> (ix, iy) without an integer division (a one-column lattice has iy = elem)
__device__ __forceinline__ void elem_xy(const Geo &G, int elem, int &ix, int &iy)
{
    iy = G.lat_nx == 1 ? elem : (int)__umulhi((unsigned int)elem, G.lat_magic);
    ix = elem - iy * G.lat_nx;
}

// element-centred coordinates, recomputed from the global position every time (R14)
__device__ __forceinline__ void local_xy(const Geo &G, int elem, double x, double y, double &xl, double &yl)
{
    int ix, iy;
    elem_xy(G, elem, ix, iy);
    xl = x - (G.lat_x0 + (ix + 0.5) * G.lat_px);
    yl = y - (G.lat_y0 + (iy + 0.5) * G.lat_py);
}

__device__ __forceinline__ int elem_universe(const Geo &G, int elem) { return __ldg(&G.lat_info[elem].x) & UNIV_MASK; }

// second-level lattice k: lower-left corner in its universe's coordinates (centred on the origin, R37)
__device__ __forceinline__ double l2_x0(const Geo &G, int k) { return -0.5 * (__ldg(G.l2_nx + k) * __ldg(G.l2_px + k)); }
__device__ __forceinline__ double l2_y0(const Geo &G, int k) { return -0.5 * (__ldg(G.l2_ny + k) * __ldg(G.l2_py + k)); }

// coordinates centred on element `inner` of second-level lattice k, from first-level-element coordinates (xo, yo)
__device__ __forceinline__ void inner_xy(const Geo &G, int k, int inner, double xo, double yo, double &xl, double &yl)
{
    const int nx = __ldg(G.l2_nx + k);
    const int jy = inner / nx, jx = inner - jy * nx;
    xl = xo - (l2_x0(G, k) + (jx + 0.5) * __ldg(G.l2_px + k));
    yl = yo - (l2_y0(G, k) + (jy + 0.5) * __ldg(G.l2_py + k));
}

// coordinates of the innermost lattice level of the packed location `elem`
__device__ __forceinline__ void innermost_xy(const Geo &G, int elem, double x, double y, double &xl, double &yl)
{
    const int outer = outer_of(G, elem), inner = inner_of(G, elem);
    local_xy(G, outer, x, y, xl, yl);
    if (inner >= 0) {
        const double xo = xl, yo = yl;
        inner_xy(G, __ldg(G.cfill + __ldg(G.umid + elem_universe(G, outer))), inner, xo, yo, xl, yl);
    }
}

// cell of first-level element `outer` that holds the point (xo, yo, z) given in that element's coordinates, descending
// into a second-level lattice where one fills the cell; the second-level index is found by floor and clamped to the
// lattice (R37).  elem = packed location; returns the material cell or -1.
__device__ __forceinline__ int descend(const Geo &G, int outer, double xo, double yo, double z, double ux, double uy, double uz,
                                       int last, int &elem)
{
    elem = outer;
    int c = find_cell(G, elem_universe(G, outer), xo, yo, z, ux, uy, uz, last);
    if (c < 0 || G.n_lat2 == 0 || __ldg(G.cft + c) != 2) return c;
    const int k = __ldg(G.cfill + c);
    const int nx = __ldg(G.l2_nx + k), ny = __ldg(G.l2_ny + k);
    int jx = (int)floor((xo - l2_x0(G, k)) / __ldg(G.l2_px + k));
    int jy = (int)floor((yo - l2_y0(G, k)) / __ldg(G.l2_py + k));
    jx = jx < 0 ? 0 : (jx > nx - 1 ? nx - 1 : jx);
    jy = jy < 0 ? 0 : (jy > ny - 1 ? ny - 1 : jy);
    const int inner = jy * nx + jx;
    double xl, yl;
    inner_xy(G, k, inner, xo, yo, xl, yl);
    elem = outer | ((inner + 1) << INNER_SHIFT);
    return find_cell(G, __ldg(G.l2_univ + __ldg(G.l2_off + k) + inner), xl, yl, z, ux, uy, uz, last);
}

// full point location from the root universe.  cell = material cell (root cell, or the local cell inside
// lattice element elem); returns false if the point is in no cell.
__device__ __forceinline__ bool locate(const Geo &G, double x, double y, double z, double ux, double uy, double uz, int last,
                                       int &cell, int &elem)
{
    elem = -1;
    cell = find_cell(G, 0, x, y, z, ux, uy, uz, last);
    if (cell < 0) return false;
    if (__ldg(G.cft + cell) == 1) {
        int ix = (int)floor((x - G.lat_x0) / G.lat_px);
        int iy = (int)floor((y - G.lat_y0) / G.lat_py);
        if (ix < 0 || iy < 0 || ix >= G.lat_nx || iy >= G.lat_ny) { cell = -1; return false; }
        double xl, yl;
        local_xy(G, iy * G.lat_nx + ix, x, y, xl, yl);
        cell = descend(G, iy * G.lat_nx + ix, xl, yl, z, ux, uy, uz, last, elem);
        if (cell < 0) return false;
    }
    return true;
}

// positive ray distance to surface s (infinity = miss); on: the particle sits on s (R11-R13)
// inv_ux, inv_uy = 1/ux, 1/uy computed once per segment (axis planes and lattice walls share them)
__device__ __forceinline__ double surf_distance(const Geo &G, int s, double x, double y, double z, double ux, double uy,
                                                double uz, bool on, double inv_ux, double inv_uy)
{
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    const double *q = G.surf_param + 4 * s;
    int t = __ldg(G.surf_type + s);
    double q0 = __ldg(q), q1 = __ldg(q + 1), q2 = __ldg(q + 2), q3 = __ldg(q + 3);
    if (t <= 3) {
        if (on) return INF;
        double d;
        if (t == 0) { if (ux == 0.0) return INF; d = (q0 - x) * inv_ux; }
        else if (t == 1) { if (uy == 0.0) return INF; d = (q0 - y) * inv_uy; }
        else {
            double num, den;
            if (t == 2) { num = q0 - z; den = uz; }
            else { num = q3 - (q0 * x + q1 * y + q2 * z); den = q0 * ux + q1 * uy + q2 * uz; }
            if (den == 0.0) return INF;
            d = num / den;
        }
        return d > 0.0 ? d : INF;
    }
    double a, k, c;
    if (t == 7) {
        double dx = x - q0, dy = y - q1, dz = z - q2;
        a = 1.0;
        k = dx * ux + dy * uy + dz * uz;
        c = dx * dx + dy * dy + dz * dz - q3 * q3;
    } else {
        double pa, pb, va, vb;
        if (t == 4) { pa = y; pb = z; va = uy; vb = uz; }
        else if (t == 5) { pa = x; pb = z; va = ux; vb = uz; }
        else { pa = x; pb = y; va = ux; vb = uy; }
        double da = pa - q0, db = pb - q1;
        a = va * va + vb * vb;
        k = da * va + db * vb;
        c = da * da + db * db - q2 * q2;
    }
    if (a == 0.0) return INF;
    if (on) {  // c is exactly 0: only the far root, only when heading inward
        if (k >= 0.0) return INF;
        double d = -2.0 * k / a;
        return d > 0.0 ? d : INF;
    }
    double disc = k * k - a * c;
    if (disc < 0.0) return INF;
    double sq = sqrt(disc);
    double d = c < 0.0 ? (-k + sq) / a : (-k - sq) / a;
    return d > 0.0 ? d : INF;
}

// nearest boundary of the current location, generic path; candidate order: enclosing-cell surfaces, local-cell
// surfaces, lattice walls -x,+x,-y,+y; ties keep the first (R12, R14).  hit = surface id, or n_surf+k for wall k.
__device__ __noinline__ double nearest(const Geo &G, double x, double y, double z, double ux, double uy, double uz, int cell,
                                       int elem, int last, int &hit, unsigned int root_mask)
{
    double best = __longlong_as_double(0x7ff0000000000000LL);
    hit = -1;
    const double inv_ux = 1.0 / ux, inv_uy = 1.0 / uy;  // +-inf when the component is zero: guarded at use
    int c0 = elem >= 0 ? G.lat_cell : cell;
    int k1 = __ldg(G.cso + c0 + 1);
    if (root_mask) {
        // candidates in list order (ties keep the first, R12): the listed bits, then anything past the 32nd surface
        const int k0 = __ldg(G.cso + c0);
        unsigned int m = k1 - k0 >= 32 ? root_mask : root_mask & ((1u << (k1 - k0)) - 1u);
        while (m) {
            int s = __ldg(G.csi + k0 + __ffs(m) - 1);
            m &= m - 1u;
            double d = surf_distance(G, s, x, y, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
        for (int k = k0 + 32; k < k1; k++) {
            int s = __ldg(G.csi + k);
            double d = surf_distance(G, s, x, y, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
    }
    if (elem >= 0) {
        int ix, iy;
        elem_xy(G, elem, ix, iy);
        const double xl = x - (G.lat_x0 + (ix + 0.5) * G.lat_px);
        const double yl = y - (G.lat_y0 + (iy + 0.5) * G.lat_py);
        k1 = __ldg(G.cso + cell + 1);
        for (int k = __ldg(G.cso + cell); k < k1; k++) {
            int s = __ldg(G.csi + k);
            double d = surf_distance(G, s, xl, yl, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
        // only the wall ahead on each axis; the lattice's outermost walls are never events (R14)
        if (ux < 0.0 && ix > 0) {
            double d = (G.lat_x0 + ix * G.lat_px - x) * inv_ux;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 0; }
        }
        if (ux > 0.0 && ix + 1 < G.lat_nx) {
            double d = (G.lat_x0 + (ix + 1) * G.lat_px - x) * inv_ux;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 1; }
        }
        if (uy < 0.0 && iy > 0) {
            double d = (G.lat_y0 + iy * G.lat_py - y) * inv_uy;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 2; }
        }
        if (uy > 0.0 && iy + 1 < G.lat_ny) {
            double d = (G.lat_y0 + (iy + 1) * G.lat_py - y) * inv_uy;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 3; }
        }
    }
    return best;
}

// nearest boundary of a location inside a second-level lattice (generic path only); candidate order: enclosing-cell surfaces, [surfaces of the
// cell a second-level lattice fills,] local-cell surfaces, [second-level walls -x,+x,-y,+y,] first-level walls
// -x,+x,-y,+y; ties keep the first (R12, R14, R37).  hit = surface id, n_surf+k for first-level wall k, n_surf+4+k
// for second-level wall k.
__device__ __noinline__ double nearest2(const Geo &G, double x, double y, double z, double ux, double uy, double uz, int cell,
                                       int elem, int last, int &hit, unsigned int root_mask)
{
    double best = __longlong_as_double(0x7ff0000000000000LL);
    hit = -1;
    const double inv_ux = 1.0 / ux, inv_uy = 1.0 / uy;  // +-inf when the component is zero: guarded at use
    int c0 = elem >= 0 ? G.lat_cell : cell;
    int k1 = __ldg(G.cso + c0 + 1);
    if (root_mask) {
        // candidates in list order (ties keep the first, R12): the listed bits, then anything past the 32nd surface
        const int k0 = __ldg(G.cso + c0);
        unsigned int m = k1 - k0 >= 32 ? root_mask : root_mask & ((1u << (k1 - k0)) - 1u);
        while (m) {
            int s = __ldg(G.csi + k0 + __ffs(m) - 1);
            m &= m - 1u;
            double d = surf_distance(G, s, x, y, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
        for (int k = k0 + 32; k < k1; k++) {
            int s = __ldg(G.csi + k);
            double d = surf_distance(G, s, x, y, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
    }
    if (elem >= 0) {
        int ix, iy;
        const int outer = outer_of(G, elem), inner = inner_of(G, elem);
        elem_xy(G, outer, ix, iy);
        const double xo = x - (G.lat_x0 + (ix + 0.5) * G.lat_px);
        const double yo = y - (G.lat_y0 + (iy + 0.5) * G.lat_py);
        double xl = xo, yl = yo;
        int k2 = 0;
        if (inner >= 0) {
            const int mid = __ldg(G.umid + elem_universe(G, outer));
            k1 = __ldg(G.cso + mid + 1);
            for (int k = __ldg(G.cso + mid); k < k1; k++) {
                int s = __ldg(G.csi + k);
                double d = surf_distance(G, s, xo, yo, z, ux, uy, uz, s == last, inv_ux, inv_uy);
                if (d < best) { best = d; hit = s; }
            }
            k2 = __ldg(G.cfill + mid);
            inner_xy(G, k2, inner, xo, yo, xl, yl);
        }
        k1 = __ldg(G.cso + cell + 1);
        for (int k = __ldg(G.cso + cell); k < k1; k++) {
            int s = __ldg(G.csi + k);
            double d = surf_distance(G, s, xl, yl, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
        if (inner >= 0) {
            // second-level walls, in first-level-element coordinates: only the wall ahead, never the outermost ones
            const int nx2 = __ldg(G.l2_nx + k2), ny2 = __ldg(G.l2_ny + k2);
            const double px2 = __ldg(G.l2_px + k2), py2 = __ldg(G.l2_py + k2);
            const int jy = inner / nx2, jx = inner - jy * nx2;
            if (ux < 0.0 && jx > 0) {
                double d = (l2_x0(G, k2) + jx * px2 - xo) * inv_ux;
                if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 4; }
            }
            if (ux > 0.0 && jx + 1 < nx2) {
                double d = (l2_x0(G, k2) + (jx + 1) * px2 - xo) * inv_ux;
                if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 5; }
            }
            if (uy < 0.0 && jy > 0) {
                double d = (l2_y0(G, k2) + jy * py2 - yo) * inv_uy;
                if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 6; }
            }
            if (uy > 0.0 && jy + 1 < ny2) {
                double d = (l2_y0(G, k2) + (jy + 1) * py2 - yo) * inv_uy;
                if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 7; }
            }
        }
        // only the wall ahead on each axis; the lattice's outermost walls are never events (R14)
        if (ux < 0.0 && ix > 0) {
            double d = (G.lat_x0 + ix * G.lat_px - x) * inv_ux;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 0; }
        }
        if (ux > 0.0 && ix + 1 < G.lat_nx) {
            double d = (G.lat_x0 + (ix + 1) * G.lat_px - x) * inv_ux;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 1; }
        }
        if (uy < 0.0 && iy > 0) {
            double d = (G.lat_y0 + iy * G.lat_py - y) * inv_uy;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 2; }
        }
        if (uy > 0.0 && iy + 1 < G.lat_ny) {
            double d = (G.lat_y0 + (iy + 1) * G.lat_py - y) * inv_uy;
            if (d > 0.0 && d < best) { best = d; hit = G.n_surf + 3; }
        }
        if (inner >= 0) {  // the second-level element's tally-bin offset rides on the hit code (R37)
            const int off = __ldg(G.l2_bin + __ldg(G.l2_off + k2) + inner);
            if (off) hit = (hit & ((1 << HIT_BITS) - 1)) | (off << HIT_BITS);
        }
    }
    return best;
}

// Straight-line path (see Geo): per axis ONE candidate, named by the location's boundary code for the direction of
// flight (lattice wall ahead, or an axis plane), plus at most one z-cylinder (centred on the lattice element, or in
// global coordinates outside a lattice).  Same formulas and the same candidate order as `nearest` (planes of the
// cell, cylinder, lattice walls); no loops, no surface-type switch: all lanes do the same work.
__device__ __forceinline__ double nearest_fast(const Geo &G, int codes_xy, int codes_z, int cyl, double x, double y, double z,
                                               double ux, double uy, double uz, int elem, int last, int &hit)
{
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    int ix = 0, iy = 0;
    double cx0 = 0.0, cy0 = 0.0;  // centre of the lattice element (origin of the cylinder's coordinates)
    if (elem >= 0) {
        elem_xy(G, elem, ix, iy);
        cx0 = G.lat_x0 + (ix + 0.5) * G.lat_px;
        cy0 = G.lat_y0 + (iy + 0.5) * G.lat_py;
    }
    const double inv_ux = 1.0 / ux, inv_uy = 1.0 / uy;
    const bool xp = ux > 0.0, yp = uy > 0.0, zp = uz > 0.0;
    const int cx = (codes_xy >> (xp ? 8 : 0)) & 255, cy = (codes_xy >> (yp ? 24 : 16)) & 255, cz = (codes_z >> (zp ? 8 : 0)) & 255;
    double px = G.lat_x0 + (ix + (xp ? 1 : 0)) * G.lat_px, py = G.lat_y0 + (iy + (yp ? 1 : 0)) * G.lat_py, pz = 0.0;
    int hx = G.n_surf + (xp ? 1 : 0), hy = G.n_surf + (yp ? 3 : 2), hz = -1;
    if (cx >= 2) { px = __ldg(G.ap_pos + cx - 2); hx = __ldg(G.ap_sid + cx - 2); }
    if (cy >= 2) { py = __ldg(G.ap_pos + cy - 2); hy = __ldg(G.ap_sid + cy - 2); }
    if (cz >= 2) { pz = __ldg(G.ap_pos + cz - 2); hz = __ldg(G.ap_sid + cz - 2); }
    double dx = (px - x) * inv_ux, dy = (py - y) * inv_uy, dz = INF;
    if (cz >= 2 && uz != 0.0 && hz != last) { dz = (pz - z) / uz; if (!(dz > 0.0)) dz = INF; }
    if (cx == 0 || ux == 0.0 || hx == last || !(dx > 0.0)) dx = INF;
    if (cy == 0 || uy == 0.0 || hy == last || !(dy > 0.0)) dy = INF;
    double dc = INF;
    if (cyl >= 0) {
        const double *q = G.surf_param + 4 * cyl;
        const double da = x - cx0 - __ldg(q);
        const double db = y - cy0 - __ldg(q + 1);
        const double r = __ldg(q + 2);
        const double a = ux * ux + uy * uy, k = da * ux + db * uy;
        // numerator of the root, then ONE division for every lane (on the cylinder: c is exactly 0, only the far root
        // -2k / a, only when heading inward, R13)
        double num = -1.0;
        if (cyl == last) { if (k < 0.0) num = -2.0 * k; }
        else {
            const double cc = da * da + db * db - r * r;
            const double disc = k * k - a * cc;
            if (disc >= 0.0) {
                const double sq = sqrt(disc);
                num = cc < 0.0 ? sq - k : -k - sq;
            }
        }
        if (a != 0.0 && num > 0.0) {
            dc = num / a;
            if (!(dc > 0.0)) dc = INF;
        }
    }
    // candidate order (ties keep the first, R12): the cell's planes, the cylinder, lattice walls
    double best = INF;
    hit = -1;
    if (cx >= 2 && dx < best) { best = dx; hit = hx; }
    if (cy >= 2 && dy < best) { best = dy; hit = hy; }
    if (dz < best) { best = dz; hit = hz; }
    if (dc < best) { best = dc; hit = cyl; }
    if (cx == 1 && dx < best) { best = dx; hit = hx; }
    if (cy == 1 && dy < best) { best = dy; hit = hy; }
    return best;
}

// Straight-line path inside a second-level lattice (R37; see LAT_FAST2): per axis ONE candidate -- the second-level
// wall ahead, or at the lattice's rim what the first-level element's code names (first-level wall or an axis plane of
// the enclosing cell) -- plus the pin universe's z-cylinder.  Same formulas, coordinates (global -> first-level element
// -> second-level element, two subtractions) and candidate order as nearest2: the enclosing cell's planes, the
// cylinder, second-level walls, first-level walls.
__device__ __forceinline__ double nearest_fast2(const Geo &G, const int4 li, const int4 l2i, int cyl, double x, double y, double z,
                                                double ux, double uy, double uz, int elem, int last, int &hit)
{
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    const int outer = outer_of(G, elem), inner = inner_of(G, elem), k = li.w >> 16;
    int ix, iy;
    elem_xy(G, outer, ix, iy);
    const int nx2 = __ldg(G.l2_nx + k);
    const int jy = inner / nx2, jx = inner - jy * nx2;
    const double px2 = __ldg(G.l2_px + k), py2 = __ldg(G.l2_py + k);
    const double x02 = l2_x0(G, k), y02 = l2_y0(G, k);
    const double xo = x - (G.lat_x0 + (ix + 0.5) * G.lat_px), yo = y - (G.lat_y0 + (iy + 0.5) * G.lat_py);
    const double xl = xo - (x02 + (jx + 0.5) * px2), yl = yo - (y02 + (jy + 0.5) * py2);
    const double inv_ux = 1.0 / ux, inv_uy = 1.0 / uy;
    const bool xp = ux > 0.0, yp = uy > 0.0, zp = uz > 0.0;
    // kind per axis: 0 nothing, 1 axis plane of the enclosing cell, 2 second-level wall, 3 first-level wall
    int kx = 2, ky = 2, hx = G.n_surf + 4 + (xp ? 1 : 0), hy = G.n_surf + 6 + (yp ? 1 : 0);
    double dx = (x02 + (jx + (xp ? 1 : 0)) * px2 - xo) * inv_ux, dy = (y02 + (jy + (yp ? 1 : 0)) * py2 - yo) * inv_uy;
    if (((l2i.z >> (xp ? 8 : 0)) & 255) == 3) {
        const int co = (li.z >> (xp ? 8 : 0)) & 255;
        kx = co == 0 ? 0 : (co == 1 ? 3 : 1);
        double pw = G.lat_x0 + (ix + (xp ? 1 : 0)) * G.lat_px;
        hx = G.n_surf + (xp ? 1 : 0);
        if (co >= 2) { pw = __ldg(G.ap_pos + co - 2); hx = __ldg(G.ap_sid + co - 2); }
        dx = (pw - x) * inv_ux;
    }
    if (((l2i.z >> (yp ? 24 : 16)) & 255) == 3) {
        const int co = (li.z >> (yp ? 24 : 16)) & 255;
        ky = co == 0 ? 0 : (co == 1 ? 3 : 1);
        double pw = G.lat_y0 + (iy + (yp ? 1 : 0)) * G.lat_py;
        hy = G.n_surf + 2 + (yp ? 1 : 0);
        if (co >= 2) { pw = __ldg(G.ap_pos + co - 2); hy = __ldg(G.ap_sid + co - 2); }
        dy = (pw - y) * inv_uy;
    }
    if (kx == 0 || ux == 0.0 || hx == last || !(dx > 0.0)) dx = INF;
    if (ky == 0 || uy == 0.0 || hy == last || !(dy > 0.0)) dy = INF;
    const int cz = (li.w >> (zp ? 8 : 0)) & 255;
    double dz = INF;
    int hz = -1;
    if (cz >= 2) {
        hz = __ldg(G.ap_sid + cz - 2);
        if (uz != 0.0 && hz != last) { dz = (__ldg(G.ap_pos + cz - 2) - z) / uz; if (!(dz > 0.0)) dz = INF; }
    }
    double dc = INF;
    if (cyl >= 0) {
        const double *q = G.surf_param + 4 * cyl;
        const double da = xl - __ldg(q), db = yl - __ldg(q + 1), r = __ldg(q + 2);
        const double a = ux * ux + uy * uy, kk = da * ux + db * uy;
        double num = -1.0;
        if (cyl == last) { if (kk < 0.0) num = -2.0 * kk; }
        else {
            const double cc = da * da + db * db - r * r;
            const double disc = kk * kk - a * cc;
            if (disc >= 0.0) {
                const double sq = sqrt(disc);
                num = cc < 0.0 ? sq - kk : -kk - sq;
            }
        }
        if (a != 0.0 && num > 0.0) {
            dc = num / a;
            if (!(dc > 0.0)) dc = INF;
        }
    }
    double best = INF;
    hit = -1;
    if (kx == 1 && dx < best) { best = dx; hit = hx; }
    if (ky == 1 && dy < best) { best = dy; hit = hy; }
    if (dz < best) { best = dz; hit = hz; }
    if (dc < best) { best = dc; hit = cyl; }
    if (kx == 2 && dx < best) { best = dx; hit = hx; }
    if (ky == 2 && dy < best) { best = dy; hit = hy; }
    if (kx == 3 && dx < best) { best = dx; hit = hx; }
    if (ky == 3 && dy < best) { best = dy; hit = hy; }
    return best;
}

__device__ __forceinline__ bool surface_in_cell(const Geo &G, int c, int s)
{
    int k1 = __ldg(G.cso + c + 1);
    for (int k = __ldg(G.cso + c); k < k1; k++)
        if (__ldg(G.csi + k) == s) return true;
    return false;
}

// ------------------------------------------------------------------ particle in registers
struct Particle {
    double x, y, z, ux, uy, uz, E, t;
    double w;       // statistical weight (read and written only by the weighted kernels, R36)
    double v;       // continuous energy: speed, union-grid index and tally energy bin of E (they change only when E
    int gi, ebin;   // does: at birth and in a scatter), kept with the particle instead of recomputed every segment
    int cell, elem, g, last, tbin;
    unsigned int pend, nseg;
    unsigned long long id;
};

// Per-thread accumulator (k numerator) reduced once per kernel; event counts by code go to a block-shared
// counter array (integer shared-memory atomics) and leakage straight to the global scalar: both are kept out
// of the registers, which is what limits the occupancy of the latency-bound transport kernels.
struct Acc {
    double knum;
    double wabs;         // weight absorbed (weighted kernels only: capture share removed at collisions, fission, capture)
    unsigned int *s_ev;  // [16] in shared memory
    const double *mgs;   // multi-group table blob: the shared-memory copy, or the global blob when it does not fit
    const Geo *geo;      // the block's shared-memory copy of the Geo descriptor: what the out-of-line (generic-path)
                         // functions read, so that the kernel parameter block never has to be copied to a stack
    bool tracing;        // launch-uniform: a trace buffer is attached
    __device__ __forceinline__ void clear(unsigned int *ev) { knum = 0.0; wabs = 0.0; s_ev = ev; }
};

__device__ __forceinline__ void count_event(Acc &acc, int ev) { atomicAdd(acc.s_ev + ev, 1u); }

// the quantities of a continuous-energy particle that depend on E alone (R19, R23, R24); call whenever E is set
__device__ __forceinline__ void ce_energy_state(const CETab &ce, Particle &p)
{
    p.gi = grid_index(ce, p.E);
    p.ebin = energy_bin(ce, p.E);
    p.v = speed_of(p.E);
}

enum { ADV_DEAD = 0, ADV_SCATTER = 1, ADV_SURFACE = 2, ADV_FISSION = 3 };
// kernel variants beyond (CE, PRIVATE, W), template parameter X: the problem has second-level lattices (generic geometry
// through nearest2 / do_surface2); the problem is time-dependent multi-group (clock, time edges, delayed neutrons).
// One-level, time-independent problems compile exactly the code they had before these were added.
enum { X_L2 = 1, X_TD = 2 };

struct TraceRec {  // = mcdc_trace_rec
    unsigned long long id;
    unsigned int cycle, seq;
    int ev, c0, elem, c1, surf, gi;
    double x, y, z, d, E, t;
};

__device__ __noinline__ void trace_event(const Trace &tr, unsigned int cycle, int lat_cell, unsigned long long id, double x,
                                         double y, double z, double t, int ev, int cell0, int elem0, int surf, int gi, double d,
                                         double E)
{
    unsigned long long rel = id - tr.first;
    if (id < tr.first || rel >= tr.n_ids) return;
    unsigned long long slot = (unsigned long long)cycle * tr.n_ids + rel;
    if (slot >= tr.cap_slots) return;
    unsigned int seq = tr.count[slot]++;
    if (seq >= tr.max_events) return;
    TraceRec *r = (TraceRec *)tr.rec + slot * tr.max_events + seq;
    r->id = id; r->cycle = cycle; r->seq = seq; r->ev = ev;
    r->c0 = elem0 >= 0 ? lat_cell : cell0;
    r->elem = elem0;
    r->c1 = elem0 >= 0 ? cell0 : -1;
    r->surf = surf; r->gi = gi;
    r->x = x; r->y = y; r->z = z; r->d = d; r->E = E; r->t = t;
}

// tally flavours: FLUX_PRIVATE = one shared-memory column per thread (tiny tallies: no atomics at all until
// the per-block flush); FLUX_GLOBAL = float64 atomics straight to L2, warp-aggregated over equal bins.
template <bool PRIVATE>
__device__ __forceinline__ void flux_add(const Ctx &c, double *s_flux, long long tix, double v)
{
    if (PRIVATE) {
        s_flux[tix * blockDim.x + threadIdx.x] += v;
    } else {
        double *dst = c.flux + (size_t)(blockIdx.x & c.flux_copy_mask) * c.n_tally + tix;
        if (!c.flux_aggregate) { atomicAdd(dst, v); return; }
        // warp-aggregated: lanes that hit the same bin elect a leader which adds the group's sum
        unsigned int act = __activemask();
        unsigned int grp = __match_any_sync(act, tix);
        int leader = __ffs(grp) - 1;
        int lane = threadIdx.x & 31;
        if (grp == (1u << lane)) {
            atomicAdd(dst, v);
        } else {
            double sum = v;
            unsigned int rest = grp & ~(1u << leader);
            // the leader walks the other members (groups are small except in tiny-tally problems, which use
            // the PRIVATE flavour)
            while (rest) {
                int src = __ffs(rest) - 1;
                double o = __shfl_sync(grp, v, src);
                if (lane == leader) sum += o;
                rest &= rest - 1;
            }
            if (lane == leader) atomicAdd(dst, sum);
        }
    }
}

__device__ __forceinline__ double mgv(const Acc &acc, int off) { return acc.mgs[off]; }

// One segment up to and including the event decision (steps a2/a3, a5, a6, a7 of SURVEY.md 8a and the
// reaction choice of a8): cross sections, distance to collision, nearest boundary, time edge, move, tallies.
// Returns ADV_*; the event that still has to be finished is left in p.pend (scatter column, hit code, time edge);
// aux = number of children (fission).  Lanes in a LAT_FAST lattice element take the straight-line geometry path; a
// warp whose lanes all do (the normal case inside a pin lattice) never enters the generic loops.
// W: the weighted variant (implicit capture with roulette, R36): the particle carries its own weight p.w, every
// collision removes the capture share, the reaction is chosen among scatter / fission, and a scattered particle whose
// weight fell below w_roulette plays roulette (one draw).  W = false is the analog path (R2): weight = the launch
// constant w0, p.w is never read.
template <bool CE, bool PRIVATE, bool W, int X = 0>
__device__ __forceinline__ int advance(const Ctx &c, Particle &p, Rng &rng, int &aux, Acc &acc, double *s_flux)
{
    constexpr bool L2 = (X & X_L2) != 0, TD = (X & X_TD) != 0, TIMED = CE || TD;
    // implicit capture: what the weighted kernels are for -- except the time-dependent multi-group kernel, which is
    // always weighted (census survivors and combed copies carry their own weights, R40) and asks the option
    const bool IMPL = W && (TD ? c.implicit != 0 : true);
    const Geo &G = c.geo;
    const int cell0 = p.cell, elem0 = p.elem;
    const int mat = __ldg(G.cfill + p.cell);
    int bin = __ldg(G.cbin + p.cell);
    int4 li;  // boundary codes of the location (z, w), fast-path flag, cylinder
    int cyl;
    if (p.elem >= 0) {
        li = __ldg(G.lat_info + (L2 ? outer_of(G, p.elem) : p.elem));
        bin += li.y;
        cyl = (li.w >> 16) - 1;  // the pin universe's z-cylinder rides in the element's table entry (LAT_FAST elements)
    } else {
        li = __ldg(G.cell_info + p.cell);
        cyl = li.y;
    }

    double sig_t, nusf, cum[MAX_CE_COL];
    int gi, ncol = 0;
    if (!CE) {
        gi = p.g;
        sig_t = mgv(acc, c.mg.o_sig_t + mat * c.mg.G + p.g);
        nusf = mgv(acc, c.mg.o_nusf + mat * c.mg.G + p.g);
    } else {
        gi = p.gi;  // union-grid index of E, found when E last changed (ce_energy_state)
        const double2 *r0 = (const double2 *)(c.ce.tab + ((size_t)mat * c.ce.n_grid + gi) * CE_ROW);
        double2 a0 = __ldg(r0), a1 = __ldg(r0 + 1), a2 = __ldg(r0 + 2), a3 = __ldg(r0 + 3);
        double2 b0 = __ldg(r0 + 4), b1 = __ldg(r0 + 5), b2 = __ldg(r0 + 6), b3 = __ldg(r0 + 7);
        const double g0 = a3.x, g1 = b3.x;  // the rows carry their grid energies (slot 6)
        double f = (p.E - g0) / (g1 - g0);
        cum[0] = a0.x + f * (b0.x - a0.x); cum[1] = a0.y + f * (b0.y - a0.y);
        cum[2] = a1.x + f * (b1.x - a1.x); cum[3] = a1.y + f * (b1.y - a1.y);
        cum[4] = a2.x + f * (b2.x - a2.x); cum[5] = a2.y + f * (b2.y - a2.y);
        double sig_f = a3.y + f * (b3.y - a3.y);
        ncol = __ldg(c.ce.ncol + mat);
        sig_t = cum[0];
#pragma unroll
        for (int j = 1; j < MAX_CE_COL; j++)
            if (j == ncol - 1) sig_t = cum[j];
        nusf = (c.ce.nu0 + c.ce.nu1 * (p.E * 1e-6)) * sig_f;
    }

    // candidate distances: collision (one draw every segment), boundary, time edge (R12)
#if MCDC_NEXT_PRE && MCDC_INV_SIGT
    double d_coll = CE ? -log(rng.next_pre(c)) / sig_t : -log(rng.next_pre(c)) * mgv(acc, c.mg.o_inv_t + mat * c.mg.G + p.g);
#elif MCDC_NEXT_PRE
    double d_coll = -log(rng.next_pre(c)) / sig_t;
#else
    double d_coll = -log(rng.next(c)) / sig_t;
#endif
    int hit;
    double d_surf;
    int4 l2i = make_int4(0, 0, 0, 0);
    if (L2 && p.elem >= (1 << INNER_SHIFT) && (li.x & LAT_FAST2))  // second-level element of a simple assembly (R37)
        l2i = __ldg(G.l2_info + __ldg(G.l2_off + (li.w >> 16)) + inner_of(G, p.elem));
    if (L2 && (l2i.x & LAT_FAST)) {
        bin += l2i.y;
        d_surf = nearest_fast2(G, li, l2i, __ldg(&G.ufast[l2i.x & UNIV_MASK].y), p.x, p.y, p.z, p.ux, p.uy, p.uz, p.elem, p.last, hit);
    } else if (li.x & LAT_FAST) d_surf = nearest_fast(G, li.z, li.w, cyl, p.x, p.y, p.z, p.ux, p.uy, p.uz, p.elem, p.last, hit);
    else {
        unsigned int root_mask = p.elem >= 0 ? __ldg(G.lat_rmask + (L2 ? outer_of(G, p.elem) : p.elem)) : 0xffffffffu;
        if (L2) {
            d_surf = nearest2(*acc.geo, p.x, p.y, p.z, p.ux, p.uy, p.uz, p.cell, p.elem, p.last, hit, root_mask);
            if (hit >= (1 << HIT_BITS)) {  // inside a second-level lattice: its element's tally-bin offset rides on the hit code (R37)
                bin += hit >> HIT_BITS;
                hit &= (1 << HIT_BITS) - 1;
                if (hit == (1 << HIT_BITS) - 1) hit = -1;
            }
        } else d_surf = nearest(*acc.geo, p.x, p.y, p.z, p.ux, p.uy, p.uz, p.cell, p.elem, p.last, hit, root_mask);
    }
    double v = 0.0, d_time = __longlong_as_double(0x7ff0000000000000LL);
    if (TIMED) {
        v = CE ? p.v : __ldg(c.td.speed + p.g);  // R23 / the group's speed (R38)
        d_time = v * (__ldg(c.ce.t_edges + p.tbin + 1) - p.t);
    }
    int kind;
    double d;
    if (d_coll < d_surf && d_coll < d_time) { kind = 0; d = d_coll; }
    else if (d_surf <= d_time) { kind = 1; d = d_surf; }
    else { kind = 2; d = d_time; }

    // move + track-length tallies
    p.x += d * p.ux; p.y += d * p.uy; p.z += d * p.uz;
    const double E_flight = CE ? p.E : 0.0;
    long long tix;
    if (!CE) tix = TD ? ((long long)bin * c.ce.n_t + p.tbin) * c.mg.G + p.g : (long long)bin * c.mg.G + p.g;
    else tix = ((long long)bin * c.ce.n_t + p.tbin) * c.ce.n_e + p.ebin;
    if (TIMED) { if (kind == 2) p.t = __ldg(c.ce.t_edges + p.tbin + 1); else p.t += d / v; }
    const double w = W ? p.w : c.w0;
    flux_add<PRIVATE>(c, s_flux, tix, w * d);
    acc.knum += w * d * nusf;

    int ev, code, surf = -1;
    p.pend = PEND_NONE;
    if (kind == 0) {
        p.last = -1;
        if (!CE) {
            double sig_s = mgv(acc, c.mg.o_sig_s + mat * c.mg.G + p.g), sig_f = mgv(acc, c.mg.o_sig_f + mat * c.mg.G + p.g);
            double total = sig_t;
            if (IMPL) {  // the weight loses its capture share; the reaction is chosen among scatter / fission
                total = sig_s + sig_f;
                const double wn = p.w * (total / sig_t);
                acc.wabs += p.w - wn;
                p.w = wn;
            }
            double uu = rng.next(c) * total;
            if (uu < sig_s) { ev = 1; code = ADV_SCATTER; p.pend = PEND_SCATTER; }
            else if (uu < sig_s + sig_f) {
                ev = 2; code = ADV_FISSION;
                if (TD)  // time-dependent fixed source (R39): floor(prompt + delayed yields + xi) children of the parent's weight
                    aux = (int)floor(__ldg(c.td.cum_nu + ((size_t)mat * c.mg.G + p.g) * (c.td.J + 1) + c.td.J) + rng.next(c));
                else
                    aux = (int)floor((W ? p.w : c.w0) * mgv(acc, c.mg.o_nu + mat * c.mg.G + p.g) / c.k_prev + rng.next(c));
            } else { ev = 3; code = ADV_DEAD; }
        } else {
            const int nsel = IMPL ? ncol - 1 : ncol;  // columns the reaction is chosen from (implicit capture: all but capture)
            double total = sig_t;
            if (IMPL) {
                total = cum[0];
#pragma unroll
                for (int j = 1; j < MAX_CE_COL; j++)
                    if (j == nsel - 1) total = cum[j];
                const double wn = p.w * (total / sig_t);
                acc.wabs += p.w - wn;
                p.w = wn;
            }
            double uu = rng.next(c) * total;
            int r = nsel - 1;  // first column whose cumulative value exceeds uu (static indices: cum stays in registers)
#pragma unroll
            for (int j = MAX_CE_COL - 2; j >= 0; j--)
                if (j < nsel - 1 && cum[j] > uu) r = j;
            if (r < ncol - 2) { ev = 1; code = ADV_SCATTER; p.pend = PEND_SCATTER | (unsigned int)r; }
            else if (r == ncol - 2) {
                ev = 2; code = ADV_FISSION;
                double nu = c.ce.nu0 + c.ce.nu1 * (p.E * 1e-6);
                aux = (int)floor((W ? p.w : c.w0) * nu + rng.next(c));
            } else { ev = 3; code = ADV_DEAD; }
        }
        if (W) {
            if (code == ADV_SCATTER) {
                if (IMPL && p.w < c.w_roulette) {  // roulette (one draw): survive at w_survive with probability w / w_survive
                    if (rng.next(c) * c.w_survive < p.w) { atomicAdd(c.scal + 5, c.w_survive - p.w); p.w = c.w_survive; }
                    else { atomicAdd(c.scal + 4, p.w); ev = 3; code = ADV_DEAD; p.pend = PEND_NONE; }
                }
            } else acc.wabs += p.w;  // fission / capture end the history with its whole weight
        }
    } else if (kind == 1) {
        surf = hit;
        if (hit >= G.n_surf) { ev = 7; code = ADV_SURFACE; p.pend = (unsigned int)hit; }
        else {
            int bc = __ldg(G.surf_bc + hit);
            if (bc == 2) { ev = 6; code = ADV_DEAD; atomicAdd(c.scal + 1, w); }
            else { ev = bc == 1 ? 5 : 4; code = ADV_SURFACE; p.pend = (unsigned int)hit; }
        }
    } else {
        // time edge: the particle has moved off whatever surface it sat on (R11)
        p.tbin++;
        p.last = -1;
        if (p.tbin == c.ce.n_t) { ev = 9; code = ADV_DEAD; if (W) atomicAdd(c.scal + 3, w); }
        else { ev = 8; code = ADV_SURFACE; p.pend = PEND_TIME; }
    }
    if (acc.tracing)
        trace_event(*c.tr_g, c.cycle, G.lat_cell, p.id, p.x, p.y, p.z, TIMED ? p.t : 0.0, ev, cell0, elem0, surf, gi, d, E_flight);
    count_event(acc, ev);
    p.nseg++;
    if (code != ADV_DEAD && code != ADV_FISSION && p.nseg >= MAX_SEGMENTS) {  // lost-particle guard (R11)
        code = ADV_DEAD;
        count_event(acc, 10);
        atomicExch(c.err, -4);
    }
    return code;
}

// rotate the unit vector (ux, uy, uz) by polar cosine mu and azimuth (sp, cp = sin, cos), then renormalise (R21)
__device__ __forceinline__ void rotate_dir(double ux, double uy, double uz, double mu, double sp, double cp, double &ox,
                                           double &oy, double &oz)
{
    double s2 = 1.0 - mu * mu;
    double s = s2 > 0.0 ? sqrt(s2) : 0.0;
    double a2 = 1.0 - uz * uz;
    if (a2 < 1e-10) {
        ox = s * cp; oy = s * sp; oz = uz > 0.0 ? mu : -mu;
    } else {
        double r = sqrt(a2);
        ox = mu * ux + s * (ux * uz * cp - uy * sp) / r;
        oy = mu * uy + s * (uy * uz * cp + ux * sp) / r;
        oz = mu * uz - s * r * cp;
    }
    double nrm = sqrt(ox * ox + oy * oy + oz * oz);
    ox /= nrm; oy /= nrm; oz /= nrm;
}

// Free-gas elastic scattering with a constant cross section (R35), speeds in units of sqrt(eV).
// Target speed x (units of sqrt(kT/A)) and cosine mu between target and neutron from |v_n - v_T| x^2 exp(-x^2):
// with probability 1 / (1 + sqrt(pi) y / 2), y = sqrt(A E / kT): x^2 = -ln(xi1 xi2), else x^2 = -ln xi1 - ln xi2
// cos^2(pi xi4 / 2); mu = 2 xi - 1; accepted with probability sqrt(y^2 + x^2 - 2 x y mu) / (x + y).  Draws per trial,
// in order: xi1, xi2, branch, [xi4], mu, accept.  Then the target's azimuth around the neutron's direction (1 draw)
// and an isotropic direction of the relative velocity in the centre-of-mass frame (2 draws).
// Out of line (thermal collisions only): takes the stream by value, returns the new draw counter; out = E', u'.
__device__ __noinline__ uint32_t free_gas(unsigned long long seed, uint32_t cycle, unsigned long long id, uint32_t ctr, double A,
                                          double kT, double E, double ux, double uy, double uz, double *out)
{
    const double y = sqrt(A * E / kT);
    const double alpha = 1.0 / (1.0 + 1.7724538509055159 * y / 2.0);
    double x2, x, mu;
    for (;;) {
        const double r1 = draw_at(seed, id, 0u, cycle, ctr), r2 = draw_at(seed, id, 0u, cycle, ctr + 1u);
        ctr += 3u;
        if (draw_at(seed, id, 0u, cycle, ctr - 1u) < alpha) x2 = -log(r1 * r2);
        else {
            const double cs = cospi(0.5 * draw_at(seed, id, 0u, cycle, ctr++));
            x2 = -log(r1) - log(r2) * cs * cs;
        }
        x = sqrt(x2);
        mu = 2.0 * draw_at(seed, id, 0u, cycle, ctr++) - 1.0;
        const double accept = sqrt(y * y + x2 - 2.0 * x * y * mu) / (x + y);
        if (draw_at(seed, id, 0u, cycle, ctr++) < accept) break;
    }
    double sp, cp, tx, ty, tz;
    sincospi(2.0 * draw_at(seed, id, 0u, cycle, ctr++), &sp, &cp);
    rotate_dir(ux, uy, uz, mu, sp, cp, tx, ty, tz);
    const double sn = sqrt(E), st = x * sqrt(kT / A);
    const double vnx = sn * ux, vny = sn * uy, vnz = sn * uz;
    const double vcx = (vnx + A * st * tx) / (A + 1.0), vcy = (vny + A * st * ty) / (A + 1.0), vcz = (vnz + A * st * tz) / (A + 1.0);
    const double rx = vnx - vcx, ry = vny - vcy, rz = vnz - vcz;
    const double sr = sqrt(rx * rx + ry * ry + rz * rz);
    double ox, oy, oz;
    const double a = draw_at(seed, id, 0u, cycle, ctr), b = draw_at(seed, id, 0u, cycle, ctr + 1u);
    ctr += 2u;
    iso_dir(a, b, ox, oy, oz);
    const double vx = vcx + sr * ox, vy = vcy + sr * oy, vz = vcz + sr * oz;
    const double e = vx * vx + vy * vy + vz * vz;
    const double nv = sqrt(e);
    out[0] = e; out[1] = vx / nv; out[2] = vy / nv; out[3] = vz / nv;
    return ctr;
}

// Scatter event (a8).  MG: new group from the cumulative scatter row, isotropic direction (1 + 2 draws).
// CE: elastic off a target at rest with mass ratio A: mu_cm, azimuth (2 draws), rotation, energy clamp (R19, R21).
template <bool CE>
__device__ __forceinline__ void do_scatter(const Ctx &c, const Acc &acc, Particle &p, Rng &rng, int col)
{
    const int mat = __ldg(c.geo.cfill + p.cell);
    if (!CE) {
        const int G = c.mg.G;
        double sig_s = mgv(acc, c.mg.o_sig_s + mat * G + p.g);
#if MCDC_NEXT3
        double xg, a, b;
        rng.next3(c, xg, a, b);
        double vv = xg * sig_s;
#else
        double vv = rng.next(c) * sig_s;
#endif
        const int row = c.mg.o_cumS + (mat * G + p.g) * G;
#if MCDC_GROUP_COUNT == 2
        // first i with cumS[i] > vv (else G - 1) = how many of the first G - 1 running sums are <= vv (they never
        // decrease: S >= 0 is validated), found by bisection with a fixed trip count, the same for every lane
        int i = 0;
        for (int h = c.mg.half; h > 0; h >>= 1) {
            const int j = i + h;
            if (j <= G - 1 && !(mgv(acc, row + j - 1) > vv)) i = j;
        }
        p.g = i;
#elif MCDC_GROUP_COUNT
        int i = 0;
        for (int j = 0; j < G - 1; j++) i += !(mgv(acc, row + j) > vv) ? 1 : 0;
        p.g = i;
#else
        int i = 0;
        while (i < G - 1 && !(mgv(acc, row + i) > vv)) i++;
        p.g = i;
#endif
#if !MCDC_NEXT3
        double a = rng.next(c), b = rng.next(c);
#endif
        iso_dir(a, b, p.ux, p.uy, p.uz);
    } else {
        double A = __ldg(c.ce.colA + mat * CE_ROW + col);
        double En;
        if (c.kT > 0.0 && p.E < 400.0 * c.kT) {  // free gas below 400 kT, target at rest above (R35)
            double o[4];
            const uint32_t ctr = free_gas(c.seed, c.cycle, rng.id, rng.ctr, A, c.kT, p.E, p.ux, p.uy, p.uz, o);
            rng.init(rng.id, ctr);
            En = o[0]; p.ux = o[1]; p.uy = o[2]; p.uz = o[3];
        } else {
            double xi_mu, xi_phi;
            rng.next2(c, xi_mu, xi_phi);
            double mu_cm = 2.0 * xi_mu - 1.0;
            double den = A * A + 2.0 * A * mu_cm + 1.0;
            double mu = 0.0;
            if (den > 0.0) mu = (1.0 + A * mu_cm) / sqrt(den);
            En = p.E * den / ((A + 1.0) * (A + 1.0));
            double sp, cp;
            sincospi(2.0 * xi_phi, &sp, &cp);
            double ox, oy, oz;
            rotate_dir(p.ux, p.uy, p.uz, mu, sp, cp, ox, oy, oz);
            p.ux = ox; p.uy = oy; p.uz = oz;
        }
        if (En < c.ce.E_min) En = c.ce.E_min;
        if (En > c.ce.E_max) En = c.ce.E_max;
        p.E = En;
        ce_energy_state(c.ce, p);
    }
    p.last = -1;
}

// Surface event of a problem with second-level lattices (R37): the same as do_surface below, with the second-level
// walls, the surfaces of the cell a second-level lattice fills, and the descent into a second-level lattice wherever
// the cell found is filled by one.  Returns false if the particle got lost.
__device__ __noinline__ bool do_surface2(const Geo &G, Particle &p, int hit)
{
    if (hit >= G.n_surf + 4) {  // second-level wall: neighbour element of the same second-level lattice (R37)
        const int w = hit - G.n_surf - 4;
        const int outer = outer_of(G, p.elem);
        const int k2 = __ldg(G.cfill + __ldg(G.umid + elem_universe(G, outer)));
        const int nx2 = __ldg(G.l2_nx + k2);
        int jy = inner_of(G, p.elem) / nx2, jx = inner_of(G, p.elem) - jy * nx2;
        if (w == 0) jx--; else if (w == 1) jx++; else if (w == 2) jy--; else jy++;
        const int inner = jy * nx2 + jx;
        p.elem = outer | ((inner + 1) << INNER_SHIFT);
        p.last = -1;
        double xl, yl;
        innermost_xy(G, p.elem, p.x, p.y, xl, yl);
        p.cell = find_cell(G, __ldg(G.l2_univ + __ldg(G.l2_off + k2) + inner), xl, yl, p.z, p.ux, p.uy, p.uz, -1);
        return p.cell >= 0;
    }
    if (hit >= G.n_surf) {
        int w = hit - G.n_surf;
        int ix, iy;
        elem_xy(G, outer_of(G, p.elem), ix, iy);
        if (w == 0) ix--; else if (w == 1) ix++; else if (w == 2) iy--; else iy++;
        p.last = -1;
        double xl, yl;
        local_xy(G, iy * G.lat_nx + ix, p.x, p.y, xl, yl);
        p.cell = descend(G, iy * G.lat_nx + ix, xl, yl, p.z, p.ux, p.uy, p.uz, -1, p.elem);
        return p.cell >= 0;
    }
    int bc = __ldg(G.surf_bc + hit);
    // whose surface: the enclosing (root) cell's, the cell's that a second-level lattice fills (first-level-element
    // coordinates), or the local cell's (innermost coordinates)
    const bool local = p.elem >= 0 && !surface_in_cell(G, G.lat_cell, hit);
    const bool inner_loc = local && inner_of(G, p.elem) >= 0;
    const bool midlevel = inner_loc && surface_in_cell(G, __ldg(G.umid + elem_universe(G, outer_of(G, p.elem))), hit);
    double xl = p.x, yl = p.y;
    if (midlevel) local_xy(G, outer_of(G, p.elem), p.x, p.y, xl, yl);
    else if (local) innermost_xy(G, p.elem, p.x, p.y, xl, yl);
    p.last = hit;
    if (bc == 1) {
        int t = __ldg(G.surf_type + hit);
        if (t == 0) p.ux = -p.ux;
        else if (t == 1) p.uy = -p.uy;
        else if (t == 2) p.uz = -p.uz;
        else {
            double nx, ny, nz;
            surf_normal(G, hit, xl, yl, p.z, nx, ny, nz);
            double nn = sqrt(nx * nx + ny * ny + nz * nz);
            nx /= nn; ny /= nn; nz /= nn;
            double dot = p.ux * nx + p.uy * ny + p.uz * nz;
            p.ux -= 2.0 * dot * nx; p.uy -= 2.0 * dot * ny; p.uz -= 2.0 * dot * nz;
        }
        return true;
    }
    if (local) {
        if (inner_loc && !midlevel) {  // inside the same second-level element
            const int outer = outer_of(G, p.elem);
            const int k2 = __ldg(G.cfill + __ldg(G.umid + elem_universe(G, outer)));
            p.cell = find_cell(G, __ldg(G.l2_univ + __ldg(G.l2_off + k2) + inner_of(G, p.elem)), xl, yl, p.z, p.ux, p.uy, p.uz, hit);
        } else {  // inside the same first-level element: its universe, descending where a lattice fills the cell
            const int outer = outer_of(G, p.elem);
            double xo, yo;
            local_xy(G, outer, p.x, p.y, xo, yo);
            p.cell = descend(G, outer, xo, yo, p.z, p.ux, p.uy, p.uz, hit, p.elem);
        }
        return p.cell >= 0;
    }
    return locate(G, p.x, p.y, p.z, p.ux, p.uy, p.uz, hit, p.cell, p.elem);
}

// Surface event (a9), generic path: lattice wall -> neighbour element; reflect; transmit -> neighbour cell by the
// side being entered (R11, R14).  Returns false if the particle got lost.
__device__ __noinline__ bool do_surface(const Geo &G, Particle &p, int hit)
{
    if (hit >= G.n_surf) {
        int w = hit - G.n_surf;
        int ix, iy;
        elem_xy(G, p.elem, ix, iy);
        if (w == 0) ix--; else if (w == 1) ix++; else if (w == 2) iy--; else iy++;
        p.elem = iy * G.lat_nx + ix;
        p.last = -1;
        double xl, yl;
        local_xy(G, p.elem, p.x, p.y, xl, yl);
        p.cell = find_cell(G, elem_universe(G, p.elem), xl, yl, p.z, p.ux, p.uy, p.uz, -1);
        return p.cell >= 0;
    }
    int bc = __ldg(G.surf_bc + hit);
    bool local = p.elem >= 0 && !surface_in_cell(G, G.lat_cell, hit);
    double xl = p.x, yl = p.y;
    if (local) local_xy(G, p.elem, p.x, p.y, xl, yl);
    p.last = hit;
    if (bc == 1) {
        int t = __ldg(G.surf_type + hit);
        if (t == 0) p.ux = -p.ux;
        else if (t == 1) p.uy = -p.uy;
        else if (t == 2) p.uz = -p.uz;
        else {
            double nx, ny, nz;
            surf_normal(G, hit, xl, yl, p.z, nx, ny, nz);
            double nn = sqrt(nx * nx + ny * ny + nz * nz);
            nx /= nn; ny /= nn; nz /= nn;
            double dot = p.ux * nx + p.uy * ny + p.uz * nz;
            p.ux -= 2.0 * dot * nx; p.uy -= 2.0 * dot * ny; p.uz -= 2.0 * dot * nz;
        }
        return true;
    }
    if (local) {
        p.cell = find_cell(G, elem_universe(G, p.elem), xl, yl, p.z, p.ux, p.uy, p.uz, hit);
        return p.cell >= 0;
    }
    return locate(G, p.x, p.y, p.z, p.ux, p.uy, p.uz, hit, p.cell, p.elem);
}

// Surface event from inside a LAT_FAST element whose event is one of: lattice wall into another LAT_FAST element,
// the universe's own z-cylinder (transmit), a reflecting axis plane of the enclosing cell.  Returns 0 if the event
// is none of these (the caller then takes the generic path), 1 done, -1 lost.
__device__ __forceinline__ int do_surface_fast(const Geo &G, Particle &p, int hit)
{
    if (p.elem < 0) {  // a CELL_FAST cell outside a lattice: its cylinder (transmit) or a reflecting axis plane
        const int4 ci = __ldg(G.cell_info + p.cell);
        if (hit == ci.y) {
            const int nb = ci.x & CELL_NO_NEIGHBOUR;
            if (__ldg(G.surf_bc + hit) != 0 || nb == CELL_NO_NEIGHBOUR) return 0;
            p.cell = nb;
            p.last = hit;
            return 1;
        }
        if (__ldg(G.surf_bc + hit) == 1) {
            int t = __ldg(G.surf_type + hit);
            if (t > 2) return 0;
            if (t == 0) p.ux = -p.ux; else if (t == 1) p.uy = -p.uy; else p.uz = -p.uz;
            p.last = hit;
            return 1;
        }
        return 0;
    }
    if (hit >= G.n_surf) {
        int w = hit - G.n_surf;
        int e2 = p.elem + (w == 0 ? -1 : w == 1 ? 1 : w == 2 ? -G.lat_nx : G.lat_nx);
        const int4 l2 = __ldg(G.lat_info + e2);
        if (!(l2.x & LAT_FAST)) return 0;
        const int4 uf = __ldg(G.ufast + (l2.x & UNIV_MASK));
        p.elem = e2;
        p.last = -1;
        int cell = uf.z;
        if (uf.x & 2) cell = uf.w;  // the cylinder lies strictly inside the element: a particle on a wall is outside it
        else if (uf.y >= 0) {
            double xl, yl;
            local_xy(G, e2, p.x, p.y, xl, yl);
            const double *q = G.surf_param + 4 * uf.y;
            double da = xl - __ldg(q), db = yl - __ldg(q + 1), r = __ldg(q + 2);
            cell = (da * da + db * db - r * r > 0.0) ? uf.w : uf.z;
        }
        p.cell = cell;
        return 1;
    }
    const int4 uf = __ldg(G.ufast + elem_universe(G, p.elem));
    if (hit == uf.y) {
        if (__ldg(G.surf_bc + hit) != 0) return 0;
        double xl, yl;
        local_xy(G, p.elem, p.x, p.y, xl, yl);
        const double *q = G.surf_param + 4 * hit;
        double nx = xl - __ldg(q), ny = yl - __ldg(q + 1);
        p.last = hit;
        p.cell = (p.ux * nx + p.uy * ny > 0.0) ? uf.w : uf.z;  // the side being entered (R11)
        return 1;
    }
    if (__ldg(G.surf_bc + hit) == 1) {
        int t = __ldg(G.surf_type + hit);
        if (t > 2) return 0;
        if (t == 0) p.ux = -p.ux; else if (t == 1) p.uy = -p.uy; else p.uz = -p.uz;
        p.last = hit;
        return 1;
    }
    return 0;
}

// Surface event from a second-level element on the two-level straight-line path (see nearest_fast2): second-level wall
// into a simple element of the same lattice, first-level wall into a LAT_FAST2 element (the second-level index by floor,
// clamped, as in descend), the pin's z-cylinder, a reflecting axis plane.  0: none of these (generic path), 1 done.
__device__ __forceinline__ int do_surface_fast2(const Geo &G, Particle &p, int hit, const int4 li, const int4 l2i)
{
    const int outer = outer_of(G, p.elem), inner = inner_of(G, p.elem);
    if (hit >= G.n_surf) {
        int e2 = outer, k = li.w >> 16, inner2;
        double xo, yo;
        if (hit >= G.n_surf + 4) {
            const int w = hit - G.n_surf - 4, nx2 = __ldg(G.l2_nx + k);
            inner2 = inner + (w == 0 ? -1 : w == 1 ? 1 : w == 2 ? -nx2 : nx2);
            local_xy(G, outer, p.x, p.y, xo, yo);
        } else {
            const int w = hit - G.n_surf;
            e2 = outer + (w == 0 ? -1 : w == 1 ? 1 : w == 2 ? -G.lat_nx : G.lat_nx);
            const int4 li2 = __ldg(G.lat_info + e2);
            if (!(li2.x & LAT_FAST2)) return 0;
            k = li2.w >> 16;
            local_xy(G, e2, p.x, p.y, xo, yo);
            const int nx2 = __ldg(G.l2_nx + k), ny2 = __ldg(G.l2_ny + k);
            int jx = (int)floor((xo - l2_x0(G, k)) / __ldg(G.l2_px + k));
            int jy = (int)floor((yo - l2_y0(G, k)) / __ldg(G.l2_py + k));
            jx = jx < 0 ? 0 : (jx > nx2 - 1 ? nx2 - 1 : jx);
            jy = jy < 0 ? 0 : (jy > ny2 - 1 ? ny2 - 1 : jy);
            inner2 = jy * nx2 + jx;
        }
        const int4 l2n = __ldg(G.l2_info + __ldg(G.l2_off + k) + inner2);
        if (!(l2n.x & LAT_FAST)) return 0;
        const int4 uf = __ldg(G.ufast + (l2n.x & UNIV_MASK));
        int cell = uf.z;
        if (uf.x & 2) cell = uf.w;  // the cylinder lies strictly inside the element: a particle on a wall is outside it
        else if (uf.y >= 0) {
            double xl, yl;
            inner_xy(G, k, inner2, xo, yo, xl, yl);
            const double *q = G.surf_param + 4 * uf.y;
            const double da = xl - __ldg(q), db = yl - __ldg(q + 1), r = __ldg(q + 2);
            cell = (da * da + db * db - r * r > 0.0) ? uf.w : uf.z;
        }
        p.elem = e2 | ((inner2 + 1) << INNER_SHIFT);
        p.cell = cell;
        p.last = -1;
        return 1;
    }
    const int4 uf = __ldg(G.ufast + (l2i.x & UNIV_MASK));
    if (hit == uf.y) {
        if (__ldg(G.surf_bc + hit) != 0) return 0;
        double xl, yl;
        innermost_xy(G, p.elem, p.x, p.y, xl, yl);
        const double *q = G.surf_param + 4 * hit;
        const double nx = xl - __ldg(q), ny = yl - __ldg(q + 1);
        p.last = hit;
        p.cell = (p.ux * nx + p.uy * ny > 0.0) ? uf.w : uf.z;  // the side being entered (R11)
        return 1;
    }
    if (__ldg(G.surf_bc + hit) == 1) {
        const int t = __ldg(G.surf_type + hit);
        if (t > 2) return 0;
        if (t == 0) p.ux = -p.ux; else if (t == 1) p.uy = -p.uy; else p.uz = -p.uz;
        p.last = hit;
        return 1;
    }
    return 0;
}

template <bool L2 = true>
__device__ __forceinline__ bool location_is_fast(const Geo &G, int cell, int elem)
{
    return ((elem >= 0 ? __ldg(&G.lat_info[L2 ? outer_of(G, elem) : elem].x) : __ldg(&G.cell_info[cell].x)) & LAT_FAST) != 0;
}

// Watt spectrum, rejection-free (R22); MeV
__device__ __forceinline__ double watt(double a, double b, double x1, double x2, double x3, double x4)
{
    double cs = cospi(0.5 * x3);
    double W = -a * (log(x1) + log(x2) * cs * cs);
    return W + 0.25 * a * a * b + (2.0 * x4 - 1.0) * sqrt(a * a * b * W);
}

// Finish the event a banked particle is waiting on (scatter: a8; surface / lattice wall: a9; time edge: nothing).
// Returns false if the particle got lost.
template <bool CE, int X = 0>
__device__ __forceinline__ bool finish_pending(const Ctx &c, const Acc &acc, Particle &p, Rng &rng)
{
    constexpr bool L2 = (X & X_L2) != 0;
    const unsigned int pend = p.pend;
    p.pend = PEND_NONE;
    if (pend >= PEND_TIME) return true;
    if (pend >= PEND_SCATTER) { do_scatter<CE>(c, acc, p, rng, (int)(pend & 7u)); return true; }
    int r = 0;
    if (L2 && p.elem >= (1 << INNER_SHIFT)) {
        const int4 li = __ldg(c.geo.lat_info + outer_of(c.geo, p.elem));
        if (li.x & LAT_FAST2) {
            const int4 l2i = __ldg(c.geo.l2_info + __ldg(c.geo.l2_off + (li.w >> 16)) + inner_of(c.geo, p.elem));
            if (l2i.x & LAT_FAST) r = do_surface_fast2(c.geo, p, (int)pend, li, l2i);
        }
    } else if (location_is_fast<L2>(c.geo, p.cell, p.elem)) r = do_surface_fast(c.geo, p, (int)pend);
    if (r == 0) r = (L2 ? do_surface2(*acc.geo, p, (int)pend) : do_surface(*acc.geo, p, (int)pend)) ? 1 : -1;
    return r > 0;
}

}  // namespace mcdc
