// mcdc_device.cuh -- device-side data layout and per-particle device functions of the B200 transport
// library (include/mcdc.h).  Written from the readings R1..R31 of DESIGN.md section 3 (= SURVEY.md 8c);
// shares no code with oracle/.  float64 everywhere.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mcdc {

constexpr int CE_ROW = 8;          // doubles per (material, grid point) row of the macroscopic CE table
constexpr int MAX_CE_COL = 6;      // cumulative columns kept per row: [el_1..el_n, fission, capture], n <= 4
constexpr int EV_DEAD = -0x40000000;  // status value of a finished history (monolithic schedule)
constexpr int RING = 8;            // per-sweep queue-counter sets kept alive for the lagging host read-back

// ------------------------------------------------------------------ layout in HBM
// Geometry and small tables: plain arrays in the workspace (read-only, L1/L2 resident).
struct Geo {
    int n_surf, n_cell, n_univ, has_lat, lat_nx, lat_ny, lat_cell;
    unsigned int lat_magic;  // floor(2^32 / lat_nx) + 1: elem / lat_nx == umulhi(elem, lat_magic) (elem * lat_nx < 2^32)
    double lat_x0, lat_y0, lat_px, lat_py;
    const int *surf_type, *surf_bc;
    const double *surf_param;  // [n_surf][4]
    const int *cso, *csi, *css, *cft, *cfill, *cbin, *uco;
    const char *blob;  // surfaces, cells and universes are one contiguous blob (staged in shared memory)
    int blob_words;    // its size in 4-byte words
    const unsigned int *lat_rmask;  // per element: bit j set = surface j of the enclosing cell's list can be the
                                    // nearest boundary from inside the element (built exactly at create)
    const int *lat_univ, *lat_bin;  // lat_bin bit 30: the enclosing cell's surfaces can be the nearest boundary
};                                  // from inside this element (create() proves when they cannot)
constexpr int LAT_ROOT_FLAG = 1 << 30;

// All multi-group tables are one contiguous blob (blob, blob_doubles); the transport kernels copy it to shared
// memory at start-up and run on rebased pointers (stage_mg) when it fits.
struct MGTab {  // [n_mat][G] each; cumS [n_mat][G][G] running row sums; cumchi running chi sums
    int G, n_mat, blob_doubles;
    const double *blob;
    const double *sig_t, *sig_s, *sig_f, *nu, *nusf, *cumS, *cumchi, *src_cum;
};

struct CETab {
    int n_grid, n_mat, n_t, n_e, search;
    const double *grid;
    const double *tab;    // [n_mat][n_grid][CE_ROW]: cumulative macroscopic columns, then Sigma_f in slot 7
    const int *ncol;      // [n_mat] number of cumulative columns (= n_nuclides + 2)
    const double *colA;   // [n_mat][CE_ROW] mass ratio A of the nuclide behind elastic column j
    const double *t_edges, *e_edges;
    const int *hash;      // [n_hash+1] bucket b -> last grid index <= lower edge of the bucket
    int hash_shift, hash_lo, n_hash;
    double nu0, nu1, watt_a, watt_b, E_min, E_max;
};

// Particle banks ("dual particle banks"): two dense structure-of-arrays banks.  A sweep reads the
// live particles of bank[s&1] (scatter-bound ones packed at the FRONT, surface-bound ones at the BACK) and
// k_advance writes every survivor, whole, to the front or the back of bank[(s+1)&1]: the queues hold the
// particles themselves, so every load and store of every kernel is coalesced.
// gl packs the group (low 16 bits) and last_surf+1 (high 16 bits); ev = pending event code (or EV_DEAD in the
// monolithic schedule); slot = index of the particle inside its cycle / wave (= its id in eigenvalue mode, R6).
struct Bank {
    double *x, *y, *z, *ux, *uy, *uz, *E, *t;
    int *cell, *elem, *gl, *tbin, *ev;
    uint32_t *ctr, *slot;
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

// Tail kernel, continuous energy: a thread follows its particle AND the prompt-fission subtree below it depth
// first; pending siblings wait on a small per-thread stack in HBM.  If the stack is full the fission is left as
// an ordinary record in the overflow part of FisRec ([M, M + over_cap)) and its children run in the next wave.
struct StackRec {
    double x, y, z, ux, uy, uz, E, t;
    int cell, elem, tbin, pad;
    unsigned long long id;
};
constexpr int STACK_DEPTH = 24;
constexpr unsigned int OVER_CAP = 65536;

struct QCount {  // one set per sweep (ring of RING)
    unsigned int n_scat, n_surf, n_alive, pad;
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
    FisRec fis;
    unsigned int cap;   // slots per bank
    int mode;           // 0 MG, 1 CE
    int n_tally, n_bins;
    int geo_stage;       // 4-byte words of the geometry blob staged in shared memory (0: none)
    int mg_stage;        // doubles of the multi-group table blob staged in shared memory by every transport kernel (0: none)
    int flux_aggregate;  // global tally flavour: 1 = warp-aggregate equal bins before the atomic
    int flux_copy_mask;  // R - 1: the per-cycle tally is kept in R copies, copy = block index & mask
    double *flux;       // [R][n_tally] per-cycle track-length tally
    double *scal;       // [0] k numerator, [1] leakage weight
    unsigned long long *counters;  // [16]
    int *err;           // device error flag
    QCount *qc;          // [RING] per-sweep counts of the front / back regions
    StackRec *stack;     // [stack_threads][STACK_DEPTH]
    unsigned int stack_threads;
    unsigned int *n_over;  // overflow fission records of the running wave
    Trace tr;
    unsigned long long seed;
    unsigned int cycle;
    double w0, k_prev;
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

// Stream (seed, id, domain, cycle): counter = (id_lo, id_hi, domain<<24 | cycle, draw/2); one block yields the
// draws 2b (words 1:0) and 2b+1 (words 3:2); xi = ((u >> 11) + 0.5) 2^-53.  The block is kept in registers so
// that two consecutive draws of one kernel cost one Philox evaluation.
struct Rng {
    uint32_t id_lo, id_hi, w2, k0, k1, ctr, blk;
    uint64_t u0, u1;
    __device__ __forceinline__ void init(unsigned long long seed, unsigned long long id, uint32_t domain, uint32_t cycle,
                                         uint32_t ctr_)
    {
        id_lo = (uint32_t)id; id_hi = (uint32_t)(id >> 32);
        w2 = (domain << 24) | cycle;
        k0 = (uint32_t)seed; k1 = (uint32_t)(seed >> 32);
        ctr = ctr_;
        blk = 0xFFFFFFFFu;
    }
    __device__ __forceinline__ double next()
    {
        uint32_t b = ctr >> 1;
        if (b != blk) {
            uint32_t o0, o1, o2, o3;
            philox4x32_10(id_lo, id_hi, w2, b, k0, k1, o0, o1, o2, o3);
            u0 = ((uint64_t)o1 << 32) | o0;
            u1 = ((uint64_t)o3 << 32) | o2;
            blk = b;
        }
        uint64_t u = (ctr & 1u) ? u1 : u0;
        ctr++;
        return ((double)(u >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    }
};

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

// first index with cum[i] > v, else n-1 (R3)
__device__ __forceinline__ int pick(const double *__restrict__ cum, int n, double v)
{
    int i = 0;
    while (i < n - 1 && !(cum[i] > v)) i++;
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

// ------------------------------------------------------------------ geometry (R11-R14)
__device__ __forceinline__ double surf_f(const Geo &G, int s, double x, double y, double z)
{
    const double *q = G.surf_param + 4 * s;
    int t = G.surf_type[s];
    double q0 = q[0], q1 = q[1], q2 = q[2], q3 = q[3];
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
    int t = G.surf_type[s];
    double q0 = q[0], q1 = q[1], q2 = q[2];
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
    int c1 = G.uco[univ + 1];
    for (int c = G.uco[univ]; c < c1; c++) {
        bool ok = true;
        int k1 = G.cso[c + 1];
        for (int k = G.cso[c]; k < k1; k++)
            if (sense_of(G, G.csi[k], x, y, z, ux, uy, uz, last) != G.css[k]) { ok = false; break; }
        if (ok) return c;
    }
    return -1;
}

// lattice element -> (ix, iy) without an integer division
__device__ __forceinline__ void elem_xy(const Geo &G, int elem, int &ix, int &iy)
{
    iy = (int)__umulhi((unsigned int)elem, G.lat_magic);
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

// full point location from the root universe.  cell = material cell (root cell, or the local cell inside
// lattice element elem); returns false if the point is in no cell.
__device__ __forceinline__ bool locate(const Geo &G, double x, double y, double z, double ux, double uy, double uz, int last,
                                       int &cell, int &elem)
{
    elem = -1;
    cell = find_cell(G, 0, x, y, z, ux, uy, uz, last);
    if (cell < 0) return false;
    if (G.cft[cell] == 1) {
        int ix = (int)floor((x - G.lat_x0) / G.lat_px);
        int iy = (int)floor((y - G.lat_y0) / G.lat_py);
        if (ix < 0 || iy < 0 || ix >= G.lat_nx || iy >= G.lat_ny) { cell = -1; return false; }
        elem = iy * G.lat_nx + ix;
        double xl, yl;
        local_xy(G, elem, x, y, xl, yl);
        cell = find_cell(G, __ldg(G.lat_univ + elem), xl, yl, z, ux, uy, uz, last);
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
    int t = G.surf_type[s];
    double q0 = q[0], q1 = q[1], q2 = q[2], q3 = q[3];
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

// nearest boundary of the current location; candidate order: enclosing-cell surfaces, local-cell surfaces,
// lattice walls -x,+x,-y,+y; ties keep the first (R12, R14).  hit = surface id, or n_surf+k for wall k.
__device__ __forceinline__ double nearest(const Geo &G, double x, double y, double z, double ux, double uy, double uz, int cell,
                                          int elem, int last, int &hit, unsigned int root_mask = 0xffffffffu)
{
    double best = __longlong_as_double(0x7ff0000000000000LL);
    hit = -1;
    const double inv_ux = 1.0 / ux, inv_uy = 1.0 / uy;  // +-inf when the component is zero: guarded at use
    int c0 = elem >= 0 ? G.lat_cell : cell;
    int k1 = G.cso[c0 + 1];
    if (root_mask) {
        // candidates in list order (ties keep the first, R12): the listed bits, then anything past the 32nd surface
        const int k0 = G.cso[c0];
        unsigned int m = k1 - k0 >= 32 ? root_mask : root_mask & ((1u << (k1 - k0)) - 1u);
        while (m) {
            int s = G.csi[k0 + __ffs(m) - 1];
            m &= m - 1u;
            double d = surf_distance(G, s, x, y, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
        for (int k = k0 + 32; k < k1; k++) {
            int s = G.csi[k];
            double d = surf_distance(G, s, x, y, z, ux, uy, uz, s == last, inv_ux, inv_uy);
            if (d < best) { best = d; hit = s; }
        }
    }
    if (elem >= 0) {
        int ix, iy;
        elem_xy(G, elem, ix, iy);
        const double xl = x - (G.lat_x0 + (ix + 0.5) * G.lat_px);
        const double yl = y - (G.lat_y0 + (iy + 0.5) * G.lat_py);
        k1 = G.cso[cell + 1];
        for (int k = G.cso[cell]; k < k1; k++) {
            int s = G.csi[k];
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

__device__ __forceinline__ bool surface_in_cell(const Geo &G, int c, int s)
{
    int k1 = G.cso[c + 1];
    for (int k = G.cso[c]; k < k1; k++)
        if (G.csi[k] == s) return true;
    return false;
}

// ------------------------------------------------------------------ particle in registers
struct Particle {
    double x, y, z, ux, uy, uz, E, t;
    int cell, elem, g, last, tbin;
    unsigned long long id;
};

// Per-thread accumulator (k numerator) reduced once per kernel; event counts by code go to a block-shared
// counter array (integer shared-memory atomics) and leakage straight to the global scalar: both are kept out
// of the registers, which is what limits the occupancy of the latency-bound transport kernels.
struct Acc {
    double knum;
    unsigned int *s_ev;  // [16] in shared memory
    __device__ __forceinline__ void clear(unsigned int *ev) { knum = 0.0; s_ev = ev; }
};

__device__ __forceinline__ void count_event(Acc &acc, int ev) { atomicAdd(acc.s_ev + ev, 1u); }

enum { ADV_DEAD = 0, ADV_SCATTER = 1, ADV_SURFACE = 2, ADV_FISSION = 3 };
constexpr int HIT_TIME_EDGE = 0x3fff0000;  // aux code of a time-edge event in the surface queue
constexpr int HIT_NEWBORN = 0x3fff0001;    // aux code of a prompt secondary just written to the back region

struct TraceRec {  // = mcdc_trace_rec
    unsigned long long id;
    unsigned int cycle, seq;
    int ev, c0, elem, c1, surf, gi;
    double x, y, z, d, E, t;
};

__device__ __forceinline__ void trace_event(const Ctx &c, const Particle &p, int ev, int cell0, int elem0, int surf, int gi,
                                            double d, double E)
{
    if (!c.tr.rec) return;
    unsigned long long rel = p.id - c.tr.first;
    if (p.id < c.tr.first || rel >= c.tr.n_ids) return;
    unsigned long long slot = (unsigned long long)c.cycle * c.tr.n_ids + rel;
    if (slot >= c.tr.cap_slots) return;
    unsigned int seq = c.tr.count[slot]++;
    if (seq >= c.tr.max_events) return;
    TraceRec *r = (TraceRec *)c.tr.rec + slot * c.tr.max_events + seq;
    r->id = p.id; r->cycle = c.cycle; r->seq = seq; r->ev = ev;
    r->c0 = elem0 >= 0 ? c.geo.lat_cell : cell0;
    r->elem = elem0;
    r->c1 = elem0 >= 0 ? cell0 : -1;
    r->surf = surf; r->gi = gi;
    r->x = p.x; r->y = p.y; r->z = p.z; r->d = d; r->E = E; r->t = p.t;
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
            // tree over the ranks inside the group: rank r receives from rank r + step
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

// One segment up to and including the event decision (steps a2/a3, a5, a6, a7 of SURVEY.md 8a and the
// reaction choice of a8): cross sections, distance to collision, nearest boundary, time edge, move, tallies.
// Returns ADV_*; aux = elastic column (scatter), hit code (surface / time edge) or number of children (fission).
template <bool CE, bool PRIVATE>
__device__ __forceinline__ int advance(const Ctx &c, const MGTab &mg, Particle &p, Rng &rng, int &aux, Acc &acc,
                                       double *s_flux, const Geo &G)
{
    const int cell0 = p.cell, elem0 = p.elem;
    const int mat = G.cfill[p.cell];
    int bin = G.cbin[p.cell];
    unsigned int root_mask = 0xffffffffu;
    if (p.elem >= 0) {
        int lb = __ldg(G.lat_bin + p.elem);
        root_mask = (lb & LAT_ROOT_FLAG) ? __ldg(G.lat_rmask + p.elem) : 0u;
        bin += lb & (LAT_ROOT_FLAG - 1);
    }

    double sig_t, nusf, cum[MAX_CE_COL];
    int gi, ncol = 0;
    if (!CE) {
        gi = p.g;
        sig_t = mg.sig_t[mat * mg.G + p.g];
        nusf = mg.nusf[mat * mg.G + p.g];
    } else {
        gi = grid_index(c.ce, p.E);
        double g0 = __ldg(c.ce.grid + gi), g1 = __ldg(c.ce.grid + gi + 1);
        double f = (p.E - g0) / (g1 - g0);
        const double2 *r0 = (const double2 *)(c.ce.tab + ((size_t)mat * c.ce.n_grid + gi) * CE_ROW);
        double2 a0 = __ldg(r0), a1 = __ldg(r0 + 1), a2 = __ldg(r0 + 2), a3 = __ldg(r0 + 3);
        double2 b0 = __ldg(r0 + 4), b1 = __ldg(r0 + 5), b2 = __ldg(r0 + 6), b3 = __ldg(r0 + 7);
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
    double d_coll = -log(rng.next()) / sig_t;
    int hit;
    double d_surf = nearest(G, p.x, p.y, p.z, p.ux, p.uy, p.uz, p.cell, p.elem, p.last, hit, root_mask);
    double v = 0.0, d_time = __longlong_as_double(0x7ff0000000000000LL);
    if (CE) {
        v = speed_of(p.E);
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
    if (!CE) tix = (long long)bin * mg.G + p.g;
    else {
        tix = ((long long)bin * c.ce.n_t + p.tbin) * c.ce.n_e + edge_bin(c.ce.e_edges, c.ce.n_e, p.E);
        if (kind == 2) p.t = __ldg(c.ce.t_edges + p.tbin + 1); else p.t += d / v;
    }
    flux_add<PRIVATE>(c, s_flux, tix, c.w0 * d);
    acc.knum += c.w0 * d * nusf;

    int ev, code;
    if (kind == 0) {
        p.last = -1;
        double uu = rng.next() * sig_t;
        if (!CE) {
            double sig_s = mg.sig_s[mat * mg.G + p.g], sig_f = mg.sig_f[mat * mg.G + p.g];
            if (uu < sig_s) { ev = 1; code = ADV_SCATTER; aux = 0; }
            else if (uu < sig_s + sig_f) {
                ev = 2; code = ADV_FISSION;
                aux = (int)floor(c.w0 * mg.nu[mat * mg.G + p.g] / c.k_prev + rng.next());
            } else { ev = 3; code = ADV_DEAD; }
        } else {
            int r = 0;
            while (r < ncol - 1 && !(cum[r] > uu)) r++;
            if (r < ncol - 2) { ev = 1; code = ADV_SCATTER; aux = r; }
            else if (r == ncol - 2) {
                ev = 2; code = ADV_FISSION;
                double nu = c.ce.nu0 + c.ce.nu1 * (p.E * 1e-6);
                aux = (int)floor(c.w0 * nu + rng.next());
            } else { ev = 3; code = ADV_DEAD; }
        }
        trace_event(c, p, ev, cell0, elem0, -1, gi, d, E_flight);
    } else if (kind == 1) {
        if (hit >= G.n_surf) { ev = 7; code = ADV_SURFACE; aux = hit; }
        else {
            int bc = G.surf_bc[hit];
            if (bc == 2) { ev = 6; code = ADV_DEAD; atomicAdd(c.scal + 1, c.w0); }
            else { ev = bc == 1 ? 5 : 4; code = ADV_SURFACE; aux = hit; }
        }
        trace_event(c, p, ev, cell0, elem0, hit, gi, d, E_flight);
    } else {
        // time edge: the particle has moved off whatever surface it sat on (R11)
        p.tbin++;
        p.last = -1;
        if (p.tbin == c.ce.n_t) { ev = 9; code = ADV_DEAD; }
        else { ev = 8; code = ADV_SURFACE; aux = HIT_TIME_EDGE; }
        trace_event(c, p, ev, cell0, elem0, -1, gi, d, E_flight);
    }
    count_event(acc, ev);
    return code;
}

// Scatter event (a8).  MG: new group from the cumulative scatter row, isotropic direction (1 + 2 draws).
// CE: elastic off a target at rest with mass ratio A: mu_cm, azimuth (2 draws), rotation, energy clamp (R19, R21).
template <bool CE>
__device__ __forceinline__ void do_scatter(const Ctx &c, const MGTab &mg, Particle &p, Rng &rng, int col, const Geo &G)
{
    const int mat = G.cfill[p.cell];
    if (!CE) {
        const int G = mg.G;
        double sig_s = mg.sig_s[mat * G + p.g];
        double vv = rng.next() * sig_s;
        p.g = pick(mg.cumS + (mat * G + p.g) * G, G, vv);
        double a = rng.next(), b = rng.next();
        iso_dir(a, b, p.ux, p.uy, p.uz);
    } else {
        double A = __ldg(c.ce.colA + mat * CE_ROW + col);
        double mu_cm = 2.0 * rng.next() - 1.0;
        double den = A * A + 2.0 * A * mu_cm + 1.0;
        double mu = 0.0;
        if (den > 0.0) mu = (1.0 + A * mu_cm) / sqrt(den);
        double En = p.E * den / ((A + 1.0) * (A + 1.0));
        double sp, cp;
        sincospi(2.0 * rng.next(), &sp, &cp);
        double s2 = 1.0 - mu * mu;
        double s = s2 > 0.0 ? sqrt(s2) : 0.0;
        double a2 = 1.0 - p.uz * p.uz;
        double ox, oy, oz;
        if (a2 < 1e-10) {
            ox = s * cp; oy = s * sp; oz = p.uz > 0.0 ? mu : -mu;
        } else {
            double r = sqrt(a2);
            ox = mu * p.ux + s * (p.ux * p.uz * cp - p.uy * sp) / r;
            oy = mu * p.uy + s * (p.uy * p.uz * cp + p.ux * sp) / r;
            oz = mu * p.uz - s * r * cp;
        }
        double nrm = sqrt(ox * ox + oy * oy + oz * oz);
        p.ux = ox / nrm; p.uy = oy / nrm; p.uz = oz / nrm;
        if (En < c.ce.E_min) En = c.ce.E_min;
        if (En > c.ce.E_max) En = c.ce.E_max;
        p.E = En;
    }
    p.last = -1;
}

// Surface event (a9): lattice wall -> neighbour element; reflect; transmit -> neighbour cell by the side being
// entered (R11, R14).  Time-edge events need no geometry work.  Returns false if the particle got lost.
__device__ __forceinline__ bool do_surface(const Geo &G, Particle &p, int hit)
{
    if (hit == HIT_TIME_EDGE) return true;
    if (hit >= G.n_surf) {
        int w = hit - G.n_surf;
        int ix, iy;
        elem_xy(G, p.elem, ix, iy);
        if (w == 0) ix--; else if (w == 1) ix++; else if (w == 2) iy--; else iy++;
        p.elem = iy * G.lat_nx + ix;
        p.last = -1;
        double xl, yl;
        local_xy(G, p.elem, p.x, p.y, xl, yl);
        p.cell = find_cell(G, __ldg(G.lat_univ + p.elem), xl, yl, p.z, p.ux, p.uy, p.uz, -1);
        return p.cell >= 0;
    }
    int bc = G.surf_bc[hit];
    bool local = p.elem >= 0 && !surface_in_cell(G, G.lat_cell, hit);
    double xl = p.x, yl = p.y;
    if (local) local_xy(G, p.elem, p.x, p.y, xl, yl);
    p.last = hit;
    if (bc == 1) {
        int t = G.surf_type[hit];
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
        p.cell = find_cell(G, __ldg(G.lat_univ + p.elem), xl, yl, p.z, p.ux, p.uy, p.uz, hit);
        return p.cell >= 0;
    }
    return locate(G, p.x, p.y, p.z, p.ux, p.uy, p.uz, hit, p.cell, p.elem);
}

// Watt spectrum, rejection-free (R22); MeV
__device__ __forceinline__ double watt(double a, double b, double x1, double x2, double x3, double x4)
{
    double cs = cospi(0.5 * x3);
    double W = -a * (log(x1) + log(x2) * cs * cs);
    return W + 0.25 * a * a * b + (2.0 * x4 - 1.0) * sqrt(a * a * b * W);
}

}  // namespace mcdc
