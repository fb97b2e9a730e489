// mcdc_lib.cu -- host side of the C-ABI (include/mcdc.h): input validation and derived tables, workspace
// carving, the sweep / cycle drivers and result read-back.  All device work is in mcdc_kernels.cuh.
#include "../../include/mcdc.h"
#include "../../include/mcdc_test.h"
#include "mcdc_kernels.cuh"
#include "mcdc_census.cuh"
#include "mcdc_microbench.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

using namespace mcdc;

static thread_local std::string g_err;
static int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}
#define CUDA_OK(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) return fail(MCDC_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));   \
    } while (0)

// seed of the run and its ten Philox round keys (Ctx::rk)
static void set_seed(Ctx &c, uint64_t seed)
{
    c.seed = seed;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; r++) { c.rk[2 * r] = k0; c.rk[2 * r + 1] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
}

static const int LAG = 3;                 // sweeps the host may run ahead of the queue-count read-back
// live particles at or below which the persistent kernel takes over from the event sweeps.  Measured on B200
// (profiles/r02_schedules.md, ms per C4 cycle): 1.5e6 -> 36.1, 4e6 -> 33.7, 6e6 -> 32.3, 9e6 -> 30.5, always -> 29.2:
// the default is "always" -- a cycle (a whole fixed-source run) is ONE persistent launch.
#ifndef MCDC_PERSIST_DEFAULT
#define MCDC_PERSIST_DEFAULT 0x7fffffff
#endif
static const int DEFAULT_PERSIST = MCDC_PERSIST_DEFAULT;
static const int DEFAULT_PERSIST_CE = 0x7fffffff;
static const uint64_t TRACE_BYTES = 48ull << 20;
#ifndef MCDC_AGG_MAX
#define MCDC_AGG_MAX 4096
#endif
static const int AGGREGATE_TALLY_MAX = MCDC_AGG_MAX;  // above this, equal bins inside a warp are rare: plain float64 atomics
static const uint64_t MG_STAGE_MAX_BYTES = 16384;  // multi-group tables up to this size are staged in shared memory
static const int PRIVATE_TALLY_MAX = 20;  // bins for which the one-column-per-thread tally fits (20*256*8 = 40 KB)
static const int MAX_AXIS_PLANES = 250;   // axis planes a boundary code of the straight-line geometry path can name

struct HostPinned {
    QCount qc[RING];
    unsigned int census[4];  // [0] census-bank count read back, [1] particles of the next interval, [2] count to set
    double comb_w;           // total weight of the particles entering an interval
    double scal[8];
    unsigned long long counters[MCDC_N_COUNTERS];
    unsigned int total;
    int err;
};

// statistics of a run; `work` is the run in progress, `pub` the state after the last call that succeeded
// (what mcdc_get_dims / mcdc_get_tallies report: a failed call leaves it untouched)
struct RunStats {
    std::vector<double> k_cycle;
    int n_active = 0;
    double k_acc = 0, k_acc2 = 0, leak_acc = 0, leak_acc2 = 0;
    uint64_t host_counters[MCDC_N_COUNTERS] = {0};  // [0] histories started from a source bank, [11] children banked by
                                                    // k_emit, [12] largest bank, [13] kernel rounds
    uint64_t counters[MCDC_N_COUNTERS] = {0};       // merged device + host counters as reported
    int set = 0;                                    // which flux accumulator pair holds this run's tallies
    double balance[6] = {0, 0, 0, 0, 0, 0};         // weight balance summed over the run's cycles (mcdc_get_balance)
    std::vector<uint64_t> census_counts;            // per census interval: particles before / after the comb
    std::vector<double> census_weights;             // and their total weights
    int next_interval = -1;                         // fixed source by intervals: the interval the next call must name
};

struct mcdc_problem {
    Ctx ctx;
    int mode;
    cudaStream_t stream;
    int device;
    int schedule, persist;
    int persist_blocks_per_sm, n_sm;  // resident blocks of the persistent kernel (occupancy query at first use)
    uint64_t cap;  // bank slots
    // time-dependent fixed source: census banks (ping-pong), radix-sort and comb scratch
    bool timed, td;
    int first_interval;
    long long census_target;
    Bank cb[2];
    int cb_cur;
    unsigned long long *sort_key[2];
    unsigned int *sort_idx[2], *sort_hist, *comb_copies, *comb_offs;
    double *comb_w;
    uint64_t census_n;  // particles in the current census bank
    // workspace pieces not in ctx
    double *flux_acc[2], *flux_acc2[2], *flux_cycle;
    int flux_copies;
    unsigned int *part;
    Site *sites;
    char *trace_base;
    unsigned int *trace_count;
    HostPinned *pin;
    cudaEvent_t ev[RING], t0, t1;
    // run state
    uint64_t bank_count;  // sites in bank[0] to start the next cycle from
    double k_prev;
    RunStats work, pub;
    bool dirty;  // a call failed part-way: per-cycle device tallies must be cleared before the next cycle
    double ms_transport;
    uint64_t n_launches;
    bool tally_private;
    uint64_t last_N;
    // optional per-kernel-class timing (mcdc_set_profile): event pairs around every launch
    int profile;
    std::vector<cudaEvent_t> pool;
    std::vector<int> pool_class;  // class of pair k (events 2k, 2k+1)
    double prof_ms[MCDC_N_PROFILE];
    uint64_t prof_launches[MCDC_N_PROFILE];
    uint64_t prof_sweep_base;  // device counter 12 (segments run by the sweep kernels) when profiling was switched on
};

// record an event pair around one launch when profiling is on
struct ProfScope {
    mcdc_problem *p;
    size_t k;
    ProfScope(mcdc_problem *p_, int cls) : p(p_), k((size_t)-1)
    {
        if (!p->profile) return;
        k = p->pool_class.size();
        if (p->pool.size() < 2 * (k + 1)) {
            cudaEvent_t a, b;
            cudaEventCreate(&a); cudaEventCreate(&b);
            p->pool.push_back(a); p->pool.push_back(b);
        }
        p->pool_class.push_back(cls);
        cudaEventRecord(p->pool[2 * k], p->stream);
    }
    ~ProfScope() { if (k != (size_t)-1) cudaEventRecord(p->pool[2 * k + 1], p->stream); }
};

static void profile_collect(mcdc_problem *p)  // call after a stream synchronize
{
    for (size_t k = 0; k < p->pool_class.size(); k++) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p->pool[2 * k], p->pool[2 * k + 1]) == cudaSuccess) {
            p->prof_ms[p->pool_class[k]] += ms;
            p->prof_launches[p->pool_class[k]]++;
        }
    }
    p->pool_class.clear();
}

// ------------------------------------------------------------------ workspace layout
struct Carver {
    char *base;
    uint64_t off;
    explicit Carver(void *b) : base((char *)b), off(0) {}
    template <class T> T *take(uint64_t n)
    {
        off = (off + 255u) & ~255ull;
        T *p = base ? (T *)(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

struct Layout {  // everything carved from the workspace, in order
    int *surf_type, *surf_bc, *cso, *csi, *css, *cft, *cfill, *cbin, *uco, *ap_sid;
    int4 *lat_info, *ufast, *cell_info, *l2_info;
    int *l2_nx, *l2_ny, *l2_off, *l2_univ, *l2_bin, *umid;
    double *l2_px, *l2_py;
    Trace *tr_g;
    unsigned int *lat_rmask;
    double *surf_param, *ap_pos;
    double *mg_blob;
    uint64_t mg_doubles;
    double *grid, *tab, *colA, *t_edges, *e_edges;
    int *ncol, *hash, *ehash;
    Bank bank[2], cb[2];
    unsigned long long *sort_key[2];
    unsigned int *sort_idx[2], *sort_hist, *comb_copies, *comb_offs;
    double *comb_w, *td_speed, *td_cum_nu, *td_cumchi_d, *td_decay;
    FisRec fis;
    QCount *qc;
    double *flux, *flux_acc[2], *flux_acc2[2], *flux_cycle, *scal;
    unsigned long long *counters;
    int *err;
    unsigned int *work;
    unsigned int *part;
    Site *sites;
    char *trace;
    unsigned int *trace_count;
    uint64_t bytes;
};

// The per-cycle tally is replicated (copy = block index mod R) so that hot bins (e.g. one reflector bin that a
// large share of all segments hits) do not serialise on one L2 address; k_accumulate sums the copies.
static int flux_copies_for(uint64_t n_tally)
{
    int r = 64;
    while (r > 1 && (uint64_t)r * n_tally * 8 > (4ull << 20)) r >>= 1;
    return r;
}

static uint64_t n_tally_of(const mcdc_materials *mat, const mcdc_tally_spec *t)
{
    if (mat) return mat->kinetics ? (uint64_t)t->n_bins * t->n_t * mat->G : (uint64_t)t->n_bins * mat->G;
    return (uint64_t)t->n_bins * t->n_t * t->n_e;
}

static int hash_params(const double *grid, int n, int &shift, int &lo, int &n_hash)
{
    // key = top bits of the IEEE-754 pattern: exponent + m mantissa bits => 2^m buckets per octave, m chosen so that a
    // bucket holds about half a grid point on average (the bisection inside a bucket is then 0 or 1 probe)
    double octaves = std::max(1.0, std::log2(grid[n - 1] / grid[0]));
    int m = (int)std::ceil(std::log2(2.0 * n / octaves));
    m = std::max(4, std::min(m, 12));
    shift = 52 - m;
    long long klo, khi;
    double a = grid[0], b = grid[n - 1];
    memcpy(&klo, &a, 8);
    memcpy(&khi, &b, 8);
    lo = (int)(klo >> shift);
    n_hash = (int)(khi >> shift) - lo + 1;
    return 0;
}

// energy-bin edges: 16 buckets per octave
static const int EHASH_SHIFT = 52 - 4;
static int ehash_buckets(const double *edges, int n_e)
{
    long long klo, khi;
    memcpy(&klo, &edges[0], 8);
    memcpy(&khi, &edges[n_e], 8);
    return (int)(khi >> EHASH_SHIFT) - (int)(klo >> EHASH_SHIFT) + 1;
}

static void carve(Layout &L, void *ws, const mcdc_geometry *g, const mcdc_materials *m, const mcdc_xs *x,
                  const mcdc_tally_spec *t, uint64_t cap)
{
    Carver C(ws);
    int nref = g->cell_surf_off[g->n_cell];
    int nlat = g->has_lattice ? g->lat_nx * g->lat_ny : 0;
    uint64_t ns = g->n_surf, nc = g->n_cell;
    L.surf_param = C.take<double>(4 * ns); L.surf_type = C.take<int>(ns); L.surf_bc = C.take<int>(ns);
    L.cso = C.take<int>(nc + 1); L.csi = C.take<int>(nref); L.css = C.take<int>(nref);
    L.cft = C.take<int>(nc); L.cfill = C.take<int>(nc); L.cbin = C.take<int>(nc); L.uco = C.take<int>(g->n_univ + 1);
    L.ufast = C.take<int4>(g->n_univ);
    L.cell_info = C.take<int4>(nc);
    L.tr_g = C.take<Trace>(1);
    L.ap_pos = C.take<double>(MAX_AXIS_PLANES); L.ap_sid = C.take<int>(MAX_AXIS_PLANES);
    L.lat_info = C.take<int4>(nlat); L.lat_rmask = C.take<unsigned int>(nlat);
    {
        uint64_t n2 = g->n_lat2 > 0 ? g->n_lat2 : 0, ne2 = n2 ? g->lat2_off[n2] : 0;
        L.l2_nx = C.take<int>(n2); L.l2_ny = C.take<int>(n2); L.l2_off = C.take<int>(n2 + 1);
        L.l2_px = C.take<double>(n2); L.l2_py = C.take<double>(n2);
        L.l2_univ = C.take<int>(ne2); L.l2_bin = C.take<int>(ne2); L.l2_info = C.take<int4>(ne2);
        L.umid = C.take<int>(g->n_univ);
    }
    bool ce = x != nullptr;
    const bool td = !ce && m->kinetics != nullptr, timed = ce || td;
    if (!ce) {
        uint64_t mg = (uint64_t)m->n_mat * m->G;
        // one contiguous blob (staged in shared memory by the kernels): six [n_mat][G] tables, cumS, src_cum
        L.mg_doubles = 7 * mg + mg * m->G + m->G;
        L.mg_blob = C.take<double>(L.mg_doubles);
        L.grid = L.tab = L.colA = L.t_edges = L.e_edges = nullptr; L.ncol = L.hash = L.ehash = nullptr;
        L.td_speed = L.td_cum_nu = L.td_cumchi_d = L.td_decay = nullptr;
        if (td) {
            uint64_t J = m->kinetics->n_dgroup;
            L.td_speed = C.take<double>(m->G); L.td_cum_nu = C.take<double>(mg * (J + 1));
            L.td_cumchi_d = C.take<double>((uint64_t)m->n_mat * J * m->G + 1); L.td_decay = C.take<double>((uint64_t)m->n_mat * J + 1);
            L.t_edges = C.take<double>(t->n_t + 1);
        }
    } else {
        int sh, lo, nh;
        hash_params(x->grid, x->n_grid, sh, lo, nh);
        L.grid = C.take<double>(x->n_grid);
        L.tab = C.take<double>((uint64_t)x->n_mat * x->n_grid * CE_ROW);
        L.colA = C.take<double>((uint64_t)x->n_mat * CE_ROW);
        L.ncol = C.take<int>(x->n_mat);
        L.hash = C.take<int>(nh + 2);
        L.ehash = C.take<int>(ehash_buckets(t->e_edges, t->n_e) + 2);
        L.t_edges = C.take<double>(t->n_t + 1); L.e_edges = C.take<double>(t->n_e + 1);
        L.mg_blob = nullptr;
        L.mg_doubles = 0;
    }
    for (int b = 0; b < 4; b++) {  // the two particle banks; for time-dependent problems also the two census banks
        Bank &B = b < 2 ? L.bank[b] : L.cb[b - 2];
        if (b >= 2 && !timed) { memset(&B, 0, sizeof B); continue; }
        B.x = C.take<double>(cap); B.y = C.take<double>(cap); B.z = C.take<double>(cap);
        B.ux = C.take<double>(cap); B.uy = C.take<double>(cap); B.uz = C.take<double>(cap);
        B.w = C.take<double>(cap);
        B.E = ce ? C.take<double>(cap) : nullptr; B.t = timed ? C.take<double>(cap) : nullptr;
        B.cell = C.take<int>(cap); B.elem = C.take<int>(cap); B.gl = C.take<int>(cap);
        B.tbin = timed ? C.take<int>(cap) : nullptr;
        B.ev = C.take<uint32_t>(cap);
        B.ctr = C.take<uint32_t>(cap); B.slot = C.take<uint32_t>(cap);
        B.id = timed ? C.take<uint64_t>(cap) : nullptr;
    }
    if (timed) {
        for (int b = 0; b < 2; b++) { L.sort_key[b] = C.take<unsigned long long>(cap); L.sort_idx[b] = C.take<unsigned int>(cap); }
        L.sort_hist = C.take<unsigned int>(256 * (cap / RS_TILE + 1) + 4);
        L.comb_copies = C.take<unsigned int>(cap + 4); L.comb_offs = C.take<unsigned int>(cap + 4);
        L.comb_w = C.take<double>(cap);
    } else {
        L.sort_key[0] = L.sort_key[1] = nullptr; L.sort_idx[0] = L.sort_idx[1] = nullptr;
        L.sort_hist = L.comb_copies = L.comb_offs = nullptr; L.comb_w = nullptr;
    }
    {
        FisRec &F = L.fis;
        F.n = C.take<int>(cap); F.cell = C.take<int>(cap); F.elem = C.take<int>(cap);
        F.tbin = ce ? C.take<int>(cap) : nullptr;
        F.x = C.take<double>(cap); F.y = C.take<double>(cap); F.z = C.take<double>(cap);
        F.t = ce ? C.take<double>(cap) : nullptr;
        F.ctr = C.take<uint32_t>(cap);
        F.id = ce ? C.take<uint64_t>(cap) : nullptr;
    }
    L.qc = C.take<QCount>(RING);
    uint64_t nt = n_tally_of(m, t);
    L.flux = C.take<double>(nt * flux_copies_for(nt));
    for (int k = 0; k < 2; k++) { L.flux_acc[k] = C.take<double>(nt); L.flux_acc2[k] = C.take<double>(nt); }
    L.flux_cycle = C.take<double>(nt);
    L.scal = C.take<double>(8);
    L.counters = C.take<unsigned long long>(MCDC_N_COUNTERS);
    L.err = C.take<int>(4);
    L.work = C.take<unsigned int>(8);
    L.part = C.take<unsigned int>(cap / BS + 4);
    L.sites = C.take<Site>(cap);
    L.trace = C.take<char>(TRACE_BYTES);
    L.trace_count = C.take<unsigned int>(TRACE_BYTES / sizeof(TraceRec) + 1);
    C.take<char>(256);
    L.bytes = C.off;
}

static uint64_t capacity_for(uint64_t n) { return 2 * n + 1024; }  // R6: bank capacity 2N

// ------------------------------------------------------------------ validation
static int validate(const mcdc_geometry *g, const mcdc_materials *m, const mcdc_xs *x, const mcdc_source *s,
                    const mcdc_tally_spec *t)
{
    if (!g || !s || !t) return fail(MCDC_EINVAL, "null geometry / source / tally");
    if ((m != nullptr) == (x != nullptr)) return fail(MCDC_EINVAL, "exactly one of materials (MG) and xs (CE) must be given");
    if (g->n_cell < 1 || g->n_univ < 1 || g->n_surf < 0) return fail(MCDC_EINVAL, "empty geometry");
    if (g->n_surf > MAX_SURFACES) return fail(MCDC_EINVAL, "too many surfaces (at most %d)", MAX_SURFACES);
    if (t->n_bins < 1) return fail(MCDC_EINVAL, "n_bins");
    int n_mat = m ? m->n_mat : x->n_mat;
    int n_lat_cells = 0;
    if (g->cell_surf_off[0] != 0) return fail(MCDC_EINVAL, "cell_surf_off[0] must be 0");
    if (g->univ_cell_off[0] != 0 || g->univ_cell_off[g->n_univ] != g->n_cell) return fail(MCDC_EINVAL, "univ_cell_off must run from 0 to n_cell");
    for (int u = 0; u < g->n_univ; u++)
        if (g->univ_cell_off[u + 1] < g->univ_cell_off[u]) return fail(MCDC_EINVAL, "univ_cell_off not monotone");
    for (int c = 0; c < g->n_cell; c++) {
        if (g->cell_surf_off[c + 1] < g->cell_surf_off[c]) return fail(MCDC_EINVAL, "cell_surf_off not monotone");
        for (int k = g->cell_surf_off[c]; k < g->cell_surf_off[c + 1]; k++) {
            if (g->cell_surf_id[k] < 0 || g->cell_surf_id[k] >= g->n_surf) return fail(MCDC_EGEOM, "cell %d names surface %d", c, g->cell_surf_id[k]);
            if (g->cell_surf_sense[k] != 1 && g->cell_surf_sense[k] != -1) return fail(MCDC_EGEOM, "sense must be +-1");
        }
        if (g->cell_fill_type[c] == 1) {
            n_lat_cells++;
            if (c >= g->univ_cell_off[1]) return fail(MCDC_EGEOM, "the lattice-filled cell must belong to the root universe");
        } else if (g->cell_fill_type[c] == 2) {
            if (g->n_lat2 < 1 || g->cell_fill[c] < 0 || g->cell_fill[c] >= g->n_lat2) return fail(MCDC_EGEOM, "cell %d names second-level lattice %d", c, g->cell_fill[c]);
            if (c < g->univ_cell_off[1]) return fail(MCDC_EGEOM, "a second-level lattice must fill a cell of a lattice element's universe, not of the root");
        } else if (g->cell_fill_type[c] != 0) return fail(MCDC_EGEOM, "cell %d: fill type %d", c, g->cell_fill_type[c]);
        else if (g->cell_fill[c] < 0 || g->cell_fill[c] >= n_mat) return fail(MCDC_EINVAL, "cell %d material %d out of range", c, g->cell_fill[c]);
        if (t->cell_bin[c] < 0 || t->cell_bin[c] >= t->n_bins) return fail(MCDC_EINVAL, "cell_bin out of range");
    }
    for (int sidx = 0; sidx < g->n_surf; sidx++) {
        if (g->surf_type[sidx] < 0 || g->surf_type[sidx] > 7) return fail(MCDC_EGEOM, "surface type");
        if (g->surf_bc[sidx] < 0 || g->surf_bc[sidx] > 2) return fail(MCDC_EGEOM, "surface bc");
    }
    if (g->has_lattice) {
        if (n_lat_cells != 1) return fail(MCDC_EGEOM, "exactly one lattice-filled cell is supported");
        if (g->lat_nx < 1 || g->lat_ny < 1 || !(g->lat_px > 0) || !(g->lat_py > 0)) return fail(MCDC_EGEOM, "lattice shape");
        if ((unsigned long long)g->lat_nx * g->lat_nx * g->lat_ny >= 0x100000000ull) return fail(MCDC_EGEOM, "lattice too large (nx*nx*ny must be < 2^32)");
        if ((long long)g->lat_nx * g->lat_ny > (1 << 20)) return fail(MCDC_EGEOM, "lattice too large (at most 2^20 elements)");
        if (!t->lat_bin) return fail(MCDC_EINVAL, "lat_bin missing");
        int max_lat_bin = 0;
        for (int e = 0; e < g->lat_nx * g->lat_ny; e++) {
            if (g->lat_univ[e] < 1 || g->lat_univ[e] >= g->n_univ) return fail(MCDC_EGEOM, "lattice element %d names universe %d", e, g->lat_univ[e]);
            if (t->lat_bin[e] < 0 || t->lat_bin[e] >= t->n_bins) return fail(MCDC_EINVAL, "lat_bin out of range");
            max_lat_bin = std::max(max_lat_bin, t->lat_bin[e]);
        }
        // inside the lattice the bin is cell_bin[local cell] + lat_bin[element]: the sum must stay inside the tally
        for (int c = g->univ_cell_off[1]; c < g->n_cell; c++)
            if (t->cell_bin[c] + max_lat_bin >= t->n_bins) return fail(MCDC_EINVAL, "cell_bin[%d] + max lat_bin reaches past n_bins", c);
    } else if (n_lat_cells) return fail(MCDC_EGEOM, "lattice-filled cell without a lattice");
    if (g->n_lat2 < 0) return fail(MCDC_EGEOM, "n_lat2");
    if (g->n_lat2 > 0) {  // second-level lattices (R37)
        if (!g->has_lattice) return fail(MCDC_EGEOM, "second-level lattices need a first-level lattice");
        if (!g->lat2_nx || !g->lat2_ny || !g->lat2_px || !g->lat2_py || !g->lat2_off || !g->lat2_univ || !t->lat2_bin)
            return fail(MCDC_EINVAL, "second-level lattice arrays missing");
        if (g->lat2_off[0] != 0) return fail(MCDC_EINVAL, "lat2_off[0] must be 0");
        // universes that lattice elements of either level use; which of them hold a second-level lattice
        std::vector<char> has2(g->n_univ, 0);
        for (int u = 1; u < g->n_univ; u++) {
            int n2 = 0;
            for (int c = g->univ_cell_off[u]; c < g->univ_cell_off[u + 1]; c++) n2 += g->cell_fill_type[c] == 2;
            if (n2 > 1) return fail(MCDC_EGEOM, "universe %d has more than one cell filled by a second-level lattice", u);
            has2[u] = n2 == 1;
        }
        // largest cell_bin per universe; largest (lat2_bin + cell_bin) per second-level lattice
        std::vector<int> ubin(g->n_univ, 0), l2max(g->n_lat2, 0);
        for (int u = 1; u < g->n_univ; u++)
            for (int c = g->univ_cell_off[u]; c < g->univ_cell_off[u + 1]; c++) ubin[u] = std::max(ubin[u], t->cell_bin[c]);
        for (int k = 0; k < g->n_lat2; k++) {
            if (g->lat2_nx[k] < 1 || g->lat2_ny[k] < 1 || !(g->lat2_px[k] > 0) || !(g->lat2_py[k] > 0)) return fail(MCDC_EGEOM, "second-level lattice %d: shape", k);
            if ((long long)g->lat2_nx[k] * g->lat2_ny[k] > 2047) return fail(MCDC_EGEOM, "second-level lattice %d has more than 2047 elements", k);
            if (g->lat2_off[k + 1] - g->lat2_off[k] != g->lat2_nx[k] * g->lat2_ny[k]) return fail(MCDC_EINVAL, "lat2_off[%d]", k + 1);
            for (int e = g->lat2_off[k]; e < g->lat2_off[k + 1]; e++) {
                int u = g->lat2_univ[e];
                if (u < 1 || u >= g->n_univ) return fail(MCDC_EGEOM, "second-level lattice %d names universe %d", k, u);
                if (has2[u]) return fail(MCDC_EGEOM, "second-level lattice %d: universe %d holds a lattice itself (two levels at most)", k, u);
                if (t->lat2_bin[e] < 0 || t->lat2_bin[e] >= (1 << 19)) return fail(MCDC_EINVAL, "lat2_bin out of range (0 .. 2^19 - 1)");
                l2max[k] = std::max(l2max[k], t->lat2_bin[e] + ubin[u]);
            }
        }
        // inside second-level lattice k of first-level element e the bin is lat_bin[e] + lat2_bin + cell_bin
        for (int e = 0; e < g->lat_nx * g->lat_ny; e++) {
            int u = g->lat_univ[e];
            for (int c = g->univ_cell_off[u]; c < g->univ_cell_off[u + 1]; c++)
                if (g->cell_fill_type[c] == 2 && t->lat_bin[e] + l2max[g->cell_fill[c]] >= t->n_bins)
                    return fail(MCDC_EINVAL, "lat_bin[%d] + lat2_bin + cell_bin reaches past n_bins", e);
        }
    }
    for (int k = 0; k < 3; k++)
        if (!(s->hi[k] >= s->lo[k])) return fail(MCDC_EINVAL, "source box: hi < lo on axis %d", k);
    if (m) {
        if (m->G < 1 || m->G > 4096 || m->n_mat < 1) return fail(MCDC_EINVAL, "G / n_mat");
        for (int i = 0; i < m->n_mat * m->G; i++) {
            double ss = 0.0;
            for (int gp = 0; gp < m->G; gp++) {
                double v = m->S[(size_t)i * m->G + gp];
                if (!(v >= 0.0)) return fail(MCDC_EINVAL, "negative scatter matrix entry");
                ss += v;
            }
            if (!(m->sig_t[i] > 0.0) || !(m->sig_f[i] >= 0.0)) return fail(MCDC_EINVAL, "Sigma_t must be > 0, Sigma_f >= 0");
            if (ss + m->sig_f[i] > m->sig_t[i] * (1.0 + 1e-12)) return fail(MCDC_EINVAL, "Sigma_s + Sigma_f > Sigma_t (material/group %d)", i);
        }
        if (!s->group_pdf) return fail(MCDC_EINVAL, "source group pdf missing");
        if (m->kinetics) {  // time-dependent multi-group (R38-R40)
            const mcdc_kinetics *kn = m->kinetics;
            if (!kn->speed || kn->n_dgroup < 0 || kn->n_dgroup > 64) return fail(MCDC_EINVAL, "kinetics: speed / n_dgroup");
            if (kn->n_dgroup > 0 && (!kn->nu_d || !kn->decay || !kn->chi_d)) return fail(MCDC_EINVAL, "kinetics: delayed-neutron arrays missing");
            for (int gg = 0; gg < m->G; gg++) if (!(kn->speed[gg] > 0.0)) return fail(MCDC_EINVAL, "kinetics: speed must be > 0");
            for (int i = 0; i < m->n_mat * kn->n_dgroup; i++) if (!(kn->decay[i] > 0.0)) return fail(MCDC_EINVAL, "kinetics: decay constants must be > 0");
            for (int i = 0; i < m->n_mat * kn->n_dgroup * m->G; i++) if (!(kn->nu_d[i] >= 0.0) || !(kn->chi_d[i] >= 0.0)) return fail(MCDC_EINVAL, "kinetics: negative yield / spectrum");
            if (kn->census_target < 0) return fail(MCDC_EINVAL, "kinetics: census_target");
            if (t->n_t < 1 || !t->t_edges) return fail(MCDC_EINVAL, "time-dependent problem without time edges");
            for (int i = 0; i < t->n_t; i++) if (!(t->t_edges[i + 1] > t->t_edges[i])) return fail(MCDC_EINVAL, "t_edges");
            if (!(s->t >= t->t_edges[0]) || !(s->t < t->t_edges[t->n_t])) return fail(MCDC_EINVAL, "source time outside the time edges");
        }
    } else {
        if (x->n_grid < 2 || x->n_nuc < 1) return fail(MCDC_EINVAL, "CE grid");
        for (int i = 1; i < x->n_grid; i++)
            if (!(x->grid[i] > x->grid[i - 1])) return fail(MCDC_EINVAL, "union grid not strictly increasing at %d", i);
        if (!(x->grid[0] > 0.0)) return fail(MCDC_EINVAL, "grid must be positive");
        if (x->mat_nuc_off[0] != 0) return fail(MCDC_EINVAL, "mat_nuc_off[0] must be 0");
        for (int mm = 0; mm < x->n_mat; mm++) {
            int nn = x->mat_nuc_off[mm + 1] - x->mat_nuc_off[mm];
            if (nn < 1 || nn + 2 > MAX_CE_COL) return fail(MCDC_EINVAL, "material %d: 1..%d nuclides supported", mm, MAX_CE_COL - 2);
            for (int j = x->mat_nuc_off[mm]; j < x->mat_nuc_off[mm + 1]; j++)
                if (x->mat_nuc_id[j] < 0 || x->mat_nuc_id[j] >= x->n_nuc) return fail(MCDC_EINVAL, "nuclide id");
        }
        if (t->n_t < 1 || t->n_e < 1 || !t->t_edges || !t->e_edges) return fail(MCDC_EINVAL, "CE tally edges");
        for (int i = 0; i < t->n_t; i++) if (!(t->t_edges[i + 1] > t->t_edges[i])) return fail(MCDC_EINVAL, "t_edges");
        for (int i = 0; i < t->n_e; i++) if (!(t->e_edges[i + 1] > t->e_edges[i])) return fail(MCDC_EINVAL, "e_edges");
        if (!(s->t >= t->t_edges[0]) || !(s->t < t->t_edges[t->n_t])) return fail(MCDC_EINVAL, "source time outside the time edges");
        if (!(s->E > 0.0)) return fail(MCDC_EINVAL, "source energy");
    }
    return 0;
}

extern "C" int mcdc_workspace_bytes(const mcdc_geometry *geo, const mcdc_materials *mat, const mcdc_xs *xs,
                                    const mcdc_tally_spec *tally, uint64_t n_particles, uint64_t *bytes)
{
    if (!geo || !tally || !bytes || ((mat != nullptr) == (xs != nullptr))) return fail(MCDC_EINVAL, "bad arguments");
    Layout L;
    carve(L, nullptr, geo, mat, xs, tally, capacity_for(n_particles));
    *bytes = L.bytes;
    return 0;
}

template <class T> static cudaError_t up(T *dst, const T *src, uint64_t n, cudaStream_t st)
{
    if (!n) return cudaSuccess;
    return cudaMemcpyAsync(dst, src, n * sizeof(T), cudaMemcpyHostToDevice, st);
}

// Per-universe shape used by the straight-line geometry path: one cell without surfaces, or two cells that are the
// inside (-) and the outside (+) of one z-cylinder and nothing else.
static void classify_universes(const mcdc_geometry *g, std::vector<int4> &uf)
{
    uf.assign(g->n_univ, make_int4(0, -1, -1, -1));
    for (int u = 1; u < g->n_univ; u++) {
        int c0 = g->univ_cell_off[u], nc = g->univ_cell_off[u + 1] - c0;
        auto nsurf = [&](int c) { return g->cell_surf_off[c + 1] - g->cell_surf_off[c]; };
        if (nc == 1 && nsurf(c0) == 0 && g->cell_fill_type[c0] == 0) uf[u] = make_int4(1, -1, c0, c0);
        else if (nc == 2 && nsurf(c0) == 1 && nsurf(c0 + 1) == 1 && g->cell_fill_type[c0] == 0 && g->cell_fill_type[c0 + 1] == 0) {
            int ka = g->cell_surf_off[c0], kb = g->cell_surf_off[c0 + 1];
            int sa = g->cell_surf_id[ka], sb = g->cell_surf_id[kb];
            if (sa == sb && g->surf_type[sa] == MCDC_CYL_Z && g->cell_surf_sense[ka] == -g->cell_surf_sense[kb]) {
                int in = g->cell_surf_sense[ka] < 0 ? c0 : c0 + 1;
                uf[u] = make_int4(1, sa, in, in == c0 ? c0 + 1 : c0);
            }
        }
    }
}

extern "C" int mcdc_create(const mcdc_geometry *g, const mcdc_materials *m, const mcdc_xs *x, const mcdc_source *s,
                           const mcdc_tally_spec *t, const mcdc_device *dev, uint64_t max_particles, mcdc_problem **out)
{
    if (!out) return fail(MCDC_EINVAL, "out is null");
    *out = nullptr;
    int rc = validate(g, m, x, s, t);
    if (rc) return rc;
    if (!dev || !dev->workspace) return fail(MCDC_EINVAL, "device workspace missing");
    if (((uintptr_t)dev->workspace & 255u) != 0) return fail(MCDC_EINVAL, "workspace must be 256-byte aligned");
    if (max_particles < 1 || max_particles > 1000000000ull) return fail(MCDC_EINVAL, "max_particles");
    if (dev->schedule < 0 || dev->schedule > 2) return fail(MCDC_EINVAL, "schedule must be 0, 1 or 2");
    uint64_t cap = capacity_for(max_particles);
    Layout L;
    carve(L, dev->workspace, g, m, x, t, cap);
    if (L.bytes > dev->workspace_bytes) return fail(MCDC_ENOMEM, "workspace too small: need %llu bytes, have %llu", (unsigned long long)L.bytes, (unsigned long long)dev->workspace_bytes);
    CUDA_OK(cudaSetDevice(dev->device));
    cudaStream_t st = (cudaStream_t)dev->stream;

    mcdc_problem *p = new mcdc_problem();
    memset(&p->ctx, 0, sizeof(Ctx));
    p->mode = x ? 1 : 0;
    p->stream = st;
    p->device = dev->device;
    p->schedule = dev->schedule;
    p->persist = dev->persist_threshold == 0 ? (x ? DEFAULT_PERSIST_CE : DEFAULT_PERSIST) : dev->persist_threshold;
    p->cap = cap;
    Ctx &c = p->ctx;
    c.mode = p->mode;

    // ---- geometry
    int nref = g->cell_surf_off[g->n_cell];
    int nlat = g->has_lattice ? g->lat_nx * g->lat_ny : 0;
    Geo &G = c.geo;
    G.n_lat2 = g->n_lat2;
    G.l2_nx = L.l2_nx; G.l2_ny = L.l2_ny; G.l2_off = L.l2_off; G.l2_px = L.l2_px; G.l2_py = L.l2_py;
    G.l2_univ = L.l2_univ; G.l2_bin = L.l2_bin; G.umid = L.umid; G.l2_info = L.l2_info;
    G.n_surf = g->n_surf; G.n_cell = g->n_cell; G.n_univ = g->n_univ; G.has_lat = g->has_lattice;
    G.lat_nx = g->has_lattice ? g->lat_nx : 1; G.lat_ny = g->has_lattice ? g->lat_ny : 1;
    G.lat_x0 = g->lat_x0; G.lat_y0 = g->lat_y0; G.lat_px = g->lat_px; G.lat_py = g->lat_py;
    G.lat_cell = -1;
    G.lat_magic = G.lat_nx > 1 ? (unsigned int)(0x100000000ull / (unsigned long long)G.lat_nx) + 1u : 0u;
    for (int cc = 0; cc < g->n_cell; cc++) if (g->cell_fill_type[cc] == 1) G.lat_cell = cc;
    G.surf_type = L.surf_type; G.surf_bc = L.surf_bc; G.surf_param = L.surf_param;
    G.cso = L.cso; G.csi = L.csi; G.css = L.css; G.cft = L.cft; G.cfill = L.cfill; G.cbin = L.cbin; G.uco = L.uco;
    G.lat_info = L.lat_info; G.cell_info = L.cell_info; G.lat_rmask = L.lat_rmask; G.ufast = L.ufast;
    G.ap_pos = L.ap_pos; G.ap_sid = L.ap_sid;
    // host staging must outlive the async copies: keep vectors until the sync at the end
    std::vector<double> h_mg, h_tab, h_colA, h_ap_pos, h_cum_nu, h_cumchi_d;
    std::vector<int> h_ncol, h_hash, h_ehash, h_cfill(g->cell_fill, g->cell_fill + g->n_cell), h_ap_sid;
    std::vector<int4> h_ufast, h_latinfo(nlat), h_cellinfo(g->n_cell), h_l2info;
    std::vector<unsigned int> h_rmask(nlat);
    for (int cc = 0; cc < g->n_cell; cc++) if (g->cell_fill_type[cc] == 1) h_cfill[cc] = 0;
    std::vector<int> h_umid(g->n_univ, -1);
    for (int u = 1; u < g->n_univ; u++)
        for (int cc = g->univ_cell_off[u]; cc < g->univ_cell_off[u + 1]; cc++)
            if (g->cell_fill_type[cc] == 2) h_umid[u] = cc;
    cudaError_t e = cudaSuccess;
#define UP(dst, src, n) do { if (e == cudaSuccess) e = up(dst, src, (uint64_t)(n), st); } while (0)
    UP(L.surf_type, g->surf_type, g->n_surf); UP(L.surf_bc, g->surf_bc, g->n_surf);
    UP(L.surf_param, g->surf_param, 4 * g->n_surf);
    UP(L.cso, g->cell_surf_off, g->n_cell + 1); UP(L.csi, g->cell_surf_id, nref); UP(L.css, g->cell_surf_sense, nref);
    UP(L.cft, g->cell_fill_type, g->n_cell); UP(L.cfill, h_cfill.data(), g->n_cell); UP(L.cbin, t->cell_bin, g->n_cell);
    UP(L.uco, g->univ_cell_off, g->n_univ + 1);
    UP(L.umid, h_umid.data(), g->n_univ);
    if (g->n_lat2 > 0) {
        int ne2 = g->lat2_off[g->n_lat2];
        UP(L.l2_nx, g->lat2_nx, g->n_lat2); UP(L.l2_ny, g->lat2_ny, g->n_lat2); UP(L.l2_off, g->lat2_off, g->n_lat2 + 1);
        UP(L.l2_px, g->lat2_px, g->n_lat2); UP(L.l2_py, g->lat2_py, g->n_lat2);
        UP(L.l2_univ, g->lat2_univ, ne2); UP(L.l2_bin, t->lat2_bin, ne2);
    }
    classify_universes(g, h_ufast);
    {   // bit 1: the universe's cylinder lies strictly inside the smallest lattice element of the problem (with a margin far
        // above rounding), so a particle that enters the element through a wall is outside the cylinder
        double hx = 1e300, hy = 1e300;
        if (g->has_lattice) { hx = 0.5 * g->lat_px; hy = 0.5 * g->lat_py; }
        for (int k = 0; k < g->n_lat2; k++) { hx = std::min(hx, 0.5 * g->lat2_px[k]); hy = std::min(hy, 0.5 * g->lat2_py[k]); }
        for (int u = 1; u < g->n_univ; u++) {
            int cyl = h_ufast[u].y;
            if (!h_ufast[u].x || cyl < 0) continue;
            const double *q = g->surf_param + 4 * cyl;
            if (std::fabs(q[0]) + q[2] < hx * (1.0 - 1e-6) && std::fabs(q[1]) + q[2] < hy * (1.0 - 1e-6)) h_ufast[u].x |= 2;
        }
    }
    UP(L.ufast, h_ufast.data(), g->n_univ);
    // every axis plane of the problem gets an index the boundary codes can name (the first MAX_AXIS_PLANES of them)
    std::vector<int> ap_of(g->n_surf, -1);
    for (int sidx = 0; sidx < g->n_surf; sidx++)
        if (g->surf_type[sidx] <= MCDC_PLANE_Z && (int)h_ap_pos.size() < MAX_AXIS_PLANES) {
            ap_of[sidx] = (int)h_ap_pos.size();
            h_ap_pos.push_back(g->surf_param[4 * sidx]);
            h_ap_sid.push_back(sidx);
        }
    G.n_ap = (int)h_ap_pos.size();
    UP(L.ap_pos, h_ap_pos.data(), h_ap_pos.size()); UP(L.ap_sid, h_ap_sid.data(), h_ap_sid.size());
    // cells outside a lattice: the straight-line path applies when the cell is bounded by axis planes (one per
    // direction at most) and at most one z-cylinder; the cell across that cylinder is known when exactly one other
    // cell of the universe lists the cylinder with the opposite sense
    for (int cc = 0; cc < g->n_cell; cc++) {
        int code[6] = {0, 0, 0, 0, 0, 0}, cyl = -1, cyl_sense = 0;
        bool fast = g->cell_fill_type[cc] == 0;
        for (int k = g->cell_surf_off[cc]; k < g->cell_surf_off[cc + 1] && fast; k++) {
            int sidx = g->cell_surf_id[k], sense = g->cell_surf_sense[k], typ = g->surf_type[sidx];
            if (typ <= MCDC_PLANE_Z) {
                int slot = 2 * typ + (sense > 0 ? 0 : 1);
                if (ap_of[sidx] < 0 || code[slot] != 0) fast = false;
                else code[slot] = 2 + ap_of[sidx];
            } else if (typ == MCDC_CYL_Z && cyl < 0) { cyl = sidx; cyl_sense = sense; }
            else fast = false;
        }
        int nb = CELL_NO_NEIGHBOUR;
        if (fast && cyl >= 0) {
            int u = 0;
            while (cc >= g->univ_cell_off[u + 1]) u++;
            int found = 0;
            for (int c2 = g->univ_cell_off[u]; c2 < g->univ_cell_off[u + 1]; c2++)
                for (int k = g->cell_surf_off[c2]; k < g->cell_surf_off[c2 + 1]; k++)
                    if (c2 != cc && g->cell_surf_id[k] == cyl && g->cell_surf_sense[k] == -cyl_sense) { nb = c2; found++; }
            if (found != 1 || g->cell_fill_type[nb] != 0) nb = CELL_NO_NEIGHBOUR;
        }
        h_cellinfo[cc] = make_int4((fast ? CELL_FAST : 0) | nb, fast ? cyl : -1, code[0] | (code[1] << 8) | (code[2] << 16) | (code[3] << 24),
                                   code[4] | (code[5] << 8));
    }
    UP(L.cell_info, h_cellinfo.data(), g->n_cell);
    // Per lattice element: which of the enclosing cell's surfaces must be tested from inside it (bit mask over the
    // cell's surface list).  A surface is dropped only where it is provably never the nearest candidate: an axis
    // plane x = p (y = p) lying strictly beyond a wall of the element that is itself an event (an interior lattice
    // wall, R14) -- the ray crosses that wall first.  Any other surface type, and planes beyond an outermost
    // (non-event) wall, stay in the mask.  Then the boundary codes of the straight-line path: per direction either
    // the lattice wall (an event) or ONE needed axis plane of the enclosing cell; an element whose needed surfaces
    // do not fit this pattern, or whose universe is not of the simple shape, keeps the generic path.
    if (nlat) {
        int lc = G.lat_cell;
        int k0 = g->cell_surf_off[lc], nroot = g->cell_surf_off[lc + 1] - k0;
        for (int iy = 0; iy < g->lat_ny; iy++)
            for (int ix = 0; ix < g->lat_nx; ix++) {
                unsigned int mask = 0u;
                double xlo = g->lat_x0 + ix * g->lat_px, xhi = g->lat_x0 + (ix + 1) * g->lat_px;
                double ylo = g->lat_y0 + iy * g->lat_py, yhi = g->lat_y0 + (iy + 1) * g->lat_py;
                double tx = 1e-9 * g->lat_px, ty = 1e-9 * g->lat_py;
                // codes: slots 0..5 = -x,+x,-y,+y,-z,+z; walls that are events first
                int code[6] = {ix > 0 ? 1 : 0, ix + 1 < g->lat_nx ? 1 : 0, iy > 0 ? 1 : 0, iy + 1 < g->lat_ny ? 1 : 0, 0, 0};
                bool fast = nroot <= 32;
                for (int j = 0; j < nroot; j++) {
                    int sidx = g->cell_surf_id[k0 + j], sense = g->cell_surf_sense[k0 + j];
                    double pp = g->surf_param[4 * sidx];
                    int typ = g->surf_type[sidx];
                    bool need = true;
                    if (typ == MCDC_PLANE_X)
                        need = !((pp > xhi + tx && ix + 1 < g->lat_nx) || (pp < xlo - tx && ix > 0));
                    else if (typ == MCDC_PLANE_Y)
                        need = !((pp > yhi + ty && iy + 1 < g->lat_ny) || (pp < ylo - ty && iy > 0));
                    if (j >= 32) { if (need) mask |= 0x80000000u; }  // past the 32nd surface: always tested
                    else if (need) mask |= 1u << j;
                    if (!need) continue;
                    if (typ > MCDC_PLANE_Z || ap_of[sidx] < 0) { fast = false; continue; }
                    // the cell lies on the `sense` side of the plane: it bounds the flight in the opposite direction
                    int slot = 2 * typ + (sense > 0 ? 0 : 1);
                    if (code[slot] != 0) fast = false;  // a lattice wall or another plane already bounds that direction
                    else code[slot] = 2 + ap_of[sidx];
                }
                int e_ = iy * g->lat_nx + ix;
                int u = g->lat_univ[e_];
                // two-level straight-line path: the universe is one cell without surfaces that lattice k2 fills
                int k2 = -1;
                if (fast && g->n_lat2 > 0 && g->univ_cell_off[u + 1] - g->univ_cell_off[u] == 1) {
                    int cc = g->univ_cell_off[u];
                    if (g->cell_fill_type[cc] == 2 && g->cell_surf_off[cc + 1] == g->cell_surf_off[cc] && g->cell_fill[cc] < 65536) k2 = g->cell_fill[cc];
                }
                if (!h_ufast[u].x) fast = false;
                h_rmask[e_] = mask;
                h_latinfo[e_] = make_int4(u | (fast ? LAT_FAST : 0) | (k2 >= 0 ? LAT_FAST2 : 0), t->lat_bin[e_],
                                          code[0] | (code[1] << 8) | (code[2] << 16) | (code[3] << 24),
                                          code[4] | (code[5] << 8) | ((k2 >= 0 ? k2 : h_ufast[u].y + 1) << 16));
            }
        UP(L.lat_info, h_latinfo.data(), nlat); UP(L.lat_rmask, h_rmask.data(), nlat);
    }
    if (g->n_lat2 > 0) {  // per second-level element: universe (| LAT_FAST if simple), bin offset, wall / rim codes
        h_l2info.resize(g->lat2_off[g->n_lat2]);
        for (int k = 0; k < g->n_lat2; k++)
            for (int jy = 0; jy < g->lat2_ny[k]; jy++)
                for (int jx = 0; jx < g->lat2_nx[k]; jx++) {
                    int i = g->lat2_off[k] + jy * g->lat2_nx[k] + jx, u = g->lat2_univ[i];
                    int cd[4] = {jx > 0 ? 1 : 3, jx + 1 < g->lat2_nx[k] ? 1 : 3, jy > 0 ? 1 : 3, jy + 1 < g->lat2_ny[k] ? 1 : 3};
                    h_l2info[i] = make_int4(u | (h_ufast[u].x ? LAT_FAST : 0), t->lat2_bin[i], cd[0] | (cd[1] << 8) | (cd[2] << 16) | (cd[3] << 24), 0);
                }
        UP(L.l2_info, h_l2info.data(), h_l2info.size());
    }

    // ---- cross sections: derived tables built here, in plain left-to-right float64 sums
    if (m) {
        int Gn = m->G, nm = m->n_mat;
        size_t mg = (size_t)nm * Gn;
        MGTab &T = c.mg;
        T.G = Gn; T.n_mat = nm; T.blob = L.mg_blob; T.blob_doubles = (int)L.mg_doubles;
        T.o_sig_t = 0; T.o_sig_s = (int)mg; T.o_sig_f = (int)(2 * mg); T.o_nu = (int)(3 * mg); T.o_nusf = (int)(4 * mg);
        T.o_cumchi = (int)(5 * mg); T.o_cumS = (int)(6 * mg); T.o_src_cum = (int)(6 * mg + mg * Gn);
        T.o_inv_t = (int)(6 * mg + mg * Gn + Gn);
        T.half = 0;
        while (2 * std::max(T.half, 1) <= Gn - 1 || (T.half == 0 && Gn - 1 >= 1)) T.half = T.half ? 2 * T.half : 1;
        h_mg.assign(L.mg_doubles, 0.0);
        for (int mm = 0; mm < nm; mm++) {
            double cc = 0.0;
            for (int gg = 0; gg < Gn; gg++) {
                double cs = 0.0;
                for (int gp = 0; gp < Gn; gp++) {
                    cs += m->S[((size_t)mm * Gn + gg) * Gn + gp];
                    h_mg[T.o_cumS + ((size_t)mm * Gn + gg) * Gn + gp] = cs;
                }
                int i = mm * Gn + gg;
                h_mg[T.o_sig_t + i] = m->sig_t[i]; h_mg[T.o_sig_f + i] = m->sig_f[i]; h_mg[T.o_nu + i] = m->nu[i];
                h_mg[T.o_sig_s + i] = cs;
                cc += m->chi[i];
                h_mg[T.o_cumchi + i] = cc;
                h_mg[T.o_nusf + i] = m->nu[i] * m->sig_f[i];
                h_mg[T.o_inv_t + i] = 1.0 / m->sig_t[i];
            }
        }
        double cs = 0.0;
        for (int gg = 0; gg < Gn; gg++) { cs += s->group_pdf[gg]; h_mg[T.o_src_cum + gg] = cs; }
        if (!(cs > 0.0)) { delete p; return fail(MCDC_EINVAL, "source group pdf sums to zero"); }
        UP(L.mg_blob, h_mg.data(), h_mg.size());
        c.mg_stage = L.mg_doubles * 8 <= MG_STAGE_MAX_BYTES ? (int)L.mg_doubles : 0;
        c.n_tally = t->n_bins * Gn;
        if (m->kinetics) {  // time-dependent multi-group: cumulative yields / delayed spectra, plain left-to-right sums
            const mcdc_kinetics *kn = m->kinetics;
            const int J = kn->n_dgroup;
            h_cum_nu.assign(mg * (J + 1), 0.0);
            h_cumchi_d.assign((size_t)nm * J * Gn + 1, 0.0);
            for (int mm = 0; mm < nm; mm++) {
                for (int j = 0; j < J; j++) {
                    double cc = 0.0;
                    for (int gg = 0; gg < Gn; gg++) { cc += kn->chi_d[((size_t)mm * J + j) * Gn + gg]; h_cumchi_d[((size_t)mm * J + j) * Gn + gg] = cc; }
                }
                for (int gg = 0; gg < Gn; gg++) {
                    double cn = m->nu[mm * Gn + gg];
                    h_cum_nu[((size_t)mm * Gn + gg) * (J + 1)] = cn;
                    for (int j = 0; j < J; j++) { cn += kn->nu_d[((size_t)mm * J + j) * Gn + gg]; h_cum_nu[((size_t)mm * Gn + gg) * (J + 1) + 1 + j] = cn; }
                }
            }
            UP(L.td_speed, kn->speed, Gn); UP(L.td_cum_nu, h_cum_nu.data(), h_cum_nu.size());
            UP(L.td_cumchi_d, h_cumchi_d.data(), (size_t)nm * J * Gn); UP(L.td_decay, kn->decay, (size_t)nm * J);
            UP(L.t_edges, t->t_edges, t->n_t + 1);
            c.td.on = 1; c.td.J = J; c.td.speed = L.td_speed; c.td.cum_nu = L.td_cum_nu; c.td.cumchi_d = L.td_cumchi_d; c.td.decay = L.td_decay;
            c.ce.n_t = t->n_t; c.ce.t_edges = L.t_edges;
            c.n_tally = t->n_bins * t->n_t * Gn;
            if (dev->schedule != 0 || dev->persist_threshold < 0) { delete p; return fail(MCDC_EINVAL, "time-dependent multi-group runs use the default schedule (persistent kernel) only"); }
            if ((uint64_t)kn->census_target > cap) { delete p; return fail(MCDC_EINVAL, "census_target exceeds the bank capacity"); }
        }
    } else {
        int ng = x->n_grid, nm = x->n_mat;
        h_tab.assign((size_t)nm * ng * CE_ROW, 0.0); h_colA.assign((size_t)nm * CE_ROW, 1.0); h_ncol.assign(nm, 0);
        for (int mm = 0; mm < nm; mm++) {
            int n0 = x->mat_nuc_off[mm], nn = x->mat_nuc_off[mm + 1] - n0;
            h_ncol[mm] = nn + 2;
            for (int j = 0; j < nn; j++) h_colA[mm * CE_ROW + j] = x->nuc_A[x->mat_nuc_id[n0 + j]];
            for (int i = 0; i < ng; i++) {
                double *row = &h_tab[((size_t)mm * ng + i) * CE_ROW];
                double cum = 0.0, sf = 0.0, sc = 0.0;
                for (int j = 0; j < nn; j++) {
                    int nuc = x->mat_nuc_id[n0 + j];
                    double dens = x->mat_nuc_dens[n0 + j];
                    cum += dens * x->nuc_el[(size_t)nuc * ng + i];
                    row[j] = cum;
                    sf += dens * x->nuc_f[(size_t)nuc * ng + i];
                    sc += dens * x->nuc_c[(size_t)nuc * ng + i];
                }
                cum += sf; row[nn] = cum;
                cum += sc; row[nn + 1] = cum;
                for (int j = nn + 2; j < MAX_CE_COL; j++) row[j] = cum;
                row[6] = x->grid[i];
                row[7] = sf;
                if (!(cum > 0.0)) { delete p; return fail(MCDC_EINVAL, "material %d has zero total cross section at grid point %d", mm, i); }
            }
        }
        int sh, lo, nh;
        hash_params(x->grid, ng, sh, lo, nh);
        h_hash.assign(nh + 2, 0);
        for (int b = 0; b <= nh; b++) {
            long long bits = ((long long)(lo + b)) << sh;
            double edge;
            memcpy(&edge, &bits, 8);
            // last grid index <= lower edge of bucket b (0 if the edge lies below the grid)
            int idx = (int)(std::upper_bound(x->grid, x->grid + ng, edge) - x->grid) - 1;
            h_hash[b] = idx < 0 ? 0 : idx;
        }
        h_hash[nh + 1] = ng - 1;
        // the same for the tally's energy-bin edges
        {
            long long klo;
            memcpy(&klo, &t->e_edges[0], 8);
            int elo = (int)(klo >> EHASH_SHIFT), neh = ehash_buckets(t->e_edges, t->n_e);
            h_ehash.assign(neh + 2, 0);
            for (int b = 0; b <= neh; b++) {
                long long bits = ((long long)(elo + b)) << EHASH_SHIFT;
                double edge;
                memcpy(&edge, &bits, 8);
                int idx = (int)(std::upper_bound(t->e_edges, t->e_edges + t->n_e + 1, edge) - t->e_edges) - 1;
                h_ehash[b] = idx < 0 ? 0 : idx;
            }
            h_ehash[neh + 1] = t->n_e;
            c.ce.ehash = L.ehash; c.ce.ehash_shift = EHASH_SHIFT; c.ce.ehash_lo = elo; c.ce.n_ehash = neh;
            UP(L.ehash, h_ehash.data(), neh + 2);
        }
        UP(L.grid, x->grid, ng); UP(L.tab, h_tab.data(), h_tab.size()); UP(L.colA, h_colA.data(), h_colA.size());
        UP(L.ncol, h_ncol.data(), nm); UP(L.hash, h_hash.data(), nh + 2);
        UP(L.t_edges, t->t_edges, t->n_t + 1); UP(L.e_edges, t->e_edges, t->n_e + 1);
        CETab &ce = c.ce;
        ce.n_grid = ng; ce.n_mat = nm; ce.n_t = t->n_t; ce.n_e = t->n_e; ce.search = x->search;
        ce.grid = L.grid; ce.tab = L.tab; ce.ncol = L.ncol; ce.colA = L.colA; ce.t_edges = L.t_edges; ce.e_edges = L.e_edges;
        ce.hash = L.hash; ce.hash_shift = sh; ce.hash_lo = lo; ce.n_hash = nh;
        ce.nu0 = x->nu0; ce.nu1 = x->nu1; ce.watt_a = x->watt_a; ce.watt_b = x->watt_b;
        ce.E_min = x->grid[0]; ce.E_max = x->grid[ng - 1];
        c.n_tally = t->n_bins * t->n_t * t->n_e;
    }
    c.n_bins = t->n_bins;
    for (int b = 0; b < 2; b++) { c.bank[b] = L.bank[b]; p->cb[b] = L.cb[b]; p->sort_key[b] = L.sort_key[b]; p->sort_idx[b] = L.sort_idx[b]; }
    p->sort_hist = L.sort_hist; p->comb_copies = L.comb_copies; p->comb_offs = L.comb_offs; p->comb_w = L.comb_w;
    p->td = m && m->kinetics; p->timed = x || p->td;
    p->census_target = p->td ? (long long)m->kinetics->census_target : 0;
    p->first_interval = 0;
    if (p->timed) {
        while (p->first_interval + 1 < t->n_t && s->t >= t->t_edges[p->first_interval + 1]) p->first_interval++;
        if (p->td) p->persist = 0x7fffffff;  // one persistent launch per census interval
    }
    p->cb_cur = 0; p->census_n = 0;
    c.cbank = L.cb[0]; c.census_stop = 0;
    c.fis = L.fis;
    c.work = L.work;
    c.cap = (unsigned int)cap;
    c.qc = L.qc; c.flux = L.flux; c.scal = L.scal; c.counters = L.counters; c.err = L.err;
    c.tr.rec = nullptr;
    c.tr_g = L.tr_g;
    if (e == cudaSuccess) e = cudaMemcpyAsync(L.tr_g, &c.tr, sizeof(Trace), cudaMemcpyHostToDevice, st);
    for (int k = 0; k < 3; k++) { c.src_lo[k] = s->lo[k]; c.src_hi[k] = s->hi[k]; c.src_dir[k] = s->dir[k]; }
    c.src_iso = s->isotropic; c.src_E = s->E; c.src_t = s->t;
    c.w0 = 1.0; c.k_prev = 1.0;
    c.max_secondaries = ~0ull;
    for (int k = 0; k < 2; k++) { p->flux_acc[k] = L.flux_acc[k]; p->flux_acc2[k] = L.flux_acc2[k]; }
    p->flux_cycle = L.flux_cycle;
    p->flux_copies = flux_copies_for((uint64_t)c.n_tally);
    c.flux_copy_mask = p->flux_copies - 1;
    p->part = L.part; p->sites = L.sites;
    p->trace_base = L.trace; p->trace_count = L.trace_count;
    p->tally_private = c.n_tally <= PRIVATE_TALLY_MAX && !p->td && g->n_lat2 == 0;  // those variants exist with the global tally only
    if (p->tally_private && (size_t)c.mg_stage * 8 + (size_t)c.n_tally * BS * 8 > 48 * 1024)
        c.mg_stage = 0;  // 48 KB default dynamic shared memory limit
    c.flux_aggregate = c.n_tally <= AGGREGATE_TALLY_MAX ? 1 : 0;
    if (e == cudaSuccess) e = cudaMemsetAsync(L.flux, 0, sizeof(double) * c.n_tally * p->flux_copies, st);
    for (int k = 0; k < 2 && e == cudaSuccess; k++) {
        e = cudaMemsetAsync(L.flux_acc[k], 0, sizeof(double) * c.n_tally, st);
        if (e == cudaSuccess) e = cudaMemsetAsync(L.flux_acc2[k], 0, sizeof(double) * c.n_tally, st);
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(L.scal, 0, 64, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.counters, 0, 8 * MCDC_N_COUNTERS, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.err, 0, 16, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.work, 0, 32, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.qc, 0, sizeof(QCount) * RING, st);
    if (e == cudaSuccess) e = cudaMallocHost((void **)&p->pin, sizeof(HostPinned));
    for (int k = 0; k < RING && e == cudaSuccess; k++) e = cudaEventCreateWithFlags(&p->ev[k], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreate(&p->t0);
    if (e == cudaSuccess) e = cudaEventCreate(&p->t1);
    // the source box must lie inside the geometry: every point of a 9 x 9 x 9 grid over it has to be in a cell
    int src_err = 0;
    if (e == cudaSuccess) {
        const int n1 = 9;
        k_check_source_box<<<(n1 * n1 * n1 + 255) / 256, 256, 0, st>>>(c, n1);
        e = cudaMemcpyAsync(&src_err, L.err, sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemsetAsync(L.err, 0, 16, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) { mcdc_destroy(p); return fail(MCDC_ECUDA, "mcdc_create: %s", cudaGetErrorString(e)); }
    if (src_err) { mcdc_destroy(p); return fail(MCDC_EGEOM, "the source box is not inside the geometry (a point of it lies in no cell)"); }
    p->bank_count = 0; p->k_prev = 1.0;
    p->dirty = false;
    p->ms_transport = 0.0; p->n_launches = 0; p->last_N = 0;
    p->profile = 0;
    memset(p->prof_ms, 0, sizeof p->prof_ms); memset(p->prof_launches, 0, sizeof p->prof_launches);
    *out = p;
    return 0;
}

extern "C" void mcdc_destroy(mcdc_problem *p)
{
    if (!p) return;
    cudaStreamSynchronize(p->stream);
    for (int k = 0; k < RING; k++) if (p->ev[k]) cudaEventDestroy(p->ev[k]);
    for (cudaEvent_t e : p->pool) cudaEventDestroy(e);
    if (p->t0) cudaEventDestroy(p->t0);
    if (p->t1) cudaEventDestroy(p->t1);
    if (p->pin) cudaFreeHost(p->pin);
    delete p;
}

extern "C" const char *mcdc_last_error(void) { return g_err.c_str(); }

#ifndef MCDC_BUILD_ID
#define MCDC_BUILD_ID "unknown"
#endif
extern "C" const char *mcdc_build_id(void) { return MCDC_BUILD_ID; }

// ------------------------------------------------------------------ drivers
#ifndef MCDC_GRID_PER_SM
#define MCDC_GRID_PER_SM 16ull  // measured (ms per C4 cycle): 4 -> 42.9, 8 -> 41.5, 16 -> 40.9, 64 -> 42.3, 1024 -> 45.1
#endif
static unsigned int grid_for(uint64_t n)
{
    uint64_t b = (n + BS - 1) / BS;
    const uint64_t cap = 148ull * MCDC_GRID_PER_SM * 256 / BS;  // persistent-style: at most MCDC_GRID_PER_SM x 256 threads' worth per SM
    return (unsigned int)std::max<uint64_t>(1, std::min(b, cap));
}

// the persistent kernel: at most the blocks that are resident at once (its idle warps wait for other warps' pushes,
// so every block of the grid must be running)
template <bool CE, bool PRIV, bool W, int X> static unsigned int grid_persist(mcdc_problem *p, uint64_t n, size_t smem)
{
    if (p->persist_blocks_per_sm == 0) {
        int nb = 0, sms = 148;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_persist<CE, PRIV, W, X>, BS, smem) != cudaSuccess || nb < 1) nb = 1;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device);
        p->persist_blocks_per_sm = nb;
        p->n_sm = sms;
    }
    uint64_t b = (n + BS - 1) / BS;
    const uint64_t cap = (uint64_t)p->n_sm * p->persist_blocks_per_sm;
    return (unsigned int)std::max<uint64_t>(1, std::min(b, cap));
}

// start a new run in the accumulator set the published results do not use
static int begin_run(mcdc_problem *p)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    p->work = RunStats();
    p->work.set = 1 - p->pub.set;
    CUDA_OK(cudaMemsetAsync(c.flux, 0, sizeof(double) * c.n_tally * p->flux_copies, st));
    CUDA_OK(cudaMemsetAsync(p->flux_acc[p->work.set], 0, sizeof(double) * c.n_tally, st));
    CUDA_OK(cudaMemsetAsync(p->flux_acc2[p->work.set], 0, sizeof(double) * c.n_tally, st));
    CUDA_OK(cudaMemsetAsync(c.counters, 0, 8 * MCDC_N_COUNTERS, st));
    CUDA_OK(cudaMemsetAsync(c.err, 0, 16, st));
    CUDA_OK(cudaMemsetAsync(c.fis.n, 0, sizeof(int) * (size_t)p->cap, st));
    if (c.tr.rec) CUDA_OK(cudaMemsetAsync(c.tr.count, 0, sizeof(unsigned int) * c.tr.cap_slots, st));
    p->k_prev = 1.0;
    p->bank_count = 0;
    p->ms_transport = 0.0;
    p->n_launches = 0;
    p->dirty = false;
    return 0;
}

// the call succeeded: what it computed becomes the reported state
static void publish(mcdc_problem *p)
{
    RunStats &w = p->work;
    for (int i = 0; i < MCDC_N_COUNTERS; i++) w.counters[i] = p->pin->counters[i];
    // histories started / children made: source-bank histories are counted on the host, secondaries that joined the
    // running population (continuous energy) on the device (counter 15)
    w.counters[0] = w.host_counters[0] + p->pin->counters[15];
    w.counters[11] = w.host_counters[11] + p->pin->counters[15];
    w.counters[12] = w.host_counters[12];
    w.counters[13] = w.host_counters[13];
    w.counters[15] = 0;
    p->pub = w;
}

static int device_error_code(mcdc_problem *p, int e)
{
    if (e == -2) return fail(MCDC_EGEOM, "particle in no cell (lost)");
    if (e == -3) return fail(MCDC_EBANK, "fission / secondary bank overflow (capacity %llu)", (unsigned long long)p->cap);
    if (e == -4) return fail(MCDC_ELOST, "segment guard exceeded (%u segments in one history)", MAX_SEGMENTS);
    if (e != 0) return fail(MCDC_ECUDA, "device error flag %d", e);
    return 0;
}

template <bool CE, bool PRIV, bool W, int X> static int transport_t(mcdc_problem *p, uint64_t M)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    const size_t smem_mg = CE ? 0 : (size_t)c.mg_stage * sizeof(double);
    const size_t smem = smem_mg + (PRIV ? (size_t)c.n_tally * BS * sizeof(double) : 0);
    CUDA_OK(cudaMemsetAsync(c.qc, 0, sizeof(QCount) * RING, st));
    uint64_t upper = M;
    long long known = -1;  // newest sweep whose counts the host has seen
    unsigned int s = 0;
    const unsigned int n0 = (unsigned int)M;
    while (upper > 0) {
        if (s > 4000000u) return fail(MCDC_ELOST, "sweep guard exceeded");
        if (p->schedule != 1 && p->persist > 0 && upper <= (uint64_t)p->persist) {
            CUDA_OK(cudaMemsetAsync(c.work, 0, 16, st));  // head, pushed, ended, born; work[4] (census count) is kept
            if (CE) CUDA_OK(cudaMemsetAsync(c.bank[(s + 1) & 1].ev, 0, sizeof(uint32_t) * (size_t)p->cap, st));
            { ProfScope ps(p, MCDC_PROF_PERSIST); k_persist<CE, PRIV, W, X><<<grid_persist<CE, PRIV, W, X>(p, upper, smem), BS, smem, st>>>(c, s, n0); }
            p->n_launches++;
            p->work.host_counters[13]++;
            break;
        }
        unsigned int gr = grid_for(upper);
        if (p->schedule != 1) {
            { ProfScope ps(p, MCDC_PROF_SWEEP); k_sweep<CE, PRIV, W, X><<<gr, BS, smem, st>>>(c, s, n0); }
            p->n_launches++;
            if (p->schedule == 2) {
                { ProfScope ps(p, MCDC_PROF_SCATTER); k_scatter<CE><<<gr, BS, smem_mg, st>>>(c, s); }
                { ProfScope ps(p, MCDC_PROF_SURFACE); k_surface<<<gr, BS, 0, st>>>(c, s); }
                p->n_launches += 2;
            }
        } else {
            { ProfScope ps(p, MCDC_PROF_SEGMENT); k_segment<CE, PRIV, W, X><<<grid_for(M), BS, smem, st>>>(c, s, n0); }
            p->n_launches++;
        }
        p->work.host_counters[13]++;
        CUDA_OK(cudaMemcpyAsync(&p->pin->qc[s % RING], c.qc + (s % RING), sizeof(QCount), cudaMemcpyDeviceToHost, st));
        CUDA_OK(cudaEventRecord(p->ev[s % RING], st));
        s++;
        bool stop = false;
        while (known < (long long)s - 1) {
            long long r = known + 1;
            if ((long long)s - 1 - r >= LAG) CUDA_OK(cudaEventSynchronize(p->ev[r % RING]));
            else {
                cudaError_t q = cudaEventQuery(p->ev[r % RING]);
                if (q == cudaErrorNotReady) break;
                if (q != cudaSuccess) return fail(MCDC_ECUDA, "event query: %s", cudaGetErrorString(q));
            }
            const QCount &h = p->pin->qc[r % RING];
            upper = p->schedule != 1 ? (uint64_t)h.n_scat + h.n_surf : (uint64_t)h.n_alive;
            if (h.err != 0) stop = true;  // a kernel raised the device error flag: the caller reads and reports it
            known = r;
        }
        if (stop) break;
    }
    CUDA_OK(cudaGetLastError());
    return 0;
}

// time-dependent multi-group: persistent kernel only (the host never launches anything else for it), weighted, global
// tally; the sweep / monolithic branches of transport_t are dead code for it
template <int X> static int transport_td(mcdc_problem *p, uint64_t M)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    const size_t smem = (size_t)c.mg_stage * sizeof(double);
    CUDA_OK(cudaMemsetAsync(c.qc, 0, sizeof(QCount) * RING, st));
    CUDA_OK(cudaMemsetAsync(c.work, 0, 16, st));  // head, pushed, ended, born; work[4] (census count) is kept
    CUDA_OK(cudaMemsetAsync(c.bank[1].ev, 0, sizeof(uint32_t) * (size_t)p->cap, st));
    { ProfScope ps(p, MCDC_PROF_PERSIST); k_persist<false, false, true, X><<<grid_persist<false, false, true, X>(p, M, smem), BS, smem, st>>>(c, 0u, (unsigned int)M); }
    p->n_launches++;
    p->work.host_counters[13]++;
    CUDA_OK(cudaGetLastError());
    return 0;
}

static int transport(mcdc_problem *p, uint64_t M)
{
    const bool W = p->ctx.implicit != 0, priv = p->tally_private;
    if (p->td) return p->ctx.geo.n_lat2 ? transport_td<X_TD | X_L2>(p, M) : transport_td<X_TD>(p, M);
    if (p->ctx.geo.n_lat2) {  // second-level lattices (R37): generic-geometry variants, global tally
        if (p->mode == 0) return W ? transport_t<false, false, true, X_L2>(p, M) : transport_t<false, false, false, X_L2>(p, M);
        return W ? transport_t<true, false, true, X_L2>(p, M) : transport_t<true, false, false, X_L2>(p, M);
    }
    if (W) {  // weighted kernels (implicit capture, R36)
        if (p->mode == 0) return priv ? transport_t<false, true, true, 0>(p, M) : transport_t<false, false, true, 0>(p, M);
        return priv ? transport_t<true, true, true, 0>(p, M) : transport_t<true, false, true, 0>(p, M);
    }
    if (p->mode == 0) return priv ? transport_t<false, true, false, 0>(p, M) : transport_t<false, false, false, 0>(p, M);
    return priv ? transport_t<true, true, false, 0>(p, M) : transport_t<true, false, false, 0>(p, M);
}

// Weight balance of the transport just finished (the scalars and counters are in pinned memory): source weight,
// absorbed, leaked, cut off, roulette loss / gain.  Analog: every ended history carried w0, so the terms follow from
// the event-counter increments; weighted: the kernels summed them (scal[2..5]).
static void add_balance(mcdc_problem *p, double source_weight, const uint64_t *before)
{
    RunStats &w = p->work;
    const double *sc = p->pin->scal;
    const unsigned long long *cn = p->pin->counters;
    w.balance[0] += source_weight;
    w.balance[2] += sc[1];
    if (p->ctx.implicit || p->td) {  // the weighted kernels ran
        w.balance[1] += sc[2]; w.balance[3] += sc[3]; w.balance[4] += sc[4]; w.balance[5] += sc[5];
    } else {
        w.balance[1] += p->ctx.w0 * (double)((cn[2] - before[2]) + (cn[3] - before[3]));
        w.balance[3] += p->ctx.w0 * (double)(cn[9] - before[9]);
    }
}

// children of the M parents' fission records -> bank[0]; returns their number.  Also brings the cycle's scalars,
// the device counters and the error flag to the host (one synchronisation).
// wait = false: everything is queued and the caller synchronises (one wait per cycle), then reads p->pin->total
static int emit_children(mcdc_problem *p, uint64_t M, uint64_t *total, bool wait = true)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    unsigned int nb = (unsigned int)((M + BS - 1) / BS);
    {
    ProfScope ps(p, MCDC_PROF_BANK);
    k_scan_partial<<<nb, BS, 0, st>>>(c, (unsigned int)M, p->part);
    k_scan_top<<<1, 1024, 0, st>>>(p->part, nb);
    if (p->mode == 0) k_emit<false><<<nb, BS, 0, st>>>(c, (unsigned int)M, p->part, (unsigned int)p->cap);
    else k_emit<true><<<nb, BS, 0, st>>>(c, (unsigned int)M, p->part, (unsigned int)p->cap);
    k_clear_counts<<<nb, BS, 0, st>>>(c, (unsigned int)M);
    }
    p->n_launches += 4;
    CUDA_OK(cudaMemcpyAsync(&p->pin->total, p->part + nb, sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaMemcpyAsync(p->pin->scal, c.scal, 6 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaMemcpyAsync(p->pin->counters, c.counters, sizeof p->pin->counters, cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaMemcpyAsync(&p->pin->err, c.err, sizeof(int), cudaMemcpyDeviceToHost, st));
    if (!wait) return 0;
    CUDA_OK(cudaStreamSynchronize(st));
    CUDA_OK(cudaGetLastError());
    profile_collect(p);
    *total = p->pin->total;
    return 0;
}

// a call failed after device work was queued: drain the stream, clear the error flag and mark the per-cycle
// tallies for clearing, so that the problem stays usable
static int abandon(mcdc_problem *p, int rc)
{
    std::string keep = g_err;
    cudaStreamSynchronize(p->stream);
    cudaMemsetAsync(p->ctx.err, 0, 16, p->stream);
    cudaMemsetAsync(p->ctx.fis.n, 0, sizeof(int) * (size_t)p->cap, p->stream);
    cudaStreamSynchronize(p->stream);
    p->dirty = true;
    p->work.next_interval = -1;  // fixed source: the next call has to name the first interval again
    g_err = keep;
    return rc;
}

// one power-iteration cycle; sample: draw the source (cycle 0) instead of starting from bank[0]
static int cycle_internal(mcdc_problem *p, uint64_t N, uint32_t cycle, int active, uint64_t seed, bool sample,
                          double *flux_cycle_host)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    if (N < 1 || capacity_for(N) > p->cap) return fail(MCDC_EINVAL, "n_particles %llu exceeds the capacity this problem was created for", (unsigned long long)N);
    if (cycle >= (1u << 24)) return fail(MCDC_EINVAL, "cycle index too large for the RNG counter layout");
    uint64_t M = sample ? N : p->bank_count;
    if (M == 0) return fail(MCDC_EBANK, "empty source bank");
    set_seed(c, seed); c.cycle = cycle;
    c.w0 = sample ? 1.0 : (double)N / (double)M;  // source renormalisation (R6)
    c.k_prev = p->k_prev;
    c.max_secondaries = ~0ull;
    if (p->dirty) {
        CUDA_OK(cudaMemsetAsync(c.flux, 0, sizeof(double) * c.n_tally * p->flux_copies, st));
        p->dirty = false;
    }
    CUDA_OK(cudaMemsetAsync(c.scal, 0, 64, st));
    CUDA_OK(cudaEventRecord(p->t0, st));
    if (sample) {
        k_source<false><<<(unsigned int)((M + BS - 1) / BS), BS, 0, st>>>(c, (unsigned int)M);
        p->n_launches++;
    }
    uint64_t before[MCDC_N_COUNTERS];
    for (int i = 0; i < MCDC_N_COUNTERS; i++) before[i] = cycle == 0 ? 0 : p->pin->counters[i];
    int rc = transport(p, M);
    if (rc) return abandon(p, rc);
    // the fission bank, the read-backs and the cycle's tally statistics are queued together: ONE wait per cycle (a
    // cycle that turns out to have failed has then added to the work accumulators, which the next run clears)
    uint64_t total = 0;
    rc = emit_children(p, M, &total, false);
    if (rc) return abandon(p, rc);
    CUDA_OK(cudaEventRecord(p->t1, st));
    k_accumulate<<<(c.n_tally + BS - 1) / BS, BS, 0, st>>>(c.flux, p->flux_copies, p->flux_cycle, p->flux_acc[p->work.set],
                                                          p->flux_acc2[p->work.set], c.n_tally, 1.0 / (double)N, active);
    if (flux_cycle_host) CUDA_OK(cudaMemcpyAsync(flux_cycle_host, p->flux_cycle, sizeof(double) * c.n_tally, cudaMemcpyDeviceToHost, st));
    p->n_launches++;
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return abandon(p, fail(MCDC_ECUDA, "cycle: %s", cudaGetErrorString(cudaGetLastError())));
    profile_collect(p);
    total = p->pin->total;
    rc = device_error_code(p, p->pin->err);
    if (rc) return abandon(p, rc);
    add_balance(p, c.w0 * (double)M, before);
    float ms = 0.f;
    CUDA_OK(cudaEventElapsedTime(&ms, p->t0, p->t1));
    p->ms_transport += ms;
    RunStats &w = p->work;
    double k_c = p->pin->scal[0] / (double)N, leak = p->pin->scal[1] / (double)N;
    w.k_cycle.push_back(k_c);
    if (active) {
        w.k_acc += k_c; w.k_acc2 += k_c * k_c;
        w.leak_acc += leak; w.leak_acc2 += leak * leak;
        w.n_active++;
    }
    p->k_prev = k_c;
    w.host_counters[0] += M;
    w.host_counters[11] += total;
    if (total > w.host_counters[12]) w.host_counters[12] = total;
    p->bank_count = total;
    p->last_N = N;
    return 0;
}

// ------------------------------------------------------------------ fixed source by census intervals (R40)
// one draw of stream (seed, id, domain, cycle) on the host: the comb's offset (same Philox4x32-10 as the device's)
static double host_draw(uint64_t seed, uint64_t id, uint32_t domain, uint32_t cycle, uint32_t index)
{
    uint32_t c0 = (uint32_t)id, c1 = (uint32_t)(id >> 32), c2 = (domain << 24) | cycle, c3 = index >> 1;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; r++) {
        uint64_t p0 = 0xD2511F53ull * c0, p1 = 0xCD9E8D57ull * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    uint64_t u = (index & 1u) ? (((uint64_t)c3 << 32) | c2) : (((uint64_t)c1 << 32) | c0);
    return ((double)(u >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

// The census bank becomes the source bank of interval k: its particles are keyed by id (those of later intervals get
// the largest key), radix-sorted, the first M -- the particles of interval k in id order -- moved to bank[0], through
// the comb if population control is on, and the rest kept in the other census bank.
template <bool CE> static int census_to_source_t(mcdc_problem *p, int k, uint64_t seed, uint64_t *M_out)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    RunStats &w = p->work;
    const unsigned int n = (unsigned int)p->census_n;
    *M_out = 0;
    if (n == 0) {
        w.census_counts.push_back(0); w.census_counts.push_back(0);
        w.census_weights.push_back(0.0); w.census_weights.push_back(0.0);
        return 0;
    }
    const Bank &S = p->cb[p->cb_cur], &KEEP = p->cb[1 - p->cb_cur];
    const unsigned int nb = (n + BS - 1) / BS, nbt = (n + RS_TILE - 1) / RS_TILE;
    CUDA_OK(cudaMemsetAsync(c.work + 5, 0, 4, st));
    k_census_keys<<<nb, BS, 0, st>>>(S, n, k, p->sort_key[0], p->sort_idx[0], c.work + 5);
    int a = 0;
    for (int pass = 0; pass < 8; pass++, a ^= 1) {
        k_rs_hist<<<nbt, BS, 0, st>>>(p->sort_key[a], n, 8 * pass, p->sort_hist);
        k_scan_top<<<1, 1024, 0, st>>>(p->sort_hist, 256u * nbt);
        k_rs_scatter<<<nbt, BS, 0, st>>>(p->sort_key[a], p->sort_idx[a], p->sort_key[1 - a], p->sort_idx[1 - a], n, 8 * pass, p->sort_hist);
    }
    p->n_launches += 25;
    CUDA_OK(cudaMemcpyAsync(&p->pin->census[1], c.work + 5, 4, cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaStreamSynchronize(st));
    const unsigned int M = p->pin->census[1];
    const unsigned int *idx = p->sort_idx[0];
    // total weight of the interval's particles (left-to-right sums in id order; the comb's running sums)
    double W = (double)M;
    const bool weighted = c.implicit || p->td;
    if (M > 0 && weighted) {
        k_comb_weights<<<(M + BS - 1) / BS, BS, 0, st>>>(S, idx, M, p->comb_w);
        k_dscan<<<1, 1024, 0, st>>>(p->comb_w, M);
        CUDA_OK(cudaMemcpyAsync(&p->pin->comb_w, p->comb_w + (M - 1), 8, cudaMemcpyDeviceToHost, st));
        CUDA_OK(cudaStreamSynchronize(st));
        W = p->pin->comb_w;
        p->n_launches += 2;
    }
    uint64_t M_run = M;
    double W_run = W;
    const bool comb = p->census_target > 0 && M > 0 && weighted;
    if (comb) {
        const unsigned int T = (unsigned int)p->census_target;
        const double xi = host_draw(seed, (uint64_t)k, 3u, 0u, 0u);  // the comb's own stream: domain 3, id = interval
        k_comb_copies<<<(M + BS - 1) / BS, BS, 0, st>>>(p->comb_w, M, T, xi, p->comb_copies);
        CUDA_OK(cudaMemcpyAsync(p->comb_offs, p->comb_copies, sizeof(unsigned int) * M, cudaMemcpyDeviceToDevice, st));
        k_scan_top<<<1, 1024, 0, st>>>(p->comb_offs, M);
        k_comb_write<CE><<<(M + BS - 1) / BS, BS, 0, st>>>(S, idx, p->comb_copies, p->comb_offs, p->comb_w, M, T, seed, k, c.bank[0]);
        p->n_launches += 3;
        M_run = T;
        W_run = W / (double)T * (double)T;
    }
    k_census_move<CE><<<nb, BS, 0, st>>>(S, idx, M, n, c.bank[0], KEEP, comb ? 0 : 1);
    p->n_launches++;
    // the kept particles are the new census bank; the interval's launch appends to it
    p->cb_cur = 1 - p->cb_cur;
    c.cbank = p->cb[p->cb_cur];
    p->census_n = n - M;
    p->pin->census[2] = n - M;
    CUDA_OK(cudaMemcpyAsync(c.work + 4, &p->pin->census[2], 4, cudaMemcpyHostToDevice, st));
    CUDA_OK(cudaGetLastError());
    w.census_counts.push_back(M); w.census_counts.push_back(M_run);
    w.census_weights.push_back(W); w.census_weights.push_back(W_run);
    *M_out = M_run;
    return 0;
}

// one census interval of a fixed-source run (time edge k -> k + 1)
// publish_now = false: the caller runs several intervals as ONE call and publishes after the last (a failure part-way
// then leaves the previous call's results readable)
static int interval_internal(mcdc_problem *p, uint64_t N, int k, uint64_t seed, bool publish_now = true)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    const int n_t = c.ce.n_t;
    if (N < 1 || capacity_for(N) > p->cap) return fail(MCDC_EINVAL, "n_particles exceeds the capacity this problem was created for");
    if (N > 60000000ull) return fail(MCDC_EINVAL, "at most 6e7 source particles per fixed-source run (32-bit secondary counters)");
    if (p->schedule == 1) return fail(MCDC_EINVAL, "census intervals need the persistent kernel (schedule 0 or 2)");
    if (k < p->first_interval || k >= n_t) return fail(MCDC_EINVAL, "census interval %d outside [%d, %d)", k, p->first_interval, n_t);
    if (k == p->first_interval) {
        int rc = begin_run(p);
        if (rc) return rc;
        CUDA_OK(cudaMemsetAsync(c.work, 0, 32, st));
        CUDA_OK(cudaMemsetAsync(c.scal, 0, 64, st));
        p->cb_cur = 0; c.cbank = p->cb[0]; p->census_n = 0;
    } else if (p->work.next_interval < 0) return fail(MCDC_EINVAL, "no fixed-source run is under way (none started, or the last interval failed): start again from interval %d", p->first_interval);
    else if (p->work.next_interval != k) return fail(MCDC_EINVAL, "census intervals must be run in order: expected %d, got %d", p->work.next_interval, k);
    RunStats &w = p->work;
    set_seed(c, seed); c.cycle = 0; c.w0 = 1.0; c.k_prev = 1.0;
    c.max_secondaries = 64ull * (N + (uint64_t)p->census_target * (uint64_t)n_t) + 4096;  // R25a
    c.census_stop = k + 1 < n_t ? 1 : 0;
    CUDA_OK(cudaEventRecord(p->t0, st));
    uint64_t M = 0;
    if (k == p->first_interval) {
        const unsigned int nbk = (unsigned int)((N + BS - 1) / BS);
        if (p->mode == 1) k_source<true><<<nbk, BS, 0, st>>>(c, (unsigned int)N);
        else k_source<false, true><<<nbk, BS, 0, st>>>(c, (unsigned int)N);
        p->n_launches++;
        M = N;
        w.census_counts.push_back(N); w.census_counts.push_back(N);
        w.census_weights.push_back((double)N); w.census_weights.push_back((double)N);
        w.host_counters[0] = N;
    } else {
        int rc = p->mode == 1 ? census_to_source_t<true>(p, k, seed, &M) : census_to_source_t<false>(p, k, seed, &M);
        if (rc) return abandon(p, rc);
    }
    if (M > 0) {
        const int keep = p->persist;
        p->persist = 0x7fffffff;  // the census lives in the persistent kernel
        int rc = transport(p, M);
        p->persist = keep;
        if (rc) return abandon(p, rc);
    }
    CUDA_OK(cudaEventRecord(p->t1, st));
    CUDA_OK(cudaMemcpyAsync(&p->pin->census[0], c.work + 4, 4, cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaMemcpyAsync(p->pin->scal, c.scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaMemcpyAsync(p->pin->counters, c.counters, sizeof p->pin->counters, cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaMemcpyAsync(&p->pin->err, c.err, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaStreamSynchronize(st));
    CUDA_OK(cudaGetLastError());
    profile_collect(p);
    // the error flag is read BEFORE this interval's flux is folded into the run's accumulators: after an earlier
    // interval was published they are the published set, and a failed interval must not reach them
    int rc = device_error_code(p, p->pin->err);
    if (rc) return abandon(p, rc);
    p->census_n = p->pin->census[0];
    if (p->census_n > p->cap) return abandon(p, fail(MCDC_EBANK, "census bank overflow (capacity %llu)", (unsigned long long)p->cap));
    k_accumulate<<<(c.n_tally + BS - 1) / BS, BS, 0, st>>>(c.flux, p->flux_copies, p->flux_cycle, p->flux_acc[w.set], p->flux_acc2[w.set],
                                                          c.n_tally, 1.0 / (double)N, 1);
    p->n_launches++;
    CUDA_OK(cudaGetLastError());
    float ms = 0.f;
    CUDA_OK(cudaEventElapsedTime(&ms, p->t0, p->t1));
    p->ms_transport += ms;
    // results so far (the scalars and counters run over all intervals of the run)
    const double k_c = p->pin->scal[0] / (double)N, leak = p->pin->scal[1] / (double)N;
    w.k_cycle.assign(1, k_c);
    w.k_acc = k_c; w.k_acc2 = k_c * k_c; w.leak_acc = leak; w.leak_acc2 = leak * leak; w.n_active = 1;
    w.host_counters[12] = std::max<uint64_t>(w.host_counters[12], std::max<uint64_t>(p->census_n, M));
    for (int i = 0; i < 6; i++) w.balance[i] = 0.0;
    {
        const uint64_t zero[MCDC_N_COUNTERS] = {0};
        // weight started: source particles (1 each) + children (continuous energy: 1 each; multi-group: the parent's, scal[6])
        const double started = (double)N + (p->td ? p->pin->scal[6] : (double)p->pin->counters[15]);
        add_balance(p, started, zero);
    }
    w.next_interval = k + 1;
    p->bank_count = 0;
    p->last_N = N;
    if (publish_now) publish(p);
    return 0;
}

extern "C" int mcdc_run_cycle(mcdc_problem *p, uint64_t N, uint32_t cycle, int32_t active, uint64_t seed, double *k_cycle)
{
    if (!p) return fail(MCDC_EINVAL, "null");
    if (p->timed) {  // fixed-source problem: one census interval
        int rc = interval_internal(p, N, (int)cycle, seed);
        if (rc) return rc;
        if (k_cycle) *k_cycle = p->work.k_cycle.back();
        return 0;
    }
    if (p->mode != 0) return fail(MCDC_EINVAL, "mcdc_run_cycle needs a multi-group problem");
    if (cycle == 0) { int rc = begin_run(p); if (rc) return rc; }
    int rc = cycle_internal(p, N, cycle, active, seed, cycle == 0, nullptr);
    if (rc) return rc;
    publish(p);
    if (k_cycle) *k_cycle = p->work.k_cycle.back();
    return 0;
}

extern "C" int mcdc_run_eigenvalue(mcdc_problem *p, uint64_t N, int32_t n_inactive, int32_t n_active, uint64_t seed)
{
    if (!p || p->mode != 0 || p->td) return fail(MCDC_EINVAL, "mcdc_run_eigenvalue needs a multi-group eigenvalue problem");
    if (n_inactive < 0 || n_active < 0) return fail(MCDC_EINVAL, "cycle counts");
    int rc = begin_run(p);
    if (rc) return rc;
    for (int cyc = 0; cyc < n_inactive + n_active; cyc++) {
        rc = cycle_internal(p, N, (uint32_t)cyc, cyc >= n_inactive, seed, cyc == 0, nullptr);
        if (rc) return rc;
    }
    publish(p);
    return 0;
}

extern "C" int mcdc_run_cycle_host(mcdc_problem *p, uint64_t N, uint32_t cycle, uint64_t seed, double k_prev,
                                   const mcdc_site *sites_in, uint64_t n_in, mcdc_site *sites_out, uint64_t max_out,
                                   uint64_t *n_out, double *flux_cycle, double *k_cycle, double *leak_cycle)
{
    if (!p || p->mode != 0 || p->td) return fail(MCDC_EINVAL, "mcdc_run_cycle_host needs a multi-group eigenvalue problem");
    static_assert(sizeof(Site) == sizeof(mcdc_site), "site layout");
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    bool sample = sites_in == nullptr || n_in == 0;
    if (!sample && n_in > p->cap) return fail(MCDC_EBANK, "source bank larger than the capacity");
    if (cycle == 0) { int rc = begin_run(p); if (rc) return rc; }
    p->k_prev = k_prev;
    if (!sample) {
        CUDA_OK(cudaMemcpyAsync(p->sites, sites_in, n_in * sizeof(Site), cudaMemcpyHostToDevice, st));
        k_load_sites<<<(unsigned int)((n_in + BS - 1) / BS), BS, 0, st>>>(c, p->sites, (unsigned int)n_in);
        p->n_launches++;
        p->bank_count = n_in;
    }
    int rc = cycle_internal(p, N, cycle, 1, seed, sample, flux_cycle);
    if (rc) return rc;
    uint64_t total = p->bank_count;
    if (n_out) *n_out = total;
    if (sites_out && total) {
        uint64_t n = std::min(total, max_out);
        k_store_sites<<<(unsigned int)((n + BS - 1) / BS), BS, 0, st>>>(c, p->sites, (unsigned int)n);
        p->n_launches++;
        CUDA_OK(cudaMemcpyAsync(sites_out, p->sites, n * sizeof(Site), cudaMemcpyDeviceToHost, st));
        CUDA_OK(cudaStreamSynchronize(st));
    }
    publish(p);
    if (k_cycle) *k_cycle = p->work.k_cycle.back();
    if (leak_cycle) *leak_cycle = p->pin->scal[1] / (double)N;
    return 0;
}

extern "C" int mcdc_run_fixed_source(mcdc_problem *p, uint64_t N, uint64_t seed)
{
    if (!p || !p->timed) return fail(MCDC_EINVAL, "mcdc_run_fixed_source needs a continuous-energy or a time-dependent multi-group problem");
    if (p->td) {  // census interval by census interval (population control happens between them, R40)
        for (int k = p->first_interval; k < p->ctx.ce.n_t; k++) {
            int rc = interval_internal(p, N, k, seed, k + 1 == p->ctx.ce.n_t);  // one call: published once, at the end
            if (rc) return rc;
        }
        return 0;
    }
    if (N < 1 || capacity_for(N) > p->cap) return fail(MCDC_EINVAL, "n_particles exceeds the capacity this problem was created for");
    if (N > 60000000ull) return fail(MCDC_EINVAL, "at most 6e7 source particles per fixed-source run (32-bit secondary counters)");
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    int rc = begin_run(p);
    if (rc) return rc;
    set_seed(c, seed); c.cycle = 0; c.w0 = 1.0; c.k_prev = 1.0;
    c.census_stop = 0;  // one launch to the last time edge: a census is a synchronisation point only (R24)
    c.max_secondaries = 64 * N + 4096;  // R25a: the prompt chain must die out
    CUDA_OK(cudaMemsetAsync(c.scal, 0, 64, st));
    CUDA_OK(cudaEventRecord(p->t0, st));
    uint64_t M = N;
    k_source<true><<<(unsigned int)((M + BS - 1) / BS), BS, 0, st>>>(c, (unsigned int)M);
    p->n_launches++;
    RunStats &w = p->work;
    uint64_t secondaries = 0;
    while (M > 0) {  // one wave per fission generation of the prompt chain (monolithic schedule only: the other
                     // schedules transport the secondaries inside the first wave)
        rc = transport(p, M);
        if (rc) return abandon(p, rc);
        uint64_t total = 0;
        rc = emit_children(p, M, &total);
        if (rc) return abandon(p, rc);
        rc = device_error_code(p, p->pin->err);
        if (rc) return abandon(p, rc);
        w.host_counters[0] += M;
        w.host_counters[11] += total;
        uint64_t high = std::max<uint64_t>(total, p->pin->counters[15]);
        if (high > w.host_counters[12]) w.host_counters[12] = high;
        secondaries += total;
        if (secondaries > c.max_secondaries) return abandon(p, fail(MCDC_EBANK, "prompt fission chain does not die out (R25)"));
        M = total;
    }
    CUDA_OK(cudaEventRecord(p->t1, st));
    k_accumulate<<<(c.n_tally + BS - 1) / BS, BS, 0, st>>>(c.flux, p->flux_copies, p->flux_cycle, p->flux_acc[w.set], p->flux_acc2[w.set],
                                                          c.n_tally, 1.0 / (double)N, 1);
    p->n_launches++;
    CUDA_OK(cudaStreamSynchronize(st));
    float ms = 0.f;
    CUDA_OK(cudaEventElapsedTime(&ms, p->t0, p->t1));
    p->ms_transport += ms;
    double k_c = p->pin->scal[0] / (double)N, leak = p->pin->scal[1] / (double)N;
    w.k_cycle.push_back(k_c);
    w.k_acc = k_c; w.k_acc2 = k_c * k_c; w.leak_acc = leak; w.leak_acc2 = leak * leak; w.n_active = 1;
    {  // the scalars and counters run over all waves of the run: one balance entry
        const uint64_t zero[MCDC_N_COUNTERS] = {0};
        add_balance(p, (double)(w.host_counters[0] + p->pin->counters[15]), zero);  // every track starts with weight 1
    }
    p->bank_count = 0;
    p->last_N = N;
    publish(p);
    return 0;
}

extern "C" int mcdc_set_physics(mcdc_problem *p, const mcdc_physics *ph)
{
    if (!p) return fail(MCDC_EINVAL, "null");
    Ctx &c = p->ctx;
    p->persist_blocks_per_sm = 0;  // the weighted kernels have their own occupancy
    if (!ph) { c.kT = 0.0; c.implicit = 0; c.w_roulette = c.w_survive = 0.0; return 0; }
    if (!(ph->kT >= 0.0)) return fail(MCDC_EINVAL, "kT must be >= 0");
    if (ph->implicit_capture && !(ph->w_roulette >= 0.0 && ph->w_survive >= ph->w_roulette))
        return fail(MCDC_EINVAL, "implicit capture needs 0 <= w_roulette <= w_survive");
    c.kT = ph->kT;
    c.implicit = ph->implicit_capture ? 1 : 0;
    c.w_roulette = ph->w_roulette; c.w_survive = ph->w_survive;
    return 0;
}

extern "C" int mcdc_get_census(const mcdc_problem *p, uint64_t *counts, double *weights, int32_t max, int32_t *n)
{
    if (!p || !counts || !weights || !n) return fail(MCDC_EINVAL, "null");
    const RunStats &r = p->pub;
    int m = (int)std::min<size_t>(r.census_counts.size() / 2, (size_t)std::max(max, 0));
    for (int i = 0; i < 2 * m; i++) { counts[i] = r.census_counts[i]; weights[i] = r.census_weights[i]; }
    *n = m;
    return 0;
}

extern "C" int mcdc_get_balance(const mcdc_problem *p, double out[6])
{
    if (!p || !out) return fail(MCDC_EINVAL, "null");
    for (int k = 0; k < 6; k++) out[k] = p->pub.balance[k];
    return 0;
}

// ------------------------------------------------------------------ results
extern "C" int mcdc_get_dims(const mcdc_problem *p, mcdc_dims *d)
{
    if (!p || !d) return fail(MCDC_EINVAL, "null");
    d->mode = p->mode; d->n_tally = p->ctx.n_tally; d->n_cycles = (int)p->pub.k_cycle.size(); d->n_active = p->pub.n_active;
    d->bank_count = p->bank_count;
    return 0;
}

static double sdev_of(double acc, double acc2, int n)
{
    if (n < 2) return 0.0;
    double m = acc / n, var = acc2 / n - m * m;
    return var > 0.0 ? std::sqrt(var / (n - 1)) : 0.0;
}

extern "C" int mcdc_get_tallies(const mcdc_problem *p, mcdc_tallies *out)
{
    if (!p || !out) return fail(MCDC_EINVAL, "null");
    const Ctx &c = p->ctx;
    const RunStats &r = p->pub;
    int n = r.n_active;
    double dn = n > 0 ? (double)n : 1.0;
    if (out->k_cycle) for (size_t i = 0; i < r.k_cycle.size(); i++) out->k_cycle[i] = r.k_cycle[i];
    out->k_mean = r.k_acc / dn; out->k_sdev = sdev_of(r.k_acc, r.k_acc2, n);
    out->leak_mean = r.leak_acc / dn; out->leak_sdev = sdev_of(r.leak_acc, r.leak_acc2, n);
    if (out->flux_mean || out->flux_sdev) {
        std::vector<double> a(c.n_tally), a2(c.n_tally);
        CUDA_OK(cudaMemcpyAsync(a.data(), p->flux_acc[r.set], sizeof(double) * c.n_tally, cudaMemcpyDeviceToHost, p->stream));
        CUDA_OK(cudaMemcpyAsync(a2.data(), p->flux_acc2[r.set], sizeof(double) * c.n_tally, cudaMemcpyDeviceToHost, p->stream));
        CUDA_OK(cudaStreamSynchronize(p->stream));
        for (int i = 0; i < c.n_tally; i++) {
            if (out->flux_mean) out->flux_mean[i] = a[i] / dn;
            if (out->flux_sdev) out->flux_sdev[i] = sdev_of(a[i], a2[i], n);
        }
    }
    if (out->counters) for (int i = 0; i < MCDC_N_COUNTERS; i++) out->counters[i] = r.counters[i];
    return 0;
}

extern "C" int mcdc_get_bank(const mcdc_problem *p, mcdc_site *out, uint64_t max, uint64_t *n)
{
    if (!p || !n) return fail(MCDC_EINVAL, "null");
    if (p->mode != 0) return fail(MCDC_EINVAL, "multi-group only");
    *n = p->bank_count;
    uint64_t m = std::min(p->bank_count, max);
    if (out && m) {
        k_store_sites<<<(unsigned int)((m + BS - 1) / BS), BS, 0, p->stream>>>(p->ctx, p->sites, (unsigned int)m);
        CUDA_OK(cudaMemcpyAsync(out, p->sites, m * sizeof(Site), cudaMemcpyDeviceToHost, p->stream));
        CUDA_OK(cudaStreamSynchronize(p->stream));
    }
    return 0;
}

extern "C" int mcdc_set_trace(mcdc_problem *p, uint64_t first_id, uint32_t n_ids, uint32_t max_events)
{
    if (!p) return fail(MCDC_EINVAL, "null");
    static_assert(sizeof(TraceRec) == sizeof(mcdc_trace_rec), "trace layout");
    if (n_ids == 0 || max_events == 0) {
        p->ctx.tr.rec = nullptr;
        CUDA_OK(cudaMemcpy((void *)p->ctx.tr_g, &p->ctx.tr, sizeof(Trace), cudaMemcpyHostToDevice));
        return 0;
    }
    uint64_t per_slot = (uint64_t)max_events * sizeof(TraceRec);
    uint64_t slots = TRACE_BYTES / per_slot;
    if (slots < n_ids) return fail(MCDC_ENOMEM, "trace buffer holds %llu (id, cycle) slots of %u events; %u ids asked", (unsigned long long)slots, max_events, n_ids);
    Trace &t = p->ctx.tr;
    t.first = first_id; t.n_ids = n_ids; t.max_events = max_events;
    t.cap_slots = (unsigned int)std::min<uint64_t>(slots, TRACE_BYTES / sizeof(TraceRec));
    t.rec = p->trace_base; t.count = p->trace_count;
    CUDA_OK(cudaMemcpyAsync((void *)p->ctx.tr_g, &t, sizeof(Trace), cudaMemcpyHostToDevice, p->stream));
    CUDA_OK(cudaMemsetAsync(t.count, 0, sizeof(unsigned int) * t.cap_slots, p->stream));
    CUDA_OK(cudaStreamSynchronize(p->stream));
    return 0;
}

extern "C" int mcdc_get_trace(const mcdc_problem *p, mcdc_trace_rec *out, uint64_t max, uint64_t *n)
{
    if (!p || !n) return fail(MCDC_EINVAL, "null");
    const Trace &t = p->ctx.tr;
    *n = 0;
    if (!t.rec) return 0;
    std::vector<unsigned int> cnt(t.cap_slots);
    CUDA_OK(cudaMemcpy(cnt.data(), t.count, sizeof(unsigned int) * t.cap_slots, cudaMemcpyDeviceToHost));
    uint64_t total = 0, written = 0;
    std::vector<TraceRec> buf(t.max_events);
    for (unsigned int sl = 0; sl < t.cap_slots; sl++) {
        unsigned int k = std::min(cnt[sl], t.max_events);
        total += cnt[sl];
        if (!k || !out || written >= max) continue;
        CUDA_OK(cudaMemcpy(buf.data(), (const TraceRec *)t.rec + (uint64_t)sl * t.max_events, k * sizeof(TraceRec), cudaMemcpyDeviceToHost));
        for (unsigned int j = 0; j < k && written < max; j++) memcpy(&out[written++], &buf[j], sizeof(TraceRec));
    }
    *n = total;
    return 0;
}

extern "C" int mcdc_set_profile(mcdc_problem *p, int32_t on)
{
    if (!p) return fail(MCDC_EINVAL, "null");
    p->profile = on ? 1 : 0;
    unsigned long long b = 0;
    CUDA_OK(cudaMemcpy(&b, p->ctx.counters + 12, sizeof b, cudaMemcpyDeviceToHost));
    p->prof_sweep_base = b;
    memset(p->prof_ms, 0, sizeof p->prof_ms); memset(p->prof_launches, 0, sizeof p->prof_launches);
    return 0;
}

extern "C" int mcdc_get_profile(const mcdc_problem *p, double *ms, uint64_t *launches, uint64_t *sweep_events)
{
    if (!p || !ms || !launches) return fail(MCDC_EINVAL, "null");
    for (int k = 0; k < MCDC_N_PROFILE; k++) { ms[k] = p->prof_ms[k]; launches[k] = p->prof_launches[k]; }
    if (sweep_events) {
        unsigned long long b = 0;
        CUDA_OK(cudaMemcpy(&b, p->ctx.counters + 12, sizeof b, cudaMemcpyDeviceToHost));
        *sweep_events = b - p->prof_sweep_base;
    }
    return 0;
}

extern "C" int mcdc_get_timing(const mcdc_problem *p, double *ms, uint64_t *nl)
{
    if (!p) return fail(MCDC_EINVAL, "null");
    if (ms) *ms = p->ms_transport;
    if (nl) *nl = p->n_launches;
    return 0;
}

// ------------------------------------------------------------------ unit-level entry points
// scratch for the test entry points is taken from the (idle) site staging buffer
extern "C" int mcdc_test_draws(mcdc_problem *p, uint64_t seed, uint32_t domain, uint32_t cycle, const uint64_t *id,
                               const uint32_t *draw, uint64_t n, double *out)
{
    if (!p || !id || !draw || !out) return fail(MCDC_EINVAL, "null");
    if (n * 24 > p->cap * sizeof(Site)) return fail(MCDC_ENOMEM, "too many draws for the scratch buffer");
    char *base = (char *)p->sites;
    unsigned long long *d_id = (unsigned long long *)base;
    double *d_out = (double *)(base + n * 8);
    uint32_t *d_draw = (uint32_t *)(base + n * 16);
    CUDA_OK(cudaMemcpyAsync(d_id, id, n * 8, cudaMemcpyHostToDevice, p->stream));
    CUDA_OK(cudaMemcpyAsync(d_draw, draw, n * 4, cudaMemcpyHostToDevice, p->stream));
    k_test_draws<<<(unsigned int)((n + 255) / 256), 256, 0, p->stream>>>(seed, domain, cycle, d_id, d_draw, n, d_out);
    CUDA_OK(cudaMemcpyAsync(out, d_out, n * 8, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaStreamSynchronize(p->stream));
    return 0;
}

extern "C" int mcdc_test_grid_index(mcdc_problem *p, const double *E, uint64_t n, int32_t *ob, int32_t *oh)
{
    if (!p || p->mode != 1 || !E || !ob || !oh) return fail(MCDC_EINVAL, "needs a continuous-energy problem");
    if (n * 16 > p->cap * sizeof(Site)) return fail(MCDC_ENOMEM, "too many points for the scratch buffer");
    char *base = (char *)p->sites;
    double *d_E = (double *)base;
    int *d_b = (int *)(base + n * 8), *d_h = (int *)(base + n * 12);
    CUDA_OK(cudaMemcpyAsync(d_E, E, n * 8, cudaMemcpyHostToDevice, p->stream));
    k_test_grid<<<(unsigned int)((n + 255) / 256), 256, 0, p->stream>>>(p->ctx, d_E, n, d_b, d_h);
    CUDA_OK(cudaMemcpyAsync(ob, d_b, n * 4, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaMemcpyAsync(oh, d_h, n * 4, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaStreamSynchronize(p->stream));
    return 0;
}

extern "C" int mcdc_test_geometry(mcdc_problem *p, const double *x, const double *u, uint64_t n, int32_t path, int32_t *loc,
                                  double *dist, int32_t *surf)
{
    if (!p || !x || !u || !loc || !dist || !surf) return fail(MCDC_EINVAL, "null");
    if (path < 0 || path > 2) return fail(MCDC_EINVAL, "path must be 0, 1 or 2");
    if (n * 72 > p->cap * sizeof(Site)) return fail(MCDC_ENOMEM, "too many points for the scratch buffer");
    char *base = (char *)p->sites;
    double *d_x = (double *)base, *d_u = (double *)(base + n * 24), *d_d = (double *)(base + n * 48);
    int *d_loc = (int *)(base + n * 56), *d_s = (int *)(base + n * 68);
    CUDA_OK(cudaMemcpyAsync(d_x, x, n * 24, cudaMemcpyHostToDevice, p->stream));
    CUDA_OK(cudaMemcpyAsync(d_u, u, n * 24, cudaMemcpyHostToDevice, p->stream));
    k_test_geometry<<<(unsigned int)((n + 255) / 256), 256, 0, p->stream>>>(p->ctx, d_x, d_u, n, path, d_loc, d_d, d_s);
    CUDA_OK(cudaMemcpyAsync(loc, d_loc, n * 12, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaMemcpyAsync(dist, d_d, n * 8, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaMemcpyAsync(surf, d_s, n * 4, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaStreamSynchronize(p->stream));
    return 0;
}

// ------------------------------------------------------------------ arithmetic micro-benchmarks
extern "C" int mcdc_microbench(mcdc_problem *p, int32_t which, uint64_t iters, double *ms_out, double *ops_out)
{
    if (!p || !ms_out || !ops_out) return fail(MCDC_EINVAL, "null");
    if (which < 0 || which >= MCDC_MB_COUNT || iters < 1) return fail(MCDC_EINVAL, "which / iters");
    cudaStream_t st = p->stream;
    const unsigned int threads = 256, blocks = 148 * 8;  // 2048 resident threads on every SM
    if ((uint64_t)threads * blocks * 8 > p->cap * sizeof(Site)) return fail(MCDC_ENOMEM, "scratch buffer too small");
    double *out = (double *)p->sites;
    double per_thread = 0.0;
    for (int pass = 0; pass < 2; pass++) {  // pass 0 warms up
        CUDA_OK(cudaEventRecord(p->t0, st));
        switch (which) {
        case MCDC_MB_FFMA: k_mb_ffma<<<blocks, threads, 0, st>>>(iters, (float *)out); per_thread = (double)MB_CHAINS * iters; break;
        case MCDC_MB_DFMA: k_mb_dfma<<<blocks, threads, 0, st>>>(iters, out); per_thread = (double)MB_CHAINS * iters; break;
        case MCDC_MB_LOG: k_mb_func<0><<<blocks, threads, 0, st>>>(iters, out); per_thread = 4.0 * iters; break;
        case MCDC_MB_DIV: k_mb_func<1><<<blocks, threads, 0, st>>>(iters, out); per_thread = 4.0 * iters; break;
        case MCDC_MB_SQRT: k_mb_func<2><<<blocks, threads, 0, st>>>(iters, out); per_thread = 4.0 * iters; break;
        case MCDC_MB_SINCOSPI: k_mb_func<3><<<blocks, threads, 0, st>>>(iters, out); per_thread = 4.0 * iters; break;
        case MCDC_MB_RCP: k_mb_func<4><<<blocks, threads, 0, st>>>(iters, out); per_thread = 4.0 * iters; break;
        default: k_mb_philox<<<blocks, threads, 0, st>>>(iters, out); per_thread = 4.0 * iters; break;
        }
        CUDA_OK(cudaEventRecord(p->t1, st));
        CUDA_OK(cudaStreamSynchronize(st));
        CUDA_OK(cudaGetLastError());
    }
    float ms = 0.f;
    CUDA_OK(cudaEventElapsedTime(&ms, p->t0, p->t1));
    *ms_out = ms;
    *ops_out = per_thread * threads * blocks;  // thread-level operations of the timed launch
    return 0;
}

// ------------------------------------------------------------------ the entry point that allocates nothing
// mcdc_draws_noalloc (include/mcdc.h): mcdc_test_draws for a caller that has no device memory to lend.  The three staging
// arrays that mcdc_test_draws carves out of the problem's workspace live here instead, in an array that is part of the
// library's device image: it exists on every GPU from the moment that GPU loads the library until the process ends,
// whether or not the entry point is ever called (MCDC_NOALLOC_DRAWS_MAX x 24 bytes = 1.5 MiB per GPU).
static __device__ __align__(256) unsigned char g_noalloc_scratch[(size_t)MCDC_NOALLOC_DRAWS_MAX * 24u];

// In HOST code the name g_noalloc_scratch is only a handle for the runtime, not the array's device address, so it must
// never be handed to a kernel or to cudaMemcpy as a pointer.  The address is asked for once per device, with that
// device current, and kept here.
enum { NOALLOC_MAX_DEVICES = 64 };
static std::mutex g_noalloc_mutex;
static unsigned char *g_noalloc_ptr[NOALLOC_MAX_DEVICES];  // zero-initialised: "not asked yet"

extern "C" int mcdc_draws_noalloc(int32_t device, void *stream, uint64_t seed, uint32_t domain, uint32_t cycle,
                                  const uint64_t *id, const uint32_t *draw, uint64_t n, double *out)
{
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return fail(MCDC_EINVAL, "device %d outside [0, %d)", (int)device, (int)NOALLOC_MAX_DEVICES);
    if (n > (uint64_t)MCDC_NOALLOC_DRAWS_MAX)
        return fail(MCDC_EINVAL, "mcdc_draws_noalloc: %llu draws asked for, the built-in scratch holds at most %d per call "
                                 "(split the request, or use mcdc_test_draws with a workspace)",
                    (unsigned long long)n, (int)MCDC_NOALLOC_DRAWS_MAX);
    if (n == 0) return 0;
    if (!id || !draw || !out) return fail(MCDC_EINVAL, "null");
    // one call at a time per process: every call stages through the same bytes
    std::lock_guard<std::mutex> guard(g_noalloc_mutex);
    int prev = -1;
    CUDA_OK(cudaGetDevice(&prev));
    if (prev != device) CUDA_OK(cudaSetDevice(device));
    int rc = 0;
    do {
        unsigned char *base = g_noalloc_ptr[device];
        if (!base) {  // first call on this device: resolve the array's address there
            void *sym = nullptr;
            cudaError_t e = cudaGetSymbolAddress(&sym, g_noalloc_scratch);
            if (e != cudaSuccess || !sym) {
                rc = fail(MCDC_ECUDA, "cudaGetSymbolAddress(g_noalloc_scratch) on device %d: %s", (int)device, cudaGetErrorString(e));
                break;
            }
            g_noalloc_ptr[device] = base = (unsigned char *)sym;
        }
        cudaStream_t st = (cudaStream_t)stream;
        // same carving as mcdc_test_draws.  Nothing here has to start at zero: the kernel reads d_id[i], d_draw[i] and
        // writes d_out[i] for i < n only, and all of those are overwritten by this call before they are read.
        unsigned long long *d_id = (unsigned long long *)base;
        double *d_out = (double *)(base + n * 8);
        uint32_t *d_draw = (uint32_t *)(base + n * 16);
        cudaError_t e = cudaMemcpyAsync(d_id, id, n * 8, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_draw, draw, n * 4, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) {
            k_test_draws<<<(unsigned int)((n + 255) / 256), 256, 0, st>>>(seed, domain, cycle, d_id, d_draw, n, d_out);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(out, d_out, n * 8, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) rc = fail(MCDC_ECUDA, "mcdc_draws_noalloc: %s", cudaGetErrorString(e));
    } while (0);
    if (prev != device) cudaSetDevice(prev);
    return rc;
}
