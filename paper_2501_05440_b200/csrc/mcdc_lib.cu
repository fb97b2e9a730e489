// mcdc_lib.cu -- host side of the C-ABI (include/mcdc.h): input validation and derived tables, workspace
// carving, the sweep / cycle drivers and result read-back.  All device work is in mcdc_kernels.cuh.
#include "../../include/mcdc.h"
#include "mcdc_kernels.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
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

static const int LAG = 3;                 // sweeps the host may run ahead of the queue-count read-back
static const int DEFAULT_TAIL = 32768;    // live particles at which the tail kernel takes over (multi-group)
static const int DEFAULT_TAIL_CE = -1;    // continuous energy: no tail kernel by default (measured: 64 -> 91, 16 -> 88, none -> 83.6 ms on C5)
// live particles below which a sweep is one fused multi-segment launch (measured on B200, profiles/r01_step4*.md)
static const int DEFAULT_FUSE = 2000000, DEFAULT_FUSE_CE = 4000000;
static const int DEFAULT_FUSE_SEGMENTS = 8, DEFAULT_FUSE_SEGMENTS_CE = 16;
static const uint64_t TRACE_BYTES = 48ull << 20;
#ifndef MCDC_AGG_MAX
#define MCDC_AGG_MAX 4096
#endif
static const int AGGREGATE_TALLY_MAX = MCDC_AGG_MAX;  // above this, equal bins inside a warp are rare: plain float64 atomics
static const uint64_t GEO_STAGE_MAX_BYTES = 8192;  // CSG tables up to this size are staged in shared memory
static const uint64_t MG_STAGE_MAX_BYTES = 16384;  // multi-group tables up to this size are staged in shared memory
static const int PRIVATE_TALLY_MAX = 20;  // bins for which the one-column-per-thread tally fits (20*256*8 = 40 KB)

struct HostPinned {
    QCount qc[RING];
    double scal[4];
    unsigned int total;
    int err;
};

struct mcdc_problem {
    Ctx ctx;
    int mode;
    cudaStream_t stream;
    int device;
    int schedule, tail, fuse, fuse_segments;
    uint64_t cap;  // bank slots
    // workspace pieces not in ctx
    double *flux_acc, *flux_acc2, *flux_cycle;
    int flux_copies;
    unsigned int *part;
    Site *sites;
    char *trace_base;
    unsigned int *trace_count;
    HostPinned *pin;
    cudaEvent_t ev[RING], t0, t1;
    // run state
    uint64_t bank_count;  // sites in bank[cur] to start the next cycle from
    double k_prev;
    std::vector<double> k_cycle;
    int n_active;
    double k_acc, k_acc2, leak_acc, leak_acc2;
    uint64_t host_counters[MCDC_N_COUNTERS];
    double ms_transport;
    uint64_t n_launches;
    bool tally_private;
    uint64_t trace_first;
    uint32_t trace_n_ids, trace_max_events;
    uint32_t trace_cap_slots;
    uint64_t last_N;
    // optional per-kernel-class timing (mcdc_set_profile): event pairs around every launch
    int profile;
    std::vector<cudaEvent_t> pool;
    std::vector<int> pool_class;  // class of pair k (events 2k, 2k+1)
    double prof_ms[MCDC_N_PROFILE];
    uint64_t prof_launches[MCDC_N_PROFILE];
    uint64_t prof_adv_base;  // device counter 12 (events processed by k_advance) when profiling was switched on
};

// RAII-free helper: record an event pair around one launch when profiling is on
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
    // small tables
    int *surf_type, *surf_bc, *cso, *csi, *css, *cft, *cfill, *cbin, *uco, *lat_univ, *lat_bin;
    unsigned int *lat_rmask;
    double *surf_param;
    double *sig_t, *sig_s, *sig_f, *nu, *nusf, *cumS, *cumchi, *src_cum;
    double *grid, *tab, *colA, *t_edges, *e_edges;
    int *ncol, *hash;
    uint64_t mg_doubles, geo_words;
    Bank bank[2];
    FisRec fis;
    StackRec *stack;
    uint64_t stack_threads;
    QCount *qc;
    double *flux, *flux_acc, *flux_acc2, *flux_cycle, *scal;
    unsigned long long *counters;
    int *err;
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
    return mat ? (uint64_t)t->n_bins * mat->G : (uint64_t)t->n_bins * t->n_t * t->n_e;
}

static int hash_params(const double *grid, int n, int &shift, int &lo, int &n_hash)
{
    // key = top bits of the IEEE-754 pattern: exponent + 8 mantissa bits => 256 buckets per octave
    shift = 52 - 8;
    long long klo, khi;
    double a = grid[0], b = grid[n - 1];
    memcpy(&klo, &a, 8);
    memcpy(&khi, &b, 8);
    lo = (int)(klo >> shift);
    n_hash = (int)(khi >> shift) - lo + 1;
    return 0;
}

static void carve(Layout &L, void *ws, const mcdc_geometry *g, const mcdc_materials *m, const mcdc_xs *x,
                  const mcdc_tally_spec *t, uint64_t cap)
{
    Carver C(ws);
    int nref = g->cell_surf_off[g->n_cell];
    int nlat = g->has_lattice ? g->lat_nx * g->lat_ny : 0;
    // one contiguous blob (staged in shared memory by the kernels): surface parameters first (8-byte aligned),
    // then the int tables
    {
        uint64_t ns = g->n_surf, nc = g->n_cell;
        uint64_t n_int = 2 * ns + (nc + 1) + 2 * (uint64_t)nref + 3 * nc + (g->n_univ + 1);
        L.geo_words = 8 * ns + n_int;
        L.surf_param = C.take<double>(4 * ns + (n_int + 1) / 2);
        int *ip = (int *)(L.surf_param + 4 * ns);
        L.surf_type = ip; ip += ns; L.surf_bc = ip; ip += ns;
        L.cso = ip; ip += nc + 1; L.csi = ip; ip += nref; L.css = ip; ip += nref;
        L.cft = ip; ip += nc; L.cfill = ip; ip += nc; L.cbin = ip; ip += nc;
        L.uco = ip;
    }
    L.lat_univ = C.take<int>(nlat); L.lat_bin = C.take<int>(nlat); L.lat_rmask = C.take<unsigned int>(nlat);
    bool ce = x != nullptr;
    if (!ce) {
        uint64_t mg = (uint64_t)m->n_mat * m->G;
        // one contiguous blob (staged in shared memory by the kernels): six [n_mat][G] tables, cumS, src_cum
        L.mg_doubles = 6 * mg + mg * m->G + m->G;
        L.sig_t = C.take<double>(L.mg_doubles);
        L.sig_s = L.sig_t + mg; L.sig_f = L.sig_s + mg; L.nu = L.sig_f + mg; L.nusf = L.nu + mg; L.cumchi = L.nusf + mg;
        L.cumS = L.cumchi + mg; L.src_cum = L.cumS + mg * m->G;
        L.grid = L.tab = L.colA = L.t_edges = L.e_edges = nullptr; L.ncol = L.hash = nullptr;
    } else {
        int sh, lo, nh;
        hash_params(x->grid, x->n_grid, sh, lo, nh);
        L.grid = C.take<double>(x->n_grid);
        L.tab = C.take<double>((uint64_t)x->n_mat * x->n_grid * CE_ROW);
        L.colA = C.take<double>((uint64_t)x->n_mat * CE_ROW);
        L.ncol = C.take<int>(x->n_mat);
        L.hash = C.take<int>(nh + 2);
        L.t_edges = C.take<double>(t->n_t + 1); L.e_edges = C.take<double>(t->n_e + 1);
        L.sig_t = L.sig_s = L.sig_f = L.nu = L.nusf = L.cumS = L.cumchi = L.src_cum = nullptr;
        L.mg_doubles = 0;
    }
    for (int b = 0; b < 2; b++) {
        Bank &B = L.bank[b];
        B.x = C.take<double>(cap); B.y = C.take<double>(cap); B.z = C.take<double>(cap);
        B.ux = C.take<double>(cap); B.uy = C.take<double>(cap); B.uz = C.take<double>(cap);
        B.E = ce ? C.take<double>(cap) : nullptr; B.t = ce ? C.take<double>(cap) : nullptr;
        B.cell = C.take<int>(cap); B.elem = C.take<int>(cap); B.gl = C.take<int>(cap);
        B.tbin = ce ? C.take<int>(cap) : nullptr;
        B.ev = C.take<int>(cap);
        B.ctr = C.take<uint32_t>(cap); B.slot = C.take<uint32_t>(cap);
        B.id = ce ? C.take<uint64_t>(cap) : nullptr;
    }
    {
        FisRec &F = L.fis;
        const uint64_t fc = cap + OVER_CAP;  // the wave's slots + the tail kernel's overflow records
        F.n = C.take<int>(fc); F.cell = C.take<int>(fc); F.elem = C.take<int>(fc);
        F.tbin = ce ? C.take<int>(fc) : nullptr;
        F.x = C.take<double>(fc); F.y = C.take<double>(fc); F.z = C.take<double>(fc);
        F.t = ce ? C.take<double>(fc) : nullptr;
        F.ctr = C.take<uint32_t>(fc);
        F.id = ce ? C.take<uint64_t>(fc) : nullptr;
    }
    L.stack_threads = ce ? std::min<uint64_t>(148ull * 16ull * 256, (cap + BS - 1) / BS * BS) : 0;
    L.stack = C.take<StackRec>(L.stack_threads * STACK_DEPTH);
    L.qc = C.take<QCount>(RING);
    uint64_t nt = n_tally_of(m, t);
    L.flux = C.take<double>(nt * flux_copies_for(nt)); L.flux_acc = C.take<double>(nt); L.flux_acc2 = C.take<double>(nt);
    L.flux_cycle = C.take<double>(nt);
    L.scal = C.take<double>(8);
    L.counters = C.take<unsigned long long>(MCDC_N_COUNTERS);
    L.err = C.take<int>(4);
    L.part = C.take<unsigned int>((cap + OVER_CAP) / BS + 4);
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
    if (g->n_surf > 30000) return fail(MCDC_EINVAL, "too many surfaces");
    int n_mat = m ? m->n_mat : x->n_mat;
    int n_lat_cells = 0;
    for (int c = 0; c < g->n_cell; c++) {
        if (g->cell_surf_off[c + 1] < g->cell_surf_off[c]) return fail(MCDC_EINVAL, "cell_surf_off not monotone");
        for (int k = g->cell_surf_off[c]; k < g->cell_surf_off[c + 1]; k++) {
            if (g->cell_surf_id[k] < 0 || g->cell_surf_id[k] >= g->n_surf) return fail(MCDC_EGEOM, "cell %d names surface %d", c, g->cell_surf_id[k]);
            if (g->cell_surf_sense[k] != 1 && g->cell_surf_sense[k] != -1) return fail(MCDC_EGEOM, "sense must be +-1");
        }
        if (g->cell_fill_type[c] == 1) n_lat_cells++;
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
        if (!t->lat_bin) return fail(MCDC_EINVAL, "lat_bin missing");
        for (int e = 0; e < g->lat_nx * g->lat_ny; e++) {
            if (g->lat_univ[e] < 1 || g->lat_univ[e] >= g->n_univ) return fail(MCDC_EGEOM, "lattice element %d names universe %d", e, g->lat_univ[e]);
            if (t->lat_bin[e] < 0 || t->lat_bin[e] >= t->n_bins) return fail(MCDC_EINVAL, "lat_bin out of range");
        }
    } else if (n_lat_cells) return fail(MCDC_EGEOM, "lattice-filled cell without a lattice");
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
    } else {
        if (x->n_grid < 2 || x->n_nuc < 1) return fail(MCDC_EINVAL, "CE grid");
        for (int i = 1; i < x->n_grid; i++)
            if (!(x->grid[i] > x->grid[i - 1])) return fail(MCDC_EINVAL, "union grid not strictly increasing at %d", i);
        if (!(x->grid[0] > 0.0)) return fail(MCDC_EINVAL, "grid must be positive");
        for (int mm = 0; mm < x->n_mat; mm++) {
            int nn = x->mat_nuc_off[mm + 1] - x->mat_nuc_off[mm];
            if (nn < 1 || nn + 2 > MAX_CE_COL) return fail(MCDC_EINVAL, "material %d: 1..%d nuclides supported", mm, MAX_CE_COL - 2);
            for (int j = x->mat_nuc_off[mm]; j < x->mat_nuc_off[mm + 1]; j++)
                if (x->mat_nuc_id[j] < 0 || x->mat_nuc_id[j] >= x->n_nuc) return fail(MCDC_EINVAL, "nuclide id");
        }
        if (t->n_t < 1 || t->n_e < 1 || !t->t_edges || !t->e_edges) return fail(MCDC_EINVAL, "CE tally edges");
        for (int i = 0; i < t->n_t; i++) if (!(t->t_edges[i + 1] > t->t_edges[i])) return fail(MCDC_EINVAL, "t_edges");
        for (int i = 0; i < t->n_e; i++) if (!(t->e_edges[i + 1] > t->e_edges[i])) return fail(MCDC_EINVAL, "e_edges");
    }
    if (t->n_bins < 1) return fail(MCDC_EINVAL, "n_bins");
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
    p->tail = dev->tail_threshold == 0 ? (x ? DEFAULT_TAIL_CE : DEFAULT_TAIL) : dev->tail_threshold;
    p->fuse = dev->fuse_threshold == 0 ? (x ? DEFAULT_FUSE_CE : DEFAULT_FUSE) : dev->fuse_threshold;
    p->fuse_segments = dev->fuse_segments <= 0 ? (x ? DEFAULT_FUSE_SEGMENTS_CE : DEFAULT_FUSE_SEGMENTS) : dev->fuse_segments;
    p->cap = cap;
    Ctx &c = p->ctx;
    c.mode = p->mode;

    // ---- geometry
    int nref = g->cell_surf_off[g->n_cell];
    int nlat = g->has_lattice ? g->lat_nx * g->lat_ny : 0;
    Geo &G = c.geo;
    G.n_surf = g->n_surf; G.n_cell = g->n_cell; G.n_univ = g->n_univ; G.has_lat = g->has_lattice;
    G.lat_nx = g->has_lattice ? g->lat_nx : 1; G.lat_ny = g->has_lattice ? g->lat_ny : 1;
    G.lat_x0 = g->lat_x0; G.lat_y0 = g->lat_y0; G.lat_px = g->lat_px; G.lat_py = g->lat_py;
    G.lat_cell = -1;
    G.lat_magic = (unsigned int)(0x100000000ull / (unsigned long long)G.lat_nx) + 1u;
    for (int cc = 0; cc < g->n_cell; cc++) if (g->cell_fill_type[cc] == 1) G.lat_cell = cc;
    G.surf_type = L.surf_type; G.surf_bc = L.surf_bc; G.surf_param = L.surf_param;
    G.cso = L.cso; G.csi = L.csi; G.css = L.css; G.cft = L.cft; G.cfill = L.cfill; G.cbin = L.cbin; G.uco = L.uco;
    G.lat_univ = L.lat_univ; G.lat_bin = L.lat_bin; G.lat_rmask = L.lat_rmask;
    G.blob = (const char *)L.surf_param; G.blob_words = (int)L.geo_words;
    c.geo_stage = L.geo_words * 4 <= GEO_STAGE_MAX_BYTES ? (int)L.geo_words : 0;
    // host staging must outlive the async copies: keep vectors until the sync at the end
    std::vector<double> h_sig_s, h_nusf, h_cumS, h_cumchi, h_srccum, h_tab, h_colA;
    std::vector<int> h_ncol, h_hash, h_cfill(g->cell_fill, g->cell_fill + g->n_cell);
    for (int cc = 0; cc < g->n_cell; cc++) if (g->cell_fill_type[cc] == 1) h_cfill[cc] = 0;
    cudaError_t e = cudaSuccess;
#define UP(dst, src, n) do { if (e == cudaSuccess) e = up(dst, src, (uint64_t)(n), st); } while (0)
    UP(L.surf_type, g->surf_type, g->n_surf); UP(L.surf_bc, g->surf_bc, g->n_surf);
    UP(L.surf_param, g->surf_param, 4 * g->n_surf);
    UP(L.cso, g->cell_surf_off, g->n_cell + 1); UP(L.csi, g->cell_surf_id, nref); UP(L.css, g->cell_surf_sense, nref);
    UP(L.cft, g->cell_fill_type, g->n_cell); UP(L.cfill, h_cfill.data(), g->n_cell); UP(L.cbin, t->cell_bin, g->n_cell);
    UP(L.uco, g->univ_cell_off, g->n_univ + 1);
    // lattice element -> tally bin, plus which of the enclosing cell's surfaces must be tested from inside the
    // element (bit mask over the cell's surface list; flag bit 30 of lat_bin = mask != 0).  A surface is dropped
    // only where it is provably never the nearest candidate: an axis plane x = p (y = p) lying strictly beyond a
    // wall of the element that is itself an event (an interior lattice wall, R14) -- the ray crosses that wall
    // first.  Any other surface type, and planes beyond an outermost (non-event) wall, stay in the mask.
    std::vector<int> h_latbin(nlat);
    std::vector<unsigned int> h_rmask(nlat);
    if (nlat) {
        int lc = G.lat_cell;
        for (int iy = 0; iy < g->lat_ny; iy++)
            for (int ix = 0; ix < g->lat_nx; ix++) {
                unsigned int mask = 0u;
                double xlo = g->lat_x0 + ix * g->lat_px, xhi = g->lat_x0 + (ix + 1) * g->lat_px;
                double ylo = g->lat_y0 + iy * g->lat_py, yhi = g->lat_y0 + (iy + 1) * g->lat_py;
                double tx = 1e-9 * g->lat_px, ty = 1e-9 * g->lat_py;
                for (int k = g->cell_surf_off[lc]; k < g->cell_surf_off[lc + 1]; k++) {
                    int sidx = g->cell_surf_id[k], j = k - g->cell_surf_off[lc];
                    double pp = g->surf_param[4 * sidx];
                    bool need = true;
                    if (g->surf_type[sidx] == MCDC_PLANE_X)
                        need = !((pp > xhi + tx && ix + 1 < g->lat_nx) || (pp < xlo - tx && ix > 0));
                    else if (g->surf_type[sidx] == MCDC_PLANE_Y)
                        need = !((pp > yhi + ty && iy + 1 < g->lat_ny) || (pp < ylo - ty && iy > 0));
                    if (j >= 32) { if (need) mask |= 0x80000000u; }  // past the 32nd surface: always tested
                    else if (need) mask |= 1u << j;
                }
                int e_ = iy * g->lat_nx + ix;
                h_rmask[e_] = mask;
                h_latbin[e_] = t->lat_bin[e_] | (mask ? LAT_ROOT_FLAG : 0);
            }
        UP(L.lat_univ, g->lat_univ, nlat); UP(L.lat_bin, h_latbin.data(), nlat); UP(L.lat_rmask, h_rmask.data(), nlat);
    }

    // ---- cross sections: derived tables built here, in plain left-to-right float64 sums
    if (m) {
        int Gn = m->G, nm = m->n_mat;
        h_sig_s.assign((size_t)nm * Gn, 0.0); h_nusf.assign((size_t)nm * Gn, 0.0);
        h_cumS.assign((size_t)nm * Gn * Gn, 0.0); h_cumchi.assign((size_t)nm * Gn, 0.0); h_srccum.assign(Gn, 0.0);
        for (int mm = 0; mm < nm; mm++) {
            double cc = 0.0;
            for (int gg = 0; gg < Gn; gg++) {
                double cs = 0.0;
                for (int gp = 0; gp < Gn; gp++) {
                    cs += m->S[((size_t)mm * Gn + gg) * Gn + gp];
                    h_cumS[((size_t)mm * Gn + gg) * Gn + gp] = cs;
                }
                h_sig_s[mm * Gn + gg] = cs;
                cc += m->chi[mm * Gn + gg];
                h_cumchi[mm * Gn + gg] = cc;
                h_nusf[mm * Gn + gg] = m->nu[mm * Gn + gg] * m->sig_f[mm * Gn + gg];
            }
        }
        double cs = 0.0;
        for (int gg = 0; gg < Gn; gg++) { cs += s->group_pdf[gg]; h_srccum[gg] = cs; }
        if (!(cs > 0.0)) { delete p; return fail(MCDC_EINVAL, "source group pdf sums to zero"); }
        UP(L.sig_t, m->sig_t, nm * Gn); UP(L.sig_f, m->sig_f, nm * Gn); UP(L.nu, m->nu, nm * Gn);
        UP(L.sig_s, h_sig_s.data(), nm * Gn); UP(L.nusf, h_nusf.data(), nm * Gn);
        UP(L.cumS, h_cumS.data(), (size_t)nm * Gn * Gn); UP(L.cumchi, h_cumchi.data(), nm * Gn);
        UP(L.src_cum, h_srccum.data(), Gn);
        c.mg.G = Gn; c.mg.n_mat = nm; c.mg.blob = L.sig_t; c.mg.blob_doubles = (int)L.mg_doubles;
        c.mg_stage = L.mg_doubles * 8 <= MG_STAGE_MAX_BYTES ? (int)L.mg_doubles : 0;
        c.mg.sig_t = L.sig_t; c.mg.sig_s = L.sig_s; c.mg.sig_f = L.sig_f; c.mg.nu = L.nu; c.mg.nusf = L.nusf;
        c.mg.cumS = L.cumS; c.mg.cumchi = L.cumchi; c.mg.src_cum = L.src_cum;
        c.n_tally = t->n_bins * Gn;
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
    for (int b = 0; b < 2; b++) c.bank[b] = L.bank[b];
    c.fis = L.fis;
    c.stack = L.stack; c.stack_threads = (unsigned int)L.stack_threads; c.n_over = (unsigned int *)(L.err + 1);
    c.cap = (unsigned int)cap;
    c.qc = L.qc; c.flux = L.flux; c.scal = L.scal; c.counters = L.counters; c.err = L.err;
    c.tr.rec = nullptr;
    for (int k = 0; k < 3; k++) { c.src_lo[k] = s->lo[k]; c.src_hi[k] = s->hi[k]; c.src_dir[k] = s->dir[k]; }
    c.src_iso = s->isotropic; c.src_E = s->E; c.src_t = s->t;
    c.w0 = 1.0; c.k_prev = 1.0;
    p->flux_acc = L.flux_acc; p->flux_acc2 = L.flux_acc2; p->flux_cycle = L.flux_cycle;
    p->flux_copies = flux_copies_for((uint64_t)c.n_tally);
    c.flux_copy_mask = p->flux_copies - 1;
    p->part = L.part; p->sites = L.sites;
    p->trace_base = L.trace; p->trace_count = L.trace_count;
    p->tally_private = c.n_tally <= PRIVATE_TALLY_MAX;
    if (p->tally_private && (size_t)c.mg_stage * 8 + (size_t)c.geo_stage * 4 + 8 + (size_t)c.n_tally * BS * 8 > 48 * 1024)
        c.mg_stage = c.geo_stage = 0;  // 48 KB default dynamic shared memory limit
    c.flux_aggregate = c.n_tally <= AGGREGATE_TALLY_MAX ? 1 : 0;
    if (e == cudaSuccess) e = cudaMemsetAsync(L.flux, 0, sizeof(double) * c.n_tally * p->flux_copies, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.flux_acc, 0, sizeof(double) * c.n_tally, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.flux_acc2, 0, sizeof(double) * c.n_tally, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.scal, 0, 64, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.counters, 0, 8 * MCDC_N_COUNTERS, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.err, 0, 16, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(L.qc, 0, sizeof(QCount) * RING, st);
    if (e == cudaSuccess) e = cudaMallocHost((void **)&p->pin, sizeof(HostPinned));
    for (int k = 0; k < RING && e == cudaSuccess; k++) e = cudaEventCreateWithFlags(&p->ev[k], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreate(&p->t0);
    if (e == cudaSuccess) e = cudaEventCreate(&p->t1);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess && p->tally_private) {
        int bytes = c.n_tally * BS * 8;
        // opt in to > 48 KB is not needed (<= 40 KB), nothing to set
        (void)bytes;
    }
    if (e != cudaSuccess) { delete p; return fail(MCDC_ECUDA, "mcdc_create: %s", cudaGetErrorString(e)); }
    p->bank_count = 0; p->k_prev = 1.0; p->n_active = 0;
    p->k_acc = p->k_acc2 = p->leak_acc = p->leak_acc2 = 0.0;
    memset(p->host_counters, 0, sizeof p->host_counters);
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
    for (int k = 0; k < RING; k++) cudaEventDestroy(p->ev[k]);
    for (cudaEvent_t e : p->pool) cudaEventDestroy(e);
    cudaEventDestroy(p->t0); cudaEventDestroy(p->t1);
    cudaFreeHost(p->pin);
    delete p;
}

extern "C" const char *mcdc_last_error(void) { return g_err.c_str(); }

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

static int reset_run(mcdc_problem *p)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    CUDA_OK(cudaMemsetAsync(c.flux, 0, sizeof(double) * c.n_tally * p->flux_copies, st));
    CUDA_OK(cudaMemsetAsync(p->flux_acc, 0, sizeof(double) * c.n_tally, st));
    CUDA_OK(cudaMemsetAsync(p->flux_acc2, 0, sizeof(double) * c.n_tally, st));
    CUDA_OK(cudaMemsetAsync(c.counters, 0, 8 * MCDC_N_COUNTERS, st));
    CUDA_OK(cudaMemsetAsync(c.err, 0, 16, st));
    CUDA_OK(cudaMemsetAsync(c.fis.n, 0, sizeof(int) * (size_t)(p->cap + OVER_CAP), st));
    if (c.tr.rec) CUDA_OK(cudaMemsetAsync(c.tr.count, 0, sizeof(unsigned int) * c.tr.cap_slots, st));
    p->k_cycle.clear();
    p->n_active = 0;
    p->k_acc = p->k_acc2 = p->leak_acc = p->leak_acc2 = 0.0;
    memset(p->host_counters, 0, sizeof p->host_counters);
    p->k_prev = 1.0;
    p->bank_count = 0;
    p->ms_transport = 0.0;
    p->n_launches = 0;
    return 0;
}

template <bool CE, bool PRIV> static int transport_t(mcdc_problem *p, uint64_t M)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    const size_t smem_mg = CE ? 0 : (size_t)c.mg_stage * sizeof(double);
    const size_t smem_geo = (size_t)((c.geo_stage + 1) / 2) * sizeof(double);
    const size_t smem = smem_mg + smem_geo + (PRIV ? (size_t)c.n_tally * BS * sizeof(double) : 0);
    CUDA_OK(cudaMemsetAsync(c.qc, 0, sizeof(QCount) * RING, st));
    CUDA_OK(cudaMemsetAsync(c.n_over, 0, sizeof(unsigned int), st));
    uint64_t upper = M;
    long long known = -1;  // newest sweep whose counts the host has seen
    unsigned int s = 0;
    const unsigned int n0 = (unsigned int)M;
    while (upper > 0) {
        if (s > 4000000u) return fail(MCDC_ELOST, "sweep guard exceeded");
        if (p->schedule == 0 && p->tail > 0 && upper <= (uint64_t)p->tail) {
            { ProfScope ps(p, MCDC_PROF_TAIL); k_finish<CE, PRIV><<<grid_for(upper), BS, smem, st>>>(c, s, n0); }
            p->n_launches++;
            p->host_counters[13]++;
            break;
        }
        unsigned int gr = grid_for(upper);
        if (p->schedule == 0 && p->fuse > 0 && upper <= (uint64_t)p->fuse) {
            ProfScope ps(p, MCDC_PROF_FUSED);
            k_multi<CE, PRIV><<<gr, BS, smem, st>>>(c, s, n0, (unsigned int)p->fuse_segments);
            p->n_launches++;
        } else if (p->schedule == 0) {
            { ProfScope ps(p, MCDC_PROF_ADVANCE); k_advance<CE, PRIV><<<gr, BS, smem, st>>>(c, s, n0); }
            { ProfScope ps(p, MCDC_PROF_SCATTER); k_scatter<CE><<<gr, BS, smem_mg, st>>>(c, s); }
            { ProfScope ps(p, MCDC_PROF_SURFACE); k_surface<<<gr, BS, smem_geo, st>>>(c, s); }
            p->n_launches += 3;
        } else {
            { ProfScope ps(p, MCDC_PROF_SEGMENT); k_segment<CE, PRIV><<<grid_for(M), BS, smem, st>>>(c, s, n0); }
            p->n_launches++;
        }
        p->host_counters[13]++;
        CUDA_OK(cudaMemcpyAsync(&p->pin->qc[s % RING], c.qc + (s % RING), sizeof(QCount), cudaMemcpyDeviceToHost, st));
        CUDA_OK(cudaEventRecord(p->ev[s % RING], st));
        s++;
        while (known < (long long)s - 1) {
            long long r = known + 1;
            if ((long long)s - 1 - r >= LAG) CUDA_OK(cudaEventSynchronize(p->ev[r % RING]));
            else {
                cudaError_t q = cudaEventQuery(p->ev[r % RING]);
                if (q == cudaErrorNotReady) break;
                if (q != cudaSuccess) return fail(MCDC_ECUDA, "event query: %s", cudaGetErrorString(q));
            }
            const QCount &h = p->pin->qc[r % RING];
            upper = p->schedule == 0 ? (uint64_t)h.n_scat + h.n_surf : (uint64_t)h.n_alive;
            known = r;
        }
    }
    CUDA_OK(cudaGetLastError());
    return 0;
}

static int transport(mcdc_problem *p, uint64_t M)
{
    if (p->mode == 0) return p->tally_private ? transport_t<false, true>(p, M) : transport_t<false, false>(p, M);
    return p->tally_private ? transport_t<true, true>(p, M) : transport_t<true, false>(p, M);
}

// children of bank[cur] (M parents) -> bank[1-cur]; returns their number
static int emit_children(mcdc_problem *p, uint64_t M, uint64_t *total)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    unsigned int nb = (unsigned int)((M + (p->mode == 1 ? OVER_CAP : 0) + BS - 1) / BS);
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
    CUDA_OK(cudaMemcpyAsync(p->pin->scal, c.scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaMemcpyAsync(&p->pin->err, c.err, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaStreamSynchronize(st));
    CUDA_OK(cudaGetLastError());
    profile_collect(p);
    *total = p->pin->total;
    return 0;
}

static int device_error(mcdc_problem *p)
{
    int e = p->pin->err;
    if (e == -2) return fail(MCDC_EGEOM, "particle in no cell (lost)");
    if (e == -3) return fail(MCDC_EBANK, "fission / secondary bank overflow (capacity %llu)", (unsigned long long)p->cap);
    if (e == -4) return fail(MCDC_ELOST, "segment guard exceeded");
    return 0;
}

// one power-iteration cycle; source: 0 = from bank[cur] (bank_count sites), 1 = sample
static int cycle_internal(mcdc_problem *p, uint64_t N, uint32_t cycle, int active, uint64_t seed, bool sample,
                          double *flux_cycle_host)
{
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    if (N < 1 || capacity_for(N) > p->cap) return fail(MCDC_EINVAL, "n_particles %llu exceeds the capacity this problem was created for", (unsigned long long)N);
    if (cycle >= (1u << 24)) return fail(MCDC_EINVAL, "cycle index too large for the RNG counter layout");
    uint64_t M = sample ? N : p->bank_count;
    if (M == 0) return fail(MCDC_EBANK, "empty source bank");
    c.seed = seed; c.cycle = cycle;
    c.w0 = sample ? 1.0 : (double)N / (double)M;  // source renormalisation (R6)
    c.k_prev = p->k_prev;
    CUDA_OK(cudaMemsetAsync(c.scal, 0, 64, st));
    CUDA_OK(cudaEventRecord(p->t0, st));
    if (sample) {
        k_source<false><<<(unsigned int)((M + BS - 1) / BS), BS, 0, st>>>(c, (unsigned int)M);
        p->n_launches++;
    }
    int rc = transport(p, M);
    if (rc) return rc;
    uint64_t total = 0;
    rc = emit_children(p, M, &total);
    if (rc) return rc;
    CUDA_OK(cudaEventRecord(p->t1, st));
    k_accumulate<<<(c.n_tally + BS - 1) / BS, BS, 0, st>>>(c.flux, p->flux_copies, p->flux_cycle, p->flux_acc, p->flux_acc2, c.n_tally, 1.0 / (double)N, active);
    if (flux_cycle_host) CUDA_OK(cudaMemcpyAsync(flux_cycle_host, p->flux_cycle, sizeof(double) * c.n_tally, cudaMemcpyDeviceToHost, st));
    p->n_launches++;
    CUDA_OK(cudaStreamSynchronize(st));
    float ms = 0.f;
    CUDA_OK(cudaEventElapsedTime(&ms, p->t0, p->t1));
    p->ms_transport += ms;
    rc = device_error(p);
    if (rc) return rc;
    double k_c = p->pin->scal[0] / (double)N, leak = p->pin->scal[1] / (double)N;
    p->k_cycle.push_back(k_c);
    if (active) {
        p->k_acc += k_c; p->k_acc2 += k_c * k_c;
        p->leak_acc += leak; p->leak_acc2 += leak * leak;
        p->n_active++;
    }
    p->k_prev = k_c;
    p->host_counters[0] += M;
    p->host_counters[11] += total;
    if (total > p->host_counters[12]) p->host_counters[12] = total;
    p->bank_count = total;
    p->last_N = N;
    return 0;
}

extern "C" int mcdc_run_cycle(mcdc_problem *p, uint64_t N, uint32_t cycle, int32_t active, uint64_t seed, double *k_cycle)
{
    if (!p || p->mode != 0) return fail(MCDC_EINVAL, "mcdc_run_cycle needs a multi-group problem");
    if (cycle == 0) { int rc = reset_run(p); if (rc) return rc; }
    int rc = cycle_internal(p, N, cycle, active, seed, cycle == 0, nullptr);
    if (rc) return rc;
    if (k_cycle) *k_cycle = p->k_cycle.back();
    return 0;
}

extern "C" int mcdc_run_eigenvalue(mcdc_problem *p, uint64_t N, int32_t n_inactive, int32_t n_active, uint64_t seed)
{
    if (!p || p->mode != 0) return fail(MCDC_EINVAL, "mcdc_run_eigenvalue needs a multi-group problem");
    if (n_inactive < 0 || n_active < 0) return fail(MCDC_EINVAL, "cycle counts");
    int rc = reset_run(p);
    if (rc) return rc;
    for (int cyc = 0; cyc < n_inactive + n_active; cyc++) {
        rc = cycle_internal(p, N, (uint32_t)cyc, cyc >= n_inactive, seed, cyc == 0, nullptr);
        if (rc) return rc;
    }
    return 0;
}

extern "C" int mcdc_run_cycle_host(mcdc_problem *p, uint64_t N, uint32_t cycle, uint64_t seed, double k_prev,
                                   const mcdc_site *sites_in, uint64_t n_in, mcdc_site *sites_out, uint64_t max_out,
                                   uint64_t *n_out, double *flux_cycle, double *k_cycle, double *leak_cycle)
{
    if (!p || p->mode != 0) return fail(MCDC_EINVAL, "mcdc_run_cycle_host needs a multi-group problem");
    static_assert(sizeof(Site) == sizeof(mcdc_site), "site layout");
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    bool sample = sites_in == nullptr || n_in == 0;
    if (!sample && n_in > p->cap) return fail(MCDC_EBANK, "source bank larger than the capacity");
    if (cycle == 0) { int rc = reset_run(p); if (rc) return rc; }
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
    if (k_cycle) *k_cycle = p->k_cycle.back();
    if (leak_cycle) *leak_cycle = p->pin->scal[1] / (double)N;
    return 0;
}

extern "C" int mcdc_run_fixed_source(mcdc_problem *p, uint64_t N, uint64_t seed)
{
    if (!p || p->mode != 1) return fail(MCDC_EINVAL, "mcdc_run_fixed_source needs a continuous-energy problem");
    if (N < 1 || capacity_for(N) > p->cap) return fail(MCDC_EINVAL, "n_particles exceeds the capacity this problem was created for");
    Ctx &c = p->ctx;
    cudaStream_t st = p->stream;
    int rc = reset_run(p);
    if (rc) return rc;
    c.seed = seed; c.cycle = 0; c.w0 = 1.0; c.k_prev = 1.0;
    CUDA_OK(cudaMemsetAsync(c.scal, 0, 64, st));
    CUDA_OK(cudaEventRecord(p->t0, st));
    uint64_t M = N;
    k_source<true><<<(unsigned int)((M + BS - 1) / BS), BS, 0, st>>>(c, (unsigned int)M);
    p->n_launches++;
    uint64_t secondaries = 0;
    while (M > 0) {  // one wave per fission generation of the prompt chain
        rc = transport(p, M);
        if (rc) return rc;
        uint64_t total = 0;
        rc = emit_children(p, M, &total);
        if (rc) return rc;
        rc = device_error(p);
        if (rc) return rc;
        p->host_counters[0] += M;
        p->host_counters[11] += total;
        if (total > p->host_counters[12]) p->host_counters[12] = total;
        secondaries += total;
        if (secondaries > 64 * N + 4096) return fail(MCDC_EBANK, "prompt fission chain does not die out (R25)");
        M = total;
    }
    CUDA_OK(cudaEventRecord(p->t1, st));
    k_accumulate<<<(c.n_tally + BS - 1) / BS, BS, 0, st>>>(c.flux, p->flux_copies, p->flux_cycle, p->flux_acc, p->flux_acc2, c.n_tally, 1.0 / (double)N, 1);
    p->n_launches++;
    CUDA_OK(cudaStreamSynchronize(st));
    float ms = 0.f;
    CUDA_OK(cudaEventElapsedTime(&ms, p->t0, p->t1));
    p->ms_transport += ms;
    double k_c = p->pin->scal[0] / (double)N, leak = p->pin->scal[1] / (double)N;
    p->k_cycle.push_back(k_c);
    p->k_acc = k_c; p->k_acc2 = k_c * k_c; p->leak_acc = leak; p->leak_acc2 = leak * leak; p->n_active = 1;
    p->bank_count = 0;
    p->last_N = N;
    return 0;
}

// ------------------------------------------------------------------ results
extern "C" int mcdc_get_dims(const mcdc_problem *p, mcdc_dims *d)
{
    if (!p || !d) return fail(MCDC_EINVAL, "null");
    d->mode = p->mode; d->n_tally = p->ctx.n_tally; d->n_cycles = (int)p->k_cycle.size(); d->n_active = p->n_active;
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
    int n = p->n_active;
    double dn = n > 0 ? (double)n : 1.0;
    if (out->k_cycle) for (size_t i = 0; i < p->k_cycle.size(); i++) out->k_cycle[i] = p->k_cycle[i];
    out->k_mean = p->k_acc / dn; out->k_sdev = sdev_of(p->k_acc, p->k_acc2, n);
    out->leak_mean = p->leak_acc / dn; out->leak_sdev = sdev_of(p->leak_acc, p->leak_acc2, n);
    std::vector<double> a(c.n_tally), a2(c.n_tally);
    CUDA_OK(cudaMemcpyAsync(a.data(), p->flux_acc, sizeof(double) * c.n_tally, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaMemcpyAsync(a2.data(), p->flux_acc2, sizeof(double) * c.n_tally, cudaMemcpyDeviceToHost, p->stream));
    unsigned long long dc[MCDC_N_COUNTERS];
    CUDA_OK(cudaMemcpyAsync(dc, c.counters, sizeof dc, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaStreamSynchronize(p->stream));
    for (int i = 0; i < c.n_tally; i++) {
        if (out->flux_mean) out->flux_mean[i] = a[i] / dn;
        if (out->flux_sdev) out->flux_sdev[i] = sdev_of(a[i], a2[i], n);
    }
    if (out->counters) {
        for (int i = 0; i < MCDC_N_COUNTERS; i++) out->counters[i] = dc[i];
        // histories started / children made inside the tail kernel (continuous energy) are counted on the device
        out->counters[0] = p->host_counters[0] + dc[15]; out->counters[11] = p->host_counters[11] + dc[15];
        out->counters[15] = 0;
        out->counters[12] = p->host_counters[12]; out->counters[13] = p->host_counters[13];
    }
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
    if (n_ids == 0 || max_events == 0) { p->ctx.tr.rec = nullptr; return 0; }
    uint64_t per_slot = (uint64_t)max_events * sizeof(TraceRec);
    uint64_t slots = TRACE_BYTES / per_slot;
    if (slots < n_ids) return fail(MCDC_ENOMEM, "trace buffer holds %llu (id, cycle) slots of %u events; %u ids asked", (unsigned long long)slots, max_events, n_ids);
    Trace &t = p->ctx.tr;
    t.first = first_id; t.n_ids = n_ids; t.max_events = max_events;
    t.cap_slots = (unsigned int)std::min<uint64_t>(slots, TRACE_BYTES / sizeof(TraceRec));
    t.rec = p->trace_base; t.count = p->trace_count;
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
    p->prof_adv_base = b;
    memset(p->prof_ms, 0, sizeof p->prof_ms); memset(p->prof_launches, 0, sizeof p->prof_launches);
    return 0;
}

extern "C" int mcdc_get_profile(const mcdc_problem *p, double *ms, uint64_t *launches, uint64_t *advance_events)
{
    if (!p || !ms || !launches) return fail(MCDC_EINVAL, "null");
    for (int k = 0; k < MCDC_N_PROFILE; k++) { ms[k] = p->prof_ms[k]; launches[k] = p->prof_launches[k]; }
    if (advance_events) {
        unsigned long long b = 0;
        CUDA_OK(cudaMemcpy(&b, p->ctx.counters + 12, sizeof b, cudaMemcpyDeviceToHost));
        *advance_events = b - p->prof_adv_base;
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
// scratch for the test entry points is taken from the (idle) second particle bank region: sites buffer
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

extern "C" int mcdc_test_geometry(mcdc_problem *p, const double *x, const double *u, uint64_t n, int32_t *loc, double *dist,
                                  int32_t *surf)
{
    if (!p || !x || !u || !loc || !dist || !surf) return fail(MCDC_EINVAL, "null");
    if (n * 72 > p->cap * sizeof(Site)) return fail(MCDC_ENOMEM, "too many points for the scratch buffer");
    char *base = (char *)p->sites;
    double *d_x = (double *)base, *d_u = (double *)(base + n * 24), *d_d = (double *)(base + n * 48);
    int *d_loc = (int *)(base + n * 56), *d_s = (int *)(base + n * 68);
    CUDA_OK(cudaMemcpyAsync(d_x, x, n * 24, cudaMemcpyHostToDevice, p->stream));
    CUDA_OK(cudaMemcpyAsync(d_u, u, n * 24, cudaMemcpyHostToDevice, p->stream));
    k_test_geometry<<<(unsigned int)((n + 255) / 256), 256, 0, p->stream>>>(p->ctx, d_x, d_u, n, d_loc, d_d, d_s);
    CUDA_OK(cudaMemcpyAsync(loc, d_loc, n * 12, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaMemcpyAsync(dist, d_d, n * 8, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaMemcpyAsync(surf, d_s, n * 4, cudaMemcpyDeviceToHost, p->stream));
    CUDA_OK(cudaStreamSynchronize(p->stream));
    return 0;
}
