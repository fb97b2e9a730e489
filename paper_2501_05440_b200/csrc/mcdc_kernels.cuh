// mcdc_kernels.cuh -- the kernels of the event-based transport loop.
//
// Event schedule (default): per sweep three kernels regroup the live particles by next event
//   k_advance  (a2/a3 XS lookup, a5 nearest boundary, a6 distance to collision, a7 move + tallies, reaction
//               choice) reads the live particles of bank[s&1] and writes every survivor, whole, into
//               bank[(s+1)&1]: scatter events packed at the FRONT, surface / lattice / time-edge events at the
//               BACK, positions from ballot + prefix-sum compaction with one atomic per block and queue (a11);
//   k_scatter  (a8) over the front region, in place;   k_surface (a9) over the back region, in place.
// The queues are the particles themselves (PAPER.md:55 dual banks), so all bank traffic is coalesced.
// Fission and capture end a history inside k_advance; a fission leaves a record at the parent's slot and the
// children are produced at the end of the cycle by count -> exclusive scan -> write (a10/a12), which yields
// the bank sorted by (parent id, child index) without atomics or a sort.  k_segment is the paper's monolithic
// design: one whole segment for every bank slot per launch, no compaction.  k_finish ends the
// last few histories in registers.
#pragma once
#include "mcdc_device.cuh"

namespace mcdc {

#ifndef MCDC_BS
#define MCDC_BS 256
#endif
constexpr int BS = MCDC_BS;  // threads per block of every transport kernel

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ int pack_gl(int g, int last) { return (g & 0xffff) | ((last + 1) << 16); }

// ------------------------------------------------------------------ a2: multi-group tables in shared memory
// Copies the table blob to shared memory (all threads of the block; ends with a barrier) and returns the table
// descriptor rebased onto the copy; `smem` is where the copy goes, n_stage its size in doubles (0: not staged,
// the tables are then read from global memory through L1).
__device__ __forceinline__ MGTab stage_mg(const Ctx &c, double *smem, int n_stage)
{
    MGTab mg = c.mg;
    if (n_stage > 0) {
        for (int k = threadIdx.x; k < n_stage; k += blockDim.x) smem[k] = __ldg(c.mg.blob + k);
        mg.sig_t = smem + (c.mg.sig_t - c.mg.blob); mg.sig_s = smem + (c.mg.sig_s - c.mg.blob);
        mg.sig_f = smem + (c.mg.sig_f - c.mg.blob); mg.nu = smem + (c.mg.nu - c.mg.blob);
        mg.nusf = smem + (c.mg.nusf - c.mg.blob); mg.cumS = smem + (c.mg.cumS - c.mg.blob);
        mg.cumchi = smem + (c.mg.cumchi - c.mg.blob); mg.src_cum = smem + (c.mg.src_cum - c.mg.blob);
        __syncthreads();
    }
    return mg;
}

// a4/a5: the CSG tables (surfaces, cell -> surface lists, fills, bins, universes) in shared memory, same scheme;
// `smem` must be 8-byte aligned; the lattice maps stay in global memory (L1/L2)
__device__ __forceinline__ Geo stage_geo(const Ctx &c, void *smem, int n_words)
{
    Geo G = c.geo;
    if (n_words > 0) {
        int *dst = (int *)smem;
        const int *src = (const int *)c.geo.blob;
        for (int k = threadIdx.x; k < n_words; k += blockDim.x) dst[k] = __ldg(src + k);
        const char *b = c.geo.blob;
        char *d = (char *)smem;
        G.surf_param = (const double *)(d + ((const char *)c.geo.surf_param - b));
        G.surf_type = (const int *)(d + ((const char *)c.geo.surf_type - b));
        G.surf_bc = (const int *)(d + ((const char *)c.geo.surf_bc - b));
        G.cso = (const int *)(d + ((const char *)c.geo.cso - b)); G.csi = (const int *)(d + ((const char *)c.geo.csi - b));
        G.css = (const int *)(d + ((const char *)c.geo.css - b)); G.cft = (const int *)(d + ((const char *)c.geo.cft - b));
        G.cfill = (const int *)(d + ((const char *)c.geo.cfill - b)); G.cbin = (const int *)(d + ((const char *)c.geo.cbin - b));
        G.uco = (const int *)(d + ((const char *)c.geo.uco - b));
        __syncthreads();
    }
    return G;
}

// ------------------------------------------------------------------ bank access (dense, position-indexed)
template <bool CE>
__device__ __forceinline__ void load_full(const Bank &B, unsigned int i, Particle &p, uint32_t &ctr, uint32_t &slot)
{
    p.x = B.x[i]; p.y = B.y[i]; p.z = B.z[i];
    p.ux = B.ux[i]; p.uy = B.uy[i]; p.uz = B.uz[i];
    p.cell = B.cell[i]; p.elem = B.elem[i];
    int gl = B.gl[i];
    p.g = gl & 0xffff; p.last = (gl >> 16) - 1;
    ctr = B.ctr[i];
    slot = B.slot[i];
    if (CE) { p.E = B.E[i]; p.t = B.t[i]; p.tbin = B.tbin[i]; p.id = B.id[i]; }
    else { p.E = 0.0; p.t = 0.0; p.tbin = 0; p.id = slot; }
}

template <bool CE>
__device__ __forceinline__ void store_full(const Bank &B, unsigned int i, const Particle &p, uint32_t ctr, uint32_t slot,
                                           int ev)
{
    B.x[i] = p.x; B.y[i] = p.y; B.z[i] = p.z; B.ux[i] = p.ux; B.uy[i] = p.uy; B.uz[i] = p.uz;
    B.cell[i] = p.cell; B.elem[i] = p.elem; B.gl[i] = pack_gl(p.g, p.last); B.ctr[i] = ctr; B.slot[i] = slot;
    B.ev[i] = ev;
    if (CE) { B.E[i] = p.E; B.t[i] = p.t; B.tbin[i] = p.tbin; B.id[i] = p.id; }
}

// a fission ends the history: leave what k_emit needs at the parent's slot
template <bool CE>
__device__ __forceinline__ void record_fission(const Ctx &c, const Particle &p, uint32_t ctr, uint32_t slot, int n)
{
    const FisRec &F = c.fis;
    F.n[slot] = n;
    if (n <= 0) return;
    F.x[slot] = p.x; F.y[slot] = p.y; F.z[slot] = p.z;
    F.cell[slot] = p.cell; F.elem[slot] = p.elem; F.ctr[slot] = ctr;
    if (CE) { F.t[slot] = p.t; F.tbin[slot] = p.tbin; F.id[slot] = p.id; }
}

// position of live particle t of a sweep's input bank: front region first, then the back region
__device__ __forceinline__ unsigned int live_pos(unsigned int cap, unsigned int n_front, unsigned int t)
{
    return t < n_front ? t : cap - 1u - (t - n_front);
}

// per-block flush: k numerator (warp shuffles + one atomic per block) and the shared event counters
__device__ __forceinline__ void flush_acc(const Ctx &c, const Acc &acc)
{
    __shared__ double s_k[BS / 32];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double k = warp_sum(acc.knum);
    if (lane == 0) s_k[w] = k;
    __syncthreads();
    if (threadIdx.x == 0) {
        double ks = 0.0;
        for (int i = 0; i < BS / 32; i++) ks += s_k[i];
        if (ks != 0.0) atomicAdd(c.scal + 0, ks);
    }
    if (threadIdx.x >= 1 && threadIdx.x < 11 && acc.s_ev[threadIdx.x])
        atomicAdd(c.counters + threadIdx.x, (unsigned long long)acc.s_ev[threadIdx.x]);
}

// block-shared event counters: declare + clear (call at kernel start, before any event is counted)
#define MCDC_EVENT_COUNTERS(acc)                         \
    __shared__ unsigned int s_evc[16];                   \
    if (threadIdx.x < 16) s_evc[threadIdx.x] = 0u;       \
    __syncthreads();                                     \
    Acc acc;                                             \
    acc.clear(s_evc)

// shared-memory tally columns (one per thread) -> one float64 atomic per bin and block
__device__ __forceinline__ void flush_private_flux(const Ctx &c, const double *s_flux)
{
    __syncthreads();
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int b = w; b < c.n_tally; b += BS / 32) {
        double v = 0.0;
        for (int t = lane; t < BS; t += 32) v += s_flux[b * BS + t];
        v = warp_sum(v);
        if (lane == 0 && v != 0.0) atomicAdd(c.flux + (size_t)(blockIdx.x & c.flux_copy_mask) * c.n_tally + b, v);
    }
}

// ballot + prefix-sum compaction (a11): output position of this thread's particle in the next bank, front
// region for scatter events, back region for surface events; one atomic per block and region.
// `par` alternates 0/1 between consecutive calls of a block: two scratch sets make two barriers per call enough.
__device__ __forceinline__ unsigned int block_slot(bool to_front, bool to_back, QCount *oc, unsigned int cap, int par)
{
    __shared__ unsigned int s_n[2][2][BS / 32];
    __shared__ unsigned int s_base[2][2];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned int mf = __ballot_sync(0xffffffffu, to_front), mb = __ballot_sync(0xffffffffu, to_back);
    if (lane == 0) { s_n[par][0][w] = __popc(mf); s_n[par][1][w] = __popc(mb); }
    __syncthreads();
    if (threadIdx.x < 2) {  // exclusive prefix over the warps, then the block's base in the region
        unsigned int tot = 0;
#pragma unroll
        for (int i = 0; i < BS / 32; i++) { unsigned int n = s_n[par][threadIdx.x][i]; s_n[par][threadIdx.x][i] = tot; tot += n; }
        s_base[par][threadIdx.x] = tot ? atomicAdd(threadIdx.x == 0 ? &oc->n_scat : &oc->n_surf, tot) : 0u;
    }
    __syncthreads();
    unsigned int lt = (1u << lane) - 1u;
    unsigned int pos = 0xffffffffu;
    if (to_front || to_back) {
        int q = to_front ? 0 : 1;
        unsigned int off = s_base[par][q] + s_n[par][q][w] + __popc((to_front ? mf : mb) & lt);
        pos = to_front ? off : cap - 1u - off;
    }
    return pos;
}

// same with a COUNT of back-region slots per thread (a continuous-energy fission puts its n children, alive, into
// the next bank: secondaries carry their own id-keyed streams, so they simply join the running population)
__device__ __forceinline__ void block_slot_n(bool to_front, unsigned int n_back, QCount *oc, unsigned int cap, int par,
                                             unsigned int &pos_front, unsigned int &off_back)
{
    __shared__ unsigned int s_n[2][2][BS / 32];
    __shared__ unsigned int s_base[2][2];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned int mf = __ballot_sync(0xffffffffu, to_front);
    unsigned int incl = n_back;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) { s_n[par][0][w] = __popc(mf); s_n[par][1][w] = incl; }
    __syncthreads();
    if (threadIdx.x < 2) {
        unsigned int tot = 0;
#pragma unroll
        for (int i = 0; i < BS / 32; i++) { unsigned int n = s_n[par][threadIdx.x][i]; s_n[par][threadIdx.x][i] = tot; tot += n; }
        s_base[par][threadIdx.x] = tot ? atomicAdd(threadIdx.x == 0 ? &oc->n_scat : &oc->n_surf, tot) : 0u;
    }
    __syncthreads();
    pos_front = s_base[par][0] + s_n[par][0][w] + __popc(mf & ((1u << lane) - 1u));
    off_back = s_base[par][1] + s_n[par][1][w] + incl - n_back;  // slot k of this thread = cap - 1 - (off_back + k)
}

// ------------------------------------------------------------------ a1: source
template <bool CE>
__global__ void __launch_bounds__(BS) k_source(Ctx c, unsigned int n)
{
    unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Bank &B = c.bank[0];
    Rng rng;
    rng.init(c.seed, i, 0u, c.cycle, 0u);
    double xi[6];
#pragma unroll
    for (int k = 0; k < 6; k++) xi[k] = rng.next();  // always six draws
    Particle p;
    p.x = c.src_lo[0] + xi[0] * (c.src_hi[0] - c.src_lo[0]);
    p.y = c.src_lo[1] + xi[1] * (c.src_hi[1] - c.src_lo[1]);
    p.z = c.src_lo[2] + xi[2] * (c.src_hi[2] - c.src_lo[2]);
    p.ux = c.src_dir[0]; p.uy = c.src_dir[1]; p.uz = c.src_dir[2];
    if (c.src_iso) iso_dir(xi[3], xi[4], p.ux, p.uy, p.uz);
    p.g = 0;
    if (!CE) p.g = pick(c.mg.src_cum, c.mg.G, xi[5] * __ldg(c.mg.src_cum + c.mg.G - 1));
    if (!locate(c.geo, p.x, p.y, p.z, p.ux, p.uy, p.uz, -1, p.cell, p.elem)) { atomicExch(c.err, -2); p.cell = -1; }
    p.last = -1; p.id = i;
    p.E = c.src_E; p.t = c.src_t; p.tbin = 0;
    if (CE) p.tbin = edge_bin(c.ce.t_edges, c.ce.n_t, c.src_t);
    store_full<CE>(B, i, p, 6u, i, p.cell < 0 ? EV_DEAD : 0);
    c.fis.n[i] = 0;
}

struct Site { double x, y, z, ux, uy, uz; int g, pad; };

// source particles from a bank of sites handed in by the host (no draws at birth)
__global__ void __launch_bounds__(BS) k_load_sites(Ctx c, const Site *sites, unsigned int n)
{
    unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Site s = sites[i];
    Particle p;
    p.x = s.x; p.y = s.y; p.z = s.z; p.ux = s.ux; p.uy = s.uy; p.uz = s.uz; p.g = s.g; p.last = -1; p.id = i;
    p.E = 0.0; p.t = 0.0; p.tbin = 0;
    if (!locate(c.geo, p.x, p.y, p.z, p.ux, p.uy, p.uz, -1, p.cell, p.elem)) { atomicExch(c.err, -2); p.cell = -1; }
    store_full<false>(c.bank[0], i, p, 0u, i, p.cell < 0 ? EV_DEAD : 0);
    c.fis.n[i] = 0;
}

__global__ void __launch_bounds__(BS) k_store_sites(Ctx c, Site *sites, unsigned int n)
{
    unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Bank &B = c.bank[0];
    Site s;
    s.x = B.x[i]; s.y = B.y[i]; s.z = B.z[i]; s.ux = B.ux[i]; s.uy = B.uy[i]; s.uz = B.uz[i];
    s.g = B.gl[i] & 0xffff; s.pad = 0;
    sites[i] = s;
}

// child j of a fission at the parent's site, drawn from the parent's stream (R5).  MG: group ~ chi and an
// isotropic direction (1 + 2 draws).  CE: Watt energy (4 draws) + direction (2 draws), own id from the domain-1
// block keyed by (parent id, parent draw counter after the multiplicity draw, j) (R10).
template <bool CE>
__device__ __forceinline__ void make_child(const Ctx &c, Rng &rng, int mat, unsigned long long pid, uint32_t ctr0, int j,
                                           Particle &p)
{
    if (!CE) {
        const double *cc = c.mg.cumchi + (size_t)mat * c.mg.G;
        p.g = pick(cc, c.mg.G, rng.next() * __ldg(cc + c.mg.G - 1));
        double a = rng.next(), b = rng.next();
        iso_dir(a, b, p.ux, p.uy, p.uz);
    } else {
        double a1 = rng.next(), a2 = rng.next(), a3 = rng.next(), a4 = rng.next();
        double En = 1e6 * watt(c.ce.watt_a, c.ce.watt_b, a1, a2, a3, a4);
        if (En < c.ce.E_min) En = c.ce.E_min;
        if (En > c.ce.E_max) En = c.ce.E_max;
        double a = rng.next(), b = rng.next();
        iso_dir(a, b, p.ux, p.uy, p.uz);
        p.E = En;
        p.id = child_id(c.seed, pid, ctr0, (uint32_t)j);
    }
    p.last = -1;
}

// ------------------------------------------------------------------ per-event kernels
#ifndef MCDC_ADV_MINBLOCKS
#define MCDC_ADV_MINBLOCKS 4  // measured on B200: 2 -> 30.2, 3 -> 25.2, 4 -> 22.5, 5 -> 24.1 ms of k_advance per C4 cycle
#endif
template <bool CE, bool PRIVATE>
__global__ void __launch_bounds__(BS, MCDC_ADV_MINBLOCKS * 256 / BS) k_advance(Ctx c, unsigned int s, unsigned int n0)
{
    extern __shared__ double s_dyn[];
    const MGTab mg = stage_mg(c, s_dyn, CE ? 0 : c.mg_stage);
    const Geo geo = stage_geo(c, s_dyn + (CE ? 0 : c.mg_stage), c.geo_stage);
    double *s_flux = s_dyn + (CE ? 0 : c.mg_stage) + (c.geo_stage + 1) / 2;
    unsigned int n_front = n0, n_in = n0;
    if (s > 0) {
        QCount pc = c.qc[(s - 1) % RING];
        n_front = pc.n_scat; n_in = pc.n_scat + pc.n_surf;
    }
    QCount *oc = c.qc + (s % RING);
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(c.counters + 12, (unsigned long long)n_in);  // events of k_advance
    if (PRIVATE) {
        for (int k = threadIdx.x; k < c.n_tally * BS; k += BS) s_flux[k] = 0.0;
        __syncthreads();
    }
    MCDC_EVENT_COUNTERS(acc);
    const Bank &B = c.bank[s & 1];
    const Bank &O = c.bank[(s + 1) & 1];
    int par = 0;
    for (unsigned int base = blockIdx.x * BS; base < n_in; base += gridDim.x * BS, par ^= 1) {
        unsigned int t = base + threadIdx.x;
        int code = ADV_DEAD, aux = 0;
        Particle p;
        uint32_t ctr = 0, slot = 0;
        Rng rng;
        if (t < n_in) {
            unsigned int i = live_pos(c.cap, n_front, t);
            if (B.cell[i] >= 0) {
                load_full<CE>(B, i, p, ctr, slot);
                rng.init(c.seed, p.id, 0u, c.cycle, ctr);
                code = advance<CE, PRIVATE>(c, mg, p, rng, aux, acc, s_flux, geo);
                if (!CE && code == ADV_FISSION) { record_fission<CE>(c, p, rng.ctr, slot, aux); code = ADV_DEAD; }
            }
        }
        if (!CE) {
            unsigned int o = block_slot(code == ADV_SCATTER, code == ADV_SURFACE, oc, c.cap, par);
            if (code != ADV_DEAD) store_full<CE>(O, o, p, rng.ctr, slot, aux);
        } else {
            unsigned int nb = code == ADV_SURFACE ? 1u : (code == ADV_FISSION ? (unsigned int)aux : 0u);
            unsigned int pf, ob;
            block_slot_n(code == ADV_SCATTER, nb, oc, c.cap, par, pf, ob);
            if (code == ADV_SCATTER) { if (pf < c.cap) store_full<CE>(O, pf, p, rng.ctr, slot, aux); }
            else if (code == ADV_SURFACE) { if (ob < c.cap) store_full<CE>(O, c.cap - 1u - ob, p, rng.ctr, slot, aux); }
            else if (code == ADV_FISSION && nb) {
                // prompt secondaries: born alive at the parent's site, first segment in the next sweep
                const int mat = c.geo.cfill[p.cell];
                const unsigned long long pid = p.id;
                const uint32_t ctr0 = rng.ctr;
                for (unsigned int j = 0; j < nb; j++) {
                    make_child<CE>(c, rng, mat, pid, ctr0, (int)j, p);
                    if (ob + j < c.cap) store_full<CE>(O, c.cap - 1u - (ob + j), p, 0u, slot, HIT_NEWBORN);
                }
                atomicAdd(c.counters + 15, (unsigned long long)nb);
            }
        }
    }
    if (PRIVATE) flush_private_flux(c, s_flux);
    flush_acc(c, acc);
}

template <bool CE>
__global__ void __launch_bounds__(BS) k_scatter(Ctx c, unsigned int s)
{
    extern __shared__ double s_dyn[];
    const MGTab mg = stage_mg(c, s_dyn, CE ? 0 : c.mg_stage);
    const QCount oc = c.qc[s % RING];
    const Bank &B = c.bank[(s + 1) & 1];
    // queue-counter housekeeping: clear the set the next sweep appends to
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        QCount z = {0u, 0u, 0u, 0u};
        c.qc[(s + 1) % RING] = z;
        if ((unsigned long long)oc.n_scat + oc.n_surf > c.cap) atomicExch(c.err, -3);  // the two regions met
    }
    for (unsigned int i = blockIdx.x * BS + threadIdx.x; i < oc.n_scat && i < c.cap; i += gridDim.x * BS) {
        Particle p;
        int gl = B.gl[i];
        p.g = gl & 0xffff;
        p.cell = B.cell[i];
        p.id = CE ? B.id[i] : (unsigned long long)B.slot[i];
        if (CE) { p.E = B.E[i]; p.ux = B.ux[i]; p.uy = B.uy[i]; p.uz = B.uz[i]; }
        Rng rng;
        rng.init(c.seed, p.id, 0u, c.cycle, B.ctr[i]);
        do_scatter<CE>(c, mg, p, rng, B.ev[i], c.geo);
        B.ux[i] = p.ux; B.uy[i] = p.uy; B.uz[i] = p.uz;
        B.gl[i] = pack_gl(p.g, -1);
        B.ctr[i] = rng.ctr;
        if (CE) B.E[i] = p.E;
    }
}

__global__ void __launch_bounds__(BS) k_surface(Ctx c, unsigned int s)
{
    extern __shared__ double s_dyn[];
    const Geo geo = stage_geo(c, s_dyn, c.geo_stage);
    const QCount oc = c.qc[s % RING];
    const Bank &B = c.bank[(s + 1) & 1];
    for (unsigned int t = blockIdx.x * BS + threadIdx.x; t < oc.n_surf; t += gridDim.x * BS) {
        unsigned int i = c.cap - 1u - t;
        int hit = B.ev[i];
        if (hit == HIT_TIME_EDGE || hit == HIT_NEWBORN) continue;
        Particle p;
        p.x = B.x[i]; p.y = B.y[i]; p.z = B.z[i];
        p.ux = B.ux[i]; p.uy = B.uy[i]; p.uz = B.uz[i];
        p.cell = B.cell[i]; p.elem = B.elem[i];
        int gl = B.gl[i];
        p.g = gl & 0xffff; p.last = (gl >> 16) - 1;
        const int cell0 = p.cell, elem0 = p.elem;
        const double ux0 = p.ux, uy0 = p.uy, uz0 = p.uz;
        if (!do_surface(geo, p, hit)) {
            atomicExch(c.err, -2);
            atomicAdd(c.counters + 10, 1ull);
            p.cell = -1;
        }
        if (p.cell != cell0) B.cell[i] = p.cell;
        if (p.elem != elem0) B.elem[i] = p.elem;
        B.gl[i] = pack_gl(p.g, p.last);
        if (p.ux != ux0) B.ux[i] = p.ux;
        if (p.uy != uy0) B.uy[i] = p.uy;
        if (p.uz != uz0) B.uz[i] = p.uz;
    }
}

// whole segment in registers (shared by the monolithic schedule and the tail kernel):
// returns 1 = still alive, 0 = history ended, 2 = ended in a fission with n_children
template <bool CE, bool PRIVATE>
__device__ __forceinline__ int segment(const Ctx &c, const MGTab &mg, const Geo &G, Particle &p, Rng &rng, Acc &acc,
                                       double *s_flux, int &n_children)
{
    int aux = 0;
    int code = advance<CE, PRIVATE>(c, mg, p, rng, aux, acc, s_flux, G);
    if (code == ADV_SCATTER) { do_scatter<CE>(c, mg, p, rng, aux, G); return 1; }
    if (code == ADV_SURFACE) {
        if (!do_surface(G, p, aux)) {
            atomicExch(c.err, -2);
            atomicAdd(c.counters + 10, 1ull);
            p.cell = -1;
            return 0;
        }
        return 1;
    }
    if (code == ADV_FISSION) { n_children = aux; return 2; }
    return 0;
}

// Fused sweep for a thinned-out population: up to max_seg whole segments per particle in registers, then the same
// ballot / prefix-sum compaction of the survivors into the next bank (front region; continuous-energy fission
// children go, alive, to the back region).  One launch replaces 3 * max_seg launches of the per-event kernels
// when a sweep is launch-latency bound; divergence is irrelevant at these sizes.
#ifndef MCDC_MULTI_MINBLOCKS
#define MCDC_MULTI_MINBLOCKS 3  // measured: 2 -> 11.4, 3 -> 9.7, 4 -> 9.6 ms of fused sweeps per C4 cycle
#endif
#ifndef MCDC_MULTI_MINBLOCKS_CE
#define MCDC_MULTI_MINBLOCKS_CE 3
#endif
template <bool CE, bool PRIVATE>
__global__ void __launch_bounds__(BS, (CE ? MCDC_MULTI_MINBLOCKS_CE : MCDC_MULTI_MINBLOCKS) * 256 / BS) k_multi(Ctx c, unsigned int s, unsigned int n0, unsigned int max_seg)
{
    extern __shared__ double s_dyn[];
    const MGTab mg = stage_mg(c, s_dyn, CE ? 0 : c.mg_stage);
    const Geo geo = stage_geo(c, s_dyn + (CE ? 0 : c.mg_stage), c.geo_stage);
    double *s_flux = s_dyn + (CE ? 0 : c.mg_stage) + (c.geo_stage + 1) / 2;
    unsigned int n_front = n0, n_in = n0;
    if (s > 0) {
        QCount pc = c.qc[(s - 1) % RING];
        n_front = pc.n_scat; n_in = pc.n_scat + pc.n_surf;
    }
    QCount *oc = c.qc + (s % RING);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        QCount z = {0u, 0u, 0u, 0u};
        c.qc[(s + 1) % RING] = z;
        if (n_in > c.cap) atomicExch(c.err, -3);
    }
    if (PRIVATE) {
        for (int k = threadIdx.x; k < c.n_tally * BS; k += BS) s_flux[k] = 0.0;
        __syncthreads();
    }
    MCDC_EVENT_COUNTERS(acc);
    const Bank &B = c.bank[s & 1];
    const Bank &O = c.bank[(s + 1) & 1];
    int par = 0;
    for (unsigned int base = blockIdx.x * BS; base < n_in; base += gridDim.x * BS, par ^= 1) {
        unsigned int t = base + threadIdx.x;
        int st = 0, nch = 0;
        Particle p;
        uint32_t ctr = 0, slot = 0;
        Rng rng;
        if (t < n_in && t < c.cap) {
            unsigned int i = live_pos(c.cap, n_front, t);
            if (B.cell[i] >= 0) {
                load_full<CE>(B, i, p, ctr, slot);
                rng.init(c.seed, p.id, 0u, c.cycle, ctr);
                unsigned int k = 0;
                do { st = segment<CE, PRIVATE>(c, mg, geo, p, rng, acc, s_flux, nch); } while (st == 1 && ++k < max_seg);
                if (!CE && st == 2) record_fission<CE>(c, p, rng.ctr, slot, nch);
            }
        }
        unsigned int nb = (CE && st == 2) ? (unsigned int)nch : 0u;
        unsigned int pf, ob;
        block_slot_n(st == 1, nb, oc, c.cap, par, pf, ob);
        if (st == 1) { if (pf < c.cap) store_full<CE>(O, pf, p, rng.ctr, slot, 0); }
        else if (nb) {
            const int mat = c.geo.cfill[p.cell];
            const unsigned long long pid = p.id;
            const uint32_t ctr0 = rng.ctr;
            for (unsigned int j = 0; j < nb; j++) {
                make_child<CE>(c, rng, mat, pid, ctr0, (int)j, p);
                if (ob + j < c.cap) store_full<CE>(O, c.cap - 1u - (ob + j), p, 0u, slot, HIT_NEWBORN);
            }
            atomicAdd(c.counters + 15, (unsigned long long)nb);
        }
    }
    if (PRIVATE) flush_private_flux(c, s_flux);
    flush_acc(c, acc);
}

// monolithic schedule: every slot of bank 0, one segment, no compaction; counts the survivors
template <bool CE, bool PRIVATE>
__global__ void __launch_bounds__(BS) k_segment(Ctx c, unsigned int s, unsigned int n)
{
    extern __shared__ double s_dyn[];
    const MGTab mg = stage_mg(c, s_dyn, CE ? 0 : c.mg_stage);
    const Geo geo = stage_geo(c, s_dyn + (CE ? 0 : c.mg_stage), c.geo_stage);
    double *s_flux = s_dyn + (CE ? 0 : c.mg_stage) + (c.geo_stage + 1) / 2;
    if (PRIVATE) {
        for (int k = threadIdx.x; k < c.n_tally * BS; k += BS) s_flux[k] = 0.0;
        __syncthreads();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        QCount z = {0u, 0u, 0u, 0u};
        c.qc[(s + 1) % RING] = z;
    }
    MCDC_EVENT_COUNTERS(acc);
    const Bank &B = c.bank[0];
    unsigned int alive = 0;
    for (unsigned int i = blockIdx.x * BS + threadIdx.x; i < n; i += gridDim.x * BS) {
        if (B.ev[i] == EV_DEAD) continue;
        Particle p;
        uint32_t ctr, slot;
        load_full<CE>(B, i, p, ctr, slot);
        Rng rng;
        rng.init(c.seed, p.id, 0u, c.cycle, ctr);
        int nch = 0;
        int st = segment<CE, PRIVATE>(c, mg, geo, p, rng, acc, s_flux, nch);
        if (st == 2) record_fission<CE>(c, p, rng.ctr, slot, nch);
        store_full<CE>(B, i, p, rng.ctr, slot, st == 1 ? 0 : EV_DEAD);
        if (st == 1) alive++;
    }
    alive = __reduce_add_sync(0xffffffffu, alive);
    if ((threadIdx.x & 31) == 0 && alive) atomicAdd(&c.qc[s % RING].n_alive, alive);
    if (PRIVATE) flush_private_flux(c, s_flux);
    flush_acc(c, acc);
}

// tail: finish the few remaining histories of the live regions inside one kernel
template <bool CE, bool PRIVATE>
__global__ void __launch_bounds__(BS) k_finish(Ctx c, unsigned int s, unsigned int n0)
{
    extern __shared__ double s_dyn[];
    const MGTab mg = stage_mg(c, s_dyn, CE ? 0 : c.mg_stage);
    const Geo geo = stage_geo(c, s_dyn + (CE ? 0 : c.mg_stage), c.geo_stage);
    double *s_flux = s_dyn + (CE ? 0 : c.mg_stage) + (c.geo_stage + 1) / 2;
    if (PRIVATE) {
        for (int k = threadIdx.x; k < c.n_tally * BS; k += BS) s_flux[k] = 0.0;
        __syncthreads();
    }
    unsigned int n_front = n0, n_in = n0;
    if (s > 0) {
        QCount pc = c.qc[(s - 1) % RING];
        n_front = pc.n_scat; n_in = pc.n_scat + pc.n_surf;
    }
    MCDC_EVENT_COUNTERS(acc);
    const Bank &B = c.bank[s & 1];
    unsigned int done = 0, born = 0, pops = 0;
    for (unsigned int t = blockIdx.x * BS + threadIdx.x; t < n_in; t += gridDim.x * BS) {
        unsigned int i = live_pos(c.cap, n_front, t);
        if (B.cell[i] < 0) continue;
        Particle p;
        uint32_t ctr, slot;
        load_full<CE>(B, i, p, ctr, slot);
        Rng rng;
        rng.init(c.seed, p.id, 0u, c.cycle, ctr);
        unsigned int guard = 0, depth = 0;
        StackRec *stk = CE ? c.stack + (size_t)(blockIdx.x * BS + threadIdx.x) * STACK_DEPTH : nullptr;
        for (;;) {
            int nch = 0, st;
            while ((st = segment<CE, PRIVATE>(c, mg, geo, p, rng, acc, s_flux, nch)) == 1) {
                if (++guard > 1000000u) { atomicExch(c.err, -4); atomicAdd(c.counters + 10, 1ull); break; }  // R11 guard
            }
            done++;
            if (st == 2) {
                if (!CE) record_fission<CE>(c, p, rng.ctr, slot, nch);
                else if (nch > 0) {
                    if (depth + (unsigned int)nch <= STACK_DEPTH) {
                        const int mat = c.geo.cfill[p.cell];
                        const unsigned long long pid = p.id;
                        const uint32_t ctr0 = rng.ctr;
                        Particle ch = p;
                        for (int j = 0; j < nch; j++) {
                            make_child<CE>(c, rng, mat, pid, ctr0, j, ch);
                            StackRec r;
                            r.x = ch.x; r.y = ch.y; r.z = ch.z; r.ux = ch.ux; r.uy = ch.uy; r.uz = ch.uz; r.E = ch.E; r.t = ch.t;
                            r.cell = ch.cell; r.elem = ch.elem; r.tbin = ch.tbin; r.pad = 0; r.id = ch.id;
                            stk[depth++] = r;
                        }
                        born += (unsigned int)nch;
                    } else {  // stack full: an ordinary fission record in the overflow region, next wave
                        unsigned int k = atomicAdd(c.n_over, 1u);
                        if (k < OVER_CAP) record_fission<CE>(c, p, rng.ctr, n0 + k, nch);
                        else atomicExch(c.err, -3);
                    }
                }
            }
            if (!CE || depth == 0) break;
            if (++pops > 4000000u) { atomicExch(c.err, -3); break; }  // R25a: diverging chain
            StackRec r = stk[--depth];
            p.x = r.x; p.y = r.y; p.z = r.z; p.ux = r.ux; p.uy = r.uy; p.uz = r.uz; p.E = r.E; p.t = r.t;
            p.cell = r.cell; p.elem = r.elem; p.tbin = r.tbin; p.id = r.id; p.last = -1; p.g = 0;
            rng.init(c.seed, p.id, 0u, c.cycle, 0u);
            guard = 0;
        }
    }
    done = __reduce_add_sync(0xffffffffu, done);
    born = __reduce_add_sync(0xffffffffu, born);
    if ((threadIdx.x & 31) == 0 && done) atomicAdd(c.counters + 14, (unsigned long long)done);
    if ((threadIdx.x & 31) == 0 && born) atomicAdd(c.counters + 15, (unsigned long long)born);
    if (PRIVATE) flush_private_flux(c, s_flux);
    flush_acc(c, acc);
}

// ------------------------------------------------------------------ a10/a12: fission bank by count-scan-write
// number of fission-record slots of the running wave: its M particles plus the overflow records
__device__ __forceinline__ unsigned int record_count(const Ctx &c, unsigned int m)
{
    unsigned int k = *c.n_over;
    return m + (k < OVER_CAP ? k : OVER_CAP);
}

__global__ void __launch_bounds__(BS) k_scan_partial(Ctx c, unsigned int m, unsigned int *part)
{
    __shared__ unsigned int s_w[BS / 32];
    const unsigned int n = record_count(c, m);
    unsigned int i = blockIdx.x * BS + threadIdx.x;
    unsigned int v = i < n ? (unsigned int)c.fis.n[i] : 0u;
    v = __reduce_add_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int t = 0;
        for (int k = 0; k < BS / 32; k++) t += s_w[k];
        part[blockIdx.x] = t;
    }
}

// exclusive scan of the per-block counts by one block; total -> part[nb]
__global__ void __launch_bounds__(1024) k_scan_top(unsigned int *part, unsigned int nb)
{
    __shared__ unsigned int s_sum[1024];
    unsigned int per = (nb + 1023u) / 1024u;
    unsigned int lo = threadIdx.x * per, hi = lo + per < nb ? lo + per : nb;
    unsigned int t = 0;
    for (unsigned int k = lo; k < hi; k++) t += part[k];
    s_sum[threadIdx.x] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int run = 0;
        for (int k = 0; k < 1024; k++) { unsigned int v = s_sum[k]; s_sum[k] = run; run += v; }
        part[nb] = run;
    }
    __syncthreads();
    unsigned int run = s_sum[threadIdx.x];
    for (unsigned int k = lo; k < hi; k++) { unsigned int v = part[k]; part[k] = run; run += v; }
}

// every fission parent writes its children into bank 0 at [offset(parent), +n): sorted by (parent id, child
// index) by construction.  MG: child group ~ chi, isotropic direction (1 + 2 draws per child) from the parent's
// stream (R5).  CE: Watt energy (4 draws) + direction (2 draws), own id from the domain-1 block (R10).
// The children's fission counts are cleared through a second array (nn) because n is still being read.
template <bool CE>
__global__ void __launch_bounds__(BS) k_emit(Ctx c, unsigned int m, const unsigned int *part, unsigned int cap)
{
    __shared__ unsigned int s_w[BS / 32];
    const FisRec &F = c.fis;
    const Bank &O = c.bank[0];
    const unsigned int n = record_count(c, m);
    unsigned int i = blockIdx.x * BS + threadIdx.x;
    int nc = i < n ? F.n[i] : 0;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned int incl = (unsigned int)nc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) s_w[w] = incl;
    __syncthreads();
    unsigned int wbase = 0;
    for (int k = 0; k < w; k++) wbase += s_w[k];
    unsigned int off = part[blockIdx.x] + wbase + incl - (unsigned int)nc;
    if (nc <= 0) return;
    if (off + (unsigned int)nc > cap) { atomicExch(c.err, -3); return; }  // bank overflow (R6)
    Particle p;
    p.x = F.x[i]; p.y = F.y[i]; p.z = F.z[i];
    p.cell = F.cell[i]; p.elem = F.elem[i];
    p.last = -1; p.g = 0; p.E = 0.0; p.t = 0.0; p.tbin = 0; p.id = 0;
    if (CE) { p.t = F.t[i]; p.tbin = F.tbin[i]; }
    const int mat = c.geo.cfill[p.cell];
    unsigned long long pid = CE ? F.id[i] : (unsigned long long)i;
    uint32_t ctr0 = F.ctr[i];
    Rng rng;
    rng.init(c.seed, pid, 0u, c.cycle, ctr0);
    for (int j = 0; j < nc; j++) {
        make_child<CE>(c, rng, mat, pid, ctr0, j, p);
        store_full<CE>(O, off + j, p, 0u, off + j, 0);
    }
}

__global__ void __launch_bounds__(BS) k_clear_counts(Ctx c, unsigned int m)
{
    unsigned int i = blockIdx.x * BS + threadIdx.x;
    if (i < record_count(c, m)) c.fis.n[i] = 0;
}

// cycle end: per-source-particle flux into the running mean / mean-square, clear the per-cycle tally (R17)
__global__ void __launch_bounds__(BS) k_accumulate(double *flux, int copies, double *flux_cycle, double *acc, double *acc2,
                                                   int n_tally, double inv_n, int active)
{
    int i = blockIdx.x * BS + threadIdx.x;
    if (i >= n_tally) return;
    double f = 0.0;
    for (int r = 0; r < copies; r++) {  // the replicated per-cycle tally (see flux_add)
        f += flux[(size_t)r * n_tally + i];
        flux[(size_t)r * n_tally + i] = 0.0;
    }
    f *= inv_n;
    flux_cycle[i] = f;
    if (active) { acc[i] += f; acc2[i] += f * f; }
}

// ------------------------------------------------------------------ unit-level test kernels
__global__ void k_test_draws(unsigned long long seed, uint32_t domain, uint32_t cycle, const unsigned long long *id,
                             const uint32_t *draw, unsigned long long n, double *out)
{
    unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    Rng rng;
    rng.init(seed, id[i], domain, cycle, draw[i]);
    out[i] = rng.next();
}

__global__ void k_test_grid(Ctx c, const double *E, unsigned long long n, int *ob, int *oh)
{
    unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    ob[i] = grid_index_binary(c.ce, E[i]);
    oh[i] = grid_index_hash(c.ce, E[i]);
}

__global__ void k_test_geometry(Ctx c, const double *x, const double *u, unsigned long long n, int *loc, double *dist,
                                int *surf)
{
    unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    int cell, elem, hit = -1;
    bool ok = locate(c.geo, x[3 * i], x[3 * i + 1], x[3 * i + 2], u[3 * i], u[3 * i + 1], u[3 * i + 2], -1, cell, elem);
    double d = -1.0;
    if (ok) d = nearest(c.geo, x[3 * i], x[3 * i + 1], x[3 * i + 2], u[3 * i], u[3 * i + 1], u[3 * i + 2], cell, elem, -1, hit);
    loc[3 * i] = !ok ? -1 : (elem >= 0 ? c.geo.lat_cell : cell);
    loc[3 * i + 1] = ok ? elem : -1;
    loc[3 * i + 2] = ok && elem >= 0 ? cell : -1;
    dist[i] = d;
    surf[i] = hit;
}

}  // namespace mcdc
