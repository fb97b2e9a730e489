// mcdc_kernels.cuh -- the kernels of the event-based transport loop.
//
// A banked particle carries the event it is waiting on (Bank::ev: scatter, surface / lattice wall, time edge or
// nothing).  Event schedule (default), one kernel per sweep while the population is large:
//   k_sweep    reads the live particles of bank[s&1] -- scatter-pending ones are packed at the FRONT, surface-pending
//              ones at the BACK, so warps are homogeneous in the event they finish -- finishes that event (a8 / a9),
//              then runs the next segment up to its event decision (a2/a3 XS lookup, a5 nearest boundary, a6 distance
//              to collision, a7 move + tallies, reaction choice) and writes every survivor, whole, into
//              bank[(s+1)&1]: front or back by its new pending event, positions from ballot + prefix-sum compaction
//              with one atomic per block and queue (a11).  The queues are the particles themselves (PAPER.md:55
//              dual banks), so all bank traffic is coalesced.
//   k_persist  (PAPER.md:49 asynchronous scheduling) takes over when the population is thin: a persistent grid whose
//              warps pull particles from a global cursor, run whole segments in registers and refill dead lanes from
//              the queue; continuous-energy fission secondaries are pushed to the queue's tail for any warp to take.
// k_scatter / k_surface finish the pending events of one region in place (schedule 2: split per-event kernels, kept
// for the comparison).  Fission and capture end a history inside the segment; a multi-group fission leaves a record
// at the parent's slot and the children are produced at the end of the cycle by count -> exclusive scan -> write
// (a10/a12), which yields the bank sorted by (parent id, child index) without atomics or a sort.  k_segment is the
// paper's monolithic design: one whole segment for every bank slot per launch, no compaction.
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
// Copies the table blob to shared memory (all threads of the block; ends with a barrier) and returns the base the
// kernel reads the tables from: the copy, or the global blob when it does not fit (n_stage = 0).
__device__ __forceinline__ const double *stage_mg(const Ctx &c, double *smem, int n_stage)
{
    if (n_stage <= 0) return c.mg.blob;
    for (int k = threadIdx.x; k < n_stage; k += blockDim.x) smem[k] = __ldg(c.mg.blob + k);
    __syncthreads();
    return smem;
}

// ------------------------------------------------------------------ bank access (dense, position-indexed)
// W (weighted kernels): a particle that has not run a segment yet starts with the launch weight w0 (source
// renormalisation, R6; secondaries of a fixed-source run: 1), later its own banked weight
// TD (time-dependent multi-group): the clock, time bin and 64-bit id are banked as for continuous energy, and the
// weight is always the banked one (census survivors and combed copies carry their own, R40).
template <bool CE, bool W = false, bool TD = false>
__device__ __forceinline__ void load_full(const Bank &B, unsigned int i, Particle &p, uint32_t &ctr, uint32_t &slot,
                                          double w0 = 1.0)
{
    p.x = B.x[i]; p.y = B.y[i]; p.z = B.z[i];
    p.ux = B.ux[i]; p.uy = B.uy[i]; p.uz = B.uz[i];
    p.cell = B.cell[i]; p.elem = B.elem[i];
    int gl = B.gl[i];
    p.g = gl & 0xffff; p.last = (gl >> 16) - 1;
    uint32_t ev = B.ev[i];
    p.pend = ev & PEND_MASK; p.nseg = ev >> 12;
    ctr = B.ctr[i];
    slot = B.slot[i];
    p.v = 0.0; p.gi = 0; p.ebin = 0;
    if (CE) { p.E = B.E[i]; p.t = B.t[i]; p.tbin = B.tbin[i]; p.id = B.id[i]; }
    else if (TD) { p.E = 0.0; p.t = B.t[i]; p.tbin = B.tbin[i]; p.id = B.id[i]; }
    else { p.E = 0.0; p.t = 0.0; p.tbin = 0; p.id = slot; }
    p.w = w0;
    if (W && (TD || p.nseg != 0)) p.w = B.w[i];
}

template <bool CE, bool W = false, bool TD = false>
__device__ __forceinline__ void store_full(const Bank &B, unsigned int i, const Particle &p, uint32_t ctr, uint32_t slot)
{
    B.x[i] = p.x; B.y[i] = p.y; B.z[i] = p.z; B.ux[i] = p.ux; B.uy[i] = p.uy; B.uz[i] = p.uz;
    B.cell[i] = p.cell; B.elem[i] = p.elem; B.gl[i] = pack_gl(p.g, p.last); B.ctr[i] = ctr; B.slot[i] = slot;
    B.ev[i] = p.pend | (p.nseg << 12);
    if (CE) { B.E[i] = p.E; B.t[i] = p.t; B.tbin[i] = p.tbin; B.id[i] = p.id; }
    if (TD) { B.t[i] = p.t; B.tbin[i] = p.tbin; B.id[i] = p.id; }
    if (W) B.w[i] = p.w;
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

// counts of the live regions a sweep reads (clamped to the capacity: a continuous-energy run whose secondaries
// outgrew the bank has already raised the overflow error; the clamp keeps every index inside the arrays)
__device__ __forceinline__ void live_counts(const Ctx &c, unsigned int s, unsigned int n0, unsigned int &n_front,
                                            unsigned int &n_in)
{
    n_front = n0; n_in = n0;
    if (s > 0) {
        QCount pc = c.qc[(s - 1) % RING];
        n_front = pc.n_scat < c.cap ? pc.n_scat : c.cap;
        unsigned long long tot = (unsigned long long)pc.n_scat + pc.n_surf;
        n_in = tot < c.cap ? (unsigned int)tot : c.cap;
    }
}

// per-block flush: k numerator (warp shuffles + one atomic per block) and the shared event counters
template <bool W = false>
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
    if (W) {  // absorbed weight (scal[2]); one atomic per warp
        double a = warp_sum(acc.wabs);
        if (lane == 0 && a != 0.0) atomicAdd(c.scal + 2, a);
    }
    if (threadIdx.x >= 1 && threadIdx.x < 11 && acc.s_ev[threadIdx.x])
        atomicAdd(c.counters + threadIdx.x, (unsigned long long)acc.s_ev[threadIdx.x]);
}

// kernel prologue shared by the transport kernels: stage the multi-group tables, clear the private tally columns
// and the block-shared event counters
#define MCDC_TRANSPORT_PROLOGUE(acc, s_flux)                                               \
    extern __shared__ double s_dyn[];                                                      \
    __shared__ unsigned int s_evc[16];                                                     \
    __shared__ Geo s_geo;                                                                  \
    if (threadIdx.x == 0) s_geo = c.geo;                                                   \
    Acc acc;                                                                               \
    acc.clear(s_evc);                                                                      \
    acc.geo = &s_geo;                                                                      \
    acc.tracing = c.tr.rec != nullptr;                                                     \
    acc.mgs = stage_mg(c, s_dyn, CE ? 0 : c.mg_stage);                                     \
    double *s_flux = s_dyn + (CE ? 0 : c.mg_stage);                                        \
    if (PRIVATE)                                                                           \
        for (int k = threadIdx.x; k < c.n_tally * BS; k += BS) s_flux[k] = 0.0;            \
    if (threadIdx.x < 16) s_evc[threadIdx.x] = 0u;                                         \
    __syncthreads()

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
template <bool CE, bool TD = false>
__global__ void __launch_bounds__(BS) k_source(Ctx c, unsigned int n)
{
    unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Bank &B = c.bank[0];
    Rng rng;
    rng.init(i, 0u);
    double xi[6];
#pragma unroll
    for (int k = 0; k < 6; k++) xi[k] = rng.next(c);  // always six draws
    Particle p;
    p.x = c.src_lo[0] + xi[0] * (c.src_hi[0] - c.src_lo[0]);
    p.y = c.src_lo[1] + xi[1] * (c.src_hi[1] - c.src_lo[1]);
    p.z = c.src_lo[2] + xi[2] * (c.src_hi[2] - c.src_lo[2]);
    p.ux = c.src_dir[0]; p.uy = c.src_dir[1]; p.uz = c.src_dir[2];
    if (c.src_iso) iso_dir(xi[3], xi[4], p.ux, p.uy, p.uz);
    p.g = 0;
    if (!CE) p.g = pick(c.mg.blob + c.mg.o_src_cum, c.mg.G, xi[5] * __ldg(c.mg.blob + c.mg.o_src_cum + c.mg.G - 1));
    if (!locate(c.geo, p.x, p.y, p.z, p.ux, p.uy, p.uz, -1, p.cell, p.elem)) { atomicExch(c.err, -2); p.cell = -1; }
    p.last = -1; p.id = i; p.pend = PEND_NONE; p.nseg = 0;
    p.E = c.src_E; p.t = c.src_t; p.tbin = 0;
    if (CE || TD) p.tbin = edge_bin(c.ce.t_edges, c.ce.n_t, c.src_t);
    p.w = 1.0;
    store_full<CE, TD, TD>(B, i, p, 6u, i);
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
    p.E = 0.0; p.t = 0.0; p.tbin = 0; p.pend = PEND_NONE; p.nseg = 0;
    if (!locate(c.geo, p.x, p.y, p.z, p.ux, p.uy, p.uz, -1, p.cell, p.elem)) { atomicExch(c.err, -2); p.cell = -1; }
    store_full<false>(c.bank[0], i, p, 0u, i);
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
        const double *cc = c.mg.blob + c.mg.o_cumchi + (size_t)mat * c.mg.G;
        p.g = pick(cc, c.mg.G, rng.next(c) * __ldg(cc + c.mg.G - 1));
        double a = rng.next(c), b = rng.next(c);
        iso_dir(a, b, p.ux, p.uy, p.uz);
    } else {
        double a1 = rng.next(c), a2 = rng.next(c), a3 = rng.next(c), a4 = rng.next(c);
        double En = 1e6 * watt(c.ce.watt_a, c.ce.watt_b, a1, a2, a3, a4);
        if (En < c.ce.E_min) En = c.ce.E_min;
        if (En > c.ce.E_max) En = c.ce.E_max;
        double a = rng.next(c), b = rng.next(c);
        iso_dir(a, b, p.ux, p.uy, p.uz);
        p.E = En;
        p.id = child_id(c.seed, pid, ctr0, (uint32_t)j);
    }
    p.last = -1; p.pend = PEND_NONE; p.nseg = 0;
}

// prompt secondaries made so far (R25a): more than max_secondaries is the bank-overflow error
__device__ __forceinline__ bool count_secondaries(const Ctx &c, unsigned int n)
{
    unsigned long long old = atomicAdd(c.counters + 15, (unsigned long long)n);
    if (old + n > c.max_secondaries) { atomicExch(c.err, -3); return false; }
    return true;
}

// the same limit looked at BEFORE children are made (time-dependent multi-group: only the children that are really born
// are counted afterwards, so the count cannot be taken up front as the continuous-energy branch does).  The read is not
// atomic with the later count: lanes that fission at the same moment can overshoot the limit by their own children, which
// a runaway guard tolerates.
__device__ __forceinline__ bool secondaries_allowed(const Ctx &c, unsigned int n)
{
    if (*(volatile unsigned long long *)(c.counters + 15) + n > c.max_secondaries) { atomicExch(c.err, -3); return false; }
    return true;
}

__device__ __forceinline__ void mark_lost(const Ctx &c)
{
    atomicExch(c.err, -2);
    atomicAdd(c.counters + 10, 1ull);
}

// ------------------------------------------------------------------ the sweep kernel (large populations)
#ifndef MCDC_SWEEP_MINBLOCKS
#define MCDC_SWEEP_MINBLOCKS 4
#endif
template <bool CE, bool PRIVATE, bool W, int X>
__global__ void __launch_bounds__(BS, MCDC_SWEEP_MINBLOCKS * 256 / BS) k_sweep(Ctx c, unsigned int s, unsigned int n0)
{
    MCDC_TRANSPORT_PROLOGUE(acc, s_flux);
    unsigned int n_front, n_in;
    live_counts(c, s, n0, n_front, n_in);
    QCount *oc = c.qc + (s % RING);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        QCount z = {0u, 0u, 0u, 0u};
        c.qc[(s + 1) % RING] = z;  // the set the next sweep appends to
        atomicAdd(c.counters + 12, (unsigned long long)n_in);  // segments run by the sweep kernels
        int e = *c.err;
        if (s > 0) {
            QCount pc = c.qc[(s - 1) % RING];
            if ((unsigned long long)pc.n_scat + pc.n_surf > c.cap) { atomicExch(c.err, -3); e = -3; }  // the two regions met
        }
        oc->err = (unsigned int)e;
    }
    const Bank &B = c.bank[s & 1];
    const Bank &O = c.bank[(s + 1) & 1];
    int par = 0;
    for (unsigned int base = blockIdx.x * BS; base < n_in; base += gridDim.x * BS, par ^= 1) {
        unsigned int t = base + threadIdx.x;
        int code = ADV_DEAD, aux = 0;
        Particle p;
        uint32_t ctr = 0, slot = 0;
        Rng rng;
        rng.init(0ull, 0u);
        const unsigned int i = t < n_in ? live_pos(c.cap, n_front, t) : 0u;
        const bool live = t < n_in && B.cell[i] >= 0;
        const unsigned int amask = __ballot_sync(0xffffffffu, live);
        if (live) {
            load_full<CE, W>(B, i, p, ctr, slot, c.w0);
            if (CE) ce_energy_state(c.ce, p);
            rng.init(p.id, ctr);
            const bool ok = finish_pending<CE, X>(c, acc, p, rng);
            __syncwarp(amask);  // the lanes went different ways by pending event: run the segment together again
            if (!ok) mark_lost(c);
            else {
                code = advance<CE, PRIVATE, W, X>(c, p, rng, aux, acc, s_flux);
                if (!CE && code == ADV_FISSION) { record_fission<CE>(c, p, rng.ctr, slot, aux); code = ADV_DEAD; }
            }
        }
        if (!CE) {
            unsigned int o = block_slot(code == ADV_SCATTER, code == ADV_SURFACE, oc, c.cap, par);
            if (code != ADV_DEAD) store_full<CE, W>(O, o, p, rng.ctr, slot);
        } else {
            unsigned int nb = code == ADV_SURFACE ? 1u : (code == ADV_FISSION ? (unsigned int)aux : 0u);
            unsigned int pf, ob;
            block_slot_n(code == ADV_SCATTER, nb, oc, c.cap, par, pf, ob);
            if (code == ADV_SCATTER) { if (pf < c.cap) store_full<CE, W>(O, pf, p, rng.ctr, slot); }
            else if (code == ADV_SURFACE) { if (ob < c.cap) store_full<CE, W>(O, c.cap - 1u - ob, p, rng.ctr, slot); }
            else if (code == ADV_FISSION && nb) {
                // prompt secondaries: born alive at the parent's site, first segment in the next sweep
                const int mat = c.geo.cfill[p.cell];
                const unsigned long long pid = p.id;
                const uint32_t ctr0 = rng.ctr;
                count_secondaries(c, nb);
                for (unsigned int j = 0; j < nb; j++) {
                    make_child<CE>(c, rng, mat, pid, ctr0, (int)j, p);
                    if (ob + j < c.cap) store_full<CE>(O, c.cap - 1u - (ob + j), p, 0u, slot);  // nseg = 0: weight w0
                }
            }
        }
    }
    if (PRIVATE) flush_private_flux(c, s_flux);
    flush_acc<W>(c, acc);
}

// ------------------------------------------------------------------ split per-event kernels (schedule 2)
// finish the scatter events of the front region / the surface events of the back region of bank[(s+1)&1] in place
template <bool CE>
__global__ void __launch_bounds__(BS) k_scatter(Ctx c, unsigned int s)
{
    extern __shared__ double s_dyn[];
    Acc acc;
    acc.clear(nullptr);
    acc.tracing = false;
    acc.geo = nullptr;
    acc.mgs = stage_mg(c, s_dyn, CE ? 0 : c.mg_stage);
    const QCount oc = c.qc[s % RING];
    const Bank &B = c.bank[(s + 1) & 1];
    for (unsigned int i = blockIdx.x * BS + threadIdx.x; i < oc.n_scat && i < c.cap; i += gridDim.x * BS) {
        Particle p;
        int gl = B.gl[i];
        uint32_t ev = B.ev[i];
        p.g = gl & 0xffff;
        p.cell = B.cell[i];
        p.id = CE ? B.id[i] : (unsigned long long)B.slot[i];
        if (CE) { p.E = B.E[i]; p.ux = B.ux[i]; p.uy = B.uy[i]; p.uz = B.uz[i]; }
        Rng rng;
        rng.init(p.id, B.ctr[i]);
        do_scatter<CE>(c, acc, p, rng, (int)(ev & 7u));
        B.ux[i] = p.ux; B.uy[i] = p.uy; B.uz[i] = p.uz;
        B.gl[i] = pack_gl(p.g, -1);
        B.ctr[i] = rng.ctr;
        B.ev[i] = (ev & ~PEND_MASK) | PEND_NONE;
        if (CE) B.E[i] = p.E;
    }
}

__global__ void __launch_bounds__(BS) k_surface(Ctx c, unsigned int s)
{
    __shared__ Geo s_geo;
    if (threadIdx.x == 0) s_geo = c.geo;
    __syncthreads();
    const QCount oc = c.qc[s % RING];
    const Bank &B = c.bank[(s + 1) & 1];
    for (unsigned int t = blockIdx.x * BS + threadIdx.x; t < oc.n_surf && t < c.cap; t += gridDim.x * BS) {
        unsigned int i = c.cap - 1u - t;
        uint32_t ev = B.ev[i];
        unsigned int hit = ev & PEND_MASK;
        if (hit >= PEND_SCATTER) continue;  // time edge / newborn: nothing to finish
        Particle p;
        p.x = B.x[i]; p.y = B.y[i]; p.z = B.z[i];
        p.ux = B.ux[i]; p.uy = B.uy[i]; p.uz = B.uz[i];
        p.cell = B.cell[i]; p.elem = B.elem[i];
        int gl = B.gl[i];
        p.g = gl & 0xffff; p.last = (gl >> 16) - 1;
        const int cell0 = p.cell, elem0 = p.elem;
        const double ux0 = p.ux, uy0 = p.uy, uz0 = p.uz;
        int r = 0;
        if (location_is_fast(c.geo, p.cell, p.elem)) r = do_surface_fast(c.geo, p, (int)hit);
        if (r == 0) r = (c.geo.n_lat2 ? do_surface2(s_geo, p, (int)hit) : do_surface(s_geo, p, (int)hit)) ? 1 : -1;
        if (r < 0) { mark_lost(c); p.cell = -1; }
        if (p.cell != cell0) B.cell[i] = p.cell;
        if (p.elem != elem0) B.elem[i] = p.elem;
        B.gl[i] = pack_gl(p.g, p.last);
        B.ev[i] = (ev & ~PEND_MASK) | PEND_NONE;
        if (p.ux != ux0) B.ux[i] = p.ux;
        if (p.uy != uy0) B.uy[i] = p.uy;
        if (p.uz != uz0) B.uz[i] = p.uz;
    }
}

// ------------------------------------------------------------------ the persistent kernel (thin populations)
// PAPER.md:49 asynchronous scheduling: the grid stays resident; each warp keeps 32 histories in registers, runs one
// whole segment per loop trip (finish the pending event, then advance) and refills the lanes whose history has ended
// from the global work queue.  Queue entry k < n_in is live particle k of bank[s&1]; entry n_in + a is the a-th
// secondary pushed by a continuous-energy fission (the fissioning lane continues as its first child and pushes the
// rest) into bank[(s+1)&1], used as a ring of `cap` slots.  A dead lane takes a TICKET (fetch-add on the queue head:
// no retries however many warps ask at once); a ticket for an entry that does not exist yet is kept, and the lane
// looks at its slot again every trip without holding up the live lanes of its warp.  Every ring slot has a sequence
// word (the bank's ev array, zero at launch): 2 lap = free for lap `lap`, 2 lap + 1 = holds that lap's entry; the
// pusher writes the particle, then the word; the ticket holder reads the particle when the word says so and hands
// the slot to the next lap.  The launch is over when every history has ended: ended == n_in + born.
#ifndef MCDC_PERSIST_MINBLOCKS
#define MCDC_PERSIST_MINBLOCKS 3
#endif
#ifndef MCDC_PERSIST_MINBLOCKS_CE
#define MCDC_PERSIST_MINBLOCKS_CE 3  // resident blocks per SM the continuous-energy variant is compiled for
#endif
#ifndef MCDC_REFILL
#define MCDC_REFILL 4  // dead lanes without a ticket at which a warp goes back to the queue
#endif
#ifndef MCDC_DENSE
#define MCDC_DENSE 12  // live lanes from which a continuous-energy warp keeps tickets for entries not pushed yet
#endif
// a particle that waits for a later census interval (it reached a time edge, or it is a delayed neutron that will be
// emitted there): appended to the census bank (R40); more than `cap` of them is the bank-overflow error
template <bool CE, bool W, bool TD>
__device__ __forceinline__ void census_put(const Ctx &c, const Particle &p, uint32_t ctr, uint32_t slot)
{
    const unsigned int i = atomicAdd(c.work + 4, 1u);
    if (i >= c.cap) { atomicExch(c.err, -3); return; }
    store_full<CE, W, TD>(c.cbank, i, p, ctr, slot);
}

// write a secondary into entry `a` of the persistent kernel's ring (bank O) and publish it (see k_persist); returns
// false when the run has to stop (bank overflow)
template <bool CE, bool W, bool TD>
__device__ __forceinline__ bool ring_put(const Ctx &c, const Bank &O, const unsigned int *head, unsigned int n_in, unsigned int a,
                                         const Particle &p, uint32_t slot)
{
    const unsigned int i = a % c.cap, free_ = 2u * (a / c.cap);
    // the slot still holds the previous lap's entry: if no ticket has been issued for that entry, nobody is about to take
    // it -- more than `cap` secondaries wait: bank overflow
    if (*(volatile uint32_t *)(O.ev + i) != free_) {
        if (*(volatile const unsigned int *)head + c.cap <= n_in + a) atomicExch(c.err, -3);
        // A ticket for the previous lap's entry has been issued; its holder takes the entry on its next loop trip.  The
        // wait is short when the holder is a lane of another warp.  It cannot end when the holder is a lane of THIS warp
        // (it is parked at the loop top until this lane gets there), which takes `cap` pushes within one loop trip, i.e.
        // a ring about as small as the number of resident lanes: the bounded wait (tens of milliseconds) then reports
        // the bank as too small (MCDC_EBANK), which it is.  DESIGN.md section 5 lists this limit.
        unsigned int spins = 0;
        while (*(volatile uint32_t *)(O.ev + i) != free_ && *(volatile int *)c.err == 0)
            if (++spins > (1u << 16)) atomicExch(c.err, -3);
        if (*(volatile int *)c.err != 0) return false;
    }
    O.x[i] = p.x; O.y[i] = p.y; O.z[i] = p.z; O.ux[i] = p.ux; O.uy[i] = p.uy; O.uz[i] = p.uz;
    O.cell[i] = p.cell; O.elem[i] = p.elem; O.slot[i] = slot;
    O.t[i] = p.t; O.tbin[i] = p.tbin; O.id[i] = p.id;
    if (CE) O.E[i] = p.E;
    if (TD) { O.gl[i] = pack_gl(p.g, -1); if (W) O.w[i] = p.w; }
    __threadfence();
    *(volatile uint32_t *)(O.ev + i) = free_ + 1u;
    return true;
}

// child j of a time-dependent multi-group fission (R39): type (prompt / precursor group) by xi nu against the cumulative
// yields, group from the type's spectrum, emission time (delayed: t - ln(xi) / lambda), isotropic direction; own id
// (R10).  Returns false for a delayed neutron emitted after the last time edge: it is never born.
__device__ __forceinline__ bool make_child_td(const Ctx &c, Rng &rng, int mat, int g_parent, double t_parent,
                                              unsigned long long pid, uint32_t ctr0, int j, Particle &p)
{
    const int J = c.td.J, G = c.mg.G;
    const double *cn = c.td.cum_nu + ((size_t)mat * G + g_parent) * (J + 1);
    const int typ = pick(cn, J + 1, rng.next(c) * __ldg(cn + J));
    const double *cc = typ == 0 ? c.mg.blob + c.mg.o_cumchi + (size_t)mat * G : c.td.cumchi_d + ((size_t)mat * J + typ - 1) * G;
    p.g = pick(cc, G, rng.next(c) * __ldg(cc + G - 1));
    double tj = t_parent;
    if (typ > 0) tj = t_parent - log(rng.next(c)) / __ldg(c.td.decay + mat * J + typ - 1);
    const double a = rng.next(c), b = rng.next(c);
    iso_dir(a, b, p.ux, p.uy, p.uz);
    p.last = -1; p.pend = PEND_NONE; p.nseg = 0;
    p.id = child_id(c.seed, pid, ctr0, (uint32_t)j);
    if (!(tj < __ldg(c.ce.t_edges + c.ce.n_t))) return false;
    p.t = tj;
    p.tbin = edge_bin(c.ce.t_edges, c.ce.n_t, tj);
    return true;
}

template <bool CE, bool PRIVATE, bool W, int X>
#ifndef MCDC_PERSIST_BLOCKS_RAW
#define MCDC_PERSIST_BLOCKS_RAW ((CE ? MCDC_PERSIST_MINBLOCKS_CE : MCDC_PERSIST_MINBLOCKS) * 256 / BS)
#endif
__global__ void __launch_bounds__(BS, MCDC_PERSIST_BLOCKS_RAW)
k_persist(Ctx c, unsigned int s, unsigned int n0)
{
    constexpr bool TD = (X & X_TD) != 0;
    constexpr bool GROW = CE || TD;  // fissions put secondaries into the running population: the work queue grows
    MCDC_TRANSPORT_PROLOGUE(acc, s_flux);
    unsigned int n_front, n_in;
    live_counts(c, s, n0, n_front, n_in);
    const Bank &B = c.bank[s & 1];
    const Bank &O = c.bank[(s + 1) & 1];
    // work[0] head of the queue, [1] secondaries pushed, [2] histories ended, [3] secondaries born in this launch
    // (32-bit: a run makes fewer than 2^32 secondaries, checked by the host)
    unsigned int *head = c.work, *tail = c.work + 1, *ended = c.work + 2, *born = c.work + 3;
    const unsigned int FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    bool alive = false, ticketed = false, drained = false;
    unsigned int ticket = 0, t_slot = 0, t_full = 0;  // ring slot and the sequence word that says "entry written"
    Particle p;
    uint32_t slot = 0;
    Rng rng;
    rng.init(0ull, 0u);
    unsigned int taken = 0, n_end = 0, idle_ns = 500;
    for (;;) {
        const unsigned int want = __ballot_sync(FULL, !alive && !ticketed && !drained);
        const int nw = __popc(want);
        const bool none_alive = !__any_sync(FULL, alive);
        // Multi-group: dead lanes go back to the queue as soon as MCDC_REFILL of them are free.  Continuous energy: a
        // DENSE warp does the same (its free lanes wait, ticket in hand, for secondaries to be pushed); a sparse or
        // idle warp only takes entries that already exist, so that a thin population stays concentrated in few warps
        // instead of keeping every resident warp busy with one or two lanes.
        unsigned int n_take = 0;
        if (!GROW) n_take = (nw >= MCDC_REFILL || (none_alive && nw > 0)) ? (unsigned int)nw : 0u;
        else if (nw >= MCDC_REFILL) {
            if (__popc(__ballot_sync(FULL, alive)) >= MCDC_DENSE) n_take = (unsigned int)nw;
            else {
                unsigned int backlog = 0;
                if (lane == 0) {
                    unsigned int h = *(volatile unsigned int *)head, t = *(volatile unsigned int *)tail;
                    backlog = n_in + t > h ? n_in + t - h : 0u;
                }
                backlog = __shfl_sync(FULL, backlog, 0);
                n_take = min((unsigned int)nw, backlog);
            }
        }
        if (GROW && n_take) {  // the run is being stopped (bank overflow, lost particle): hand out no more work
            int e = 0;
            if (lane == 0) e = *(volatile int *)c.err;
            if (__shfl_sync(FULL, e, 0)) n_take = 0;
        }
        const bool take = n_take > 0;
        if (take) {
            unsigned int base = 0;
            if (lane == 0) base = atomicAdd(head, n_take);
            base = __shfl_sync(FULL, base, 0);
            const unsigned int rank = __popc(want & ((1u << lane) - 1u));
            if (!alive && !ticketed && !drained && rank < n_take) {
                ticket = base + rank;
                ticketed = GROW || ticket < n_in;  // eigenvalue cycle: the queue never grows, a ticket past its end is void
                drained = !ticketed;
                if (GROW && ticket >= n_in) {
                    const unsigned int a = ticket - n_in;
                    t_slot = a % c.cap;
                    t_full = 2u * (a / c.cap) + 1u;
                }
            }
        }
        if (ticketed) {
            uint32_t ctr = 0;
            bool have = false;
            if (ticket < n_in) {
                load_full<CE, W, TD>(B, live_pos(c.cap, n_front, ticket), p, ctr, slot, c.w0);
                have = true;
            } else if (GROW && *(volatile uint32_t *)(O.ev + t_slot) == t_full) {
                const unsigned int i = t_slot;
                __threadfence();
                p.x = __ldcg(O.x + i); p.y = __ldcg(O.y + i); p.z = __ldcg(O.z + i);
                p.ux = __ldcg(O.ux + i); p.uy = __ldcg(O.uy + i); p.uz = __ldcg(O.uz + i);
                p.cell = __ldcg(O.cell + i); p.elem = __ldcg(O.elem + i);
                p.g = 0; p.last = -1; p.pend = PEND_NONE; p.nseg = 0;
                p.w = c.w0;
                slot = __ldcg(O.slot + i);
                p.E = 0.0;
                if (CE) p.E = __ldcg(O.E + i);
                if (TD) { p.g = __ldcg(O.gl + i) & 0xffff; if (W) p.w = __ldcg(O.w + i); }
                p.t = __ldcg(O.t + i); p.tbin = __ldcg(O.tbin + i); p.id = __ldcg(O.id + i);
                __threadfence();
                *(volatile uint32_t *)(O.ev + i) = t_full + 1u;  // free for the next lap
                have = true;
            }
            if (have) {
                ticketed = false;
                if (CE) ce_energy_state(c.ce, p);
                if (p.cell >= 0) { alive = true; rng.init(p.id, ctr); taken++; }
                else n_end++;  // a particle that was lost at birth
            }
        }
        if (!__any_sync(FULL, alive)) {
            // nothing to run.  Multi-group: leave once every lane's ticket is void.  Continuous energy: other warps may
            // still push secondaries; sleep, then look again, until every history of the launch has ended:
            // ended == n_in + born, with `ended` read first (a parent's children are counted in `born` before the
            // parent is counted in `ended`, so the test cannot pass early).
            unsigned int fin = 0;
            if (!GROW) fin = __all_sync(FULL, drained) ? 1u : 0u;
            else {
                const unsigned int ne = __reduce_add_sync(FULL, n_end);
                n_end = 0;
                if (lane == 0) {
                    if (ne) atomicAdd(ended, ne);
                    unsigned int e = *(volatile unsigned int *)ended;
                    __threadfence();
                    unsigned int b = *(volatile unsigned int *)born;
                    fin = (e == n_in + b || *(volatile int *)c.err != 0) ? 1u : 0u;
                }
                fin = __shfl_sync(FULL, fin, 0);
            }
            if (fin) break;
            if (GROW) { __nanosleep(idle_ns); if (idle_ns < 16000) idle_ns *= 2; }
            continue;
        }
        idle_ns = 500;
        const unsigned int amask = __ballot_sync(FULL, alive);
        if (alive) {
            int aux = 0, code = ADV_DEAD;
            const bool ok = finish_pending<CE, X>(c, acc, p, rng);
            __syncwarp(amask);  // the lanes went different ways by pending event: run the segment together again
            if (!ok) mark_lost(c);
            else code = advance<CE, PRIVATE, W, X>(c, p, rng, aux, acc, s_flux);
            if (GROW && code == ADV_SURFACE && p.pend == PEND_TIME && c.census_stop) {
                // the census (R40): the particle waits in the census bank for the next interval
                p.pend = PEND_NONE;
                census_put<CE, W, TD>(c, p, rng.ctr, slot);
                code = ADV_DEAD;
            }
            if (code == ADV_DEAD) { alive = false; n_end++; }
            else if (code == ADV_FISSION) {
                alive = false;
                n_end++;
                if (!GROW) record_fission<CE>(c, p, rng.ctr, slot, aux);
                else if (TD) {
                    if (aux > 0 && secondaries_allowed(c, (unsigned int)aux)) {
                        // every child is counted as born first; one that is never born, or that waits for a later
                        // interval, is counted as ended at once (the termination test stays ended == n_in + born)
                        atomicAdd(born, (unsigned int)aux);
                        const int mat = c.geo.cfill[p.cell], g_parent = p.g, tbin_parent = p.tbin;
                        const double t_parent = p.t;
                        const unsigned long long pid = p.id;
                        const uint32_t ctr0 = rng.ctr;
                        Particle first = p;
                        bool have_first = false;
                        unsigned int n_born = 0;
                        for (int j = 0; j < aux; j++) {
                            if (!make_child_td(c, rng, mat, g_parent, t_parent, pid, ctr0, j, p)) { n_end++; continue; }
                            n_born++;
                            if (p.tbin != tbin_parent) { census_put<CE, W, TD>(c, p, 0u, slot); n_end++; continue; }
                            if (!have_first) { first = p; have_first = true; continue; }
                            if (!ring_put<CE, W, TD>(c, O, head, n_in, atomicAdd(tail, 1u), p, slot)) break;
                        }
                        if (n_born) { count_secondaries(c, n_born); if (W) atomicAdd(c.scal + 6, (double)n_born * first.w); }
                        if (have_first) {
                            p = first;
                            rng.init(p.id, 0u);
                            alive = true;
                        }
                    }
                } else if (aux > 0 && count_secondaries(c, (unsigned int)aux)) {
                    atomicAdd(born, (unsigned int)aux);
                    const int mat = c.geo.cfill[p.cell];
                    const unsigned long long pid = p.id;
                    const uint32_t ctr0 = rng.ctr;
                    unsigned int at = 0;
                    if (aux > 1) at = atomicAdd(tail, (unsigned int)(aux - 1));
                    Particle first = p;
                    for (int j = 0; j < aux; j++) {
                        make_child<CE>(c, rng, mat, pid, ctr0, j, p);
                        if (j == 0) first = p;
                        else if (!ring_put<CE, W, false>(c, O, head, n_in, at + (unsigned int)(j - 1), p, slot)) break;
                    }
                    p = first;
                    p.w = c.w0;
                    ce_energy_state(c.ce, p);
                    rng.init(p.id, 0u);
                    alive = true;
                }
            }
        }
    }
    taken = __reduce_add_sync(FULL, taken);
    if (lane == 0 && taken) atomicAdd(c.counters + 14, (unsigned long long)taken);
    if (PRIVATE) flush_private_flux(c, s_flux);
    flush_acc<W>(c, acc);
}

// ------------------------------------------------------------------ monolithic schedule
// every slot of bank 0, one whole segment (advance + the event it ends in), in place, no compaction; counts the
// survivors.  A dead slot has cell = -1.
template <bool CE, bool PRIVATE, bool W, int X>
__global__ void __launch_bounds__(BS) k_segment(Ctx c, unsigned int s, unsigned int n)
{
    MCDC_TRANSPORT_PROLOGUE(acc, s_flux);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        QCount z = {0u, 0u, 0u, 0u};
        c.qc[(s + 1) % RING] = z;
        c.qc[s % RING].err = (unsigned int)*c.err;
    }
    const Bank &B = c.bank[0];
    unsigned int alive = 0;
    for (unsigned int i = blockIdx.x * BS + threadIdx.x; i < n; i += gridDim.x * BS) {
        if (B.cell[i] < 0) continue;
        Particle p;
        uint32_t ctr, slot;
        load_full<CE, W>(B, i, p, ctr, slot, c.w0);
        if (CE) ce_energy_state(c.ce, p);
        Rng rng;
        rng.init(p.id, ctr);
        int aux = 0;
        int code = advance<CE, PRIVATE, W, X>(c, p, rng, aux, acc, s_flux);
        if (code == ADV_FISSION) { record_fission<CE>(c, p, rng.ctr, slot, aux); code = ADV_DEAD; }
        else if (code != ADV_DEAD && !finish_pending<CE, X>(c, acc, p, rng)) { mark_lost(c); code = ADV_DEAD; }
        if (code == ADV_DEAD) p.cell = -1;
        store_full<CE, W>(B, i, p, rng.ctr, slot);
        if (code != ADV_DEAD) alive++;
    }
    alive = __reduce_add_sync(0xffffffffu, alive);
    if ((threadIdx.x & 31) == 0 && alive) atomicAdd(&c.qc[s % RING].n_alive, alive);
    if (PRIVATE) flush_private_flux(c, s_flux);
    flush_acc<W>(c, acc);
}

// ------------------------------------------------------------------ a10/a12: fission bank by count-scan-write
__global__ void __launch_bounds__(BS) k_scan_partial(Ctx c, unsigned int n, unsigned int *part)
{
    __shared__ unsigned int s_w[BS / 32];
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
// The parents' counts are cleared by k_clear_counts afterwards (a child slot may be another parent's record).
template <bool CE>
__global__ void __launch_bounds__(BS) k_emit(Ctx c, unsigned int n, const unsigned int *part, unsigned int cap)
{
    __shared__ unsigned int s_w[BS / 32];
    const FisRec &F = c.fis;
    const Bank &O = c.bank[0];
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
    rng.init(pid, ctr0);
    for (int j = 0; j < nc; j++) {
        make_child<CE>(c, rng, mat, pid, ctr0, j, p);
        store_full<CE>(O, off + j, p, 0u, off + j);
    }
}

__global__ void __launch_bounds__(BS) k_clear_counts(Ctx c, unsigned int n)
{
    unsigned int i = blockIdx.x * BS + threadIdx.x;
    if (i < n) c.fis.n[i] = 0;
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
    out[i] = draw_at(seed, id[i], domain, cycle, draw[i]);
}

__global__ void k_test_grid(Ctx c, const double *E, unsigned long long n, int *ob, int *oh)
{
    unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    ob[i] = grid_index_binary(c.ce, E[i]);
    oh[i] = grid_index_hash(c.ce, E[i]);
}

// locate + nearest boundary of n points; path: 0 = the path the transport kernels take from that point (straight-line
// in LAT_FAST elements, pruned enclosing-cell list elsewhere), 1 = generic loops with the pruned list, 2 = generic
// loops over every surface of the enclosing cell (no pruning)
__global__ void k_test_geometry(Ctx c, const double *x, const double *u, unsigned long long n, int path, int *loc,
                                double *dist, int *surf)
{
    unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
    __shared__ Geo s_geo;
    if (threadIdx.x == 0) s_geo = c.geo;
    __syncthreads();
    if (i >= n) return;
    const Geo &G = c.geo;
    int cell, elem, hit = -1;
    const double px = x[3 * i], py = x[3 * i + 1], pz = x[3 * i + 2], ux = u[3 * i], uy = u[3 * i + 1], uz = u[3 * i + 2];
    bool ok = locate(G, px, py, pz, ux, uy, uz, -1, cell, elem);
    double d = -1.0;
    if (ok) {
        const int4 li = elem >= 0 ? __ldg(G.lat_info + outer_of(G, elem)) : __ldg(G.cell_info + cell);
        const int cyl = elem >= 0 ? __ldg(&G.ufast[li.x & UNIV_MASK].y) : li.y;
        int4 l2i = make_int4(0, 0, 0, 0);
        if (path == 0 && elem >= (1 << INNER_SHIFT) && (li.x & LAT_FAST2))
            l2i = __ldg(G.l2_info + __ldg(G.l2_off + (li.w >> 16)) + inner_of(G, elem));
        if (l2i.x & LAT_FAST) d = nearest_fast2(G, li, l2i, __ldg(&G.ufast[l2i.x & UNIV_MASK].y), px, py, pz, ux, uy, uz, elem, -1, hit);
        else if (path == 0 && (li.x & LAT_FAST)) d = nearest_fast(G, li.z, li.w, cyl, px, py, pz, ux, uy, uz, elem, -1, hit);
        else {
            unsigned int mask = (elem >= 0 && path != 2) ? __ldg(G.lat_rmask + outer_of(G, elem)) : 0xffffffffu;
            d = G.n_lat2 ? nearest2(s_geo, px, py, pz, ux, uy, uz, cell, elem, -1, hit, mask) : nearest(s_geo, px, py, pz, ux, uy, uz, cell, elem, -1, hit, mask);
            if (hit >= (1 << HIT_BITS)) { hit &= (1 << HIT_BITS) - 1; if (hit == (1 << HIT_BITS) - 1) hit = -1; }
        }
    }
    loc[3 * i] = !ok ? -1 : (elem >= 0 ? G.lat_cell : cell);
    loc[3 * i + 1] = ok ? elem : -1;
    loc[3 * i + 2] = ok && elem >= 0 ? cell : -1;
    dist[i] = d;
    surf[i] = hit;
}

// any point of an nx x ny x nz grid over the source box that lies in no cell raises the geometry error (mcdc_create)
__global__ void k_check_source_box(Ctx c, int n1)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n1 * n1 * n1) return;
    const int a[3] = {i % n1, (i / n1) % n1, i / (n1 * n1)};
    double x[3];
    for (int k = 0; k < 3; k++) {
        double f = n1 > 1 ? (double)a[k] / (n1 - 1) : 0.5;
        f = 1e-9 + f * (1.0 - 2e-9);  // just inside the faces
        x[k] = c.src_lo[k] + f * (c.src_hi[k] - c.src_lo[k]);
    }
    int cell, elem;
    if (!locate(c.geo, x[0], x[1], x[2], 0.0, 0.0, 1.0, -1, cell, elem)) atomicExch(c.err, -2);
}

}  // namespace mcdc
