// mcdc_census.cuh -- what happens between two census intervals of a time-dependent fixed-source run (R40;
// PAPER.md:31 "fully dynamic simulations"): the particles waiting in the census bank are keyed by particle id, sorted
// (LSD radix sort, 8 bits per pass, stable), those of the next interval are moved to the source bank in id order --
// optionally through the population-control comb -- and the rest is kept for later intervals.  The id order makes the
// comb reproducible: it is the order the CPU oracle combs in.
#pragma once
#include "mcdc_kernels.cuh"

namespace mcdc {

constexpr int RS_ITEMS = 8;               // keys per thread and tile
constexpr int RS_TILE = BS * RS_ITEMS;    // keys per block

// key of census particle i: its id if it belongs to interval k, the largest key otherwise (sorted to the end); counts
// the particles of interval k
__global__ void __launch_bounds__(BS) k_census_keys(Bank CB, unsigned int n, int k, unsigned long long *key, unsigned int *idx,
                                                    unsigned int *n_match)
{
    unsigned int i = blockIdx.x * BS + threadIdx.x;
    bool m = false;
    if (i < n) {
        m = CB.tbin[i] == k;
        key[i] = m ? (unsigned long long)CB.id[i] : ~0ull;
        idx[i] = i;
    }
    unsigned int cnt = __popc(__ballot_sync(0xffffffffu, m));
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(n_match, cnt);
}

// radix-sort pass, step 1: digit histogram of every tile, stored digit-major (hist[digit * n_blocks + block]) so that
// ONE exclusive scan of the whole array gives every (digit, block) its first output position
__global__ void __launch_bounds__(BS) k_rs_hist(const unsigned long long *key, unsigned int n, int shift, unsigned int *hist)
{
    __shared__ unsigned int s_h[256];
    s_h[threadIdx.x] = 0u;  // BS == 256
    __syncthreads();
    const unsigned int base = blockIdx.x * RS_TILE;
    for (int r = 0; r < RS_ITEMS; r++) {
        unsigned int i = base + r * BS + threadIdx.x;
        if (i < n) atomicAdd(&s_h[(unsigned int)(key[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[threadIdx.x * gridDim.x + blockIdx.x] = s_h[threadIdx.x];
}

// step 3 (step 2 is the scan): stable scatter.  Keys of a tile are taken in order, BS at a time; inside a round the
// rank of a key among equal digits is (equal digits in earlier warps) + (equal digits in lower lanes of its warp).
__global__ void __launch_bounds__(BS) k_rs_scatter(const unsigned long long *key_in, const unsigned int *idx_in,
                                                   unsigned long long *key_out, unsigned int *idx_out, unsigned int n, int shift,
                                                   const unsigned int *hist)
{
    __shared__ unsigned int s_run[256];            // next output position of each digit for this block
    __shared__ unsigned int s_wc[BS / 32][256];    // per warp: keys of each digit in the current round
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    s_run[threadIdx.x] = hist[threadIdx.x * gridDim.x + blockIdx.x];
    for (int k = 0; k < BS / 32; k++) s_wc[k][threadIdx.x] = 0u;
    __syncthreads();
    const unsigned int base = blockIdx.x * RS_TILE;
    for (int r = 0; r < RS_ITEMS; r++) {
        const unsigned int i = base + r * BS + threadIdx.x;
        const bool live = i < n;
        unsigned long long kv = 0ull;
        unsigned int d = 256u + lane;  // a digit nobody else has: a dead lane matches only itself
        if (live) { kv = key_in[i]; d = (unsigned int)(kv >> shift) & 255u; }
        const unsigned int peers = __match_any_sync(0xffffffffu, d);
        const unsigned int rank = __popc(peers & ((1u << lane) - 1u));
        if (live && rank == 0) s_wc[w][d] = __popc(peers);
        __syncthreads();
        if (live) {
            unsigned int before = 0;
            for (int k = 0; k < w; k++) before += s_wc[k][d];
            const unsigned int o = s_run[d] + before + rank;
            key_out[o] = kv;
            idx_out[o] = idx_in[i];
        }
        __syncthreads();
        unsigned int tot = 0;
        for (int k = 0; k < BS / 32; k++) { tot += s_wc[k][threadIdx.x]; s_wc[k][threadIdx.x] = 0u; }
        s_run[threadIdx.x] += tot;
        __syncthreads();
    }
}

// copy one banked particle (all fields the problem has)
template <bool CE>
__device__ __forceinline__ void copy_particle(const Bank &S, unsigned int i, const Bank &D, unsigned int o)
{
    D.x[o] = S.x[i]; D.y[o] = S.y[i]; D.z[o] = S.z[i]; D.ux[o] = S.ux[i]; D.uy[o] = S.uy[i]; D.uz[o] = S.uz[i];
    D.cell[o] = S.cell[i]; D.elem[o] = S.elem[i]; D.gl[o] = S.gl[i]; D.ev[o] = S.ev[i]; D.ctr[o] = S.ctr[i];
    D.slot[o] = S.slot[i]; D.t[o] = S.t[i]; D.tbin[o] = S.tbin[i]; D.id[o] = S.id[i]; D.w[o] = S.w[i];
    if (CE) D.E[o] = S.E[i];
}

// sorted position r < M: particle of the next interval -> source bank slot r (no population control);
// r >= M: a later interval's particle -> slot r - M of the other census bank
template <bool CE>
__global__ void __launch_bounds__(BS) k_census_move(Bank S, const unsigned int *idx, unsigned int M, unsigned int n, Bank dst,
                                                    Bank keep, int move_first)
{
    unsigned int r = blockIdx.x * BS + threadIdx.x;
    if (r >= n) return;
    const unsigned int i = idx[r];
    if (r < M) { if (move_first) copy_particle<CE>(S, i, dst, r); }
    else copy_particle<CE>(S, i, keep, r - M);
}

// ---- the comb (R40)
__global__ void __launch_bounds__(BS) k_comb_weights(Bank S, const unsigned int *idx, unsigned int M, double *w)
{
    unsigned int r = blockIdx.x * BS + threadIdx.x;
    if (r < M) w[r] = S.w[idx[r]];
}

// inclusive prefix sum of n doubles in place, one block: every thread sums a contiguous chunk left to right, the chunk
// totals are summed left to right by one thread, every thread rewrites its chunk.  (The oracle sums in one chain: the
// two differ by rounding order, ~1e-16 relative, like every other tally.)
__global__ void __launch_bounds__(1024) k_dscan(double *a, unsigned int n)
{
    __shared__ double s_sum[1024];
    const unsigned int per = (n + 1023u) / 1024u;
    const unsigned int lo = threadIdx.x * per, hi = lo + per < n ? lo + per : n;
    double t = 0.0;
    for (unsigned int k = lo; k < hi; k++) t += a[k];
    s_sum[threadIdx.x] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double run = 0.0;
        for (int k = 0; k < 1024; k++) { double v = s_sum[k]; s_sum[k] = run; run += v; }
    }
    __syncthreads();
    double run = s_sum[threadIdx.x];
    for (unsigned int k = lo; k < hi; k++) { run += a[k]; a[k] = run; }
}

// first tooth j (0..N) with off + j delta >= C: the comb's own comparison, so that the count of teeth inside a
// particle's weight interval is exactly what a left-to-right walk finds
__device__ __forceinline__ unsigned int first_tooth(double C, double off, double delta, unsigned int N)
{
    double e = ceil((C - off) / delta);
    long long j = e < 0.0 ? 0ll : (e > (double)N ? (long long)N : (long long)e);
    while (j > 0 && !(off + (double)(j - 1) * delta < C)) j--;
    while (j < (long long)N && off + (double)j * delta < C) j++;
    return (unsigned int)j;
}

// copies of sorted particle r = teeth in [C_{r-1}, C_r); the last particle also gets a tooth lost to rounding.
// prm[0] = xi (the comb's draw); W = C[M-1]
__global__ void __launch_bounds__(BS) k_comb_copies(const double *C, unsigned int M, unsigned int N, double xi, unsigned int *copies)
{
    unsigned int r = blockIdx.x * BS + threadIdx.x;
    if (r >= M) return;
    const double W = C[M - 1], delta = W / (double)N, off = xi * delta;
    const unsigned int j0 = r == 0 ? 0u : first_tooth(C[r - 1], off, delta, N);
    const unsigned int j1 = r == M - 1 ? N : first_tooth(C[r], off, delta, N);
    copies[r] = j1 > j0 ? j1 - j0 : 0u;
}

// every copy is a new track: weight W / N, id from the domain-2 Philox block (parent id, interval, copy index), draw
// and segment counters reset
template <bool CE>
__global__ void __launch_bounds__(BS) k_comb_write(Bank S, const unsigned int *idx, const unsigned int *copies,
                                                   const unsigned int *offs, const double *C, unsigned int M, unsigned int N,
                                                   unsigned long long seed, int k, Bank dst)
{
    unsigned int r = blockIdx.x * BS + threadIdx.x;
    if (r >= M) return;
    const unsigned int nc = copies[r];
    if (!nc) return;
    const unsigned int i = idx[r], o0 = offs[r];
    const double delta = C[M - 1] / (double)N;
    const unsigned long long pid = S.id[i];
    for (unsigned int cidx = 0; cidx < nc; cidx++) {
        const unsigned int o = o0 + cidx;
        copy_particle<CE>(S, i, dst, o);
        uint32_t o0w, o1w, o2w, o3w;
        philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), (2u << 24) | (uint32_t)k, cidx, (uint32_t)seed, (uint32_t)(seed >> 32), o0w,
                      o1w, o2w, o3w);
        dst.id[o] = ((unsigned long long)o1w << 32) | o0w;
        dst.w[o] = delta;
        dst.ctr[o] = 0u;
        dst.ev[o] = PEND_NONE;  // no pending event, segment counter 0
        dst.slot[o] = o;
    }
}

}  // namespace mcdc
