/* mcdc_test.h -- unit-level and micro-benchmark entry points of the same library (libmcdc_b200.so).
 *
 * They are NOT part of the product boundary (SURVEY.md 8b lists none of them; include/mcdc.h is that boundary): the parity
 * tests use them to compare single steps of the path (random-number draws, union-grid search, cell lookup and distance to
 * the nearest surface) with the oracle, and bench.py uses mcdc_microbench for the denominators of the issue-slot roofline.
 * Conventions as in mcdc.h: HOST pointers in and out, caller-owned, 0 or a negative MCDC_E* code returned; the device
 * staging is taken from the problem's (idle) workspace, so n is limited by the problem's capacity (MCDC_ENOMEM beyond it).
 */
#ifndef MCDC_TEST_H
#define MCDC_TEST_H
#include "mcdc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* n uniform draws of stream (seed, id[i], domain, cycle) at index draw[i] */
int mcdc_test_draws(mcdc_problem *p, uint64_t seed, uint32_t domain, uint32_t cycle, const uint64_t *id,
                    const uint32_t *draw, uint64_t n, double *out);
/* union-grid index of E[i] with the binary (out_bin) and the hashed (out_hash) search */
int mcdc_test_grid_index(mcdc_problem *p, const double *E, uint64_t n, int32_t *out_bin, int32_t *out_hash);
/* locate + nearest boundary for n points: loc[i][3] = (c0, elem, c1), dist[i], surf[i].  path 0: the code path the
 * transport kernels take from that point (straight-line inside simple lattice elements, else the generic loops over
 * the enclosing cell's surfaces that create() could not rule out); 1: generic loops with that pruned list; 2: generic
 * loops over every surface (no pruning).  All three must agree. */
int mcdc_test_geometry(mcdc_problem *p, const double *x, const double *u, uint64_t n, int32_t path, int32_t *loc,
                       double *dist, int32_t *surf);

/* Arithmetic micro-benchmarks of this GPU (the ALU roofline's denominators): runs `iters` loop trips of
 * independent register-only chains of one operation on 148 x 8 blocks of 256 threads; returns the device time of the
 * launch and the thread-level operations it performed (FFMA / DFMA: fused multiply-adds; LOG, DIV, SQRT, SINCOSPI, RCP:
 * float64 library calls; PHILOX: Philox4x32-10 blocks = two draws each). */
enum { MCDC_MB_FFMA = 0, MCDC_MB_DFMA, MCDC_MB_LOG, MCDC_MB_DIV, MCDC_MB_SQRT, MCDC_MB_SINCOSPI, MCDC_MB_RCP, MCDC_MB_PHILOX,
       MCDC_MB_COUNT };
int mcdc_microbench(mcdc_problem *p, int32_t which, uint64_t iters, double *ms, double *ops);

#ifdef __cplusplus
}
#endif
#endif
