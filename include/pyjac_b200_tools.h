/* pyjac_b200_tools.h -- bench / test helpers beside the product library (libpyjac_b200_tools.so).
 *
 * Nothing here is on the evaluation path of include/pyjac_b200.h: table statistics for the
 * design notes and the host-side tests, and the two machine-peak probes the roofline discussion
 * refers to (`bench.py --peaks`).
 */
#ifndef PYJAC_B200_TOOLS_H
#define PYJAC_B200_TOOLS_H

#include "pyjac_b200.h"

#ifdef __cplusplus
extern "C" {
#endif

#define PYJAC_TOOLS_NSTATS 24

/* Host-only: validates and packs `host_desc` exactly as pyjac_mech_create_shaped does (no CUDA
 * call, the same self-check of everything the kernels read without bounds checks) and reports the
 * size of the evaluation tables.  stats[0..23] =
 *   0 elements of the per-state array E      1 entries of all Jacobian cell lists
 *   2 gather steps of the streaming phase    3 gather steps of the summing phase
 *   4 Jacobian cells with a list             5 chunks of the summing phase
 *   6 shared-memory bytes of one CTA         7 groups of 32 reactions
 *   8 states per CTA iteration               9 threads per CTA
 *  10 reserved (1)                          11 CTAs per SM the footprint is sized for
 *  12 cells summed piecewise                13 pieces
 *  14 bytes of the summing-phase tables     15 bytes of the streaming-phase tables
 *  16..19 summing-phase steps by kind (three sums at once, one sum, products, all reactions)
 *  20, 21 shared-memory wavefronts beyond the minimum that the entry placement leaves, per CTA
 *         iteration (summing phase, streaming phase; the bank model of mech_pack.cu)
 *  22, 23 bank-group excess of the gather groups before / after the layout search of the per-reaction terms
 * Errors as pyjac_mech_create_shaped (PYJAC_EINVAL, PYJAC_ELIMIT, PYJAC_ENOMEM). */
int pyjac_tools_pack_stats(const pyjac_mech_desc *host_desc, const pyjac_launch_shape *shape,
                           int64_t *stats);

/* Machine peaks measured with the same instructions the Jacobian kernel uses.  Device pointers,
 * enqueued on `stream` (a cudaStream_t), no allocation.
 *   pyjac_tools_peak_store_stream: writes n_doubles (a multiple of 2) doubles of `buf` once with
 *     16-byte streaming stores (st.global.cs.v2.f64), the store of the streaming phase; bytes
 *     moved = 8 n_doubles.
 *   pyjac_tools_peak_dfma: every thread of a full-occupancy grid runs 8 independent chains of
 *     `iters` fp64 FMAs and writes one result per thread to out[0 .. *n_threads) (out must hold
 *     148 * 2048 doubles at least; the thread count used is returned); flops = 2 * 8 * iters *
 *     *n_threads. */
int pyjac_tools_peak_store_stream(double *buf, int64_t n_doubles, void *stream);
/*   pyjac_tools_peak_tile_store: the output path of a kernel that assembles each state's Jacobian in
 *     shared memory first.  n_tiles tiles of tile_doubles doubles (even; 8 tile_doubles a multiple of
 *     16 bytes) are each written element by element with 8-byte shared-memory stores and then moved
 *     to buf[t * tile_doubles ..) by mode 0: one cp.async.bulk.global.shared::cta per tile (bulk-copy
 *     engine, two buffers per CTA so that a copy drains while the next tile is filled), mode 1: a
 *     read-back with 16-byte shared loads and st.global.cs.v2.f64.  256 threads per CTA,
 *     ctas_per_sm x SM count CTAs; bytes moved = 8 n_tiles tile_doubles.  PYJAC_ELIMIT if two tiles
 *     exceed the shared memory of one CTA. */
int pyjac_tools_peak_tile_store(double *buf, int64_t n_tiles, int32_t tile_doubles, int32_t mode,
                                int32_t ctas_per_sm, void *stream);
int pyjac_tools_peak_dfma(double *out, int64_t iters, int64_t *n_threads, void *stream);

/* Gather probe -- a TIMING PROTOTYPE, not an evaluation: the output half of a Jacobian kernel whose
 * gathers carry no padding, on the REAL contribution lists of the mechanism's Jacobian cells but with
 * stand-in values for the per-reaction terms they sum.  Per batch of S (1..3) states a CTA writes the
 * rank-one part of every cell to a per-state tile in shared memory, adds the cells' sparse sums (cells
 * sorted by list length, 32 cells of nearly equal length per warp chunk, one shared-memory load per
 * entry and state) and moves each tile to out[state][(N_sp+1)^2] with one cp.async.bulk; n_buf = 2
 * tile sets overlap the copies with the next batch.  Builds and uploads its tables, runs 2 warm-up and
 * `reps` timed launches (CUDA events on `stream`), frees the tables.  Outputs: ms_best / ms_mean per
 * launch; expected_host[(N_sp+1)^2] = the tile every state must hold (the stand-in values do not
 * depend on the state) for the caller to compare with `out` (DEVICE pointer, n_states tiles);
 * stats[8] = list entries, entries with chunk padding, chunks, E elements per state, shared memory
 * per CTA in bytes, non-empty cells, cells, grid.  PYJAC_ELIMIT if the shape does not fit shared
 * memory; allocates (probe only). */
int pyjac_tools_gather_probe(const pyjac_mech_desc *host_desc, int32_t S, int32_t threads,
                             int32_t ctas_per_sm, int32_t n_buf, int64_t n_states, double *out,
                             double *expected_host, int64_t *stats, int32_t reps, float *ms_best,
                             float *ms_mean, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* PYJAC_B200_TOOLS_H */
