/* pixreco_driver.h — a multi-threaded C++ client of the C ABI (pixreco.h) for the paper's own usage pattern:
 * one pr_acquire per event on the event's own stream, issued from several host threads at once, completion by
 * polling, never a blocking wait (TBB tasks on many threads; BASELINE.json
 * configs[2]; SURVEY 8(d) "issuing host threads in {1, 2, 4}").  It uses nothing but pixreco.h: it is a caller of
 * the library, not part of the hot path.  Built as libpixreco_driver.so next to libpixreco.so.
 */
#ifndef PIXRECO_DRIVER_H
#define PIXRECO_DRIVER_H

#include <stdint.h>

#include "pixreco.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  double   wall_s;                 /* first pr_acquire to last pr_produce, over all threads (A24)                  */
  double   acquire_us_median, acquire_us_mean, acquire_us_p99;   /* host time inside pr_acquire, per call           */
  uint64_t events, digis, clusters;
  uint64_t produce_polls;          /* pr_produce calls that answered PR_NOT_READY                                  */
  int32_t  status;                 /* PR_OK or the first error any thread saw                                      */
  uint32_t threads;
} prd_result;

/* Run `n_events` events: event e takes input pool[(first + e) % n_pool], slot e % n_slots and stream e % n_slots
 * (A25); a slot is acquired again only after its previous event was produced and released.  Thread t of `n_threads`
 * drives the slots s with s % n_threads == t, each slot through its own sequence of events (s, s + n_slots, ...), serving
 * whichever of its slots has completed (polling pr_produce): no slot waits for another slot's event.  t_start_ns / t_end_ns (may be NULL, else [n_events]) receive the
 * device time stamps of every event (pr_output.t_start_ns / t_end_ns).  `want` and `mem_kind` come with the inputs.
 * Returns res->status.                                                                                            */
int prd_run_streams(pr_event* const* slots, void* const* streams, uint32_t n_slots,
                    const pr_input* pool, uint32_t n_pool, uint32_t first, uint32_t n_events, uint32_t n_threads,
                    uint64_t* t_start_ns, uint64_t* t_end_ns, prd_result* res);

/* What one event produced, as the issuing thread saw it in pr_produce: the counters, and FNV-1a (64-bit, over
 * 32-bit words) fingerprints of the pinned-host mirrors h_label[n_digis] and h_cl_label[n_clusters] (0 when the
 * input's `want` did not ask for that mirror), so that a caller can check EVERY event of a multi-threaded run
 * against its own expectation.                                                                                   */
typedef struct {
  uint64_t event_id;
  uint32_t n_digis, n_errors, n_kept_digis, n_clusters_all, n_clusters, status_bits;
  uint32_t thread, pad;
  uint64_t hash_label, hash_cl_label;
} prd_event_record;

/* As prd_run_streams; rec (may be NULL, else [n_events]) receives one record per event.                          */
int prd_run_streams_rec(pr_event* const* slots, void* const* streams, uint32_t n_slots,
                        const pr_input* pool, uint32_t n_pool, uint32_t first, uint32_t n_events, uint32_t n_threads,
                        uint64_t* t_start_ns, uint64_t* t_end_ns, prd_event_record* rec, prd_result* res);

/* The consumer of the transfer stage: a "legacy" CPU module that wants one record per
 * cluster (array of structures) instead of the library's structure of arrays.  It reads the pinned-host mirrors of a
 * produced event — so the event must have been acquired with PR_WANT_CLUSTERS (| PR_WANT_HITS), or those must have
 * been fetched after the fact with pr_transfer — and writes min(n_clusters, cap) records into dst (host memory of the
 * caller).  Returns the number of records written, or PR_ERR_INVALID_ARG (NULL arguments) / PR_ERR_BAD_STATE (the
 * cluster mirrors are not there).  Hit fields are zero when the hit mirrors are absent.  Pure host code.          */
typedef struct {
  uint32_t label;                 /* canonical label = minimum digi index of the cluster (A10)                      */
  uint32_t size;
  uint16_t module, flags;         /* flags: hit border bits (A29)                                                   */
  float charge, row, col;         /* electrons; charge-weighted centroid in pixel units (A13)                       */
  float x_um, y_um, xerr_um, yerr_um;   /* hit position and error estimate (A26, A27, A30)                          */
  uint16_t row_min, row_max, col_min, col_max;   /* bounding box (A28)                                              */
} prd_cluster_aos;

int prd_clusters_to_aos(const pr_output* out, prd_cluster_aos* dst, uint32_t cap);

#ifdef __cplusplus
}
#endif
#endif /* PIXRECO_DRIVER_H */
