/* pixreco.h — C ABI of libpixreco: pixel-detector local reconstruction on one B200, behind the
 * acquire/produce split of arXiv:2004.04334.
 *
 * No C++ types and no exceptions cross this boundary.  `P:Lnn` cites /root/reference/PAPER.md
 * line nn; `BJ` cites BASELINE.json; `A<n>` cites the readings listed in DESIGN.md.
 *
 * The offload pattern (paper section 2 and 4):
 *   - acquire() launches the offloaded work and returns; produce() runs later, once the work is
 *     known to be complete ("External Worker").  Here: pr_acquire / pr_produce.
 *   - Completion is signalled by a callback queued into the CUDA stream, able to carry an error
 *     (P:L35), never by a blocking wait (P:L31 fn.1 lists the banned calls).  Here: the
 *     optional `done` callback and/or polling pr_query (cudaEventQuery, or a completion word in mapped memory).
 *   - Only asynchronous CUDA calls during event processing; work of one event is queued into ONE
 *     stream, different events' streams run concurrently.  The caller owns the stream.
 *   - Device and pinned-host memory come from a caching pool so that no runtime allocation API is
 *     called in steady state.  Here: pr_pool_* (hand-written, stream-aware).
 *   - A product carries {device, stream, completion event}; a consumer on another stream
 *     waits with cudaStreamWaitEvent.  Here: pr_event_cuda_event.
 *   - Transfers to the host happen only when asked for.  Here: pr_input.want.
 *
 * What is computed (BJ north_star (2); the paper itself describes no kernel):
 *   a1 unpack   raw u32 word -> digi (module,row,col,adc,wordIdx) or error (word,idx); both lists
 *               stable (original order); word format bit31=error, 30:20 module, 19:12 row,
 *               11:3 col, 2:0 reserved (A1-A4)
 *   a2 calib    charge = fmaf((float)adc, gain[module], pedestal[module]); kept iff >= pixel thr
 *   a3 cluster  per module, 8-connected components of kept digis; label = min digi index (A10)
 *   a4 reduce   per cluster exact int64 fixed-point (2^-14 e) sums -> size, charge, charge-
 *               weighted (row,col) centroid; kept iff charge >= cluster thr; kept clusters
 *               numbered in ascending label order (A9, A12, A13)
 *   hits        the step after clustering in the paper's Fig. 1: one hit per kept cluster —
 *               bounding box, local position from the exact sums (pixel centre = index + 0.5, origin
 *               at the module centre, times the pitch), border flags, error estimate (A26-A30)
 *
 * Threading: any host thread may use different pr_event objects concurrently; one pr_event is
 * used by one thread at a time.  Every entry point sets the CUDA device of its handle.
 * Non-blocking guarantee: pr_acquire, pr_query, pr_produce, pr_release never call a synchronising
 * CUDA API, and in steady state (pool warm) no cudaMalloc/cudaHostAlloc/cudaFree.
 * pr_create / pr_destroy / pr_event_create / pr_event_destroy / pr_pool_trim may block.
 */
#ifndef PIXRECO_H
#define PIXRECO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PR_ABI_VERSION 4

/* ---- return codes (int).  Negative = error.  pr_strerror() names them. ---- */
#define PR_OK               0
#define PR_NOT_READY        1   /* work still running: poll again or wait for the callback        */
#define PR_ERR_INVALID_ARG (-1)
#define PR_ERR_BAD_STATE   (-2) /* e.g. acquire on a busy slot, produce before acquire            */
#define PR_ERR_CAPACITY    (-3) /* an internal capacity was exceeded; never silent truncation     */
#define PR_ERR_INPUT_ORDER (-4) /* valid words not grouped by non-decreasing module (A5)          */
#define PR_ERR_BAD_CALIB   (-5) /* gain not finite / not in (0,128), |pedestal| >= 65536, thr<512 */
#define PR_ERR_OOM         (-6)
#define PR_ERR_CUDA        (-7) /* a CUDA call failed; sticky for the handle                      */

#define PR_INVALID_LABEL 0xFFFFFFFFu

/* pr_input.mem_kind: where `words` / `adc` live */
#define PR_MEM_HOST_PINNED 1u   /* page-locked host memory (pr_host_alloc or cudaHostAlloc)       */
#define PR_MEM_DEVICE      2u   /* device memory on the handle's device, 16-byte aligned, used in place */

/* pr_input.want: which outputs get a pinned-host mirror (exact-size copy) */
#define PR_WANT_DIGIS    0x01u  /* module,row,col,adc,word_idx, mod_digi_start */
#define PR_WANT_CHARGE   0x02u
#define PR_WANT_LABELS   0x04u  /* label, clus */
#define PR_WANT_CLUSTERS 0x08u  /* cluster SoA, mod_clus_start */
#define PR_WANT_ERRORS   0x10u
#define PR_WANT_HITS     0x20u  /* hit SoA (one hit per kept cluster: local position, errors, bounding box, edge flags) */
#define PR_WANT_ALL      0x3Fu

/* pr_output.status_bits (device-detected conditions) */
#define PR_STATUS_INPUT_ORDER 0x1u
#define PR_STATUS_CAPACITY    0x2u

typedef struct pr_handle pr_handle;  /* one per (process, device): calibration tables + pools      */
typedef struct pr_event  pr_event;   /* one in-flight event slot; reusable after pr_release        */
typedef struct pr_pool   pr_pool;    /* caching allocator                                  */

/* Completion callback.  Runs exactly once per pr_acquire that returned PR_OK, on a
 * CUDA-internal thread, after every output (and requested host mirror) is visible.  `status` is
 * what pr_produce will return.  It must not call any CUDA or pr_* function that enqueues work. */
typedef void (*pr_done_fn)(void* user, int status);

typedef struct {
  uint32_t struct_size;           /* = sizeof(pr_config); ABI versioning                          */
  int32_t  device;                /* CUDA ordinal                                                 */
  uint32_t n_modules;             /* 1..2048 (11-bit field)                                       */
  uint16_t n_rows, n_cols;        /* 1..256, 1..512 (8/9-bit fields); BJ configs: 160 x 416       */
  const float* gain;              /* host, [n_modules], finite, in (0,128); copied at create      */
  const float* pedestal;          /* host, [n_modules], finite, |p| < 65536; copied at create     */
  float    pixel_threshold_e;     /* keep digi iff charge >= this; must be >= 512 (A9)            */
  float    cluster_threshold_e;   /* keep cluster iff summed charge >= this                       */
  uint32_t max_words_hint;        /* pre-warm the pools for events of this many words (0 = none)  */
  uint32_t max_events_in_flight;  /* ... and this many concurrent events                          */
  uint64_t max_cached_bytes_device, max_cached_bytes_host;   /* pool caps, 0 = unlimited          */
  uint32_t flags;                 /* PR_FLAG_* mask                                               */
  float    pitch_row_um, pitch_col_um;   /* pixel pitch along the row index (local x) and the col index (local y) in um for
                                     the hits (A26); 0 = the defaults 100 and 150                  */
} pr_config;

/* pr_config.flags */
#define PR_FLAG_KERNEL_TIMING 0x1u /* record CUDA events around each kernel on its stream and sum the
                                      per-kernel device times into pr_stats (measurement aid; adds
                                      four cudaEventRecord per acquire)                            */

#define PR_FLAG_NO_GRAPH      0x2u /* never replay a single event's chain from a CUDA graph (see pr_acquire); for A/B
                                      measurements                                                 */

#define PR_FLAG_UNPACK_OVERSUBSCRIBE 0x4u /* test aid: launch k_unpack with eight times as many CTAs as fit the device
                                      at once.  Tiles are handed out by ticket, so a tile only ever waits for tiles of
                                      CTAs that are already running: the launch must end all the same    */

#define PR_FLAG_UNORDERED_INPUT 0x8u /* the words of an event may come in ANY order (reading A31; the step before the decode in
                                      the paper's Fig. 1): pr_acquire / pr_acquire_batch first bucket them
                                      stably by module on the device (error and out-of-range words last), then run the
                                      chain on the bucketed stream.  The digi list is then "by module, input order inside
                                      a module", the error list in input order, word_idx / err_idx are positions in the
                                      INPUT.  Costs three more launches and ~10 bytes per word of slab; the chained
                                      modules (pr_digis_acquire) answer PR_ERR_INVALID_ARG on such a handle           */

typedef struct {                  /* one event's input, filled by the caller before pr_acquire    */
  const uint32_t* words;          /* [n_words] raw words; caller-owned, valid until completion    */
  const uint16_t* adc;            /* [n_words] parallel ADC values (<= 4095)                      */
  uint32_t n_words;               /* may be 0 (A20)                                               */
  uint32_t mem_kind;              /* PR_MEM_HOST_PINNED | PR_MEM_DEVICE                           */
  uint32_t want;                  /* PR_WANT_* mask of pinned-host mirrors; 0 = counters only     */
  uint64_t event_id;              /* opaque, echoed in pr_output                                  */
  pr_done_fn done; void* user;    /* may be NULL: caller polls pr_query                           */
} pr_input;

/* Views into library-owned buffers; valid from a PR_OK pr_produce until pr_release(ev).
 * d_* are device pointers (always set); h_* are pinned-host mirrors (NULL unless in `want`).
 * Lengths: digi arrays n_digis; err arrays n_errors; cluster and hit arrays n_clusters;
 * mod_*_start n_modules+1.                                                                        */
typedef struct {
  uint64_t event_id;
  uint32_t n_words, n_digis, n_errors, n_kept_digis, n_clusters_all, n_clusters, status_bits, n_modules;
  uint64_t t_start_ns, t_end_ns;  /* device %globaltimer when the first kernel of the acquire started and when this
                                     event's counters were published: kernels of events on different streams may
                                     overlap; the intervals show whether they did                         */
  const uint16_t *d_module, *d_row, *d_col, *d_adc; const uint32_t* d_word_idx;
  const float* d_charge; const uint32_t* d_label; const int32_t* d_clus;
  const uint32_t *d_mod_digi_start, *d_mod_clus_start;
  const uint32_t *d_cl_label, *d_cl_size; const uint16_t* d_cl_module;
  const float *d_cl_charge, *d_cl_row, *d_cl_col;
  const uint32_t *d_err_word, *d_err_idx;
  const float *d_ht_x, *d_ht_y, *d_ht_xerr, *d_ht_yerr;   /* [n_clusters] um; hit k belongs to cluster k (A26, A27, A30) */
  const uint32_t *d_ht_rows, *d_ht_cols;                  /* minRow | maxRow << 16, minCol | maxCol << 16 (A28)          */
  const uint16_t* d_ht_flags;                             /* bit 0: touches row 0 or R-1, bit 1: col 0 or C-1 (A29)      */
  const uint16_t *h_module, *h_row, *h_col, *h_adc; const uint32_t* h_word_idx;
  const float* h_charge; const uint32_t* h_label; const int32_t* h_clus;
  const uint32_t *h_mod_digi_start, *h_mod_clus_start;
  const uint32_t *h_cl_label, *h_cl_size; const uint16_t* h_cl_module;
  const float *h_cl_charge, *h_cl_row, *h_cl_col;
  const uint32_t *h_err_word, *h_err_idx;
  const float *h_ht_x, *h_ht_y, *h_ht_xerr, *h_ht_yerr;
  const uint32_t *h_ht_rows, *h_ht_cols;
  const uint16_t* h_ht_flags;
} pr_output;

typedef struct {
  uint64_t hits, misses;            /* allocations served from the cache / by the backend         */
  uint64_t backend_allocs, backend_frees;   /* cudaMalloc|cudaHostAlloc and cudaFree|cudaFreeHost */
  uint64_t bytes_live, bytes_cached, bytes_peak;  /* handed out / idle in the cache / max(live+cached) */
  uint64_t cross_stream_reuses;     /* blocks reused on a different stream after their event completed */
} pr_pool_stats;

typedef struct {
  uint64_t events_acquired, events_produced, words, digis, clusters;
  uint64_t kernel_launches, memcpy_calls, callbacks_fired;
  uint32_t events_in_flight, max_events_in_flight;
  pr_pool_stats device_pool, host_pool;
  /* PR_FLAG_KERNEL_TIMING only: device time summed over `timed_acquires` completed acquires */
  uint64_t timed_acquires;
  double   unpack_ms, cluster_ms, finalize_ms, export_ms;
} pr_stats;

/* ---- handle: job start / job end (may block and allocate) ---- */
/* Validates cfg (PR_ERR_INVALID_ARG, PR_ERR_BAD_CALIB), uploads the calibration tables, creates
 * the two pools and pre-warms them per the hints.  *out is NULL on error.                        */
int pr_create(const pr_config* cfg, pr_handle** out);
/* Waits for the device to go idle, destroys remaining event slots, frees both pools.             */
int pr_destroy(pr_handle* h);

/* ---- event slots ---- */
int pr_event_create(pr_handle* h, pr_event** out);   /* creates the slot's cudaEvent; may allocate */
int pr_event_destroy(pr_event* ev);                  /* PR_ERR_BAD_STATE while work is in flight   */

/* acquire: enqueue ALL work of one event — optional H2D staging, unpack+calibrate+compact,
 * cluster+reduce, optional exact-size host mirrors, completion event, optional callback — on
 * `cuda_stream` (a cudaStream_t passed as void*, e.g. torch.cuda.Stream().cuda_stream; NULL is
 * the legacy default stream) and return at once.  Argument/state errors are returned here and
 * nothing is enqueued.  The slot must be idle (fresh or released).
 * A device-resident event without host mirrors is enqueued with ONE launch: the slot keeps an instantiated CUDA graph of
 * its chain (the three kernels and the completion event; the kernels leave the control words cleared behind them),
 * everything that changes from event to event travels in the descriptor, which is set as a parameter of the three
 * kernel nodes before the launch; the graph is rebuilt only when the event size class changes.  The paper
 * found CUDA graphs "too restrictive" for its modules in 2020; for one module's fixed chain they fit.     */
int pr_acquire(pr_event* ev, const pr_input* in, void* cuda_stream);
/* Same for a batch of n independent events processed by ONE chain of launches on one stream
 * (B200-first: one Run-3 event is ~1000x too small to fill the GPU).  All inputs share mem_kind
 * and want; `done` of inputs[0] fires once for the batch.  n in 1..4096.                          */
int pr_acquire_batch(pr_event* ev, const pr_input* inputs, uint32_t n, void* cuda_stream);
/* PR_OK when the slot's work is complete, PR_NOT_READY if not (never waits): cudaEventQuery on the
 * slot's event, or — for a one-event acquire replayed from the slot's CUDA graph — a load of the
 * completion word that the last CTA of the last kernel raises in mapped pinned memory after a
 * system-scope fence (every result of the acquire is visible to the host and to any stream then).  */
int pr_query(pr_event* ev);
/* produce: non-blocking.  PR_NOT_READY if called too early; otherwise fills *out and
 * returns PR_OK or the device-detected error (PR_ERR_INPUT_ORDER, PR_ERR_CAPACITY), in which case
 * the counters are set, array contents are undefined and the slot stays usable.                  */
int pr_produce(pr_event* ev, pr_output* out);
int pr_produce_batch(pr_event* ev, pr_output* outs, uint32_t n);   /* outs[n]; worst status returned */
/* Return the slot's buffers to the pools; invalidates pr_output views.  PR_NOT_READY if the work
 * has not completed yet, or its completion callback has not returned yet (nothing is released then).
 * The caller must have seen its own consumers of the d_* views complete (or use pr_release_on).  */
int pr_release(pr_event* ev);
/* The same when a consumer kernel queued on `consumer_stream` may still be reading the d_* views:
 * the buffers go back to the pool tagged with that stream and an event recorded on it now, so another stream
 * reuses them only after the consumer's work has completed (queried, never waited on).            */
int pr_release_on(pr_event* ev, void* consumer_stream);
/* Transfer on demand as a stage of its own (the copy to the host is a module of its own, run
 * only if something consumes it, and it learns about completion like any External Worker).  After a
 * pr_produce that returned PR_OK, enqueue exact-size DMA copies (cudaMemcpyAsync, sizes taken from the
 * event's counters) of the outputs in `want` that have no host mirror yet, on `cuda_stream` (any stream
 * of the device: the slot's work is complete), and return at once.  The slot is in flight again:
 * pr_query / pr_produce (/ `done`, may be NULL) as after pr_acquire; the next PR_OK pr_produce also fills
 * the h_* views of what was requested here.  PR_ERR_BAD_STATE unless the slot is complete and not
 * released; PR_ERR_INVALID_ARG for unknown bits; an event with a device-detected error transfers nothing. */
int pr_transfer(pr_event* ev, uint32_t want, void* cuda_stream, pr_done_fn done, void* user);
/* The slot's completion cudaEvent_t (as void*) for cudaStreamWaitEvent on a consumer's stream
 * (P:L108), valid between pr_acquire and pr_release.                                             */
void* pr_event_cuda_event(pr_event* ev);
/* Consumer-side synchronisation of P:L106-108: if the slot's work has already completed
 * (cudaEventQuery) return at once; otherwise make `consumer_stream` wait for it with
 * cudaStreamWaitEvent.  Never blocks the host.  After it returns PR_OK, work queued on
 * `consumer_stream` may read the slot's device buffers (addresses: a previous pr_produce of a same-
 * sized event on this slot, or any pr_produce after completion).                                 */
int pr_stream_wait_event(pr_event* ev, void* consumer_stream);

/* ---- chained modules (section 4.2; P:L76 Product<T> / ScopedContext) -------------------------------
 * The chain of pr_acquire as separate modules that hand a PRODUCT to one another without a host wait:
 *     raw --pr_digis_acquire--> digis --pr_clusters_acquire--> clusters + hits
 *                                  \--pr_occupancy_acquire--> kept digis and ADC sum per module (a parallel branch)
 * A product is what the paper's Product<T> carries: {device, the stream the producer's work was queued in, an event
 * recorded after it} plus the device views.  It is available as soon as the producer's acquire has returned — the
 * producer need not be complete — and stays valid until the producer's slot is released; pr_release of the producer
 * answers PR_NOT_READY while a consumer that took the product has not been released.
 * A consumer's acquire is the ScopedContext rule of P:L100 and L106-108: the FIRST consumer to ask for the product
 * reuses the producer's stream (its work is simply queued behind the producer's: no synchronisation at all); every
 * other consumer runs on the stream it brings along (`own_stream`) and makes it wait for the product's event with
 * cudaStreamWaitEvent, unless cudaEventQuery says the event has completed already.  *used_stream (may be NULL) receives
 * the stream the work went to.  Every module's slot completes like any other: pr_query / pr_produce / callback of
 * pr_input (digis) / pr_release; a consumer's pr_produce fills the digi views of the product it consumed as well.   */
typedef struct pr_product pr_product;
/* raw -> digis: optional H2D staging, unpack + calibrate + compact, digi counters to the host.  pr_produce on this slot
 * gives the digi and error views and n_digis / n_errors (cluster views NULL); `want` may hold DIGIS, CHARGE, ERRORS.  */
int pr_digis_acquire(pr_event* ev, const pr_input* in, void* cuda_stream);
/* The product of the slot's digis acquire (PR_ERR_BAD_STATE if there is none).  Never blocks.                         */
int pr_digis_product(pr_event* ev, pr_product** out);
/* {device, stream, event} of a product, as the paper's Product<T> exposes them.                             */
int pr_product_info(const pr_product* p, int32_t* device, void** cuda_stream, void** cuda_event);
/* digis -> clusters + hits on slot `ev` (idle, another slot than the producer's): the clustering and hit kernels of
 * pr_acquire on the product's digi views.  `want`: mirrors as in pr_input (any PR_WANT_* bit); `done`/`user`: completion
 * callback as in pr_input (may be NULL).  pr_produce on this slot gives everything pr_acquire's does.                   */
int pr_clusters_acquire(pr_event* ev, pr_product* digis, uint32_t want, void* own_stream, void** used_stream,
                        pr_done_fn done, void* user);
/* digis -> occupancy on slot `ev`: per module the number of kept digis (charge >= pixel threshold) and the sum of
 * their ADC values; both arrays [n_modules] are mirrored to pinned host memory (they are small).  All zero if the
 * product's input order was violated (PR_STATUS_INPUT_ORDER: module boundaries undefined).                            */
int pr_occupancy_acquire(pr_event* ev, pr_product* digis, void* own_stream, void** used_stream, pr_done_fn done, void* user);
/* produce of an occupancy slot: PR_NOT_READY if early; views valid until pr_release(ev).                             */
int pr_occupancy_produce(pr_event* ev, const uint32_t** d_count, const uint32_t** d_adc_sum,
                         const uint32_t** h_count, const uint32_t** h_adc_sum);

/* ---- raw -> digis without any allocation (for callers that cannot reach cudaMalloc) --------------------------------
 * The first step of the path — raw words -> digis + charge, the k_unpack of pr_acquire / pr_digis_acquire (the "raw to
 * digi" step of the paper's Fig. 1; readings A1-A7) — as ONE call that allocates nothing, for code under CUDA
 * graph capture, tight serving loops or harnesses that forbid cudaMalloc.  Inputs and outputs are the CALLER's device
 * buffers on the handle's device; the kernel's scratch (launch control words, counters, one look-back state per
 * 2048-word tile) is a file-scope __device__ array of pr_static_scratch_bytes() = 65792 bytes that every GPU holds from
 * the moment it loads the library until exit, which bounds the input: n_words <= PR_STATIC_MAX_WORDS, beyond that
 * PR_ERR_CAPACITY and nothing is enqueued.  The call enqueues one memset (what must start at zero is cleared on every
 * call: the array keeps the last call's contents) and two kernels on `cuda_stream` and returns at once; it calls no
 * cudaMalloc / cudaFree, no pool and no allocating library routine, and it waits for nothing.  Completion is the
 * caller's business (its stream).  ALL calls on one device share the one array: two calls whose work overlaps on the
 * GPU (different streams without an ordering between them) race on it — order them, or use pr_digis_acquire.
 * Arguments: d_words [n_words] u32 and d_adc [n_words] u16 (device, 16-byte aligned, used in place; may be NULL when
 * n_words == 0).  pr_digis_out: device buffers, every base 16-byte aligned, owned by the caller before and after:
 * d_module, d_row, d_col, d_adc u16 [cap]; d_word_idx u32 [cap]; d_charge f32 [cap]; d_err_word, d_err_idx u32 [cap],
 * cap = n_words rounded up to a multiple of 8 (at least 8); d_mod_digi_start u32 [n_modules + 1]; d_counters u32 [8]
 * = {n_words, n_digis, n_errors, 0, 0, 0, status_bits, 0}.  Elements beyond n_digis / n_errors are not written.  The
 * same values, bit for bit, as the digi part of pr_acquire (status bit 0 = PR_ERR_INPUT_ORDER: then
 * d_mod_digi_start is undefined).  Returns PR_OK, PR_ERR_INVALID_ARG (NULL or misaligned pointer), PR_ERR_CAPACITY,
 * PR_ERR_CUDA.  pr_static_setup looks the array's device address up (cudaGetSymbolAddress, once per device) ahead of
 * the first call — pr_unpack_static does it itself otherwise; call it before a stream capture begins.              */
#define PR_STATIC_MAX_WORDS (1u << 24)
typedef struct pr_digis_out {
  uint16_t *d_module, *d_row, *d_col, *d_adc;
  uint32_t* d_word_idx;
  float* d_charge;
  uint32_t *d_err_word, *d_err_idx;
  uint32_t* d_mod_digi_start;
  uint32_t* d_counters;
} pr_digis_out;
size_t pr_static_scratch_bytes(void);
int pr_static_setup(pr_handle* h);
int pr_unpack_static(pr_handle* h, const uint32_t* d_words, const uint16_t* d_adc, uint32_t n_words, const pr_digis_out* out,
                     void* cuda_stream);

/* ---- pinned host memory from the handle's host pool, for inputs ---- */
void* pr_host_alloc(pr_handle* h, size_t bytes);     /* NULL on failure */
int   pr_host_free(pr_handle* h, void* p);

int pr_get_stats(pr_handle* h, pr_stats* out);
const char* pr_strerror(int code);
/* Text of the last CUDA error seen by this handle ("" if none). Valid until the next pr_* call. */
const char* pr_last_cuda_error(pr_handle* h);
int pr_abi_version(void);

/* ---- the caching allocator itself (reading A23) ----
 * Requests are rounded up to bins (256 B .. 2^36 B, four bins per octave); a freed block
 * remembers the stream it was last used on and an event recorded at free; it is reused at once on
 * the same stream and on another stream only after that event is complete (queried, never
 * waited on).  Nothing is returned to the backend except by pr_pool_trim / pr_pool_destroy or when
 * the backend is out of memory.                                                                  */
#define PR_POOL_DEVICE 0   /* cudaMalloc / cudaFree on `device`                                   */
#define PR_POOL_PINNED 1   /* cudaHostAlloc(portable|mapped) / cudaFreeHost                       */
#define PR_POOL_FAKE   2   /* no CUDA at all: fake addresses + scripted event completion (tests)  */
int   pr_pool_create(int kind, int device, uint64_t max_cached_bytes, pr_pool** out);
void* pr_pool_alloc(pr_pool* p, size_t bytes, void* cuda_stream);            /* NULL on failure   */
/* `completed` != 0: the caller knows all work touching the block has finished (no event needed). */
int   pr_pool_free(pr_pool* p, void* ptr, void* cuda_stream, int completed);
int   pr_pool_trim(pr_pool* p, uint64_t keep_cached_bytes);                  /* may block         */
int   pr_pool_get_stats(pr_pool* p, pr_pool_stats* out);
int   pr_pool_destroy(pr_pool* p);
/* PR_POOL_FAKE only: declare everything recorded so far on `cuda_stream` complete.               */
int   pr_pool_fake_complete(pr_pool* p, void* cuda_stream);
/* Size a request of `bytes` is rounded up to (pure function; 0 if bytes exceeds the largest bin). */
uint64_t pr_pool_bin_bytes(uint64_t bytes);

#ifdef __cplusplus
}
#endif
#endif /* PIXRECO_H */
