// pixreco_api.cu — the C-ABI boundary of include/pixreco.h: handle, event slots, acquire/produce.
//
// pr_acquire is the body of the paper's acquire() with a ScopedContext around it (PAPER.md
// L76, L94, L100): set the device, take buffers from the caching pool (L88-90), enqueue copies
// and kernels on the event's own stream (L82-86), record the completion event and queue the
// completion callback (L94) — and return.  pr_produce is produce(): it only reads what the
// callback / event already made visible.  No blocking CUDA call appears in either (L31 fn.1).
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/pixreco.h"
#include "kernels.cuh"
#include "pool.hpp"

using namespace pixreco;

namespace {
enum SlotState { kIdle = 0, kInFlight = 1, kDone = 2 };
constexpr uint32_t kMaxBatch = 4096;
constexpr uint32_t kMaxExportItems = 25;      // arrays of one event that can get a host mirror

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
}  // namespace

struct pr_handle {
  pr_config cfg{};
  Geom geom{};
  float2* dCalib = nullptr;
  CachingPool *devPool = nullptr, *hostPool = nullptr;
  int smCount = 0, clusterBlocksPerSM = 1, unpackBlocksPerSM = 1;
  size_t clusterSmem = 0, denseSmem = 0;
  int denseBlocksPerSM = 1;
  std::mutex mu;
  std::vector<pr_event*> slots;
  std::atomic<uint64_t> evAcquired{0}, evProduced{0}, words{0}, digis{0}, clusters{0}, launches{0}, memcpys{0}, callbacks{0};
  std::atomic<uint32_t> inFlight{0}, maxInFlight{0};
  std::atomic<int> sticky{0};
  bool timing = false, noGraph = false;
  uint64_t timedAcquires = 0; double msUnpack = 0, msCluster = 0, msFinalize = 0, msExport = 0;   // guarded by mu
  std::string lastCuda;
};

struct SubEvent {            // host-side record of one event of the slot's batch
  pr_input in{};
  uint32_t cap = 0;
  EvDesc desc{};
  // pinned mirrors (nullptr unless wanted)
  pr_output hostViews{};
};

// What a module puts into the event for its consumers (the paper's Product<T>): device, the stream its work was
// queued in, the event recorded after it — and the device views (the digi part of the descriptor).
struct pr_product {
  pr_event* producer = nullptr;
  int device = 0;
  cudaStream_t stream = nullptr;
  cudaEvent_t event = nullptr;
  std::atomic<int> streamTaken{0};   // the first consumer to ask reuses `stream`
  std::atomic<int> consumers{0};     // consumers that took the product and have not been released yet
  EvDesc desc{};                     // digi views, modDigiStart, result (the producer's final counters on the device)
  uint32_t nWords = 0;
  bool valid = false;
};

enum ModuleKind { kFullChain = 0, kDigisModule = 1, kClustersModule = 2, kOccupancyModule = 3 };

struct pr_event {
  pr_handle* h = nullptr;
  int module = kFullChain;           // which module's work the slot holds (chained modules: P:L98-108)
  pr_product product;                // kDigisModule: what consumers take
  pr_product* consumed = nullptr;    // consumers: the product they took (released with the slot)
  uint32_t *occCount = nullptr, *occAdcSum = nullptr, *occHost = nullptr;   // kOccupancyModule: views into devSlab / hostSlab
  int state = kIdle;
  cudaEvent_t done = nullptr;
  cudaStream_t stream = nullptr;
  uint32_t n = 0;
  std::vector<SubEvent> sub;                 // grows only: no heap traffic in steady state
  std::vector<uint32_t*> stW; std::vector<uint16_t*> stA; std::vector<ExportItem> items;   // per-acquire scratch, kept
  // per-acquire pool blocks
  void* devSlab = nullptr; void* hostSlab = nullptr; void* descStage = nullptr; void* descDev = nullptr;
  bool ctlDirty = false;                    // the control block holds the counters of an acquire that ran outside the slot's graph
  // persistent per-slot blocks (grown on demand).  Control block: [LaunchCtl | counters | group counts | big-module list]
  // zeroed by one small memset per acquire, then [look-back states of k_unpack], which k_unpack's last CTA puts back
  // to zero itself (so that part is cleared only when the block is (re)allocated).
  void* ctl = nullptr; size_t ctlBytes = 0;
  size_t ctlZeroLast = 0;    // where the self-cleaning part began at the last acquire: if that moves, the whole block is cleared again
  HostCounters* hostCounters = nullptr; size_t hostCountersCap = 0;
  int status = PR_OK;        // filled when completion is observed
  pr_done_fn doneFn = nullptr; void* doneUser = nullptr;
  std::atomic<int> cbPending{0};             // a completion callback is queued and has not returned yet
  cudaEvent_t tev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // PR_FLAG_KERNEL_TIMING: start, unpack, cluster, finalize, export
  bool exported = false;
  bool transferStage = false;  // the work in flight is a pr_transfer: completion does not count the events again
  std::vector<void*> extraHost, extraDev;  // pinned / device blocks of pr_transfer stages, returned at release
  // last validated input pointers (their memory kind is not asked again)
  const void *lastWords = nullptr, *lastAdc = nullptr; uint32_t lastKind = 0;
  // the single-event chain as an instantiated CUDA graph: everything that changes between events travels in the
  // descriptor (gDescHost -> gDescDev by a copy node); rebuilt when the control block or the size class changes
  cudaGraphExec_t gExec = nullptr; cudaStream_t capStream = nullptr;
  EvDesc gDesc{}; bool gDescSet = false;   // the descriptor that the graph's k_cluster and k_finalize nodes hold
  bool flagDone = false;                    // this acquire went through the slot's graph: k_finalize's last CTA raises seq in the mapped counters when
                                            // everything is written, and poll() reads that word instead of asking the driver about `done`
  cudaGraph_t gGraph = nullptr; cudaGraphNode_t gNode[3] = {nullptr, nullptr, nullptr};   // the three kernel nodes: their parameters are set per launch
  uint32_t gUnpackGrid = 0, gPro = 0, gClusterGrid = 0, gModBatch = 0, gUnits = 0;
  LaunchCtl* gLc = nullptr; u64* gTileState = nullptr;
  EvDesc* gDescHost = nullptr; char* gDescDev = nullptr;      // [EvDesc][tile -> event map: zeros]
  void* gCtl = nullptr; uint32_t gTilesClass = 0; size_t gCtlZero = 0;
  uint64_t graphLaunches = 0, graphBuilds = 0;
};

namespace {

int cuda_fail(pr_handle* h, cudaError_t e, const char* what) {
  if (h) {
    std::lock_guard<std::mutex> g(h->mu);
    h->lastCuda = std::string(what) + ": " + cudaGetErrorString(e);
    h->sticky.store(1);
  }
  cudaGetLastError();
  return PR_ERR_CUDA;
}
#define PR_CUDA(h, call)                                   \
  do {                                                     \
    cudaError_t e__ = (call);                              \
    if (e__ != cudaSuccess) return cuda_fail((h), e__, #call); \
  } while (0)

// Carves arrays out of one slab; first pass (base == nullptr) only measures.
struct Carver {
  char* base; size_t off = 0;
  explicit Carver(void* b) : base((char*)b) {}
  template <typename T> T* take(size_t count) {
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += align_up(count * sizeof(T), 256);
    return p;
  }
};

// Device slab of one sub-event, digi part (what k_unpack writes).  `stage`: room for the H2D copy of the inputs.
void carve_digis(Carver& c, EvDesc& d, uint32_t cap, uint32_t M, bool stage, uint32_t** stageWords, uint16_t** stageAdc) {
  if (stage) { *stageWords = c.take<uint32_t>(cap); *stageAdc = c.take<uint16_t>(cap); }
  d.module = c.take<u16>(cap); d.row = c.take<u16>(cap); d.col = c.take<u16>(cap); d.adcOut = c.take<u16>(cap);
  d.wordIdx = c.take<u32>(cap); d.charge = c.take<float>(cap);
  d.errWord = c.take<u32>(cap); d.errIdx = c.take<u32>(cap);
  d.modDigiStart = c.take<u32>(M + 4);
  d.result = c.take<DevCounters>(1);
}
// ... and the cluster part (k_cluster / k_dense / k_finalize).
void carve_clusters(Carver& c, EvDesc& d, uint32_t cap, uint32_t M) {
  d.label = c.take<u32>(cap); d.clus = c.take<int32_t>(cap);
  d.modClusStart = c.take<u32>(M + 4);
  d.clLabel = c.take<u32>(cap); d.clSize = c.take<u32>(cap); d.clModule = c.take<u16>(cap);
  d.clCharge = c.take<float>(cap); d.clRow = c.take<float>(cap); d.clCol = c.take<float>(cap);
  d.htX = c.take<float>(cap); d.htY = c.take<float>(cap); d.htXerr = c.take<float>(cap); d.htYerr = c.take<float>(cap);
  d.htRows = c.take<u32>(cap); d.htCols = c.take<u32>(cap); d.htFlags = c.take<u16>(cap);
  d.modCount = c.take<u32>(M + 4);
  d.staged = c.take<StagedCluster>(cap);
  // touched only by modules beyond the shared-memory tiers
  d.wsPerm = c.take<u32>(cap); d.wsParent = c.take<u32>(cap); d.wsRoot = c.take<u32>(cap);
  d.wsKnum = c.take<int32_t>(cap); d.wsSize = c.take<u32>(cap);
  d.wsS = c.take<u64>(cap); d.wsSx = c.take<u64>(cap); d.wsSy = c.take<u64>(cap); d.wsBox = c.take<u32>((size_t)cap * 4);
}
// ... and the bucketed copy of the input for words in arbitrary order (A31; k_bucket.cuh)
void carve_bucket(Carver& c, BucketDesc& b, uint32_t cap, uint32_t M, uint32_t nTiles) {
  b.dstW = c.take<u32>(cap); b.dstA = c.take<u16>(cap); b.orig = c.take<u32>(cap);
  b.hist = c.take<u32>((size_t)(M + 1) * nTiles);
}
void carve_device(Carver& c, EvDesc& d, uint32_t cap, uint32_t M, bool stage, uint32_t** stageWords, uint16_t** stageAdc) {
  carve_digis(c, d, cap, M, stage, stageWords, stageAdc);
  carve_clusters(c, d, cap, M);
}

void carve_host(Carver& c, pr_output& o, uint32_t want, uint32_t cap, uint32_t M) {
  if (want & PR_WANT_DIGIS) {
    o.h_module = c.take<uint16_t>(cap); o.h_row = c.take<uint16_t>(cap); o.h_col = c.take<uint16_t>(cap);
    o.h_adc = c.take<uint16_t>(cap); o.h_word_idx = c.take<uint32_t>(cap); o.h_mod_digi_start = c.take<uint32_t>(M + 4);
  }
  if (want & PR_WANT_CHARGE) o.h_charge = c.take<float>(cap);
  if (want & PR_WANT_LABELS) { o.h_label = c.take<uint32_t>(cap); o.h_clus = c.take<int32_t>(cap); }
  if (want & PR_WANT_CLUSTERS) {
    o.h_cl_label = c.take<uint32_t>(cap); o.h_cl_size = c.take<uint32_t>(cap); o.h_cl_module = c.take<uint16_t>(cap);
    o.h_cl_charge = c.take<float>(cap); o.h_cl_row = c.take<float>(cap); o.h_cl_col = c.take<float>(cap);
    o.h_mod_clus_start = c.take<uint32_t>(M + 4);
  }
  if (want & PR_WANT_ERRORS) { o.h_err_word = c.take<uint32_t>(cap); o.h_err_idx = c.take<uint32_t>(cap); }
  if (want & PR_WANT_HITS) {
    o.h_ht_x = c.take<float>(cap); o.h_ht_y = c.take<float>(cap); o.h_ht_xerr = c.take<float>(cap); o.h_ht_yerr = c.take<float>(cap);
    o.h_ht_rows = c.take<uint32_t>(cap); o.h_ht_cols = c.take<uint32_t>(cap); o.h_ht_flags = c.take<uint16_t>(cap);
  }
}

int status_to_code(uint32_t bits) {
  if (bits & PR_STATUS_INPUT_ORDER) return PR_ERR_INPUT_ORDER;
  if (bits & PR_STATUS_CAPACITY) return PR_ERR_CAPACITY;
  return PR_OK;
}

// Runs on a CUDA-internal thread: translate device status into the code for done().
void CUDART_CB trampoline(void* p) {
  pr_event* ev = static_cast<pr_event*>(p);
  int worst = PR_OK;
  for (uint32_t k = 0; k < ev->n; ++k) {
    int c = status_to_code(ev->hostCounters[k].status);
    if (c < worst) worst = c;
  }
  ev->h->callbacks.fetch_add(1);
  if (ev->doneFn) ev->doneFn(ev->doneUser, worst);
  ev->cbPending.store(0, std::memory_order_release);   // only now may the slot be released, re-armed or destroyed
}

void destroy_graph(pr_event* ev) {
  pr_handle* h = ev->h;
  if (ev->gExec) { cudaGraphExecDestroy(ev->gExec); ev->gExec = nullptr; }
  if (ev->gGraph) { cudaGraphDestroy(ev->gGraph); ev->gGraph = nullptr; }
  if (ev->capStream) { cudaStreamDestroy(ev->capStream); ev->capStream = nullptr; }
  if (ev->gDescHost) { h->hostPool->free(ev->gDescHost, nullptr, true); ev->gDescHost = nullptr; }
  if (ev->gDescDev) { h->devPool->free(ev->gDescDev, nullptr, true); ev->gDescDev = nullptr; }
}

void release_blocks(pr_event* ev, bool completed) {
  pr_handle* h = ev->h;
  if (ev->consumed) { ev->consumed->consumers.fetch_sub(1); ev->consumed = nullptr; }   // the producer may be released now
  ev->product.valid = false;
  ev->module = kFullChain;
  if (ev->devSlab) { h->devPool->free(ev->devSlab, ev->stream, completed); ev->devSlab = nullptr; }
  if (ev->descDev) { h->devPool->free(ev->descDev, ev->stream, completed); ev->descDev = nullptr; }
  if (ev->hostSlab) { h->hostPool->free(ev->hostSlab, ev->stream, completed); ev->hostSlab = nullptr; }
  if (ev->descStage) { h->hostPool->free(ev->descStage, ev->stream, completed); ev->descStage = nullptr; }
  for (void* p : ev->extraHost) h->hostPool->free(p, ev->stream, completed);
  for (void* p : ev->extraDev) h->devPool->free(p, ev->stream, completed);
  ev->extraHost.clear(); ev->extraDev.clear();
}

// Whether [p, p + bytes) is memory of the kind the caller declared.  Pointers inside a live block of the handle's own
// pinned pool (pr_host_alloc) and the pointers validated by the slot's previous acquire need no CUDA call.
bool kind_ok(pr_event* ev, const void* words, const void* adc, uint32_t kind) {
  if (ev->lastKind == kind && ev->lastWords == words && ev->lastAdc == adc) return true;
  pr_handle* h = ev->h;
  bool ok;
  uintptr_t base; size_t bytes;
  if (kind == PR_MEM_HOST_PINNED && h->hostPool->find_live(words, &base, &bytes) && h->hostPool->find_live(adc, &base, &bytes)) ok = true;
  else {
    cudaPointerAttributes pa{}, pb{};
    if (cudaPointerGetAttributes(&pa, words) != cudaSuccess || cudaPointerGetAttributes(&pb, adc) != cudaSuccess) {
      cudaGetLastError();
      return false;
    }
    const cudaMemoryType need = kind == PR_MEM_DEVICE ? cudaMemoryTypeDevice : cudaMemoryTypeHost;
    ok = pa.type == need && pb.type == need;     // pageable host memory would make the copy synchronous
  }
  if (ok) { ev->lastWords = words; ev->lastAdc = adc; ev->lastKind = kind; }
  return ok;
}

// Something failed after work was queued: the slot goes back to idle, its blocks return to the pool tagged with the
// stream (reused elsewhere only after what was queued has run), the control block is dropped (its zeros are not
// guaranteed any more).  The handle is sticky-failed by PR_CUDA already.
int fail_after_enqueue(pr_event* ev, int code) {
  pr_handle* h = ev->h;
  release_blocks(ev, false);
  if (ev->ctl) { h->devPool->free(ev->ctl, ev->stream, false); ev->ctl = nullptr; ev->ctlBytes = 0; }
  ev->state = kIdle; ev->n = 0;
  return code;
}
#define PR_CUDA_Q(ev, call)                                 \
  do {                                                      \
    cudaError_t e__ = (call);                               \
    if (e__ != cudaSuccess) return fail_after_enqueue((ev), cuda_fail((ev)->h, e__, #call)); \
  } while (0)

// The chain of ONE device-resident event as a CUDA graph, recorded by stream capture on the slot's private stream (thread-
// local capture mode: other threads' CUDA calls are not affected) and instantiated: clear the per-acquire control words,
// upload the descriptor, k_unpack / k_cluster / k_finalize in their batch form with one event (the descriptor is read
// from device memory), record the completion event.  Grids are those of the size class; CTAs without a tile or a ticket
// leave at once.  Only here may a slot's acquire allocate (first use of a size class).
int build_graph(pr_event* ev, uint32_t tilesClass, size_t ctlZero, LaunchCtl* lc, u64* tileState, cudaStream_t stream) {
  (void)stream;
  pr_handle* h = ev->h;
  const uint32_t M = h->cfg.n_modules;
  if (ev->gExec) { cudaGraphExecDestroy(ev->gExec); ev->gExec = nullptr; }
  if (ev->gGraph) { cudaGraphDestroy(ev->gGraph); ev->gGraph = nullptr; }
  const uint32_t unitsPerEvent = (M + kFinMods - 1) / kFinMods;
  const uint64_t warpsResident = (uint64_t)h->smCount * h->clusterBlocksPerSM * (kClusterThreads / 32);
  const uint32_t modBatch = (uint64_t)M >= 4 * warpsResident ? kModBatch : (uint64_t)M >= 2 * warpsResident ? 2u : 1u;
  const uint64_t warpTickets = ((uint64_t)((M + modBatch - 1) / modBatch) + 7) / 8, maxDense = (uint64_t)tilesClass * kTileWords / (kWarpCap + 1);
  uint64_t wantCtas = warpTickets > maxDense ? warpTickets : maxDense;
  uint32_t clusterGrid = (uint32_t)(h->smCount * h->clusterBlocksPerSM);
  if (clusterGrid > wantCtas) clusterGrid = (uint32_t)wantCtas;
  if (clusterGrid < 1) clusterGrid = 1;
  uint32_t unpackGrid = (uint32_t)(h->smCount * h->unpackBlocksPerSM) * ((h->cfg.flags & PR_FLAG_UNPACK_OVERSUBSCRIBE) ? 8u : 1u);
  if (unpackGrid > tilesClass) unpackGrid = tilesClass;
  uint32_t pro = (tilesClass + unpackGrid - 1) / unpackGrid;
  if (pro >= 4) pro = 7;
  const uint32_t finSplits = 1;                                  // (the class stays below 8192 words per module group on average)
  cudaStream_t cs = ev->capStream;
  cudaGraph_t graph = nullptr;
  cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaStreamBeginCapture");
  // Three kernel nodes and the completion event, nothing else.  No memset node: the kernels leave the control words zeroed
  // behind them (k_unpack: tile ticket and look-back states; k_finalize with selfClean: module ticket, counters, group
  // counts).  No copy node: the event's descriptor is a kernel PARAMETER (the one-event form of the kernels), set on the
  // three nodes before every launch (graph_set_event) — a copy node cost ~4 us at the head of every event's chain, reading
  // the descriptor from mapped pinned memory inside k_unpack two PCIe round trips.
  const EvDesc& d0 = ev->sub[0].desc;
  k_unpack<true><<<unpackGrid, kUnpackThreads + 64, sizeof(UnpackShared), cs>>>(d0, nullptr, nullptr, d0.nTiles, pro, lc, tileState, h->geom, nullptr);
  k_cluster<true><<<clusterGrid, kClusterThreads, h->clusterSmem, cs>>>(d0, nullptr, 1, lc, nullptr, modBatch, h->geom);
  k_finalize<true><<<unitsPerEvent * finSplits, 256, 0, cs>>>(d0, nullptr, 1, unitsPerEvent, finSplits, 1u, lc, h->geom, 1u);
  cudaEventRecordWithFlags(ev->done, cs, cudaEventRecordExternal);   // an event-record NODE: ev->done stays an ordinary event the host can query
  e = cudaStreamEndCapture(cs, &graph);
  if (e != cudaSuccess || !graph) { cudaGetLastError(); return cuda_fail(h, e, "cudaStreamEndCapture"); }
  // the kernel nodes, by the function they launch
  cudaGraphNode_t nodes[8]; size_t nNodes = 8;
  ev->gNode[0] = ev->gNode[1] = ev->gNode[2] = nullptr;
  if (cudaGraphGetNodes(graph, nodes, &nNodes) == cudaSuccess) {
    for (size_t k = 0; k < nNodes && k < 8; ++k) {
      cudaGraphNodeType ty;
      cudaKernelNodeParams kp{};
      if (cudaGraphNodeGetType(nodes[k], &ty) != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
      if (cudaGraphKernelNodeGetParams(nodes[k], &kp) != cudaSuccess) continue;
      if (kp.func == (void*)k_unpack<true>) ev->gNode[0] = nodes[k];
      else if (kp.func == (void*)k_cluster<true>) ev->gNode[1] = nodes[k];
      else if (kp.func == (void*)k_finalize<true>) ev->gNode[2] = nodes[k];
    }
  }
  if (!ev->gNode[0] || !ev->gNode[1] || !ev->gNode[2]) { cudaGetLastError(); cudaGraphDestroy(graph); return cuda_fail(h, cudaErrorUnknown, "graph kernel nodes"); }
  e = cudaGraphInstantiate(&ev->gExec, graph, 0);
  if (e != cudaSuccess) { ev->gExec = nullptr; cudaGraphDestroy(graph); return cuda_fail(h, e, "cudaGraphInstantiate"); }
  ev->gGraph = graph;                                        // (the nodes belong to it)
  ev->gCtl = ev->ctl; ev->gTilesClass = tilesClass; ev->gCtlZero = ctlZero;
  ev->gUnpackGrid = unpackGrid; ev->gPro = pro; ev->gClusterGrid = clusterGrid; ev->gModBatch = modBatch; ev->gUnits = unitsPerEvent;
  ev->gLc = lc; ev->gTileState = tileState;
  ev->gDescSet = false;
  ++ev->graphBuilds;
  return PR_OK;
}

// The event of this launch: its descriptor (and its tile count) into the parameters of the graph's three kernel nodes.
int graph_set_event(pr_event* ev, const EvDesc& d0) {
  pr_handle* h = ev->h;
  const EvDesc* noBatch = nullptr; const u16* noMap = nullptr; u32* noList = nullptr; const EvDesc* noHost = nullptr;
  u32 one = 1, nTiles = d0.nTiles, pro = ev->gPro, modBatch = ev->gModBatch, units = ev->gUnits, splits = 1, groups = 1, clean = 1;
  LaunchCtl* lc = ev->gLc; u64* ts = ev->gTileState;
  void* aU[] = {(void*)&d0, &noBatch, &noMap, &nTiles, &pro, &lc, &ts, &h->geom, &noHost};
  void* aC[] = {(void*)&d0, &noBatch, &one, &lc, &noList, &modBatch, &h->geom};
  void* aF[] = {(void*)&d0, &noBatch, &one, &units, &splits, &groups, &lc, &h->geom, &clean};
  cudaKernelNodeParams kp{};
  kp.extra = nullptr;
  kp.func = (void*)k_unpack<true>; kp.gridDim = dim3(ev->gUnpackGrid); kp.blockDim = dim3(kUnpackThreads + 64); kp.sharedMemBytes = (unsigned)sizeof(UnpackShared); kp.kernelParams = aU;
  PR_CUDA(h, cudaGraphExecKernelNodeSetParams(ev->gExec, ev->gNode[0], &kp));
  // k_cluster and k_finalize read nothing of the descriptor that names the input (words, adc, nWords, tileBase, nTiles:
  // its first 28 bytes); the rest names the slot's own buffers, which the caching pool hands back event after event
  constexpr size_t kInputPart = offsetof(EvDesc, cap);
  if (ev->gDescSet && memcmp((const char*)&d0 + kInputPart, (const char*)&ev->gDesc + kInputPart, sizeof(EvDesc) - kInputPart) == 0) return PR_OK;
  kp.func = (void*)k_cluster<true>; kp.gridDim = dim3(ev->gClusterGrid); kp.blockDim = dim3(kClusterThreads); kp.sharedMemBytes = (unsigned)h->clusterSmem; kp.kernelParams = aC;
  PR_CUDA(h, cudaGraphExecKernelNodeSetParams(ev->gExec, ev->gNode[1], &kp));
  kp.func = (void*)k_finalize<true>; kp.gridDim = dim3(units * splits); kp.blockDim = dim3(256); kp.sharedMemBytes = 0; kp.kernelParams = aF;
  PR_CUDA(h, cudaGraphExecKernelNodeSetParams(ev->gExec, ev->gNode[2], &kp));
  ev->gDesc = d0; ev->gDescSet = true;
  return PR_OK;
}

int acquire_impl(pr_event* ev, const pr_input* ins, uint32_t n, void* cuda_stream) {
  if (!ev || !ins || n == 0 || n > kMaxBatch) return PR_ERR_INVALID_ARG;
  pr_handle* h = ev->h;
  if (h->sticky.load()) return PR_ERR_CUDA;
  if (ev->state != kIdle) return PR_ERR_BAD_STATE;
  const uint32_t M = h->cfg.n_modules, kind = ins[0].mem_kind, want = ins[0].want;
  if (kind != PR_MEM_HOST_PINNED && kind != PR_MEM_DEVICE) return PR_ERR_INVALID_ARG;
  if (want & ~PR_WANT_ALL) return PR_ERR_INVALID_ARG;
  PR_CUDA(h, cudaSetDevice(h->cfg.device));
  for (uint32_t k = 0; k < n; ++k) {
    const pr_input& in = ins[k];
    if (in.mem_kind != kind || in.want != want) return PR_ERR_INVALID_ARG;
    if (in.n_words && (!in.words || !in.adc)) return PR_ERR_INVALID_ARG;
    if (in.n_words > 0xFFFFFFF0u - kTileWords) return PR_ERR_INVALID_ARG;
    if (in.n_words) {
      if (kind == PR_MEM_DEVICE && (((uintptr_t)in.words | (uintptr_t)in.adc) & 15u)) return PR_ERR_INVALID_ARG;
      if (!kind_ok(ev, in.words, in.adc, kind)) return PR_ERR_INVALID_ARG;
    }
  }
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const bool stage = kind == PR_MEM_HOST_PINNED;
  const bool unordered = (h->cfg.flags & PR_FLAG_UNORDERED_INPUT) != 0;      // A31: bucket the words by module first

  // ---- host inputs of a batch that lie in ONE pinned block of the handle's pool and form a nearly dense span per array (a
  // DAQ buffer from pr_host_alloc, the bench's pool) are staged by ONE copy per array, each event keeping its offset
  // inside the span; anything else gets one copy per event and array (the gaps of a span were never handed to the library)
  uintptr_t wLo = ~(uintptr_t)0, wHi = 0, aLo = ~(uintptr_t)0, aHi = 0;
  bool merged = false;
  if (stage && n > 1) {
    size_t wSum = 0, aSum = 0;
    for (uint32_t k = 0; k < n; ++k) {
      if (!ins[k].n_words) continue;
      const uintptr_t w = (uintptr_t)ins[k].words, a = (uintptr_t)ins[k].adc;
      wLo = w < wLo ? w : wLo; wHi = w + 4 * (size_t)ins[k].n_words > wHi ? w + 4 * (size_t)ins[k].n_words : wHi;
      aLo = a < aLo ? a : aLo; aHi = a + 2 * (size_t)ins[k].n_words > aHi ? a + 2 * (size_t)ins[k].n_words : aHi;
      wSum += 4 * (size_t)ins[k].n_words; aSum += 2 * (size_t)ins[k].n_words;
    }
    merged = wSum > 0 && wHi - wLo <= wSum + wSum / 4 + 4096 && aHi - aLo <= aSum + aSum / 4 + 4096;
    if (merged) {
      uintptr_t bw, ba; size_t sw, sa;
      merged = h->hostPool->find_live((const void*)wLo, &bw, &sw) && wHi <= bw + sw &&
               h->hostPool->find_live((const void*)aLo, &ba, &sa) && aHi <= ba + sa;
    }
    for (uint32_t k = 0; merged && k < n; ++k)
      if (ins[k].n_words && ((((uintptr_t)ins[k].words - wLo) | ((uintptr_t)ins[k].adc - aLo)) & 15u)) merged = false;   // TMA wants 16-byte alignment
  }

  // ---- layout
  if (ev->sub.size() < n) { ev->sub.resize(n); ev->stW.resize(n); ev->stA.resize(n); }
  size_t devBytes = merged ? align_up(wHi - wLo, 256) + align_up(aHi - aLo, 256) : 0, hostBytes = 0;
  uint32_t totalTiles = 0;
  uint64_t totalWords = 0;
  for (uint32_t k = 0; k < n; ++k) {
    SubEvent& s = ev->sub[k];
    s.in = ins[k];
    s.cap = (uint32_t)align_up(s.in.n_words ? s.in.n_words : 1, 8);
    Carver cd(nullptr); EvDesc tmp{}; uint32_t* sw; uint16_t* sa;
    carve_device(cd, tmp, s.cap, M, stage && !merged, &sw, &sa);
    s.desc = EvDesc{};
    s.desc.tileBase = totalTiles;
    s.desc.nTiles = s.in.n_words ? (s.in.n_words + kTileWords - 1) / kTileWords : 1;
    if (unordered) { BucketDesc b{}; carve_bucket(cd, b, s.cap, M, s.desc.nTiles); }
    devBytes += cd.off;
    if (want) { Carver ch(nullptr); pr_output o{}; carve_host(ch, o, want, s.cap, M); hostBytes += ch.off; }
    totalTiles += s.desc.nTiles;
    totalWords += s.in.n_words;
  }
  const size_t grpPerEv = align_up((M + 31) / 32, 16);      // u32 per event
  // launches whose modules are large on average (configs[4]) hand their large modules to k_dense
  const bool denseKernel = totalWords > (uint64_t)kWarpCap * M * n;
  const size_t bigCap = denseKernel ? (size_t)(totalWords / (kWarpCap + 1) + 2) : 0;
  // control block: [LaunchCtl | counters | group counts | big list] (zeroed per acquire), [tile states] (self-cleaning)
  const size_t ctlZero = align_up(sizeof(LaunchCtl) + align_up(sizeof(DevCounters) * n, 64) + 4 * grpPerEv * n + 4 * bigCap, 256);
  // one device-resident event without mirrors: replayed from the slot's CUDA graph, built for its size class (tiles
  // rounded up to a power of two, at least 8) — the whole class must stay on the warp-ticket path
  uint32_t tilesClass = 8;
  while (tilesClass < totalTiles) tilesClass <<= 1;
  const bool useGraph = n == 1 && !stage && want == 0 && !h->timing && !h->noGraph && !unordered && ev->capStream &&
                        (uint64_t)tilesClass * kTileWords <= (uint64_t)kWarpCap * M && tilesClass <= 4096;
  const size_t ctlNeed = ctlZero + (size_t)8 * (useGraph ? tilesClass : totalTiles);

  // ---- buffers from the pools (steady state: cache hits only)
  bool ctlFresh = false;
  if (ev->ctlBytes < ctlNeed) {
    if (ev->ctl) h->devPool->free(ev->ctl, ev->stream, true);
    ev->ctl = h->devPool->alloc(ctlNeed, stream);
    ev->ctlBytes = ev->ctl ? (size_t)bin_bytes_for(ctlNeed) : 0;
    if (!ev->ctl) return PR_ERR_OOM;
    ctlFresh = true;
  }
  if (ev->ctlZeroLast != ctlZero) { ctlFresh = true; ev->ctlZeroLast = ctlZero; }   // another layout: its look-back states must start at zero too
  if (ev->hostCountersCap < n) {
    if (ev->hostCounters) h->hostPool->free(ev->hostCounters, ev->stream, true);
    ev->hostCounters = (HostCounters*)h->hostPool->alloc(sizeof(HostCounters) * n, stream);
    ev->hostCountersCap = ev->hostCounters ? n : 0;
    if (!ev->hostCounters) return PR_ERR_OOM;
  }
  ev->stream = stream;
  ev->devSlab = h->devPool->alloc(devBytes, stream);
  if (!ev->devSlab) return PR_ERR_OOM;
  if (want) {
    ev->hostSlab = h->hostPool->alloc(hostBytes, stream);
    if (!ev->hostSlab) { release_blocks(ev, true); return PR_ERR_OOM; }
  }
  // one block, one H2D copy: event descriptors and the tile -> event map (batches), then the export table (mirrors)
  const size_t descPart = n > 1 ? align_up(sizeof(EvDesc) * n + sizeof(u16) * totalTiles, 16) : 0;
  const size_t descBytes = descPart + (want ? sizeof(ExportItem) * kMaxExportItems * n : 0);
  if (descBytes) {
    ev->descStage = h->hostPool->alloc(descBytes, stream);
    ev->descDev = h->devPool->alloc(descBytes, stream);
    if (!ev->descStage || !ev->descDev) { release_blocks(ev, true); return PR_ERR_OOM; }
  }

  BucketDesc* bkHost = nullptr; BucketDesc* bkDev = nullptr;
  const size_t bkBytes = unordered ? sizeof(BucketDesc) * n + align_up(sizeof(u16) * totalTiles, 16) : 0;
  if (unordered) {
    bkHost = (BucketDesc*)h->hostPool->alloc(bkBytes, stream);
    bkDev = (BucketDesc*)h->devPool->alloc(bkBytes, stream);
    if (bkHost) ev->extraHost.push_back(bkHost);
    if (bkDev) ev->extraDev.push_back(bkDev);
    if (!bkHost || !bkDev) { release_blocks(ev, true); return PR_ERR_OOM; }
  }

  // ---- carve
  char* ctl = (char*)ev->ctl;
  LaunchCtl* lc = (LaunchCtl*)ctl;
  DevCounters* counters = (DevCounters*)(ctl + sizeof(LaunchCtl));
  u32* grpCount = (u32*)(ctl + sizeof(LaunchCtl) + align_up(sizeof(DevCounters) * n, 64));
  u32* bigList = denseKernel ? grpCount + grpPerEv * n : nullptr;
  u64* tileState = (u64*)(ctl + ctlZero);
  Carver cd(ev->devSlab), ch(ev->hostSlab);
  char *spanW = nullptr, *spanA = nullptr;
  if (merged) { spanW = cd.take<char>(wHi - wLo); spanA = cd.take<char>(aHi - aLo); }
  for (uint32_t k = 0; k < n; ++k) {
    SubEvent& s = ev->sub[k];
    EvDesc& d = s.desc;
    ev->stW[k] = nullptr; ev->stA[k] = nullptr;
    carve_device(cd, d, s.cap, M, stage && !merged, &ev->stW[k], &ev->stA[k]);
    if (merged && s.in.n_words) {
      ev->stW[k] = (uint32_t*)(spanW + ((uintptr_t)s.in.words - wLo)); ev->stA[k] = (uint16_t*)(spanA + ((uintptr_t)s.in.adc - aLo));
    }
    d.words = stage ? ev->stW[k] : s.in.words;
    d.adc = stage ? ev->stA[k] : s.in.adc;
    d.nWords = s.in.n_words; d.cap = s.cap;
    if (unordered) {                               // k_unpack reads the bucketed stream
      BucketDesc& b = bkHost[k];
      b = BucketDesc{};
      carve_bucket(cd, b, s.cap, M, d.nTiles);
      b.srcW = d.words; b.srcA = d.adc; b.wordIdx = d.wordIdx; b.errIdx = d.errIdx; b.counters = counters + k;
      b.nWords = d.nWords; b.nTiles = d.nTiles; b.tileBase = d.tileBase;
      d.words = b.dstW; d.adc = b.dstA;
      u16* te = (u16*)(bkHost + n);
      for (uint32_t t = 0; t < d.nTiles; ++t) te[d.tileBase + t] = (u16)k;
    }
    d.counters = counters + k; d.hostCounters = ev->hostCounters + k;
    d.tileState = tileState + d.tileBase;
    d.grpCount = grpCount + grpPerEv * k;
    s.hostViews = pr_output{};
    if (want) carve_host(ch, s.hostViews, want, s.cap, M);
    ev->hostCounters[k] = HostCounters{};
  }

  // ---- enqueue (all asynchronous, one stream: P:L82).  From here on a failure goes through fail_after_enqueue.
  uint64_t nMemcpy = 0, nLaunch = 0;
  if (useGraph) {
    // a new control block (look-back states too), or one that an acquire outside the graph left with its counters in it
    if (ctlFresh || ev->ctlDirty) PR_CUDA_Q(ev, cudaMemsetAsync(ev->ctl, 0, ctlFresh ? ev->ctlBytes : ctlZero, stream));
    ev->ctlDirty = false;
    if (!ev->gExec || ev->gCtl != ev->ctl || ev->gTilesClass != tilesClass || ev->gCtlZero != ctlZero) {
      int rc = build_graph(ev, tilesClass, ctlZero, lc, tileState, stream);
      if (rc != PR_OK) return fail_after_enqueue(ev, rc);
    }
    {
      int rc = graph_set_event(ev, ev->sub[0].desc);
      if (rc != PR_OK) return fail_after_enqueue(ev, rc);
    }
    PR_CUDA_Q(ev, cudaGraphLaunch(ev->gExec, stream));
    ev->flagDone = true;
    ++ev->graphLaunches;
    nLaunch = 3; nMemcpy = 0;
  } else {
  // tickets, counters, group counts: one small memset; the look-back states only when the block is new (k_unpack's last
  // CTA puts their zeros back, and those of its two ticket words, harmlessly cleared again here)
  PR_CUDA_Q(ev, cudaMemsetAsync(ev->ctl, 0, ctlFresh ? ev->ctlBytes : ctlZero, stream));
  ev->ctlDirty = true;                             // (only the slot's graph leaves the control words zeroed behind it)
  ev->flagDone = false;
  if (merged) {
    PR_CUDA_Q(ev, cudaMemcpyAsync(spanW, (const void*)wLo, wHi - wLo, cudaMemcpyHostToDevice, stream));
    PR_CUDA_Q(ev, cudaMemcpyAsync(spanA, (const void*)aLo, aHi - aLo, cudaMemcpyHostToDevice, stream));
    nMemcpy += 2;
  } else if (stage)
    for (uint32_t k = 0; k < n; ++k) {
      const SubEvent& s = ev->sub[k];
      if (!s.in.n_words) continue;
      PR_CUDA_Q(ev, cudaMemcpyAsync(ev->stW[k], s.in.words, (size_t)s.in.n_words * 4, cudaMemcpyHostToDevice, stream));
      PR_CUDA_Q(ev, cudaMemcpyAsync(ev->stA[k], s.in.adc, (size_t)s.in.n_words * 2, cudaMemcpyHostToDevice, stream));
      nMemcpy += 2;
    }
  // k_cluster: persistent CTAs (dense scan + warp tickets).  A small launch gets one CTA per warp
  // ticket or per possible dense module (a dense module has more than kWarpCap digis).
  // k_finalize: a CTA takes one group of 32 modules of one event; launches with many small groups (a Run-3-like batch:
  // under 1k digis per group) hand out 4 or 2 groups at a time (measured: 3 % less time there, 4 % more on the high
  // pile-up batch with its 3.4k digis per group, which keeps one group per CTA)
  const uint64_t finGroups = (uint64_t)n * ((M + kFinMods - 1) / kFinMods), wordsPerGroup = totalWords / (finGroups ? finGroups : 1);
  const uint32_t finGroupsPerUnit = finGroups < 32ull * h->smCount ? 1u : wordsPerGroup <= 1024 ? 4u : wordsPerGroup <= 2048 ? 2u : 1u;
  const uint32_t unitsPerEvent = (M + kFinMods * finGroupsPerUnit - 1) / (kFinMods * finGroupsPerUnit);
  // tickets of 4 modules when there are plenty, of 2 or 1 when the launch is small (a single event): every warp gets work
  const uint64_t warpsResident = (uint64_t)h->smCount * h->clusterBlocksPerSM * (kClusterThreads / 32);
  const uint32_t modBatch = (uint64_t)n * M >= 4 * warpsResident ? kModBatch : (uint64_t)n * M >= 2 * warpsResident ? 2u : 1u;
  const uint64_t warpTickets = ((uint64_t)n * ((M + modBatch - 1) / modBatch) + 7) / 8, maxDense = totalWords / (kWarpCap + 1);
  const uint64_t wantCtas = warpTickets > maxDense ? warpTickets : maxDense;
  uint32_t clusterGrid = (uint32_t)(h->smCount * h->clusterBlocksPerSM);
  if (clusterGrid > wantCtas) clusterGrid = (uint32_t)wantCtas;
  if (clusterGrid < 1) clusterGrid = 1;
  // k_finalize: one CTA per (event, 32 modules); huge events get several CTAs per group (about 8k words each)
  uint32_t finSplits = (uint32_t)(totalWords / ((uint64_t)n * unitsPerEvent * 8192 * finGroupsPerUnit) + 1);
  if (finSplits > 64) finSplits = 64;
  uint32_t denseGrid = (uint32_t)(h->smCount * h->denseBlocksPerSM);
  if (denseGrid > bigCap) denseGrid = bigCap ? (uint32_t)bigCap : 1u;
  // k_unpack: persistent CTAs taking tiles by ticket; a CTA holds at most `pro` tiles at a time (7 = a full pipeline)
  uint32_t unpackGrid = (uint32_t)(h->smCount * h->unpackBlocksPerSM) * ((h->cfg.flags & PR_FLAG_UNPACK_OVERSUBSCRIBE) ? 8u : 1u);
  if (unpackGrid > totalTiles) unpackGrid = totalTiles;
  uint32_t pro = (totalTiles + unpackGrid - 1) / unpackGrid;
  if (pro >= 4) pro = 7;
  // descriptor block: [EvDesc x n][tile -> event map] for batches, then the export table (exact-size mirrors)
  std::vector<ExportItem>& items = ev->items;
  items.clear();
  if (want) {
    for (uint32_t k = 0; k < n; ++k) {
      const EvDesc& d = ev->sub[k].desc; const pr_output& o = ev->sub[k].hostViews;
      auto add = [&](const void* src, const void* dst, uint32_t eb, uint32_t sel, uint32_t fixed) {
        if (dst) items.push_back(ExportItem{src, const_cast<void*>(dst), d.result, eb, sel, fixed, 0u});
      };
      add(d.module, o.h_module, 2, 0, 0); add(d.row, o.h_row, 2, 0, 0); add(d.col, o.h_col, 2, 0, 0);
      add(d.adcOut, o.h_adc, 2, 0, 0); add(d.wordIdx, o.h_word_idx, 4, 0, 0);
      add(d.modDigiStart, o.h_mod_digi_start, 4, 3, M + 1);
      add(d.charge, o.h_charge, 4, 0, 0); add(d.label, o.h_label, 4, 0, 0); add(d.clus, o.h_clus, 4, 0, 0);
      add(d.clLabel, o.h_cl_label, 4, 2, 0); add(d.clSize, o.h_cl_size, 4, 2, 0); add(d.clModule, o.h_cl_module, 2, 2, 0);
      add(d.clCharge, o.h_cl_charge, 4, 2, 0); add(d.clRow, o.h_cl_row, 4, 2, 0); add(d.clCol, o.h_cl_col, 4, 2, 0);
      add(d.modClusStart, o.h_mod_clus_start, 4, 3, M + 1);
      add(d.errWord, o.h_err_word, 4, 1, 0); add(d.errIdx, o.h_err_idx, 4, 1, 0);
      add(d.htX, o.h_ht_x, 4, 2, 0); add(d.htY, o.h_ht_y, 4, 2, 0); add(d.htXerr, o.h_ht_xerr, 4, 2, 0); add(d.htYerr, o.h_ht_yerr, 4, 2, 0);
      add(d.htRows, o.h_ht_rows, 4, 2, 0); add(d.htCols, o.h_ht_cols, 4, 2, 0); add(d.htFlags, o.h_ht_flags, 2, 2, 0);
    }
  }
  if (descBytes) {
    char* st8 = (char*)ev->descStage;
    if (n > 1) {
      EvDesc* st = (EvDesc*)st8;
      u16* te = (u16*)(st + n);
      for (uint32_t k = 0; k < n; ++k) {
        st[k] = ev->sub[k].desc;
        for (uint32_t t = 0; t < st[k].nTiles; ++t) te[st[k].tileBase + t] = (u16)k;
      }
    }
    if (!items.empty()) memcpy(st8 + descPart, items.data(), items.size() * sizeof(ExportItem));
    PR_CUDA_Q(ev, cudaMemcpyAsync(ev->descDev, st8, descPart + items.size() * sizeof(ExportItem), cudaMemcpyHostToDevice, stream));
    ++nMemcpy;
  }
  if (h->timing) PR_CUDA_Q(ev, cudaEventRecord(ev->tev[0], stream));
  if (unordered) {
    PR_CUDA_Q(ev, cudaMemcpyAsync(bkDev, bkHost, bkBytes, cudaMemcpyHostToDevice, stream));
    ++nMemcpy;
    const u16* te = (const u16*)(bkDev + n);
    k_bucket<false><<<totalTiles, kBucketThreads, 0, stream>>>(bkDev, te, h->geom);
    k_bucket_scan<<<n, 1024, 0, stream>>>(bkDev, h->geom);
    k_bucket<true><<<totalTiles, kBucketThreads, 0, stream>>>(bkDev, te, h->geom);
    nLaunch += 3;
  }
  const EvDesc& d0 = ev->sub[0].desc;
  if (n == 1) {
    k_unpack<true><<<unpackGrid, kUnpackThreads + 64, sizeof(UnpackShared), stream>>>(d0, nullptr, nullptr, totalTiles, pro, lc, tileState, h->geom, nullptr);
    if (h->timing) PR_CUDA_Q(ev, cudaEventRecord(ev->tev[1], stream));
    k_cluster<true><<<clusterGrid, kClusterThreads, h->clusterSmem, stream>>>(d0, nullptr, 1, lc, bigList, modBatch, h->geom);
    if (denseKernel) k_dense<true><<<denseGrid, kDenseThreads, h->denseSmem, stream>>>(d0, nullptr, lc, bigList, h->geom);
    if (h->timing) PR_CUDA_Q(ev, cudaEventRecord(ev->tev[2], stream));
    k_finalize<true><<<unitsPerEvent * finSplits, 256, 0, stream>>>(d0, nullptr, 1, unitsPerEvent, finSplits, finGroupsPerUnit, lc, h->geom, 0u);
  } else {
    const EvDesc* dd = (const EvDesc*)ev->descDev;
    k_unpack<false><<<unpackGrid, kUnpackThreads + 64, sizeof(UnpackShared), stream>>>(d0, dd, (const u16*)(dd + n), totalTiles, pro, lc, tileState, h->geom, nullptr);
    if (h->timing) PR_CUDA_Q(ev, cudaEventRecord(ev->tev[1], stream));
    k_cluster<false><<<clusterGrid, kClusterThreads, h->clusterSmem, stream>>>(d0, dd, n, lc, bigList, modBatch, h->geom);
    if (denseKernel) k_dense<false><<<denseGrid, kDenseThreads, h->denseSmem, stream>>>(d0, dd, lc, bigList, h->geom);
    if (h->timing) PR_CUDA_Q(ev, cudaEventRecord(ev->tev[2], stream));
    k_finalize<false><<<n * unitsPerEvent * finSplits, 256, 0, stream>>>(d0, dd, n, unitsPerEvent, finSplits, finGroupsPerUnit, lc, h->geom, 0u);
  }
  nLaunch += denseKernel ? 4 : 3;
  if (unordered) {                                 // wordIdx / errIdx: positions in the input, not in the bucketed stream
    uint32_t gx = (uint32_t)((totalWords / n + 1023) / 1024);
    if (gx < 1) gx = 1;
    if (gx > 256) gx = 256;
    k_unbucket_idx<<<dim3(gx, n), 256, 0, stream>>>(bkDev);
    ++nLaunch;
  }
  PR_CUDA_Q(ev, cudaGetLastError());
  if (h->timing) PR_CUDA_Q(ev, cudaEventRecord(ev->tev[3], stream));
  ev->exported = want != 0;
  if (want && !items.empty()) {
    const ExportItem* itab = (const ExportItem*)((const char*)ev->descDev + descPart);   // device-resident export table
    // The copies are bound by PCIe, not by the SMs: a few dozen CTAs with four 16-byte vectors in flight per thread
    // saturate the link, stay out of the way of the other acquires' kernels and stream item after item (a grid with
    // a CTA per item and 1024-vector slice measured 29.0k events/s end to end on the 256-event batches, this one 34-35k)
    uint32_t gy = (uint32_t)items.size();
    if (gy > 32) gy = 32;
    uint32_t gx = 32 / gy;
    k_export<<<dim3(gx, gy), 256, 0, stream>>>(itab, (uint32_t)items.size());
    ++nLaunch;
    PR_CUDA_Q(ev, cudaGetLastError());
  }
  if (h->timing && want) PR_CUDA_Q(ev, cudaEventRecord(ev->tev[4], stream));
  PR_CUDA_Q(ev, cudaEventRecord(ev->done, stream));
  }
  ev->n = n;
  ev->doneFn = ins[0].done; ev->doneUser = ins[0].user;
  ev->status = PR_OK;
  ev->state = kInFlight;
  ev->transferStage = false;
  if (ev->doneFn) {
    ev->cbPending.store(1, std::memory_order_release);
    cudaError_t ce = cudaLaunchHostFunc(stream, trampoline, ev);
    if (ce != cudaSuccess) {                      // the work is queued and will complete; only the callback is missing
      ev->cbPending.store(0);
      cuda_fail(h, ce, "cudaLaunchHostFunc");
    }
  }
  h->evAcquired.fetch_add(n); h->launches.fetch_add(nLaunch); h->memcpys.fetch_add(nMemcpy);
  h->words.fetch_add(totalWords);
  uint32_t f = h->inFlight.fetch_add(1) + 1, mx = h->maxInFlight.load();
  while (f > mx && !h->maxInFlight.compare_exchange_weak(mx, f)) {}
  return h->sticky.load() ? PR_ERR_CUDA : PR_OK;
}

// Non-blocking completion check; moves kInFlight -> kDone.
int poll(pr_event* ev) {
  if (ev->state == kDone) return PR_OK;
  if (ev->state != kInFlight) return PR_ERR_BAD_STATE;
  if (ev->flagDone) {
    if (*reinterpret_cast<const volatile uint32_t*>(&ev->hostCounters[0].seq) == 0u) return PR_NOT_READY;
    std::atomic_thread_fence(std::memory_order_acquire);
  } else {
    cudaError_t r = cudaEventQuery(ev->done);
    if (r == cudaErrorNotReady) { cudaGetLastError(); return PR_NOT_READY; }
    if (r != cudaSuccess) return cuda_fail(ev->h, r, "cudaEventQuery");
  }
  int worst = PR_OK; uint64_t dg = 0, cl = 0;
  for (uint32_t k = 0; k < ev->n; ++k) {
    const HostCounters& c = ev->hostCounters[k];
    int code = status_to_code(c.status);
    if (code < worst) worst = code;
    dg += c.nDigis; cl += c.nClusters;
  }
  ev->status = worst;
  ev->state = kDone;
  if (ev->transferStage) { ev->transferStage = false; ev->h->inFlight.fetch_sub(1); return PR_OK; }
  if (ev->h->timing) {
    float a = 0, b = 0, c = 0, f = 0;
    if (cudaEventElapsedTime(&a, ev->tev[0], ev->tev[1]) == cudaSuccess && cudaEventElapsedTime(&b, ev->tev[1], ev->tev[2]) == cudaSuccess &&
        cudaEventElapsedTime(&f, ev->tev[2], ev->tev[3]) == cudaSuccess) {
      if (ev->exported && cudaEventElapsedTime(&c, ev->tev[3], ev->tev[4]) != cudaSuccess) c = 0;
      std::lock_guard<std::mutex> g(ev->h->mu);
      ev->h->timedAcquires++; ev->h->msUnpack += a; ev->h->msCluster += b; ev->h->msFinalize += f; ev->h->msExport += c;
    } else cudaGetLastError();
  }
  ev->h->inFlight.fetch_sub(1);
  // chained modules: an event counts once, where it enters (digis) — its clusters where they are made
  if (ev->module == kFullChain || ev->module == kDigisModule) { ev->h->evProduced.fetch_add(ev->n); ev->h->digis.fetch_add(dg); }
  if (ev->module == kFullChain || ev->module == kClustersModule) ev->h->clusters.fetch_add(cl);
  return PR_OK;
}

void fill_output(pr_event* ev, uint32_t k, pr_output* out) {
  const SubEvent& s = ev->sub[k];
  const EvDesc& d = s.desc;
  const HostCounters& c = ev->hostCounters[k];
  *out = s.hostViews;
  out->event_id = s.in.event_id;
  out->n_words = c.nWords; out->n_digis = c.nDigis; out->n_errors = c.nErrors; out->n_kept_digis = c.nKept;
  out->n_clusters_all = c.nClustersAll; out->n_clusters = c.nClusters; out->status_bits = c.status;
  out->n_modules = ev->h->cfg.n_modules;
  out->t_start_ns = c.tStart; out->t_end_ns = c.tEnd;
  out->d_module = d.module; out->d_row = d.row; out->d_col = d.col; out->d_adc = d.adcOut; out->d_word_idx = d.wordIdx;
  out->d_charge = d.charge; out->d_label = d.label; out->d_clus = d.clus;
  out->d_mod_digi_start = d.modDigiStart; out->d_mod_clus_start = d.modClusStart;
  out->d_cl_label = d.clLabel; out->d_cl_size = d.clSize; out->d_cl_module = d.clModule;
  out->d_cl_charge = d.clCharge; out->d_cl_row = d.clRow; out->d_cl_col = d.clCol;
  out->d_err_word = d.errWord; out->d_err_idx = d.errIdx;
  out->d_ht_x = d.htX; out->d_ht_y = d.htY; out->d_ht_xerr = d.htXerr; out->d_ht_yerr = d.htYerr;
  out->d_ht_rows = d.htRows; out->d_ht_cols = d.htCols; out->d_ht_flags = d.htFlags;
}

}  // namespace

extern "C" {

int pr_abi_version(void) { return PR_ABI_VERSION; }

const char* pr_strerror(int code) {
  switch (code) {
    case PR_OK: return "ok";
    case PR_NOT_READY: return "not ready";
    case PR_ERR_INVALID_ARG: return "invalid argument";
    case PR_ERR_BAD_STATE: return "bad state for this call";
    case PR_ERR_CAPACITY: return "internal capacity exceeded";
    case PR_ERR_INPUT_ORDER: return "input words not grouped by non-decreasing module";
    case PR_ERR_BAD_CALIB: return "bad calibration table or threshold";
    case PR_ERR_OOM: return "out of memory";
    case PR_ERR_CUDA: return "CUDA error (see pr_last_cuda_error)";
    default: return "unknown code";
  }
}

const char* pr_last_cuda_error(pr_handle* h) {
  if (!h) return "";
  std::lock_guard<std::mutex> g(h->mu);
  return h->lastCuda.c_str();
}

int pr_create(const pr_config* cfg, pr_handle** out) {
  if (!out) return PR_ERR_INVALID_ARG;
  *out = nullptr;
  if (!cfg || cfg->struct_size != sizeof(pr_config)) return PR_ERR_INVALID_ARG;
  if (cfg->n_modules < 1 || cfg->n_modules > 2048 || cfg->n_rows < 1 || cfg->n_rows > 256 || cfg->n_cols < 1 ||
      cfg->n_cols > 512 || !cfg->gain || !cfg->pedestal || (cfg->flags & ~(PR_FLAG_KERNEL_TIMING | PR_FLAG_NO_GRAPH | PR_FLAG_UNPACK_OVERSUBSCRIBE | PR_FLAG_UNORDERED_INPUT)))
    return PR_ERR_INVALID_ARG;
  // A9/A21: ranges that make the 2^-14 fixed-point sums exact and overflow-free
  if (!(cfg->pixel_threshold_e >= 512.0f) || !std::isfinite(cfg->pixel_threshold_e) ||
      !std::isfinite(cfg->cluster_threshold_e) || !(std::fabs(cfg->cluster_threshold_e) < 1e12f))
    return PR_ERR_BAD_CALIB;
  if (!(cfg->pitch_row_um >= 0.0f) || !(cfg->pitch_col_um >= 0.0f) || !std::isfinite(cfg->pitch_row_um) || !std::isfinite(cfg->pitch_col_um))
    return PR_ERR_INVALID_ARG;
  for (uint32_t m = 0; m < cfg->n_modules; ++m) {
    const float g = cfg->gain[m], p = cfg->pedestal[m];
    if (!std::isfinite(g) || !(g > 0.0f) || !(g < 128.0f) || !std::isfinite(p) || !(std::fabs(p) < 65536.0f)) return PR_ERR_BAD_CALIB;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return PR_ERR_CUDA; }
  if (cfg->device < 0 || cfg->device >= ndev) return PR_ERR_INVALID_ARG;

  pr_handle* h = new (std::nothrow) pr_handle();
  if (!h) return PR_ERR_OOM;
  h->cfg = *cfg;
  h->cfg.gain = h->cfg.pedestal = nullptr;
  h->timing = (cfg->flags & PR_FLAG_KERNEL_TIMING) != 0;
  h->noGraph = (cfg->flags & PR_FLAG_NO_GRAPH) != 0;
  auto fail = [&](int code) { pr_destroy(h); return code; };
  if (cudaSetDevice(cfg->device) != cudaSuccess) { cudaGetLastError(); return fail(PR_ERR_CUDA); }
  cudaDeviceProp prop{};
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) { cudaGetLastError(); return fail(PR_ERR_CUDA); }
  h->smCount = prop.multiProcessorCount;
  {
    std::vector<float2> cal(cfg->n_modules);
    for (uint32_t m = 0; m < cfg->n_modules; ++m) cal[m] = make_float2(cfg->gain[m], cfg->pedestal[m]);
    const size_t tb = cal.size() * sizeof(float2);
    if (cudaMalloc(&h->dCalib, tb) != cudaSuccess) { cudaGetLastError(); return fail(PR_ERR_OOM); }
    if (cudaMemcpy(h->dCalib, cal.data(), tb, cudaMemcpyHostToDevice) != cudaSuccess) { cudaGetLastError(); return fail(PR_ERR_CUDA); }
  }
  Geom& g = h->geom;
  g.M = cfg->n_modules; g.R = cfg->n_rows; g.C = cfg->n_cols;
  g.stride = (g.C + 2 + 31) / 32;
  g.bitmapWords = (g.R + 2) * g.stride + 1;
  g.pixThr = cfg->pixel_threshold_e;
  g.clusThrFixed = (i64)llrint((double)cfg->cluster_threshold_e * 16384.0);
  g.pitchRow = cfg->pitch_row_um > 0.0f ? (double)cfg->pitch_row_um : 100.0;       // A26
  g.pitchCol = cfg->pitch_col_um > 0.0f ? (double)cfg->pitch_col_um : 150.0;
  g.calib = h->dCalib;
  h->clusterSmem = cluster_smem_bytes(g.bitmapWords);
  if (cudaFuncSetAttribute(k_cluster<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->clusterSmem) != cudaSuccess ||
      cudaFuncSetAttribute(k_cluster<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->clusterSmem) != cudaSuccess) {
    cudaGetLastError(); return fail(PR_ERR_CUDA);
  }
  h->denseSmem = dense_smem_bytes(g.bitmapWords, kDenseDigis, kDenseClusters);
  if (cudaFuncSetAttribute(k_dense<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->denseSmem) != cudaSuccess ||
      cudaFuncSetAttribute(k_dense<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->denseSmem) != cudaSuccess) {
    cudaGetLastError(); return fail(PR_ERR_CUDA);
  }
  int dps = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&dps, k_dense<true>, kDenseThreads, h->denseSmem) != cudaSuccess) { cudaGetLastError(); dps = 1; }
  h->denseBlocksPerSM = dps < 1 ? 1 : dps;
  int bps = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_cluster<true>, kClusterThreads, h->clusterSmem) != cudaSuccess) { cudaGetLastError(); bps = 1; }
  h->clusterBlocksPerSM = bps < 1 ? 1 : bps;
  if (cudaFuncSetAttribute(k_unpack<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(UnpackShared)) != cudaSuccess ||
      cudaFuncSetAttribute(k_unpack<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(UnpackShared)) != cudaSuccess) {
    cudaGetLastError(); return fail(PR_ERR_CUDA);
  }
  int ups = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ups, k_unpack<false>, kUnpackThreads + 64, sizeof(UnpackShared)) != cudaSuccess) { cudaGetLastError(); ups = 1; }
  h->unpackBlocksPerSM = ups < 1 ? 1 : ups;
  h->devPool = new CachingPool(make_device_backend(cfg->device), cfg->max_cached_bytes_device);
  h->hostPool = new CachingPool(make_pinned_backend(cfg->device), cfg->max_cached_bytes_host);

  // Pre-warm: run the allocation pattern of `max_events_in_flight` events of `max_words_hint`
  // words once, so the first real events hit the cache (the paper amortises API cost).
  if (cfg->max_words_hint && cfg->max_events_in_flight) {
    const uint32_t cap = (uint32_t)align_up(cfg->max_words_hint, 8);
    Carver cd(nullptr); EvDesc tmp{}; uint32_t* sw; uint16_t* sa;
    carve_device(cd, tmp, cap, g.M, true, &sw, &sa);
    const uint32_t tiles = (cap + kTileWords - 1) / kTileWords;
    const size_t ctlNeed = align_up(sizeof(LaunchCtl) + 64 + 4 * align_up((g.M + 31) / 32, 16), 256) + (size_t)8 * tiles;
    std::vector<void*> a, b, c;
    for (uint32_t i = 0; i < cfg->max_events_in_flight; ++i) {
      a.push_back(h->devPool->alloc(cd.off, nullptr));
      b.push_back(h->devPool->alloc(ctlNeed, nullptr));
      c.push_back(h->hostPool->alloc(sizeof(HostCounters), nullptr));
    }
    for (void* p : a) if (p) h->devPool->free(p, nullptr, true);
    for (void* p : b) if (p) h->devPool->free(p, nullptr, true);
    for (void* p : c) if (p) h->hostPool->free(p, nullptr, true);
  }
  *out = h;
  return PR_OK;
}

int pr_destroy(pr_handle* h) {
  if (!h) return PR_ERR_INVALID_ARG;
  cudaSetDevice(h->cfg.device);
  cudaDeviceSynchronize();                       // job end: allowed to block
  std::vector<pr_event*> slots;
  { std::lock_guard<std::mutex> g(h->mu); slots.swap(h->slots); }
  for (pr_event* ev : slots) {
    release_blocks(ev, true);
    if (ev->ctl) h->devPool->free(ev->ctl, nullptr, true);
    if (ev->hostCounters) h->hostPool->free(ev->hostCounters, nullptr, true);
    if (ev->done) cudaEventDestroy(ev->done);
    for (int i = 0; i < 5; ++i) if (ev->tev[i]) cudaEventDestroy(ev->tev[i]);
    destroy_graph(ev);
    delete ev;
  }
  delete h->devPool; delete h->hostPool;
  if (h->dCalib) cudaFree(h->dCalib);
  cudaGetLastError();
  delete h;
  return PR_OK;
}

int pr_event_create(pr_handle* h, pr_event** out) {
  if (!h || !out) return PR_ERR_INVALID_ARG;
  *out = nullptr;
  PR_CUDA(h, cudaSetDevice(h->cfg.device));
  pr_event* ev = new (std::nothrow) pr_event();
  if (!ev) return PR_ERR_OOM;
  ev->h = h;
  cudaError_t e = cudaEventCreateWithFlags(&ev->done, cudaEventDisableTiming);
  if (e != cudaSuccess) { delete ev; return cuda_fail(h, e, "cudaEventCreateWithFlags"); }
  if (h->timing)
    for (int i = 0; i < 5; ++i) PR_CUDA(h, cudaEventCreate(&ev->tev[i]));
  if (!h->noGraph && cudaStreamCreateWithFlags(&ev->capStream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); ev->capStream = nullptr; }
  { std::lock_guard<std::mutex> g(h->mu); h->slots.push_back(ev); }
  *out = ev;
  return PR_OK;
}

int pr_event_destroy(pr_event* ev) {
  if (!ev) return PR_ERR_INVALID_ARG;
  pr_handle* h = ev->h;
  if (ev->state == kInFlight && poll(ev) != PR_OK) return PR_ERR_BAD_STATE;
  if (ev->cbPending.load(std::memory_order_acquire)) return PR_ERR_BAD_STATE;   // its completion callback has not returned yet
  if (ev->product.consumers.load() > 0) return PR_ERR_BAD_STATE;               // a consumer still holds its product
  release_blocks(ev, true);
  if (ev->ctl) h->devPool->free(ev->ctl, ev->stream, true);
  if (ev->hostCounters) h->hostPool->free(ev->hostCounters, ev->stream, true);
  if (ev->done) cudaEventDestroy(ev->done);
  for (int i = 0; i < 5; ++i) if (ev->tev[i]) cudaEventDestroy(ev->tev[i]);
  destroy_graph(ev);
  {
    std::lock_guard<std::mutex> g(h->mu);
    for (size_t i = 0; i < h->slots.size(); ++i)
      if (h->slots[i] == ev) { h->slots.erase(h->slots.begin() + i); break; }
  }
  delete ev;
  return PR_OK;
}

int pr_acquire(pr_event* ev, const pr_input* in, void* cuda_stream) { return acquire_impl(ev, in, 1, cuda_stream); }
int pr_acquire_batch(pr_event* ev, const pr_input* ins, uint32_t n, void* cuda_stream) { return acquire_impl(ev, ins, n, cuda_stream); }

int pr_query(pr_event* ev) {
  if (!ev) return PR_ERR_INVALID_ARG;
  if (ev->state == kIdle) return PR_ERR_BAD_STATE;
  return poll(ev);
}

int pr_produce_batch(pr_event* ev, pr_output* outs, uint32_t n) {
  if (!ev || !outs) return PR_ERR_INVALID_ARG;
  if (ev->state == kIdle) return PR_ERR_BAD_STATE;
  int r = poll(ev);
  if (r != PR_OK) return r;
  if (n != ev->n) return PR_ERR_INVALID_ARG;
  for (uint32_t k = 0; k < n; ++k) fill_output(ev, k, outs + k);
  return ev->status;
}
int pr_produce(pr_event* ev, pr_output* out) { return pr_produce_batch(ev, out, 1); }

int pr_release(pr_event* ev) {
  if (!ev) return PR_ERR_INVALID_ARG;
  if (ev->state == kIdle) return PR_ERR_BAD_STATE;
  int r = poll(ev);
  if (r != PR_OK) return r;
  if (ev->cbPending.load(std::memory_order_acquire)) return PR_NOT_READY;   // the callback still reads the slot
  if (ev->product.consumers.load() > 0) return PR_NOT_READY;                // a consumer still holds this slot's product
  release_blocks(ev, true);                      // completion observed: reusable by any stream at once
  ev->state = kIdle;
  ev->n = 0;
  return PR_OK;
}

int pr_release_on(pr_event* ev, void* consumer_stream) {
  if (!ev) return PR_ERR_INVALID_ARG;
  if (ev->state == kIdle) return PR_ERR_BAD_STATE;
  int r = poll(ev);
  if (r != PR_OK) return r;
  if (ev->cbPending.load(std::memory_order_acquire)) return PR_NOT_READY;
  if (ev->product.consumers.load() > 0) return PR_NOT_READY;
  PR_CUDA(ev->h, cudaSetDevice(ev->h->cfg.device));
  ev->stream = (cudaStream_t)consumer_stream;    // the pool records an event on it and defers reuse by other streams
  release_blocks(ev, false);
  ev->state = kIdle;
  ev->n = 0;
  return PR_OK;
}

int pr_transfer(pr_event* ev, uint32_t want, void* cuda_stream, pr_done_fn done, void* user) {
  if (!ev || (want & ~PR_WANT_ALL)) return PR_ERR_INVALID_ARG;
  pr_handle* h = ev->h;
  if (h->sticky.load()) return PR_ERR_CUDA;
  if (ev->state == kIdle) return PR_ERR_BAD_STATE;
  if (ev->state == kInFlight && poll(ev) != PR_OK) return PR_ERR_BAD_STATE;
  if (ev->cbPending.load(std::memory_order_acquire)) return PR_ERR_BAD_STATE;
  PR_CUDA(h, cudaSetDevice(h->cfg.device));
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const uint32_t M = h->cfg.n_modules;
  struct Copy { const void* src; const void** view; size_t bytes; };
  std::vector<Copy> copies;
  size_t total = 0;
  for (uint32_t k = 0; k < ev->n; ++k) {
    SubEvent& s = ev->sub[k];
    const HostCounters& c = ev->hostCounters[k];
    if (status_to_code(c.status) != PR_OK) continue;           // outputs undefined: nothing to copy
    const EvDesc& d = s.desc; pr_output& o = s.hostViews;
    auto add = [&](const void* src, const void** view, size_t count, size_t eb) {
      if (*view) return;                                        // already mirrored
      copies.push_back(Copy{src, view, count * eb});
      total += align_up(count * eb ? count * eb : 1, 256);
    };
    const size_t D = c.nDigis, E = c.nErrors, N = c.nClusters;
    if (want & PR_WANT_DIGIS) {
      add(d.module, (const void**)&o.h_module, D, 2); add(d.row, (const void**)&o.h_row, D, 2); add(d.col, (const void**)&o.h_col, D, 2);
      add(d.adcOut, (const void**)&o.h_adc, D, 2); add(d.wordIdx, (const void**)&o.h_word_idx, D, 4);
      add(d.modDigiStart, (const void**)&o.h_mod_digi_start, M + 1, 4);
    }
    if (want & PR_WANT_CHARGE) add(d.charge, (const void**)&o.h_charge, D, 4);
    if (want & PR_WANT_LABELS) { add(d.label, (const void**)&o.h_label, D, 4); add(d.clus, (const void**)&o.h_clus, D, 4); }
    if (want & PR_WANT_CLUSTERS) {
      add(d.clLabel, (const void**)&o.h_cl_label, N, 4); add(d.clSize, (const void**)&o.h_cl_size, N, 4);
      add(d.clModule, (const void**)&o.h_cl_module, N, 2); add(d.clCharge, (const void**)&o.h_cl_charge, N, 4);
      add(d.clRow, (const void**)&o.h_cl_row, N, 4); add(d.clCol, (const void**)&o.h_cl_col, N, 4);
      add(d.modClusStart, (const void**)&o.h_mod_clus_start, M + 1, 4);
    }
    if (want & PR_WANT_ERRORS) { add(d.errWord, (const void**)&o.h_err_word, E, 4); add(d.errIdx, (const void**)&o.h_err_idx, E, 4); }
    if (want & PR_WANT_HITS) {
      add(d.htX, (const void**)&o.h_ht_x, N, 4); add(d.htY, (const void**)&o.h_ht_y, N, 4);
      add(d.htXerr, (const void**)&o.h_ht_xerr, N, 4); add(d.htYerr, (const void**)&o.h_ht_yerr, N, 4);
      add(d.htRows, (const void**)&o.h_ht_rows, N, 4); add(d.htCols, (const void**)&o.h_ht_cols, N, 4);
      add(d.htFlags, (const void**)&o.h_ht_flags, N, 2);
    }
  }
  char* slab = nullptr;
  if (total) {
    slab = (char*)h->hostPool->alloc(total, stream);
    if (!slab) return PR_ERR_OOM;
    ev->extraHost.push_back(slab);
  }
  size_t off = 0; uint64_t nMemcpy = 0, nLaunch = 0;
  if (copies.size() <= 4) {
    for (const Copy& c : copies) {
      *c.view = slab + off;
      if (c.bytes) { PR_CUDA(h, cudaMemcpyAsync(slab + off, c.src, c.bytes, cudaMemcpyDeviceToHost, stream)); ++nMemcpy; }
      off += align_up(c.bytes ? c.bytes : 1, 256);
    }
  } else {
    // many arrays (a batch): gather them on the device into one block laid out like the host slab, then ONE DMA copy.
    // The gather table goes up with one small copy; the sizes are exact because the counters are already on the host.
    const size_t tabBytes = align_up(sizeof(ExportItem) * copies.size(), 256);
    char* dstage = (char*)h->devPool->alloc(total + tabBytes, stream);
    ExportItem* htab = (ExportItem*)h->hostPool->alloc(tabBytes, stream);
    if (dstage) ev->extraDev.push_back(dstage);
    if (htab) ev->extraHost.push_back(htab);
    if (!dstage || !htab) return PR_ERR_OOM;
    uint32_t nItems = 0;
    for (const Copy& c : copies) {
      *c.view = slab + off;
      if (c.bytes) htab[nItems++] = ExportItem{c.src, dstage + tabBytes + off, nullptr, 1u, 3u, (uint32_t)c.bytes, 0u};
      off += align_up(c.bytes ? c.bytes : 1, 256);
    }
    if (nItems) {
      PR_CUDA(h, cudaMemcpyAsync(dstage, htab, sizeof(ExportItem) * nItems, cudaMemcpyHostToDevice, stream));
      k_export<<<dim3(4, nItems < 2048u ? nItems : 2048u), 256, 0, stream>>>((const ExportItem*)dstage, nItems);
      PR_CUDA(h, cudaGetLastError());
      PR_CUDA(h, cudaMemcpyAsync(slab, dstage + tabBytes, total, cudaMemcpyDeviceToHost, stream));
      nMemcpy += 2; nLaunch += 1;
    }
  }
  h->launches.fetch_add(nLaunch);
  PR_CUDA(h, cudaEventRecord(ev->done, stream));
  ev->stream = stream;
  ev->doneFn = done; ev->doneUser = user;
  ev->state = kInFlight;
  ev->transferStage = true;
  ev->flagDone = false;                          // this stage ends with `done`, recorded above
  if (done) {
    ev->cbPending.store(1, std::memory_order_release);
    cudaError_t ce = cudaLaunchHostFunc(stream, trampoline, ev);
    if (ce != cudaSuccess) { ev->cbPending.store(0); return cuda_fail(h, ce, "cudaLaunchHostFunc"); }
  }
  h->memcpys.fetch_add(nMemcpy);
  uint32_t f = h->inFlight.fetch_add(1) + 1, mx = h->maxInFlight.load();
  while (f > mx && !h->maxInFlight.compare_exchange_weak(mx, f)) {}
  return PR_OK;
}

void* pr_event_cuda_event(pr_event* ev) { return ev ? (void*)ev->done : nullptr; }

int pr_stream_wait_event(pr_event* ev, void* consumer_stream) {
  if (!ev) return PR_ERR_INVALID_ARG;
  if (ev->state == kIdle) return PR_ERR_BAD_STATE;
  if (ev->state == kDone) return PR_OK;
  PR_CUDA(ev->h, cudaSetDevice(ev->h->cfg.device));
  cudaError_t r = cudaEventQuery(ev->done);
  if (r == cudaSuccess) return PR_OK;
  if (r != cudaErrorNotReady) return cuda_fail(ev->h, r, "cudaEventQuery");
  cudaGetLastError();
  PR_CUDA(ev->h, cudaStreamWaitEvent((cudaStream_t)consumer_stream, ev->done, 0));
  return PR_OK;
}

void* pr_host_alloc(pr_handle* h, size_t bytes) { return h ? h->hostPool->alloc(bytes, nullptr) : nullptr; }
int pr_host_free(pr_handle* h, void* p) { return h ? h->hostPool->free(p, nullptr, true) : PR_ERR_INVALID_ARG; }

int pr_get_stats(pr_handle* h, pr_stats* out) {
  if (!h || !out) return PR_ERR_INVALID_ARG;
  memset(out, 0, sizeof *out);
  out->events_acquired = h->evAcquired.load(); out->events_produced = h->evProduced.load();
  out->words = h->words.load(); out->digis = h->digis.load(); out->clusters = h->clusters.load();
  out->kernel_launches = h->launches.load(); out->memcpy_calls = h->memcpys.load(); out->callbacks_fired = h->callbacks.load();
  out->events_in_flight = h->inFlight.load(); out->max_events_in_flight = h->maxInFlight.load();
  h->devPool->stats(&out->device_pool); h->hostPool->stats(&out->host_pool);
  {
    std::lock_guard<std::mutex> g(h->mu);
    out->timed_acquires = h->timedAcquires; out->unpack_ms = h->msUnpack; out->cluster_ms = h->msCluster; out->finalize_ms = h->msFinalize; out->export_ms = h->msExport;
  }
  return PR_OK;
}

}  // extern "C"

#include "chain_api.cuh"
#include "static_api.cuh"
