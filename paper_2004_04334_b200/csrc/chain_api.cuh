// chain_api.cuh — the chained modules of include/pixreco.h (section 4.2; L76 Product<T> and
// ScopedContext): raw -> digis | digis -> clusters + hits | digis -> occupancy, each an acquire/produce module of its
// own on its own slot, passing a product {device, stream, event, views} and never waiting on the host in between.
// Included at the end of pixreco_api.cu (same translation unit: it uses that file's slot state machine and helpers).
#pragma once

namespace {

// Completion bookkeeping shared by the three chained acquires (the tail of acquire_impl).
int chained_finish(pr_event* ev, cudaStream_t stream, pr_done_fn done, void* user, uint64_t nLaunch, uint64_t nMemcpy, uint64_t words, bool entry) {
  pr_handle* h = ev->h;
  PR_CUDA_Q(ev, cudaGetLastError());
  PR_CUDA_Q(ev, cudaEventRecord(ev->done, stream));
  ev->n = 1;
  ev->doneFn = done; ev->doneUser = user;
  ev->status = PR_OK;
  ev->state = kInFlight;
  ev->transferStage = false;
  ev->exported = false;
  if (done) {
    ev->cbPending.store(1, std::memory_order_release);
    cudaError_t ce = cudaLaunchHostFunc(stream, trampoline, ev);
    if (ce != cudaSuccess) { ev->cbPending.store(0); cuda_fail(h, ce, "cudaLaunchHostFunc"); }
  }
  if (entry) h->evAcquired.fetch_add(1);      // an event counts once, where it enters the chain
  h->launches.fetch_add(nLaunch); h->memcpys.fetch_add(nMemcpy); h->words.fetch_add(words);
  uint32_t f = h->inFlight.fetch_add(1) + 1, mx = h->maxInFlight.load();
  while (f > mx && !h->maxInFlight.compare_exchange_weak(mx, f)) {}
  return h->sticky.load() ? PR_ERR_CUDA : PR_OK;
}

// The slot's persistent blocks for one event: control block of at least `ctlNeed` bytes (`*fresh` if it is new and
// needs a full clear) and one HostCounters record.
int chained_blocks(pr_event* ev, size_t ctlNeed, size_t ctlZero, cudaStream_t stream, bool* fresh) {
  pr_handle* h = ev->h;
  *fresh = false;
  if (ev->ctlBytes < ctlNeed) {
    if (ev->ctl) h->devPool->free(ev->ctl, ev->stream, true);
    ev->ctl = h->devPool->alloc(ctlNeed, stream);
    ev->ctlBytes = ev->ctl ? (size_t)bin_bytes_for(ctlNeed) : 0;
    if (!ev->ctl) return PR_ERR_OOM;
    *fresh = true;
  }
  if (ev->ctlZeroLast != ctlZero) { *fresh = true; ev->ctlZeroLast = ctlZero; }
  if (ev->hostCountersCap < 1) {
    if (ev->hostCounters) h->hostPool->free(ev->hostCounters, ev->stream, true);
    ev->hostCounters = (HostCounters*)h->hostPool->alloc(sizeof(HostCounters), stream);
    ev->hostCountersCap = ev->hostCounters ? 1 : 0;
    if (!ev->hostCounters) return PR_ERR_OOM;
  }
  if (ev->sub.size() < 1) { ev->sub.resize(1); ev->stW.resize(1); ev->stA.resize(1); }
  return PR_OK;
}

// ScopedContext of a consumer: the first consumer of a product reuses the producer's stream; any
// other one runs on its own stream, which waits for the product's event unless that has completed already.
int consumer_stream(pr_handle* h, pr_product* p, void* own_stream, cudaStream_t* out) {
  if (!p->streamTaken.exchange(1)) { *out = p->stream; return PR_OK; }
  cudaStream_t s = (cudaStream_t)own_stream;
  cudaError_t r = cudaEventQuery(p->event);
  if (r == cudaErrorNotReady) {
    cudaGetLastError();
    PR_CUDA(h, cudaStreamWaitEvent(s, p->event, 0));
  } else if (r != cudaSuccess) return cuda_fail(h, r, "cudaEventQuery");
  *out = s;
  return PR_OK;
}

int product_ok(pr_event* ev, pr_product* p) {
  if (!ev || !p || !p->valid || !p->producer) return PR_ERR_INVALID_ARG;
  if (p->producer == ev || p->producer->h != ev->h) return PR_ERR_INVALID_ARG;
  if (ev->h->sticky.load()) return PR_ERR_CUDA;
  if (ev->state != kIdle) return PR_ERR_BAD_STATE;
  if (p->producer->state == kIdle) return PR_ERR_BAD_STATE;
  return PR_OK;
}

}  // namespace

extern "C" {

int pr_digis_acquire(pr_event* ev, const pr_input* in, void* cuda_stream) {
  if (!ev || !in) return PR_ERR_INVALID_ARG;
  pr_handle* h = ev->h;
  if (h->sticky.load()) return PR_ERR_CUDA;
  if (ev->state != kIdle) return PR_ERR_BAD_STATE;
  if (h->cfg.flags & PR_FLAG_UNORDERED_INPUT) return PR_ERR_INVALID_ARG;                       // A31 is built into pr_acquire* only
  const uint32_t M = h->cfg.n_modules, kind = in->mem_kind, want = in->want;
  if (kind != PR_MEM_HOST_PINNED && kind != PR_MEM_DEVICE) return PR_ERR_INVALID_ARG;
  if (want & ~(PR_WANT_DIGIS | PR_WANT_CHARGE | PR_WANT_ERRORS)) return PR_ERR_INVALID_ARG;   // this module makes nothing else
  if (in->n_words && (!in->words || !in->adc)) return PR_ERR_INVALID_ARG;
  if (in->n_words > 0xFFFFFFF0u - kTileWords) return PR_ERR_INVALID_ARG;
  PR_CUDA(h, cudaSetDevice(h->cfg.device));
  if (in->n_words) {
    if (kind == PR_MEM_DEVICE && (((uintptr_t)in->words | (uintptr_t)in->adc) & 15u)) return PR_ERR_INVALID_ARG;
    if (!kind_ok(ev, in->words, in->adc, kind)) return PR_ERR_INVALID_ARG;
  }
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const bool stage = kind == PR_MEM_HOST_PINNED;
  const uint32_t cap = (uint32_t)align_up(in->n_words ? in->n_words : 1, 8);
  const uint32_t nTiles = in->n_words ? (in->n_words + kTileWords - 1) / kTileWords : 1;
  const size_t ctlZero = align_up(sizeof(LaunchCtl) + align_up(sizeof(DevCounters), 64), 256);
  bool fresh;
  int rc = chained_blocks(ev, ctlZero + (size_t)8 * nTiles, ctlZero, stream, &fresh);
  if (rc != PR_OK) return rc;
  SubEvent& s = ev->sub[0];
  s.in = *in; s.cap = cap; s.desc = EvDesc{}; s.hostViews = pr_output{};
  Carver measure(nullptr); EvDesc tmp{}; uint32_t* sw = nullptr; uint16_t* sa = nullptr;
  carve_digis(measure, tmp, cap, M, stage, &sw, &sa);
  size_t hostBytes = 0;
  if (want) { Carver ch(nullptr); pr_output o{}; carve_host(ch, o, want, cap, M); hostBytes = ch.off; }
  ev->stream = stream;
  ev->devSlab = h->devPool->alloc(measure.off, stream);
  if (!ev->devSlab) return PR_ERR_OOM;
  if (want) {
    ev->hostSlab = h->hostPool->alloc(hostBytes, stream);
    const size_t tab = sizeof(ExportItem) * kMaxExportItems;
    ev->descStage = h->hostPool->alloc(tab, stream);
    ev->descDev = h->devPool->alloc(tab, stream);
    if (!ev->hostSlab || !ev->descStage || !ev->descDev) { release_blocks(ev, true); return PR_ERR_OOM; }
  }
  char* ctl = (char*)ev->ctl;
  LaunchCtl* lc = (LaunchCtl*)ctl;
  EvDesc& d = s.desc;
  Carver cd(ev->devSlab), ch(ev->hostSlab);
  carve_digis(cd, d, cap, M, stage, &ev->stW[0], &ev->stA[0]);
  d.words = stage ? ev->stW[0] : in->words;
  d.adc = stage ? ev->stA[0] : in->adc;
  d.nWords = in->n_words; d.cap = cap; d.tileBase = 0; d.nTiles = nTiles;
  d.counters = (DevCounters*)(ctl + sizeof(LaunchCtl)); d.hostCounters = ev->hostCounters;
  d.tileState = (u64*)(ctl + ctlZero);
  if (want) carve_host(ch, s.hostViews, want, cap, M);
  ev->hostCounters[0] = HostCounters{};
  ev->module = kDigisModule;

  // ---- enqueue: clear the control words, stage the input, unpack, close the product
  uint64_t nMemcpy = 0, nLaunch = 0;
  PR_CUDA_Q(ev, cudaMemsetAsync(ev->ctl, 0, fresh ? ev->ctlBytes : ctlZero, stream));
  ev->ctlDirty = true; ev->flagDone = false;
  if (stage && in->n_words) {
    PR_CUDA_Q(ev, cudaMemcpyAsync(ev->stW[0], in->words, (size_t)in->n_words * 4, cudaMemcpyHostToDevice, stream));
    PR_CUDA_Q(ev, cudaMemcpyAsync(ev->stA[0], in->adc, (size_t)in->n_words * 2, cudaMemcpyHostToDevice, stream));
    nMemcpy += 2;
  }
  uint32_t unpackGrid = (uint32_t)(h->smCount * h->unpackBlocksPerSM);
  if (unpackGrid > nTiles) unpackGrid = nTiles;
  uint32_t pro = (nTiles + unpackGrid - 1) / unpackGrid;
  if (pro >= 4) pro = 7;
  k_unpack<true><<<unpackGrid, kUnpackThreads + 64, sizeof(UnpackShared), stream>>>(d, nullptr, nullptr, nTiles, pro, lc, d.tileState, h->geom, nullptr);
  k_publish_digis<<<1, 32, 0, stream>>>(d, lc);
  nLaunch += 2;
  if (want) {
    std::vector<ExportItem>& items = ev->items;
    items.clear();
    const pr_output& o = s.hostViews;
    auto add = [&](const void* src, const void* dst, uint32_t eb, uint32_t sel, uint32_t fixed) {
      if (dst) items.push_back(ExportItem{src, const_cast<void*>(dst), d.result, eb, sel, fixed, 0u});
    };
    add(d.module, o.h_module, 2, 0, 0); add(d.row, o.h_row, 2, 0, 0); add(d.col, o.h_col, 2, 0, 0);
    add(d.adcOut, o.h_adc, 2, 0, 0); add(d.wordIdx, o.h_word_idx, 4, 0, 0);
    add(d.modDigiStart, o.h_mod_digi_start, 4, 3, M + 1);
    add(d.charge, o.h_charge, 4, 0, 0);
    add(d.errWord, o.h_err_word, 4, 1, 0); add(d.errIdx, o.h_err_idx, 4, 1, 0);
    memcpy(ev->descStage, items.data(), items.size() * sizeof(ExportItem));
    PR_CUDA_Q(ev, cudaMemcpyAsync(ev->descDev, ev->descStage, items.size() * sizeof(ExportItem), cudaMemcpyHostToDevice, stream));
    uint32_t gx = (uint32_t)(((size_t)cap * 4 / 16 + 1023) / 1024);
    gx = gx < 1 ? 1 : gx > 64 ? 64 : gx;
    k_export<<<dim3(gx, (uint32_t)items.size()), 256, 0, stream>>>((const ExportItem*)ev->descDev, (uint32_t)items.size());
    ++nMemcpy; ++nLaunch;
  }
  rc = chained_finish(ev, stream, in->done, in->user, nLaunch, nMemcpy, in->n_words, true);
  if (rc != PR_OK) return rc;
  // the product: available at once; consumers synchronise through its event
  pr_product& p = ev->product;
  p.producer = ev; p.device = h->cfg.device; p.stream = stream; p.event = ev->done;
  p.streamTaken.store(0); p.consumers.store(0);
  p.desc = d; p.nWords = in->n_words; p.valid = true;
  return PR_OK;
}

// digis -> clusters + hits.  The consumer's descriptor is the product's digi views plus its own cluster part; its
// counters start as a copy of what the producer found (k_import_digis), the kernels are those of pr_acquire.
int pr_clusters_acquire(pr_event* ev, pr_product* p, uint32_t want, void* own_stream, void** used_stream, pr_done_fn done, void* user) {
  int rc = product_ok(ev, p);
  if (rc != PR_OK) return rc;
  if (want & ~PR_WANT_ALL) return PR_ERR_INVALID_ARG;
  pr_handle* h = ev->h;
  PR_CUDA(h, cudaSetDevice(h->cfg.device));
  const uint32_t M = h->cfg.n_modules, cap = p->desc.cap, nWords = p->nWords;
  const size_t grpPerEv = align_up((M + 31) / 32, 16);
  const bool denseKernel = nWords > (uint64_t)kWarpCap * M;
  const size_t bigCap = denseKernel ? (size_t)(nWords / (kWarpCap + 1) + 2) : 0;
  const size_t ctlZero = align_up(sizeof(LaunchCtl) + align_up(sizeof(DevCounters), 64) + 4 * grpPerEv + 4 * bigCap, 256);
  cudaStream_t stream;
  rc = consumer_stream(h, p, own_stream, &stream);
  if (rc != PR_OK) return rc;
  if (used_stream) *used_stream = (void*)stream;
  bool fresh;
  rc = chained_blocks(ev, ctlZero, ctlZero, stream, &fresh);
  if (rc != PR_OK) return rc;
  SubEvent& s = ev->sub[0];
  s.in = pr_input{}; s.in.n_words = nWords; s.in.want = want; s.in.event_id = p->producer->sub[0].in.event_id;
  s.cap = cap; s.hostViews = pr_output{};
  Carver measure(nullptr); EvDesc tmp{};
  carve_clusters(measure, tmp, cap, M); measure.take<DevCounters>(1);
  size_t hostBytes = 0;
  if (want) { Carver ch(nullptr); pr_output o{}; carve_host(ch, o, want, cap, M); hostBytes = ch.off; }
  ev->stream = stream;
  ev->devSlab = h->devPool->alloc(measure.off, stream);
  if (!ev->devSlab) return PR_ERR_OOM;
  if (want) {
    ev->hostSlab = h->hostPool->alloc(hostBytes, stream);
    const size_t tab = sizeof(ExportItem) * kMaxExportItems;
    ev->descStage = h->hostPool->alloc(tab, stream);
    ev->descDev = h->devPool->alloc(tab, stream);
    if (!ev->hostSlab || !ev->descStage || !ev->descDev) { release_blocks(ev, true); return PR_ERR_OOM; }
  }
  char* ctl = (char*)ev->ctl;
  LaunchCtl* lc = (LaunchCtl*)ctl;
  s.desc = p->desc;                      // the digi views are the producer's
  EvDesc& d = s.desc;
  Carver cd(ev->devSlab), ch(ev->hostSlab);
  carve_clusters(cd, d, cap, M);
  d.result = cd.take<DevCounters>(1);
  d.counters = (DevCounters*)(ctl + sizeof(LaunchCtl)); d.hostCounters = ev->hostCounters;
  d.grpCount = (u32*)(ctl + sizeof(LaunchCtl) + align_up(sizeof(DevCounters), 64));
  d.tileState = nullptr;
  u32* bigList = denseKernel ? d.grpCount + grpPerEv : nullptr;
  if (want) carve_host(ch, s.hostViews, want, cap, M);
  ev->hostCounters[0] = HostCounters{};
  ev->module = kClustersModule;
  ev->consumed = p; p->consumers.fetch_add(1);

  uint64_t nMemcpy = 0, nLaunch = 0;
  PR_CUDA_Q(ev, cudaMemsetAsync(ev->ctl, 0, fresh ? ev->ctlBytes : ctlZero, stream));
  ev->ctlDirty = true; ev->flagDone = false;
  const uint32_t unitsPerEvent = (M + kFinMods - 1) / kFinMods;
  const uint64_t warpsResident = (uint64_t)h->smCount * h->clusterBlocksPerSM * (kClusterThreads / 32);
  const uint32_t modBatch = (uint64_t)M >= 4 * warpsResident ? kModBatch : (uint64_t)M >= 2 * warpsResident ? 2u : 1u;
  const uint64_t warpTickets = ((uint64_t)((M + modBatch - 1) / modBatch) + 7) / 8, maxDense = nWords / (kWarpCap + 1);
  const uint64_t wantCtas = warpTickets > maxDense ? warpTickets : maxDense;
  uint32_t clusterGrid = (uint32_t)(h->smCount * h->clusterBlocksPerSM);
  if (clusterGrid > wantCtas) clusterGrid = (uint32_t)wantCtas;
  if (clusterGrid < 1) clusterGrid = 1;
  uint32_t finSplits = (uint32_t)(nWords / ((uint64_t)unitsPerEvent * 8192) + 1);
  if (finSplits > 64) finSplits = 64;
  uint32_t denseGrid = (uint32_t)(h->smCount * h->denseBlocksPerSM);
  if (denseGrid > bigCap) denseGrid = bigCap ? (uint32_t)bigCap : 1u;
  k_import_digis<<<1, 32, 0, stream>>>(d.counters, p->desc.result, lc);
  k_cluster<true><<<clusterGrid, kClusterThreads, h->clusterSmem, stream>>>(d, nullptr, 1, lc, bigList, modBatch, h->geom);
  if (denseKernel) k_dense<true><<<denseGrid, kDenseThreads, h->denseSmem, stream>>>(d, nullptr, lc, bigList, h->geom);
  k_finalize<true><<<unitsPerEvent * finSplits, 256, 0, stream>>>(d, nullptr, 1, unitsPerEvent, finSplits, 1u, lc, h->geom, 0u);
  nLaunch += denseKernel ? 4 : 3;
  if (want) {
    std::vector<ExportItem>& items = ev->items;
    items.clear();
    const pr_output& o = s.hostViews;
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
    memcpy(ev->descStage, items.data(), items.size() * sizeof(ExportItem));
    PR_CUDA_Q(ev, cudaMemcpyAsync(ev->descDev, ev->descStage, items.size() * sizeof(ExportItem), cudaMemcpyHostToDevice, stream));
    uint32_t gx = (uint32_t)(((size_t)cap * 4 / 16 + 1023) / 1024);
    gx = gx < 1 ? 1 : gx > 64 ? 64 : gx;
    k_export<<<dim3(gx, (uint32_t)items.size()), 256, 0, stream>>>((const ExportItem*)ev->descDev, (uint32_t)items.size());
    ++nMemcpy; ++nLaunch;
  }
  return chained_finish(ev, stream, done, user, nLaunch, nMemcpy, 0, false);
}

// digis -> occupancy: the second consumer, on a parallel branch of the module graph.
int pr_occupancy_acquire(pr_event* ev, pr_product* p, void* own_stream, void** used_stream, pr_done_fn done, void* user) {
  int rc = product_ok(ev, p);
  if (rc != PR_OK) return rc;
  pr_handle* h = ev->h;
  PR_CUDA(h, cudaSetDevice(h->cfg.device));
  const uint32_t M = h->cfg.n_modules;
  cudaStream_t stream;
  rc = consumer_stream(h, p, own_stream, &stream);
  if (rc != PR_OK) return rc;
  if (used_stream) *used_stream = (void*)stream;
  bool fresh;
  rc = chained_blocks(ev, 256, ev->ctlZeroLast, stream, &fresh);     // no control words of its own: whatever the block holds stays
  if (rc != PR_OK) return rc;
  const size_t arr = align_up((size_t)M * 4, 256);
  ev->stream = stream;
  ev->devSlab = h->devPool->alloc(2 * arr, stream);
  ev->hostSlab = h->hostPool->alloc(2 * arr, stream);
  if (!ev->devSlab || !ev->hostSlab) { release_blocks(ev, true); return PR_ERR_OOM; }
  ev->occCount = (uint32_t*)ev->devSlab; ev->occAdcSum = (uint32_t*)((char*)ev->devSlab + arr);
  ev->occHost = (uint32_t*)ev->hostSlab;
  SubEvent& s = ev->sub[0];
  s.in = pr_input{}; s.in.n_words = p->nWords; s.in.event_id = p->producer->sub[0].in.event_id;
  s.cap = p->desc.cap; s.desc = p->desc; s.hostViews = pr_output{};
  ev->hostCounters[0] = HostCounters{};
  ev->module = kOccupancyModule;
  ev->consumed = p; p->consumers.fetch_add(1);
  if (fresh) PR_CUDA_Q(ev, cudaMemsetAsync(ev->ctl, 0, ev->ctlBytes, stream));
  uint32_t grid = (M + 7) / 8;
  if (grid > (uint32_t)h->smCount * 8u) grid = (uint32_t)h->smCount * 8u;
  k_occupancy<<<grid, 256, 0, stream>>>(p->desc, p->desc.result, ev->occCount, ev->occAdcSum, ev->hostCounters, h->geom);
  PR_CUDA_Q(ev, cudaMemcpyAsync(ev->hostSlab, ev->devSlab, 2 * arr, cudaMemcpyDeviceToHost, stream));
  return chained_finish(ev, stream, done, user, 1, 1, 0, false);
}

int pr_occupancy_produce(pr_event* ev, const uint32_t** d_count, const uint32_t** d_adc_sum, const uint32_t** h_count, const uint32_t** h_adc_sum) {
  if (!ev) return PR_ERR_INVALID_ARG;
  if (ev->state == kIdle || ev->module != kOccupancyModule) return PR_ERR_BAD_STATE;
  int r = poll(ev);
  if (r != PR_OK) return r;
  const size_t arr = align_up((size_t)ev->h->cfg.n_modules * 4, 256);
  if (d_count) *d_count = ev->occCount;
  if (d_adc_sum) *d_adc_sum = ev->occAdcSum;
  if (h_count) *h_count = ev->occHost;
  if (h_adc_sum) *h_adc_sum = (const uint32_t*)((const char*)ev->occHost + arr);
  return ev->status;
}

int pr_digis_product(pr_event* ev, pr_product** out) {
  if (!ev || !out) return PR_ERR_INVALID_ARG;
  *out = nullptr;
  if (ev->state == kIdle || ev->module != kDigisModule || !ev->product.valid) return PR_ERR_BAD_STATE;
  *out = &ev->product;
  return PR_OK;
}

int pr_product_info(const pr_product* p, int32_t* device, void** cuda_stream, void** cuda_event) {
  if (!p || !p->valid) return PR_ERR_INVALID_ARG;
  if (device) *device = p->device;
  if (cuda_stream) *cuda_stream = (void*)p->stream;
  if (cuda_event) *cuda_event = (void*)p->event;
  return PR_OK;
}

}  // extern "C"
