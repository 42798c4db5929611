// static_api.cuh — pr_unpack_static: raw words -> digis + charge (k_unpack, a1 + a2) for callers that may not allocate.
// Some callers cannot reach cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
// This one entry point touches neither the caching pool nor any allocator: inputs and outputs are the caller's device
// buffers, and k_unpack's scratch — its launch control words, the event's counters and one look-back state per tile —
// lives in a file-scope __device__ array of fixed size (kStaticScratchBytes = 65792 bytes, held by every GPU that loads
// the library until exit), which bounds the input at PR_STATIC_MAX_WORDS words.
// Included at the end of pixreco_api.cu: the array, the look-up of its device address and the launch are in ONE
// translation unit.  In host code the array's name is only a host-side stand-in for the symbol, never a device address:
// the address comes from cudaGetSymbolAddress, once per device, with that device current (static_scratch_for).
#pragma once

namespace {

constexpr uint32_t kStaticMaxTiles = PR_STATIC_MAX_WORDS / kTileWords;                                   // 8192
constexpr size_t kStaticCtlBytes = 256;                     // [LaunchCtl | DevCounters], as the control block of the chained modules
constexpr size_t kStaticScratchBytes = kStaticCtlBytes + (size_t)8 * kStaticMaxTiles;                    // 65792
static_assert(PR_STATIC_MAX_WORDS % kTileWords == 0, "whole tiles");
static_assert(sizeof(LaunchCtl) + sizeof(DevCounters) <= kStaticCtlBytes && sizeof(LaunchCtl) % 8 == 0, "control words fit their part of the scratch");

static __device__ __align__(256) unsigned char g_staticScratch[kStaticScratchBytes];

constexpr int kStaticMaxDevices = 64;
std::mutex g_staticMu;
void* g_staticPtr[kStaticMaxDevices] = {};                   // device address of g_staticScratch per device ordinal

// Device address of the scratch array on `device` (made current here).  nullptr and *err on failure.
void* static_scratch_for(int device, cudaError_t* err) {
  *err = cudaSuccess;
  if (device < 0 || device >= kStaticMaxDevices) { *err = cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> g(g_staticMu);
  if (g_staticPtr[device]) return g_staticPtr[device];
  cudaError_t e = cudaSetDevice(device);
  void* p = nullptr;
  if (e == cudaSuccess) e = cudaGetSymbolAddress(&p, g_staticScratch);
  if (e != cudaSuccess || !p) { *err = e != cudaSuccess ? e : cudaErrorInvalidSymbol; return nullptr; }
  g_staticPtr[device] = p;
  return p;
}

// The event's final counters from the scratch to the caller's buffer: 8 words, the layout of DevCounters.
__global__ void k_publish_static(const DevCounters* __restrict__ c, uint32_t* __restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  out[0] = c->nWords; out[1] = c->nDigis; out[2] = c->nErrors; out[3] = 0u; out[4] = 0u; out[5] = 0u; out[6] = c->status; out[7] = 0u;
}

}  // namespace

extern "C" {

size_t pr_static_scratch_bytes(void) { return kStaticScratchBytes; }

int pr_static_setup(pr_handle* h) {
  if (!h) return PR_ERR_INVALID_ARG;
  if (h->sticky.load()) return PR_ERR_CUDA;
  cudaError_t e;
  if (!static_scratch_for(h->cfg.device, &e)) return cuda_fail(h, e, "cudaGetSymbolAddress(static scratch)");
  return PR_OK;
}

int pr_unpack_static(pr_handle* h, const uint32_t* d_words, const uint16_t* d_adc, uint32_t n_words, const pr_digis_out* out,
                     void* cuda_stream) {
  if (!h || !out) return PR_ERR_INVALID_ARG;
  if (h->sticky.load()) return PR_ERR_CUDA;
  if (n_words > PR_STATIC_MAX_WORDS) return PR_ERR_CAPACITY;                 // the scratch holds one state per tile, no more
  if (n_words && (!d_words || !d_adc)) return PR_ERR_INVALID_ARG;
  if (!out->d_module || !out->d_row || !out->d_col || !out->d_adc || !out->d_word_idx || !out->d_charge || !out->d_err_word ||
      !out->d_err_idx || !out->d_mod_digi_start || !out->d_counters) return PR_ERR_INVALID_ARG;
  const uintptr_t al = (uintptr_t)d_words | (uintptr_t)d_adc | (uintptr_t)out->d_module | (uintptr_t)out->d_row | (uintptr_t)out->d_col |
                       (uintptr_t)out->d_adc | (uintptr_t)out->d_word_idx | (uintptr_t)out->d_charge | (uintptr_t)out->d_err_word |
                       (uintptr_t)out->d_err_idx | (uintptr_t)out->d_mod_digi_start | (uintptr_t)out->d_counters;
  if (al & 15u) return PR_ERR_INVALID_ARG;                                   // TMA bulk copies: 16-byte aligned bases
  cudaError_t e;
  unsigned char* scratch = (unsigned char*)static_scratch_for(h->cfg.device, &e);
  if (!scratch) return cuda_fail(h, e, "cudaGetSymbolAddress(static scratch)");
  PR_CUDA(h, cudaSetDevice(h->cfg.device));
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const uint32_t nTiles = n_words ? (n_words + kTileWords - 1) / kTileWords : 1;
  LaunchCtl* lc = (LaunchCtl*)scratch;
  EvDesc d{};
  d.words = d_words; d.adc = d_adc;
  d.nWords = n_words; d.tileBase = 0; d.nTiles = nTiles; d.cap = (uint32_t)align_up(n_words ? n_words : 1, 8);
  d.module = out->d_module; d.row = out->d_row; d.col = out->d_col; d.adcOut = out->d_adc; d.wordIdx = out->d_word_idx;
  d.charge = out->d_charge; d.errWord = out->d_err_word; d.errIdx = out->d_err_idx; d.modDigiStart = out->d_mod_digi_start;
  d.counters = (DevCounters*)(scratch + sizeof(LaunchCtl));
  d.tileState = (u64*)(scratch + kStaticCtlBytes);
  // every call shares the array, which keeps the last call's contents: the control words, the counters and this
  // launch's look-back states start at zero
  PR_CUDA(h, cudaMemsetAsync(scratch, 0, kStaticCtlBytes + (size_t)8 * nTiles, stream));
  uint32_t unpackGrid = (uint32_t)(h->smCount * h->unpackBlocksPerSM);
  if (unpackGrid > nTiles) unpackGrid = nTiles;
  uint32_t pro = (nTiles + unpackGrid - 1) / unpackGrid;
  if (pro >= 4) pro = 7;
  k_unpack<true><<<unpackGrid, kUnpackThreads + 64, sizeof(UnpackShared), stream>>>(d, nullptr, nullptr, nTiles, pro, lc, d.tileState, h->geom, nullptr);
  k_publish_static<<<1, 32, 0, stream>>>(d.counters, out->d_counters);
  PR_CUDA(h, cudaGetLastError());
  h->launches.fetch_add(2); h->words.fetch_add(n_words);
  return PR_OK;
}

}  // extern "C"
