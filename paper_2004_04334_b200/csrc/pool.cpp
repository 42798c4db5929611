// pool.cpp — see pool.hpp.  Host-only C++; the CUDA backends use the runtime API.
#include "pool.hpp"

#include <cuda_runtime_api.h>

#include <algorithm>
#include <map>

namespace pixreco {

// Four bins per octave: 2^k * {1, 1.25, 1.5, 1.75}; every bin is a multiple of 64 B for k >= 8.
uint64_t bin_bytes_for(uint64_t bytes) {
  if (bytes <= (1ull << kMinBinLog2)) return 1ull << kMinBinLog2;
  if (bytes > (1ull << kMaxBinLog2)) return 0;
  int k = 63 - __builtin_clzll(bytes - 1);             // 2^k < bytes <= 2^(k+1)  (bytes > 256)
  uint64_t base = 1ull << k, q = base >> 2;
  for (int s = 1; s <= 4; ++s)
    if (bytes <= base + q * s) return base + q * s;
  return base << 1;
}

// ------------------------------------------------------------------ backends
namespace {
struct DeviceBackend : PoolBackend {
  int dev;
  explicit DeviceBackend(int d) : dev(d) {}
  void* mem_alloc(size_t bytes) override {
    void* p = nullptr;
    cudaSetDevice(dev);
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
  }
  void mem_free(void* p) override { cudaSetDevice(dev); cudaFree(p); }
  void* event_create() override {
    cudaEvent_t e = nullptr;
    cudaSetDevice(dev);
    if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return e;
  }
  void event_destroy(void* e) override { cudaEventDestroy((cudaEvent_t)e); }
  bool event_record(void* e, void* s) override { return cudaEventRecord((cudaEvent_t)e, (cudaStream_t)s) == cudaSuccess; }
  bool event_done(void* e) override {
    cudaError_t r = cudaEventQuery((cudaEvent_t)e);
    if (r != cudaSuccess) { cudaGetLastError(); return false; }   // not ready — or an error: never hand out a block whose completion is unknown
    return true;
  }
};
struct PinnedBackend : DeviceBackend {
  explicit PinnedBackend(int d) : DeviceBackend(d) {}
  void* mem_alloc(size_t bytes) override {
    void* p = nullptr;
    cudaSetDevice(dev);
    if (cudaHostAlloc(&p, bytes, cudaHostAllocPortable | cudaHostAllocMapped) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
  }
  void mem_free(void* p) override { cudaFreeHost(p); }
};
// Fake: addresses are never dereferenced; an event is (stream, ticket); a stream's work is
// "complete" up to the ticket last declared by fake_complete().
struct FakeBackend : PoolBackend {
  struct Ev { void* stream; uint64_t ticket; };
  uint64_t next_addr = 0x10000000ull, budget = 1ull << 40, used = 0;
  std::map<void*, uint64_t> issued, completed;
  std::map<void*, uint64_t> sizes;
  void* mem_alloc(size_t bytes) override {
    if (used + bytes > budget) return nullptr;
    void* p = (void*)next_addr; next_addr += (bytes + 4095) & ~4095ull; used += bytes; sizes[p] = bytes;
    return p;
  }
  void mem_free(void* p) override { used -= sizes[p]; sizes.erase(p); }
  void* event_create() override { return new Ev{nullptr, 0}; }
  void event_destroy(void* e) override { delete (Ev*)e; }
  bool event_record(void* e, void* s) override { ((Ev*)e)->stream = s; ((Ev*)e)->ticket = ++issued[s]; return true; }
  bool event_done(void* e) override { Ev* ev = (Ev*)e; return completed[ev->stream] >= ev->ticket; }
  void fake_complete(void* s) override { completed[s] = issued[s]; }
};
}  // namespace

PoolBackend* make_device_backend(int device) { return new DeviceBackend(device); }
PoolBackend* make_pinned_backend(int device) { return new PinnedBackend(device); }
PoolBackend* make_fake_backend() { return new FakeBackend(); }

// ------------------------------------------------------------------ pool
CachingPool::CachingPool(PoolBackend* backend, uint64_t max_cached) : backend_(backend), max_cached_(max_cached) {}

CachingPool::~CachingPool() {
  {
    std::lock_guard<std::mutex> g(mu_);
    trim_locked(0);
    for (auto& kv : free_)                               // still pending (work queued behind them when they were freed):
      for (Block* b : kv.second) {                       // destroy is the end of the job, the owner has waited for its streams
        st_.bytes_cached -= b->bytes;
        release_block_locked(b);
      }
    free_.clear();
    for (auto& kv : live_) {                             // leaked by the user: give back anyway
      if (kv.second->event) backend_->event_destroy(kv.second->event);
      backend_->mem_free(kv.second->ptr);
      delete kv.second;
    }
    live_.clear();
  }
  delete backend_;
}

void* CachingPool::alloc(size_t bytes, void* stream) {
  uint64_t bin = bin_bytes_for(bytes ? bytes : 1);
  if (!bin) return nullptr;
  std::lock_guard<std::mutex> g(mu_);
  auto it = free_.find(bin);
  if (it != free_.end()) {
    auto& v = it->second;
    // 1st choice: a block last used on this same stream (stream order makes it safe at once) or
    // one already known complete; newest first.  2nd: a pending block whose event has completed.
    int pick = -1;
    for (int i = (int)v.size() - 1; i >= 0; --i)
      if (!v[i]->pending || v[i]->stream == stream) { pick = i; break; }
    if (pick < 0)
      for (int i = 0; i < (int)v.size(); ++i)
        if (backend_->event_done(v[i]->event)) { v[i]->pending = false; pick = i; break; }
    if (pick >= 0) {
      Block* b = v[pick];
      v.erase(v.begin() + pick);
      if (b->stream != stream) st_.cross_stream_reuses++;
      b->stream = stream; b->pending = false;
      live_[(uintptr_t)b->ptr] = b;
      st_.hits++; st_.bytes_cached -= b->bytes; st_.bytes_live += b->bytes;
      return b->ptr;
    }
  }
  void* p = backend_->mem_alloc(bin);
  if (!p) {                                              // out of memory: drop the cache and retry once
    trim_locked(0);
    p = backend_->mem_alloc(bin);
    if (!p) return nullptr;
  }
  Block* b = new Block();
  b->ptr = p; b->bytes = bin; b->stream = stream;
  live_[(uintptr_t)p] = b;
  st_.misses++; st_.backend_allocs++; st_.bytes_live += bin;
  st_.bytes_peak = std::max(st_.bytes_peak, st_.bytes_live + st_.bytes_cached);
  return p;
}

int CachingPool::free(void* ptr, void* stream, bool completed) {
  if (!ptr) return PR_OK;
  std::lock_guard<std::mutex> g(mu_);
  auto it = live_.find((uintptr_t)ptr);
  if (it == live_.end()) return PR_ERR_INVALID_ARG;
  Block* b = it->second;
  live_.erase(it);
  b->stream = stream;
  if (completed) {
    b->pending = false;
  } else {
    if (!b->event) b->event = backend_->event_create();
    if (!b->event || !backend_->event_record(b->event, stream)) {
      // cannot track completion: do not cache a block that may still be in use
      st_.bytes_live -= b->bytes;
      release_block_locked(b);
      return PR_ERR_CUDA;
    }
    b->pending = true;
  }
  b->freed_seq = ++seq_;
  st_.bytes_live -= b->bytes; st_.bytes_cached += b->bytes;
  free_[b->bytes].push_back(b);
  if (max_cached_ && st_.bytes_cached > max_cached_) trim_locked(max_cached_);
  return PR_OK;
}

void CachingPool::release_block_locked(Block* b) {
  if (b->event) backend_->event_destroy(b->event);
  backend_->mem_free(b->ptr);
  st_.backend_frees++;
  delete b;
}

// Oldest-first; only blocks that are not pending (or whose event has completed) are given back.
void CachingPool::trim_locked(uint64_t keep) {
  std::vector<std::pair<uint64_t, Block*>> all;
  for (auto& kv : free_)
    for (Block* b : kv.second) all.push_back({b->freed_seq, b});
  std::sort(all.begin(), all.end());
  for (auto& sb : all) {
    if (st_.bytes_cached <= keep) break;
    Block* b = sb.second;
    if (b->pending) {
      if (!backend_->event_done(b->event)) continue;
      b->pending = false;
    }
    auto& v = free_[b->bytes];
    v.erase(std::find(v.begin(), v.end(), b));
    st_.bytes_cached -= b->bytes;
    release_block_locked(b);
  }
}

bool CachingPool::find_live(const void* p, uintptr_t* base, size_t* bytes) {
  std::lock_guard<std::mutex> g(mu_);
  auto it = live_.upper_bound((uintptr_t)p);
  if (it == live_.begin()) return false;
  --it;
  if ((uintptr_t)p >= it->first + it->second->bytes) return false;
  *base = it->first; *bytes = (size_t)it->second->bytes;
  return true;
}

int CachingPool::trim(uint64_t keep) {
  std::lock_guard<std::mutex> g(mu_);
  trim_locked(keep);
  return PR_OK;
}

void CachingPool::stats(pr_pool_stats* out) {
  std::lock_guard<std::mutex> g(mu_);
  *out = st_;
}

}  // namespace pixreco

// ------------------------------------------------------------------ C ABI
extern "C" {

int pr_pool_create(int kind, int device, uint64_t max_cached_bytes, pr_pool** out) {
  if (!out) return PR_ERR_INVALID_ARG;
  *out = nullptr;
  pixreco::PoolBackend* be = nullptr;
  if (kind == PR_POOL_DEVICE) be = pixreco::make_device_backend(device);
  else if (kind == PR_POOL_PINNED) be = pixreco::make_pinned_backend(device);
  else if (kind == PR_POOL_FAKE) be = pixreco::make_fake_backend();
  else return PR_ERR_INVALID_ARG;
  pr_pool* p = new pr_pool{new pixreco::CachingPool(be, max_cached_bytes)};
  *out = p;
  return PR_OK;
}
void* pr_pool_alloc(pr_pool* p, size_t bytes, void* s) { return p ? p->impl->alloc(bytes, s) : nullptr; }
int pr_pool_free(pr_pool* p, void* ptr, void* s, int completed) { return p ? p->impl->free(ptr, s, completed != 0) : PR_ERR_INVALID_ARG; }
int pr_pool_trim(pr_pool* p, uint64_t keep) { return p ? p->impl->trim(keep) : PR_ERR_INVALID_ARG; }
int pr_pool_get_stats(pr_pool* p, pr_pool_stats* out) {
  if (!p || !out) return PR_ERR_INVALID_ARG;
  p->impl->stats(out);
  return PR_OK;
}
int pr_pool_destroy(pr_pool* p) {
  if (!p) return PR_ERR_INVALID_ARG;
  delete p->impl;
  delete p;
  return PR_OK;
}
int pr_pool_fake_complete(pr_pool* p, void* s) {
  if (!p) return PR_ERR_INVALID_ARG;
  p->impl->fake_complete(s);
  return PR_OK;
}
uint64_t pr_pool_bin_bytes(uint64_t bytes) { return pixreco::bin_bytes_for(bytes); }

}  // extern "C"
