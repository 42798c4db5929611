// pool.hpp — stream-aware caching allocator for device and pinned-host memory.
//
// Paper: "we decided to use a memory pool for both the device and the pinned host memory ...
// the cost of the API calls gets amortized".  The paper's pool was derived from
// a library allocator; this one is written from the behavioural description in DESIGN.md (A23):
// binned sizes, per-bin free lists, a freed block remembers its last stream and an event recorded
// at free, immediate reuse on the same stream, reuse on another stream only once the event has
// completed (query, never wait), nothing returned to the backend outside trim/destroy/OOM.
#pragma once
#include <cstddef>
#include <cstdint>
#include <map>
#include <mutex>
#include <unordered_map>
#include <vector>

#include "../../include/pixreco.h"

namespace pixreco {

// Backend = where memory and completion events come from.  Three exist: CUDA device, CUDA pinned
// host, and a fake used by CPU-only tests of the host logic.
struct PoolBackend {
  virtual ~PoolBackend() {}
  virtual void* mem_alloc(size_t bytes) = 0;            // nullptr on out-of-memory
  virtual void  mem_free(void* p) = 0;
  virtual void* event_create() = 0;
  virtual void  event_destroy(void* ev) = 0;
  virtual bool  event_record(void* ev, void* stream) = 0;
  virtual bool  event_done(void* ev) = 0;               // non-blocking query
  virtual void  fake_complete(void* /*stream*/) {}
};

PoolBackend* make_device_backend(int device);
PoolBackend* make_pinned_backend(int device);
PoolBackend* make_fake_backend();

constexpr int kMinBinLog2 = 8;      // 256 B
constexpr int kMaxBinLog2 = 36;     // 64 GiB
uint64_t bin_bytes_for(uint64_t bytes);   // 0 if too large

class CachingPool {
 public:
  CachingPool(PoolBackend* backend, uint64_t max_cached_bytes);
  ~CachingPool();
  void* alloc(size_t bytes, void* stream);
  int   free(void* ptr, void* stream, bool completed);
  int   trim(uint64_t keep_cached_bytes);
  void  stats(pr_pool_stats* out);
  void  fake_complete(void* stream) { backend_->fake_complete(stream); }
  // The live (handed out) block that contains p: its start and size.  False if p is not inside one.
  bool  find_live(const void* p, uintptr_t* base, size_t* bytes);

 private:
  struct Block {
    void*    ptr = nullptr;
    uint64_t bytes = 0;
    void*    stream = nullptr;   // stream of the last use
    void*    event = nullptr;    // lazily created; recorded at free when not known complete
    bool     pending = false;    // event recorded and not yet seen complete
    uint64_t freed_seq = 0;      // for oldest-first trimming
  };
  void release_block_locked(Block* b);
  void trim_locked(uint64_t keep);

  PoolBackend* backend_;
  uint64_t max_cached_;
  std::mutex mu_;
  std::unordered_map<uint64_t, std::vector<Block*>> free_;   // bin bytes -> idle blocks
  std::map<uintptr_t, Block*> live_;                         // by start address (find_live looks up a containing block)
  pr_pool_stats st_{};
  uint64_t seq_ = 0;
};

}  // namespace pixreco

struct pr_pool {
  pixreco::CachingPool* impl;
};
