// stream_driver.cpp — see include/pixreco_driver.h.  Host-only C++17; calls the C ABI of libpixreco.so only.
#include <algorithm>
#include <atomic>
#include <chrono>
#include <thread>
#include <vector>

#include "../../include/pixreco_driver.h"

namespace {
using clk = std::chrono::steady_clock;
inline double us_since(clk::time_point t0) { return std::chrono::duration<double, std::micro>(clk::now() - t0).count(); }

// FNV-1a over 32-bit words: the per-event fingerprint a caller compares with its own hash of the expected array
inline uint64_t fnv1a32(const uint32_t* p, size_t n) {
  uint64_t h = 1469598103934665603ull;
  for (size_t i = 0; i < n; ++i) { h ^= p[i]; h *= 1099511628211ull; }
  return h;
}
}  // namespace

extern "C" int prd_run_streams_rec(pr_event* const* slots, void* const* streams, uint32_t n_slots,
                                   const pr_input* pool, uint32_t n_pool, uint32_t first, uint32_t n_events, uint32_t n_threads,
                                   uint64_t* t_start_ns, uint64_t* t_end_ns, prd_event_record* rec, prd_result* res) {
  if (!slots || !streams || !pool || !res || !n_slots || !n_pool || !n_threads) return PR_ERR_INVALID_ARG;
  if (n_threads > n_slots) n_threads = n_slots;
  std::atomic<int> status{PR_OK};
  std::atomic<uint32_t> ready{0};
  std::atomic<bool> go{false};
  std::vector<std::vector<float>> acqUs(n_threads);
  std::vector<uint64_t> digis(n_threads, 0), clusters(n_threads, 0), polls(n_threads, 0), done(n_threads, 0);
  std::vector<clk::time_point> tBegin(n_threads), tEnd(n_threads);

  auto worker = [&](uint32_t t) {
    // Every slot runs its own sequence of events (s, s + n_slots, s + 2 n_slots, ...: A25) and is served as soon as it
    // is ready: the thread goes round its slots, takes the product of a slot whose event has completed (pr_produce
    // answers PR_NOT_READY otherwise: a poll, never a wait), releases it and issues the slot's next event.  No slot
    // waits for another slot's event.
    std::vector<int64_t> inFlight(n_slots, -1), next(n_slots, -1);
    uint32_t mine = 0, open = 0;
    for (uint32_t s = t; s < n_slots; s += n_threads) { next[s] = s < n_events ? (int64_t)s : -1; ++mine; if (next[s] >= 0) ++open; }
    acqUs[t].reserve(n_events / n_threads + 8);
    pr_output out;
    bool failed = false;
    auto fail = [&](int r) { int ok = PR_OK; status.compare_exchange_strong(ok, r); failed = true; };
    ready.fetch_add(1);
    while (!go.load(std::memory_order_acquire)) {}
    tBegin[t] = clk::now();
    while (open && !failed && status.load(std::memory_order_relaxed) == PR_OK) {
      for (uint32_t s = t; s < n_slots && !failed; s += n_threads) {
        if (inFlight[s] >= 0) {
          const int r = pr_produce(slots[s], &out);
          if (r == PR_NOT_READY) { ++polls[t]; continue; }
          if (r != PR_OK) { fail(r); break; }
          const int64_t e = inFlight[s];
          digis[t] += out.n_digis; clusters[t] += out.n_clusters; ++done[t];
          if (t_start_ns) t_start_ns[e] = out.t_start_ns;
          if (t_end_ns) t_end_ns[e] = out.t_end_ns;
          if (rec) {
            prd_event_record& q = rec[e];
            q.event_id = out.event_id; q.n_digis = out.n_digis; q.n_errors = out.n_errors; q.n_kept_digis = out.n_kept_digis;
            q.n_clusters_all = out.n_clusters_all; q.n_clusters = out.n_clusters; q.status_bits = out.status_bits;
            q.thread = t;
            q.hash_label = out.h_label ? fnv1a32(out.h_label, out.n_digis) : 0;
            q.hash_cl_label = out.h_cl_label ? fnv1a32(out.h_cl_label, out.n_clusters) : 0;
          }
          int rr;
          while ((rr = pr_release(slots[s])) == PR_NOT_READY) {}
          if (rr != PR_OK) { fail(rr); break; }
          inFlight[s] = -1;
          if (next[s] < 0) --open;
        }
        if (inFlight[s] < 0 && next[s] >= 0) {
          const int64_t e = next[s];
          const auto a0 = clk::now();
          const int r = pr_acquire(slots[s], pool + (first + e) % n_pool, streams[s]);
          acqUs[t].push_back((float)us_since(a0));
          if (r != PR_OK) { fail(r); break; }
          inFlight[s] = e;
          next[s] = e + n_slots < n_events ? e + n_slots : -1;
        }
      }
    }
    (void)mine;
    tEnd[t] = clk::now();
  };

  std::vector<std::thread> th;
  for (uint32_t t = 0; t < n_threads; ++t) th.emplace_back(worker, t);
  while (ready.load() < n_threads) {}
  go.store(true, std::memory_order_release);
  for (auto& x : th) x.join();

  clk::time_point b = tBegin[0], e = tEnd[0];
  std::vector<float> all;
  *res = prd_result{};
  for (uint32_t t = 0; t < n_threads; ++t) {
    b = std::min(b, tBegin[t]); e = std::max(e, tEnd[t]);
    all.insert(all.end(), acqUs[t].begin(), acqUs[t].end());
    res->digis += digis[t]; res->clusters += clusters[t]; res->produce_polls += polls[t]; res->events += done[t];
  }
  res->wall_s = std::chrono::duration<double>(e - b).count();
  if (!all.empty()) {
    std::sort(all.begin(), all.end());
    double sum = 0;
    for (float v : all) sum += v;
    res->acquire_us_median = all[all.size() / 2];
    res->acquire_us_mean = sum / all.size();
    res->acquire_us_p99 = all[std::min(all.size() - 1, (size_t)(all.size() * 0.99))];
  }
  res->status = status.load();
  res->threads = n_threads;
  return res->status;
}

extern "C" int prd_run_streams(pr_event* const* slots, void* const* streams, uint32_t n_slots,
                               const pr_input* pool, uint32_t n_pool, uint32_t first, uint32_t n_events, uint32_t n_threads,
                               uint64_t* t_start_ns, uint64_t* t_end_ns, prd_result* res) {
  return prd_run_streams_rec(slots, streams, n_slots, pool, n_pool, first, n_events, n_threads, t_start_ns, t_end_ns, nullptr, res);
}

extern "C" int prd_clusters_to_aos(const pr_output* out, prd_cluster_aos* dst, uint32_t cap) {
  if (!out || (!dst && cap)) return PR_ERR_INVALID_ARG;
  const uint32_t n = out->n_clusters < cap ? out->n_clusters : cap;
  if (n && !(out->h_cl_label && out->h_cl_size && out->h_cl_module && out->h_cl_charge && out->h_cl_row && out->h_cl_col))
    return PR_ERR_BAD_STATE;
  const bool hits = out->h_ht_x && out->h_ht_y && out->h_ht_xerr && out->h_ht_yerr && out->h_ht_rows && out->h_ht_cols && out->h_ht_flags;
  for (uint32_t k = 0; k < n; ++k) {
    prd_cluster_aos r{};
    r.label = out->h_cl_label[k]; r.size = out->h_cl_size[k]; r.module = out->h_cl_module[k];
    r.charge = out->h_cl_charge[k]; r.row = out->h_cl_row[k]; r.col = out->h_cl_col[k];
    if (hits) {
      r.flags = out->h_ht_flags[k];
      r.x_um = out->h_ht_x[k]; r.y_um = out->h_ht_y[k]; r.xerr_um = out->h_ht_xerr[k]; r.yerr_um = out->h_ht_yerr[k];
      r.row_min = (uint16_t)(out->h_ht_rows[k] & 0xFFFFu); r.row_max = (uint16_t)(out->h_ht_rows[k] >> 16);
      r.col_min = (uint16_t)(out->h_ht_cols[k] & 0xFFFFu); r.col_max = (uint16_t)(out->h_ht_cols[k] >> 16);
    }
    dst[k] = r;
  }
  return (int)n;
}
