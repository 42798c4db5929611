// Host-only harness for tests/test_sanitizers.py: the oracle, the workload generator and the caching pool on its fake
// backend, built with -fsanitize=address,undefined (compute-sanitizer is not available on this pool; the device code
// is covered by the parity tests).  Exit code 0 = nothing reported.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../include/pixreco.h"

extern "C" {
// paper_2004_04334_b200/workloads/pixgen.c
struct pixgen_params {
  uint32_t n_modules, n_rows, n_cols; double lambda; uint32_t hot_modules; double hot_factor, compact_mean, frac_elongated,
      elongated_mean, frac_strip; uint32_t strip_min, strip_max; double p_touch; uint32_t fill_pixels; double err_frac; uint32_t adc_law;
};
struct pixgen_stats { uint64_t n_words, n_digis, n_errors, n_seeded_clusters, max_digis_per_module; };
int pixgen_default_params(uint32_t config, pixgen_params* p);
int pixgen_calib(uint64_t seed, uint32_t config, uint32_t n_modules, float* gain, float* ped);
int pixgen_event(uint64_t seed, uint32_t config, uint32_t event, const pixgen_params* p, uint32_t** words, uint16_t** adc, pixgen_stats* st);
void pixgen_free(void* p);
// oracle/pixreco_oracle.c
int po_run(const uint32_t* words, const uint16_t* adc, uint32_t W, uint32_t M, uint32_t R, uint32_t C,
           const float* gain, const float* ped, float pix_thr, float clus_thr,
           uint16_t* d_module, uint16_t* d_row, uint16_t* d_col, uint16_t* d_adc, uint32_t* d_word_idx,
           uint32_t* e_word, uint32_t* e_idx, uint32_t* mod_digi_start, float* charge, uint8_t* kept, uint32_t* label,
           uint32_t* cl_label, uint16_t* cl_module, uint32_t* cl_size, float* cl_charge, float* cl_row, float* cl_col,
           int32_t* clus, uint32_t* mod_clus_start, double pitch_row_um, double pitch_col_um,
           float* ht_x, float* ht_y, float* ht_xerr, float* ht_yerr, uint32_t* ht_rows, uint32_t* ht_cols, uint16_t* ht_flags,
           uint32_t* counters);
int po_check_exact_sums(uint32_t D, const uint32_t* label, const float* charge, const uint16_t* d_col);
}

static int run_oracle(uint32_t config, uint32_t event, uint32_t n_modules_override, uint32_t fill_override) {
  pixgen_params p;
  pixgen_default_params(config, &p);
  if (n_modules_override) p.n_modules = n_modules_override;
  if (fill_override) p.fill_pixels = fill_override;
  const uint32_t M = p.n_modules;
  std::vector<float> gain(M), ped(M);
  if (pixgen_calib(20200404ull, config, M, gain.data(), ped.data())) return 2;
  uint32_t* words = nullptr; uint16_t* adc = nullptr; pixgen_stats st;
  if (pixgen_event(20200404ull, config, event, &p, &words, &adc, &st)) return 3;
  const uint32_t W = (uint32_t)st.n_words;                    // every output array has exactly the documented capacity
  std::vector<uint16_t> dm(W), dr(W), dc(W), da(W), clm(W), hf(W);
  std::vector<uint32_t> dw(W), ew(W), ei(W), mds(M + 1), lab(W), cll(W), cls(W), mcs(M + 1), hr(W), hc(W), cnt(7);
  std::vector<float> q(W), clq(W), clr(W), clc(W), hx(W), hy(W), hxe(W), hye(W);
  std::vector<uint8_t> kept(W);
  std::vector<int32_t> clus(W);
  int rc = po_run(words, adc, W, M, p.n_rows, p.n_cols, gain.data(), ped.data(), 1000.f, 4000.f, dm.data(), dr.data(), dc.data(),
                  da.data(), dw.data(), ew.data(), ei.data(), mds.data(), q.data(), kept.data(), lab.data(), cll.data(), clm.data(),
                  cls.data(), clq.data(), clr.data(), clc.data(), clus.data(), mcs.data(), 100.0, 150.0, hx.data(), hy.data(),
                  hxe.data(), hye.data(), hr.data(), hc.data(), hf.data(), cnt.data());
  if (!rc && W < 60000) rc = po_check_exact_sums(cnt[0], lab.data(), q.data(), dc.data());
  std::printf("config %u event %u: %u words, %u digis, %u clusters, rc %d\n", config, event, W, cnt[0], cnt[4], rc);
  pixgen_free(words); pixgen_free(adc);
  return rc ? 4 : 0;
}

static int run_pool() {
  pr_pool* pool = nullptr;
  if (pr_pool_create(PR_POOL_FAKE, 0, 64ull << 20, &pool) != PR_OK) return 10;
  uint64_t x = 88172645463325252ull;
  auto rnd = [&]() { x ^= x << 13; x ^= x >> 7; x ^= x << 17; return x; };
  std::vector<std::pair<void*, uintptr_t>> live;
  for (int it = 0; it < 20000; ++it) {
    const uint64_t r = rnd();
    const uintptr_t stream = 0x100 * (1 + (r >> 8) % 8);
    if (live.size() < 64 && (r & 3) != 0) {
      const size_t bytes = 1 + (size_t)((r >> 16) % (8u << 20));
      void* ptr = pr_pool_alloc(pool, bytes, (void*)stream);
      if (!ptr) return 11;
      live.push_back({ptr, stream});
    } else if (!live.empty()) {
      const size_t k = (size_t)((r >> 40) % live.size());
      if (pr_pool_free(pool, live[k].first, (void*)live[k].second, (int)((r >> 4) & 1)) != PR_OK) return 12;
      live[k] = live.back(); live.pop_back();
    }
    if ((r & 0xFF) == 0) pr_pool_fake_complete(pool, (void*)stream);
    if ((r & 0xFFF) == 1) pr_pool_trim(pool, 1 << 20);
  }
  if (pr_pool_free(pool, (void*)0xDEAD0000, (void*)0x100, 0) != PR_ERR_INVALID_ARG) return 13;
  for (auto& b : live) pr_pool_free(pool, b.first, (void*)b.second, 1);
  pr_pool_stats st;
  if (pr_pool_get_stats(pool, &st) != PR_OK || st.bytes_live != 0) return 14;
  return pr_pool_destroy(pool) == PR_OK ? 0 : 15;
}

int main() {
  int rc = run_oracle(0, 0, 0, 0);
  if (!rc) rc = run_oracle(1, 3, 0, 0);
  if (!rc) rc = run_oracle(4, 1, 6, 1900);
  if (!rc) rc = run_pool();
  std::printf("sanitize_main: %d\n", rc);
  return rc;
}
