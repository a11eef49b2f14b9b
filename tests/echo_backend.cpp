// TEST INFRASTRUCTURE, NOT PRODUCT CODE: a host-only back end for the multi-process front end (include/pp_ipc.h),
// so that the transport can be tested on a machine without a GPU.  Built into tests/libpp_echo.so by
// tests/conftest.py; libpp.so neither contains nor loads it.
//
// Every source yields, at the next flush, one hit {event_id, source_id, photon_idx = its photon count at 1e4
// photons/GeV, dom_id = 0, time_ns = t_ns + length, weight = energy}.  With echo_set_hits_per_source(k) it yields k
// copies (photon_idx + 0..k-1), to fill a client's hit ring quickly.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <atomic>
#include <chrono>
#include <mutex>
#include <thread>
#include <vector>

#include "../include/pp_ipc.h"

namespace {

struct Echo {
  std::mutex mu;
  std::vector<pp_hit> pending, ready;
  uint64_t flushed = 0;  // sources whose hits have been made available
  uint64_t pending_sources = 0;
  uint32_t hits_per_source = 1;
  uint64_t auto_id = 0;
  std::atomic<uint32_t> collect_delay_us{0};  // a collect that found nothing dawdles this long before it returns
};

int e_submit(void* ctx, const pp_source* s, const float* len, const uint32_t* ev, const uint32_t* sid, size_t n) {
  Echo* e = static_cast<Echo*>(ctx);
  std::lock_guard<std::mutex> g(e->mu);
  for (size_t i = 0; i < n; ++i) {
    pp_hit h{};
    const double cnt = std::floor((double)s[i].energy_GeV * 1.0e4 + 0.5);
    h.event_id = ev[i]; h.source_id = sid ? sid[i] : (uint32_t)(e->auto_id + i); h.dom_id = 0;
    h.time_ns = (double)s[i].t_ns + (len ? (double)len[i] : 0.0); h.weight = s[i].energy_GeV; h.n_scatter = 0;
    for (uint32_t k = 0; k < e->hits_per_source; ++k) {
      h.photon_idx = (uint32_t)cnt + k;
      e->pending.push_back(h);
    }
  }
  e->auto_id += n;
  e->pending_sources += n;
  return PP_OK;
}
int e_flush(void* ctx) {
  Echo* e = static_cast<Echo*>(ctx);
  std::lock_guard<std::mutex> g(e->mu);
  e->ready.insert(e->ready.end(), e->pending.begin(), e->pending.end());
  e->flushed += e->pending_sources;
  e->pending_sources = 0;
  e->pending.clear();
  return PP_OK;
}
int e_completed(void* ctx, uint64_t* n_sources) {
  Echo* e = static_cast<Echo*>(ctx);
  std::lock_guard<std::mutex> g(e->mu);
  *n_sources = e->flushed;
  return PP_OK;
}
int e_collect(void* ctx, pp_hit* out, size_t cap, size_t* n_out, int* drained) {
  Echo* e = static_cast<Echo*>(ctx);
  std::lock_guard<std::mutex> g(e->mu);
  const size_t n = std::min(cap, e->ready.size());
  std::memcpy(out, e->ready.data(), n * sizeof(pp_hit));
  e->ready.erase(e->ready.begin(), e->ready.begin() + (long)n);
  *n_out = n;
  *drained = (n == 0 && e->pending.empty() && e->ready.empty()) ? 1 : 0;
  const uint32_t delay = e->collect_delay_us.load();
  if (n == 0 && delay) {
    // the answer above is now stale by `delay`: blocks handed over meanwhile are NOT covered by `drained`
    e->mu.unlock();
    std::this_thread::sleep_for(std::chrono::microseconds(delay));
    e->mu.lock();
  }
  return PP_OK;
}

}  // namespace

extern "C" {

// A fresh, independent instance; lives as long as the process.
const pp_ipc_backend* echo_backend_new(void) {
  return new pp_ipc_backend{new Echo(), e_submit, e_flush, e_collect, e_completed};
}

void echo_set_hits_per_source(const pp_ipc_backend* be, uint32_t k) {
  Echo* e = static_cast<Echo*>(be->ctx);
  std::lock_guard<std::mutex> g(e->mu);
  e->hits_per_source = k ? k : 1;
}

// Makes every empty-handed collect return late: widens the window between "the back end looked" and "the server acts on
// it" that a preempted dispatch thread opens in production.
void echo_set_collect_delay_us(const pp_ipc_backend* be, uint32_t us) {
  static_cast<Echo*>(be->ctx)->collect_delay_us.store(us);
}

}  // extern "C"
