// Several devices behind one photon server (include/pp_multi.h): a queue that cuts
// launch-sized batches of whole sources and deals each to the back end with the fewest photons outstanding.
// Host-only code: no CUDA call in this file.  Product code: shares nothing with oracle/.
#include "../../include/pp_multi.h"

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <condition_variable>
#include <deque>
#include <mutex>
#include <thread>
#include <vector>

namespace {

constexpr uint32_t kMaxDevices = 64;

// ---- back end bound to a pp_handle (the same binding the multi-process server uses) ----
int h_submit(void* ctx, const pp_source* s, const float* len, const uint32_t* ev, const uint32_t* sid, size_t n) {
  return pp_submit_segments(static_cast<pp_handle*>(ctx), s, len, ev, sid, n);
}
int h_flush(void* ctx) { return pp_flush(static_cast<pp_handle*>(ctx)); }
int h_collect(void* ctx, pp_hit* out, size_t cap, size_t* n_out, int* drained) {
  pp_handle* h = static_cast<pp_handle*>(ctx);
  int rc = pp_collect(h, out, cap, n_out, 0);
  *drained = 0;
  if (rc != PP_OK || *n_out != 0) return rc;
  pp_stats_t st;
  rc = pp_stats(h, &st);
  if (rc == PP_OK && st.photons_done == st.photons_submitted && st.hits_collected == st.photons_hit) *drained = 1;
  return rc;
}
int h_completed(void* ctx, uint64_t* n_sources) {
  pp_stats_t st;
  const int rc = pp_stats(static_cast<pp_handle*>(ctx), &st);
  *n_sources = rc == PP_OK ? st.sources_completed : 0;
  return rc;
}

struct Staged {
  pp_source s;
  float length;
  uint32_t event_id, source_id;
  uint64_t photons;
};

struct Batch {          // a dealt batch, in deal order
  uint32_t dev;
  uint64_t n_sources, photons;
  uint64_t dev_end;     // sources dealt to `dev` up to and including this batch
  bool complete;
};

struct Device {
  pp_ipc_backend be{};
  uint64_t base_completed = 0;   // the back end's completed count when the front was created
  uint64_t dealt_sources = 0, dealt_photons = 0, batches = 0;
  uint64_t outstanding = 0;      // photons dealt and not yet complete
  std::deque<size_t> open;       // indices into pp_multi::batches of this device's incomplete batches, in order
  bool dealing = false;          // a batch is being handed to this device right now, outside pp_multi::mu
};

}  // namespace

struct pp_multi {
  std::vector<Device> dev;
  uint64_t deal_photons = 100000000ull;
  float yield = 0.0f;
  std::mutex mu;                 // staging, dealing, bookkeeping
  std::condition_variable cv_dealt;  // a device has finished taking a batch (Device::dealing went false)
  std::deque<Staged> staged;
  uint64_t staged_photons = 0;
  uint64_t n_submitted = 0, ph_submitted = 0;
  uint64_t n_deals = 0;          // batches cut off the staging queue so far
  uint64_t rejected_sources = 0; // sources of batches a back end refused (dropped, counted as complete)
  std::deque<Batch> batches;     // incomplete prefix trimmed as batches complete in order
  size_t batches_base = 0;       // global index of batches.front()
  uint64_t completed_prefix = 0; // sources in the complete prefix of the deal order
  std::mutex collect_mu;
  uint32_t next_dev = 0;         // round-robin start of the next collect
};

namespace {

// Refresh the per-device outstanding counts and the global completed prefix.  Caller holds m->mu.
int refresh(pp_multi* m) {
  for (uint32_t d = 0; d < m->dev.size(); ++d) {
    Device& D = m->dev[d];
    if (D.open.empty() || !D.be.completed) continue;
    uint64_t v = 0;
    const int rc = D.be.completed(D.be.ctx, &v);
    if (rc != PP_OK) return rc;
    const uint64_t done = v > D.base_completed ? v - D.base_completed : 0;
    while (!D.open.empty()) {
      Batch& b = m->batches[D.open.front() - m->batches_base];
      if (b.dev_end > done) break;
      b.complete = true;
      D.outstanding -= b.photons;
      D.open.pop_front();
    }
  }
  while (!m->batches.empty() && m->batches.front().complete) {
    m->completed_prefix += m->batches.front().n_sources;
    m->batches.pop_front();
    m->batches_base++;
  }
  return PP_OK;
}

// Cut a batch of whole sources holding at least `want` photons (or everything, if less is staged) off the staging
// queue and hand it to the device with the fewest photons outstanding.  Caller holds m->mu through `lk`; the lock is
// RELEASED while the device takes the batch: its submit blocks while the device's source ring is full, and the
// completed count, the drained test of collect, the statistics and every other submitter need m->mu meanwhile (behind
// the multi-process server a dispatch thread that cannot ask for the completed count stops collecting, and with it
// the only thing that would ever free the ring).  The batch leaves the staging queue and enters the books before the
// lock is released; `dealing` keeps a second dealer off the same device until the hand-over is finished, so each
// device sees its batches in the order of the books.
int deal_one(pp_multi* m, uint64_t want, std::unique_lock<std::mutex>& lk) {
  uint32_t best = 0;
  for (;;) {
    if (m->staged.empty()) return PP_OK;
    const int rc0 = refresh(m);
    if (rc0 != PP_OK) return rc0;
    bool found = false;
    for (uint32_t d = 0; d < m->dev.size(); ++d)
      if (!m->dev[d].dealing && (!found || m->dev[d].outstanding < m->dev[best].outstanding)) { best = d; found = true; }
    if (found) break;
    m->cv_dealt.wait(lk);  // every device is taking a batch right now
  }
  size_t n = 0;
  uint64_t ph = 0;
  while (n < m->staged.size() && (ph < want || n == 0)) ph += m->staged[n++].photons;
  std::vector<pp_source> src(n);
  std::vector<float> len(n);
  std::vector<uint32_t> ev(n), sid(n);
  bool any_len = false;
  for (size_t i = 0; i < n; ++i) {
    const Staged& r = m->staged[i];
    src[i] = r.s; len[i] = r.length; ev[i] = r.event_id; sid[i] = r.source_id;
    any_len |= r.length != 0.0f;
  }
  Device& D = m->dev[best];
  m->staged.erase(m->staged.begin(), m->staged.begin() + (long)n);
  m->staged_photons -= ph;
  D.dealt_sources += n; D.dealt_photons += ph; D.batches++; D.outstanding += ph;
  m->batches.push_back(Batch{best, n, ph, D.dealt_sources, false});
  const size_t idx = m->batches_base + m->batches.size() - 1;
  D.open.push_back(idx);
  D.dealing = true;
  m->n_deals++;
  lk.unlock();
  int rc = D.be.submit(D.be.ctx, src.data(), any_len ? len.data() : nullptr, ev.data(), sid.data(), n);
  if (rc == PP_OK) rc = D.be.flush(D.be.ctx);  // a dealt batch is a whole launch: do not wait for more
  lk.lock();
  D.dealing = false;
  m->cv_dealt.notify_all();
  if (rc == PP_E_INVAL || rc == PP_E_OVERFLOW) {
    // the device refused the batch as a whole (pp.h: none of its sources is propagated); pp_multi_submit makes the
    // handle's own checks, so this means a back end with other rules or another light yield.  The batch is gone from
    // the staging queue already (left there, every later deal would meet it again); it is taken out of the device's
    // books and counted as complete without hits, so that whoever waits on the completed count is not stuck behind it,
    // and the caller of this deal gets the code.  (It is the device's newest batch: nobody else dealt to it meanwhile;
    // and it cannot have been found complete, since the device never got its sources.)
    D.dealt_sources -= n; D.dealt_photons -= ph; D.batches--; D.outstanding -= ph;
    D.open.pop_back();
    Batch& b = m->batches[idx - m->batches_base];
    b.photons = 0; b.dev_end = D.dealt_sources; b.complete = true;
    m->rejected_sources += n;
  }
  return rc;
}

// the front as a pp_ipc_backend
int m_submit(void* ctx, const pp_source* s, const float* len, const uint32_t* ev, const uint32_t* sid, size_t n) {
  return pp_multi_submit(static_cast<pp_multi*>(ctx), s, len, ev, sid, n);
}
int m_flush(void* ctx) { return pp_multi_flush(static_cast<pp_multi*>(ctx)); }
int m_completed(void* ctx, uint64_t* n_sources) {
  pp_multi* m = static_cast<pp_multi*>(ctx);
  std::lock_guard<std::mutex> g(m->mu);
  const int rc = refresh(m);
  *n_sources = m->completed_prefix;
  return rc;
}
int collect_once(pp_multi* m, pp_hit* out, size_t cap, size_t* n_out, int* drained) {
  *n_out = 0;
  *drained = 0;
  std::lock_guard<std::mutex> g(m->collect_mu);
  const uint32_t nd = (uint32_t)m->dev.size();
  // "drained" = every device is, and no source was on its way to one while they were asked: nothing staged, no batch
  // being handed over, and no batch dealt between the look before and the look after
  auto quiet = [&]() {
    bool q = m->staged.empty();
    for (const Device& D : m->dev) q = q && !D.dealing;
    return q;
  };
  uint64_t deals_before = 0;
  bool all_drained = true;
  {
    std::lock_guard<std::mutex> g2(m->mu);
    deals_before = m->n_deals;
    all_drained = quiet();
  }
  for (uint32_t k = 0; k < nd; ++k) {
    Device& D = m->dev[(m->next_dev + k) % nd];
    size_t got = 0;
    int dr = 0;
    const int rc = D.be.collect(D.be.ctx, out, cap, &got, &dr);
    if (rc != PP_OK) return rc;
    if (got > 0) {
      *n_out = got;
      m->next_dev = (m->next_dev + k + 1) % nd;  // the next call starts with the next device
      return PP_OK;
    }
    all_drained = all_drained && dr != 0;
  }
  if (all_drained) {
    std::lock_guard<std::mutex> g2(m->mu);
    *drained = (quiet() && m->n_deals == deals_before) ? 1 : 0;
  }
  return PP_OK;
}
int m_collect(void* ctx, pp_hit* out, size_t cap, size_t* n_out, int* drained) {
  return collect_once(static_cast<pp_multi*>(ctx), out, cap, n_out, drained);
}

}  // namespace

extern "C" {

int pp_multi_create_backends(const pp_ipc_backend* backends, uint32_t n, const pp_multi_config* cfg, pp_multi** out) {
  if (!backends || n == 0 || n > kMaxDevices || !cfg || !out) return PP_E_INVAL;
  *out = nullptr;
  if (!(cfg->photons_per_GeV > 0.0f) || !std::isfinite(cfg->photons_per_GeV)) return PP_E_INVAL;
  for (uint32_t d = 0; d < n; ++d)
    if (!backends[d].submit || !backends[d].flush || !backends[d].collect) return PP_E_INVAL;
  auto* m = new pp_multi();
  m->dev.resize(n);
  for (uint32_t d = 0; d < n; ++d) {
    m->dev[d].be = backends[d];
    if (backends[d].completed) backends[d].completed(backends[d].ctx, &m->dev[d].base_completed);
  }
  if (cfg->deal_photons) m->deal_photons = cfg->deal_photons;
  m->yield = cfg->photons_per_GeV;
  *out = m;
  return PP_OK;
}

int pp_multi_create(pp_handle* const* handles, uint32_t n, const pp_multi_config* cfg, pp_multi** out) {
  if (!handles || n == 0 || n > kMaxDevices) return PP_E_INVAL;
  std::vector<pp_ipc_backend> be(n);
  for (uint32_t d = 0; d < n; ++d) {
    if (!handles[d]) return PP_E_INVAL;
    be[d] = pp_ipc_backend{handles[d], h_submit, h_flush, h_collect, h_completed};
  }
  return pp_multi_create_backends(be.data(), n, cfg, out);
}

void pp_multi_destroy(pp_multi* m) { delete m; }

int pp_multi_submit(pp_multi* m, const pp_source* sources, const float* lengths_m, const uint32_t* event_ids,
                    const uint32_t* source_ids, size_t n) {
  if (!m) return PP_E_INVAL;
  if (n == 0) return PP_OK;
  if (!sources || !event_ids) return PP_E_INVAL;
  // the checks a handle makes on a source (pp.h, pp_submit) and the photon counts, before anything is staged: a bad
  // call fails as a whole, here and now, in the caller that made it -- not later in some other caller's deal
  std::vector<uint64_t> cnt(n);
  for (size_t i = 0; i < n; ++i) {
    const pp_source& a = sources[i];
    const float f8[8] = {a.x, a.y, a.z, a.dx, a.dy, a.dz, a.t_ns, a.energy_GeV};
    for (float f : f8)
      if (!std::isfinite(f)) return PP_E_INVAL;
    const double n2 = (double)a.dx * a.dx + (double)a.dy * a.dy + (double)a.dz * a.dz;
    if (std::fabs(n2 - 1.0) > 1e-4 || a.energy_GeV < 0.0f) return PP_E_INVAL;
    if (lengths_m && !(std::isfinite(lengths_m[i]) && lengths_m[i] >= 0.0f)) return PP_E_INVAL;
    const int rc = pp_photon_count(a.energy_GeV, m->yield, &cnt[i]);
    if (rc != PP_OK) return rc;
  }
  std::unique_lock<std::mutex> g(m->mu);
  for (size_t i = 0; i < n; ++i) {
    Staged r;
    r.s = sources[i]; r.length = lengths_m ? lengths_m[i] : 0.0f; r.event_id = event_ids[i];
    r.source_id = source_ids ? source_ids[i] : (uint32_t)(m->n_submitted + i);  // the FRONT's running record number
    r.photons = cnt[i];
    m->staged.push_back(r);
    m->staged_photons += cnt[i];
  }
  m->n_submitted += n;
  for (size_t i = 0; i < n; ++i) m->ph_submitted += cnt[i];
  while (m->staged_photons >= m->deal_photons) {
    const int rc = deal_one(m, m->deal_photons, g);
    if (rc != PP_OK) return rc;
  }
  return PP_OK;
}

int pp_multi_flush(pp_multi* m) {
  if (!m) return PP_E_INVAL;
  std::unique_lock<std::mutex> g(m->mu);
  while (!m->staged.empty()) {
    const int rc = deal_one(m, m->deal_photons, g);
    if (rc != PP_OK) return rc;
  }
  // (a batch another thread is still handing over is flushed by that thread)
  for (auto& D : m->dev) {
    const int rc = D.be.flush(D.be.ctx);
    if (rc != PP_OK) return rc;
  }
  return PP_OK;
}

int pp_multi_collect(pp_multi* m, pp_hit* out, size_t cap, size_t* n_out, int block) {
  if (!m || !n_out || (!out && cap)) return PP_E_INVAL;
  *n_out = 0;
  for (;;) {
    int drained = 0;
    const int rc = collect_once(m, out, cap, n_out, &drained);
    if (rc != PP_OK || *n_out > 0 || drained || !block || cap == 0) return rc;
    std::this_thread::sleep_for(std::chrono::microseconds(100));
  }
}

int pp_multi_get_stats(pp_multi* m, pp_multi_stats* out) {
  if (!m || !out) return PP_E_INVAL;
  std::lock_guard<std::mutex> g(m->mu);
  const int rc = refresh(m);
  *out = pp_multi_stats{};
  out->n_devices = (uint32_t)m->dev.size();
  out->sources_submitted = m->n_submitted; out->photons_submitted = m->ph_submitted;
  out->sources_staged = m->staged.size();
  out->sources_completed = m->completed_prefix;
  for (size_t d = 0; d < m->dev.size(); ++d) {
    out->batches[d] = m->dev[d].batches; out->photons[d] = m->dev[d].dealt_photons;
    out->photons_outstanding[d] = m->dev[d].outstanding;
  }
  return rc;
}

int pp_multi_backend(pp_multi* m, pp_ipc_backend* out) {
  if (!m || !out) return PP_E_INVAL;
  *out = pp_ipc_backend{m, m_submit, m_flush, m_collect, m_completed, nullptr};
  return PP_OK;
}

}  // extern "C"
