// TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Host stand-ins for the launch wrappers of pp_kernels.cu (pp_internal.h), used
// only by the ThreadSanitizer build of the host side (tests/tsan/).  No physics: the fake propagation "finishes" every
// photon of the launch at once, makes one hit for every kHitStride-th photon of the batch, and honours the bounded hit
// ring with the same stop / resume-list protocol the real kernel uses (so relaunches are exercised too).
#include <algorithm>
#include <atomic>
#include <cstring>

#include "../../paper_2405_05700_b200/csrc/pp_internal.h"

namespace pp {

constexpr unsigned long long kHitStride = 997;

static std::atomic<uint64_t> g_launches{0};
uint64_t kernel_launch_count() { return g_launches.load(); }

cudaError_t launch_ingest(const pp_source* s, const uint32_t* ev, const uint32_t* sid, uint32_t sid_base, uint32_t n,
                          float yield, SrcRec* out, unsigned int* overflow, cudaStream_t) {
  for (uint32_t i = 0; i < n; ++i) {
    unsigned long long cnt = host_photon_count(s[i].energy_GeV, yield);
    if (cnt > 0xFFFFFFFFull) { *overflow = 1; cnt = 0; }
    SrcRec r{};
    r.x = s[i].x; r.y = s[i].y; r.z = s[i].z; r.dx = s[i].dx; r.dy = s[i].dy; r.dz = s[i].dz; r.t = s[i].t_ns;
    r.energy = s[i].energy_GeV; r.event_id = ev[i]; r.source_id = sid ? sid[i] : sid_base + i;
    r.n_photons = (uint32_t)cnt; r.length = 0.0f;
    out[i] = r;
  }
  g_launches++;
  return cudaSuccess;
}

cudaError_t launch_scan(const SrcRec* src, uint32_t n, unsigned long long* cum, cudaStream_t) {
  unsigned long long run = 0;
  for (uint32_t i = 0; i < n; ++i) { cum[i] = run; run += src[i].n_photons; }
  cum[n] = run;
  g_launches++;
  return cudaSuccess;
}

cudaError_t launch_tiles(const unsigned long long*, uint32_t, unsigned long long, uint32_t, uint32_t, uint32_t*, uint32_t*,
                         Status* status, cudaStream_t) {
  if (status) *status = Status{};
  g_launches++;
  return cudaSuccess;  // the fake propagation walks the prefix sums itself
}

cudaError_t launch_prologue(const SrcRec* src, uint32_t n_src, unsigned long long* cum, unsigned long long, uint32_t,
                            uint32_t, uint32_t*, uint32_t*, Status* status, cudaStream_t st) {
  *status = Status{};
  return launch_scan(src, n_src, cum, st);
}

cudaError_t launch_propagate(const LaunchParams& P, bool, bool, int, size_t, cudaStream_t) {
  g_launches++;
  Status* st = P.status;
  pp_hit* ring = static_cast<pp_hit*>(P.ring);
  uint32_t n_out = 0;
  bool stopped = false;
  auto run_range = [&](unsigned long long g0, unsigned long long g1) {
    if (stopped) {
      if (g0 < g1 && n_out < P.resume_cap) P.resume_out[n_out++] = WorkItem{g0, g1, 0u, 0u};
      return;
    }
    unsigned long long g = (g0 + kHitStride - 1) / kHitStride * kHitStride;
    unsigned long long started_to = g1;
    for (; g < g1; g += kHitStride) {
      if (st->hit_count >= P.ring_cap) {  // ring full: the rest of this range is replayed by the next launch
        stopped = true;
        started_to = g;
        if (n_out < P.resume_cap) P.resume_out[n_out++] = WorkItem{g, g1, 0u, 0u};
        break;
      }
      // the source holding batch photon g
      const unsigned long long* it = std::upper_bound(P.cum, P.cum + P.n_src + 1, g);
      const uint32_t s = (uint32_t)(it - P.cum) - 1;
      pp_hit h{};
      h.event_id = P.src[s].event_id; h.source_id = P.src[s].source_id; h.photon_idx = (uint32_t)(g - P.cum[s]);
      h.dom_id = 0; h.time_ns = (double)P.src[s].t; h.weight = 1.0f; h.n_scatter = 0;
      ring[st->hit_count++] = h;
      st->photons_hit++;
    }
    st->photons_started += started_to - g0;
    st->flights += started_to - g0;
  };
  for (uint32_t r = 0; r < P.n_resume_in; ++r) run_range(P.resume_in[r].g0, P.resume_in[r].g1);
  st->resume_counter = P.n_resume_in;
  const unsigned long long fresh0 = std::min(P.g_end, P.g_begin + st->tile_counter * (unsigned long long)P.tile_photons);
  run_range(fresh0, P.g_end);
  st->tile_counter = P.n_tiles;
  st->n_resume_out = n_out;
  st->stop = stopped ? 1u : 0u;
  return cudaSuccess;
}

cudaError_t propagate_occupancy(bool, bool, size_t, int* blocks_per_sm) { *blocks_per_sm = 2; return cudaSuccess; }
int propagate_warps_per_block() { return 8; }

}  // namespace pp
