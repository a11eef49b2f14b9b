// TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Drives the host side of the library (built with -fsanitize=thread against
// the fake CUDA runtime and fake kernels of this directory) from many threads, the way the paper's clients drive the
// photon server, and checks the bookkeeping.  ThreadSanitizer reports go to stderr and make the
// exit code non-zero (TSAN_OPTIONS=exitcode=66 halt_on_error=1: the first report ends the run).
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <thread>
#include <unistd.h>
#include <vector>

#include "../../include/pp_ipc.h"
#include "../../include/pp_multi.h"

static int g_fail = 0;
#define CHECK(c) do { if (!(c)) { std::fprintf(stderr, "CHECK failed at %s:%d: %s\n", __FILE__, __LINE__, #c); g_fail = 1; } } while (0)

static const unsigned long long kHitStride = 997;

static std::vector<pp_source> make_sources(int n, float energy) {
  std::vector<pp_source> v(n);
  for (int i = 0; i < n; ++i) v[i] = pp_source{(float)i, 0.f, 0.f, 0.f, 0.f, 1.f, (float)i, energy};
  return v;
}

static pp_handle* make_handle(uint64_t target, uint64_t ring_bytes, uint64_t src_ring_bytes) {
  static const float xyz[3] = {0.f, 0.f, 0.f};
  static const float la[2] = {100.f, 80.f}, ls[2] = {25.f, 20.f};
  pp_geometry geo{1, xyz, 0.2f};
  pp_ice ice{2, 10.f, 10.f, la, ls, 0.9f, 1.35f, 0.75f, 1.0e4f};
  pp_config cfg{};
  cfg.launch_photons_target = target; cfg.hit_ring_bytes = ring_bytes; cfg.source_ring_bytes = src_ring_bytes;
  pp_handle* h = nullptr;
  const int rc = pp_create(&geo, &ice, &cfg, &h);
  CHECK(rc == PP_OK && h);
  return h;
}

// many producers, one consumer, small rings (back-pressure both ways), a tiny hit ring (relaunches), stats polled
static void test_threads() {
  pp_handle* h = make_handle(200000, 2 * 64 * 32, 256 * 48);  // launches of 2e5 photons, 64-hit ring, 256-source ring
  const int n_thr = 8, per = 40, blk = 25;
  const float e = 1.0f;  // 1e4 photons per source
  std::atomic<bool> done{false};
  std::atomic<uint64_t> hits{0};
  std::thread consumer([&] {
    std::vector<pp_hit> buf(4096);
    for (;;) {
      size_t n = 0;
      const int rc = pp_collect(h, buf.data(), buf.size(), &n, 1);
      CHECK(rc == PP_OK);
      hits += n;
      if (n == 0) { if (done.load()) return; usleep(200); }
    }
  });
  std::thread poll([&] { pp_stats_t st; while (!done.load()) { pp_stats(h, &st); usleep(300); } });
  std::vector<std::thread> prod;
  for (int t = 0; t < n_thr; ++t)
    prod.emplace_back([&, t] {
      auto src = make_sources(blk, e);
      std::vector<uint32_t> ev(blk, (uint32_t)t), sid(blk);
      for (int b = 0; b < per; ++b) {
        for (int i = 0; i < blk; ++i) sid[i] = (uint32_t)(b * blk + i);
        CHECK(pp_submit(h, src.data(), ev.data(), (b & 1) ? sid.data() : nullptr, blk) == PP_OK);
        if (b % 7 == 0) pp_flush(h);
      }
    });
  for (auto& t : prod) t.join();
  pp_flush(h);
  // drain
  for (;;) {
    pp_stats_t st;
    pp_stats(h, &st);
    if (st.photons_done == st.photons_submitted && st.sources_completed == st.sources_submitted) break;
    usleep(500);
  }
  done.store(true);
  consumer.join(); poll.join();
  std::vector<pp_hit> buf(4096);
  size_t n = 0;
  while (pp_collect(h, buf.data(), buf.size(), &n, 0) == PP_OK && n) hits += n;
  pp_stats_t st;
  pp_stats(h, &st);
  const uint64_t photons = (uint64_t)n_thr * per * blk * 10000ull;
  CHECK(st.photons_submitted == photons && st.photons_done == photons);
  CHECK(st.photons_hit == hits.load() && st.hits_collected == hits.load());
  CHECK(st.relaunches > 0 && st.launches >= photons / 200000);
  CHECK(hits.load() >= photons / kHitStride - st.launches - 8 && hits.load() <= photons / kHitStride + st.launches + 8);
  std::printf("threads: %llu photons, %llu hits, %llu launches, %llu relaunches\n", (unsigned long long)photons,
              (unsigned long long)hits.load(), (unsigned long long)st.launches, (unsigned long long)st.relaunches);
  pp_destroy(h);
}

// the multi-process front end with its clients as threads of this process (the shared-memory protocol is the same)
static void test_ipc(bool over_multi) {
  pp_handle* h0 = make_handle(100000, 0, 0);
  pp_handle* h1 = over_multi ? make_handle(100000, 0, 0) : nullptr;
  pp_multi* m = nullptr;
  pp_ipc_server* srv = nullptr;
  char name[64];
  std::snprintf(name, sizeof name, "/pp_tsan_%d_%d", (int)getpid(), over_multi ? 1 : 0);
  pp_ipc_config cfg{4, 0, 64 * 48, 64 * 32};  // rings of 64 sources / 64 hits: back-pressure both ways
  if (over_multi) {
    pp_handle* hs[2] = {h0, h1};
    pp_multi_config mc{150000, 1.0e4f, 0};
    CHECK(pp_multi_create(hs, 2, &mc, &m) == PP_OK);
    pp_ipc_backend be;
    CHECK(pp_multi_backend(m, &be) == PP_OK);
    CHECK(pp_ipc_server_create_backend(&be, name, &cfg, &srv) == PP_OK);
  } else {
    CHECK(pp_ipc_server_create(h0, name, &cfg, &srv) == PP_OK);
  }
  const int n_cl = 4, blocks = 12, blk = 30;
  std::atomic<uint64_t> hits{0};
  std::vector<std::thread> cl;
  for (int c = 0; c < n_cl; ++c)
    cl.emplace_back([&, c] {
      pp_ipc_client* k = nullptr;
      CHECK(pp_ipc_client_open(name, &k) == PP_OK);
      auto src = make_sources(blk, 2.0f);
      std::vector<pp_hit> buf(512);
      uint64_t mine = 0;
      for (int b = 0; b < blocks; ++b) {
        std::vector<uint32_t> ev(blk, (uint32_t)(c * 1000 + b));
        CHECK(pp_ipc_submit(k, src.data(), nullptr, ev.data(), nullptr, blk) == PP_OK);
        size_t n = 0;
        CHECK(pp_ipc_collect(k, buf.data(), buf.size(), &n, 0) == PP_OK);
        for (size_t i = 0; i < n; ++i) CHECK(buf[i].event_id / 1000 == (uint32_t)c);
        mine += n;
      }
      pp_ipc_flush(k);
      for (;;) {
        size_t n = 0;
        CHECK(pp_ipc_collect(k, buf.data(), buf.size(), &n, 1) == PP_OK);
        if (n == 0) break;
        for (size_t i = 0; i < n; ++i) CHECK(buf[i].event_id / 1000 == (uint32_t)c);
        mine += n;
      }
      hits += mine;
      pp_ipc_client_close(k);
    });
  for (auto& t : cl) t.join();
  pp_ipc_server_stats st;
  CHECK(pp_ipc_server_get_stats(srv, &st) == PP_OK);
  CHECK(st.hits_unrouted == 0 && st.sources_ingested == (uint64_t)n_cl * blocks * blk);
  CHECK(st.hits_routed == hits.load() && hits.load() > 0);
  std::printf("ipc%s: %llu sources, %llu hits routed\n", over_multi ? " over 2 devices" : "",
              (unsigned long long)st.sources_ingested, (unsigned long long)st.hits_routed);
  pp_ipc_server_destroy(srv);
  if (m) pp_multi_destroy(m);
  pp_destroy(h0);
  if (h1) pp_destroy(h1);
}

int main() {
  test_threads();
  test_ipc(false);
  test_ipc(true);
  std::printf(g_fail ? "FAILED\n" : "OK\n");
  return g_fail;
}
