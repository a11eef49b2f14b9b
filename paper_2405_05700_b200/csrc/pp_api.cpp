// Host side of the photon propagator: C ABI (include/pp.h), DOM-lookup construction, launch engine
// (two slots = two CUDA streams, double-buffered), and the batching server thread that turns a
// stream of pp_submit() calls from many producer threads into large GPU launches.
// Product code: shares nothing with oracle/.  No CPU fallback anywhere: every photon is tracked
// by the kernels in pp_kernels.cu.
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <condition_variable>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <deque>
#include <map>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include "pp_internal.h"

using namespace pp;

namespace {

constexpr double kC = 0.299792458;  // m/ns
constexpr size_t kStageBytes = 4u << 20;  // pinned D2H staging chunk per slot (x2)
constexpr size_t kHeadBytes = 128;        // the Status record sits this far in front of the hit ring (device and pinned)
constexpr uint64_t kFirstHits = 2048;     // hits read back in the same copy as the Status record (64 KiB)
static_assert(sizeof(Status) <= kHeadBytes, "Status must fit the ring head");
using Clock = std::chrono::steady_clock;

inline uint64_t align_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

#ifdef PP_GUARD
// Test-only guard build (tests/test_gpu_guard.py; pp_guard.cuh): every piece of the DEVICE workspace is followed by a
// zone of kGuardBytes filled with kGuardByte, which the host reads back and checks after every launch.
constexpr uint64_t kGuardBytes = 256;
constexpr unsigned char kGuardByte = 0xA5;
std::atomic<uint64_t> g_guard_zone_checks{0};
#endif

struct Carver {  // hands out aligned pieces of one workspace
  unsigned char* base;
  uint64_t off = 0;
  explicit Carver(void* b) : base(static_cast<unsigned char*>(b)) {}
#ifdef PP_GUARD
  std::vector<unsigned char*>* zones = nullptr;  // where the guard zones of the pieces handed out are noted
#endif
  template <class T>
  T* take(uint64_t count) {
    off = align_up(off, 256);
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += count * sizeof(T);
#ifdef PP_GUARD
    if (zones) {
      if (base) zones->push_back(base + off);
      off += kGuardBytes;
    }
#endif
    return p;
  }
};

struct HostGeometry {
  std::vector<StringRec> strings;
  std::vector<float4> dom_xyzw;
  std::vector<uint16_t> cell_sid;  // cell table, see pp_types.h
  uint32_t nx = 1, ny = 1;
  float cell_ox = 0, cell_oy = 0, inv_cell = 1, xy_cap = 1;
  bool fast_ok = false;
  std::string why;
};

struct Sizes {
  uint64_t cap_src = 0;      // records in the pinned source ring == per-slot device source capacity
  uint64_t max_tiles = 0;    // per launch
  uint64_t resume_cap = 0;   // WorkItems per resume list
  uint64_t ring_cap = 0;     // hits per slot ring
  uint64_t target = 0;       // photons per launch
};

struct Slot {
  cudaStream_t stream = nullptr;
  // device
  SrcRec* d_src = nullptr;
  unsigned long long* d_cum = nullptr;
  uint32_t* d_cum_rel = nullptr;
  uint32_t* d_tile_src = nullptr;
  Status* d_status = nullptr;
  WorkItem* d_resume[2] = {nullptr, nullptr};
  pp_hit* d_ring = nullptr;
  // pinned host
  Status* h_status = nullptr;     // D2H target; the first kFirstHits hits of the ring follow at kHeadBytes
  pp_hit* h_first = nullptr;
  Status* h_status_in = nullptr;  // H2D source of the cleared Status record
  unsigned long long* h_cum = nullptr;  // host-side prologue of a server launch: prefix sums and tile table
  uint32_t* h_cum_rel = nullptr;
  uint32_t* h_tile_src = nullptr;
  unsigned char* h_stage[2] = {nullptr, nullptr};
  cudaEvent_t ev_h2d = nullptr, ev_k0 = nullptr, ev_k1 = nullptr, ev_done = nullptr, ev_stage[2] = {nullptr, nullptr};
  // state of the launch in flight
  bool in_flight = false;
  uint64_t sources_end = 0;  // sources [0, sources_end) of the submit order are complete once this launch has retired
  int resume_sel = 0;  // which of d_resume[] is the OUT list of the launch in flight
  LaunchParams P;
  uint64_t seq = 0;
  bool fates = false;
  uint64_t photons = 0;       // photons of the launch in flight (fresh tiles)
  Clock::time_point t_enq{};  // when the launch was enqueued, and how long it should take once it has the GPU
  double expect_us = 0.0;
};

}  // namespace

struct pp_handle {
  pp_config cfg{};
  pp_ice ice{};
  int device = 0;
  int n_sm = 0, grid = 0;
  size_t smem = 0;
  bool brute = false;
  Sizes sz;
  HostGeometry hg;
  LaunchParams base{};  // medium + geometry filled in once
  std::vector<unsigned char> image;  // shared-memory tables as the kernel stages them (LaunchParams::smem_image)
  uint64_t image_bytes = 0;

  // memory
  void* dev_ws = nullptr; bool own_dev = false;
  void* pin_ws = nullptr; bool own_pin = false;
  bool own_streams = false;
  Slot slot[2];
  SrcRec* d_res_src = nullptr;            // resident batch
  unsigned long long* d_res_cum = nullptr;
  unsigned int* d_res_overflow = nullptr;
  unsigned long long* h_res_total = nullptr;  // pinned
  unsigned int* h_res_overflow = nullptr;     // pinned
  cudaEvent_t ev_base = nullptr, ev_job = nullptr;

  // source ring (pinned), positions are monotonically increasing record numbers
  SrcRec* ring = nullptr;
  std::mutex mu;  // the source ring, the launch bookkeeping and the stats below; NOT the hit queue (hit_mu)
  std::condition_variable cv_space, cv_work, cv_pub;
  uint64_t ring_reserve = 0;  // next record a producer may claim: producers copy into [ring_head, ring_reserve) outside the lock
  uint64_t next_auto_id = 0;  // running record number handed to sources submitted without ids
  uint64_t ring_head = 0;     // records below it are written and published (in order)
  uint64_t ring_launch = 0;   // first record not yet fully launched
  uint64_t ring_tail = 0;     // first record still needed
  uint64_t launch_offset = 0; // photons of record ring_launch already launched
  uint64_t queued_photons = 0;
  uint64_t flush_upto = 0;    // records below this position must be launched even if under target
  std::atomic<bool> shutdown{false};
  bool resident_active = false;
  int n_in_flight = 0;
  uint64_t inflight_photons = 0;  // photons of the launches in flight
  uint64_t launch_seq = 0;
  double us_per_photon = 7.0e-5;     // running estimate of the kernel time per photon (server thread's polling)
  Clock::time_point t_last_retire{};
  int space_waiters = 0;

  // finished hits waiting for pp_collect: a lock of their own, so that collecting never waits for a producer
  // copying sources or for the server cutting a launch (and vice versa).  Never held together with mu.
  std::mutex hit_mu;
  std::condition_variable cv_hits, cv_hit_space;
  std::deque<std::vector<pp_hit>> hitq;
  size_t hitq_front_off = 0;
  uint64_t hitq_bytes = 0, hitq_budget = 0;
  uint64_t hits_collected = 0, hit_high_water = 0;  // under hit_mu; folded into pp_stats

  // stats
  pp_stats_t st{};
  bool wall_started = false;
  Clock::time_point wall_t0, wall_t1;
  double busy_end_ms = 0;

#ifdef PP_GUARD
  std::vector<unsigned char*> guard_zones;  // device addresses of the guard zones behind the workspace pieces
#endif

  // error state
  std::atomic<int> sticky{PP_OK};
  std::string err;
  std::mutex err_mu;

  std::thread server;
};

namespace {

int fail(pp_handle* h, int code, const std::string& msg) {
  if (h) {
    std::lock_guard<std::mutex> g(h->err_mu);
    h->err = msg;
    if (code == PP_E_CUDA) h->sticky.store(PP_E_CUDA);
  }
  return code;
}

#define PP_CUDA(h, call)                                                                        \
  do {                                                                                          \
    cudaError_t e__ = (call);                                                                   \
    if (e__ != cudaSuccess)                                                                     \
      return fail((h), PP_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__));         \
  } while (0)

// ---------------------------------------------------------------------------------------------
// validation
// ---------------------------------------------------------------------------------------------
bool finite_f(float x) { return std::isfinite(x); }

int validate_inputs(const pp_geometry* geo, const pp_ice* ice, std::string* why) {
  if (!geo || !ice || !geo->xyz || !ice->abs_len || !ice->scat_len) { *why = "null pointer"; return PP_E_INVAL; }
  if (geo->n_dom == 0 || !(geo->radius > 0.0f) || !finite_f(geo->radius)) { *why = "bad geometry"; return PP_E_INVAL; }
  for (uint32_t i = 0; i < 3 * geo->n_dom; ++i)
    if (!finite_f(geo->xyz[i])) { *why = "non-finite DOM coordinate"; return PP_E_INVAL; }
  if (ice->n_layers == 0 || ice->n_layers > PP_MAX_LAYERS) { *why = "n_layers out of range"; return PP_E_INVAL; }
  if (!(ice->dz > 0.0f) || !finite_f(ice->dz) || !finite_f(ice->z_top)) { *why = "bad layer grid"; return PP_E_INVAL; }
  for (uint32_t i = 0; i < ice->n_layers; ++i)
    if (!(ice->abs_len[i] > 0.0f) || !(ice->scat_len[i] > 0.0f) || std::isnan(ice->abs_len[i]) ||
        std::isnan(ice->scat_len[i])) { *why = "non-positive length in ice table"; return PP_E_INVAL; }
  if (!(std::fabs(ice->g) < 1.0f)) { *why = "|g| must be < 1"; return PP_E_INVAL; }
  if (!(ice->n_group > 0.0f) || !finite_f(ice->n_group)) { *why = "bad n_group"; return PP_E_INVAL; }
  if (!(ice->cos_cherenkov >= -1.0f && ice->cos_cherenkov <= 1.0f)) { *why = "bad cos_cherenkov"; return PP_E_INVAL; }
  if (!(ice->photons_per_GeV >= 0.0f) || !finite_f(ice->photons_per_GeV)) { *why = "bad yield"; return PP_E_INVAL; }
  return PP_OK;
}

// ---------------------------------------------------------------------------------------------
// a5 (host part): group DOMs into vertical lines, build the 2-D cell grid over the footprint
// ---------------------------------------------------------------------------------------------
void build_geometry(const pp_geometry* geo, bool brute, HostGeometry* out) {
  const uint32_t n = geo->n_dom;
  out->fast_ok = false;
  if (brute) {
    // validation mode: every DOM in input order (the cell table of the fast path is still built when the
    // geometry allows it, only to report the same xy cap)
    HostGeometry fast;
    build_geometry(geo, false, &fast);
    out->xy_cap = fast.fast_ok ? fast.xy_cap : 100.0f;
    out->dom_xyzw.resize(n);
    for (uint32_t j = 0; j < n; ++j) {
      float4 v;
      v.x = geo->xyz[3 * j]; v.y = geo->xyz[3 * j + 1]; v.z = geo->xyz[3 * j + 2];
      std::memcpy(&v.w, &j, 4);
      out->dom_xyzw[j] = v;
    }
    out->cell_sid.assign(1, kNoString);
    return;
  }
  struct Dom { float z; uint32_t id; };
  std::map<std::pair<uint32_t, uint32_t>, std::vector<Dom>> lines;  // key = bit patterns of (x, y)
  for (uint32_t j = 0; j < n; ++j) {
    uint32_t bx, by;
    float x = geo->xyz[3 * j] + 0.0f, y = geo->xyz[3 * j + 1] + 0.0f;  // +0: fold -0 into +0
    std::memcpy(&bx, &x, 4); std::memcpy(&by, &y, 4);
    lines[{bx, by}].push_back(Dom{geo->xyz[3 * j + 2], j});
  }
  if (lines.size() > (size_t)kMaxStringsSmem) { out->why = "more than 512 vertical lines of DOMs"; return; }
  out->dom_xyzw.reserve(n);
  std::vector<std::pair<float, float>> xy;
  for (auto& kv : lines) {
    auto& v = kv.second;
    std::sort(v.begin(), v.end(), [](const Dom& a, const Dom& b) { return a.z > b.z || (a.z == b.z && a.id < b.id); });
    float x, y;
    std::memcpy(&x, &kv.first.first, 4); std::memcpy(&y, &kv.first.second, 4);
    StringRec r{};
    r.x = x; r.y = y; r.z0 = v[0].z; r.n = (uint32_t)v.size(); r.base = (uint32_t)out->dom_xyzw.size();
    double pitch = 1.0;
    if (v.size() > 1) {
      pitch = ((double)v.front().z - (double)v.back().z) / (double)(v.size() - 1);
      if (!(pitch > 0.0)) { out->why = "two DOMs at the same position"; return; }
      for (size_t k = 0; k < v.size(); ++k)
        if (std::fabs((double)v[k].z - ((double)v[0].z - k * pitch)) > 1e-3 * pitch + 1e-4) {
          out->why = "DOMs of a vertical line are not uniformly spaced";
          return;
        }
    }
    r.pitch = (float)pitch; r.inv_pitch = (float)(1.0 / pitch);
    out->strings.push_back(r);
    xy.push_back({x, y});
    for (auto& d : v) {
      float4 c; c.x = x; c.y = y; c.z = d.z;
      std::memcpy(&c.w, &d.id, 4);
      out->dom_xyzw.push_back(c);
    }
  }
  // ---- cell table: THE candidate line for a piece of flight whose xy midpoint lies in a cell ----
  // A piece of xy length <= L that passes within Rm of a line has its midpoint within L/2 + Rm of it.
  // If every cell is within reach = L/2 + Rm + slack of at most one line, the cell names that line; this
  // holds when 2 reach + (cell diagonal) < d_min, the smallest distance between two lines.
  const size_t ns = xy.size();
  double d_min = 1e30;
  for (size_t i = 0; i < ns; ++i)
    for (size_t j = i + 1; j < ns; ++j)
      d_min = std::min(d_min, std::hypot((double)xy[i].first - xy[j].first, (double)xy[i].second - xy[j].second));
  const double Rm = (double)geo->radius + 5e-3, slack = 0.02;
  const double L_max = 112.0;   // longest piece of flight looked up at once (metres): as long as the line spacing allows
  const double cell_div = 12.0;  // cells per smallest line distance: finer cells leave room for longer pieces (a
                                 // flight is then cut into 1.42 instead of 1.54 pieces on average: +1.8 %, profiles/r02_v13.md)
  double cell = ns > 1 ? d_min / cell_div : 32.0;
  double L = ns > 1 ? std::min(L_max, d_min - 2.0 * (Rm + slack) - cell * std::sqrt(2.0) - slack) : L_max;
  double x0 = 1e30, x1 = -1e30, y0 = 1e30, y1 = -1e30;
  for (auto& p : xy) { x0 = std::min(x0, (double)p.first); x1 = std::max(x1, (double)p.first);
                       y0 = std::min(y0, (double)p.second); y1 = std::max(y1, (double)p.second); }
  for (int attempt = 0;; ++attempt) {
    if (!(L >= 1.0) || attempt > 60) { out->why = "lines of DOMs too dense for the cell table"; return; }
    const double reach = 0.5 * L + Rm + slack, pad = reach + 2.0 * cell;  // >= one ring of empty cells all around
    const double gx0 = x0 - pad, gy0 = y0 - pad;
    const uint64_t nx = (uint64_t)std::ceil((x1 + pad - gx0) / cell) + 1, ny = (uint64_t)std::ceil((y1 + pad - gy0) / cell) + 1;
    if (nx * ny > 40000) {  // keep the table in shared memory: coarser cells, shorter pieces
      cell *= 1.25;
      L = std::min(L, d_min - 2.0 * (Rm + slack) - cell * std::sqrt(2.0) - slack);
      continue;
    }
    out->cell_sid.assign((size_t)(nx * ny), kNoString);
    bool clash = false;
    for (size_t s = 0; s < ns && !clash; ++s) {
      const double sx = xy[s].first, sy = xy[s].second;
      const int64_t ix0 = std::max<int64_t>(0, (int64_t)std::floor((sx - reach - gx0) / cell) - 1);
      const int64_t ix1 = std::min<int64_t>((int64_t)nx - 1, (int64_t)std::floor((sx + reach - gx0) / cell) + 1);
      const int64_t iy0 = std::max<int64_t>(0, (int64_t)std::floor((sy - reach - gy0) / cell) - 1);
      const int64_t iy1 = std::min<int64_t>((int64_t)ny - 1, (int64_t)std::floor((sy + reach - gy0) / cell) + 1);
      for (int64_t iy = iy0; iy <= iy1 && !clash; ++iy)
        for (int64_t ix = ix0; ix <= ix1; ++ix) {
          // distance from the line's axis to the cell rectangle
          const double cx0 = gx0 + ix * cell, cy0 = gy0 + iy * cell;
          const double ddx = std::max({cx0 - sx, 0.0, sx - (cx0 + cell)}), ddy = std::max({cy0 - sy, 0.0, sy - (cy0 + cell)});
          if (ddx * ddx + ddy * ddy > reach * reach) continue;
          uint16_t& c = out->cell_sid[(size_t)iy * nx + (size_t)ix];
          if (c != kNoString) { clash = true; break; }
          c = (uint16_t)s;
        }
    }
    if (clash) { L *= 0.9; continue; }
    // the clamp in the kernel relies on an empty outer ring
    for (uint64_t ix = 0; ix < nx; ++ix)
      if (out->cell_sid[ix] != kNoString || out->cell_sid[(ny - 1) * nx + ix] != kNoString) { out->why = "internal: cell ring"; return; }
    for (uint64_t iy = 0; iy < ny; ++iy)
      if (out->cell_sid[iy * nx] != kNoString || out->cell_sid[iy * nx + nx - 1] != kNoString) { out->why = "internal: cell ring"; return; }
    out->nx = (uint32_t)nx; out->ny = (uint32_t)ny;
    out->inv_cell = (float)(1.0 / cell);
    out->cell_ox = (float)(-gx0 / cell); out->cell_oy = (float)(-gy0 / cell);
    out->xy_cap = (float)L;
    break;
  }
  out->fast_ok = true;
}

// Medium and geometry constants of a handle and the image of the shared-memory tables (a4, a5; layout in
// pp_types.h).  Host only: pp_workspace_size() needs the image size, pp_create() uploads the image.
int build_tables(pp_handle* h, const pp_geometry* geo, const pp_ice* ice, const pp_config* cfg) {
  LaunchParams& B = h->base;
  const double scat_scale = (cfg->flags & PP_FLAG_EFFECTIVE_SCATTERING) ? 1.0 - (double)ice->g : 1.0;
  if (!(scat_scale > 0.0)) return PP_E_INVAL;
  const uint32_t nl = ice->n_layers;
  std::vector<LayerRec> layers(nl + 1);
  for (uint32_t i = 0; i < nl; ++i) {
    // R-20: an effective scattering length is turned into the geometric mean free path here, once
    const double ls = (double)ice->scat_len[i] * scat_scale;
    layers[i].lb = (float)ls;
    layers[i].a = layers[i].a2 = (float)(1.0 / (double)ice->abs_len[i]); layers[i].b = (float)(1.0 / ls);
  }
  layers[nl] = layers[nl - 1];
  B.n_layers = nl; B.last_layer = (int32_t)nl - 1;
  B.z_top = ice->z_top; B.dz_layer = ice->dz; B.inv_dz_layer = (float)(1.0 / (double)ice->dz);
  const double g = ice->g;
  B.hg_one_minus_g = (float)(1.0 - g); B.hg_two_g = (float)(2.0 * g); B.hg_one_minus_g2 = (float)(1.0 - g * g);
  B.one_minus_cos_c = (float)(1.0 - (double)ice->cos_cherenkov);
  B.inv_v = (double)ice->n_group / kC;
  B.inv_c = (float)(1.0 / kC);
  {
    uint32_t k0 = (uint32_t)cfg->seed, k1 = (uint32_t)(cfg->seed >> 32);
    for (int r = 0; r < 10; ++r) { B.rk[r][0] = k0; B.rk[r][1] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
  }
  if (cfg->max_flights >= 0x80000000u) return PP_E_INVAL;  // the kernel keeps a flag in the counter's top bit
  B.max_flights = cfg->max_flights ? cfg->max_flights : 100000u;
  B.tile_photons = kTilePhotons;
  const uint32_t ns = (uint32_t)h->hg.strings.size();
  B.n_strings = ns; B.n_dom = geo->n_dom;
  B.nx = h->hg.nx; B.nx_m1 = h->hg.nx - 1u; B.ny_m1 = h->hg.ny - 1u;
  B.cell_ox = h->hg.cell_ox; B.cell_oy = h->hg.cell_oy; B.inv_cell = h->hg.inv_cell;
  B.radius = geo->radius; B.radius_margin = geo->radius + 5e-3f;
  B.rm2 = B.radius_margin * B.radius_margin;
  B.xy_cap2 = h->hg.xy_cap * h->hg.xy_cap; B.inv_xy_cap = 1.0f / h->hg.xy_cap;
  // ---- a4: tables of the direct layer walk (pp_types.h) ----
  std::vector<uint16_t> inv_tab;  // layer holding a cumulative SCATTERING depth (the walk follows absorption along)
  {
    std::vector<double> cum[2] = {std::vector<double>(nl + 1, 0.0), std::vector<double>(nl + 1, 0.0)};  // B, A
    for (uint32_t i = 0; i < nl; ++i) {
      cum[0][i + 1] = cum[0][i] + (double)ice->dz / ((double)ice->scat_len[i] * scat_scale);
      cum[1][i + 1] = cum[1][i] + (double)ice->dz / (double)ice->abs_len[i];
    }
    for (uint32_t i = 0; i <= nl; ++i) {
      const float bh = (float)cum[0][i], ah = (float)cum[1][i];
      layers[i].Bh = bh; layers[i].Ah = ah;
      layers[i].Bl = (float)(cum[0][i] - (double)bh); layers[i].Al = (float)(cum[1][i] - (double)ah);
    }
    layers[nl].Bh = layers[nl].Ah = INFINITY; layers[nl].Bl = layers[nl].Al = 0.0f;
    B.walk_loop = 0;
    {
      const int t = 0;
      // bin width: just under the thinnest layer, so that a bin holds at most one boundary; coarser (and the
      // kernel then loops) if that would need more than kMaxWalkInv bins
      double thin = 1e300;
      for (uint32_t i = 0; i < nl; ++i) thin = std::min(thin, cum[t][i + 1] - cum[t][i]);
      const double top = nl > 1 ? cum[t][nl - 1] : 0.0;  // cumulative depth at the upper edge of the last layer
      double step = 0.99 * thin;
      if (top / step + 3.0 > (double)kMaxWalkInv) { step = top / ((double)kMaxWalkInv - 3.0); B.walk_loop = 1; }
      const uint32_t m = (uint32_t)std::ceil(top / step) + 1;  // bins 0..m
      inv_tab.resize(m + 1);
      uint32_t j = 0;
      for (uint32_t b = 0; b <= m; ++b) {
        // a lower bound of the layer for every depth that can land in bin b (index rounding slack 4e-3 bins)
        const double x = ((double)b - 4e-3) * step;
        while (j + 1 < nl && (double)layers[j + 1].Bh <= x) ++j;
        inv_tab[b] = (uint16_t)j;
      }
      B.m_b = m;
      B.k_b = (float)(1.0 / step);
    }
  }
  // ---- the image ----
  std::vector<float2> str_xy(ns + 1);
  std::vector<float4> str_a(ns);
  std::vector<uint2> str_b(ns);
  for (uint32_t i = 0; i < ns; ++i) {
    const StringRec& r = h->hg.strings[i];
    str_xy[i] = make_float2(r.x, r.y);
    str_a[i] = make_float4(r.x, r.y, r.z0, r.inv_pitch);
    str_b[i] = make_uint2(r.n, r.base);
  }
  str_xy[ns] = make_float2(NAN, NAN);  // what an empty cell names: fails the pre-filter
  std::vector<uint16_t> cell(h->hg.cell_sid);
  for (auto& c : cell) if (c == kNoString) c = (uint16_t)ns;
  std::vector<unsigned char>& img = h->image;
  img.clear();
  auto put = [&](const void* src, size_t bytes) {
    const size_t off = (img.size() + 15) & ~(size_t)15;
    img.resize(off + bytes, 0);
    if (bytes) std::memcpy(img.data() + off, src, bytes);
    return (uint32_t)off;
  };
  put(layers.data(), layers.size() * sizeof(LayerRec));
  {
    std::vector<LayerRec> rec_b(layers);
    for (uint32_t i = 0; i < nl; ++i) {
      const LayerRec& lo = layers[std::min(i + 1, nl - 1)];  // finite at the bottom edge (pp_types.h)
      rec_b[i].Bh = lo.Bh; rec_b[i].Ah = lo.Ah; rec_b[i].Bl = lo.Bl; rec_b[i].Al = lo.Al;
    }
    rec_b[nl] = rec_b[nl - 1];
    B.off_rec_b = put(rec_b.data(), rec_b.size() * sizeof(LayerRec));
  }
  B.off_inv_b = put(inv_tab.data(), inv_tab.size() * sizeof(uint16_t));
  B.off_str_xy = put(str_xy.data(), str_xy.size() * sizeof(float2));
  B.off_cell = put(cell.data(), cell.size() * sizeof(uint16_t));
  B.off_str_a = put(str_a.data(), str_a.size() * sizeof(float4));
  B.off_str_b = put(str_b.data(), str_b.size() * sizeof(uint2));
  img.resize((img.size() + 15) & ~(size_t)15, 0);
  h->image_bytes = img.size();
  B.smem_image_bytes = (uint32_t)img.size();
  h->smem = img.size();
  return PP_OK;
}

void fill_sizes(const pp_config& cfg, int n_sm, Sizes* s) {
  s->target = cfg.launch_photons_target ? cfg.launch_photons_target : 100000000ull;
  const uint64_t src_bytes = cfg.source_ring_bytes ? cfg.source_ring_bytes : (64ull << 20);
  s->cap_src = std::max<uint64_t>(64, src_bytes / sizeof(SrcRec));
  // large launches: target / kTilePhotons tiles; small ones use smaller tiles but never more than 8 per warp
  s->max_tiles = std::max<uint64_t>((s->target + kTilePhotons - 1) / kTilePhotons, (uint64_t)n_sm * 64ull * 8ull) + 2;
  s->resume_cap = (uint64_t)n_sm * 2048ull * 2ull + 4096ull;
  const uint64_t hit_bytes = cfg.hit_ring_bytes ? cfg.hit_ring_bytes : (256ull << 20);
  s->ring_cap = std::max<uint64_t>(32, std::min<uint64_t>(hit_bytes / 2 / sizeof(pp_hit), 0xFFFFFF00ull));
}

// Carve (or, with null base, just measure) the device workspace.
uint64_t carve_device(pp_handle* h, void* base) {
  Carver c(base);
#ifdef PP_GUARD
  h->guard_zones.clear();
  c.zones = &h->guard_zones;
#endif
  const HostGeometry& g = h->hg;
  h->base.smem_image = c.take<uint4>(h->image_bytes / 16);
  h->base.dom_xyzw = c.take<float4>(g.dom_xyzw.size());
  for (int i = 0; i < 2; ++i) {
    Slot& s = h->slot[i];
    s.d_src = c.take<SrcRec>(h->sz.cap_src);
    s.d_cum = c.take<unsigned long long>(h->sz.cap_src + 1);
    s.d_cum_rel = c.take<uint32_t>(h->sz.cap_src + 1);
    s.d_tile_src = c.take<uint32_t>(h->sz.max_tiles);
    s.d_resume[0] = c.take<WorkItem>(h->sz.resume_cap);
    s.d_resume[1] = c.take<WorkItem>(h->sz.resume_cap);
    // [Status | pad to kHeadBytes | pp_hit x ring_cap]: one device-to-host copy brings the status and the first hits
    unsigned char* sr = c.take<unsigned char>(kHeadBytes + h->sz.ring_cap * sizeof(pp_hit));
    s.d_status = reinterpret_cast<Status*>(sr);
    s.d_ring = reinterpret_cast<pp_hit*>(sr ? sr + kHeadBytes : nullptr);
  }
  h->d_res_src = c.take<SrcRec>(h->sz.cap_src);
  h->d_res_cum = c.take<unsigned long long>(h->sz.cap_src + 1);
  h->d_res_overflow = c.take<unsigned int>(4);
  return align_up(c.off, 256);
}

uint64_t carve_pinned(pp_handle* h, void* base) {
  Carver c(base);
  h->ring = c.take<SrcRec>(h->sz.cap_src);
  for (int i = 0; i < 2; ++i) {
    Slot& s = h->slot[i];
    unsigned char* hs = c.take<unsigned char>(kHeadBytes + kFirstHits * sizeof(pp_hit));
    s.h_status = reinterpret_cast<Status*>(hs);
    s.h_first = reinterpret_cast<pp_hit*>(hs ? hs + kHeadBytes : nullptr);
    s.h_status_in = c.take<Status>(1);
    s.h_cum = c.take<unsigned long long>(h->sz.cap_src + 1);
    s.h_cum_rel = c.take<uint32_t>(h->sz.cap_src + 1);
    s.h_tile_src = c.take<uint32_t>(h->sz.max_tiles);
    s.h_stage[0] = c.take<unsigned char>(kStageBytes);
    s.h_stage[1] = c.take<unsigned char>(kStageBytes);
  }
  h->h_res_total = c.take<unsigned long long>(2);
  h->h_res_overflow = c.take<unsigned int>(4);
  return align_up(c.off, 256);
}

// ---------------------------------------------------------------------------------------------
// launch engine
// ---------------------------------------------------------------------------------------------

// a9, first part: the Status record and the first kFirstHits hits of the ring in ONE device-to-host copy (they are
// contiguous on both sides): a launch with few hits -- every small launch -- needs no second copy.
cudaError_t read_back_head(pp_handle* h, Slot& s) {
  const size_t bytes = kHeadBytes + (size_t)std::min<uint64_t>(kFirstHits, h->sz.ring_cap) * sizeof(pp_hit);
  return cudaMemcpyAsync(s.h_status, s.d_status, bytes, cudaMemcpyDeviceToHost, s.stream);
}

// Tile size of a launch: 1024 photons for large launches; a small launch is cut finer so that every resident warp
// gets work (about 4 tiles per warp), which is what sets the latency of a launch the GPU is too big for (C3).
void pick_tiles(const pp_handle* h, uint64_t n_ph, uint32_t* tile_photons, uint32_t* n_tiles) {
  uint32_t tile = kTilePhotons;
  const uint64_t want_tiles = (uint64_t)h->grid * (uint64_t)propagate_warps_per_block() * 4ull;
  while (tile > (uint32_t)kMinTilePhotons && n_ph / tile < want_tiles) tile >>= 1;
  *tile_photons = tile;
  *n_tiles = (uint32_t)std::min<uint64_t>((n_ph + tile - 1) / tile, 0xFFFFFFFFull);
}

// cum[s] - g_begin in 32 bits as the kernels read it (LaunchParams::cum_rel)
inline uint32_t rel32(uint64_t c, uint64_t g_begin) {
  return c < g_begin ? (uint32_t)(c - g_begin) : (uint32_t)std::min<uint64_t>(c - g_begin, 0xFFFFFFFFull);
}

// a2 on the host, for launches cut by the batching server: the server walks the queued records anyway, so it
// writes the prefix sums, their launch-relative form and the tile -> source table itself, into pinned memory that
// travels with the records.  A launch then needs no kernel in front of the propagation kernel, which matters because
// that kernel could not start before the previous launch has left an SM: with the tables uploaded by the copy engine
// the next launch's CTAs move in as the previous launch's move out.  `count_at(q)` = photons of the launch's q-th
// record.  Returns the total.
template <class CountAt>
uint64_t host_prologue(Slot& s, CountAt count_at, uint32_t n_src, uint64_t g_begin, uint32_t tile, uint32_t n_tiles) {
  uint64_t run = 0;
  for (uint32_t q = 0; q < n_src; ++q) {
    s.h_cum[q] = run; s.h_cum_rel[q] = rel32(run, g_begin);
    run += count_at(q);
  }
  s.h_cum[n_src] = run; s.h_cum_rel[n_src] = rel32(run, g_begin);
  uint32_t si = 0;  // tile_src[j] = the last source with cum <= the tile's first photon (skips sources without photons)
  for (uint32_t j = 0; j < n_tiles; ++j) {
    const uint64_t g = g_begin + (uint64_t)j * tile;
    while (si + 1 < n_src && s.h_cum[si + 1] <= g) ++si;
    s.h_tile_src[j] = si;
  }
  *s.h_status_in = Status{};
  return run;
}

// Enqueue tiles + propagate (+ status read-back) for photons [g_begin, g_end) of the batch
// (src, cum, n_src), which must already be (or be enqueued to become) resident on slot.stream.
// `host_tables`: host_prologue() has filled the slot's pinned tables for exactly this launch; they are uploaded
// instead of being computed by the scan / tiles kernels.
int enqueue_launch(pp_handle* h, Slot& s, const SrcRec* src, unsigned long long* cum, uint32_t n_src,
                   uint64_t g_begin, uint64_t g_end, pp_fate* fates, bool has_segments, bool need_scan,
                   bool host_tables = false) {
  const uint64_t n_ph = g_end - g_begin;
  uint32_t tile = 0, n_tiles = 0;
  pick_tiles(h, n_ph, &tile, &n_tiles);
  if (n_tiles > h->sz.max_tiles) return fail(h, PP_E_NOMEM, "launch larger than launch_photons_target");
  if (host_tables) {
    PP_CUDA(h, cudaMemcpyAsync(cum, s.h_cum, ((size_t)n_src + 1) * sizeof(unsigned long long), cudaMemcpyHostToDevice, s.stream));
    PP_CUDA(h, cudaMemcpyAsync(s.d_cum_rel, s.h_cum_rel, ((size_t)n_src + 1) * sizeof(uint32_t), cudaMemcpyHostToDevice, s.stream));
    PP_CUDA(h, cudaMemcpyAsync(s.d_tile_src, s.h_tile_src, (size_t)n_tiles * sizeof(uint32_t), cudaMemcpyHostToDevice, s.stream));
    PP_CUDA(h, cudaMemcpyAsync(s.d_status, s.h_status_in, sizeof(Status), cudaMemcpyHostToDevice, s.stream));
  } else if (need_scan && n_src <= kPrologueMax && n_tiles <= kPrologueMax) {
    // a2 on the device (resident path): prefix sums (unless the batch is scanned already), tile -> source table,
    // launch-relative prefix sums; the status record is cleared by the same kernel.  Small launches do all of it in
    // one single-CTA kernel.
    PP_CUDA(h, launch_prologue(src, n_src, cum, g_begin, n_tiles, tile, s.d_tile_src, s.d_cum_rel, s.d_status, s.stream));
  } else {
    if (need_scan) PP_CUDA(h, launch_scan(src, n_src, cum, s.stream));
    PP_CUDA(h, launch_tiles(cum, n_src, g_begin, n_tiles, tile, s.d_tile_src, s.d_cum_rel, s.d_status, s.stream));
  }
  LaunchParams P = h->base;
  P.src = src; P.cum = cum; P.cum_rel = s.d_cum_rel; P.tile_src = s.d_tile_src;
  P.g_begin = g_begin; P.g_end = g_end; P.n_src = n_src; P.n_tiles = n_tiles; P.tile_photons = tile;
  P.has_segments = has_segments ? 1u : 0u;
  s.resume_sel = 0;
  P.resume_in = s.d_resume[1]; P.resume_out = s.d_resume[0];
  P.n_resume_in = 0; P.resume_cap = (uint32_t)h->sz.resume_cap;
  P.status = s.d_status; P.ring = s.d_ring; P.ring_cap = (uint32_t)h->sz.ring_cap;
  P.fates = fates;
  s.fates = fates != nullptr;
  s.P = P;
  PP_CUDA(h, cudaEventRecord(s.ev_k0, s.stream));
  PP_CUDA(h, launch_propagate(P, h->brute, s.fates, h->grid, h->smem, s.stream));
  PP_CUDA(h, cudaEventRecord(s.ev_k1, s.stream));
  PP_CUDA(h, read_back_head(h, s));
  PP_CUDA(h, cudaEventRecord(s.ev_done, s.stream));
  s.in_flight = true;
  s.seq = ++h->launch_seq;
  s.t_enq = Clock::now();
  s.expect_us = 60.0 + (double)n_ph * h->us_per_photon;
  return PP_OK;
}

// Push finished hits to the collect queue (bounded: blocks the server while the consumer is behind,
// which in turn back-pressures pp_submit; the resident path fails instead of dead-locking).
int push_hits(pp_handle* h, std::vector<pp_hit>&& v, bool may_block) {
  if (v.empty()) return PP_OK;
  std::unique_lock<std::mutex> lk(h->hit_mu);
  const uint64_t bytes = v.size() * sizeof(pp_hit);
  while (h->hitq_bytes + bytes > h->hitq_budget && h->hitq_bytes > 0) {
    if (!may_block) return fail(h, PP_E_NOMEM, "host hit queue budget exceeded in pp_run_resident; collect more often");
    if (h->shutdown.load()) break;
    h->cv_hit_space.wait_for(lk, std::chrono::milliseconds(20));
  }
  h->hitq_bytes += bytes;
  h->hit_high_water = std::max<uint64_t>(h->hit_high_water, bytes);
  h->hitq.push_back(std::move(v));
  h->cv_hits.notify_all();
  return PP_OK;
}

// Wait for the slot's launch, stream its hits to the host in chunks, relaunch if the ring filled up.
int finish_slot(pp_handle* h, Slot& s, bool may_block) {
  PP_CUDA(h, cudaEventSynchronize(s.ev_done));
  const Status hs = *s.h_status;
  if (hs.error) return fail(h, PP_E_CUDA, hs.error == 1u ? std::string("internal: resume list overflow")
                                                          : "internal: guard check " + std::to_string(hs.error) + " failed in the kernel");
#ifdef PP_GUARD
  {
    // every launch: the zones behind the workspace pieces must still hold their pattern (one small copy per zone; the
    // guard build is not timed)
    unsigned char z[kGuardBytes];
    for (size_t q = 0; q < h->guard_zones.size(); ++q) {
      PP_CUDA(h, cudaMemcpyAsync(z, h->guard_zones[q], kGuardBytes, cudaMemcpyDeviceToHost, s.stream));
      PP_CUDA(h, cudaStreamSynchronize(s.stream));
      for (uint64_t b = 0; b < kGuardBytes; ++b)
        if (z[b] != kGuardByte)
          return fail(h, PP_E_CUDA, "internal: guard zone " + std::to_string(q) + " behind a workspace piece was overwritten at byte " + std::to_string(b));
      g_guard_zone_checks++;
    }
  }
#endif
  float t0 = 0, t1 = 0;
  PP_CUDA(h, cudaEventElapsedTime(&t0, h->ev_base, s.ev_k0));
  PP_CUDA(h, cudaEventElapsedTime(&t1, h->ev_base, s.ev_k1));
  // ---- a9: stream the valid part of the ring to the host through two pinned staging chunks ----
  const uint64_t n_valid = std::min<uint64_t>(hs.hit_count, h->sz.ring_cap);
  std::vector<pp_hit> hits(n_valid);
  {
    // the first hits came with the status record; the rest through the two staging chunks, two copies in flight
    const uint64_t n_first = std::min<uint64_t>(n_valid, kFirstHits);
    std::memcpy(hits.data(), s.h_first, n_first * sizeof(pp_hit));
    const uint64_t per = kStageBytes / sizeof(pp_hit);
    uint64_t issued = n_first, done = n_first;
    uint64_t n_issued = 0, n_done = 0;
    uint64_t cnt[2] = {0, 0};
    while (done < n_valid) {
      while (issued < n_valid && n_issued - n_done < 2) {
        const int bi = (int)(n_issued & 1);
        cnt[bi] = std::min<uint64_t>(per, n_valid - issued);
        PP_CUDA(h, cudaMemcpyAsync(s.h_stage[bi], s.d_ring + issued, cnt[bi] * sizeof(pp_hit), cudaMemcpyDeviceToHost,
                                   s.stream));
        PP_CUDA(h, cudaEventRecord(s.ev_stage[bi], s.stream));
        issued += cnt[bi];
        n_issued++;
      }
      const int b = (int)(n_done & 1);
      PP_CUDA(h, cudaEventSynchronize(s.ev_stage[b]));
      std::memcpy(hits.data() + done, s.h_stage[b], cnt[b] * sizeof(pp_hit));
      done += cnt[b];
      n_done++;
    }
  }
  {
    std::lock_guard<std::mutex> g(h->mu);
    h->st.photons_done += hs.photons_started;
    h->st.photons_hit += hs.photons_hit;
    h->st.photons_aborted += hs.photons_aborted;
    h->st.photons_rejected += hs.photons_rejected;
    h->st.photons_absorbed += hs.photons_started - hs.photons_hit - hs.photons_aborted - hs.photons_rejected;
    h->st.flights += hs.flights;
    h->st.launches += 1;
    // time this launch had the GPU to itself: from the end of the launch before it (its CTAs move in as that one's
    // move out) or from its own start, whichever is later
    const double own_ms = std::max(0.0, (double)t1 - std::max((double)t0, h->busy_end_ms));
    h->st.kernel_busy_ms += own_ms;
    h->busy_end_ms = std::max(h->busy_end_ms, (double)t1);
    if (hs.photons_started > 1000000ull && own_ms > 0.0)
      h->us_per_photon = 0.75 * h->us_per_photon + 0.25 * (own_ms * 1e3 / (double)hs.photons_started);
    h->t_last_retire = Clock::now();
  }
  int rc = push_hits(h, std::move(hits), may_block);
  if (rc != PP_OK) return rc;
  // items of this launch's resume list that no warp fetched before the ring filled up again
  const uint32_t res_consumed = std::min<uint32_t>(hs.resume_counter, s.P.n_resume_in);
  const uint32_t res_rest = s.P.n_resume_in - res_consumed;
  if (hs.n_resume_out > 0 || res_rest > 0) {
    // ---- ring filled up: relaunch for the deferred photons, the unfinished tiles and the fresh tiles ----
    Status ns{};
    ns.tile_counter = hs.tile_counter;
    *s.h_status_in = ns;
    PP_CUDA(h, cudaMemcpyAsync(s.d_status, s.h_status_in, sizeof(Status), cudaMemcpyHostToDevice, s.stream));
    LaunchParams& P = s.P;
    uint32_t n_next = std::min<uint32_t>(hs.n_resume_out, P.resume_cap);
    if (res_rest > 0) {
      // carry the unfetched items over: append them to the list the launch wrote
      if ((uint64_t)n_next + res_rest > P.resume_cap) return fail(h, PP_E_CUDA, "internal: resume list overflow");
      PP_CUDA(h, cudaMemcpyAsync(s.d_resume[s.resume_sel] + n_next, P.resume_in + res_consumed,
                                 (size_t)res_rest * sizeof(WorkItem), cudaMemcpyDeviceToDevice, s.stream));
      n_next += res_rest;
    }
    P.resume_in = s.d_resume[s.resume_sel];
    P.n_resume_in = n_next;
    s.resume_sel ^= 1;
    P.resume_out = s.d_resume[s.resume_sel];
    PP_CUDA(h, cudaEventRecord(s.ev_k0, s.stream));
    PP_CUDA(h, launch_propagate(P, h->brute, s.fates, h->grid, h->smem, s.stream));
    PP_CUDA(h, cudaEventRecord(s.ev_k1, s.stream));
    PP_CUDA(h, read_back_head(h, s));
    PP_CUDA(h, cudaEventRecord(s.ev_done, s.stream));
    std::lock_guard<std::mutex> g(h->mu);
    h->st.relaunches += 1;
    return PP_OK;  // still in flight
  }
  s.in_flight = false;
  return PP_OK;
}

// Finish a slot completely (all relaunches).
int drain_slot(pp_handle* h, Slot& s, bool may_block) {
  while (s.in_flight) {
    int rc = finish_slot(h, s, may_block);
    if (rc != PP_OK) { s.in_flight = false; return rc; }
  }
  return PP_OK;
}

// ---------------------------------------------------------------------------------------------
// a1: the batching server thread
// ---------------------------------------------------------------------------------------------

// Launch cutting (a1).  `count_at(i)` is the photon count of the i-th queued source, the first of
// which has `first_offset` photons already launched.  Takes sources until `target` photons are
// reached, splitting the last source's photon range if needed.  Pure function: also exposed for
// CPU tests through pp_debug_plan_launches().
struct Cut {
  uint64_t n_rec;       // queued sources that take part in this launch (the last may be partial)
  uint64_t g_begin;     // first photon of the launch, numbered within the launch's own prefix sum
  uint64_t g_end;       // one past the last photon
  uint64_t photons;     // g_end - g_begin
  bool last_partial;    // the last source continues in the next launch ...
  uint64_t next_offset; // ... from this photon index
};

template <class CountAt>
bool plan_cut(CountAt count_at, uint64_t n_avail, uint64_t first_offset, uint64_t target, Cut* c) {
  uint64_t acc = 0, cum_all = 0;
  c->g_begin = first_offset; c->last_partial = false; c->next_offset = 0;
  uint64_t i = 0;
  while (i < n_avail) {
    const uint64_t np = count_at(i);
    const uint64_t skip = (i == 0 ? first_offset : 0);
    const uint64_t avail = np - skip;
    if (acc + avail > target) {  // split this source across launches
      const uint64_t take = target - acc;
      c->n_rec = i + 1;
      c->g_end = cum_all + skip + take;
      c->photons = acc + take;
      c->last_partial = true;
      c->next_offset = skip + take;
      return c->photons > 0;
    }
    acc += avail; cum_all += np;
    ++i;
    if (acc == target) break;
  }
  c->n_rec = i; c->g_end = cum_all; c->photons = acc;
  return acc > 0;
}

void server_main(pp_handle* h) {
  cudaSetDevice(h->device);
  std::unique_lock<std::mutex> lk(h->mu);
  int next_slot = 0;
  for (;;) {
    if (h->sticky.load() != PP_OK) {  // poisoned: wake everybody, do nothing more
      h->cv_space.notify_all(); h->cv_hits.notify_all();
      if (h->shutdown) return;
      h->cv_work.wait_for(lk, std::chrono::milliseconds(50));
      continue;
    }
    if (h->shutdown) {  // pp_destroy: queued-but-unlaunched work is dropped, launches in flight finish
      h->ring_launch = h->ring_tail = h->ring_head; h->launch_offset = 0; h->queued_photons = 0;
    }
    bool progressed = false;
    // 1. retire finished launches (oldest first)
    for (int pass = 0; pass < 2 && !h->resident_active; ++pass) {
      Slot* oldest = nullptr;
      for (auto& s : h->slot)
        if (s.in_flight && (!oldest || s.seq < oldest->seq)) oldest = &s;
      if (!oldest) break;
      const cudaError_t q = cudaEventQuery(oldest->ev_done);
      if (q == cudaErrorNotReady) break;
      lk.unlock();
      const int rc = finish_slot(h, *oldest, true);
      lk.lock();
      if (rc != PP_OK) { oldest->in_flight = false; }
      if (!oldest->in_flight) {
        h->n_in_flight--; h->inflight_photons -= std::min(h->inflight_photons, oldest->photons); h->wall_t1 = Clock::now();
        // launches retire oldest first and their hits are queued by now: everything before sources_end is complete
        h->st.sources_completed = std::max<uint64_t>(h->st.sources_completed, oldest->sources_end);
        h->cv_hits.notify_all();
      }
      progressed = true;
    }
    // 2. launch if a slot is free and enough work is queued
    if (!h->resident_active && h->n_in_flight < 2 && h->sticky.load() == PP_OK) {
      Slot& s = h->slot[next_slot].in_flight ? h->slot[next_slot ^ 1] : h->slot[next_slot];
      Cut c{};
      // a GPU that is idle, or about to be, is fed early: while less than half a target is in flight, a launch is
      // cut as soon as an eighth of the target is queued ("to keep the GPU as busy as possible"), so a
      // job ramps up through launches of growing size instead of waiting for a full one; once enough is in flight
      // the queue fills to the target
      const bool idle_feed = h->inflight_photons < h->sz.target / 2 &&
                             h->queued_photons >= std::max<uint64_t>(1, h->sz.target / 8);
      const bool force = h->flush_upto > h->ring_launch || h->space_waiters > 0 || idle_feed;
      bool have = false;
      if (!s.in_flight) {
        if (h->queued_photons == 0) {  // nothing but zero-photon sources (or nothing at all): drop them
          h->ring_launch = h->ring_tail = h->ring_head; h->launch_offset = 0;
          if (h->n_in_flight == 0) h->st.sources_completed = std::max<uint64_t>(h->st.sources_completed, h->ring_head);
          h->cv_space.notify_all();
        } else if (h->queued_photons >= h->sz.target || force) {
          const uint64_t cap = h->sz.cap_src, base = h->ring_launch;
          const uint64_t b0 = base % cap;  // (one division, not one per record: a cut walks 2e5 records of C2)
          have = plan_cut([&](uint64_t i) { const uint64_t k = b0 + i; return (uint64_t)h->ring[k < cap ? k : k - cap].n_photons; },
                          h->ring_head - base, h->launch_offset, h->sz.target, &c);
        }
      }
      if (have) {
        const uint32_t n_src = (uint32_t)c.n_rec;
        const uint64_t rec_a = h->ring_launch;
        // bookkeeping under the lock; the records stay valid until ring_tail passes them
        h->queued_photons -= c.photons;
        if (c.last_partial) { h->ring_launch = rec_a + c.n_rec - 1; h->launch_offset = c.next_offset; }
        else { h->ring_launch = rec_a + c.n_rec; h->launch_offset = 0; }
        const bool idle_gpu = h->n_in_flight == 0;
        s.in_flight = true;  // reserve
        s.sources_end = h->ring_launch;  // a source split across launches completes with the launch that ends it
        h->n_in_flight++;
        s.photons = c.photons; h->inflight_photons += c.photons;
        lk.unlock();
        int rc = PP_OK;
        {
          const uint64_t cap = h->sz.cap_src;
          const uint64_t a = rec_a % cap;
          const uint64_t first = std::min<uint64_t>(n_src, cap - a);
          cudaError_t e = cudaMemcpyAsync(s.d_src, h->ring + a, first * sizeof(SrcRec), cudaMemcpyHostToDevice, s.stream);
          if (e == cudaSuccess && first < n_src)
            e = cudaMemcpyAsync(s.d_src + first, h->ring, (n_src - first) * sizeof(SrcRec), cudaMemcpyHostToDevice, s.stream);
          if (e == cudaSuccess) e = cudaEventRecord(s.ev_h2d, s.stream);
          if (e != cudaSuccess) rc = fail(h, PP_E_CUDA, std::string("upload: ") + cudaGetErrorString(e));
          bool seg = false;  // any track segment among the records of this launch?
          auto rec = [&](uint32_t q) -> const SrcRec& { const uint64_t k = a + q; return h->ring[k < cap ? k : k - cap]; };
          uint32_t tile = 0, n_tiles = 0;
          pick_tiles(h, c.photons, &tile, &n_tiles);
          // a small launch onto an idle GPU keeps the single prologue kernel (one launch instead of four copies:
          // 20 us of a 0.15 ms launch, C3); every other launch gets its tables from the host
          const bool host_tables = !(idle_gpu && n_src <= kPrologueMax && n_tiles <= kPrologueMax);
          if (rc == PP_OK && host_tables && n_tiles <= h->sz.max_tiles)
            host_prologue(s, [&](uint32_t q) { const SrcRec& r = rec(q); seg |= r.length > 0.0f; return (uint64_t)r.n_photons; },
                          n_src, c.g_begin, tile, n_tiles);  // (one pass over the records: sums and the segment flag)
          else
            for (uint32_t q = 0; q < n_src && !seg; ++q) seg = rec(q).length > 0.0f;
          if (rc == PP_OK)
            rc = enqueue_launch(h, s, s.d_src, s.d_cum, n_src, c.g_begin, c.g_end, nullptr, seg, true, host_tables);
          if (rc == PP_OK && cudaEventSynchronize(s.ev_h2d) != cudaSuccess) rc = fail(h, PP_E_CUDA, "upload sync failed");
        }
        lk.lock();
        if (rc != PP_OK) { s.in_flight = false; h->n_in_flight--; h->inflight_photons -= std::min(h->inflight_photons, s.photons); }
        // the uploaded records are free again (a split record stays for the next launch)
        h->ring_tail = h->ring_launch;
        h->cv_space.notify_all();
        next_slot ^= 1;
        progressed = true;
      }
    }
    if (progressed) continue;
    if (h->shutdown && h->n_in_flight == 0 && h->queued_photons == 0) return;
    if (h->n_in_flight > 0 && !h->resident_active) {
      // nothing launchable and the GPU is busy: sleep through most of the time the oldest launch should still take
      // (a running estimate of the kernel time per photon), then poll its completion event (bounded spinning, only
      // around the expected end), so that the latency of a launch is not rounded up to a sleep period (C3)
      Slot* oldest = nullptr;
      for (auto& s : h->slot)
        if (s.in_flight && (!oldest || s.seq < oldest->seq)) oldest = &s;
      bool ready = false;
      if (oldest) {
        const auto t_ref = std::max(oldest->t_enq, h->t_last_retire);
        const double elapsed = std::chrono::duration<double, std::micro>(Clock::now() - t_ref).count();
        const double left = oldest->expect_us - elapsed;
        if (left > 250.0) {
          h->cv_work.wait_for(lk, std::chrono::microseconds((long)std::min(left - 150.0, 2000.0)));
          continue;  // new sources may have arrived meanwhile
        }
        lk.unlock();
        const auto t_end = Clock::now() + std::chrono::microseconds((long)(std::max(left, 0.0) + 250.0));
        do {
          ready = cudaEventQuery(oldest->ev_done) != cudaErrorNotReady;
          if (!ready) std::this_thread::yield();
        } while (!ready && Clock::now() < t_end);
        lk.lock();
      }
      if (!ready) h->cv_work.wait_for(lk, std::chrono::microseconds(100));
    } else {
      h->cv_work.wait_for(lk, std::chrono::milliseconds(20));
    }
  }
}

void destroy_events(Slot& s) {
  for (cudaEvent_t* e : {&s.ev_h2d, &s.ev_k0, &s.ev_k1, &s.ev_done, &s.ev_stage[0], &s.ev_stage[1]})
    if (*e) { cudaEventDestroy(*e); *e = nullptr; }
}

bool idle_locked(pp_handle* h) {
  return h->n_in_flight == 0 && h->queued_photons == 0 && !h->resident_active;
}

}  // namespace

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" {

const char* pp_version(void) { return "pp 0.5 (sm_100a)"; }

int pp_check_inputs(const pp_geometry* geo, const pp_ice* ice, uint32_t flags) {
  std::string why;
  int rc = validate_inputs(geo, ice, &why);
  if (rc != PP_OK) return rc;
  HostGeometry hg;
  const bool brute = (flags & PP_FLAG_BRUTE_FORCE_DOMS) != 0;
  build_geometry(geo, brute, &hg);
  return (brute || hg.fast_ok) ? PP_OK : PP_E_UNSUPPORTED;
}

int pp_photon_count(float energy_GeV, float photons_per_GeV, uint64_t* n_out) {
  if (!n_out || !std::isfinite(energy_GeV) || !std::isfinite(photons_per_GeV) || energy_GeV < 0.0f ||
      photons_per_GeV < 0.0f)
    return PP_E_INVAL;
  const unsigned long long n = host_photon_count(energy_GeV, photons_per_GeV);
  *n_out = n;
  return n > 0xFFFFFFFFull ? PP_E_OVERFLOW : PP_OK;
}

int pp_debug_plan_launches(const uint32_t* photon_counts, size_t n, uint64_t target, pp_launch_plan* out, size_t cap,
                           size_t* n_out) {
  if ((!photon_counts && n) || !n_out || (!out && cap) || target == 0) return PP_E_INVAL;
  size_t k = 0;
  uint64_t first = 0, offset = 0;
  while (first < n) {
    Cut c{};
    const bool ok = plan_cut([&](uint64_t i) { return (uint64_t)photon_counts[first + i]; }, n - first, offset, target, &c);
    if (!ok) break;  // only zero-photon sources are left
    if (k < cap) out[k] = pp_launch_plan{first, c.n_rec, c.g_begin, c.g_end};
    ++k;
    if (c.last_partial) { first += c.n_rec - 1; offset = c.next_offset; }
    else { first += c.n_rec; offset = 0; }
  }
  *n_out = k;
  return k > cap ? PP_E_NOMEM : PP_OK;
}
uint64_t pp_kernel_launch_count(void) { return kernel_launch_count(); }

int pp_workspace_size(const pp_geometry* geo, const pp_ice* ice, const pp_config* cfg, uint64_t* device_bytes,
                      uint64_t* pinned_bytes) {
  std::string why;
  if (!cfg) return PP_E_INVAL;
  int rc = validate_inputs(geo, ice, &why);
  if (rc != PP_OK) return rc;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PP_E_CUDA;
  if (cfg->device > 0 || (cfg->device == 0 && (cfg->flags & PP_FLAG_DEVICE_ORDINAL))) dev = cfg->device;
  int n_sm = 0;
  if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PP_E_CUDA;
  pp_handle tmp;
  tmp.cfg = *cfg; tmp.ice = *ice;
  tmp.brute = (cfg->flags & PP_FLAG_BRUTE_FORCE_DOMS) != 0;
  build_geometry(geo, tmp.brute, &tmp.hg);
  if (!tmp.brute && !tmp.hg.fast_ok) return PP_E_UNSUPPORTED;
  fill_sizes(*cfg, n_sm, &tmp.sz);
  rc = build_tables(&tmp, geo, ice, cfg);
  if (rc != PP_OK) return rc;
  if (device_bytes) *device_bytes = carve_device(&tmp, nullptr);
  if (pinned_bytes) *pinned_bytes = carve_pinned(&tmp, nullptr);
  return PP_OK;
}

int pp_create(const pp_geometry* geo, const pp_ice* ice, const pp_config* cfg, pp_handle** out) {
  if (!out || !cfg) return PP_E_INVAL;
  *out = nullptr;
  std::string why;
  int rc = validate_inputs(geo, ice, &why);
  if (rc != PP_OK) return rc;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) return PP_E_CUDA;  // no CPU fallback
  auto* h = new pp_handle();
  h->cfg = *cfg;
  h->ice = *ice;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { delete h; return PP_E_CUDA; }
  const int callers_dev = dev;  // made current again before pp_create returns, whatever the outcome
  if (cfg->device > 0 || (cfg->device == 0 && (cfg->flags & PP_FLAG_DEVICE_ORDINAL))) dev = cfg->device;
  h->device = dev;
  auto bail = [&](int code) { pp_destroy(h); cudaSetDevice(callers_dev); return code; };
  if (cudaSetDevice(dev) != cudaSuccess) return bail(PP_E_CUDA);
  if (cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return bail(PP_E_CUDA);
  h->brute = (cfg->flags & PP_FLAG_BRUTE_FORCE_DOMS) != 0;
  build_geometry(geo, h->brute, &h->hg);
  if (!h->brute && !h->hg.fast_ok) return bail(PP_E_UNSUPPORTED);
  fill_sizes(*cfg, h->n_sm, &h->sz);
  rc = build_tables(h, geo, ice, cfg);
  if (rc != PP_OK) return bail(rc);
  h->hitq_budget = 1ull << 30;

  // ---- workspaces ----
  const uint64_t need_dev = carve_device(h, nullptr), need_pin = carve_pinned(h, nullptr);
  if (cfg->device_workspace) {
    if (cfg->device_workspace_bytes < need_dev) return bail(PP_E_NOMEM);
    h->dev_ws = cfg->device_workspace;
  } else {
    if (cudaMalloc(&h->dev_ws, need_dev) != cudaSuccess) return bail(PP_E_NOMEM);
    h->own_dev = true;
  }
  if (cfg->pinned_workspace) {
    if (cfg->pinned_workspace_bytes < need_pin) return bail(PP_E_NOMEM);
    h->pin_ws = cfg->pinned_workspace;
  } else {
    if (cudaHostAlloc(&h->pin_ws, need_pin, cudaHostAllocDefault) != cudaSuccess) return bail(PP_E_NOMEM);
    h->own_pin = true;
  }
  carve_device(h, h->dev_ws);
  carve_pinned(h, h->pin_ws);
#ifdef PP_GUARD
  for (unsigned char* z : h->guard_zones)
    if (cudaMemset(z, kGuardByte, kGuardBytes) != cudaSuccess) return bail(PP_E_CUDA);
#endif
  if (cfg->stream0 && cfg->stream1) {
    h->slot[0].stream = (cudaStream_t)cfg->stream0;
    h->slot[1].stream = (cudaStream_t)cfg->stream1;
  } else {
    h->own_streams = true;
    for (auto& s : h->slot)
      if (cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking) != cudaSuccess) return bail(PP_E_CUDA);
  }
  for (auto& s : h->slot) {
    for (cudaEvent_t* e : {&s.ev_h2d, &s.ev_k0, &s.ev_k1, &s.ev_done, &s.ev_stage[0], &s.ev_stage[1]})
      if (cudaEventCreate(e) != cudaSuccess) return bail(PP_E_CUDA);
  }
  if (cudaEventCreate(&h->ev_base) != cudaSuccess || cudaEventCreate(&h->ev_job) != cudaSuccess) return bail(PP_E_CUDA);

  // ---- tables and constants to the device ----
  LaunchParams& B = h->base;
  auto up = [&](const void* dst, const void* src, size_t bytes) {
    return bytes == 0 || cudaMemcpy(const_cast<void*>(dst), src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  if (!up(B.smem_image, h->image.data(), h->image.size()) ||
      !up(B.dom_xyzw, h->hg.dom_xyzw.data(), h->hg.dom_xyzw.size() * sizeof(float4)))
    return bail(PP_E_CUDA);

  // ---- persistent grid: every SM filled to the kernel's occupancy ----
  {
    // make the opt-in dynamic shared memory size known before asking for the occupancy
    int bps = 0;
    // a zero-work launch sets the function attribute (launch_propagate does it on first use)
    Status zero{};
    if (cudaMemcpy(h->slot[0].d_status, &zero, sizeof(zero), cudaMemcpyHostToDevice) != cudaSuccess) return bail(PP_E_CUDA);
    LaunchParams P = B;
    P.status = h->slot[0].d_status; P.n_tiles = 0; P.g_begin = P.g_end = 0; P.n_resume_in = 0;
    P.resume_out = h->slot[0].d_resume[0]; P.resume_in = h->slot[0].d_resume[1]; P.resume_cap = (uint32_t)h->sz.resume_cap;
    P.ring = h->slot[0].d_ring; P.ring_cap = (uint32_t)h->sz.ring_cap; P.src = h->slot[0].d_src; P.cum = h->slot[0].d_cum;
    P.tile_src = h->slot[0].d_tile_src; P.cum_rel = h->slot[0].d_cum_rel;
    for (int f = 0; f < 6; ++f) {  // every kernel variant this handle can launch: fates x flight-loop physics
      P.spec_n = (f >> 1) == 1 ? 1u : 0u;   // wavelength bins only
      P.emit_on = (f >> 1) == 2 ? 1u : 0u;  // (any of the other switches selects the same, fullest variant)
      if (launch_propagate(P, h->brute, (f & 1) != 0, 1, h->smem, h->slot[0].stream) != cudaSuccess) return bail(PP_E_CUDA);
    }
    if (cudaStreamSynchronize(h->slot[0].stream) != cudaSuccess) return bail(PP_E_CUDA);
    if (propagate_occupancy(h->brute, false, h->smem, &bps) != cudaSuccess || bps < 1) return bail(PP_E_CUDA);
    h->grid = h->n_sm * bps;
  }
  if (cudaEventRecord(h->ev_base, h->slot[0].stream) != cudaSuccess) return bail(PP_E_CUDA);
  if (cudaEventSynchronize(h->ev_base) != cudaSuccess) return bail(PP_E_CUDA);
  h->server = std::thread(server_main, h);
  if (callers_dev != dev) cudaSetDevice(callers_dev);
  *out = h;
  return PP_OK;
}

int pp_submit(pp_handle* h, const pp_source* src, const uint32_t* event_ids, const uint32_t* source_ids, size_t n) {
  return pp_submit_segments(h, src, nullptr, event_ids, source_ids, n);
}

}  // extern "C"

namespace {
// One light source as the submit path sees it, whatever the caller's layout.
struct SrcView { const pp_source* s; float length; uint32_t event_id; bool has_id; uint32_t source_id; };

// pp_submit / pp_submit_segments / pp_submit_packed: `at(i)` is the i-th source of the call.
template <class At>
int submit_generic(pp_handle* h, size_t n, At at, uint64_t* records_end = nullptr) {
  const float yield = h->ice.photons_per_GeV;
  const uint64_t cap = h->sz.cap_src;
  // the checks of one source, branch-free: non-zero = bad; also gives its photon count
  auto check = [&](const SrcView& v, uint32_t* count) -> uint32_t {
    const pp_source& a = *v.s;
    uint32_t w[8];
    std::memcpy(w, &a, sizeof w);  // x, y, z, dx, dy, dz, t, E
    uint32_t nonfinite = 0;
    for (int q = 0; q < 8; ++q) nonfinite |= (uint32_t)((w[q] & 0x7f800000u) == 0x7f800000u);
    const double n2 = (double)a.dx * a.dx + (double)a.dy * a.dy + (double)a.dz * a.dz;
    const unsigned long long cnt = host_photon_count(a.energy_GeV, yield);
    *count = (uint32_t)cnt;
    return nonfinite | (uint32_t)(std::fabs(n2 - 1.0) > 1e-4) | (uint32_t)(a.energy_GeV < 0.0f) |
           (uint32_t)!(v.length >= 0.0f && v.length <= 3.0e38f) | (uint32_t)(cnt > 0xFFFFFFFFull);
  };
  // the slow pass that names the offender (runs only if there is one)
  auto name_offender = [&]() -> int {
    for (size_t i = 0; i < n; ++i) {
      const SrcView v = at(i);
      const pp_source& a = *v.s;
      const float f8[8] = {a.x, a.y, a.z, a.dx, a.dy, a.dz, a.t_ns, a.energy_GeV};
      for (float f : f8)
        if (!std::isfinite(f)) return fail(h, PP_E_INVAL, "non-finite field in source " + std::to_string(i));
      const double n2 = (double)a.dx * a.dx + (double)a.dy * a.dy + (double)a.dz * a.dz;
      if (std::fabs(n2 - 1.0) > 1e-4) return fail(h, PP_E_INVAL, "source direction is not a unit vector");
      if (a.energy_GeV < 0.0f) return fail(h, PP_E_INVAL, "negative source energy");
      if (!(std::isfinite(v.length) && v.length >= 0.0f)) return fail(h, PP_E_INVAL, "bad source length");
      if (host_photon_count(a.energy_GeV, yield) > 0xFFFFFFFFull)
        return fail(h, PP_E_OVERFLOW, "source " + std::to_string(i) + " has more than 2^32-1 photons");
    }
    return fail(h, PP_E_INVAL, "bad source");
  };
  auto write_rec = [&](uint64_t p0, size_t j, const SrcView& v, uint32_t count, uint64_t auto_id) {
    const pp_source& a = *v.s;
    const uint64_t kk = p0 + j;
    SrcRec& r = h->ring[kk < cap ? kk : kk - cap];
    r.x = a.x; r.y = a.y; r.z = a.z; r.dx = a.dx; r.dy = a.dy; r.dz = a.dz; r.t = a.t_ns; r.energy = a.energy_GeV;
    r.event_id = v.event_id;
    r.source_id = v.has_id ? v.source_id : (uint32_t)(auto_id + j);  // running record number
    r.n_photons = count;
    r.length = v.length;
  };
  auto publish = [&](std::unique_lock<std::mutex>& lk, uint64_t pos, size_t m, uint64_t ph) {  // lk held
    h->cv_pub.wait(lk, [&] { return h->ring_head == pos; });  // earlier reservations publish first
    h->ring_head = pos + m;
    h->cv_pub.notify_all();
    h->queued_photons += ph;
    h->st.sources_submitted += m;
    h->st.photons_submitted += ph;
    h->st.source_ring_high_water =
        std::max<uint64_t>(h->st.source_ring_high_water, (h->ring_reserve - h->ring_tail) * sizeof(SrcRec));
    if (h->queued_photons >= h->sz.target ||
        (h->inflight_photons < h->sz.target / 2 && h->queued_photons >= std::max<uint64_t>(1, h->sz.target / 8)))
      h->cv_work.notify_all();
  };
  // Everything is validated before anything is enqueued.
  // Fast path: the whole call fits into the ring right now.  ONE pass checks, counts and copies into reserved slots
  // that nobody can see yet (the multi-process front end pushes 4e7 sources/s through here); a bad source takes the
  // reservation back (always possible for a lone producer such as that front end; if other producers have reserved
  // behind it meanwhile, the slots are published as sources without photons, which the server drops).
  {
    std::unique_lock<std::mutex> lk(h->mu);
    if (h->shutdown.load()) return PP_E_STATE;
    if ((h->sz.cap_src - (h->ring_reserve - h->ring_tail)) >= n) {
      if (!h->wall_started) { h->wall_started = true; h->wall_t0 = Clock::now(); h->wall_t1 = h->wall_t0; }
      const uint64_t pos = h->ring_reserve, auto_id = h->next_auto_id, p0 = pos % cap;
      h->ring_reserve += n;
      h->next_auto_id += n;
      lk.unlock();
      uint32_t bad = 0;
      uint64_t ph = 0;
      for (size_t j = 0; j < n; ++j) {
        const SrcView v = at(j);
        uint32_t cnt;
        bad |= check(v, &cnt);
        write_rec(p0, j, v, cnt, auto_id);
        ph += cnt;
      }
      if (bad) {
        for (size_t j = 0; j < n; ++j) { const uint64_t kk = p0 + j; h->ring[kk < cap ? kk : kk - cap].n_photons = 0u; }
        ph = 0;
      }
      lk.lock();
      if (bad && h->ring_reserve == pos + n) {
        h->ring_reserve = pos; h->next_auto_id = auto_id;  // nobody reserved behind us: as if nothing had happened
        lk.unlock();
        return name_offender();
      }
      publish(lk, pos, n, ph);
      if (bad) { lk.unlock(); return name_offender(); }
      if (records_end) *records_end = pos + n;
      return PP_OK;
    }
  }
  // General path (the call does not fit into the ring at once): a checking pass that keeps the photon counts, then
  // the copy in as many pieces as the ring has room for.
  thread_local std::vector<uint32_t> counts;
  if (counts.size() < n) counts.resize(n);
  {
    uint32_t bad = 0;
    for (size_t i = 0; i < n; ++i) bad |= check(at(i), &counts[i]);
    if (bad) return name_offender();
  }
  const bool nonblock = (h->cfg.flags & PP_FLAG_NONBLOCKING_SUBMIT) != 0;
  size_t i = 0;
  std::unique_lock<std::mutex> lk(h->mu);
  if (h->shutdown.load()) return PP_E_STATE;
  if (!h->wall_started) { h->wall_started = true; h->wall_t0 = Clock::now(); h->wall_t1 = h->wall_t0; }
  if (nonblock) {
    if (n > h->sz.cap_src) return fail(h, PP_E_NOMEM, "batch larger than the source ring");
    if (h->sz.cap_src - (h->ring_reserve - h->ring_tail) < n) { h->cv_work.notify_all(); return PP_E_WOULDBLOCK; }
  }
  while (i < n) {
    const uint64_t space = h->sz.cap_src - (h->ring_reserve - h->ring_tail);
    if (space == 0) {
      h->space_waiters++;
      h->cv_work.notify_all();
      h->cv_space.wait(lk, [&] { return h->sz.cap_src - (h->ring_reserve - h->ring_tail) > 0 || h->shutdown.load() ||
                                        h->sticky.load() != PP_OK; });
      h->space_waiters--;
      if (h->shutdown.load()) return PP_E_STATE;
      if (h->sticky.load() != PP_OK) return h->sticky.load();
      continue;
    }
    // reserve under the lock, copy outside it, publish in order: producers fill the ring in parallel and the server
    // thread never waits for a copy
    const size_t m = (size_t)std::min<uint64_t>(space, n - i);
    const uint64_t pos = h->ring_reserve, auto_id = h->next_auto_id;
    h->ring_reserve += m;
    h->next_auto_id += m;
    lk.unlock();
    uint64_t ph = 0;
    const uint64_t p0 = pos % cap;
    for (size_t j = 0; j < m; ++j, ++i) {
      write_rec(p0, j, at(i), counts[i], auto_id);
      ph += counts[i];
    }
    lk.lock();
    publish(lk, pos, m, ph);
    if (records_end) *records_end = pos + m;
  }
  return PP_OK;
}
}  // namespace

extern "C" {

int pp_submit_segments(pp_handle* h, const pp_source* src, const float* lengths, const uint32_t* event_ids,
                       const uint32_t* source_ids, size_t n) {
  if (!h) return PP_E_INVAL;
  if (h->sticky.load() != PP_OK) return h->sticky.load();
  if (n == 0) return PP_OK;
  if (!src || !event_ids) return fail(h, PP_E_INVAL, "null sources or event_ids");
  return submit_generic(h, n, [&](size_t i) {
    return SrcView{src + i, lengths ? lengths[i] : 0.0f, event_ids[i], source_ids != nullptr, source_ids ? source_ids[i] : 0u};
  });
}

int pp_submit_packed(pp_handle* h, const pp_packed_source* recs, size_t n, uint64_t* records_end) {
  if (!h) return PP_E_INVAL;
  if (h->sticky.load() != PP_OK) return h->sticky.load();
  if (n == 0) {
    if (records_end) { std::lock_guard<std::mutex> g(h->mu); *records_end = h->ring_reserve; }
    return PP_OK;
  }
  if (!recs) return fail(h, PP_E_INVAL, "null records");
  return submit_generic(h, n, [&](size_t i) {
    return SrcView{&recs[i].s, recs[i].length_m, recs[i].event_id, true, recs[i].source_id};
  }, records_end);
}

int pp_flush(pp_handle* h) {
  if (!h) return PP_E_INVAL;
  if (h->sticky.load() != PP_OK) return h->sticky.load();
  std::lock_guard<std::mutex> g(h->mu);
  h->flush_upto = h->ring_head;
  h->cv_work.notify_all();
  return PP_OK;
}

int pp_collect(pp_handle* h, pp_hit* out, size_t cap, size_t* n_out, int block) {
  if (!h || !n_out || (!out && cap)) return PP_E_INVAL;
  *n_out = 0;
  // a blocking caller first polls for a short while (a small launch is back within ~0.1 ms, less than a sleep and
  // wake-up costs), then sleeps on the condition variable
  const auto spin_until = Clock::now() + std::chrono::microseconds(200);
  for (;;) {
    {
      std::unique_lock<std::mutex> lk(h->hit_mu);
      size_t got = 0;
      while (got < cap && !h->hitq.empty()) {
        auto& v = h->hitq.front();
        const size_t m = std::min(cap - got, v.size() - h->hitq_front_off);
        std::memcpy(out + got, v.data() + h->hitq_front_off, m * sizeof(pp_hit));
        got += m;
        h->hitq_front_off += m;
        if (h->hitq_front_off == v.size()) {
          h->hitq_bytes -= v.size() * sizeof(pp_hit);
          h->hitq.pop_front();
          h->hitq_front_off = 0;
        }
      }
      if (got) {
        *n_out = got;
        h->hits_collected += got;
        h->cv_hit_space.notify_all();
        return PP_OK;
      }
    }
    if (h->sticky.load() != PP_OK) return h->sticky.load();
    if (!block || cap == 0) return PP_OK;
    bool idle;
    {
      std::lock_guard<std::mutex> g(h->mu);
      idle = idle_locked(h) && h->ring_launch == h->ring_reserve;
    }
    std::unique_lock<std::mutex> lk(h->hit_mu);
    if (!h->hitq.empty()) continue;
    // a launch's hits are queued before the launch is retired, so "idle" seen first and the queue still empty now
    // means drained
    if (idle) return PP_OK;
    if (Clock::now() < spin_until) { lk.unlock(); std::this_thread::yield(); continue; }
    h->cv_hits.wait_for(lk, std::chrono::milliseconds(5));
  }
}

int pp_set_acceptance(pp_handle* h, uint32_t mode, const float* coef, uint32_t n_coef) {
  if (!h) return PP_E_INVAL;
  if (mode > PP_ACCEPT_WEIGHTED) return fail(h, PP_E_INVAL, "pp_set_acceptance: unknown mode");
  if (mode != PP_ACCEPT_OFF) {
    if (!coef || n_coef == 0 || n_coef > PP_MAX_ACCEPT_COEF) return fail(h, PP_E_INVAL, "pp_set_acceptance: n_coef out of range");
    for (uint32_t k = 0; k < n_coef; ++k)
      if (!finite_f(coef[k])) return fail(h, PP_E_INVAL, "pp_set_acceptance: non-finite coefficient");
  }
  std::lock_guard<std::mutex> g(h->mu);
  if (!idle_locked(h)) return PP_E_STATE;
  h->base.acc_mode = mode;
  h->base.acc_n = mode == PP_ACCEPT_OFF ? 0u : n_coef;
  for (uint32_t k = 0; k < PP_MAX_ACCEPT_COEF; ++k) h->base.acc_coef[k] = (mode != PP_ACCEPT_OFF && k < n_coef) ? coef[k] : 0.0f;
  return PP_OK;
}

int pp_set_spectrum(pp_handle* h, uint32_t n_bins, const float* cdf, const float* abs_scale, const float* scat_scale,
                    const float* n_group, const float* acc_scale) {
  if (!h) return PP_E_INVAL;
  if (n_bins > PP_MAX_SPECTRUM_BINS) return fail(h, PP_E_INVAL, "pp_set_spectrum: too many bins");
  if (n_bins && (!cdf || !abs_scale || !scat_scale || !n_group || !acc_scale)) return fail(h, PP_E_INVAL, "pp_set_spectrum: null array");
  for (uint32_t j = 0; j < n_bins; ++j) {
    const bool ok = finite_f(cdf[j]) && cdf[j] > 0.0f && cdf[j] <= 1.0f && (j == 0 || cdf[j] >= cdf[j - 1]) &&
                    finite_f(abs_scale[j]) && abs_scale[j] > 0.0f && finite_f(scat_scale[j]) && scat_scale[j] > 0.0f &&
                    finite_f(n_group[j]) && n_group[j] >= 1.0f && finite_f(acc_scale[j]) && acc_scale[j] >= 0.0f;
    if (!ok) return fail(h, PP_E_INVAL, "pp_set_spectrum: bad value in bin " + std::to_string(j));
  }
  std::lock_guard<std::mutex> g(h->mu);
  if (!idle_locked(h)) return PP_E_STATE;
  LaunchParams& B = h->base;
  B.spec_n = n_bins;
  for (uint32_t j = 0; j < PP_MAX_SPECTRUM_BINS; ++j) {
    const bool in = j < n_bins;
    B.spec_cdf[j] = in ? cdf[j] : 2.0f;
    B.spec_inv_a[j] = in ? (float)(1.0 / (double)abs_scale[j]) : 1.0f;
    B.spec_inv_b[j] = in ? (float)(1.0 / (double)scat_scale[j]) : 1.0f;
    B.spec_acc[j] = in ? acc_scale[j] : 1.0f;
    B.spec_inv_v[j] = in ? (double)n_group[j] / kC : B.inv_v;
  }
  return PP_OK;
}

int pp_set_emission_smearing(pp_handle* h, float g_axis) {
  if (!h) return PP_E_INVAL;
  if (!finite_f(g_axis) || !(g_axis > -1.0f && g_axis <= 1.0f) || g_axis == 0.0f)
    return fail(h, PP_E_INVAL, "pp_set_emission_smearing: g_axis must be in (-1, 1] and not 0");
  std::lock_guard<std::mutex> g(h->mu);
  if (!idle_locked(h)) return PP_E_STATE;
  const double ga = g_axis;
  h->base.emit_on = g_axis < 1.0f ? 1u : 0u;
  h->base.emit_one_minus_g = (float)(1.0 - ga); h->base.emit_two_g = (float)(2.0 * ga);
  h->base.emit_one_minus_g2 = (float)(1.0 - ga * ga);
  return PP_OK;
}

int pp_set_segment_profile(pp_handle* h, uint32_t n_knots, const float* cum_fraction) {
  if (!h) return PP_E_INVAL;
  if (n_knots == 1 || n_knots > PP_MAX_PROFILE_KNOTS || (n_knots && !cum_fraction))
    return fail(h, PP_E_INVAL, "pp_set_segment_profile: n_knots must be 0 or 2..33");
  for (uint32_t i = 0; i < n_knots; ++i)
    if (!finite_f(cum_fraction[i]) || cum_fraction[i] < 0.0f || cum_fraction[i] > 1.0f ||
        (i > 0 && cum_fraction[i] < cum_fraction[i - 1]))
      return fail(h, PP_E_INVAL, "pp_set_segment_profile: table must be non-decreasing in [0, 1]");
  std::lock_guard<std::mutex> g(h->mu);
  if (!idle_locked(h)) return PP_E_STATE;
  h->base.seg_n = n_knots;
  for (uint32_t i = 0; i < PP_MAX_PROFILE_KNOTS; ++i) h->base.seg_tab[i] = i < n_knots ? cum_fraction[i] : 1.0f;
  return PP_OK;
}

int pp_stats(pp_handle* h, pp_stats_t* out) {
  if (!h || !out) return PP_E_INVAL;
  {
    std::lock_guard<std::mutex> g(h->mu);
    *out = h->st;
    if (h->wall_started) out->wall_ms = std::chrono::duration<double, std::milli>(h->wall_t1 - h->wall_t0).count();
  }
  std::lock_guard<std::mutex> g(h->hit_mu);
  out->hits_collected = h->hits_collected;
  out->hit_ring_high_water = h->hit_high_water;
  return PP_OK;
}

const char* pp_last_error(pp_handle* h) {
  if (!h) return "null handle";
  std::lock_guard<std::mutex> g(h->err_mu);
  return h->err.c_str();
}

void pp_destroy(pp_handle* h) {
  if (!h) return;
  {
    std::lock_guard<std::mutex> g(h->mu);
    h->shutdown.store(true);
    h->cv_work.notify_all(); h->cv_space.notify_all(); h->cv_pub.notify_all();
  }
  {
    std::lock_guard<std::mutex> g(h->hit_mu);
    h->cv_hits.notify_all(); h->cv_hit_space.notify_all();
  }
  if (h->server.joinable()) h->server.join();
  cudaSetDevice(h->device);
  for (auto& s : h->slot) {
    if (s.stream) cudaStreamSynchronize(s.stream);
    destroy_events(s);
    if (h->own_streams && s.stream) cudaStreamDestroy(s.stream);
  }
  if (h->ev_base) cudaEventDestroy(h->ev_base);
  if (h->ev_job) cudaEventDestroy(h->ev_job);
  if (h->own_dev && h->dev_ws) cudaFree(h->dev_ws);
  if (h->own_pin && h->pin_ws) cudaFreeHost(h->pin_ws);
  delete h;
}

int pp_run_resident(pp_handle* h, const pp_source* d_sources, const uint32_t* d_event_ids, const uint32_t* d_source_ids,
                    size_t n, pp_fate* d_fates, uint64_t* photons_out, double* device_ms_out) {
  if (!h) return PP_E_INVAL;
  if (h->sticky.load() != PP_OK) return h->sticky.load();
  if (photons_out) *photons_out = 0;
  if (device_ms_out) *device_ms_out = 0.0;
  if (n == 0) return PP_OK;
  if (!d_sources || !d_event_ids) return fail(h, PP_E_INVAL, "null device pointer");
  if (n > h->sz.cap_src) return fail(h, PP_E_NOMEM, "more sources than the source ring holds; raise source_ring_bytes");
  uint32_t sid_base = 0;  // source ids when d_source_ids is NULL: the handle's running record number
  {
    std::unique_lock<std::mutex> lk(h->mu);
    if (h->shutdown) return PP_E_STATE;
    if (!idle_locked(h) || h->ring_launch != h->ring_reserve)
      return fail(h, PP_E_STATE, "pp_run_resident needs an idle server (flush and collect first)");
    h->resident_active = true;
    sid_base = (uint32_t)h->next_auto_id;
    h->next_auto_id += n;
    if (!h->wall_started) { h->wall_started = true; h->wall_t0 = Clock::now(); h->wall_t1 = h->wall_t0; }
  }
  auto leave = [&](int rc) {
    std::lock_guard<std::mutex> g(h->mu);
    h->resident_active = false;
    h->wall_t1 = Clock::now();
    h->cv_hits.notify_all();
    return rc;
  };
  cudaSetDevice(h->device);
  Slot& s0 = h->slot[0];
  cudaStream_t st = s0.stream;
  // ---- a2: ingest + count + scan, once for the whole resident batch ----
  cudaError_t e = cudaEventRecord(h->ev_job, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(h->d_res_overflow, 0, sizeof(unsigned int), st);
  if (e == cudaSuccess)
    e = launch_ingest(d_sources, d_event_ids, d_source_ids, sid_base, (uint32_t)n, h->ice.photons_per_GeV, h->d_res_src,
                      h->d_res_overflow, st);
  if (e == cudaSuccess) e = launch_scan(h->d_res_src, (uint32_t)n, h->d_res_cum, st);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(h->h_res_total, h->d_res_cum + n, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(h->h_res_overflow, h->d_res_overflow, sizeof(unsigned int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaEventRecord(s0.ev_h2d, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return leave(fail(h, PP_E_CUDA, std::string("expansion: ") + cudaGetErrorString(e)));
  if (*h->h_res_overflow) return leave(fail(h, PP_E_OVERFLOW, "a source has more than 2^32-1 photons"));
  const uint64_t total = *h->h_res_total;
  {
    std::lock_guard<std::mutex> g(h->mu);
    h->st.sources_submitted += n;
    h->st.photons_submitted += total;
  }
  // the second stream must see the expansion results
  if (cudaStreamWaitEvent(h->slot[1].stream, s0.ev_h2d, 0) != cudaSuccess) return leave(fail(h, PP_E_CUDA, "wait event"));
  // ---- launches of at most `target` photons, alternating between the two slots ----
  int rc = PP_OK;
  int which = 0;
  for (uint64_t g0 = 0; g0 < total && rc == PP_OK; g0 += h->sz.target) {
    Slot& s = h->slot[which];
    rc = drain_slot(h, s, false);
    if (rc != PP_OK) break;
    const uint64_t g1 = std::min(total, g0 + h->sz.target);
    rc = enqueue_launch(h, s, h->d_res_src, h->d_res_cum, (uint32_t)n, g0, g1, d_fates, false, false);
    which ^= 1;
  }
  // retire in launch order
  for (int pass = 0; pass < 2; ++pass) {
    Slot& s = h->slot[which];
    const int r2 = drain_slot(h, s, false);
    if (rc == PP_OK) rc = r2;
    which ^= 1;
  }
  if (rc == PP_OK) {
    float ms0 = 0, ms1 = 0;
    cudaEventElapsedTime(&ms0, h->ev_job, h->slot[0].ev_done);
    if (total > h->sz.target) cudaEventElapsedTime(&ms1, h->ev_job, h->slot[1].ev_done);
    if (device_ms_out) *device_ms_out = std::max(ms0, ms1);
    if (photons_out) *photons_out = total;
  }
  return leave(rc);
}

}  // extern "C"

// What the entry point without allocations (pp_run_resident_noalloc, pp_kernels.cu) reads from a handle.
namespace pp {

int handle_launch_info(pp_handle* h, HandleLaunchInfo* out) {
  if (!h || !out) return PP_E_INVAL;
  if (h->sticky.load() != PP_OK) return h->sticky.load();
  std::lock_guard<std::mutex> g(h->mu);  // (pp_set_* write the template under this lock)
  if (h->shutdown) return PP_E_STATE;
  out->base = h->base;
  out->device = h->device; out->grid = h->grid; out->smem = h->smem; out->brute = h->brute;
  out->photons_per_GeV = h->ice.photons_per_GeV;
  return PP_OK;
}

int handle_fail(pp_handle* h, int code, const char* msg) { return fail(h, code, msg ? msg : ""); }

}  // namespace pp

#ifdef PP_GUARD
// guard build only: how many guard zones have been read back and found intact so far in this process
extern "C" uint64_t pp_guard_zone_checks(void) { return g_guard_zone_checks.load(); }
#endif
