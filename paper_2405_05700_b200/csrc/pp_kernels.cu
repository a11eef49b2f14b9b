// CUDA kernels of the photon propagator (sm_100a): source expansion (a2) and the persistent
// propagation kernel (a3-a8).  See DESIGN.md sections 2 and 5.  Product code: shares nothing with oracle/.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/pp.h"
#include "pp_internal.h"
#include "pp_device.cuh"
#include "pp_guard.cuh"

#ifndef PP_MIN_BLOCKS
#define PP_MIN_BLOCKS 1  // resident CTAs per SM the propagation kernel is compiled for (one CTA of 1024 threads)
#endif

namespace pp {

static_assert(sizeof(SrcRec) == 48, "SrcRec layout");
static_assert(sizeof(pp_hit) == 32, "pp_hit layout");
static_assert(sizeof(pp_fate) == 40, "pp_fate layout");
static_assert(sizeof(WorkItem) == 24, "WorkItem layout");
static_assert(sizeof(LayerRec) == 32, "LayerRec layout");

// =============================================================================================
// a2  Source expansion
// =============================================================================================

// Step 1 (R-12b): N = floor(double(E) * double(yield) + 0.5); exact in fp64 for fp32 inputs with
// N < 2^32, so host and device agree bit for bit.  Returns 2^32 or more on overflow.
__host__ __device__ inline unsigned long long photon_count(float energy, float yield) {
  const double n = floor((double)energy * (double)yield + 0.5);
  if (!(n > 0.0)) return 0ull;
  if (n >= 1.8e19) return ~0ull;
  return (unsigned long long)n;
}

// Resident path only: build SrcRec[] from the caller's device arrays and count photons.
__global__ void ingest_kernel(const pp_source* __restrict__ s, const uint32_t* __restrict__ ev,
                              const uint32_t* __restrict__ sid, uint32_t sid_base, uint32_t n, float yield,
                              SrcRec* __restrict__ out,
                              unsigned int* __restrict__ overflow) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const pp_source a = s[i];
  unsigned long long cnt = photon_count(a.energy_GeV, yield);
  if (cnt > 0xFFFFFFFFull) { atomicExch(overflow, 1u); cnt = 0; }
  SrcRec r;
  r.x = a.x; r.y = a.y; r.z = a.z; r.dx = a.dx; r.dy = a.dy; r.dz = a.dz; r.t = a.t_ns; r.energy = a.energy_GeV;
  r.event_id = ev[i]; r.source_id = sid ? sid[i] : sid_base + i; r.n_photons = (uint32_t)cnt; r.length = 0.0f;
  out[i] = r;
}

// Exclusive prefix sum of n_photons into cum[0..n] (64-bit).  One CTA of 1024 threads; each
// thread owns a contiguous chunk.  n is at most a few 1e5-1e6 per launch, so one CTA suffices
// (the scan is ~1e-4 of a launch).
__global__ void __launch_bounds__(1024) scan_kernel(const SrcRec* __restrict__ src, uint32_t n,
                                                    unsigned long long* __restrict__ cum) {
  __shared__ unsigned long long part[1024];
  const uint32_t t = threadIdx.x;
  const uint32_t per = (n + 1023u) / 1024u;
  const uint32_t lo = min(n, t * per), hi = min(n, lo + per);
  unsigned long long s = 0;
  for (uint32_t i = lo; i < hi; ++i) s += src[i].n_photons;
  part[t] = s;
  __syncthreads();
  // Hillis-Steele inclusive scan over the 1024 partials
  for (uint32_t off = 1; off < 1024; off <<= 1) {
    unsigned long long v = (t >= off) ? part[t - off] : 0ull;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  unsigned long long run = (t == 0) ? 0ull : part[t - 1];
  for (uint32_t i = lo; i < hi; ++i) {
    cum[i] = run;
    run += src[i].n_photons;
  }
  if (t == 1023) cum[n] = part[1023];
}

// tile_src[j] = index of the source that holds batch-global photon g_begin + j * tile_photons,
// i.e. the last s with cum[s] <= g (sources with zero photons are skipped by construction); and
// cum_rel[s] = cum[s] - g_begin in 32 bits for the refill (see LaunchParams::cum_rel).
__device__ __forceinline__ void tile_entry(const unsigned long long* __restrict__ cum, uint32_t n_src,
                                           unsigned long long g_begin, uint32_t tile_photons, uint32_t j,
                                           uint32_t* __restrict__ tile_src) {
  const unsigned long long g = g_begin + (unsigned long long)j * tile_photons;
  uint32_t lo = 0, hi = n_src;  // invariant: cum[lo] <= g < cum[hi]
  while (hi - lo > 1) {
    const uint32_t mid = (lo + hi) >> 1;
    if (cum[mid] <= g) lo = mid; else hi = mid;
  }
  tile_src[j] = lo;
}
__device__ __forceinline__ uint32_t rel32(unsigned long long c, unsigned long long g_begin) {
  return c < g_begin ? (uint32_t)(c - g_begin) : (uint32_t)min(c - g_begin, 0xFFFFFFFFull);
}

// Also clears the launch's Status record (the propagation kernel that follows on the stream counts from zero).
__global__ void tiles_kernel(const unsigned long long* __restrict__ cum, uint32_t n_src, unsigned long long g_begin,
                             uint32_t n_tiles, uint32_t tile_photons, uint32_t* __restrict__ tile_src,
                             uint32_t* __restrict__ cum_rel, Status* __restrict__ status) {
  const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j == 0 && status) *status = Status{};
  if (j <= n_src) cum_rel[j] = rel32(cum[j], g_begin);
  if (j < n_tiles) tile_entry(cum, n_src, g_begin, tile_photons, j, tile_src);
}

// Small launches (a few thousand sources and tiles; C3's 1e5-photon end): scan + tiles + status in ONE kernel of one
// CTA, so that the fixed cost of a launch is one kernel less (small batches underuse the GPU; what can
// be saved is the host-side latency around the kernel).
__global__ void __launch_bounds__(1024) prologue_kernel(const SrcRec* __restrict__ src, uint32_t n_src,
                                                        unsigned long long* __restrict__ cum, unsigned long long g_begin,
                                                        uint32_t n_tiles, uint32_t tile_photons,
                                                        uint32_t* __restrict__ tile_src, uint32_t* __restrict__ cum_rel,
                                                        Status* __restrict__ status) {
  __shared__ unsigned long long part[1024];
  const uint32_t t = threadIdx.x;
  const uint32_t per = (n_src + 1023u) / 1024u;
  const uint32_t lo = min(n_src, t * per), hi = min(n_src, lo + per);
  unsigned long long s = 0;
  for (uint32_t i = lo; i < hi; ++i) s += src[i].n_photons;
  part[t] = s;
  __syncthreads();
  for (uint32_t off = 1; off < 1024; off <<= 1) {
    unsigned long long v = (t >= off) ? part[t - off] : 0ull;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  unsigned long long run = (t == 0) ? 0ull : part[t - 1];
  for (uint32_t i = lo; i < hi; ++i) {
    cum[i] = run;
    cum_rel[i] = rel32(run, g_begin);
    run += src[i].n_photons;
  }
  if (t == 1023) { cum[n_src] = part[1023]; cum_rel[n_src] = rel32(part[1023], g_begin); }
  if (t == 0) *status = Status{};
  __threadfence_block();
  __syncthreads();
  for (uint32_t j = t; j < n_tiles; j += 1024u) tile_entry(cum, n_src, g_begin, tile_photons, j, tile_src);
}


// =============================================================================================
// a3-a8  Persistent propagation kernel
// =============================================================================================
#ifndef PP_BLOCK_THREADS
#define PP_BLOCK_THREADS 1024  // 64 registers per thread either way; one big CTA per SM stages the tables once (+1 %)
#endif
constexpr int kBlockThreads = PP_BLOCK_THREADS;
constexpr int kMaxDevices = 64;
constexpr uint32_t kDeadBit = 0x80000000u;  // top bit of a lane's flight counter: the lane holds no photon

// Shared-memory tables: one image built by the host (LaunchParams::smem_image), copied verbatim by every CTA.

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

struct Best {  // nearest DOM entry found so far on the current flight
  float t;
  uint32_t dom;
};

__device__ __forceinline__ void sphere_test(const float4 c, float R, float phx, float phy, float phz, float plx,
                                            float ply, float plz, float dx, float dy, float dz, float s, Best& best) {
  // Step 7: first point of [0, s] inside the closed ball; compensated position ph + pl (R-5, R-8)
  const float ox = (phx - c.x) + plx, oy = (phy - c.y) + ply, oz = (phz - c.z) + plz;
  const float b = fmaf(ox, dx, fmaf(oy, dy, oz * dz));
  const float qx = fmaf(-b, dx, ox), qy = fmaf(-b, dy, oy), qz = fmaf(-b, dz, oz);  // closest-approach vector
  const float disc = fmaf(R, R, -fmaf(qx, qx, fmaf(qy, qy, qz * qz)));
  if (disc < 0.0f) return;
  const float h = sqrtf(disc);
  const float t_in = -b - h, t_out = -b + h;
  if (t_out < 0.0f || t_in > s) return;
  const float t = fmaxf(t_in, 0.0f);
  const uint32_t dom = __float_as_uint(c.w);
  if (t < best.t || (t == best.t && dom < best.dom)) { best.t = t; best.dom = dom; }
}

// Step 7 (slow path, rare): the flight passes within the pre-filter radius of the axis of line
// `si`; test the DOMs whose z lies in the swept interval with the exact ray-sphere solve.
__device__ __noinline__ Best test_string(const LaunchParams& P, uint32_t si, float phx, float phy, float phz, float plx,
                                         float ply, float plz, float dx, float dy, float dz, float s, Best best) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const float4 sa = reinterpret_cast<const float4*>(smem_raw + P.off_str_a)[si];
  const uint2 sb = reinterpret_cast<const uint2*>(smem_raw + P.off_str_b)[si];
  const uint32_t n = sb.x, base = sb.y;
  // interval of the flight inside the infinite cylinder of radius Rm about the axis
  const float Rm = P.radius_margin;
  const float ax = (sa.x - phx) - plx, ay = (sa.y - phy) - ply;
  const float rho2 = fmaf(dx, dx, dy * dy);
  float ta = 0.0f, tb = s;
  if (rho2 > 1e-12f) {
    // (approximate reciprocal and square root: the interval only selects candidate DOMs, and Rm carries a margin
    // five orders of magnitude above their error)
    const float inv = fast_rcp(rho2);
    const float tc = fmaf(ax, dx, ay * dy) * inv;
    const float cr = fmaf(ax, dy, -ay * dx);
    const float h2 = fmaf(Rm * Rm, rho2, -cr * cr);
    if (h2 < 0.0f) return best;
    const float h = fast_sqrt(h2) * inv;
    ta = fmaxf(0.0f, tc - h);
    tb = fminf(s, tc + h);
    if (ta > tb) return best;
  } else if (fmaf(ax, ax, ay * ay) > Rm * Rm) {
    return best;
  }
  const float za = fmaf(dz, ta, phz), zb = fmaf(dz, tb, phz);
  const float zhi = fmaxf(za, zb) + Rm, zlo = fminf(za, zb) - Rm;
  int k_lo = (int)ceilf((sa.z - zhi) * sa.w);
  int k_hi = (int)floorf((sa.z - zlo) * sa.w);
  k_lo = max(k_lo - 1, 0);  // one extra on each side: the arithmetic lookup is only a candidate filter
  k_hi = min(k_hi + 1, (int)n - 1);
  for (int k = k_lo; k <= k_hi; ++k)
    sphere_test(__ldg(&P.dom_xyzw[base + k]), P.radius, phx, phy, phz, plx, ply, plz, dx, dy, dz, s, best);
  return best;
}

// Validation variant of step 7: every DOM, every flight.
__device__ __noinline__ Best test_all_doms(const LaunchParams& P, float phx, float phy, float phz, float plx, float ply,
                                           float plz, float dx, float dy, float dz, float s, Best best) {
  for (uint32_t j = 0; j < P.n_dom; ++j)
    sphere_test(__ldg(&P.dom_xyzw[j]), P.radius, phx, phy, phz, plx, ply, plz, dx, dy, dz, s, best);
  return best;
}

// R-21: the wavelength uniform is made of the low 9 bits of words 0, 1, 2 of the photon's Philox block 0 (the
// uniforms of R-3 use the top 23 bits of a word); bin j = the first with cdf[j] > u.  Entries past spec_n hold 2, and
// the count below runs over the warp-uniform bound spec_n, so the constant-bank loads are uniform.
__device__ __forceinline__ uint32_t spectrum_bin_from_words(const LaunchParams& P, uint32_t w0, uint32_t w1, uint32_t w2) {
  const float u = uniform_from_word(((w0 & 0x1FFu) << 23) | ((w1 & 0x1FFu) << 14) | ((w2 & 0x1FFu) << 5));
  uint32_t j = 0;
  for (uint32_t i = 0; i + 1u < P.spec_n; ++i) j += (P.spec_cdf[i] > u) ? 0u : 1u;
  return j;
}
// the same, recomputed from scratch where a hit's time or acceptance is formed (rare)
__device__ __noinline__ uint32_t spectrum_bin(const LaunchParams& P, uint32_t pidx, uint32_t sid, uint32_t ev) {
  uint32_t b0 = pidx, b1 = sid, b2 = ev, b3 = 0u;
  philox4x32_10(b0, b1, b2, b3, P.rk);
  return spectrum_bin_from_words(P, b0, b1, b2);
}

// R-23: fraction of a source's length at which a photon is emitted, F(u) piecewise linear through the knots
__device__ __forceinline__ float segment_fraction(const LaunchParams& P, float u) {
  if (P.seg_n < 2u) return u;
  const float x = u * (float)(P.seg_n - 1u);
  const uint32_t i = min(__float2uint_rz(x), P.seg_n - 2u);
  const float f0 = P.seg_tab[i], f1 = P.seg_tab[i + 1u];
  return fmaf(x - (float)i, f1 - f0, f0);
}

// Step 6, rare path.  The fast walk only finds where the SCATTERING budget runs out and how much absorption budget is
// left there; a remainder <= 0 means the photon was absorbed before that point.  Where that was matters only if a DOM
// was met on the flight (or for the fate dump): walk the absorption budget tau_a forward from the photon, layer by
// layer.  Returns the distance along the ray to the absorption point.
__device__ __noinline__ float absorb_distance(const LaunchParams& P, float phz, float plz, float dz, float tau_a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const float w = fmaxf(fabsf(dz), 1e-9f);
  const int last = P.last_layer;
  const bool up = dz > 0.0f;
  int l = (int)floorf((P.z_top - phz) * P.inv_dz_layer);
  l = max(0, min(l, last));
  const int i1 = l + (up ? 0 : 1);
  float h = fabsf((fmaf(-P.dz_layer, (float)i1, P.z_top) - phz) - plz);  // to the boundary ahead (two-float z)
  float T = tau_a * w, V = 0.0f;                                         // vertical budget, vertical distance so far
  for (;;) {
    const float a = *reinterpret_cast<const float*>(smem_raw + (uint32_t)l * 32u);  // absorption coefficient
    const bool open = up ? (l == 0) : (l == last);  // the end layers are infinite (R-6)
    const float need = a * h;
    if (open || T <= need) return (V + T / a) / w;
    T -= need;
    V += h;
    l += up ? -1 : 1;
    h = P.dz_layer;
  }
}

// DOM acceptance (R-17), rare path: p(eta) in the arrival direction cosine eta = d_z of a photon that met a DOM on
// flight k_hit.  Returns the weight of the hit (1 in the probabilistic mode, p in the weighted mode), or a negative
// number if the photon makes no photoelectron.
__device__ __noinline__ float dom_accepts(const LaunchParams& P, float dz, uint32_t pidx, uint32_t sid, uint32_t ev,
                                          uint32_t k_hit) {
  float pa = 0.0f;
  for (int c = (int)P.acc_n - 1; c >= 0; --c) pa = fmaf(pa, dz, P.acc_coef[c]);
  pa = fminf(fmaxf(pa, 0.0f), 1.0f);
  if (P.spec_n != 0u) pa = fminf(1.0f, pa * P.spec_acc[spectrum_bin(P, pidx, sid, ev)]);  // R-21
  if (P.acc_mode == 1u) {
    uint32_t a0 = pidx, a1 = sid, a2 = ev, a3 = 0x80000000u | k_hit;
    philox4x32_10(a0, a1, a2, a3, P.rk);
    return (uniform_from_word(a0) < pa) ? 1.0f : -1.0f;
  }
  return (pa > 0.0f) ? pa : -1.0f;
}

// Fetch the next work item of the launch for a warp (lane 0 talks to the queues; rare: once per tile).
// Returns the warp-uniform (t_next, t_end, s_cur, resume list not yet empty); t_next == t_end means no work is left.
__device__ __noinline__ uint4 fetch_work(const LaunchParams& P, unsigned lane, bool use_resume) {
  Status* const st = P.status;
  unsigned long long a = 0, b = 0;
  uint32_t sh = 0, res_left = use_resume ? 1u : 0u;
  if (lane == 0 && *(volatile unsigned int*)&st->stop == 0u) {
    if (use_resume) {
      const unsigned r = atomicAdd(&st->resume_counter, 1u);
      if (r < P.n_resume_in) {
        const WorkItem w = P.resume_in[r];
        a = w.g0; b = w.g1; sh = w.src;
      } else {
        res_left = 0u;
      }
    }
    if (a == b) {
      const unsigned long long j = atomicAdd(&st->tile_counter, 1ull);
      if (j < P.n_tiles) {
        a = P.g_begin + j * P.tile_photons;
        b = min(a + (unsigned long long)P.tile_photons, P.g_end);
        sh = __ldg(&P.tile_src[j]);
        (void)PP_GUARD_CHECK(st, sh < P.n_src, PP_GUARD_TILE_SRC);
        if (*(volatile unsigned int*)&st->stop != 0u) {
          // the ring filled up while we were fetching: hand the whole tile to the next launch
          const unsigned o = atomicAdd(&st->n_resume_out, 1u);
          if (o < P.resume_cap) P.resume_out[o] = WorkItem{a, b, sh, 0u}; else atomicExch(&st->error, 1u);
          a = b = 0;
        }
      }
    }
  }
  uint4 r;
  r.x = __shfl_sync(0xffffffffu, (uint32_t)(a - P.g_begin), 0);
  r.y = __shfl_sync(0xffffffffu, (uint32_t)(b - P.g_begin), 0);
  r.z = __shfl_sync(0xffffffffu, sh, 0);
  r.w = __shfl_sync(0xffffffffu, res_left, 0);
  return r;
}

// kExt: which of the optional physics that touches the flight loop is compiled in.  0: none.  1: wavelength bins
// (R-21) only, switched on (no run-time test in the loop).  2: wavelength bins, track-segment sources (R-18) and
// emission smearing (R-22), each behind its run-time switch.  The DOM acceptance (R-17) is in every variant, in the
// rare hit block.  kLoop: the inverse walk tables are coarser than the thinnest layer (pathological
// ice, LaunchParams::walk_loop), so the layer found may be several layers short
template <bool kBrute, bool kFates, int kExt, bool kLoop>
__global__ void __launch_bounds__(kBlockThreads, PP_MIN_BLOCKS) propagate_kernel(const __grid_constant__ LaunchParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // ---- stage the medium and the DOM lookup in shared memory (a4, a5): one verbatim copy of the host-built image ----
  {
    uint4* const dst = reinterpret_cast<uint4*>(smem_raw);
    const uint32_t n16 = P.smem_image_bytes >> 4;
    for (uint32_t i = threadIdx.x; i < n16; i += blockDim.x) dst[i] = __ldg(P.smem_image + i);
  }
  // R-21: (1 / abs_scale, 1 / scat_scale) of the wavelength bins, where a lane can index them freely
  __shared__ float2 s_spec[kExt != 0 ? PP_MAX_SPECTRUM_BINS : 1];
  if (kExt != 0 && threadIdx.x < PP_MAX_SPECTRUM_BINS)
    s_spec[threadIdx.x] = make_float2(P.spec_inv_a[threadIdx.x], P.spec_inv_b[threadIdx.x]);
  __syncthreads();
  // layer records at offset 0: coefficients (a, b, 1/b, a) of layer i, cumulative depths at boundary i
  auto walk_B = [&](int i) { return *reinterpret_cast<const float*>(smem_raw + (uint32_t)i * 32u + 16u); };
  const uint16_t* const s_inv_b = reinterpret_cast<const uint16_t*>(smem_raw + P.off_inv_b);
  const float2* const s_str_xy = reinterpret_cast<const float2*>(smem_raw + P.off_str_xy);
  const uint16_t* const s_cell = reinterpret_cast<const uint16_t*>(smem_raw + P.off_cell);
  // the warp's current source record (a2): staged once per (tile, source) run, read by the lanes that refill
  __shared__ float4 s_wsrc[kBlockThreads / 32][3];
  const unsigned wslot = threadIdx.x >> 5;
  uint32_t wsrc_addr;  // shared-window address of this warp's record, pinned in a register (not rematerialised)
  asm volatile("mov.u32 %0, %1;" : "=r"(wsrc_addr) : "r"((uint32_t)__cvta_generic_to_shared(&s_wsrc[wslot][0])));

  const unsigned lt = lanemask_lt();
  Status* const st = P.status;
  const float inf = __int_as_float(0x7f800000);

  // ---- warp-uniform work state: photons [t_next, t_end) of the launch (numbered from g_begin) are this warp's
  // current work item; [t_next, run_end) of them belong to source s_cur, whose photon 0 is launch photon pbase ----
  uint32_t t_next = 0, t_end = 0, run_end = 0, s_cur = 0, pbase = 0;
  bool refill_ok = true;   // false once the queues are empty or the hit ring filled up
  bool use_resume = P.n_resume_in > 0;
  uint32_t w_started = 0, w_hits = 0, w_flights = 0;

  // ---- per-lane photon state (a dead lane keeps computing on its stale state; nothing it produces is used) ----
  float phx = 0, phy = 0, phz = 0, plx = 0, ply = 0, plz = 0;  // position, two-float (hi + lo)
  float dx = 0, dy = 0, dz = 1;
  float Lh = 0, Ll = 0;  // path length, two-float
  float tau_a = 0;
  float sc_b = 1.0f;  // kExt only: 1 / scat_scale of the photon's wavelength bin (R-21)
  const bool spectrum_on = kExt == 1 || (kExt == 2 && P.spec_n != 0u);  // (a compile-time constant unless kExt == 2)
  // k = flights started so far = index of the next Philox block; its top bit marks a DEAD lane (no register for a
  // flag; max_flights < 2^31 is checked at pp_create)
  uint32_t ev = 0, sid = 0, pidx = 0, k = kDeadBit, s_mine = 0;

  // A new run (rare: once per source of a work item): the next source of the current work item, or a new work item
  // (resume list first, then tiles).  Leaves t_next < run_end, or refill_ok = false when no work is left.
  auto next_run = [&]() {
    if (t_next == t_end) {
      const uint4 wk = fetch_work(P, __popc(lt), use_resume);
      t_next = wk.x; t_end = wk.y; s_cur = wk.z; use_resume = wk.w != 0u;
      w_started += t_end - t_next;  // counted per work item; what is handed back at the end is taken out again
    } else {
      ++s_cur;
    }
    if (t_next != t_end) {
      uint32_t hi = 0u;
      while (PP_GUARD_CHECK(st, s_cur < P.n_src, PP_GUARD_SRC_INDEX) &&
             (hi = __ldg(&P.cum_rel[s_cur + 1])) <= t_next) ++s_cur;  // skips sources without photons
      pbase = __ldg(&P.cum_rel[s_cur]);  // mod 2^32: right for the launch's first (split) source too
      run_end = min(t_end, hi);
      __syncwarp();
      if (__popc(lt) < 3) s_wsrc[wslot][__popc(lt)] = __ldg(reinterpret_cast<const float4*>(P.src + s_cur) + __popc(lt));
      __syncwarp();
    } else {
      run_end = t_end;
      refill_ok = false;
    }
  };
  next_run();

  for (;;) {
    // =========================== refill dead lanes (a2 -> a3) ===========================
    // t_next < run_end whenever refill_ok: the next run is fetched as soon as the current one is used up, and a
    // refill that uses it up goes on with the next one, so lanes stay dead only when the launch has run dry
    // (no test in front of the loop: nearly every iteration has dead lanes, and with none, or with nothing to refill
    // from -- run_end == t_next then --, the body assigns nothing and leaves at once)
    unsigned need_mask = __ballot_sync(0xffffffffu, (int)k < 0);
    for (;;) {
      // ---- a2/a3: initial state of photon r of the launch (fused expansion) ----
      // (compared as "rank < photons left in the run": t_next + rank may wrap for a warp that holds no work item
      // in a launch whose first photon is not the first of its source)
      const uint32_t rank = __popc(need_mask & lt), avail = run_end - t_next;
      const uint32_t r = t_next + rank;
      if ((int)k < 0 && rank < avail) {
        float4 r0; float2 r1; uint2 r2;
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r0.x), "=f"(r0.y), "=f"(r0.z), "=f"(r0.w) : "r"(wsrc_addr));
        asm volatile("ld.shared.v2.f32 {%0,%1}, [%2+16];" : "=f"(r1.x), "=f"(r1.y) : "r"(wsrc_addr));
        asm volatile("ld.shared.v2.u32 {%0,%1}, [%2+32];" : "=r"(r2.x), "=r"(r2.y) : "r"(wsrc_addr));
        phx = r0.x; phy = r0.y; phz = r0.z; plx = ply = plz = 0.0f;
        dx = r0.w; dy = r1.x; dz = r1.y;
        Lh = 0.0f; Ll = 0.0f;
        ev = r2.x; sid = r2.y;
        pidx = r - pbase;
        (void)PP_GUARD_CHECK(st, pidx < __ldg(&P.src[s_cur].n_photons), PP_GUARD_PHOTON_INDEX);
        k = 0; s_mine = s_cur;  // alive
      }
      t_next += min((uint32_t)__popc(need_mask), avail);
      if (t_next != run_end || !refill_ok) break;
      next_run();
      need_mask = __ballot_sync(0xffffffffu, (int)k < 0);
    }
    const bool alive = (int)k >= 0;
    const unsigned alive_mask = __ballot_sync(0xffffffffu, alive);
    if (alive_mask == 0u) break;  // nothing left to refill from
    w_flights += __popc(alive_mask);  // every live lane flies once per iteration

    // =========================== a7': Philox block k of this photon ===========================
    uint32_t c0 = pidx, c1 = sid, c2 = ev, c3 = k;
    philox4x32_10(c0, c1, c2, c3, P.rk);
    const float u_az = uniform_from_word(c0), u_hg = uniform_from_word(c1);
    const float u_dist = uniform_from_word(c2), u_abs = uniform_from_word(c3);
    // =========================== a7: emission (k = 0) or scatter (k > 0) ======================
    const float m_hg = hg_one_minus_cos(u_hg, P.hg_one_minus_g, P.hg_two_g, P.hg_one_minus_g2);
    const float m = (k == 0) ? P.one_minus_cos_c : m_hg;
    if (kExt == 2 && P.has_segments != 0u && k == 0) {
      // R-18: a source with a length emits from a point uniform along it; u_hg is free on flight 0
      const float ell = segment_fraction(P, u_hg) * __ldg(&P.src[s_mine].length);
      const float nx_ = fmaf(dx, ell, phx); plx += fmaf(dx, ell, phx - nx_); phx = nx_;
      const float ny_ = fmaf(dy, ell, phy); ply += fmaf(dy, ell, phy - ny_); phy = ny_;
      const float nz_ = fmaf(dz, ell, phz); plz += fmaf(dz, ell, phz - nz_); phz = nz_;
    }
    if (kExt == 2 && P.emit_on != 0u && k == 0) {
      // R-22: the axis the photon is emitted about = the source axis deflected by an HG(g_axis) polar angle
      uint32_t e0 = pidx, e1 = sid, e2 = ev, e3 = 0x20000000u;
      philox4x32_10(e0, e1, e2, e3, P.rk);
      rotate(dx, dy, dz, hg_one_minus_cos(uniform_from_word(e0), P.emit_one_minus_g, P.emit_two_g, P.emit_one_minus_g2),
             uniform_from_word(e1));
    }
    rotate(dx, dy, dz, m, u_az);
    // =========================== a3: absorption budget (once per photon) ======================
    float tau_new = neg_log_fast(u_abs);
    if (spectrum_on && k == 0) {
      // R-21: the photon's wavelength bin from the spare bits of block 0.  Both optical-depth budgets are kept in
      // units of the unscaled ice table: tau_a is divided by abs_scale once, sc_b = 1 / scat_scale multiplies
      // every tau_s.
      // The bin's two scales come from shared memory: a per-lane index into the constant bank (where the tables
      // arrive) is replayed once per distinct value in the warp, a shared-memory read is not.
      const float2 sc = s_spec[spectrum_bin_from_words(P, c0, c1, c2)];
      tau_new *= sc.x;
      sc_b = sc.y;
    }
    tau_a = (k == 0) ? tau_new : tau_a;
    // =========================== a4: optical depth to the next scatter ========================
    float tau_s = neg_log_fast(u_dist);
    if (spectrum_on) tau_s *= sc_b;
    // =========================== a4: layer walk in vertical optical depth ======================
    // Along a straight ray the optical depth spent between two heights is (vertical optical depth)/|d_z|,
    // so the budgets are scaled by w = |d_z| once and the walk works in vertical metres.
    const float w = fmaxf(fabsf(dz), 1e-9f);
    const float inv_w = fast_rcp(w);
    const bool up = dz > 0.0f;
    const int last = P.last_layer;
    // Direct walk, branch-free.  h0 is the vertical distance to the boundary ahead, i1; the flight reaches it with
    // budgets t1 (scattering), t2 (absorption) left (negative: it ends before).  With B(i), A(i) the cumulative
    // vertical optical depths at the boundaries (two-float sums), the cumulative depth X = B(i1) +- t1 at which the
    // scattering budget runs out names the layer js (inverse table + one compare-and-step); clamped to the photon's
    // side of its own layer it is the layer lj where the flight would scatter.  lj = li (always so in an end layer
    // with no boundary ahead, R-6): the budgets are spent in layer li, as they are.  Otherwise the budgets left at
    // lj's entry boundary come from the two-float sums, so their error is relative to the budget, not to the
    // cumulative depth.  Coefficients and sums come from one record each at the start and at the end (LayerRec,
    // pp_types.h).  The absorption budget is only FOLLOWED to the scatter point: what is left of it there becomes
    // the new tau_a, and a remainder <= 0 means the photon was absorbed on the way (where exactly is worked out in
    // the rare path, absorb_distance, when a DOM was met on the flight).
    const float sgn = up ? -1.0f : 1.0f;
    int li = (int)floorf((P.z_top - phz) * P.inv_dz_layer);
    li = max(0, min(li, last));
    const int i1 = li + (up ? 0 : 1);
    const float h0 = fabsf((fmaf(-P.dz_layer, (float)i1, P.z_top) - phz) - plz);  // two-float z
    const unsigned char* const rec0 = smem_raw + (up ? 0u : P.off_rec_b) + (uint32_t)li * 32u;
    const float2 L0 = *reinterpret_cast<const float2*>(rec0);  // a, b of layer li
    const float4 W1 = *reinterpret_cast<const float4*>(rec0 + 16);
    const float Ts0 = tau_s * w, Ta0 = tau_a * w;
    const float t1 = fmaf(-L0.y, h0, Ts0), t2 = fmaf(-L0.x, h0, Ta0);
    const float Xs = fmaf(sgn, t1, W1.x);
    const float xs_l = fmaf(sgn, t1, W1.z), xa_l = fmaf(sgn, t2, W1.w);  // lo parts of the two-float X
    int js = s_inv_b[min(__float2uint_rz(fmaf(Xs, P.k_b, -1e-3f)), P.m_b)];
    js += (walk_B(js + 1) <= Xs) ? 1 : 0;
    if (kLoop) {
      while (js < last && walk_B(js + 1) <= Xs) ++js;
    }
    const int lj = up ? min(js, li) : max(js, li);
    const unsigned char* const rec1 = smem_raw + (up ? P.off_rec_b : 0u) + (uint32_t)lj * 32u;
    const float2 L4 = *reinterpret_cast<const float2*>(rec1 + 8);  // 1/b, a of layer lj
    const float4 Wb = *reinterpret_cast<const float4*>(rec1 + 16);
    // (selects through select_eq: the compiler would otherwise branch around the three right-hand sides, and nearly
    // every warp holds lanes of both kinds)
    const float Ts = select_eq(lj, li, Ts0, sgn * ((W1.x - Wb.x) + (xs_l - Wb.z)));
    const float Ta = select_eq(lj, li, Ta0, sgn * ((W1.y - Wb.y) + (xa_l - Wb.w)));
    const float Vb = select_eq(lj, li, 0.0f, fmaf(P.dz_layer, (float)(abs(lj - li) - 1), h0));
    const float vs = Ts * L4.x;                   // vertical distance to the scatter point in the final layer
    // ... and the flight's length if the photon gets that far; kept finite (a near-horizontal flight in ice that
    // hardly scatters overflows), so that "no DOM" (t = inf) never compares as a hit
    const float s = fminf((Vb + vs) * inv_w, 3.0e38f);
    const float Ta_left = fmaf(-L4.y, vs, Ta);    // absorption budget left at the scatter point (vertical)
    const bool absorbed = !(Ta_left > 0.0f);      // ties: absorbed (s_abs <= s_scat)
    const float tau_a0 = tau_a;                   // (kept for the rare path below)
    tau_a = Ta_left * inv_w;
    // =========================== a5: DOM intersection on [0, s] ===============================
    Best best{inf, 0xFFFFFFFFu};
    if (kBrute) {
      if (alive) best = test_all_doms(P, phx, phy, phz, plx, ply, plz, dx, dy, dz, s, best);
    } else {
      // the one line of DOMs a piece of flight no longer than xy_cap in the xy-plane can meet is named by the
      // cell of the piece's xy midpoint; a longer flight is looked up piece by piece
      const float rho2 = fmaf(dx, dx, dy * dy);
      const float sxy2 = s * s * rho2;
      float ds = s;
      int n_ch = 1;
      if (sxy2 > P.xy_cap2) {
        const float f = floorf(fast_sqrt(sxy2) * P.inv_xy_cap) + 1.0f;
        if (f > 64.0f) {
          // a flight of more than 64 pieces (far longer than the detector is wide): every line, here in the rare
          // path; the one look-up below then repeats a line already tested, which changes nothing
          if (alive)
            for (uint32_t si = 0; si < P.n_strings; ++si)
              best = test_string(P, si, phx, phy, phz, plx, ply, plz, dx, dy, dz, s, best);
        } else {
          n_ch = (int)f;
          ds = s * fast_rcp(f);
        }
      }
      const float rm2 = fmaf(P.rm2, rho2, 1e-12f);
      float tm = 0.5f * ds;
#pragma unroll 1
      for (;;) {
        // cell of the piece's midpoint; the saturating conversion sends negative coordinates to cell 0.  An empty
        // cell names the NaN entry of the line table, which fails the pre-filter.
        const uint32_t cx = min(__float2uint_rz(fmaf(fmaf(tm, dx, phx), P.inv_cell, P.cell_ox)), P.nx_m1);
        const uint32_t cy = min(__float2uint_rz(fmaf(fmaf(tm, dy, phy), P.inv_cell, P.cell_oy)), P.ny_m1);
        const uint32_t si = s_cell[cy * P.nx + cx];
        const float2 sxy = s_str_xy[si];
        const float cr = fmaf(sxy.x - phx, dy, -(sxy.y - phy) * dx);
        if (cr * cr <= rm2 && alive)
          best = test_string(P, si, phx, phy, phz, plx, ply, plz, dx, dy, dz, s, best);
        if (--n_ch <= 0) break;
        tm += ds;
      }
    }
    bool hit = best.t <= s;  // (a dead lane never looks for DOMs: its best.t is inf)
    const uint32_t hit_dom = best.dom;
    // =========================== a6: advance / terminate ======================================
    float s_end = s;
    if (kFates && alive && absorbed) {
      // the fate dump wants the end point of every absorbed photon: where was it absorbed?
      s_end = fminf(s, absorb_distance(P, phz, plz, dz, tau_a0));
      hit = hit && best.t <= s_end;
    }
    // (the lean variant asks that question only for a photon that also met a DOM on this flight, in the rare
    // block below; until then `hit` may hold a DOM that lies behind the absorption point)
    const float adv = hit ? best.t : s_end;
    {
      // compensated position: sum = fl(p + d*adv); the rounding error is recovered with one
      // more fma (exact unless |p| << |d*adv| ulp-wise, where it is negligible anyway)
      const float nx_ = fmaf(dx, adv, phx); plx += fmaf(dx, adv, phx - nx_); phx = nx_;
      const float ny_ = fmaf(dy, adv, phy); ply += fmaf(dy, adv, phy - ny_); phy = ny_;
      const float nz_ = fmaf(dz, adv, phz); plz += fmaf(dz, adv, phz - nz_); phz = nz_;
      const float nl = Lh + adv; Ll += adv - (nl - Lh); Lh = nl;
    }
    k += 1u;  // k counts the free flights started = index of the next Philox block
    const bool aborted = alive && !hit && !absorbed && k >= P.max_flights;
    const bool done = hit || absorbed || aborted;

    // =========================== a8: hit write (warp-aggregated); rare =============================
    bool deferred = false, rejected = false;
    unsigned hit_mask = __ballot_sync(0xffffffffu, hit || aborted);
    if (hit_mask) {
      if (aborted) atomicAdd(&st->photons_aborted, 1ull);  // never in practice (R-10)
      if (!kFates && hit && absorbed) {
        // absorbed before the scatter point AND a DOM on the way: which came first?  The photon has been advanced to
        // the DOM already (it is dead either way), so its start height is recovered from there, as a two-float.
        const float z0 = fmaf(-dz, adv, phz);
        const float z0l = plz + fmaf(-dz, adv, phz - z0);
        hit = adv <= absorb_distance(P, z0, z0l, dz, tau_a0);
      }
      hit_mask = __ballot_sync(0xffffffffu, hit);
      float weight = 1.0f;
      if (P.acc_mode != 0u && hit_mask) {
        // ---- DOM acceptance (R-17): asked only here, where a lane of the warp has met a DOM (4e-5 of the photons
        // in C1), behind a warp-uniform run-time switch: every kernel variant has it, and it costs the others nothing
        if (hit) {
          weight = dom_accepts(P, dz, pidx, sid, ev, k - 1u);  // k was advanced: the hit flight is k - 1
          rejected = weight < 0.0f;
          hit = !rejected;
        }
        const unsigned rej_mask = __ballot_sync(0xffffffffu, rejected);
        if (rej_mask && __popc(lt) == __ffs(rej_mask) - 1) atomicAdd(&st->photons_rejected, (unsigned long long)__popc(rej_mask));
        hit_mask &= ~rej_mask;
      }
      if (hit_mask) {
        const unsigned n_hit = __popc(hit_mask);
        unsigned base = 0;
        const int leader = __ffs(hit_mask) - 1;
        if (__popc(lt) == leader) base = atomicAdd(&st->hit_count, n_hit);
        base = __shfl_sync(0xffffffffu, base, leader);
        if (hit) {
          const unsigned slot = base + __popc(hit_mask & lt);
          if (slot < P.ring_cap && PP_GUARD_CHECK(st, base + n_hit >= base, PP_GUARD_HIT_SLOT)) {
            double t0 = (double)__ldg(&P.src[s_mine].t);
            if (kExt == 2 && P.has_segments != 0u) {
              // R-18: emitted l / c after the source time; l is recomputed from block 0 instead of being carried
              uint32_t e0 = pidx, e1 = sid, e2 = ev, e3 = 0u;
              philox4x32_10(e0, e1, e2, e3, P.rk);
              t0 += (double)(segment_fraction(P, uniform_from_word(e1)) * __ldg(&P.src[s_mine].length)) * (double)P.inv_c;
            }
            pp_hit h;
            h.event_id = ev; h.source_id = sid; h.photon_idx = pidx; h.dom_id = hit_dom;
            double inv_v = P.inv_v;
            if (spectrum_on) inv_v = P.spec_inv_v[spectrum_bin(P, pidx, sid, ev)];  // R-21
            h.time_ns = t0 + ((double)Lh + (double)Ll) * inv_v;
            h.weight = weight; h.n_scatter = k - 1;
            uint4* dst = reinterpret_cast<uint4*>(reinterpret_cast<pp_hit*>(P.ring) + slot);
            const uint4* srcv = reinterpret_cast<const uint4*>(&h);
            dst[0] = srcv[0];
            dst[1] = srcv[1];
          } else {
            // ring full: this photon is replayed from scratch by the next launch (counter-based RNG)
            deferred = true;
            const unsigned long long g = __ldg(&P.cum[s_mine]) + pidx;
            const unsigned o = atomicAdd(&st->n_resume_out, 1u);
            if (o < P.resume_cap) P.resume_out[o] = WorkItem{g, g + 1, s_mine, 0u}; else atomicExch(&st->error, 1u);
            atomicExch(&st->stop, 1u);
          }
        }
        const unsigned def_mask = __ballot_sync(0xffffffffu, deferred);
        w_hits += n_hit - __popc(def_mask);
        if (def_mask) {
          // the replay will count these photons (and their flights) again: take them out here
          refill_ok = false;
          run_end = t_next;  // (nothing more is handed out; [t_next, t_end) goes to the resume list at the end)
          w_started -= __popc(def_mask);
          w_flights -= __reduce_add_sync(0xffffffffu, deferred ? k : 0u);
        }
      }
    }

    if (kFates) {
      if (alive && done && !deferred) {
        const unsigned long long g = __ldg(&P.cum[s_mine]) + pidx;
        pp_fate f;
        f.x = phx + plx; f.y = phy + ply; f.z = phz + plz;
        f.path_m = Lh + Ll;
        f.time_ns = (double)__ldg(&P.src[s_mine].t) + ((double)Lh + (double)Ll) *
                    (spectrum_on ? P.spec_inv_v[spectrum_bin(P, pidx, sid, ev)] : P.inv_v);
        f.n_flights = k;
        f.dom = (hit || rejected) ? (int32_t)hit_dom : -1;
        f.fate = hit ? 1u : (rejected ? 3u : (aborted ? 2u : 0u));
        f.photon_idx = pidx;
        if (PP_GUARD_CHECK(st, g < P.g_end, PP_GUARD_FATE_INDEX)) reinterpret_cast<pp_fate*>(P.fates)[g] = f;
      }
    }
    k |= done ? kDeadBit : 0u;  // (a dead lane stays dead whatever its stale state says)
  }

  // ---- leftovers of a stopped warp go to the next launch; fold the counters ----
  if (lt == 0u) {
    if (t_next < t_end) {
      w_started -= t_end - t_next;
      const unsigned o = atomicAdd(&st->n_resume_out, 1u);
      if (o < P.resume_cap) P.resume_out[o] = WorkItem{P.g_begin + t_next, P.g_begin + t_end, s_cur, 0u};
      else atomicExch(&st->error, 1u);
    }
    atomicAdd(&st->photons_started, (unsigned long long)w_started);
    atomicAdd(&st->flights, (unsigned long long)w_flights);  // < 2^32 per warp for any launch of < 2^32 photons
    if (w_hits) atomicAdd(&st->photons_hit, (unsigned long long)w_hits);
  }
}

// =============================================================================================
// host-side launch wrappers (declared in pp_internal.h)
// =============================================================================================
static std::atomic<uint64_t> g_launches{0};
uint64_t kernel_launch_count() { return g_launches.load(); }

cudaError_t launch_ingest(const pp_source* d_s, const uint32_t* d_ev, const uint32_t* d_sid, uint32_t sid_base, uint32_t n,
                          float yield, SrcRec* d_out, unsigned int* d_overflow, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  ingest_kernel<<<(n + 255) / 256, 256, 0, st>>>(d_s, d_ev, d_sid, sid_base, n, yield, d_out, d_overflow);
  g_launches++;
  return cudaGetLastError();
}

cudaError_t launch_scan(const SrcRec* d_src, uint32_t n, unsigned long long* d_cum, cudaStream_t st) {
  scan_kernel<<<1, 1024, 0, st>>>(d_src, n, d_cum);
  g_launches++;
  return cudaGetLastError();
}

cudaError_t launch_tiles(const unsigned long long* d_cum, uint32_t n_src, unsigned long long g_begin, uint32_t n_tiles,
                         uint32_t tile_photons, uint32_t* d_tile_src, uint32_t* d_cum_rel, Status* d_status,
                         cudaStream_t st) {
  const uint32_t n_thr = max(max(n_tiles, n_src + 1), 1u);
  tiles_kernel<<<(n_thr + 255) / 256, 256, 0, st>>>(d_cum, n_src, g_begin, n_tiles, tile_photons, d_tile_src, d_cum_rel,
                                                      d_status);
  g_launches++;
  return cudaGetLastError();
}

cudaError_t launch_prologue(const SrcRec* d_src, uint32_t n_src, unsigned long long* d_cum, unsigned long long g_begin,
                            uint32_t n_tiles, uint32_t tile_photons, uint32_t* d_tile_src, uint32_t* d_cum_rel,
                            Status* d_status, cudaStream_t st) {
  prologue_kernel<<<1, 1024, 0, st>>>(d_src, n_src, d_cum, g_begin, n_tiles, tile_photons, d_tile_src, d_cum_rel, d_status);
  g_launches++;
  return cudaGetLastError();
}

// Opt-in dynamic shared memory size of one kernel variant: raised when a handle needs more than any before it on
// this device (the attribute is per device and per function; it is never lowered).
template <bool B, bool F, int A, bool L>
static cudaError_t ensure_smem(size_t smem) {
  static std::atomic<size_t> attr_smem[kMaxDevices];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (smem > attr_smem[dev].load()) {
    e = cudaFuncSetAttribute(propagate_kernel<B, F, A, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_smem[dev].store(smem);
  }
  return cudaSuccess;
}

template <bool B, bool F, int A, bool L>
static cudaError_t launch_prop_t(const LaunchParams& P, int grid, size_t smem, cudaStream_t st) {
  const cudaError_t e = ensure_smem<B, F, A, L>(smem);
  if (e != cudaSuccess) return e;
  propagate_kernel<B, F, A, L><<<grid, kBlockThreads, smem, st>>>(P);
  g_launches++;
  return cudaGetLastError();
}

template <bool B, bool F, bool L>
static cudaError_t launch_prop_ext(int ext, const LaunchParams& P, int grid, size_t smem, cudaStream_t st) {
  switch (ext) {
    case 0: return launch_prop_t<B, F, 0, L>(P, grid, smem, st);
    case 1: return launch_prop_t<B, F, 1, L>(P, grid, smem, st);
    default: return launch_prop_t<B, F, 2, L>(P, grid, smem, st);
  }
}
template <bool B, bool F>
static cudaError_t launch_prop_loop(bool loop, int ext, const LaunchParams& P, int grid, size_t smem, cudaStream_t st) {
  return loop ? launch_prop_ext<B, F, true>(ext, P, grid, smem, st) : launch_prop_ext<B, F, false>(ext, P, grid, smem, st);
}

// the kernel variant is picked by (brute-force DOM test, fate dump, flight-loop physics in use, coarse walk tables)
cudaError_t launch_propagate(const LaunchParams& P, bool brute, bool fates, int grid, size_t smem, cudaStream_t st) {
  // (the DOM acceptance needs no variant of its own: it sits in the rare hit block of every variant)
  const int ext = (P.has_segments != 0u || P.emit_on != 0u) ? 2 : (P.spec_n != 0u ? 1 : 0);
  const bool loop = P.walk_loop != 0u;
  if (brute) return fates ? launch_prop_loop<true, true>(loop, ext, P, grid, smem, st)
                          : launch_prop_loop<true, false>(loop, ext, P, grid, smem, st);
  return fates ? launch_prop_loop<false, true>(loop, ext, P, grid, smem, st)
               : launch_prop_loop<false, false>(loop, ext, P, grid, smem, st);
}

int propagate_warps_per_block() { return kBlockThreads / 32; }

template <bool B, bool F, int A, bool L>
static cudaError_t occupancy_t(size_t smem, int* n) {
  const cudaError_t e = ensure_smem<B, F, A, L>(smem);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(n, propagate_kernel<B, F, A, L>, kBlockThreads, smem);
}

cudaError_t propagate_occupancy(bool brute, bool fates, size_t smem, int* blocks_per_sm) {
  // all variants are compiled for the same launch bounds; the leanest and the fullest bracket the rest
  int a = 0, b = 0;
  cudaError_t e = brute ? occupancy_t<true, true, 2, true>(smem, &a) : occupancy_t<false, true, 2, true>(smem, &a);
  if (e != cudaSuccess) return e;
  e = brute ? occupancy_t<true, false, 0, false>(smem, &b) : occupancy_t<false, false, 0, false>(smem, &b);
  (void)fates;
  *blocks_per_sm = a < b ? a : b;
  return e;
}

// =============================================================================================
// pp_run_resident_noalloc (include/pp.h): a small resident run whose scratch is a static device array
// =============================================================================================
// For callers that cannot get device memory when they need photons propagated (a framework's pool owns the device; a
// latency-bound loop that cannot afford cudaMalloc's wait for running kernels; a process in which a stream is being
// captured).  Everything pp_run_resident keeps in the handle's workspace for a launch -- expanded source records,
// prefix sums, tile table, Status -- sits here in one array that is part of the library image.  One array per device,
// shared by every call: see the rules in pp.h.

constexpr uint32_t kNoallocMaxSrc = PP_NOALLOC_MAX_SOURCES;
constexpr uint32_t kNoallocMaxPhotons = PP_NOALLOC_MAX_PHOTONS;
constexpr uint32_t kNoallocMaxTiles = 65536;  // >= 2 x (tiles wanted for a small launch: 4 per resident warp) up to 256 SMs

struct NoallocHead {  // what the host reads back after the prologue
  unsigned long long total;  // photons of the call
  unsigned int overflow;     // a source with more than 2^32 - 1 photons
  unsigned int tile_photons, n_tiles;
  unsigned int too_big;      // more photons or tiles than the array is laid out for: no tile table was written
};
struct NoallocScratch {
  Status status;  // counters of the propagation launch: cleared by the prologue of every call
  NoallocHead head;
  alignas(16) SrcRec src[kNoallocMaxSrc];
  unsigned long long cum[kNoallocMaxSrc + 1];
  uint32_t cum_rel[kNoallocMaxSrc + 1];
  uint32_t tile_src[kNoallocMaxTiles];
};
constexpr size_t kNoallocBytes = (sizeof(NoallocScratch) + 255) / 256 * 256;
static_assert(kNoallocBytes <= (512u << 10), "pp.h promises at most 512 KiB");

// THE scratch.  In host code this name is only a handle for cudaGetSymbolAddress -- not a device address: a kernel given
// `g_noalloc_scratch` from the host side would fault, or scribble over host memory the GPU can reach.  The device
// address is looked up once per device in noalloc_scratch() below.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocBytes];

// Variant of prologue_kernel for the array above: ingest (build the source records, count photons) + prefix sums +
// choice of the tile size + tile table + cleared Status, one CTA.  g_begin is 0: the call is one launch.
// Everything a later kernel of the same call reads is written here first, so nothing left by an earlier call matters.
__global__ void __launch_bounds__(1024) noalloc_prologue_kernel(NoallocScratch* __restrict__ S,
                                                                const pp_source* __restrict__ s,
                                                                const uint32_t* __restrict__ ev,
                                                                const uint32_t* __restrict__ sid, uint32_t n, float yield,
                                                                uint32_t want_tiles) {
  __shared__ unsigned long long part[1024];
  __shared__ unsigned int s_overflow;
  const uint32_t t = threadIdx.x;
  if (t == 0) s_overflow = 0u;
  __syncthreads();
  const uint32_t per = (n + 1023u) / 1024u;
  const uint32_t lo = min(n, t * per), hi = min(n, lo + per);
  unsigned long long sum = 0;
  for (uint32_t i = lo; i < hi; ++i) {
    const pp_source a = s[i];
    unsigned long long cnt = photon_count(a.energy_GeV, yield);
    if (cnt > 0xFFFFFFFFull) { s_overflow = 1u; cnt = 0; }
    SrcRec r;
    r.x = a.x; r.y = a.y; r.z = a.z; r.dx = a.dx; r.dy = a.dy; r.dz = a.dz; r.t = a.t_ns; r.energy = a.energy_GeV;
    r.event_id = ev[i]; r.source_id = sid[i]; r.n_photons = (uint32_t)cnt; r.length = 0.0f;
    S->src[i] = r;
    sum += cnt;
  }
  part[t] = sum;
  __syncthreads();
  for (uint32_t off = 1; off < 1024; off <<= 1) {
    unsigned long long v = (t >= off) ? part[t - off] : 0ull;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  unsigned long long run = (t == 0) ? 0ull : part[t - 1];
  for (uint32_t i = lo; i < hi; ++i) {
    S->cum[i] = run;
    S->cum_rel[i] = rel32(run, 0ull);
    run += S->src[i].n_photons;  // (this thread wrote it)
  }
  const unsigned long long total = part[1023];
  if (t == 1023) { S->cum[n] = total; S->cum_rel[n] = rel32(total, 0ull); }
  // tile size as pick_tiles (pp_api.cpp) chooses it for a small launch: about `want_tiles` tiles, 32..1024 photons each
  uint32_t tile = kTilePhotons;
  while (tile > (uint32_t)kMinTilePhotons && total / tile < want_tiles) tile >>= 1;
  const unsigned long long n_tiles = (total + tile - 1) / tile;
  const bool too_big = total > kNoallocMaxPhotons || n_tiles > kNoallocMaxTiles;
  if (t == 0) {
    S->status = Status{};
    S->head.total = total; S->head.overflow = s_overflow; S->head.tile_photons = tile;
    S->head.n_tiles = too_big ? 0u : (uint32_t)n_tiles; S->head.too_big = too_big ? 1u : 0u;
  }
  __threadfence_block();
  __syncthreads();  // the tile search reads prefix sums other threads wrote
  if (!too_big)
    for (uint32_t j = t; j < (uint32_t)n_tiles; j += 1024u) tile_entry(S->cum, n, 0ull, tile, j, S->tile_src);
}

// Device address of the array on the CURRENT device; looked up on the first call for that device, kept afterwards.
static cudaError_t noalloc_scratch(int dev, NoallocScratch** out) {
  static std::mutex mu;
  static NoallocScratch* addr[kMaxDevices] = {};
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> g(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    addr[dev] = static_cast<NoallocScratch*>(p);
  }
  *out = addr[dev];
  return cudaSuccess;
}

static int run_noalloc(pp_handle* h, const HandleLaunchInfo& info, const pp_source* d_sources, const uint32_t* d_event_ids,
                       const uint32_t* d_source_ids, uint32_t n, pp_hit* d_hits, uint32_t ring_cap, size_t* n_hits_out,
                       uint64_t* photons_out, cudaStream_t st) {
  char msg[256];
  auto cuda_fail = [&](const char* what, cudaError_t e) {
    snprintf(msg, sizeof msg, "pp_run_resident_noalloc: %s: %s", what, cudaGetErrorString(e));
    return handle_fail(h, PP_E_CUDA, msg);
  };
  NoallocScratch* S = nullptr;  // DEVICE address: only ever used for address arithmetic on the host
  cudaError_t e = noalloc_scratch(info.device, &S);
  if (e != cudaSuccess) return cuda_fail("cudaGetSymbolAddress", e);
  // ---- a2: expansion into the static array; the host needs the totals before it can launch ----
  const uint32_t want_tiles = (uint32_t)info.grid * (uint32_t)(kBlockThreads / 32) * 4u;
  noalloc_prologue_kernel<<<1, 1024, 0, st>>>(S, d_sources, d_event_ids, d_source_ids, n, info.photons_per_GeV, want_tiles);
  g_launches++;
  e = cudaGetLastError();
  NoallocHead head{};
  if (e == cudaSuccess) e = cudaMemcpyAsync(&head, &S->head, sizeof head, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail("expansion", e);
  if (head.overflow) return handle_fail(h, PP_E_OVERFLOW, "pp_run_resident_noalloc: a source has more than 2^32-1 photons");
  if (head.too_big) {
    snprintf(msg, sizeof msg,
             "pp_run_resident_noalloc: the batch has %llu photons; the static scratch array is laid out for at most %u "
             "(PP_NOALLOC_MAX_PHOTONS): split the batch or use pp_run_resident",
             head.total, kNoallocMaxPhotons);
    return handle_fail(h, PP_E_NOMEM, msg);
  }
  if (photons_out) *photons_out = head.total;
  if (head.total == 0) return PP_OK;
  // ---- a3-a8: one propagation launch; the hit "ring" is the caller's buffer, and there are no resume lists: a
  // buffer that fills up makes the kernel stop and flag an error instead of handing work to a next launch ----
  LaunchParams P = info.base;
  P.src = S->src; P.cum = S->cum; P.cum_rel = S->cum_rel; P.tile_src = S->tile_src;
  P.g_begin = 0; P.g_end = head.total; P.n_src = n; P.n_tiles = head.n_tiles; P.tile_photons = head.tile_photons;
  P.has_segments = 0u;
  P.resume_in = nullptr; P.resume_out = nullptr; P.n_resume_in = 0; P.resume_cap = 0;
  P.status = &S->status; P.ring = d_hits; P.ring_cap = ring_cap;
  P.fates = nullptr;
  e = launch_propagate(P, info.brute, false, info.grid, info.smem, st);
  Status hs{};
  if (e == cudaSuccess) e = cudaMemcpyAsync(&hs, &S->status, sizeof hs, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail("propagation", e);
  if (hs.stop || hs.error || hs.hit_count > ring_cap) {
    *n_hits_out = hs.hit_count;
    snprintf(msg, sizeof msg,
             "pp_run_resident_noalloc: hit buffer too small: the batch makes at least %u hits, hit_cap is %u", hs.hit_count,
             ring_cap);
    return handle_fail(h, PP_E_NOMEM, msg);
  }
  if (hs.photons_started != head.total) return handle_fail(h, PP_E_CUDA, "pp_run_resident_noalloc: internal: photons lost");
  *n_hits_out = hs.hit_count;
  return PP_OK;
}

}  // namespace pp

extern "C" int pp_run_resident_noalloc(pp_handle* h, const pp_source* d_sources, const uint32_t* d_event_ids,
                                       const uint32_t* d_source_ids, size_t n, pp_hit* d_hits, size_t hit_cap,
                                       size_t* n_hits_out, uint64_t* photons_out, void* stream) {
  using namespace pp;
  if (!h || !n_hits_out) return PP_E_INVAL;
  *n_hits_out = 0;
  if (photons_out) *photons_out = 0;
  HandleLaunchInfo info;
  const int rc = handle_launch_info(h, &info);
  if (rc != PP_OK) return rc;
  if (n == 0) return PP_OK;
  if (!d_sources || !d_event_ids || !d_source_ids)
    return handle_fail(h, PP_E_INVAL, "pp_run_resident_noalloc: null device pointer (source ids are required here)");
  if ((hit_cap > 0 && !d_hits) || (reinterpret_cast<uintptr_t>(d_hits) & 15u))
    return handle_fail(h, PP_E_INVAL, "pp_run_resident_noalloc: d_hits is null or not 16-byte aligned");
  if (n > kNoallocMaxSrc) {
    char msg[200];
    snprintf(msg, sizeof msg,
             "pp_run_resident_noalloc: %zu sources; the static scratch array is laid out for at most %u "
             "(PP_NOALLOC_MAX_SOURCES): split the batch or use pp_run_resident", n, kNoallocMaxSrc);
    return handle_fail(h, PP_E_NOMEM, msg);
  }
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
  if (cudaSetDevice(info.device) != cudaSuccess) return handle_fail(h, PP_E_CUDA, "pp_run_resident_noalloc: cudaSetDevice");
  const uint32_t ring_cap = (uint32_t)(hit_cap < 0xFFFFFF00ull ? hit_cap : 0xFFFFFF00ull);
  const int out = run_noalloc(h, info, d_sources, d_event_ids, d_source_ids, (uint32_t)n, d_hits, ring_cap, n_hits_out,
                              photons_out, static_cast<cudaStream_t>(stream));
  if (prev >= 0 && prev != info.device) cudaSetDevice(prev);
  return out;
}
