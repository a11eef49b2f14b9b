// ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.  C entry points over oracle.hpp for ctypes
// (oracle/oracle.py).  See oracle.hpp for what each function computes and its citation.
#include <atomic>
#include <cstring>
#include <thread>

#include "oracle.hpp"

using namespace oracle;

extern "C" {

struct orc_ice {
  int32_t n_layers;
  double z_top, dz;
  const float* abs_len;
  const float* scat_len;
  double g, n_group, cos_cherenkov, photons_per_gev;
  int32_t effective_scattering, pad;
};

struct orc_geometry {
  int32_t n_dom;
  const float* xyz;
  double radius;
};

struct orc_hit {
  uint32_t event_id, source_id, photon_idx, dom_id;
  double time_ns;
  double weight;
};

struct orc_fate {
  int32_t fate, dom;
  uint32_t n_flights, pad;
  double x, y, z, time_ns, path_m;
  double dx, dy, dz;  // direction of the last flight
};

struct orc_stats {
  uint64_t photons, absorbed, hit, aborted, flights, rejected;
};

struct orc_job {
  orc_geometry geo;
  orc_ice ice;
  uint64_t seed;
  uint64_t n_sources;
  const float* src;            // [n_sources][8]
  const uint32_t* event_id;    // [n_sources]
  const uint32_t* source_id;   // [n_sources]
  const uint64_t* first;       // nullable: first photon index per source (default 0)
  const uint64_t* count;       // nullable: number of photon indices per source (default N_s - first)
  uint64_t stride, offset;     // photon i is run iff first <= i < first+count and i % stride == offset
  int32_t brute_force;         // 1: test every DOM; 0: exact vertical-line pre-filter
  int32_t real_type;           // 0: fp64 (the oracle); 1: fp32 (diagnostic only)
  int32_t n_threads;           // <= 0: hardware_concurrency
  int32_t pad;
  orc_hit* hits;               // out, capacity hit_cap
  uint64_t hit_cap;
  orc_fate* fates;             // nullable out, capacity fate_cap, in (source, photon) order
  uint64_t fate_cap;
  int32_t acc_mode;            // DOM acceptance (oracle.hpp, R-17): 0 off, 1 probabilistic, 2 weighted
  int32_t acc_n_coef;
  double acc_coef[8];
  const float* length;         // nullable: source lengths in metres (oracle.hpp, R-18); default 0 = point sources
  int32_t spec_n, pad2;        // wavelength bins (oracle.hpp, R-21); 0 = monochromatic
  const float* spec_cdf;
  const float* spec_abs_scale;
  const float* spec_scat_scale;
  const float* spec_n_group;
  const float* spec_acc_scale;
  double g_axis;               // angular smearing of the emission axis (oracle.hpp, R-22); 1 = off
  int32_t prof_n, pad3;        // longitudinal profile of extended sources (oracle.hpp, R-23); 0 = uniform
  const float* prof_f;
};

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
double orc_uniform(uint32_t w) { return uniform_from_word(w); }
uint64_t orc_photon_count(float e, float y) { return photon_count(e, y); }
double orc_hg_cos(double g, double u) { return hg_cos<double>(g, u); }
double orc_segment_fraction(const float* f, int32_t n, double u) {
  const SegmentProfile p{n, f};
  return segment_fraction(&p, u);
}
uint32_t orc_spectrum_word(const uint32_t* w) { return spectrum_word(w); }
double orc_acceptance(const double* coef, int32_t n_coef, double eta) {
  Acceptance a{1, n_coef, {0}};
  for (int k = 0; k < n_coef && k < 8; ++k) a.coef[k] = coef[k];
  return acceptance(a, eta);
}
void orc_rotate(const double* d, double cos_t, double phi, double* out) {
  double v[3] = {d[0], d[1], d[2]};
  rotate<double>(v, cos_t, phi);
  out[0] = v[0]; out[1] = v[1]; out[2] = v[2];
}

static Ice to_ice(const orc_ice* i) {
  return Ice{i->n_layers, i->z_top, i->dz, i->abs_len, i->scat_len, i->g, i->n_group, i->cos_cherenkov,
             i->photons_per_gev, i->effective_scattering};
}
static Geometry to_geo(const orc_geometry* g) { return Geometry{g->n_dom, g->xyz, g->radius}; }

int32_t orc_layer_of(const orc_ice* ice, double z) { return layer_of<double>(to_ice(ice), z); }
// which: 0 = scattering table, 1 = absorption table
double orc_walk(const orc_ice* ice, int32_t which, double z, double dir_z, double tau) {
  const Ice i = to_ice(ice);
  return walk<double>(i, which ? i.abs_len : i.scat_len, z, dir_z, tau);
}
double orc_depth(const orc_ice* ice, int32_t which, double z, double dir_z, double s) {
  const Ice i = to_ice(ice);
  return depth<double>(i, which ? i.abs_len : i.scat_len, z, dir_z, s);
}
int32_t orc_intersect(const orc_geometry* geo, int32_t brute, const double* p, const double* d, double s,
                      double* t_hit) {
  const Geometry g = to_geo(geo);
  if (brute) return intersect_brute<double>(g, p, d, s, t_hit);
  StringIndex idx(g);
  return intersect_lines<double>(g, idx, p, d, s, t_hit);
}

// Runs the selected photons of every source.  Returns the number of hits found (which may exceed
// hit_cap: only the first hit_cap, in (source order, photon_idx) order, are stored), or -1 on bad input.
int64_t orc_propagate(const orc_job* job, orc_stats* stats_out) {
  if (!job || job->stride == 0) return -1;
  const Geometry geo = to_geo(&job->geo);
  const Ice ice = to_ice(&job->ice);
  StringIndex idx(geo);
  const StringIndex* pidx = job->brute_force ? nullptr : &idx;
  if (job->acc_n_coef < 0 || job->acc_n_coef > 8 || job->acc_mode < 0 || job->acc_mode > 2) return -1;
  Acceptance acc{job->acc_mode, job->acc_n_coef, {0}};
  for (int k = 0; k < job->acc_n_coef; ++k) acc.coef[k] = job->acc_coef[k];
  if (job->spec_n < 0 || job->spec_n > 32 || job->prof_n < 0 || job->prof_n == 1 || job->prof_n > 33) return -1;
  const SegmentProfile prof{job->prof_n, job->prof_f};
  const Spectrum spec{job->spec_n, job->spec_cdf, job->spec_abs_scale, job->spec_scat_scale, job->spec_n_group,
                      job->spec_acc_scale};

  // flatten the selection into work units of (source, [lo, hi)) so threads can share big sources
  struct Unit { uint64_t s, lo, hi, fate_base; };
  std::vector<Unit> units;
  uint64_t n_sel = 0;
  const uint64_t chunk = 1 << 14;
  for (uint64_t s = 0; s < job->n_sources; ++s) {
    const uint64_t n_s = photon_count(job->src[8 * s + 7], float(ice.photons_per_gev));
    uint64_t lo = job->first ? job->first[s] : 0;
    uint64_t hi = job->count ? std::min(n_s, lo + job->count[s]) : n_s;
    if (lo >= hi) continue;
    // first selected index >= lo
    uint64_t i0 = lo + ((job->offset + job->stride - (lo % job->stride)) % job->stride);
    for (uint64_t a = i0; a < hi; a += chunk * job->stride) {
      const uint64_t b = std::min(hi, a + chunk * job->stride);
      units.push_back(Unit{s, a, b, n_sel});
      n_sel += (b - a + job->stride - 1) / job->stride;
    }
  }
  int nt = job->n_threads > 0 ? job->n_threads : int(std::thread::hardware_concurrency());
  if (nt < 1) nt = 1;
  std::atomic<size_t> next{0};
  std::vector<std::vector<orc_hit>> hits(nt);
  std::vector<orc_stats> st(nt);
  for (auto& x : st) std::memset(&x, 0, sizeof(x));
  auto worker = [&](int tid) {
    for (;;) {
      const size_t u = next.fetch_add(1);
      if (u >= units.size()) break;
      const Unit& un = units[u];
      uint64_t fi = un.fate_base;
      for (uint64_t i = un.lo; i < un.hi; i += job->stride, ++fi) {
        const float* src = job->src + 8 * un.s;
        const uint32_t ev = job->event_id[un.s], sid = job->source_id[un.s];
        const float len = job->length ? job->length[un.s] : 0.0f;
        PhotonResult r = job->real_type == 1
                             ? propagate_photon<float>(geo, pidx, ice, job->seed, src, ev, sid, uint32_t(i), &acc, len, &spec, job->g_axis, &prof)
                             : propagate_photon<double>(geo, pidx, ice, job->seed, src, ev, sid, uint32_t(i), &acc, len, &spec, job->g_axis, &prof);
        st[tid].photons++;
        st[tid].flights += r.n_flights;
        if (r.fate == kAbsorbed) st[tid].absorbed++;
        else if (r.fate == kHit) { st[tid].hit++; hits[tid].push_back(orc_hit{ev, sid, uint32_t(i), uint32_t(r.dom), r.time_ns, r.weight}); }
        else if (r.fate == kRejected) st[tid].rejected++;
        else st[tid].aborted++;
        if (job->fates && fi < job->fate_cap) {
          orc_fate& f = job->fates[fi];
          f.fate = r.fate; f.dom = r.dom; f.n_flights = r.n_flights; f.pad = 0;
          f.x = r.x; f.y = r.y; f.z = r.z; f.time_ns = r.time_ns; f.path_m = r.path_m;
          f.dx = r.dx; f.dy = r.dy; f.dz = r.dz;
        }
      }
    }
  };
  std::vector<std::thread> th;
  for (int t = 1; t < nt; ++t) th.emplace_back(worker, t);
  worker(0);
  for (auto& t : th) t.join();

  std::vector<orc_hit> all;
  orc_stats tot;
  std::memset(&tot, 0, sizeof(tot));
  for (int t = 0; t < nt; ++t) {
    all.insert(all.end(), hits[t].begin(), hits[t].end());
    tot.photons += st[t].photons; tot.absorbed += st[t].absorbed; tot.hit += st[t].hit;
    tot.aborted += st[t].aborted; tot.flights += st[t].flights; tot.rejected += st[t].rejected;
  }
  std::sort(all.begin(), all.end(), [](const orc_hit& a, const orc_hit& b) {
    if (a.event_id != b.event_id) return a.event_id < b.event_id;
    if (a.source_id != b.source_id) return a.source_id < b.source_id;
    return a.photon_idx < b.photon_idx;
  });
  const uint64_t n_copy = std::min<uint64_t>(all.size(), job->hit_cap);
  if (n_copy && job->hits) std::memcpy(job->hits, all.data(), n_copy * sizeof(orc_hit));
  if (stats_out) *stats_out = tot;
  return int64_t(all.size());
}

}  // extern "C"
