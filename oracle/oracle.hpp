// ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow, obviously-correct CPU implementation of the photon-propagation hot path of
// arXiv:2405.05700 (layered ice, "calculate the distance to the next scatter
// for each photon and then picking a new angle based on the physics of scattering ... repeated
// until the photon intersects a detector or is absorbed").  It follows the algorithm step by
// step in the order of DESIGN.md section 2 ("The path, step by step"); every function cites
// the passage / reading it implements.  fp64 throughout (the template parameter exists only so
// that an fp32 instantiation can be used to *diagnose* mismatches; parity is always against
// Real = double).
//
// Independence: this file shares NO code with paper_2405_05700_b200/csrc (own Philox, own
// geometry handling, own everything) and is never linked into or called by the product.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may use it.
//
// Parity pins (tests/test_oracle_*.py, all -m "not gpu"):
//   philox4x32_10        published known-answer vectors (tests/golden/philox_kat.txt)
//   uniform_from_word    closed form; range/never 0 or 1
//   photon_count         closed form
//   hg_cos               <cos> = g, <cos^2> = (1+2g^2)/3 by quadrature; g=0 uniform; analytic CDF inverse
//   rotate               unit output, d'.d = cos(theta), azimuth uniformity, pole branch limit
//   walk / depth         piecewise closed form on a hand-built 3-layer table; walk(depth(s)) = s
//   intersect_*          analytic chord through a sphere; brute force == string pre-filter
//   propagate            homogeneous-ice closed forms (segments ~ Geom, path ~ Exp(lambda_a),
//                        <displacement> = 1/(a+b(1-g))), unscattered survival exp(-(d-R)(a+b)),
//                        arrival time (d-R)/v, causality, conservation
//   propagate, step 8 in LAYERED ice with scattering on (absorption budget carried across flights and layers)
//                        g -> 1 vertical beam: total path over many flights ~ 1 - exp(-sum a_i dz_i) from the table only;
//                        abs_len = 4 scat_len in every layer: flights per photon geometric with mean exactly 5
//   acceptance / propagate with acceptance (NEXT-1, R-17)
//                        polynomial values by hand; photons started inside a DOM: accepted fraction = p(cos theta_c)
//                        and every weight = p(cos theta_c); pencil beam: hit fraction = survival x p(d_z);
//                        weighted and probabilistic modes agree in expectation; mode 0 unchanged
//   propagate with a source length (NEXT-2, R-18)
//                        beam along the axis at a DOM ahead: hit fraction (lambda/L) e^{-(D-R)/lambda} (e^{L/lambda} - 1),
//                        arrival times l/c + (D-R-l)/v and the mean emission offset of the hits; mean end-point
//                        displacement L/2 + 1/(a+b(1-g)); L = 0 is the point source bit for bit
//   effective scattering lengths (NEXT-2, R-20): table 200 m at g = 0.875 == table 25 m geometric, bit for bit;
//                        mean displacement 1/(a + 1/lambda_e)
//   wavelength bins (NEXT-2, R-21): one bin with unit scales == monochromatic bit for bit; two bins: bin frequencies,
//                        mean path sum_j w_j lambda_a / abs_scale_j, flights per photon per bin, two arrival times
//                        (d-R) n_j / c at a DOM with frequencies ~ w_j exp(-(d-R) a_j)
//   angular smearing (NEXT-2, R-22): <cos> and <P2> of the emission angle about the source axis are
//                        g cos(theta_c) and g^2 P2(cos theta_c) (Legendre moments multiply); azimuthal symmetry;
//                        g_axis = 1 == exact cone bit for bit
//   longitudinal profile (NEXT-2, R-23): table values by hand; mean and variance of the emission offset for a
//                        triangular-density table; identity table == no table to rounding
//   full layered C1-C4 hit lists: PARITY UNPINNED by anything external (no published values);
//                        pinned only through the invariants above.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <limits>
#include <vector>

namespace oracle {

// ------------------------------------------------------------------------------------------
// Random numbers: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), reading R-3.
// ------------------------------------------------------------------------------------------
inline void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c[4] = {ctr_in[0], ctr_in[1], ctr_in[2], ctr_in[3]};
  uint32_t k[2] = {key_in[0], key_in[1]};
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = M0 * c[0];
    const uint64_t p1 = M1 * c[2];
    const uint32_t hi0 = uint32_t(p0 >> 32), lo0 = uint32_t(p0);
    const uint32_t hi1 = uint32_t(p1 >> 32), lo1 = uint32_t(p1);
    const uint32_t n0 = hi1 ^ c[1] ^ k[0];
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c[3] ^ k[1];
    const uint32_t n3 = lo0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
    k[0] += W0; k[1] += W1;
  }
  out[0] = c[0]; out[1] = c[1]; out[2] = c[2]; out[3] = c[3];
}

// u = (x >> 9) * 2^-23 + 2^-24: 23 random bits, exactly representable in fp32, in
// [2^-24, 1 - 2^-24], never 0 or 1 (R-3).
inline double uniform_from_word(uint32_t x) {
  return double(x >> 9) * (1.0 / 8388608.0) + (1.0 / 16777216.0);
}

// Step 1 (R-12b): N_s = floor(double(E) * double(yield) + 0.5).
inline uint64_t photon_count(float energy_gev, float photons_per_gev) {
  const double n = std::floor(double(energy_gev) * double(photons_per_gev) + 0.5);
  return n <= 0.0 ? 0 : uint64_t(n);
}

// ------------------------------------------------------------------------------------------
// Inputs
// ------------------------------------------------------------------------------------------
struct Ice {
  int n_layers;
  double z_top;  // upper edge of layer 0 (z up)
  double dz;     // layer thickness (10 m)
  const float* abs_len;   // [n_layers] metres
  const float* scat_len;  // [n_layers] metres, geometric mean free path (R-7)
  double g, n_group, cos_cherenkov, photons_per_gev;
  // NEXT-2 option (R-20): scat_len holds EFFECTIVE scattering lengths lambda_e = lambda_s / (1 - g), the
  // convention of measured ice tables; the geometric mean free path of R-7 is then lambda_e (1 - g).
  int effective_scattering = 0;
};

struct Geometry {
  int n_dom;
  const float* xyz;  // [n_dom][3]
  double radius;
};

constexpr double kC = 0.299792458;  // m/ns

// ------------------------------------------------------------------------------------------
// Step 9a: Henyey-Greenstein inverse CDF (R-1).  u -> 1 is forward.
// ------------------------------------------------------------------------------------------
template <class Real>
inline Real hg_cos(Real g, Real u) {
  if (g == Real(0)) return Real(2) * u - Real(1);
  const Real q = (Real(1) - g * g) / (Real(1) - g + Real(2) * g * u);
  Real c = (Real(1) + g * g - q * q) / (Real(2) * g);
  return std::min(Real(1), std::max(Real(-1), c));
}

// ------------------------------------------------------------------------------------------
// Step 2 / 9b: rotate unit vector d by polar angle theta (given as cos) and azimuth phi about
// itself, then renormalise (R-9, pinned azimuth reference).
// ------------------------------------------------------------------------------------------
template <class Real>
inline void rotate(Real d[3], Real cos_t, Real phi) {
  const Real sin_t = std::sqrt(std::max(Real(0), (Real(1) - cos_t) * (Real(1) + cos_t)));
  const Real cp = std::cos(phi), sp = std::sin(phi);
  const Real rho2 = d[0] * d[0] + d[1] * d[1];
  Real n[3];
  if (rho2 > Real(1e-10)) {
    const Real rho = std::sqrt(rho2);
    n[0] = d[0] * cos_t + sin_t * (d[0] * d[2] * cp - d[1] * sp) / rho;
    n[1] = d[1] * cos_t + sin_t * (d[1] * d[2] * cp + d[0] * sp) / rho;
    n[2] = d[2] * cos_t - sin_t * cp * rho;
  } else {
    n[0] = sin_t * cp;
    n[1] = sin_t * sp;
    n[2] = (d[2] >= Real(0) ? Real(1) : Real(-1)) * cos_t;
  }
  const Real norm = std::sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
  d[0] = n[0] / norm; d[1] = n[1] / norm; d[2] = n[2] / norm;
}

// ------------------------------------------------------------------------------------------
// Step 6: layer walk (R-6).  Layer index of height z; the end layers extend to infinity.
// ------------------------------------------------------------------------------------------
template <class Real>
inline int layer_of(const Ice& ice, Real z) {
  const Real f = std::floor((Real(ice.z_top) - z) / Real(ice.dz));
  if (f <= Real(0)) return 0;
  if (f >= Real(ice.n_layers - 1)) return ice.n_layers - 1;
  return int(f);
}

// Distance s along a ray starting at height z with direction cosine dir_z at which the optical
// depth  integral_0^s c(z(s')) ds'  reaches tau, with c_i = 1/len[i] per layer.
template <class Real>
inline Real walk(const Ice& ice, const float* len, Real z, Real dir_z, Real tau) {
  int i = layer_of(ice, z);
  Real s = 0;
  const Real inf = std::numeric_limits<Real>::infinity();
  for (;;) {
    const Real c = Real(1) / Real(len[i]);
    Real l = inf;  // distance to the next horizontal boundary along the ray
    if (dir_z > Real(0) && i > 0) {
      const Real zb = Real(ice.z_top) - Real(i) * Real(ice.dz);  // upper edge of layer i
      l = std::max(Real(0), (zb - z) / dir_z);
    } else if (dir_z < Real(0) && i < ice.n_layers - 1) {
      const Real zb = Real(ice.z_top) - Real(i + 1) * Real(ice.dz);  // lower edge of layer i
      l = std::max(Real(0), (zb - z) / dir_z);
    }
    if (tau <= c * l) return s + tau / c;
    tau -= c * l;
    s += l;
    z += dir_z * l;
    i += (dir_z > Real(0)) ? -1 : 1;
  }
}

// Optical depth  integral_0^s c(z(s')) ds'  along the same ray (step 8: absorption budget used
// up by a flight of length s).
template <class Real>
inline Real depth(const Ice& ice, const float* len, Real z, Real dir_z, Real s) {
  int i = layer_of(ice, z);
  Real tau = 0;
  const Real inf = std::numeric_limits<Real>::infinity();
  for (;;) {
    const Real c = Real(1) / Real(len[i]);
    Real l = inf;
    if (dir_z > Real(0) && i > 0) {
      l = std::max(Real(0), (Real(ice.z_top) - Real(i) * Real(ice.dz) - z) / dir_z);
    } else if (dir_z < Real(0) && i < ice.n_layers - 1) {
      l = std::max(Real(0), (Real(ice.z_top) - Real(i + 1) * Real(ice.dz) - z) / dir_z);
    }
    if (s <= l) return tau + c * s;
    tau += c * l;
    s -= l;
    z += dir_z * l;
    i += (dir_z > Real(0)) ? -1 : 1;
  }
}

// ------------------------------------------------------------------------------------------
// Step 7: first point of the flight [0, s] that lies in the closed ball of a DOM (R-5, R-8).
// Returns true and t_hit if the ball |x - c| <= R meets the segment.
// ------------------------------------------------------------------------------------------
template <class Real>
inline bool hit_sphere(const Real p[3], const Real d[3], Real s, const Real c[3], Real R, Real* t_hit) {
  const Real oc[3] = {p[0] - c[0], p[1] - c[1], p[2] - c[2]};
  const Real b = oc[0] * d[0] + oc[1] * d[1] + oc[2] * d[2];
  const Real perp[3] = {oc[0] - b * d[0], oc[1] - b * d[1], oc[2] - b * d[2]};  // closest approach vector
  const Real disc = R * R - (perp[0] * perp[0] + perp[1] * perp[1] + perp[2] * perp[2]);
  if (disc < Real(0)) return false;  // tangent (disc == 0) counts as a hit (R-8b)
  const Real h = std::sqrt(disc);
  const Real t_in = -b - h, t_out = -b + h;
  if (t_out < Real(0) || t_in > s) return false;
  *t_hit = std::max(Real(0), t_in);  // start inside a DOM: hit at distance 0 (R-5)
  return true;
}

// Brute force over every DOM: smallest t_hit, ties to the smaller dom id.
template <class Real>
inline int intersect_brute(const Geometry& geo, const Real p[3], const Real d[3], Real s, Real* t_best) {
  int best = -1;
  Real tb = std::numeric_limits<Real>::infinity();
  for (int j = 0; j < geo.n_dom; ++j) {
    const Real c[3] = {Real(geo.xyz[3 * j]), Real(geo.xyz[3 * j + 1]), Real(geo.xyz[3 * j + 2])};
    Real t;
    if (hit_sphere(p, d, s, c, Real(geo.radius), &t) && t < tb) { tb = t; best = j; }
  }
  *t_best = tb;
  return best;
}

// Exact pre-filter: DOMs are grouped into vertical lines of equal (x, y);
// a line whose axis is farther than R from the xy-projection of the flight cannot hold a hit
// DOM, so its DOMs are skipped.  Tested identical to brute force (tests/test_oracle_geometry.py).
struct StringIndex {
  struct Line { double x, y; std::vector<int> doms; };
  std::vector<Line> lines;
  explicit StringIndex(const Geometry& geo) {
    for (int j = 0; j < geo.n_dom; ++j) {
      const double x = geo.xyz[3 * j], y = geo.xyz[3 * j + 1];
      bool found = false;
      for (auto& l : lines)
        if (l.x == x && l.y == y) { l.doms.push_back(j); found = true; break; }
      if (!found) lines.push_back(Line{x, y, {j}});
    }
  }
};

template <class Real>
inline int intersect_lines(const Geometry& geo, const StringIndex& idx, const Real p[3], const Real d[3], Real s,
                           Real* t_best) {
  int best = -1;
  Real tb = std::numeric_limits<Real>::infinity();
  const Real R = Real(geo.radius);
  // xy-projection of the flight: q(t) = p_xy + t d_xy, t in [0, s]; distance from the axis point a
  const Real ex = d[0] * s, ey = d[1] * s;
  const Real e2 = ex * ex + ey * ey;
  for (const auto& l : idx.lines) {
    const Real ax = Real(l.x) - p[0], ay = Real(l.y) - p[1];
    Real f = e2 > Real(0) ? (ax * ex + ay * ey) / e2 : Real(0);
    f = std::min(Real(1), std::max(Real(0), f));
    const Real rx = ax - f * ex, ry = ay - f * ey;
    // small safety margin so that rounding in this filter can never reject a true hit
    if (rx * rx + ry * ry > (R * Real(1.0001) + Real(1e-9)) * (R * Real(1.0001) + Real(1e-9))) continue;
    for (int j : l.doms) {
      const Real c[3] = {Real(geo.xyz[3 * j]), Real(geo.xyz[3 * j + 1]), Real(geo.xyz[3 * j + 2])};
      Real t;
      if (hit_sphere(p, d, s, c, R, &t) && (t < tb || (t == tb && j < best))) { tb = t; best = j; }
    }
  }
  *t_best = tb;
  return best;
}

// ------------------------------------------------------------------------------------------
// One photon, steps 2-10.
// ------------------------------------------------------------------------------------------
enum Fate : int { kAbsorbed = 0, kHit = 1, kAborted = 2, kRejected = 3 };

// ------------------------------------------------------------------------------------------
// DOM acceptance (NEXT-1; "When a photon intersects a detector, it creates a photoelectron
// with a probability calculated from its position, direction, time, and wavelength"; the
// hit record carries a weight).  Reading R-17: the probability depends on the arrival
// direction only, p(eta) = clamp(sum_k c_k eta^k, 0, 1) with eta = d_z, the cosine between the photon's
// travel direction at the intersection and +z (the PMT looks down, so an upgoing photon meets its face).
//   mode 0: every intersection is a hit of weight 1 (acceptance off).
//   mode 1 (probabilistic): one more uniform, word 0 of Philox block (photon, source, event, 2^31 | k) for an
//           intersection on flight k; hit of weight 1 iff u < p(eta), otherwise the photon ends in the DOM
//           without a photoelectron (kRejected).
//   mode 2 (weighted): no draw; hit of weight p(eta) iff p(eta) > 0, otherwise kRejected.
// Either way the photon stops at the DOM (R-8).
// ------------------------------------------------------------------------------------------
struct Acceptance {
  int mode;
  int n_coef;
  double coef[8];
};

inline double acceptance(const Acceptance& acc, double eta) {
  double p = 0, x = 1;
  for (int k = 0; k < acc.n_coef; ++k) { p += acc.coef[k] * x; x *= eta; }
  return std::min(1.0, std::max(0.0, p));
}

// ------------------------------------------------------------------------------------------
// Wavelength bins (NEXT-2; the photoelectron probability depends on "position, direction, time, and
// wavelength"; the optical properties vary).  Reading R-21: a photon belongs to one of
// n <= 32 wavelength bins for its whole life, bin j = the first with cdf[j] > u, u = the uniform of the word made of
// the low 9 bits of words 0, 1, 2 of the photon's Philox block 0 (spectrum_word); in bin j the absorption and scattering coefficients of every layer are multiplied by
// abs_scale[j] and scat_scale[j], the group index is n_group[j], and the acceptance probability becomes
// min(1, p(eta) acc_scale[j]).  n = 0: monochromatic (R-4b).
// ------------------------------------------------------------------------------------------
struct Spectrum {
  int n;
  const float* cdf;         // [n] cumulative bin probabilities, non-decreasing, cdf[n-1] >= 1
  const float* abs_scale;   // [n] > 0
  const float* scat_scale;  // [n] > 0
  const float* n_group;     // [n] >= 1
  const float* acc_scale;   // [n] >= 0
};

// The wavelength draw costs no extra Philox block: a uniform takes the top 23 bits of its word (R-3), so the low 9
// bits of the words of block 0 are unused; the low 9 bits of words 0, 1, 2 make the word of the wavelength uniform.
inline uint32_t spectrum_word(const uint32_t w[4]) {
  return ((w[0] & 0x1FFu) << 23) | ((w[1] & 0x1FFu) << 14) | ((w[2] & 0x1FFu) << 5);
}

inline int spectrum_bin(const Spectrum& sp, double u) {
  int j = 0;
  while (j + 1 < sp.n && !(double(sp.cdf[j]) > u)) ++j;
  return j;
}

// ------------------------------------------------------------------------------------------
// Longitudinal profile of an extended source (NEXT-2, R-23): where along its length a source of length L emits.
// The offset is L F(u), u the uniform of R-18, F piecewise linear through n knots f[0..n-1] at u = i/(n-1)
// (an inverse cumulative distribution given as a table: no rejection sampling, one uniform).  No table: F(u) = u,
// the uniform segment of R-18.
// ------------------------------------------------------------------------------------------
struct SegmentProfile {
  int n;           // knots, 0 or 2..33
  const float* f;  // [n] non-decreasing, in [0, 1]
};

inline double segment_fraction(const SegmentProfile* p, double u) {
  if (!p || p->n < 2) return u;
  const double x = u * double(p->n - 1);
  int i = int(x);
  if (i > p->n - 2) i = p->n - 2;
  const double t = x - double(i);
  return double(p->f[i]) + t * (double(p->f[i + 1]) - double(p->f[i]));
}

struct PhotonResult {
  double weight;      // hit weight (1 unless the acceptance is in weighted mode)
  int fate;
  int dom;            // hit DOM or -1
  uint32_t n_flights;  // number of flights (segments) started
  double x, y, z;     // end point
  double dx, dy, dz;  // direction of the last flight (diagnostics: incidence angle at a DOM)
  double time_ns;     // end time (hit time if fate == kHit)
  double path_m;      // total geometric path
};

constexpr uint32_t kMaxFlights = 100000;  // R-10

template <class Real>
inline PhotonResult propagate_photon(const Geometry& geo, const StringIndex* idx, const Ice& ice, uint64_t seed,
                                     const float src[8], uint32_t event_id, uint32_t source_id,
                                     uint32_t photon_idx, const Acceptance* acc = nullptr, float length = 0.0f,
                                     const Spectrum* spec = nullptr, double g_axis = 1.0,
                                     const SegmentProfile* prof = nullptr) {
  const uint32_t key[2] = {uint32_t(seed), uint32_t(seed >> 32)};
  // R-21: the photon's wavelength bin fixes its coefficient scales and its group index
  Real sc_a = 1, sc_b = 1, sc_acc = 1;
  double n_group = ice.n_group;
  if (spec && spec->n > 0) {
    const uint32_t sctr[4] = {photon_idx, source_id, event_id, 0u};
    uint32_t sw[4];
    philox4x32_10(sctr, key, sw);
    const int j = spectrum_bin(*spec, uniform_from_word(spectrum_word(sw)));
    sc_a = Real(spec->abs_scale[j]); sc_b = Real(spec->scat_scale[j]); sc_acc = Real(spec->acc_scale[j]);
    n_group = double(spec->n_group[j]);
  }
  const Real v = Real(kC / n_group);  // group velocity, m/ns
  const Real two_pi = Real(6.283185307179586476925286766559);
  Real p[3] = {Real(src[0]), Real(src[1]), Real(src[2])};
  Real d[3] = {Real(src[3]), Real(src[4]), Real(src[5])};  // source axis; rotated below (step 2)
  double t = double(src[6]);  // time and path are kept in fp64 even in the fp32 diagnostic instantiation
  double path = 0;
  Real tau_a = 0;
  PhotonResult r{};
  r.dom = -1;
  for (uint32_t k = 0;; ++k) {
    if (k >= kMaxFlights) { r.fate = kAborted; break; }  // step 10
    // R-3: Philox block k of this photon serves flight k: words -> (azimuth, HG, distance, absorption)
    const uint32_t ctr[4] = {photon_idx, source_id, event_id, k};
    uint32_t w[4];
    philox4x32_10(ctr, key, w);
    const Real u_az = Real(uniform_from_word(w[0])), u_hg = Real(uniform_from_word(w[1]));
    const Real u_dist = Real(uniform_from_word(w[2])), u_abs = Real(uniform_from_word(w[3]));
    Real cos_t;
    if (k == 0) {
      // R-18 (NEXT-2, track segments: PAPER.md:29 continuous losses, "photon emitting steps"): a source of
      // length L > 0 emits from a point uniform on [0, L] along its axis, at the time the muon (speed c, R-11b) is
      // there; the offset uses the word of block 0 that flight 0 leaves unused (u_hg).  L = 0: point cascade (R-4).
      if (length > 0.0f) {
        const Real ell = Real(segment_fraction(prof, double(u_hg))) * Real(length);
        for (int a = 0; a < 3; ++a) p[a] += d[a] * ell;  // d is still the source axis here
        t += double(ell) / kC;
      }
      // R-22 (NEXT-2, angular smearing; the light of a cascade comes from its secondaries, "parameterized
      // light yields"): with g_axis < 1 the axis the photon is emitted about is the source axis deflected by a polar
      // angle drawn from the Henyey-Greenstein law of parameter g_axis and a uniform azimuth -- words 0 and 1 of Philox
      // block (photon, source, event, 2^29).  g_axis = 1: the exact cone of R-4.
      if (g_axis < 1.0) {
        const uint32_t ectr[4] = {photon_idx, source_id, event_id, 0x20000000u};
        uint32_t ew[4];
        philox4x32_10(ectr, key, ew);
        rotate(d, hg_cos(Real(g_axis), Real(uniform_from_word(ew[0]))), two_pi * Real(uniform_from_word(ew[1])));
      }
      cos_t = Real(ice.cos_cherenkov);  // step 2: emission on the Cherenkov cone about the source axis (R-4)
      tau_a = -std::log(u_abs);         // step 3: absorption budget, drawn once per photon
    } else {
      cos_t = hg_cos(Real(ice.g), u_hg);  // step 9: scatter at the end of flight k-1
    }
    rotate(d, cos_t, two_pi * u_az);
    r.n_flights = k + 1;
    // step 5/6: distance to the next scatter and to the absorption point
    // R-20: with effective scattering lengths b = 1/(lambda_e (1-g)), so the optical depth along the lambda_e table
    // that corresponds to tau_s is tau_s (1 - g)
    const Real tau_s = -std::log(u_dist) * (ice.effective_scattering ? Real(1.0 - ice.g) : Real(1));
    // R-21: coefficients scaled by sc <=> optical depth along the unscaled table divided by sc
    const Real s_scat = walk(ice, ice.scat_len, p[2], d[2], tau_s / sc_b);
    const Real s_abs = walk(ice, ice.abs_len, p[2], d[2], tau_a / sc_a);
    const bool absorbed = (s_abs <= s_scat);
    const Real s = absorbed ? s_abs : s_scat;
    // step 7: first DOM met on [0, s]
    Real t_hit;
    const int dom = idx ? intersect_lines(geo, *idx, p, d, s, &t_hit) : intersect_brute(geo, p, d, s, &t_hit);
    if (dom >= 0) {
      for (int a = 0; a < 3; ++a) p[a] += d[a] * t_hit;
      path += double(t_hit);
      t += double(t_hit) / double(v);
      r.fate = kHit; r.dom = dom; r.weight = 1.0;
      if (acc && acc->mode != 0) {  // R-17
        const double pa = std::min(1.0, acceptance(*acc, double(d[2])) * double(sc_acc));
        if (acc->mode == 1) {
          const uint32_t actr[4] = {photon_idx, source_id, event_id, 0x80000000u | k};
          uint32_t aw[4];
          philox4x32_10(actr, key, aw);
          if (!(uniform_from_word(aw[0]) < pa)) r.fate = kRejected;
        } else {
          r.weight = pa;
          if (!(pa > 0.0)) r.fate = kRejected;
        }
      }
      break;
    }
    // step 8: advance
    tau_a -= depth(ice, ice.abs_len, p[2], d[2], s) * sc_a;
    for (int a = 0; a < 3; ++a) p[a] += d[a] * s;
    path += double(s);
    t += double(s) / double(v);
    if (absorbed) { r.fate = kAbsorbed; break; }
  }
  r.x = double(p[0]); r.y = double(p[1]); r.z = double(p[2]);
  r.dx = double(d[0]); r.dy = double(d[1]); r.dz = double(d[2]);
  r.time_ns = double(t);
  r.path_m = double(path);
  return r;
}

}  // namespace oracle
