// Records shared by the host side (pp_api.cpp) and the kernels (pp_kernels.cu) of the library.
// Not part of the public ABI.  Product code: shares nothing with oracle/.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

namespace pp {

// ---------------------------------------------------------------------------------------------
// Records shared between host and device code of the library (not part of the public ABI).
// ---------------------------------------------------------------------------------------------
struct __align__(16) SrcRec {  // 48 B: one light source as the kernels see it
  float x, y, z, dx;
  float dy, dz, t, energy;
  uint32_t event_id, source_id, n_photons;
  float length;  // metres; 0 = point source (R-18)
};

struct __align__(16) IceLayer {  // per-layer coefficients (1/m) and lengths (m)
  float a, b, la, lb;
};

struct __align__(16) StringRec {  // one vertical line of DOMs with uniform pitch
  float x, y, z0, pitch;          // z0 = z of DOM k = 0 (the highest); DOM k at z0 - k*pitch
  float inv_pitch;
  uint32_t n, base, pad;          // n DOMs; rows [base, base+n) of dom_xyzw
};

struct __align__(8) WorkItem {  // a range of batch-global photon numbers still to be run
  uint64_t g0, g1;
  uint32_t src, pad;
};

struct Status {                 // one per launch slot, device memory, copied back after every launch
  unsigned long long tile_counter;    // next fresh tile
  unsigned long long photons_started;
  unsigned long long photons_hit;
  unsigned long long photons_aborted;
  unsigned long long flights;
  unsigned long long photons_rejected;  // met a DOM, no photoelectron (acceptance)
  unsigned int hit_count;       // hits reserved in the ring this launch (may exceed ring_cap)
  unsigned int resume_counter;  // next resume_in item
  unsigned int n_resume_out;    // items written to resume_out
  unsigned int stop;            // set when the hit ring filled up
  unsigned int error;           // internal invariant broken (resume list overflow)
  unsigned int pad[3];
};

constexpr int kTilePhotons = 1024;  // photons per fresh work tile of a large launch (small launches use smaller tiles)
constexpr int kMinTilePhotons = 32;
constexpr int kMaxStringsSmem = 512;
constexpr float kPoleRho2 = 1e-10f;  // R-9
constexpr uint32_t kMaxWalkInv = 4096;  // entries per inverse walk table (device and shared memory)
constexpr uint16_t kNoString = 0xFFFFu;  // host-side marker while the cell table is built: no line within reach

// One record per layer boundary i (= upper edge of layer i), i = 0..n_layers; 32 B, shared memory (a4).
// The first half is layer i's coefficients, the second half the cumulative vertical optical depth at the boundary as
// two-float sums (B scattering, A absorption).  Record n_layers repeats the last layer's coefficients and holds +inf
// in the hi parts (only ever compared against).  A second array (LaunchParams::off_rec_b) pairs layer i's
// coefficients with the sums at its LOWER boundary i + 1 (record n_layers - 1 and n_layers: the finite sums of
// boundary n_layers - 1, never used for arithmetic), so that a flight reads the coefficients of a layer and the sums
// of the boundary it faces (start) or entered through (end) from ONE record: the first array going up at the start
// and down at the end, the second one otherwise.
struct __align__(16) LayerRec {
  float a, b;             // absorption and scattering coefficients, 1/m: what a flight needs where it starts ...
  float lb, a2;           // ... and where it ends: the scattering length (m) and the absorption coefficient again,
                          // so that either pair is one 8-byte load
  float Bh, Ah, Bl, Al;
};

// Everything a propagation launch needs.  Passed by value (kernel parameter space = constant bank).  The fields the
// loop touches every iteration sit in 16-byte groups so that one constant load fetches a group.
struct LaunchParams {
  // ---- hot groups (each 16 B, 16 B aligned) ----
  uint32_t rk[10][2];                                   // Philox round keys (5 groups)
  float hg_one_minus_g, hg_two_g, hg_one_minus_g2;      // 1-g, 2g, 1-g^2
  float one_minus_cos_c;                                // 1 - cos(theta_c)
  float z_top, inv_dz_layer, dz_layer;
  int32_t last_layer;                                   // n_layers - 1
  float k_b;                                            // inverse-table index = cumulative scattering depth * k_b
  uint32_t m_b;                                         // largest inverse-table index
  uint32_t off_inv_b, off_rec_b;                        // byte offsets into dynamic shared memory (layer records at 0)
  uint32_t off_str_xy, off_cell, pad0, pad1;
  float inv_cell, cell_ox, cell_oy;                     // cell coordinate = x * inv_cell + cell_ox
  float rm2;                                            // radius_margin^2 (pre-filter)
  uint32_t nx_m1, ny_m1, nx;
  float xy_cap2;                                        // (longest piece of flight looked up at once, xy)^2
  float inv_xy_cap;
  uint32_t max_flights;
  uint32_t ring_cap;
  uint32_t pad2;
  // ---- work ----
  const SrcRec* src;
  const unsigned long long* cum;  // [n_src + 1] exclusive prefix of n_photons (batch-global photon numbers)
  const uint32_t* cum_rel;        // [n_src + 1] cum[s] - g_begin as 32 bits: wraps below 0 (only the launch's first
                                  // source can be there, and it is never compared), saturates at 2^32 - 1 above
  const uint32_t* tile_src;       // [n_tiles] source holding the first photon of each tile
  unsigned long long g_begin, g_end;
  uint32_t n_src, n_tiles;
  uint32_t tile_photons;          // photons per fresh tile of this launch: kMinTilePhotons..kTilePhotons, a power of two
  uint32_t n_resume_in, resume_cap;
  const WorkItem* resume_in;
  WorkItem* resume_out;
  Status* status;
  void* ring;         // pp_hit[ring_cap]
  void* fates;        // pp_fate[g_end] or nullptr
  // ---- tables ----
  // Image of the shared-memory tables, copied verbatim into dynamic shared memory by every CTA (smem_image_bytes, a
  // multiple of 16): [LayerRec x (n_layers + 1)] [LayerRec x (n_layers + 1), second array] [u16 inv_b x (m_b + 1)]
  // [float2 line xy x (n_strings + 1)] [u16 cell x (nx ny)] [float4 line (x, y, z0, 1/pitch) x n_strings]
  // [uint2 line (n, base) x n_strings].
  //  * inv_b maps a quantised cumulative scattering depth to a layer j0 such that the layer holding that depth is j0
  //    or j0 + 1 (or beyond, when walk_loop is set for a coarse table).
  //  * cell table (a5): cell (ix, iy) of a uniform grid over the footprint names THE line of DOMs whose pre-filter disc
  //    can be met by a piece of flight whose xy midpoint lies in that cell; n_strings if none: that entry of the line
  //    xy table holds NaN, so the pre-filter fails without a branch.  Unique because a piece is at most xy_cap long in
  //    xy (longer flights are looked up piece by piece), and xy_cap < (smallest distance between two lines)
  //    - 2 radius_margin - cell diagonal; the outermost ring of cells is empty, so the cell index may simply be
  //    clamped into the grid.
  const uint4* smem_image;
  uint32_t smem_image_bytes;
  uint32_t walk_loop;        // the inverse walk tables are coarse (host: picks the kLoop kernel variant)
  uint32_t off_str_a, off_str_b;
  uint32_t n_layers;
  uint32_t n_strings, n_dom;
  const float4* dom_xyzw;    // [n_dom] sorted by (string, k); w = bit pattern of the public dom_id
  float radius, radius_margin;       // radius_margin = R + safety used by the pre-filter
  double inv_v;                                      // n_group / c  [ns/m]
  // ---- optional physics (kExt variant only) ----
  // DOM acceptance (pp_set_acceptance, R-17): mode 0 off, 1 probabilistic, 2 weighted
  uint32_t acc_mode, acc_n;
  // wavelength bins (pp_set_spectrum, R-21): 0 = monochromatic
  uint32_t spec_n;
  float spec_cdf[32], spec_inv_a[32], spec_inv_b[32], spec_acc[32];  // cumulative probability, 1/abs_scale, 1/scat_scale
  double spec_inv_v[32];                                             // n_group[j] / c  [ns/m]
  // angular smearing of the emission axis (pp_set_emission_smearing, R-22): HG constants 1-g, 2g, 1-g^2; off = 0
  uint32_t emit_on;
  float emit_one_minus_g, emit_two_g, emit_one_minus_g2;
  // longitudinal profile of extended sources (pp_set_segment_profile, R-23): knots of the inverse CDF; 0 = uniform
  uint32_t seg_n;
  float seg_tab[33];
  uint32_t has_segments;  // some source of this launch has length > 0 (R-18)
  float inv_c;            // 1 / c  [ns/m]
  float acc_coef[8];
};
static_assert(offsetof(LaunchParams, hg_one_minus_g) % 16 == 0 && offsetof(LaunchParams, z_top) % 16 == 0 &&
              offsetof(LaunchParams, k_b) % 16 == 0 && offsetof(LaunchParams, off_str_xy) % 16 == 0 &&
              offsetof(LaunchParams, inv_cell) % 16 == 0 && offsetof(LaunchParams, nx_m1) % 16 == 0 &&
              offsetof(LaunchParams, inv_xy_cap) % 16 == 0, "hot parameter groups must be 16-byte aligned");

}  // namespace pp
