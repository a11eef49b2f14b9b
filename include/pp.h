/*
 * pp.h -- C ABI of the B200-native photon propagator ("pp"), the GPU photon-propagation stage of
 * arXiv:2405.05700 plus the server-side batching that feeds it.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md):
 *   - light sources: "These losses in the detector volume are then used as light sources for the
 *     photon propagator" (section 2);
 *   - medium: "The optical properties of the ice are divided into vertical layers of 10 m thickness
 *     having different coefficients of scattering and absorption";
 *   - photon loop: "calculate the distance to the next scatter for each photon and then picking a new
 *     angle based on the physics of scattering. This process is then repeated until the photon
 *     intersects a detector or is absorbed";
 *   - batching: "When the step queue is sufficiently full, a block of steps is sent to the propagation
 *     server for processing as a batch. The server aggregates steps from multiple events and clients
 *     in order to keep the GPU as busy as possible" (section 4);
 *   - hit record: "only stores the ID of the particle that produced it, the time of the hit, and the
 *     weight";
 *   - many producers, one server: "multiple instances of IceTray ... sharing a single photon propagator
 *     server".
 * Everything the paper leaves open is fixed by the readings R-1..R-23 in DESIGN.md section 3.
 *
 * Conventions: metres, nanoseconds, GeV; z up.  All pointers are HOST pointers unless the parameter
 * name starts with d_ (DEVICE pointer).  The caller owns every pointer it passes; the library copies
 * what it needs before the call returns unless stated otherwise.  Every call returns PP_OK (0) or a
 * negative pp_status; no exceptions cross the boundary; after PP_E_CUDA the handle is poisoned (every
 * later call returns PP_E_CUDA) and pp_last_error() gives the CUDA message.  There is no CPU fallback:
 * without a CUDA device pp_create fails with PP_E_CUDA.
 */
#ifndef PP_H_
#define PP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum pp_status {
  PP_OK = 0,
  PP_E_INVAL = -1,       /* bad argument (NULL, NaN, non-unit direction, non-positive length, ...) */
  PP_E_NOMEM = -2,       /* workspace too small / allocation failed */
  PP_E_CUDA = -3,        /* CUDA error (sticky) */
  PP_E_OVERFLOW = -4,    /* a per-source photon count does not fit 32 bits */
  PP_E_WOULDBLOCK = -5,  /* non-blocking call could not make progress */
  PP_E_UNSUPPORTED = -6, /* geometry the fast DOM lookup cannot represent (see pp_geometry) */
  PP_E_STATE = -7        /* call not valid in this state (e.g. submit after shutdown) */
} pp_status;

/* A light source ("photon emitting step"): a point cascade that emits
 * N = floor(double(energy_GeV) * double(photons_per_GeV) + 0.5) photons at (x,y,z), time t_ns, on the
 * Cherenkov cone about the unit axis (dx,dy,dz) (R-4, R-12b).  32 bytes. */
typedef struct pp_source {
  float x, y, z;
  float dx, dy, dz;
  float t_ns;
  float energy_GeV;
} pp_source;

/* A hit (producing particle, time, weight).  The producing photon is identified by the
 * Philox counter triple (event_id, source_id, photon_idx), which lets any hit be replayed in isolation;
 * a single 32-bit photon id would overflow for one C4-size event (5e9 photons).  32 bytes. */
typedef struct pp_hit {
  uint32_t event_id;
  uint32_t source_id;
  uint32_t photon_idx; /* index of the photon within its source, 0 <= photon_idx < N */
  uint32_t dom_id;     /* row index into pp_geometry.xyz */
  double time_ns;      /* source time (+ emission delay along a segment, R-18) + path / group velocity */
  float weight;        /* 1.0 unless pp_set_acceptance is in weighted mode (R-4b, R-17) */
  uint32_t n_scatter;  /* number of scatters before the hit (diagnostic; 0 = direct light) */
} pp_hit;

/* Detector geometry: n_dom spheres of one radius.  dom_id = row index.  The fast lookup needs DOMs
 * that sit on vertical lines (equal x,y) with a uniform z pitch per line (R-11); anything else makes
 * pp_create return PP_E_UNSUPPORTED unless PP_FLAG_BRUTE_FORCE_DOMS is set. */
typedef struct pp_geometry {
  uint32_t n_dom;
  const float* xyz; /* [n_dom][3] */
  float radius;     /* metres, > 0 */
} pp_geometry;

/* Layered ice.  Layer i spans z in (z_top-(i+1)*dz, z_top-i*dz]; layer 0 extends to
 * +infinity and layer n_layers-1 to -infinity (R-6).  Lengths in metres; scat_len is the geometric
 * mean free path between scatters (R-7) unless PP_FLAG_EFFECTIVE_SCATTERING is set (R-20). */
typedef struct pp_ice {
  uint32_t n_layers;     /* 1..PP_MAX_LAYERS */
  float z_top;
  float dz;
  const float* abs_len;  /* [n_layers] > 0 */
  const float* scat_len; /* [n_layers] > 0 */
  float g;               /* Henyey-Greenstein asymmetry, |g| < 1 (R-1) */
  float n_group;         /* group index; photon speed = c / n_group */
  float cos_cherenkov;   /* cosine of the emission cone half-angle, in [-1, 1] */
  float photons_per_GeV; /* light yield */
} pp_ice;

#define PP_MAX_LAYERS 1024u

/* pp_config.flags */
#define PP_FLAG_BRUTE_FORCE_DOMS 1u /* test every DOM on every flight (validation; any geometry) */
#define PP_FLAG_NONBLOCKING_SUBMIT 2u /* pp_submit enqueues all n sources or none: PP_E_WOULDBLOCK if the ring lacks space */
#define PP_FLAG_EFFECTIVE_SCATTERING 4u /* pp_ice.scat_len holds effective scattering lengths lambda_e = lambda_s/(1-g)
                                           (the convention of measured ice tables); the mean free path between
                                           scatters is then lambda_e (1-g) (reading R-20; needs g < 1) */

#define PP_FLAG_DEVICE_ORDINAL 8u /* pp_config.device names a CUDA device ordinal even when it is 0 (without the flag,
                                     device <= 0 means "the calling thread's current device", so that a zeroed
                                     pp_config keeps working -- and device 0 cannot be named while another is current) */

/* Sizes and resources.  Zero means "default".  device_workspace / pinned_workspace / streams may be
 * NULL: the library then allocates them itself (cudaMalloc / cudaHostAlloc / cudaStreamCreate) and
 * frees them in pp_destroy.  When given (PyTorch supplies them in the Python binding), they stay
 * owned by the caller and must outlive the handle; pp_workspace_size() says how big they must be. */
typedef struct pp_config {
  uint64_t seed;                  /* Philox key (R-3) */
  uint64_t launch_photons_target; /* photons per GPU launch the server aims for (default 1e8) */
  uint64_t hit_ring_bytes;        /* total device bytes for the two bounded hit rings (default 256 MiB) */
  uint64_t source_ring_bytes;     /* pinned host bytes for the source ring (default 64 MiB) */
  void* device_workspace;
  uint64_t device_workspace_bytes;
  void* pinned_workspace;
  uint64_t pinned_workspace_bytes;
  void* stream0; /* cudaStream_t */
  void* stream1; /* cudaStream_t */
  uint32_t flags;
  uint32_t max_flights; /* safety cap on flights per photon (default 100000, R-10); < 2^31 */
  int32_t device;       /* CUDA device ordinal; <= 0: the current device, unless PP_FLAG_DEVICE_ORDINAL makes 0 an
                           ordinal.  pp_create leaves the caller's current device as it found it. */
  uint32_t reserved;
} pp_config;

typedef struct pp_stats_t {
  uint64_t sources_submitted;
  uint64_t photons_submitted;
  uint64_t photons_done;    /* = absorbed + hit + aborted once drained */
  uint64_t photons_absorbed;
  uint64_t photons_hit;
  uint64_t photons_aborted; /* reached max_flights; must be 0 */
  uint64_t flights;         /* scattering steps (free flights) simulated */
  uint64_t launches;        /* propagation-kernel launches */
  uint64_t relaunches;      /* extra launches forced by a full hit ring */
  uint64_t hits_collected;
  double kernel_busy_ms;    /* union of the propagation kernels' device intervals (CUDA events) */
  double wall_ms;           /* first pp_submit .. last drain */
  uint64_t source_ring_high_water; /* bytes */
  uint64_t hit_ring_high_water;    /* bytes */
  uint64_t photons_rejected;       /* met a DOM but made no photoelectron (pp_set_acceptance); done = absorbed + hit + aborted + rejected */
  uint64_t sources_completed;      /* the first sources_completed sources, in pp_submit order, are fully propagated and all
                                      their hits are available to pp_collect (== sources_submitted once drained); lets a
                                      producer finish its events while others keep the server busy */
} pp_stats_t;

typedef struct pp_handle pp_handle;

/* Required workspace sizes for a configuration (cfg may have NULL workspaces). */
int pp_workspace_size(const pp_geometry* geo, const pp_ice* ice, const pp_config* cfg, uint64_t* device_bytes,
                      uint64_t* pinned_bytes);

/* Builds the DOM lookup and ice tables, uploads them, starts the batching server thread. */
int pp_create(const pp_geometry* geo, const pp_ice* ice, const pp_config* cfg, pp_handle** out);

/* Enqueues n light sources ("a block of steps").  event_ids[n] required.
 * (event_id, source_id) MUST BE UNIQUE for the life of the handle: the pair is part of the Philox counter (R-3), so
 * two sources that share it draw the same random numbers -- perfectly correlated photons, duplicated hits, no error.
 * source_ids may be NULL: a source then gets the handle's running record number (the count of sources submitted
 * before it, pp_stats.sources_submitted, mod 2^32), which is unique across calls.  Results are reproducible from run
 * to run only with explicit ids or a fixed submit order.  Thread-safe: any number of threads may submit
 * concurrently.  Copies before returning.  Blocks while the source ring is full unless
 * PP_FLAG_NONBLOCKING_SUBMIT.  Sources with N == 0 photons are accepted and ignored.  A call with a bad source
 * (non-finite field, direction not a unit vector, negative energy or length, more than 2^32 - 1 photons) fails as a
 * whole with PP_E_INVAL / PP_E_OVERFLOW: none of its sources is propagated.  (If other threads were submitting at the
 * same moment, the failed call may still be counted in pp_stats.sources_submitted, as sources without photons.) */
int pp_submit(pp_handle* h, const pp_source* sources, const uint32_t* event_ids, const uint32_t* source_ids,
              size_t n);

/* pp_submit for extended sources (NEXT-2, reading R-18 of DESIGN.md; a muon's energy loss is split into
 * continuous and stochastic losses; "photon emitting steps").  lengths_m[n] (HOST, nullable = all 0):
 * a source with length L > 0 is a straight track segment from its position along its direction; each of its
 * photons starts at a point uniform on the segment, offset l = u L with u = word 1 of the photon's Philox block 0
 * (the word flight 0 leaves unused), at time t_ns + l / c (the muon moves at c), on the Cherenkov cone about the
 * direction as for a point source.  L = 0 is the point cascade of pp_submit.  PP_E_INVAL for a negative or
 * non-finite length.  Everything else as pp_submit. */
int pp_submit_segments(pp_handle* h, const pp_source* sources, const float* lengths_m, const uint32_t* event_ids,
                       const uint32_t* source_ids, size_t n);

/* One light source with everything pp_submit_segments takes for it, as ONE 48-byte record (array of structures). */
typedef struct pp_packed_source {
  pp_source s;
  float length_m;     /* 0 = point source (R-18) */
  uint32_t event_id;
  uint32_t source_id;
  uint32_t reserved;  /* ignored */
} pp_packed_source;

/* pp_submit_segments for n packed records (HOST): the same checks, the same semantics, explicit source ids; one pass
 * over one array instead of four.  This is what the multi-process front end (pp_ipc.h) moves from its shared-memory
 * rings into the handle: at C2's 400 photons per source a B200 consumes 4e7 sources/s ("a block of
 * steps is sent to the GPU"), which is within sight of what one ingest thread can copy. */
int pp_submit_packed(pp_handle* h, const pp_packed_source* records, size_t n, uint64_t* records_end);
/* records_end (nullable): receives the number of sources submitted to the handle up to and including the last one of
 * this call, in submit order -- the value pp_stats.sources_completed has reached when all of them are propagated.
 * (With several threads submitting, that is how each of them learns where its sources sit in the common order.) */

/* Longitudinal profile of extended sources (NEXT-2, reading R-23): where along its length a source of
 * pp_submit_segments emits.  The offset of a photon becomes l = L F(u) with the same u as above and F piecewise
 * linear through the n_knots values cum_fraction[i] at u = i / (n_knots - 1): an inverse cumulative distribution given
 * as a table (one uniform, no rejection).  cum_fraction is a HOST array, non-decreasing, in [0, 1], copied before
 * returning; 2 <= n_knots <= PP_MAX_PROFILE_KNOTS, or n_knots = 0 for the uniform segment F(u) = u (the default).
 * PP_E_INVAL otherwise; idle server required (PP_E_STATE). */
#define PP_MAX_PROFILE_KNOTS 33u
int pp_set_segment_profile(pp_handle* h, uint32_t n_knots, const float* cum_fraction);

/* Asks the server to launch whatever is queued even if it is less than launch_photons_target. */
int pp_flush(pp_handle* h);

/* Copies up to cap finished hits into out (unspecified order; hits of one event may span calls).
 * block != 0: waits until at least one hit is available or everything submitted so far has been
 * propagated and handed out.  *n_out == 0 with PP_OK then means "drained".  One collector at a time. */
int pp_collect(pp_handle* h, pp_hit* out, size_t cap, size_t* n_out, int block);

/* DOM acceptance ("When a photon intersects a detector, it creates a photoelectron with a probability
 * calculated from its position, direction, time, and wavelength"; the hit record carries a weight).
 * Reading R-17 of DESIGN.md: the probability depends on the arrival direction only,
 *   p(eta) = clamp(coef[0] + coef[1] eta + ... + coef[n_coef-1] eta^(n_coef-1), 0, 1),
 * eta = d_z of the photon at the intersection (cosine between its travel direction and +z).
 *   PP_ACCEPT_OFF            every intersection is a hit of weight 1 (the default after pp_create);
 *   PP_ACCEPT_PROBABILISTIC  one more uniform, word 0 of Philox block (photon, source, event, 2^31 | k) for an
 *                            intersection on flight k: hit of weight 1 iff u < p(eta), else the photon is counted in
 *                            photons_rejected;
 *   PP_ACCEPT_WEIGHTED       no draw: hit of weight p(eta) iff p(eta) > 0, else rejected.
 * The photon stops at the DOM in every mode (R-8).  coef is a HOST array of n_coef <= PP_MAX_ACCEPT_COEF floats,
 * copied before returning (ignored for PP_ACCEPT_OFF).  Applies to launches cut after the call; the server must be
 * idle (nothing queued or in flight), otherwise PP_E_STATE.  PP_E_INVAL for a bad mode, n_coef or a non-finite
 * coefficient. */
#define PP_ACCEPT_OFF 0u
#define PP_ACCEPT_PROBABILISTIC 1u
#define PP_ACCEPT_WEIGHTED 2u
#define PP_MAX_ACCEPT_COEF 8u
int pp_set_acceptance(pp_handle* h, uint32_t mode, const float* coef, uint32_t n_coef);

/* Wavelength bins (NEXT-2, reading R-21 of DESIGN.md; PAPER.md:33 names the wavelength among the things the
 * photoelectron probability depends on, PAPER.md:9 the varying optical properties).  A photon belongs to one of
 * n_bins <= PP_MAX_SPECTRUM_BINS bins for its whole life: bin j = the first with cdf[j] > u, u = the uniform of the word
 * made of the low 9 bits of words 0, 1, 2 of the photon's Philox block 0 (bits the other uniforms do not use, so no
 * extra block is drawn).  In bin j the absorption and scattering coefficients of every ice layer are
 * multiplied by abs_scale[j] and scat_scale[j], the photon travels at c / n_group[j], and the acceptance
 * probability of pp_set_acceptance becomes min(1, p(eta) acc_scale[j]).  All arrays are HOST arrays of n_bins
 * floats, copied before returning: cdf non-decreasing in (0, 1] (the last bin takes whatever is left), scales > 0,
 * n_group >= 1, acc_scale >= 0 (PP_E_INVAL otherwise).  n_bins = 0 switches back to monochromatic photons
 * (pp_ice.n_group, scales 1).  Applies to launches cut after the call; idle server required (PP_E_STATE). */
#define PP_MAX_SPECTRUM_BINS 32u
int pp_set_spectrum(pp_handle* h, uint32_t n_bins, const float* cdf, const float* abs_scale, const float* scat_scale,
                    const float* n_group, const float* acc_scale);

/* Angular smearing of the emission (NEXT-2, reading R-22 of DESIGN.md; a cascade's light comes from
 * its secondaries).  With g_axis < 1 the axis a photon is emitted about is the source direction deflected by a polar
 * angle drawn from the Henyey-Greenstein law of parameter g_axis and a uniform azimuth (words 0 and 1 of Philox block
 * (photon, source, event, 2^29)); the photon then leaves on the Cherenkov cone about that axis.  g_axis = 1 (the
 * default) is the exact cone of R-4.  -1 < g_axis <= 1, g_axis != 0 (PP_E_INVAL otherwise).  Applies to launches cut
 * after the call; idle server required (PP_E_STATE). */
int pp_set_emission_smearing(pp_handle* h, float g_axis);

int pp_stats(pp_handle* h, pp_stats_t* out);
const char* pp_last_error(pp_handle* h);
void pp_destroy(pp_handle* h);

/* ---- device-resident path (what bench.py times as `value`, and what the parity tests drive) ----
 * Inputs already in HBM: d_sources[n] (pp_source), d_event_ids[n], d_source_ids[n] (nullable: the running
 * record number as in pp_submit) are DEVICE pointers.  Runs source expansion + propagation for ALL photons of the n sources in
 * launches of at most launch_photons_target photons, alternating between the two streams,
 * synchronously; hits go through the bounded device hit ring to the pp_collect queue.  Needs an
 * idle server (PP_E_STATE otherwise) and n <= source ring capacity (PP_E_NOMEM otherwise).
 * d_fates, if not NULL, is a DEVICE array with one pp_fate per photon of the batch, indexed by
 * the batch-global photon number (sources in order, photons in order): validation only.
 * device_ms_out: device time from the start of expansion to the last status read-back (CUDA events). */
typedef struct pp_fate {
  float x, y, z;       /* end point */
  float path_m;        /* total geometric path */
  double time_ns;      /* end time */
  uint32_t n_flights;
  int32_t dom;         /* hit DOM or -1 */
  uint32_t fate;       /* 0 absorbed, 1 hit, 2 aborted, 3 rejected by the DOM acceptance */
  uint32_t photon_idx;
} pp_fate;

int pp_run_resident(pp_handle* h, const pp_source* d_sources, const uint32_t* d_event_ids,
                    const uint32_t* d_source_ids, size_t n, pp_fate* d_fates, uint64_t* photons_out,
                    double* device_ms_out);

/* ---- a small resident run that allocates nothing ----
 * For whom: code that must not, or cannot, get device memory at the moment it wants photons propagated.  Three such
 * callers are common.  (1) A plug-in inside a framework whose caching allocator has already taken nearly all of the
 * device for its own pool: a cudaMalloc next to that pool fails, or succeeds and later makes the framework's own
 * allocations fail.  (2) A latency-bound loop: cudaMalloc and cudaFree may wait for every kernel running on the device
 * -- here, for a 100 ms propagation launch of the batching server -- before they return.  (3) A thread in a process
 * where some other thread is capturing a stream in CUDA's default (global) capture mode: cudaMalloc is refused there
 * and breaks the capture.  pp_run_resident itself allocates nothing per call either, but it works in the handle's
 * workspace, needs the server idle, and queues its hits in host memory that grows by allocation; this call touches none
 * of that.
 *
 * What it does: pp_run_resident for a SMALL batch, in one propagation launch, with the hits written straight into the
 * caller's DEVICE buffer.  Same kernels, same Philox counters: the hits are, record for record, those pp_run_resident
 * gives for the same handle and sources (their order in d_hits is unspecified, as everywhere).  The handle supplies the
 * medium, the geometry, the seed and the optional physics set by pp_set_*; its server, queues, workspace and
 * statistics are neither used nor changed, so the call may run while the server is busy.
 *   d_sources[n], d_event_ids[n], d_source_ids[n]   DEVICE inputs, all required (no automatic source ids);
 *   d_hits[hit_cap]                                  DEVICE output, 16-byte aligned (may be NULL if hit_cap == 0);
 *   n_hits_out, photons_out                          HOST outputs (photons_out nullable);
 *   stream                                           cudaStream_t the work is enqueued on (NULL: the default stream).
 * The call returns after the stream has been synchronised: d_hits[0 .. *n_hits_out) is then complete.
 *
 * Scratch: the expanded source records, their photon prefix sums, the tile table and the launch's counters live in
 * ONE statically allocated device array of 512 KiB inside the library image (every GPU on which the library gets
 * loaded holds it until the process exits), shared by every call on that device, whatever the handle.  Hence:
 *   - limits: n <= PP_NOALLOC_MAX_SOURCES and at most PP_NOALLOC_MAX_PHOTONS photons in total; beyond either the call
 *     fails with PP_E_NOMEM and a message that names the limit (pp_last_error), and nothing is written to d_hits;
 *   - PP_E_NOMEM as well if the batch makes more than hit_cap hits (then d_hits holds an arbitrary hit_cap of them and
 *     *n_hits_out the number the batch needs at least); PP_E_OVERFLOW for a source of more than 2^32 - 1 photons;
 *   - the array keeps what the previous call left in it; each call rewrites or clears everything it reads, so calls
 *     in sequence are independent.  The library does NOT order calls against each other: two calls whose GPU work
 *     overlaps on one device (two threads, any streams, any handles) race on the array and both results are garbage.
 *     Serialise them.
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress), with that device
 *     current; make that first call before any stream capture begins in the process.
 * No cudaMalloc, cudaFree, cudaHostAlloc or other allocating CUDA call is made, on the first call or later; host
 * memory is neither allocated nor pinned except for the text of an error message.  The caller's current device is
 * restored before returning. */
#define PP_NOALLOC_MAX_SOURCES 4096u
#define PP_NOALLOC_MAX_PHOTONS 4194304u /* 2^22 */
int pp_run_resident_noalloc(pp_handle* h, const pp_source* d_sources, const uint32_t* d_event_ids,
                            const uint32_t* d_source_ids, size_t n, pp_hit* d_hits, size_t hit_cap, size_t* n_hits_out,
                            uint64_t* photons_out, void* stream);

/* ---- host-only helpers (no CUDA call inside; usable and tested on a machine without a GPU) ----
 * pp_check_inputs: the validation pp_create performs on geometry and ice (PP_E_INVAL), including whether
 * the fast DOM lookup can represent the geometry (PP_E_UNSUPPORTED unless PP_FLAG_BRUTE_FORCE_DOMS).
 * pp_photon_count: step 1 of the path, N = floor(double(E)*double(yield)+0.5); PP_E_OVERFLOW if N >= 2^32.
 * pp_debug_plan_launches: the launch cutting the batching server applies ("when the step
 * queue is sufficiently full, a block of steps is sent"): given the per-source photon counts in queue
 * order and the per-launch target, lists the launches a flush of that queue produces.  Launch k covers
 * sources [first_source, first_source + n_sources) and the photons [g_begin, g_end) of that slice's own
 * exclusive prefix sum, so a source split across launches appears as the last source of one launch and
 * the first of the next.  Returns PP_E_NOMEM (with *n_out = launches needed) if cap is too small. */
typedef struct pp_launch_plan {
  uint64_t first_source;
  uint64_t n_sources;
  uint64_t g_begin;
  uint64_t g_end;
} pp_launch_plan;

int pp_check_inputs(const pp_geometry* geo, const pp_ice* ice, uint32_t flags);
int pp_photon_count(float energy_GeV, float photons_per_GeV, uint64_t* n_out);
int pp_debug_plan_launches(const uint32_t* photon_counts, size_t n, uint64_t target, pp_launch_plan* out, size_t cap,
                           size_t* n_out);

/* Library version and the number of CUDA kernels this library launched so far in this process. */
const char* pp_version(void);
uint64_t pp_kernel_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* PP_H_ */
