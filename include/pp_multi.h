/* pp_multi.h -- several GPUs behind ONE photon server.
 *
 * arXiv:2405.05700: photon propagation is "embarrassingly parallel" and the server "aggregates steps
 * from multiple events and clients in order to keep the GPU as busy as possible".  With more than one
 * GPU in the server's node the same aggregation feeds all of them: this front owns nothing but a queue.  It stages
 * the light sources it is given, cuts them into batches of about one launch (whole sources), and deals every batch to
 * the back end -- one pp_handle per device -- that has the fewest photons outstanding.  Hits of all devices come
 * back through one pp_multi_collect.  There is no exchange between the devices and no collective: replicas only.
 *
 * Results contract: exactly pp.h's.  A photon's random numbers are keyed by (event_id, source_id, photon_idx) and the
 * handles share geometry, ice and seed, so the multiset of hits does not depend on how many devices there are or on
 * which device ran which batch.  (event_id, source_id) must be unique for the life of the front; with
 * source_ids == NULL the FRONT numbers the sources (its running record count), never the individual handles.
 *
 * All pointers are HOST pointers; records are copied before a call returns.  Return codes are pp.h's.
 */
#ifndef PP_MULTI_H_
#define PP_MULTI_H_

#include "pp.h"
#include "pp_ipc.h" /* pp_ipc_backend: the function table a device is driven through */

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pp_multi pp_multi;

typedef struct pp_multi_config {
  uint64_t deal_photons;   /* photons per dealt batch (default 1e8 = pp_config.launch_photons_target's default) */
  float photons_per_GeV;   /* the light yield of the handles' ice (pp_ice.photons_per_GeV); must be > 0 */
  uint32_t reserved;
} pp_multi_config;

/* One front over n handles (1 <= n <= 64), normally one per device (pp_config.device), all created with the same
 * geometry, ice, seed and options.  The handles stay owned by the caller, must be drained now, must outlive the front
 * and must not be used for pp_submit / pp_collect by anybody else meanwhile. */
int pp_multi_create(pp_handle* const* handles, uint32_t n, const pp_multi_config* cfg, pp_multi** out);
/* The same over any back ends (tests on a machine without a GPU use host-only ones). */
int pp_multi_create_backends(const pp_ipc_backend* backends, uint32_t n, const pp_multi_config* cfg, pp_multi** out);
void pp_multi_destroy(pp_multi* m);

/* pp_submit_segments on the front: stages the sources; whenever deal_photons photons are staged, a batch of whole
 * sources is cut and dealt to the least-loaded device (and that device is flushed, so the batch is launched).
 * Thread-safe.  Blocks while the chosen device's source ring is full.  A call with a bad source (pp.h, pp_submit:
 * non-finite field, direction not a unit vector, negative energy or length, more than 2^32 - 1 photons) fails as a
 * whole with PP_E_INVAL / PP_E_OVERFLOW before anything is staged.  Should a device still refuse a batch the front has
 * dealt (a back end with rules of its own), that batch is dropped -- counted as complete, without hits -- and the call
 * whose deal met it returns the device's code; the sources of other calls are not held up. */
int pp_multi_submit(pp_multi* m, const pp_source* sources, const float* lengths_m, const uint32_t* event_ids,
                    const uint32_t* source_ids, size_t n);
/* Deals whatever is staged (however little) and flushes every device. */
int pp_multi_flush(pp_multi* m);
/* pp_collect on the front: hits of all devices, in no particular order.  block != 0: waits until at least one hit is
 * there or everything submitted so far is propagated and handed out (*n_out == 0 then means "drained"). */
int pp_multi_collect(pp_multi* m, pp_hit* out, size_t cap, size_t* n_out, int block);

typedef struct pp_multi_stats {
  uint32_t n_devices, reserved;
  uint64_t sources_submitted, photons_submitted;
  uint64_t sources_staged;          /* submitted, not yet dealt */
  uint64_t sources_completed;       /* the first sources_completed sources, in submit order, are fully propagated */
  uint64_t batches[64];             /* per device: batches dealt */
  uint64_t photons[64];             /* per device: photons dealt */
  uint64_t photons_outstanding[64]; /* per device: dealt and not yet complete */
} pp_multi_stats;
int pp_multi_get_stats(pp_multi* m, pp_multi_stats* out);

/* The front as a back end of the multi-process server: pp_ipc_server_create_backend(&be, ...) then puts client
 * processes (pp_ipc.h) in front of all the devices.  *out stays valid until pp_multi_destroy. */
int pp_multi_backend(pp_multi* m, pp_ipc_backend* out);

#ifdef __cplusplus
}
#endif
#endif /* PP_MULTI_H_ */
