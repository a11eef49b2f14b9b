/* pp_ipc.h -- multi-process front end of the photon-propagation server.
 *
 * arXiv:2405.05700 runs the propagation clients and the photon server as separate processes that talk over
 * "interprocess communications (IPC)"; each client ships "a block of steps" when its step queue
 * is sufficiently full and "the server aggregates steps from multiple events and clients in order to keep the GPU as
 * busy as possible"; 1, 2, 4, 8 or 16 client instances share ONE photon server.
 *
 * This header is that boundary: one server process owns the pp_handle (and the GPU); any number of client processes
 * (no CUDA needed in them) attach to a POSIX shared-memory segment by name.  Per client the segment holds one
 * single-producer/single-consumer ring of light sources (client -> server) and one of hits (server -> client), both
 * bounded: a client that runs ahead of the GPU blocks in pp_ipc_submit, which is what keeps every process's memory
 * predictable.  The server's ingest threads move blocks from the rings into the handle (pp_submit_packed)
 * (so launches mix the sources of all clients); its dispatch thread routes every collected hit to the client that
 * submitted the hit's event.
 *
 * Contract: event ids are global -- an event belongs to the client that first submits a source of it, for as long as
 * a block of that client holding sources of the event is in the server (the owner table forgets an event when the
 * last such block is complete and its hits are routed, so the table stays as small as the work in flight); two
 * clients submitting the same event id at the same time is a caller error (its hits all go to the first).
 * (event_id, source_id) must be unique for the life of the server, as in pp.h: two sources with the same pair draw
 * the same random numbers.  source_ids == NULL numbers a client's sources with its running record count.
 *
 * A client that falls behind with pp_ipc_collect never holds up the others: hits its ring has no room for are parked
 * in the server, and while more than four rings' worth is parked the server takes no more sources from that client
 * (it then blocks in pp_ipc_submit).  A client whose process has died (checked with kill(pid, 0), so server and
 * clients must share a pid namespace) is treated as closed: its hits are dropped and its slot is handed out again.  The
 * hits a client receives are exactly the hits of its events, and, as everywhere in pp.h, they do not depend on how
 * many clients there are, on block sizes or on timing.
 *
 * All pointers are HOST pointers; records are copied before a call returns.  Return codes are pp.h's
 * (PP_OK, PP_E_INVAL, PP_E_NOMEM, PP_E_STATE, PP_E_WOULDBLOCK, ...).
 */
#ifndef PP_IPC_H_
#define PP_IPC_H_

#include "pp.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pp_ipc_server pp_ipc_server;
typedef struct pp_ipc_client pp_ipc_client;

typedef struct pp_ipc_config {
  uint32_t max_clients;       /* client slots in the segment (default 16) */
  uint32_t ingest_threads;    /* threads that move blocks from the rings into the back end (default: one per four
                                 client slots, 2 to 4; always 1 for a back end without submit_packed) */
  uint64_t source_ring_bytes; /* per client, client -> server (default 4 MiB = 87 381 sources) */
  uint64_t hit_ring_bytes;    /* per client, server -> client (default 4 MiB = 131 072 hits) */
} pp_ipc_config;

/* The server's back end: where blocks go and hits come from.  pp_ipc_server_create() binds it to a pp_handle
 * (submit = pp_submit_segments, flush = pp_flush, collect = pp_collect with block = 0, completed =
 * pp_stats.sources_completed); tests on a machine without a GPU bind it to a host-only back end of their own
 * (tests/echo_backend.cpp) through pp_ipc_server_create_backend(). */
typedef struct pp_ipc_backend {
  void* ctx;
  int (*submit)(void* ctx, const pp_source* sources, const float* lengths_m, const uint32_t* event_ids,
                const uint32_t* source_ids, size_t n);
  int (*flush)(void* ctx);
  int (*collect)(void* ctx, pp_hit* out, size_t cap, size_t* n_out, int* drained); /* non-blocking; *drained != 0:
                                            everything submitted before this call has been propagated and handed out */
  int (*completed)(void* ctx, uint64_t* n_sources); /* the first n_sources sources, in submit order, are fully
                                            propagated and their hits can be collected (pp_stats.sources_completed).
                                            Optional (may be NULL); when given, the server decides completion on this
                                            count alone and ignores *drained */
  int (*submit_packed)(void* ctx, const pp_packed_source* records, size_t n, uint64_t* records_end); /* optional
                                            (may be NULL): the same as submit for packed records (pp_submit_packed,
                                            which also says where the call's last record sits in the back end's submit
                                            order); the ingest threads then hand the rings' records over as they lie,
                                            in one pass, several clients at a time */
} pp_ipc_backend;

/* Creates (O_CREAT | O_EXCL) the shared-memory segment `shm_name` ("/name"), and starts the ingest and dispatch
 * threads.  cfg may be NULL (defaults).  The handle must be drained now, must outlive the server and must not be
 * used for pp_submit / pp_collect by anybody else meanwhile. */
int pp_ipc_server_create(pp_handle* h, const char* shm_name, const pp_ipc_config* cfg, pp_ipc_server** out);
int pp_ipc_server_create_backend(const pp_ipc_backend* be, const char* shm_name, const pp_ipc_config* cfg,
                                 pp_ipc_server** out);
/* Stops the threads, unlinks the segment.  Clients still attached see PP_E_STATE from then on. */
void pp_ipc_server_destroy(pp_ipc_server* s);

typedef struct pp_ipc_server_stats {
  uint64_t clients_attached; /* distinct slots ever claimed */
  uint64_t blocks_ingested;  /* calls of the back end's submit */
  uint64_t sources_ingested;
  uint64_t hits_routed;
  uint64_t hits_unrouted;    /* hits of an event no client had announced (must be 0) */
  uint64_t hits_dropped;     /* hits of clients that had left (closed, or their process died) */
  uint64_t clients_dropped;  /* clients the server declared gone because their process no longer exists */
  uint64_t events_tracked;   /* entries of the event-owner table right now (bounded by the events in flight) */
  uint64_t clients_failed;   /* clients a block of which the back end refused (see pp_ipc_submit) */
} pp_ipc_server_stats;
int pp_ipc_server_get_stats(pp_ipc_server* s, pp_ipc_server_stats* out);

/* ---- client side (any process; no CUDA call inside) ---- */
/* Attaches to the segment and claims a client slot -- one a former client has left, else a fresh one (PP_E_NOMEM if
 * none, PP_E_STATE if there is no server). */
int pp_ipc_client_open(const char* shm_name, pp_ipc_client** out);
/* Ships a block of n sources.  lengths_m and source_ids may be NULL as in pp_submit_segments.
 * Blocks while the client's source ring is full; a block larger than the ring is shipped in pieces.
 * A block with a bad source (pp.h, pp_submit) fails here with PP_E_INVAL and ships nothing.  What only the server can
 * judge -- a source of more than 2^32 - 1 photons at the server's light yield, or anything else its back end refuses
 * with PP_E_INVAL / PP_E_OVERFLOW -- fails THIS client only: the refused block is dropped as a whole, the server takes
 * no more sources from the client and drops its outstanding hits, and every later pp_ipc_submit / pp_ipc_flush /
 * pp_ipc_collect of the client returns the back end's code (hits already in its ring are still handed out first).
 * The other clients are served as before; pp_ipc_client_close frees the slot as usual. */
int pp_ipc_submit(pp_ipc_client* c, const pp_source* sources, const float* lengths_m, const uint32_t* event_ids,
                  const uint32_t* source_ids, size_t n);
/* Asks the server to launch whatever is queued (pp_flush) once it has ingested everything this client shipped. */
int pp_ipc_flush(pp_ipc_client* c);
/* Copies up to cap hits of this client's events into out.  block != 0: waits until at least one hit is there or
 * everything this client shipped has been propagated and handed out (*n_out == 0 then means "drained").  A client
 * drains on its own: it does not wait for other clients' work (the server tracks completion block by block, in the
 * order it handed the blocks to the GPU server). */
int pp_ipc_collect(pp_ipc_client* c, pp_hit* out, size_t cap, size_t* n_out, int block);
/* Detaches.  Hits not yet collected are dropped; the slot is handed out again once the blocks this client shipped
 * are complete (other clients' work does not delay that). */
void pp_ipc_client_close(pp_ipc_client* c);

#ifdef __cplusplus
}
#endif
#endif /* PP_IPC_H_ */
