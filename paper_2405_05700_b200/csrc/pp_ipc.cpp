// Multi-process front end (include/pp_ipc.h): one server process owns the
// pp_handle, client processes ship blocks of light sources through a POSIX shared-memory segment and get their
// events' hits back.  Host-only code: no CUDA call in this file.  Product code: shares nothing with oracle/.
#include "../../include/pp_ipc.h"

#include <fcntl.h>
#include <signal.h>
#include <sys/mman.h>
#include <sys/stat.h>
#include <unistd.h>

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <cerrno>
#include <cstddef>
#include <cstring>
#include <deque>
#include <mutex>
#include <new>
#include <string>
#include <thread>
#include <unordered_map>
#include <vector>

namespace {

constexpr uint64_t kMagic = 0x70705f6970633031ull;  // "pp_ipc01"
constexpr size_t kHeaderBytes = 4096;
constexpr size_t kCtlBytes = 256;
constexpr size_t kIngestChunk = 16384;  // sources per back-end submit

struct SrcSlot {  // 48 B
  pp_source s;
  float length;
  uint32_t event_id, source_id, pad;
};
static_assert(sizeof(SrcSlot) == 48, "SrcSlot layout");
static_assert(sizeof(pp_packed_source) == sizeof(SrcSlot) && offsetof(pp_packed_source, length_m) == offsetof(SrcSlot, length) &&
              offsetof(pp_packed_source, event_id) == offsetof(SrcSlot, event_id) &&
              offsetof(pp_packed_source, source_id) == offsetof(SrcSlot, source_id),
              "a ring slot is a pp_packed_source");

struct ShmHeader {
  uint64_t magic;
  uint32_t max_clients, pad;
  uint64_t src_cap, hit_cap;  // records per client ring
  uint64_t client_stride, total_bytes;
  std::atomic<uint32_t> server_alive;
  std::atomic<uint32_t> next_slot;
};
static_assert(sizeof(ShmHeader) <= kHeaderBytes, "header");

// Life of a slot: kAttached (a client owns it) -> kClosed (the client left, or its process is gone) -> kQuiesced (the
// slot's ingest thread has seen that and will not touch the slot's source ring again) -> kRecycled (the dispatch thread has
// emptied it: claimable again).  Only the ingest thread that serves a slot moves it out of kClosed, so the dispatch thread never
// recycles a slot while a block of it is being handed to the back end.
// kFailed: the back end refused a block of this client (a source the client-side checks cannot judge, e.g. more than
// 2^32 - 1 photons at the server's light yield): the server takes nothing more from it and drops its hits, every call of
// the client returns the back end's code, and the slot goes the usual way once the client closes (or is gone).
enum : uint32_t { kFree = 0, kAttached = 1, kClosed = 2, kRecycled = 3, kQuiesced = 4, kFailed = 5 };

struct ClientCtl {
  std::atomic<uint32_t> state;
  std::atomic<uint64_t> src_head;  // written by the client
  std::atomic<uint64_t> src_tail;  // written by the server: sources before it have been handed to the back end
  std::atomic<uint64_t> hit_head;  // written by the server
  std::atomic<uint64_t> hit_tail;  // written by the client
  std::atomic<uint64_t> flush_seq;      // client: src_head at its last flush request
  std::atomic<uint64_t> flushed_seq;    // server: flush requests honoured up to here
  std::atomic<uint64_t> completed_seq;  // server: sources before it are propagated and their hits are in the hit ring
  std::atomic<uint32_t> pid;            // client: its process id (the server checks that a stalled client still exists)
  std::atomic<int32_t> fail_code;       // server: why the slot is kFailed (a pp_status)
};
static_assert(sizeof(ClientCtl) <= kCtlBytes, "ctl");
static_assert(std::atomic<uint64_t>::is_always_lock_free, "address-free atomics needed in shared memory");

struct Segment {
  void* base = nullptr;
  size_t bytes = 0;
  ShmHeader* hdr() const { return reinterpret_cast<ShmHeader*>(base); }
  unsigned char* client_base(uint32_t c) const {
    return reinterpret_cast<unsigned char*>(base) + kHeaderBytes + (size_t)c * hdr()->client_stride;
  }
  ClientCtl* ctl(uint32_t c) const { return reinterpret_cast<ClientCtl*>(client_base(c)); }
  SrcSlot* src_ring(uint32_t c) const { return reinterpret_cast<SrcSlot*>(client_base(c) + kCtlBytes); }
  pp_hit* hit_ring(uint32_t c) const {
    return reinterpret_cast<pp_hit*>(client_base(c) + kCtlBytes + hdr()->src_cap * sizeof(SrcSlot));
  }
};

using Clock = std::chrono::steady_clock;
inline void nap(int us) { std::this_thread::sleep_for(std::chrono::microseconds(us)); }

// ---- back end bound to a pp_handle ----
int h_submit(void* ctx, const pp_source* s, const float* len, const uint32_t* ev, const uint32_t* sid, size_t n) {
  return pp_submit_segments(static_cast<pp_handle*>(ctx), s, len, ev, sid, n);
}
int h_submit_packed(void* ctx, const pp_packed_source* recs, size_t n, uint64_t* records_end) {
  return pp_submit_packed(static_cast<pp_handle*>(ctx), recs, n, records_end);
}
int h_flush(void* ctx) { return pp_flush(static_cast<pp_handle*>(ctx)); }
int h_collect(void* ctx, pp_hit* out, size_t cap, size_t* n_out, int* drained) {
  pp_handle* h = static_cast<pp_handle*>(ctx);
  int rc = pp_collect(h, out, cap, n_out, 0);
  *drained = 0;
  if (rc != PP_OK || *n_out != 0) return rc;
  // nothing to hand out right now: drained iff every submitted photon is done and every hit found was collected
  // (pp_stats: photons_hit is raised before the hits are queued, hits_collected when they are handed out)
  pp_stats_t st;
  rc = pp_stats(h, &st);
  if (rc == PP_OK && st.photons_done == st.photons_submitted && st.hits_collected == st.photons_hit) *drained = 1;
  return rc;
}

int h_completed(void* ctx, uint64_t* n_sources) {
  pp_stats_t st;
  const int rc = pp_stats(static_cast<pp_handle*>(ctx), &st);
  *n_sources = rc == PP_OK ? st.sources_completed : 0;
  return rc;
}

}  // namespace

struct pp_ipc_server {
  Segment seg;
  std::string name;
  pp_ipc_backend be{};
  std::vector<std::thread> ingest;  // thread t serves the client slots c with c % ingest.size() == t
  std::thread dispatch;
  std::atomic<bool> stop{false};
  // event id -> owning client slot, with the number of that client's blocks holding sources of the event that are
  // handed to the back end and not yet complete; the entry goes when the count drops to zero
  struct Owner { uint32_t client, blocks; };
  std::mutex map_mu;
  std::unordered_map<uint32_t, Owner> owner;
  std::atomic<uint64_t> blocks{0}, sources{0}, routed{0}, unrouted{0}, dropped{0}, clients_dropped{0}, clients_failed{0};
  struct Block { uint32_t client; uint64_t tail_after, global_end; std::vector<uint32_t> events; };
  std::mutex fifo_mu;
  std::deque<Block> fifo;       // blocks handed to the back end, not yet known to be complete: in hand-over order with
                                // one ingest thread, in any order with several (global_end then comes from the back end)
  uint64_t base_completed = 0;  // the back end's completed count when the server started
  // per client slot
  struct PerClient {
    std::deque<pp_hit> parked;             // dispatch thread only: hits waiting for room in the client's hit ring
    uint64_t pending_completed = 0;        // dispatch thread only: completed_seq to publish once `parked` is empty
    std::atomic<uint64_t> parked_n{0};     // read by the ingest thread: a client far behind is not ingested from
    std::atomic<uint32_t> blocks_in_flight{0};
    Clock::time_point last_alive_check{};
  };
  std::vector<PerClient> pc;
  uint64_t park_cap = 0;  // hits parked per client above which the server stops taking that client's sources

  std::atomic<int> error{PP_OK};
};

struct pp_ipc_client {
  Segment seg;
  uint32_t slot = 0;
};

namespace {

void ingest_main(pp_ipc_server* s, uint32_t me, uint32_t n_thr) {
  ShmHeader* H = s->seg.hdr();
  std::vector<pp_source> src(kIngestChunk);
  std::vector<float> len(kIngestChunk);
  std::vector<uint32_t> ev(kIngestChunk), sid(kIngestChunk);
  while (!s->stop.load()) {
    bool progressed = false;
    const uint32_t n_slots = std::min(H->next_slot.load(std::memory_order_acquire), H->max_clients);
    for (uint32_t c = me; c < n_slots; c += n_thr) {
      ClientCtl* ctl = s->seg.ctl(c);
      const uint32_t state = ctl->state.load(std::memory_order_acquire);
      if (state == kClosed) {
        // the client has left: sources it shipped and the server never took are skipped (nobody wants their hits),
        // and from here on this thread leaves the slot alone until a new client has attached
        ctl->src_tail.store(ctl->src_head.load(std::memory_order_acquire), std::memory_order_release);
        ctl->flushed_seq.store(ctl->flush_seq.load(std::memory_order_relaxed), std::memory_order_relaxed);
        if (s->pc[c].blocks_in_flight.load() != 0) {
          // blocks of it that the back end still holds must complete for the slot to come back
          const int rc = s->be.flush(s->be.ctx);
          if (rc != PP_OK) { s->error.store(rc); s->stop.store(true); break; }
        }
        uint32_t expect = kClosed;
        ctl->state.compare_exchange_strong(expect, kQuiesced, std::memory_order_acq_rel);
        continue;
      }
      if (state == kFailed) {
        // nothing more is taken from a client whose block the back end refused; what it still ships is skipped
        ctl->src_tail.store(ctl->src_head.load(std::memory_order_acquire), std::memory_order_release);
        ctl->flushed_seq.store(ctl->flush_seq.load(std::memory_order_relaxed), std::memory_order_relaxed);
        continue;
      }
      if (state != kAttached) continue;
      const uint64_t head = ctl->src_head.load(std::memory_order_acquire);
      uint64_t tail = ctl->src_tail.load(std::memory_order_relaxed);
      // a client that does not read its hits gets no more work done for it: its source ring fills up and it blocks
      // in pp_ipc_submit, which bounds what the server has to park for it
      const bool behind = s->pc[c].parked_n.load(std::memory_order_acquire) > s->park_cap;
      if (head != tail && !behind) {
        const SrcSlot* ring = s->seg.src_ring(c);
        const uint64_t t0 = tail % H->src_cap;
        // a back end that takes packed records gets them as they lie in the ring (one contiguous span per pass)
        const bool packed = s->be.submit_packed != nullptr;
        const size_t n = (size_t)std::min<uint64_t>(std::min<uint64_t>(head - tail, kIngestChunk),
                                                    packed ? H->src_cap - t0 : kIngestChunk);
        bool any_len = false;
        if (!packed)
          for (size_t i = 0; i < n; ++i) {
            const uint64_t k = t0 + i;
            const SrcSlot& r = ring[k < H->src_cap ? k : k - H->src_cap];
            src[i] = r.s; len[i] = r.length; ev[i] = r.event_id; sid[i] = r.source_id;
            any_len |= r.length != 0.0f;
          }
        pp_ipc_server::Block blk{c, tail + n, 0, {}};
        {
          // the block's distinct event ids, found outside the lock (one id per run of equal ids, then sort + unique:
          // a block of 16384 one-source events costs n log n here, not n^2 comparisons inside the lock the dispatch
          // thread needs for every run of hits it routes)
          std::vector<uint32_t>& ids = blk.events;
          uint32_t last = ~(packed ? ring[t0].event_id : ev[0]);
          for (size_t i = 0; i < n; ++i) {
            const uint32_t e = packed ? ring[t0 + i].event_id : ev[i];
            if (e != last) { ids.push_back(e); last = e; }
          }
          std::sort(ids.begin(), ids.end());
          ids.erase(std::unique(ids.begin(), ids.end()), ids.end());
          std::lock_guard<std::mutex> g(s->map_mu);  // announce the events before their hits can exist
          size_t kept = 0;
          for (const uint32_t e : ids) {
            auto it = s->owner.find(e);
            if (it == s->owner.end()) it = s->owner.emplace(e, pp_ipc_server::Owner{c, 0}).first;
            if (it->second.client == c) { it->second.blocks++; ids[kept++] = e; }  // else: caller error (pp_ipc.h)
          }
          ids.resize(kept);
        }
        s->pc[c].blocks_in_flight++;
        int rc;
        if (packed) {
          // the back end says where the block's last record sits in its submit order; the block joins the list after
          // the hand-over (a block that is complete before it is listed is simply found complete at the next look)
          uint64_t end = 0;
          rc = s->be.submit_packed(s->be.ctx, reinterpret_cast<const pp_packed_source*>(ring + t0), n, &end);
          if (rc == PP_OK) {
            blk.global_end = end - s->base_completed;
            std::lock_guard<std::mutex> g(s->fifo_mu);
            s->fifo.push_back(std::move(blk));
          }
        } else {
          {
            // one ingest thread: the block is in the list before the back end sees it, in hand-over order
            std::lock_guard<std::mutex> g(s->fifo_mu);
            blk.global_end = s->sources.load() + n;
            s->fifo.push_back(std::move(blk));
          }
          rc = s->be.submit(s->be.ctx, src.data(), any_len ? len.data() : nullptr, ev.data(), sid.data(), n);
        }
        if (rc == PP_E_INVAL || rc == PP_E_OVERFLOW) {
          // The back end refused the block as a whole (pp.h: none of its sources is propagated): a fault of this
          // client's input, not of the server.  The block is taken back out of the books, the client is marked failed,
          // and everybody else is served as before.
          if (!packed) {
            std::lock_guard<std::mutex> g(s->fifo_mu);  // (listed before the hand-over; the one ingest thread's newest)
            blk = std::move(s->fifo.back());
            s->fifo.pop_back();
          }
          {
            std::lock_guard<std::mutex> g(s->map_mu);
            for (const uint32_t e : blk.events) {
              auto it = s->owner.find(e);
              if (it != s->owner.end() && it->second.client == c && --it->second.blocks == 0) s->owner.erase(it);
            }
          }
          s->pc[c].blocks_in_flight--;
          ctl->fail_code.store(rc, std::memory_order_release);
          uint32_t expect = kAttached;
          if (ctl->state.compare_exchange_strong(expect, kFailed, std::memory_order_acq_rel)) s->clients_failed++;
          ctl->src_tail.store(ctl->src_head.load(std::memory_order_acquire), std::memory_order_release);
          progressed = true;
          continue;
        }
        if (rc != PP_OK) { s->error.store(rc); s->stop.store(true); break; }
        s->blocks++; s->sources += n;
        tail += n;
        ctl->src_tail.store(tail, std::memory_order_release);
        progressed = true;
      }
      const uint64_t fs = ctl->flush_seq.load(std::memory_order_acquire);
      if (fs > ctl->flushed_seq.load(std::memory_order_relaxed) && tail >= fs) {
        const int rc = s->be.flush(s->be.ctx);
        if (rc != PP_OK) { s->error.store(rc); s->stop.store(true); break; }
        ctl->flushed_seq.store(fs, std::memory_order_release);
        progressed = true;
      }
    }
    if (!progressed) nap(50);
  }
}

// A client is gone if it closed, or if its process no longer exists (it was killed: PAPER.md:47 names jobs that die
// at their memory limit).  The existence check costs a system call, so it is made at most every 10 ms per client and
// only for a client the server is waiting for.
bool client_gone(pp_ipc_server* s, uint32_t c) {
  ClientCtl* ctl = s->seg.ctl(c);
  const uint32_t st = ctl->state.load(std::memory_order_acquire);
  if (st != kAttached && st != kFailed) return true;
  auto& pc = s->pc[c];
  const auto now = Clock::now();
  if (now - pc.last_alive_check < std::chrono::milliseconds(10)) return false;
  pc.last_alive_check = now;
  const uint32_t pid = ctl->pid.load(std::memory_order_acquire);
  if (pid != 0 && kill((pid_t)pid, 0) != 0 && errno == ESRCH) {
    uint32_t expect = st;
    if (ctl->state.compare_exchange_strong(expect, kClosed, std::memory_order_acq_rel)) s->clients_dropped++;
    return true;
  }
  return false;
}

// Move parked hits of client c into its ring as far as there is room; drop them if the client is gone.
void drain_parked(pp_ipc_server* s, uint32_t c) {
  auto& pc = s->pc[c];
  ShmHeader* H = s->seg.hdr();
  ClientCtl* ctl = s->seg.ctl(c);
  if (!pc.parked.empty()) {
    const uint64_t head = ctl->hit_head.load(std::memory_order_relaxed);
    const uint64_t space = H->hit_cap - (head - ctl->hit_tail.load(std::memory_order_acquire));
    if (space > 0) {
      pp_hit* ring = s->seg.hit_ring(c);
      const size_t m = (size_t)std::min<uint64_t>(space, pc.parked.size());
      for (size_t q = 0; q < m; ++q) ring[(head + q) % H->hit_cap] = pc.parked[q];
      pc.parked.erase(pc.parked.begin(), pc.parked.begin() + (long)m);
      ctl->hit_head.store(head + m, std::memory_order_release);
      s->routed += m;
    } else if (client_gone(s, c)) {
      s->dropped += pc.parked.size();
      pc.parked.clear();
    }
    pc.parked_n.store(pc.parked.size(), std::memory_order_release);
  }
  if (pc.parked.empty() && pc.pending_completed > ctl->completed_seq.load(std::memory_order_relaxed))
    ctl->completed_seq.store(pc.pending_completed, std::memory_order_release);  // its hits are all in the ring now
}

void dispatch_main(pp_ipc_server* s) {
  ShmHeader* H = s->seg.hdr();
  const size_t cap = 1 << 16;
  std::vector<pp_hit> buf(cap);
  while (!s->stop.load()) {
    const uint32_t n_slots = std::min(H->next_slot.load(std::memory_order_acquire), H->max_clients);
    for (uint32_t c = 0; c < n_slots; ++c) drain_parked(s, c);
    // how many sources (in hand-over order) were complete BEFORE the collect below: their hits are already queued,
    // so once that collect comes back empty they have all been routed (or parked)
    // Both are read BEFORE the collect, never after: a block handed over while the collect was under way (an idle
    // server, a preempted dispatch thread) is not covered by what that collect reports.
    uint64_t n_complete = 0;
    if (s->be.completed) {
      uint64_t v = 0;
      const int rc0 = s->be.completed(s->be.ctx, &v);
      if (rc0 != PP_OK) { s->error.store(rc0); s->stop.store(true); break; }
      n_complete = v > s->base_completed ? v - s->base_completed : 0;
    }
    // (back ends without completed(): the sources whose hand-over had returned by now)
    const uint64_t handed_before = s->sources.load(std::memory_order_acquire);
    size_t n = 0;
    int drained = 0;
    const int rc = s->be.collect(s->be.ctx, buf.data(), cap, &n, &drained);
    if (rc != PP_OK) { s->error.store(rc); s->stop.store(true); break; }
    size_t i = 0;
    while (i < n) {
      // route a run of hits of one event in one go
      uint32_t c = ~0u;
      {
        std::lock_guard<std::mutex> g(s->map_mu);
        auto it = s->owner.find(buf[i].event_id);
        if (it != s->owner.end()) c = it->second.client;
      }
      size_t j = i + 1;
      while (j < n && buf[j].event_id == buf[i].event_id) ++j;
      if (c == ~0u) { s->unrouted += j - i; i = j; continue; }
      auto& pc = s->pc[c];
      ClientCtl* ctl = s->seg.ctl(c);
      const uint32_t st = ctl->state.load(std::memory_order_acquire);
      if (st != kAttached) { s->dropped += j - i; i = j; continue; }  // nobody will read them
      if (pc.parked.empty()) {
        // straight into the client's ring as far as there is room ...
        pp_hit* ring = s->seg.hit_ring(c);
        const uint64_t head = ctl->hit_head.load(std::memory_order_relaxed);
        const uint64_t space = H->hit_cap - (head - ctl->hit_tail.load(std::memory_order_acquire));
        const size_t m = (size_t)std::min<uint64_t>(space, j - i);
        for (size_t q = 0; q < m; ++q) ring[(head + q) % H->hit_cap] = buf[i + q];
        if (m) ctl->hit_head.store(head + m, std::memory_order_release);
        s->routed += m;
        i += m;
      }
      if (i < j) {
        // ... the rest is parked: a client that is behind (or dead) never holds up the routing for the others
        pc.parked.insert(pc.parked.end(), buf.begin() + (long)i, buf.begin() + (long)j);
        pc.parked_n.store(pc.parked.size(), std::memory_order_release);
        i = j;
      }
    }
    if (n == 0) {
      // per-client completion, block by block: a client drains without waiting for the others.  A block is complete
      // once the back end says so (n_complete, read before the collect that came back empty: its hits are routed).
      std::vector<pp_ipc_server::Block> done;
      {
        std::lock_guard<std::mutex> g(s->fifo_mu);
        // a back end with completed() is believed on that count alone; `drained` serves the ones without: everything
        // whose hand-over had returned before the collect started is done
        const uint64_t upto = s->be.completed ? n_complete : (drained ? handed_before : 0);
        for (auto it = s->fifo.begin(); it != s->fifo.end();) {
          if (it->global_end <= upto &&
              it->tail_after <= s->seg.ctl(it->client)->src_tail.load(std::memory_order_acquire)) {
            done.push_back(std::move(*it));
            it = s->fifo.erase(it);
          } else if (s->ingest.size() == 1) {
            break;  // hand-over order: nothing behind an incomplete block is complete
          } else {
            ++it;
          }
        }
      }
      if (!done.empty()) {
        std::lock_guard<std::mutex> g(s->map_mu);
        for (const auto& b : done)
          for (uint32_t e : b.events) {
            auto it = s->owner.find(e);
            if (it != s->owner.end() && it->second.client == b.client && --it->second.blocks == 0) s->owner.erase(it);
          }
      }
      for (const auto& b : done) {
        auto& pc = s->pc[b.client];
        pc.pending_completed = std::max(pc.pending_completed, b.tail_after);
        pc.blocks_in_flight--;
        drain_parked(s, b.client);
      }
      // a slot is handed out again once its client has left and nothing of it is in the server any more.  The ring
      // counters are absolute and simply carry on; hits the old client never read are skipped.
      for (uint32_t c = 0; c < n_slots; ++c) {
        ClientCtl* ctl = s->seg.ctl(c);
        const uint32_t st = ctl->state.load(std::memory_order_acquire);
        if (st == kAttached || st == kFailed) { client_gone(s, c); continue; }  // a client whose process was killed is closed here
        if (st != kQuiesced) continue;                         // the ingest thread has not let go of the slot yet
        auto& pc = s->pc[c];
        if (!pc.parked.empty()) { s->dropped += pc.parked.size(); pc.parked.clear(); pc.parked_n.store(0); }
        if (pc.blocks_in_flight.load() != 0) continue;
        ctl->hit_tail.store(ctl->hit_head.load(std::memory_order_relaxed), std::memory_order_release);
        pc.pending_completed = 0;
        ctl->completed_seq.store(ctl->src_head.load(std::memory_order_acquire), std::memory_order_release);
        ctl->pid.store(0, std::memory_order_relaxed);
        ctl->fail_code.store(0, std::memory_order_relaxed);
        ctl->state.store(kRecycled, std::memory_order_release);
      }
      nap(100);
    }
  }
}

int map_segment(const char* name, bool create, size_t bytes, Segment* seg) {
  const int fd = create ? shm_open(name, O_CREAT | O_EXCL | O_RDWR, 0600) : shm_open(name, O_RDWR, 0600);
  if (fd < 0) return PP_E_STATE;
  if (create && ftruncate(fd, (off_t)bytes) != 0) { close(fd); shm_unlink(name); return PP_E_NOMEM; }
  if (!create) {
    struct stat st;
    if (fstat(fd, &st) != 0 || (size_t)st.st_size < kHeaderBytes) { close(fd); return PP_E_STATE; }
    bytes = (size_t)st.st_size;
  }
  void* p = mmap(nullptr, bytes, PROT_READ | PROT_WRITE, MAP_SHARED, fd, 0);
  close(fd);
  if (p == MAP_FAILED) { if (create) shm_unlink(name); return PP_E_NOMEM; }
  seg->base = p; seg->bytes = bytes;
  return PP_OK;
}

}  // namespace

extern "C" {

int pp_ipc_server_create_backend(const pp_ipc_backend* be, const char* shm_name, const pp_ipc_config* cfg,
                                 pp_ipc_server** out) {
  if (!be || !be->submit || !be->flush || !be->collect || !shm_name || shm_name[0] != '/' || !out) return PP_E_INVAL;
  *out = nullptr;
  const uint32_t max_clients = cfg && cfg->max_clients ? cfg->max_clients : 16u;
  const uint64_t src_bytes = cfg && cfg->source_ring_bytes ? cfg->source_ring_bytes : (4ull << 20);
  const uint64_t hit_bytes = cfg && cfg->hit_ring_bytes ? cfg->hit_ring_bytes : (4ull << 20);
  if (max_clients > 1024) return PP_E_INVAL;
  const uint64_t src_cap = std::max<uint64_t>(1, src_bytes / sizeof(SrcSlot));
  const uint64_t hit_cap = std::max<uint64_t>(1, hit_bytes / sizeof(pp_hit));
  const uint64_t stride = (kCtlBytes + src_cap * sizeof(SrcSlot) + hit_cap * sizeof(pp_hit) + 255) / 256 * 256;
  const size_t total = kHeaderBytes + (size_t)stride * max_clients;
  auto* s = new pp_ipc_server();
  s->name = shm_name;
  s->be = *be;
  const int rc = map_segment(shm_name, true, total, &s->seg);
  if (rc != PP_OK) { delete s; return rc; }
  std::memset(s->seg.base, 0, kHeaderBytes);
  ShmHeader* H = new (s->seg.base) ShmHeader();
  H->max_clients = max_clients; H->src_cap = src_cap; H->hit_cap = hit_cap;
  H->client_stride = stride; H->total_bytes = total;
  for (uint32_t c = 0; c < max_clients; ++c) new (s->seg.ctl(c)) ClientCtl();  // ftruncate zero-filled the rings
  H->next_slot.store(0);
  s->pc = std::vector<pp_ipc_server::PerClient>(max_clients);
  s->park_cap = 4 * hit_cap;
  H->magic = kMagic;
  H->server_alive.store(1, std::memory_order_release);
  if (s->be.completed) s->be.completed(s->be.ctx, &s->base_completed);  // the back end must be drained at this point
  {
    // default: one ingest thread per four client slots, at least 2, at most 4 (measured with 8 and 16 clients)
    uint32_t n_thr = s->be.submit_packed ? (cfg && cfg->ingest_threads ? cfg->ingest_threads : std::max(2u, std::min(4u, max_clients / 4u))) : 1u;
    n_thr = std::max(1u, std::min(n_thr, std::min(max_clients, 16u)));
    s->ingest.reserve(n_thr);  // (dispatch_main reads ingest.size(): all threads exist before it starts)
    for (uint32_t t = 0; t < n_thr; ++t) s->ingest.emplace_back(ingest_main, s, t, n_thr);
  }
  s->dispatch = std::thread(dispatch_main, s);
  *out = s;
  return PP_OK;
}

int pp_ipc_server_create(pp_handle* h, const char* shm_name, const pp_ipc_config* cfg, pp_ipc_server** out) {
  if (!h) return PP_E_INVAL;
  const pp_ipc_backend be{h, h_submit, h_flush, h_collect, h_completed, h_submit_packed};
  return pp_ipc_server_create_backend(&be, shm_name, cfg, out);
}

void pp_ipc_server_destroy(pp_ipc_server* s) {
  if (!s) return;
  s->stop.store(true);
  for (auto& t : s->ingest) if (t.joinable()) t.join();
  if (s->dispatch.joinable()) s->dispatch.join();
  s->seg.hdr()->server_alive.store(0, std::memory_order_release);
  munmap(s->seg.base, s->seg.bytes);
  shm_unlink(s->name.c_str());
  delete s;
}

int pp_ipc_server_get_stats(pp_ipc_server* s, pp_ipc_server_stats* out) {
  if (!s || !out) return PP_E_INVAL;
  out->clients_attached = std::min(s->seg.hdr()->next_slot.load(), s->seg.hdr()->max_clients);
  out->blocks_ingested = s->blocks.load(); out->sources_ingested = s->sources.load();
  out->hits_routed = s->routed.load(); out->hits_unrouted = s->unrouted.load();
  out->hits_dropped = s->dropped.load(); out->clients_dropped = s->clients_dropped.load();
  out->clients_failed = s->clients_failed.load();
  {
    std::lock_guard<std::mutex> g(s->map_mu);
    out->events_tracked = s->owner.size();
  }
  return s->error.load();
}

int pp_ipc_client_open(const char* shm_name, pp_ipc_client** out) {
  if (!shm_name || !out) return PP_E_INVAL;
  *out = nullptr;
  auto* c = new pp_ipc_client();
  const int rc = map_segment(shm_name, false, 0, &c->seg);
  if (rc != PP_OK) { delete c; return rc; }
  ShmHeader* H = c->seg.hdr();
  if (H->magic != kMagic || H->total_bytes != c->seg.bytes || !H->server_alive.load(std::memory_order_acquire)) {
    munmap(c->seg.base, c->seg.bytes); delete c; return PP_E_STATE;
  }
  // a slot a former client has left (and the server has emptied) first, else a fresh one
  uint32_t slot = ~0u;
  const uint32_t used = std::min(H->next_slot.load(std::memory_order_acquire), H->max_clients);
  for (uint32_t i = 0; i < used && slot == ~0u; ++i) {
    uint32_t expect = kRecycled;
    if (c->seg.ctl(i)->state.compare_exchange_strong(expect, kAttached, std::memory_order_acq_rel)) slot = i;
  }
  if (slot == ~0u) {
    if (H->next_slot.load(std::memory_order_acquire) >= H->max_clients) { munmap(c->seg.base, c->seg.bytes); delete c; return PP_E_NOMEM; }
    slot = H->next_slot.fetch_add(1);
    if (slot >= H->max_clients) { munmap(c->seg.base, c->seg.bytes); delete c; return PP_E_NOMEM; }
    c->seg.ctl(slot)->state.store(kAttached, std::memory_order_release);
  }
  c->slot = slot;
  c->seg.ctl(slot)->pid.store((uint32_t)getpid(), std::memory_order_release);
  *out = c;
  return PP_OK;
}

int pp_ipc_submit(pp_ipc_client* c, const pp_source* sources, const float* lengths, const uint32_t* event_ids,
                  const uint32_t* source_ids, size_t n) {
  if (!c) return PP_E_INVAL;
  if (n == 0) return PP_OK;
  if (!sources || !event_ids) return PP_E_INVAL;
  {
    // the cheap checks here, so that a bad block never reaches the shared ring (one branch-free pass: a client ships
    // millions of sources per second)
    uint32_t bad = 0;
    for (size_t i = 0; i < n; ++i) {
      const pp_source& a = sources[i];
      uint32_t w[8];
      std::memcpy(w, &a, sizeof w);  // x, y, z, dx, dy, dz, t, E
      uint32_t nonfinite = 0;
      for (int q = 0; q < 8; ++q) nonfinite |= (uint32_t)((w[q] & 0x7f800000u) == 0x7f800000u);
      const double n2 = (double)a.dx * a.dx + (double)a.dy * a.dy + (double)a.dz * a.dz;
      const float len = lengths ? lengths[i] : 0.0f;
      bad |= nonfinite | (uint32_t)(a.energy_GeV < 0.0f) | (uint32_t)!(len >= 0.0f && len <= 3.0e38f) |
             (uint32_t)(std::fabs(n2 - 1.0) > 1e-4);
    }
    if (bad) return PP_E_INVAL;
  }
  ShmHeader* H = c->seg.hdr();
  ClientCtl* ctl = c->seg.ctl(c->slot);
  SrcSlot* ring = c->seg.src_ring(c->slot);
  size_t i = 0;
  while (i < n) {
    if (!H->server_alive.load(std::memory_order_acquire)) return PP_E_STATE;
    if (ctl->state.load(std::memory_order_acquire) == kFailed) return ctl->fail_code.load(std::memory_order_acquire);
    const uint64_t head = ctl->src_head.load(std::memory_order_relaxed);
    const uint64_t space = H->src_cap - (head - ctl->src_tail.load(std::memory_order_acquire));
    if (space == 0) { nap(50); continue; }  // bounded ring: the client waits for the GPU
    const size_t m = (size_t)std::min<uint64_t>(space, n - i);
    for (size_t q = 0; q < m; ++q, ++i) {
      SrcSlot& r = ring[(head + q) % H->src_cap];
      r.s = sources[i]; r.length = lengths ? lengths[i] : 0.0f; r.event_id = event_ids[i];
      r.source_id = source_ids ? source_ids[i] : (uint32_t)(head + q); r.pad = 0;  // the client's running record number
    }
    ctl->src_head.store(head + m, std::memory_order_release);
  }
  return PP_OK;
}

int pp_ipc_flush(pp_ipc_client* c) {
  if (!c) return PP_E_INVAL;
  ClientCtl* ctl = c->seg.ctl(c->slot);
  ctl->flush_seq.store(ctl->src_head.load(std::memory_order_relaxed), std::memory_order_release);
  if (ctl->state.load(std::memory_order_acquire) == kFailed) return ctl->fail_code.load(std::memory_order_acquire);
  return c->seg.hdr()->server_alive.load(std::memory_order_acquire) ? PP_OK : PP_E_STATE;
}

int pp_ipc_collect(pp_ipc_client* c, pp_hit* out, size_t cap, size_t* n_out, int block) {
  if (!c || !n_out || (!out && cap)) return PP_E_INVAL;
  *n_out = 0;
  ShmHeader* H = c->seg.hdr();
  ClientCtl* ctl = c->seg.ctl(c->slot);
  const pp_hit* ring = c->seg.hit_ring(c->slot);
  for (;;) {
    // read "complete" before the ring: hits are published before completed_seq moves
    const bool complete = ctl->completed_seq.load(std::memory_order_acquire) >= ctl->src_head.load(std::memory_order_relaxed);
    const uint64_t tail = ctl->hit_tail.load(std::memory_order_relaxed);
    const uint64_t avail = ctl->hit_head.load(std::memory_order_acquire) - tail;
    if (avail > 0) {
      const size_t m = (size_t)std::min<uint64_t>(avail, cap);
      for (size_t q = 0; q < m; ++q) out[q] = ring[(tail + q) % H->hit_cap];
      ctl->hit_tail.store(tail + m, std::memory_order_release);
      *n_out = m;
      return PP_OK;
    }
    if (ctl->state.load(std::memory_order_acquire) == kFailed) return ctl->fail_code.load(std::memory_order_acquire);
    if (complete || !block) return PP_OK;  // drained, or nothing yet
    if (!H->server_alive.load(std::memory_order_acquire)) return PP_E_STATE;
    nap(100);
  }
}

void pp_ipc_client_close(pp_ipc_client* c) {
  if (!c) return;
  c->seg.ctl(c->slot)->state.store(kClosed, std::memory_order_release);
  munmap(c->seg.base, c->seg.bytes);
  delete c;
}

}  // extern "C"
