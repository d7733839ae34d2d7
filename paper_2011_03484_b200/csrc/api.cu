// api.cu — the C ABI of include/glisse.h and the host driver behind it (layers A and B of
// DESIGN.md §1): per-chunk schedule planet-history kernel (own stream, one chunk ahead, two log
// buffers) -> particle kernel -> survivor compaction every R chunks
// (PAPER.md:127), with CUDA events for the dependencies and no host synchronisation inside
// glisse_advance.  Every step of the path runs in the kernels; there is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/glisse_test.h"
#include "glisse_internal.cuh"

using namespace glisse;

namespace {

struct LogBuffer {
  double* log = nullptr;    // [(K+1) * stride]
  double* jlog = nullptr;   // [(K+1) * 6 Np]   Jacobi state of the planets at every record
  long long start = 0;      // step index of record 0
  int len = 0;              // steps it holds (records 0..len); K except while ramping up
  cudaEvent_t ready = nullptr;     // planet-history kernel that fills it has finished   (stream P)
  cudaEvent_t consumed = nullptr;  // last particle kernel that reads it has finished    (stream Q)
};

struct TimedLaunch {
  cudaEvent_t t0, t1;
};

// Device memory of a sim comes from one stream-ordered pool per device that keeps up to 1 GiB of
// freed memory cached: a create/destroy cycle then costs microseconds instead of the ~1 ms of a
// cudaMalloc/cudaFree pair (which also synchronise the device).
std::mutex g_mu;
cudaMemPool_t g_pool[64] = {};

cudaError_t arena_pool(int dev, cudaMemPool_t* out) {
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_pool[dev]) {
    cudaMemPoolProps props{};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaError_t e = cudaMemPoolCreate(&g_pool[dev], &props);
    if (e != cudaSuccess) return e;
    unsigned long long keep = 1ull << 30;
    e = cudaMemPoolSetAttribute(g_pool[dev], cudaMemPoolAttrReleaseThreshold, &keep);
    if (e != cudaSuccess) return e;
  }
  *out = g_pool[dev];
  return cudaSuccess;
}

// The pinned word through which a sim's survivor count comes back: handed out from one pinned page
// per process (cudaMallocHost/cudaFreeHost per sim cost ~0.2 ms).
constexpr int kPinnedWords = 1024;
constexpr int kRingStepWords = 64;   // slot_step copies that may be in flight at once
int* g_pinned = nullptr;
std::vector<int> g_pinned_free;

int* pinned_word() {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_pinned) {
    if (cudaMallocHost(reinterpret_cast<void**>(&g_pinned), kPinnedWords * sizeof(int)) != cudaSuccess) {
      (void)cudaGetLastError();
      g_pinned = nullptr;
      return nullptr;
    }
    for (int i = kPinnedWords - 1; i >= 0; --i) g_pinned_free.push_back(i);
  }
  if (g_pinned_free.empty()) return nullptr;
  const int i = g_pinned_free.back();
  g_pinned_free.pop_back();
  return g_pinned + i;
}

// Streams of a sim come from a per-device cache as well: creating the two streams of a sim and
// destroying them again cost ~0.3 ms per create / destroy cycle (measured on the box), more than the
// whole upload of 10^5 particles.  A stream goes back only after it has been synchronised; at most
// kCachedStreams of each kind are kept per device, the rest are destroyed.
constexpr int kCachedStreams = 8;
std::vector<cudaStream_t> g_streams[64][2];   // [device][0 = default priority, 1 = highest]

cudaError_t take_stream(int dev, bool high_priority, cudaStream_t* out) {
  {
    std::lock_guard<std::mutex> lock(g_mu);
    auto& v = g_streams[dev][high_priority ? 1 : 0];
    if (!v.empty()) {
      *out = v.back();
      v.pop_back();
      return cudaSuccess;
    }
  }
  if (!high_priority) return cudaStreamCreateWithFlags(out, cudaStreamNonBlocking);
  int least = 0, greatest = 0;
  cudaError_t e = cudaDeviceGetStreamPriorityRange(&least, &greatest);
  if (e != cudaSuccess) return e;
  return cudaStreamCreateWithPriority(out, cudaStreamNonBlocking, greatest);
}

// st: synchronised, with nothing of the sim left on it
void give_stream(int dev, bool high_priority, cudaStream_t st) {
  if (!st) return;
  {
    std::lock_guard<std::mutex> lock(g_mu);
    auto& v = g_streams[dev][high_priority ? 1 : 0];
    if (static_cast<int>(v.size()) < kCachedStreams) {
      v.push_back(st);
      return;
    }
  }
  cudaStreamDestroy(st);
}

void release_pinned_word(int* w) {
  if (!w) return;
  std::lock_guard<std::mutex> lock(g_mu);
  g_pinned_free.push_back(static_cast<int>(w - g_pinned));
}

}  // namespace

struct glisse_sim {
  int device = 0;
  cudaStream_t q = nullptr;  // particle stream (the caller's, or owned)
  cudaStream_t p = nullptr;  // planet-history stream (owned)
  bool own_q = false;
  int np = 0;
  long long n = 0;
  double dt = 0.0, gm0 = 0.0;
  glisse_params prm{};
  int K = 1024;
  int stride = 0;
  int planet_smem = 0;  // dynamic shared memory the planet-history kernel asks for (one SM to itself)
  int status = GLISSE_OK;  // sticky

  PlanetSystem* d_sys = nullptr;
  double* d_j0 = nullptr;    // Jacobi state the planet clock was (re-)seeded with (time of `origin`)
  bool dkd = false;          // GLISSE_SCHEME_DKD: log records are the planets at the HALF steps
  double* d_jhalf = nullptr; // DKD: Jacobi state at origin + 1/2 (start of the half-step clock)
  double* d_jprev = nullptr; // DKD: Jacobi state at step - 1/2 (the last record the particles used)
  double* d_scratch_log = nullptr;   // DKD: 2 records of a one-step planet launch
  double* d_scratch_jlog = nullptr;
  double* d_ptmp = nullptr;  // [6 Np] scratch: heliocentric planet state in / out
  long long* d_fail = nullptr;  // [2] first failed planet step: [0] the sim's clock, [1] scratch of glisse_planet_log
  LogBuffer buf[2];
  int cur = 0;
  bool ahead = false;  // buf[cur ^ 1] holds (or is being filled with) the chunk after buf[cur]'s
  long long step = 0;
  long long origin = 0;        // step at which the planet clock was (re-)seeded: chunks are counted from it
  bool planets_stale = false;  // an external log moved the particles past the internal planet clock

  // particle state: two working sets (ping-pong for compaction) + original-order assembly arrays
  double* work[2][6] = {};
  int* id[2] = {};
  int* flag[2] = {};
  long long* rstep[2] = {};
  double* fin[6] = {};
  int* fin_flag = nullptr;
  long long* fin_rstep = nullptr;
  int* d_nslots = nullptr;  // [2], indexed like the working sets
  int* d_block_counts = nullptr;
  unsigned char* d_bin = nullptr;
  int w = 0;                // working set in use
  int nslots_upper = 0;     // host upper bound of d_nslots[w]
  int* h_nslots = nullptr;  // pinned
  cudaEvent_t nslots_ready = nullptr;
  bool nslots_pending = false;

  // launch chain of the particle kernel (particles.cu): completion lists and tickets, by launch parity
  int* d_list[2] = {};
  unsigned* d_ticket = nullptr;   // [2]
  int* d_error = nullptr;
  int chain_len = 0;              // launches in the open chain (0 = the next launch starts one)
  int chain_groups = 0;
  bool stats_on = false;
  bool refine = false;            // particle-kernel instantiation with the third-order Kepler starting point
  bool definition_only = false;   // ... with the definition's Kepler solver alone (kepler_iters / kepler_tol)
  bool binning = false;           // survivors ordered by Kepler-solver hardness at every resync (bin_iterations)
  unsigned long long hard_at_create = 0;   // bodies that wanted the third-order starting point at create
  unsigned long long* d_stats = nullptr;  // [3]

  // snapshot staging (glisse_snapshot): a copy in original order that stream r ships to the caller
  double* snap[6] = {};
  int* snap_flag = nullptr;
  long long* snap_rstep = nullptr;
  cudaStream_t r = nullptr;            // snapshot copy stream
  cudaEvent_t snap_ready = nullptr;    // staging written            (stream Q)
  cudaEvent_t snap_done = nullptr;     // staging copied to the caller (stream R)
  bool snap_in_flight = false;
  // output ring (glisse_snapshot_ring)
  int ring_kind = 0, ring_slots = 0;
  double* ring_data = nullptr;
  int* ring_flag = nullptr;
  long long* ring_rstep = nullptr;
  long long* ring_step = nullptr;
  long long ring_emitted = 0;
  long long* d_ring_steps = nullptr;   // device [kRingStepWords]: sources of the slot_step copies (written by the
  int ring_step_next = 0;              // sample pass, so the copy on stream r is an ordinary async D2H / D2D)

  // resonant-argument record (glisse_resonance_*), original order
  LibrationRecord lib{};
  double* d_amp_mean = nullptr;
  int res_planet = -1, res_p = 0, res_q = 0;
  double res_window = 0.0;
  long long res_samples = 0;
  std::vector<double> gm_planet_host;

  unsigned long long* d_counters = nullptr;  // [0] particle-steps, [1] scratch for counts
  long long launches = 0;

  void* arena = nullptr;  // one device allocation behind every pointer above
  ParticleArgs pa{};
  std::vector<TimedLaunch> timed_free, timed_busy;
  double timed_ms = 0.0;
  long long timed_launches = 0;
};

namespace {

#define CK(call)                                 \
  do {                                           \
    cudaError_t e__ = (call);                    \
    if (e__ != cudaSuccess) {                    \
      (void)cudaGetLastError();                  \
      return (e__ == cudaErrorMemoryAllocation) ? GLISSE_ENOMEM : GLISSE_ECUDA; \
    }                                            \
  } while (0)

// same, for use after the sim exists: a failure is sticky
#define CKS(sim, call)                           \
  do {                                           \
    cudaError_t e__ = (call);                    \
    if (e__ != cudaSuccess) {                    \
      (void)cudaGetLastError();                  \
      (sim)->status = (e__ == cudaErrorMemoryAllocation) ? GLISSE_ENOMEM : GLISSE_ECUDA; \
      return (sim)->status;                      \
    }                                            \
  } while (0)

// upper 32 bits of a double (sign, exponent, top of the mantissa)
int high_word(double v) {
  unsigned long long b;
  std::memcpy(&b, &v, sizeof(b));
  return static_cast<int>(b >> 32);
}

bool all_finite_host(const double* p, long long n) {
  for (long long i = 0; i < n; ++i)
    if (!std::isfinite(p[i])) return false;
  return true;
}

void free_sim(glisse_sim* s) {
  if (!s) return;
  cudaSetDevice(s->device);
  if (s->q) cudaStreamSynchronize(s->q);
  if (s->p) cudaStreamSynchronize(s->p);
  if (s->r) cudaStreamSynchronize(s->r);
  if (s->snap_ready) cudaEventDestroy(s->snap_ready);
  if (s->snap_done) cudaEventDestroy(s->snap_done);
  for (int b = 0; b < 2; ++b) {
    if (s->buf[b].ready) cudaEventDestroy(s->buf[b].ready);
    if (s->buf[b].consumed) cudaEventDestroy(s->buf[b].consumed);
  }
  if (s->arena) {
    cudaStream_t fs = s->q ? s->q : s->p;
    if (!fs || cudaFreeAsync(s->arena, fs) != cudaSuccess) cudaFree(s->arena);
    if (fs) cudaStreamSynchronize(fs);
  }
  release_pinned_word(s->h_nslots);
  if (s->nslots_ready) cudaEventDestroy(s->nslots_ready);
  for (auto& t : s->timed_free) { cudaEventDestroy(t.t0); cudaEventDestroy(t.t1); }
  for (auto& t : s->timed_busy) { cudaEventDestroy(t.t0); cudaEventDestroy(t.t1); }
  if (s->r && cudaStreamSynchronize(s->r) == cudaSuccess) give_stream(s->device, false, s->r);
  if (s->p && cudaStreamSynchronize(s->p) == cudaSuccess) give_stream(s->device, true, s->p);
  if (s->own_q && s->q && cudaStreamSynchronize(s->q) == cudaSuccess) give_stream(s->device, false, s->q);
  (void)cudaGetLastError();
  delete s;
}

// collect finished timed launches (non-blocking unless `block`)
void harvest_timings(glisse_sim* s, bool block) {
  size_t kept = 0;
  for (size_t i = 0; i < s->timed_busy.size(); ++i) {
    TimedLaunch t = s->timed_busy[i];
    cudaError_t e = block ? cudaEventSynchronize(t.t1) : cudaEventQuery(t.t1);
    if (e == cudaSuccess) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, t.t0, t.t1) == cudaSuccess) {
        s->timed_ms += ms;
        s->timed_launches += 1;
      }
      s->timed_free.push_back(t);
    } else {
      (void)cudaGetLastError();
      s->timed_busy[kept++] = t;
    }
  }
  s->timed_busy.resize(kept);
}

// Anything other than a particle-kernel launch that is enqueued on stream q ends the open launch chain:
// the next particle launch is an ordinary one (full stream order) and starts a new chain.
void break_chain(glisse_sim* s) { s->chain_len = 0; }

// Advance every slot of the working set by `nsteps` steps with the planet log at `log` (record 0 = the
// current step).  Issued as back-to-back launches of prm.segment_steps steps; all but the first of a
// chain ask for programmatic stream serialisation and take their particle groups from the completion
// list of the launch before (particles.cu), so the device stays full while a launch drains.  The whole
// run is bracketed by one pair of timing events (the launches overlap by design).
int launch_particles(glisse_sim* s, const double* log, int nsteps) {
  ParticleArgs& a = s->pa;
  const int w = s->w;
  for (int k = 0; k < 6; ++k) a.st[k] = s->work[w][k];
  a.flag = s->flag[w];
  a.rstep = s->rstep[w];
  a.n_slots = s->d_nslots + w;
  // a newer survivor count may have arrived from the last compaction: shrink the grid (never blocks)
  if (s->nslots_pending && cudaEventQuery(s->nslots_ready) == cudaSuccess) {
    s->nslots_upper = *s->h_nslots;
    s->nslots_pending = false;
  }
  (void)cudaGetLastError();
  const int per_group = particles_per_group();
  const int groups = std::max(1, (s->nslots_upper + per_group - 1) / per_group);
  if (groups != s->chain_groups) break_chain(s);

  TimedLaunch t{};
  bool timed = false;
  if (s->timed_free.empty() && s->timed_busy.size() >= 256) harvest_timings(s, false);
  if (!s->timed_free.empty()) {
    t = s->timed_free.back();
    s->timed_free.pop_back();
    timed = true;
  } else if (s->timed_busy.size() < 256) {
    if (cudaEventCreate(&t.t0) == cudaSuccess && cudaEventCreate(&t.t1) == cudaSuccess) timed = true;
  }
  if (timed) {
    cudaEventRecord(t.t0, s->q);
    break_chain(s);   // an event record sits between this run and the launch before it
  }
  const int seg = s->prm.segment_steps > 0 ? s->prm.segment_steps : nsteps;
  for (int off = 0; off < nsteps; off += seg) {
    const int m = std::min(seg, nsteps - off);
    const bool first = s->chain_len == 0;
    if (first) {  // a new chain: clear both completion lists and tickets
      CKS(s, cudaMemsetAsync(s->d_list[0], 0, sizeof(int) * groups, s->q));
      CKS(s, cudaMemsetAsync(s->d_list[1], 0, sizeof(int) * groups, s->q));
      CKS(s, cudaMemsetAsync(s->d_ticket, 0, 2 * sizeof(unsigned), s->q));
      s->chain_groups = groups;
    }
    const int par = s->chain_len & 1;
    a.wait_list = first ? nullptr : s->d_list[par ^ 1];
    a.done_list = s->d_list[par];
    a.done_ticket = s->d_ticket + par;
    a.ticket_base = static_cast<unsigned>(s->chain_len >> 1) * static_cast<unsigned>(groups);
    a.log = log + static_cast<size_t>(off) * s->stride;
    a.step0 = s->step + off;
    a.nsteps = m;
    CKS(s, launch_particle_kernel(a, groups, !first, s->stats_on, s->dkd, s->refine, s->definition_only, s->q));
    s->launches += 1;
    s->chain_len += 1;
  }
  if (timed) {
    cudaEventRecord(t.t1, s->q);
    break_chain(s);
    s->timed_busy.push_back(t);
  }
  return GLISSE_OK;
}

int run_compaction(glisse_sim* s) {
  break_chain(s);
  const int w = s->w, o = w ^ 1;
  CompactArgs c{};
  for (int k = 0; k < 6; ++k) {
    c.src[k] = s->work[w][k];
    c.dst[k] = s->work[o][k];
    c.fin[k] = s->fin[k];
  }
  c.src_id = s->id[w]; c.dst_id = s->id[o];
  c.src_flag = s->flag[w]; c.src_rstep = s->rstep[w];
  c.dst_flag = s->flag[o]; c.dst_rstep = s->rstep[o];
  c.fin_flag = s->fin_flag; c.fin_rstep = s->fin_rstep;
  c.n_in = s->d_nslots + w;
  c.n_out = s->d_nslots + o;
  c.n_out_host = s->h_nslots;
  c.block_counts = s->d_block_counts;
  c.bin = s->d_bin;
  c.bins = s->binning ? kCompactBins : 1;
  c.mu = s->gm0;
  c.dt = s->dkd ? 0.5 * s->dt : s->dt;
  c.refine = s->refine ? 1 : 0;
  CKS(s, launch_compaction(c, s->nslots_upper, s->q, &s->launches));
  s->w = o;
  // survivor count to the host without blocking: the scan kernel stores it into the mapped pinned word
  // itself (no copy in this stream: a device-to-host copy here queues behind a snapshot's copies on
  // the same copy engine and held the next chunk back by 0.2 ms); the next launches use it once the
  // event says it has arrived
  CKS(s, cudaEventRecord(s->nslots_ready, s->q));
  s->nslots_pending = true;
  return GLISSE_OK;
}

// Steps in the log buffer that starts at step `start`.  The first chunk after the planet clock is
// (re-)seeded is cut into pieces of 64, 64, 128, 256, ... steps (summing to K): the planet-history
// kernel is serial in time, so a full first chunk would keep the particles waiting for K x 1 us before
// their first step; after the ramp the planets stay one buffer ahead.  Results do not depend on the
// cut.  From kNoRampParticles particles on the first chunk is NOT cut: the pieces are
// separate launch chains (an event wait between two launches ends the programmatic chaining), each with
// a tail of its own that costs more than one wave of particles waiting once — 1.0 ms of the first
// chunk at 2^20 particles, where the upload alone outlasts the planet kernel's K steps.
constexpr long long kNoRampParticles = 1LL << 18;
int buffer_len(const glisse_sim* s, long long start) {
  const int K = s->K;
  const long long rel = start - s->origin;
  if (K < 256 || rel >= K || s->n >= kNoRampParticles) return K;
  if (rel == 0) return 64;
  return static_cast<int>(std::min<long long>(rel, K - rel));
}

// planet-history kernel into buffer b, starting from the Jacobi state `jin` at step `start`
int fill_log_buffer(glisse_sim* s, int b, const double* jin, long long start) {
  LogBuffer& B = s->buf[b];
  CKS(s, cudaStreamWaitEvent(s->p, B.consumed, 0));
  CKS(s, launch_planet_kernel(s->d_sys, s->np, jin, B.log, B.jlog, buffer_len(s, start), s->dt, start, s->d_fail,
                              s->planet_smem, s->p));
  B.len = buffer_len(s, start);
  s->launches += 1;
  CKS(s, cudaEventRecord(B.ready, s->p));
  B.start = start;
  return GLISSE_OK;
}

// (Re-)start the planet clock at step `start` from the synchronised Jacobi state in d_j0, into buffer 0.
// KDK: record 0 is that state.  DKD: the log holds the planets at the half steps, so the clock starts
// with ONE Wisdom-Holman step of dt/2 (a one-step planet launch into scratch) and goes on from there.
int start_planet_clock(glisse_sim* s, long long start) {
  s->origin = start;
  s->cur = 0;
  s->ahead = false;
  const double* j0 = s->d_j0;
  if (s->dkd && s->np > 0) {
    CKS(s, launch_planet_kernel(s->d_sys, s->np, s->d_j0, s->d_scratch_log, s->d_scratch_jlog, 1, 0.5 * s->dt, start,
                                s->d_fail, 0, s->p));
    s->launches += 1;
    CKS(s, cudaMemcpyAsync(s->d_jhalf, s->d_scratch_jlog + 6 * s->np, sizeof(double) * 6 * s->np,
                           cudaMemcpyDeviceToDevice, s->p));
    j0 = s->d_jhalf;
  }
  return fill_log_buffer(s, 0, j0, start);
}

// Heliocentric planet positions / velocities at the CURRENT step into d_ptmp (q | qd), on stream q.
// KDK: the Jacobi state of the current record.  DKD: the records sit at the half steps, so the state at
// the integer step is half a Wisdom-Holman step on from the last record the particles used (d_jprev),
// or the seed itself at the clock's origin.
int planets_at_current_step(glisse_sim* s) {
  const int np = s->np;
  double* d_out = s->d_ptmp;
  const double* js = nullptr;
  if (!s->dkd) {
    const LogBuffer& B = s->buf[s->cur];
    const long long off = s->step - B.start;
    CKS(s, cudaStreamWaitEvent(s->q, B.ready, 0));
    js = B.jlog + static_cast<size_t>(off) * 6 * np;
  } else if (s->step == s->origin) {
    js = s->d_j0;
  } else {
    CKS(s, launch_planet_kernel(s->d_sys, np, s->d_jprev, s->d_scratch_log, s->d_scratch_jlog, 1, 0.5 * s->dt,
                                s->step, s->d_fail + 1, 0, s->q));
    s->launches += 1;
    js = s->d_scratch_jlog + 6 * np;
  }
  CKS(s, launch_planet_read(s->d_sys, js, d_out, d_out + 3 * np, s->q));
  s->launches += 1;
  return GLISSE_OK;
}

// Waits for everything the caller has asked for.  The planet stream may still be working on a chunk
// AHEAD of the particles: that is not waited for (every chunk the particles have used is complete,
// the particle kernel waited for it), and a planet failure in it concerns the caller only once the
// particles have gone past the failed step (glisse_internal.cuh: kNoPlanetFailure).
int sync_all(glisse_sim* s) {
  CKS(s, cudaStreamSynchronize(s->q));
  if (s->nslots_pending) {
    s->nslots_upper = *s->h_nslots;
    s->nslots_pending = false;
  }
  harvest_timings(s, true);
  if (s->status == GLISSE_OK) {
    long long fail = kNoPlanetFailure;
    int err = 0;
    CKS(s, cudaMemcpy(&fail, s->d_fail, sizeof(fail), cudaMemcpyDeviceToHost));
    CKS(s, cudaMemcpy(&err, s->d_error, sizeof(err), cudaMemcpyDeviceToHost));
    if (err != 0) s->status = GLISSE_ECUDA;              // a chained warp gave up waiting (particles.cu)
    else if (!s->planets_stale && fail < s->step) s->status = GLISSE_EPLANET;
  }
  return s->status;
}

template <class T>
cudaError_t dmalloc(T** p, size_t count) {
  return cudaMalloc(reinterpret_cast<void**>(p), (count ? count : 1) * sizeof(T));
}

ScatterArgs scatter_args(const glisse_sim* s) {
  ScatterArgs g{};
  const int w = s->w;
  for (int k = 0; k < 6; ++k) {
    g.st[k] = s->work[w][k];
    g.fin[k] = s->fin[k];
  }
  g.id = s->id[w]; g.flag = s->flag[w]; g.rstep = s->rstep[w];
  g.n_slots = s->d_nslots + w;
  g.fin_flag = s->fin_flag; g.fin_rstep = s->fin_rstep;
  return g;
}

int ensure_snapshot_stream(glisse_sim* s) {
  if (!s->r) {  // first snapshot of this sim: its copy stream and events
    CKS(s, take_stream(s->device, false, &s->r));
    CKS(s, cudaEventCreateWithFlags(&s->snap_ready, cudaEventDisableTiming));
    CKS(s, cudaEventCreateWithFlags(&s->snap_done, cudaEventDisableTiming));
  }
  return GLISSE_OK;
}

// One sample of the state at the current step, on stream q: working order -> original order, then ONE
// pass that writes the snapshot staging copy (if out != null) and / or updates the resonance record
// (if resonance): the elements are computed once for both.  The staging copy is shipped to the caller's
// buffers by stream r; `slot_step` (may be null) receives the step count after the data.
int enqueue_sample(glisse_sim* s, bool snapshot, int kind, double* const out[6], int* flag, long long* removal_step,
                   long long* slot_step, bool resonance) {
  break_chain(s);
  if (snapshot) {
    const int st = ensure_snapshot_stream(s);
    if (st != GLISSE_OK) return st;
    // the staging arrays are free once the previous snapshot's copies are done (device-side wait)
    if (s->snap_in_flight) CKS(s, cudaStreamWaitEvent(s->q, s->snap_done, 0));
  }
  CKS(s, launch_scatter_to_original(scatter_args(s), s->nslots_upper, s->q));
  s->launches += 1;
  SampleArgs a{};
  for (int k = 0; k < 6; ++k) {
    a.fin[k] = s->fin[k];
    a.out[k] = s->snap[k];
  }
  a.fin_flag = s->fin_flag; a.fin_rstep = s->fin_rstep;
  a.out_flag = s->snap_flag; a.out_rstep = s->snap_rstep;
  a.n = s->n;
  a.mu = s->gm0;
  a.do_snapshot = snapshot ? 1 : 0;
  a.kind = kind;
  a.do_resonance = resonance ? 1 : 0;
  long long* step_word = nullptr;
  if (snapshot && slot_step) {  // the step count travels with the staging copy (no host-to-host copy: that
    step_word = s->d_ring_steps + (s->ring_step_next++ % kRingStepWords);   // one would stall the enqueueing thread)
    a.step = s->step;
    a.step_out = step_word;
  }
  if (resonance) {
    // planets at the current step: heliocentric q, qd
    const int np = s->np;
    double* d_out = s->d_ptmp;
    const int sp = planets_at_current_step(s);
    if (sp != GLISSE_OK) return sp;
    a.planet_q = d_out + 3 * s->res_planet;
    a.planet_qd = d_out + 3 * np + 3 * s->res_planet;
    a.mu_planet = s->gm0 + s->gm_planet_host[s->res_planet];
    a.window = s->res_window;
    a.p = s->res_p; a.q = s->res_q;
    a.lib = s->lib;
    s->res_samples += 1;
  }
  CKS(s, launch_sample(a, s->q));
  s->launches += 1;
  if (!snapshot) return GLISSE_OK;
  CKS(s, cudaEventRecord(s->snap_ready, s->q));
  // from here on the particle stream is free to go on; stream r ships the staging copy
  CKS(s, cudaStreamWaitEvent(s->r, s->snap_ready, 0));
  const size_t N = static_cast<size_t>(s->n);
  for (int k = 0; k < 6; ++k)
    if (out && out[k]) CKS(s, cudaMemcpyAsync(out[k], s->snap[k], N * sizeof(double), cudaMemcpyDefault, s->r));
  if (flag) CKS(s, cudaMemcpyAsync(flag, s->snap_flag, N * sizeof(int), cudaMemcpyDefault, s->r));
  if (removal_step)
    CKS(s, cudaMemcpyAsync(removal_step, s->snap_rstep, N * sizeof(long long), cudaMemcpyDefault, s->r));
  if (step_word)  // after the data, same stream: a host polling a pinned slot_step sees complete slots
    CKS(s, cudaMemcpyAsync(slot_step, step_word, sizeof(long long), cudaMemcpyDefault, s->r));
  CKS(s, cudaEventRecord(s->snap_done, s->r));
  s->snap_in_flight = true;
  return GLISSE_OK;
}

// What happens when the step count reaches a multiple of K (counted from the planet clock's origin): the
// periodic outputs and the resync, each at its own interval in chunks.
int chunk_boundary(glisse_sim* s) {
  const long long chunk = (s->step - s->origin) / s->K;   // chunks completed
  const glisse_params& P = s->prm;
  const bool snap = P.snapshot_chunks > 0 && s->ring_slots > 0 && chunk % P.snapshot_chunks == 0;
  const bool res = P.resonance_chunks > 0 && s->res_planet >= 0 && !s->planets_stale && chunk % P.resonance_chunks == 0;
  if (snap || res) {
    double* out[6] = {};
    int* fl = nullptr;
    long long *rs = nullptr, *ss = nullptr;
    if (snap) {
      const size_t slot = static_cast<size_t>(s->ring_emitted % s->ring_slots), N = static_cast<size_t>(s->n);
      for (int k = 0; k < 6; ++k) out[k] = s->ring_data + (slot * 6 + k) * N;
      if (s->ring_flag) fl = s->ring_flag + slot * N;
      if (s->ring_rstep) rs = s->ring_rstep + slot * N;
      if (s->ring_step) ss = s->ring_step + slot;
    }
    const int st = enqueue_sample(s, snap, s->ring_kind, out, fl, rs, ss, res);
    if (st != GLISSE_OK) return st;
    if (snap) s->ring_emitted += 1;
  }
  if (P.resync_chunks > 0 && chunk % P.resync_chunks == 0) return run_compaction(s);
  return GLISSE_OK;
}

}  // namespace

extern "C" {

void glisse_default_params(glisse_params* p) {
  if (!p) return;
  p->r_min = 0.0;
  p->r_max = std::numeric_limits<double>::infinity();
  p->kepler_iters = 5;
  p->kepler_tol = 1e-14;
  p->chunk_steps = 1024;
  p->resync_chunks = 1;
  p->device = 0;
  p->stream = nullptr;
  p->snapshot_chunks = 0;
  p->resonance_chunks = 0;
  p->bin_iterations = 2;
  p->scheme = GLISSE_SCHEME_KDK;
  p->guess_order = 0;
  p->segment_steps = 128;
}

int glisse_log_stride(int n_planets) {
  return (n_planets < 0 || n_planets > kMaxPlanets) ? 0 : log_stride(n_planets);
}

const char* glisse_strerror(int status) {
  switch (status) {
    case GLISSE_OK: return "ok";
    case GLISSE_EINVAL: return "invalid argument";
    case GLISSE_ECUDA: return "CUDA failure";
    case GLISSE_ENOMEM: return "out of memory";
    case GLISSE_EPLANET: return "a planet's Kepler drift failed (planets must be encounter-free and bound)";
    case GLISSE_ELIMIT: return "size beyond the fixed capacity of a non-allocating entry point";
    default: return "unknown status";
  }
}

int glisse_create(glisse_sim** out, double gm_star, int n_planets, const double* gm_planet, const double* planet_pos,
                  const double* planet_vel, const double* planet_rcrit, long long n_particles,
                  const double* const pos[3], const double* const vel[3], double dt, const glisse_params* params) {
  if (!out) return GLISSE_EINVAL;
  *out = nullptr;
  if (n_planets < 0 || n_planets > kMaxPlanets || n_particles < 1 || n_particles >= (1LL << 31) || !pos || !vel)
    return GLISSE_EINVAL;
  if (!(gm_star > 0.0) || !std::isfinite(gm_star) || dt == 0.0 || !std::isfinite(dt)) return GLISSE_EINVAL;
  if (n_planets > 0 && (!gm_planet || !planet_pos || !planet_vel)) return GLISSE_EINVAL;
  for (int k = 0; k < 3; ++k)
    if (!pos[k] || !vel[k]) return GLISSE_EINVAL;
  if (n_planets > 0) {
    if (!all_finite_host(gm_planet, n_planets) || !all_finite_host(planet_pos, 3LL * n_planets) ||
        !all_finite_host(planet_vel, 3LL * n_planets))
      return GLISSE_EINVAL;
    for (int j = 0; j < n_planets; ++j)
      if (!(gm_planet[j] > 0.0)) return GLISSE_EINVAL;
    if (planet_rcrit && !all_finite_host(planet_rcrit, n_planets)) return GLISSE_EINVAL;
  }
  glisse_params prm;
  glisse_default_params(&prm);
  if (params) prm = *params;
  if (prm.kepler_iters < 0 || !(prm.kepler_tol > 0.0) || prm.chunk_steps < 1 || prm.chunk_steps > 16384 ||
      prm.resync_chunks < 0 || prm.device < 0 || std::isnan(prm.r_min) || std::isnan(prm.r_max) ||
      prm.snapshot_chunks < 0 || prm.resonance_chunks < 0 || prm.segment_steps < 0 ||
      (prm.scheme != GLISSE_SCHEME_KDK && prm.scheme != GLISSE_SCHEME_DKD) ||
      (prm.guess_order != 0 && prm.guess_order != 1 && prm.guess_order != 3) || prm.bin_iterations < 0 ||
      prm.bin_iterations > 2)
    return GLISSE_EINVAL;

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || prm.device >= ndev) {
    (void)cudaGetLastError();
    return GLISSE_ECUDA;
  }
  CK(cudaSetDevice(prm.device));

  glisse_sim* s = new (std::nothrow) glisse_sim;
  if (!s) return GLISSE_ENOMEM;
  s->device = prm.device;
  s->prm = prm;
  s->np = n_planets;
  s->n = n_particles;
  s->dt = dt;
  s->gm0 = gm_star;
  s->K = prm.chunk_steps;
  s->dkd = prm.scheme == GLISSE_SCHEME_DKD;
  s->stride = log_stride(n_planets);
  const long long N = n_particles;
  const int np = n_planets;

#define CKF(call)                         \
  do {                                    \
    cudaError_t e2__ = (call);            \
    if (e2__ != cudaSuccess) {            \
      (void)cudaGetLastError();           \
      free_sim(s);                        \
      return (e2__ == cudaErrorMemoryAllocation) ? GLISSE_ENOMEM : GLISSE_ECUDA; \
    }                                     \
  } while (0)

  if (prm.stream) {
    s->q = static_cast<cudaStream_t>(prm.stream);
  } else {
    CKF(take_stream(s->device, false, &s->q));
    s->own_q = true;
  }
  {
    // the planet stream at the highest priority: when a planet-history block and the blocks of a
    // particle kernel become runnable together, the planet block (one warp, on the critical path
    // of the NEXT chunk, and needing an SM to itself) must be placed first
    CKF(take_stream(s->device, true, &s->p));
  }
  CKF(configure_particle_kernels());
  CKF(configure_planet_kernels(&s->planet_smem));

  // ---- allocations: one device arena, carved at 256-byte boundaries ------------------------------
  const int n_groups = static_cast<int>((N + particles_per_group() - 1) / particles_per_group());
  {
    struct Req { void** p; size_t bytes; };
    std::vector<Req> reqs;
    auto need = [&](auto** p, size_t count) {
      reqs.push_back({reinterpret_cast<void**>(p), (count ? count : 1) * sizeof(**p)});
    };
    for (int b = 0; b < 2; ++b) {
      need(&s->buf[b].log, static_cast<size_t>(s->K + 1) * s->stride);
      need(&s->buf[b].jlog, static_cast<size_t>(s->K + 1) * 6 * np);
      for (int k = 0; k < 6; ++k) need(&s->work[b][k], N);
      need(&s->id[b], N);
      need(&s->flag[b], N);
      need(&s->rstep[b], N);
      need(&s->d_list[b], n_groups);
    }
    for (int k = 0; k < 6; ++k) need(&s->fin[k], N);
    need(&s->fin_flag, N);
    need(&s->fin_rstep, N);
    LibrationRecord& L = s->lib;
    need(&L.phi, N); need(&L.seen0, N); need(&L.seen180, N); need(&L.phi_min, N); need(&L.phi_max, N);
    need(&L.ext_last, N); need(&L.amp_sum, N); need(&L.amp_max, N); need(&L.n_amp, N); need(&L.n_seen, N);
    need(&L.trend, N); need(&L.ext_kind, N);
    need(&s->d_amp_mean, N);
    for (int k = 0; k < 6; ++k) need(&s->snap[k], N);
    need(&s->snap_flag, N);
    need(&s->snap_rstep, N);
    need(&s->d_nslots, 2);
    need(&s->d_block_counts, static_cast<size_t>(kCompactBins) * ((N + 255) / 256 + 1) + 1);
    need(&s->d_bin, N);
    need(&s->d_counters, 3);   // d_counters, d_error, d_stats: consecutive, cleared by ONE memset at create
    need(&s->d_error, 1);
    need(&s->d_stats, 3);
    need(&s->d_ticket, 2);
    need(&s->d_ring_steps, kRingStepWords);
    need(&s->d_fail, 2);
    need(&s->d_sys, 1);
    need(&s->d_j0, static_cast<size_t>(6 * np));
    need(&s->d_jhalf, static_cast<size_t>(6 * np));
    need(&s->d_jprev, static_cast<size_t>(6 * np));
    need(&s->d_scratch_log, static_cast<size_t>(2 * s->stride));
    need(&s->d_scratch_jlog, static_cast<size_t>(2 * 6 * np));
    need(&s->d_ptmp, static_cast<size_t>(6 * np));
    size_t total = 0;
    for (auto& r : reqs) total += (r.bytes + 255) & ~static_cast<size_t>(255);
    cudaMemPool_t pool = nullptr;
    CKF(arena_pool(s->device, &pool));
    CKF(cudaMallocFromPoolAsync(&s->arena, total, pool, s->q));
    // stream-ordered memory: the planet stream may touch it only after the allocation on q
    cudaEvent_t born = nullptr;
    CKF(cudaEventCreateWithFlags(&born, cudaEventDisableTiming));
    cudaError_t eb = cudaEventRecord(born, s->q);
    if (eb == cudaSuccess) eb = cudaStreamWaitEvent(s->p, born, 0);
    cudaEventDestroy(born);
    CKF(eb);
    size_t off = 0;
    for (auto& r : reqs) {
      *r.p = static_cast<char*>(s->arena) + off;
      off += (r.bytes + 255) & ~static_cast<size_t>(255);
    }
  }
  for (int b = 0; b < 2; ++b) {
    CKF(cudaEventCreateWithFlags(&s->buf[b].ready, cudaEventDisableTiming));
    CKF(cudaEventCreateWithFlags(&s->buf[b].consumed, cudaEventDisableTiming));
  }
  s->h_nslots = pinned_word();
  if (!s->h_nslots) {
    free_sim(s);
    return GLISSE_ENOMEM;
  }
  CKF(cudaEventCreateWithFlags(&s->nslots_ready, cudaEventDisableTiming));

  // ---- planet system ----------------------------------------------------------------------------
  PlanetSystem hs{};
  hs.np = np;
  hs.gm0 = gm_star;
  double eta = gm_star;
  for (int j = 0; j < np; ++j) {
    hs.gm[j] = gm_planet[j];
    hs.eta_prev[j] = eta;
    eta += gm_planet[j];
    hs.eta[j] = eta;
  }
  const long long no_fail[2] = {kNoPlanetFailure, kNoPlanetFailure};
  s->gm_planet_host.assign(gm_planet, gm_planet + np);
  CKF(cudaMemcpyAsync(s->d_sys, &hs, sizeof(hs), cudaMemcpyHostToDevice, s->p));
  CKF(cudaMemcpyAsync(s->d_fail, no_fail, sizeof(no_fail), cudaMemcpyHostToDevice, s->p));
  if (np > 0) {
    double* d_q = s->d_ptmp;
    double* d_qd = s->d_ptmp + 3 * np;
    CKF(cudaMemcpyAsync(d_q, planet_pos, sizeof(double) * 3 * np, cudaMemcpyHostToDevice, s->p));
    CKF(cudaMemcpyAsync(d_qd, planet_vel, sizeof(double) * 3 * np, cudaMemcpyHostToDevice, s->p));
    CKF(launch_planet_init(s->d_sys, d_q, d_qd, s->d_j0, s->p));
    s->launches += 1;
  }
  CKF(cudaStreamSynchronize(s->p));  // the caller's planet arrays and `hs` are consumed
  // chunk 0 into buffer 0; the chunk after it is started by the first advance (s->ahead)
  if (start_planet_clock(s, 0) != GLISSE_OK) {
    const int st = s->status;
    free_sim(s);
    return st;
  }

  // ---- particle state ---------------------------------------------------------------------------
  // (finiteness is checked on the device after the upload, for host and device inputs alike: a
  // host loop over 6 N doubles costs more than the whole upload)
  for (int k = 0; k < 3; ++k) {
    CKF(cudaMemcpyAsync(s->work[0][k], pos[k], sizeof(double) * N, cudaMemcpyDefault, s->q));
    CKF(cudaMemcpyAsync(s->work[0][3 + k], vel[k], sizeof(double) * N, cudaMemcpyDefault, s->q));
  }
  CKF(cudaMemsetAsync(s->d_counters, 0,
                      reinterpret_cast<char*>(s->d_stats + 3) - reinterpret_cast<char*>(s->d_counters), s->q));
  {
    // One pass: identity order and cleared flags, the count of non-finite inputs, and the count of bodies that
    // want the third-order Kepler starting point.  guess_order = 0: the starting point is chosen here, once,
    // from the initial conditions (deterministic: the same inputs always give the same instantiation, whatever
    // K, R or the schedule); the same count decides automatic binning.
    CKF(launch_create_pass(s->work[0], N, gm_star, (s->dkd ? 0.5 : 1.0) * dt, s->d_counters + 1, s->id[0], s->flag[0],
                           s->rstep[0], s->fin_flag, s->fin_rstep, s->q));
    s->launches += 1;
    unsigned long long cnt[2] = {0, 0};   // non-finite inputs, bodies wanting the third-order starting point
    CKF(cudaMemcpyAsync(cnt, s->d_counters + 1, sizeof(cnt), cudaMemcpyDeviceToHost, s->q));
    CKF(cudaStreamSynchronize(s->q));
    if (cnt[0]) {
      free_sim(s);
      return GLISSE_EINVAL;
    }
    s->refine = prm.guess_order == 3 || (prm.guess_order == 0 && 20 * cnt[1] > static_cast<unsigned long long>(N));
    s->hard_at_create = cnt[1];
  }
  const int nsl[2] = {static_cast<int>(N), 0};
  CKF(cudaMemcpyAsync(s->d_nslots, nsl, sizeof(nsl), cudaMemcpyHostToDevice, s->q));
  s->nslots_upper = static_cast<int>(N);
  s->w = 0;

  // ---- constant part of the particle-kernel arguments --------------------------------------------
  ParticleArgs& a = s->pa;
  a.pstep_counter = s->d_counters;
  a.error = s->d_error;
  a.solver_stats = s->d_stats;
  a.stride = s->stride;
  a.stage_recs = stage_records(np);
  a.np = np;
  a.iters = prm.kepler_iters;
  a.hdt = 0.5 * dt;
  a.mu = gm_star;
  a.inv_mu = 1.0 / gm_star;
  a.inv_mu_dt = dt / gm_star;
  a.inv_mu_hdt = 0.5 * dt / gm_star;
  a.rmin2 = (prm.r_min > 0.0) ? prm.r_min * prm.r_min : 0.0;
  a.rmax2 = (prm.r_max > 0.0 && std::isfinite(prm.r_max)) ? prm.r_max * prm.r_max
                                                           : std::numeric_limits<double>::infinity();
  a.tol = prm.kepler_tol;
  a.two_mu = 2.0 * gm_star;
  s->definition_only = !fast_solver_allowed(prm.kepler_iters, prm.kepler_tol);
  for (int j = 0; j < kMaxPlanets; ++j) {
    a.gm[j] = (j < np) ? gm_planet[j] : 0.0;
    a.rc2[j] = (j < np && planet_rcrit) ? planet_rcrit[j] * planet_rcrit[j] : 0.0;
    a.rc2_hi[j] = high_word(a.rc2[j]);
  }
  a.rmin2_hi = high_word(a.rmin2);
  a.rmax2_hi = high_word(a.rmax2);
  // iteration-count binning: the initial order is binned too (nothing is removed by it)
  // 2 = automatic: on if at least one body in a thousand is a hard one at create (the count of bodies that
  // want the third-order starting point), or if the population was given that starting point
  s->binning = prm.bin_iterations == 1 || (prm.bin_iterations == 2 && (s->refine || s->hard_at_create * 1000ULL >= static_cast<unsigned long long>(N)));
  if (s->binning && run_compaction(s) != GLISSE_OK) {
    const int st = s->status;
    free_sim(s);
    return st;
  }
  // the caller's buffers are free again once the copies on q are done; the planet stream keeps
  // running (a planet failure is reported by a synchronising call once the particles are past it)
  CKF(cudaStreamSynchronize(s->q));
#undef CKF
  *out = s;
  return GLISSE_OK;
}

int glisse_advance(glisse_sim* s, long long n_steps) {
  if (!s || n_steps < 0) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (s->planets_stale) return GLISSE_EINVAL;  // the internal planet clock is stale: glisse_set_planets
  CKS(s, cudaSetDevice(s->device));
  const int np = s->np;
  while (n_steps > 0) {
    const LogBuffer& B = s->buf[s->cur];
    const long long off = s->step - B.start;  // 0 <= off < B.len: an exhausted buffer is left at once
    if (!s->ahead) {
      // the planet stream works one chunk ahead: the other buffer gets the chunk after this one
      // while the particles work through this one.  Queued BEFORE the particle kernel so that the
      // planet-history block (which takes an SM to itself, planets.cu) is resident before the
      // particles fill the device, and only when particles are about to be advanced: a caller that
      // stops here never pays for a chunk it does not use.
      const int sf = fill_log_buffer(s, s->cur ^ 1, B.jlog + static_cast<size_t>(B.len) * 6 * np, B.start + B.len);
      if (sf != GLISSE_OK) return sf;
      s->ahead = true;
    }
    CKS(s, cudaStreamWaitEvent(s->q, B.ready, 0));
    break_chain(s);
    const int m = static_cast<int>(std::min<long long>(n_steps, B.len - off));
    const int st = launch_particles(s, B.log + static_cast<size_t>(off) * s->stride, m);
    if (st != GLISSE_OK) return st;
    if (s->dkd && np > 0) {  // the Jacobi state at (new step) - 1/2: record off + m - 1 of this buffer
      CKS(s, cudaMemcpyAsync(s->d_jprev, B.jlog + static_cast<size_t>(off + m - 1) * 6 * np, sizeof(double) * 6 * np,
                             cudaMemcpyDeviceToDevice, s->q));
      break_chain(s);
    }
    s->step += m;
    n_steps -= m;
    if (off + m == B.len) {  // this buffer is used up: the planet stream may overwrite it
      CKS(s, cudaEventRecord(s->buf[s->cur].consumed, s->q));
      break_chain(s);
      s->cur ^= 1;
      s->ahead = false;
    }
    if ((s->step - s->origin) % s->K == 0) {  // a chunk is complete: periodic outputs, resync
      const int sc = chunk_boundary(s);
      if (sc != GLISSE_OK) return sc;
    }
  }
  return GLISSE_OK;
}

// The external log goes through the sim's own two log buffers, chunk by chunk: upload of chunk c+1 on
// the planet stream while the particle kernel works on chunk c — the paper's double-buffered PCIe
// design.  No allocation, no host synchronisation.
int glisse_advance_with_log(glisse_sim* s, long long n_steps, const double* log) {
  if (!s || n_steps < 0 || !log) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (n_steps == 0) return GLISSE_OK;
  CKS(s, cudaSetDevice(s->device));
  if (!s->planets_stale) {
    // From here on the two buffers hold the caller's planets.  The look-ahead planet kernel may still
    // be writing one of them (the uploads below follow it on the same stream p) and particle kernels
    // already queued on q may still be reading the other: the uploads wait for those through the
    // buffers' `consumed` events, recorded now.
    for (int b = 0; b < 2; ++b) CKS(s, cudaEventRecord(s->buf[b].consumed, s->q));
    break_chain(s);
    s->planets_stale = true;
    s->ahead = false;
  }
  // upload records [first, first + m] of the caller's log into buffer b as the chunk starting at `start`
  auto upload = [&](int b, long long first, long long start) -> int {
    const int m = static_cast<int>(std::min<long long>(n_steps - first, s->K));
    LogBuffer& B = s->buf[b];
    CKS(s, cudaStreamWaitEvent(s->p, B.consumed, 0));
    CKS(s, cudaMemcpyAsync(B.log, log + static_cast<size_t>(first) * s->stride,
                           static_cast<size_t>(m + 1) * s->stride * sizeof(double), cudaMemcpyDefault, s->p));
    CKS(s, cudaEventRecord(B.ready, s->p));
    B.start = start;
    B.len = m;
    return GLISSE_OK;
  };
  const long long step_at_entry = s->step;
  long long done = 0, uploaded = 0;
  int b = s->cur;
  {
    const int st = upload(b, 0, step_at_entry);
    if (st != GLISSE_OK) return st;
    uploaded = s->buf[b].len;
  }
  while (done < n_steps) {
    LogBuffer& B = s->buf[b];
    if (uploaded < n_steps) {  // next chunk into the other buffer while this one is worked through
      const int st = upload(b ^ 1, uploaded, step_at_entry + uploaded);
      if (st != GLISSE_OK) return st;
      uploaded += s->buf[b ^ 1].len;
    }
    CKS(s, cudaStreamWaitEvent(s->q, B.ready, 0));
    break_chain(s);
    const int st = launch_particles(s, B.log, B.len);
    if (st != GLISSE_OK) return st;
    s->step += B.len;
    done += B.len;
    CKS(s, cudaEventRecord(B.consumed, s->q));
    break_chain(s);
    if (B.len == s->K) {   // every full chunk of the external history counts as a chunk
      const int sc = chunk_boundary(s);
      if (sc != GLISSE_OK) return sc;
    }
    b ^= 1;
  }
  s->cur = b;
  return GLISSE_OK;
}

int glisse_set_planets(glisse_sim* s, const double* planet_pos, const double* planet_vel) {
  if (!s) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  const int np = s->np;
  if (np > 0 && (!planet_pos || !planet_vel)) return GLISSE_EINVAL;
  if (np > 0 && (!all_finite_host(planet_pos, 3LL * np) || !all_finite_host(planet_vel, 3LL * np))) return GLISSE_EINVAL;
  CKS(s, cudaSetDevice(s->device));
  // everything queued on either stream uses the old clock: let it finish, then restart at this step
  CKS(s, cudaStreamSynchronize(s->p));
  CKS(s, cudaStreamSynchronize(s->q));
  if (np > 0) {
    double* d_q = s->d_ptmp;
    double* d_qd = s->d_ptmp + 3 * np;
    CKS(s, cudaMemcpyAsync(d_q, planet_pos, sizeof(double) * 3 * np, cudaMemcpyHostToDevice, s->p));
    CKS(s, cudaMemcpyAsync(d_qd, planet_vel, sizeof(double) * 3 * np, cudaMemcpyHostToDevice, s->p));
    CKS(s, launch_planet_init(s->d_sys, d_q, d_qd, s->d_j0, s->p));
    s->launches += 1;
  }
  const long long no_fail = kNoPlanetFailure;
  CKS(s, cudaMemcpyAsync(s->d_fail, &no_fail, sizeof(no_fail), cudaMemcpyHostToDevice, s->p));
  CKS(s, cudaStreamSynchronize(s->p));   // the caller's arrays and `no_fail` are consumed
  s->planets_stale = false;
  return start_planet_clock(s, s->step);
}

int glisse_planet_log(glisse_sim* s, long long n_steps, double* log) {
  if (!s || n_steps < 0 || !log || n_steps > (1LL << 24)) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (s->planets_stale) return GLISSE_EINVAL;
  CKS(s, cudaSetDevice(s->device));
  break_chain(s);
  const int np = s->np;
  const LogBuffer& B = s->buf[s->cur];
  const long long off = s->step - B.start;
  double *d_log = nullptr, *d_jlog = nullptr;
  const size_t count = static_cast<size_t>(n_steps + 1) * s->stride;
  const long long no_fail = kNoPlanetFailure;
  long long fail = kNoPlanetFailure;
  CKS(s, dmalloc(&d_log, count));
  cudaError_t e = dmalloc(&d_jlog, static_cast<size_t>(n_steps + 1) * 6 * np);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s->q, B.ready, 0);
  // a scratch failure word: a failure somewhere in this look-ahead does not concern the sim's own clock
  if (e == cudaSuccess) e = cudaMemcpyAsync(s->d_fail + 1, &no_fail, sizeof(no_fail), cudaMemcpyHostToDevice, s->q);
  if (e == cudaSuccess)
    e = launch_planet_kernel(s->d_sys, s->np, B.jlog + static_cast<size_t>(off) * 6 * np, d_log, d_jlog,
                             static_cast<int>(n_steps), s->dt, s->step, s->d_fail + 1, 0, s->q);
  s->launches += 1;
  if (e == cudaSuccess) e = cudaMemcpyAsync(log, d_log, count * sizeof(double), cudaMemcpyDefault, s->q);
  if (e == cudaSuccess) e = cudaMemcpyAsync(&fail, s->d_fail + 1, sizeof(fail), cudaMemcpyDeviceToHost, s->q);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->q);
  cudaFree(d_log);
  cudaFree(d_jlog);
  CKS(s, e);
  const int st = sync_all(s);
  if (st != GLISSE_OK) return st;
  return fail < s->step + n_steps ? GLISSE_EPLANET : GLISSE_OK;   // not sticky: the sim itself is intact
}

long long glisse_planet_log_static_limit(int n_planets) {
  const long long lim = static_planet_log_limit(n_planets);
  return lim < 0 ? GLISSE_EINVAL : lim;
}

// glisse_planet_log without an allocation: the kernel writes the caller's device buffer, its Jacobi-state
// scratch is the static device array of planets.cu.  No cudaMalloc, cudaFree or allocating routine below.
int glisse_planet_log_static(glisse_sim* s, long long n_steps, double* log) {
  if (!s || n_steps < 0 || !log || (reinterpret_cast<uintptr_t>(log) & 15)) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (s->planets_stale) return GLISSE_EINVAL;
  if (n_steps > static_planet_log_limit(s->np)) return GLISSE_ELIMIT;
  CKS(s, cudaSetDevice(s->device));
  {
    // the kernel writes `log` directly: it must be device memory of this device
    cudaPointerAttributes at{};
    if (cudaPointerGetAttributes(&at, log) != cudaSuccess) {
      (void)cudaGetLastError();
      return GLISSE_EINVAL;
    }
    if (at.type != cudaMemoryTypeDevice || at.device != s->device) return GLISSE_EINVAL;
  }
  break_chain(s);
  const int np = s->np;
  const LogBuffer& B = s->buf[s->cur];
  const long long off = s->step - B.start;
  const long long no_fail = kNoPlanetFailure;
  long long fail = kNoPlanetFailure;
  CKS(s, cudaStreamWaitEvent(s->q, B.ready, 0));
  // a scratch failure word: a failure somewhere in this look-ahead does not concern the sim's own clock
  CKS(s, cudaMemcpyAsync(s->d_fail + 1, &no_fail, sizeof(no_fail), cudaMemcpyHostToDevice, s->q));
  CKS(s, launch_planet_kernel_static(s->d_sys, np, B.jlog + static_cast<size_t>(off) * 6 * np, log,
                                     static_cast<int>(n_steps), s->dt, s->step, s->d_fail + 1, s->q));
  s->launches += 1;
  CKS(s, cudaMemcpyAsync(&fail, s->d_fail + 1, sizeof(fail), cudaMemcpyDeviceToHost, s->q));
  const int st = sync_all(s);
  if (st != GLISSE_OK) return st;
  return fail < s->step + n_steps ? GLISSE_EPLANET : GLISSE_OK;   // not sticky: the sim itself is intact
}

int glisse_interpolate_log(glisse_sim* s, long long n_samples, const double* sample_time, const double* sample_pos,
                           const double* sample_vel, double t_first, double dt_record, long long n_records,
                           double* log) {
  if (!s || n_samples < 2 || n_samples > (1LL << 24) || n_records < 0 || n_records > (1LL << 26) || !sample_time || !log ||
      !std::isfinite(t_first) || !std::isfinite(dt_record))
    return GLISSE_EINVAL;
  const int np = s->np;
  if (np > 0 && (!sample_pos || !sample_vel)) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (n_records == 0) return GLISSE_OK;
  CKS(s, cudaSetDevice(s->device));
  break_chain(s);
  // the instants come to the host once (they may live on the device): increasing, and covering the records
  std::vector<double> t(static_cast<size_t>(n_samples));
  CKS(s, cudaMemcpyAsync(t.data(), sample_time, sizeof(double) * n_samples, cudaMemcpyDefault, s->q));
  CKS(s, cudaStreamSynchronize(s->q));
  for (long long m = 0; m + 1 < n_samples; ++m)
    if (!(t[m + 1] > t[m])) return GLISSE_EINVAL;
  const double t_last = t_first + static_cast<double>(n_records - 1) * dt_record;
  if (!(std::min(t_first, t_last) >= t[0]) || !(std::max(t_first, t_last) <= t[n_samples - 1])) return GLISSE_EINVAL;
  const size_t n_state = static_cast<size_t>(n_samples) * 3 * np;
  const size_t count = static_cast<size_t>(n_records) * s->stride;
  double *d_t = nullptr, *d_q = nullptr, *d_v = nullptr, *d_log = nullptr;
  cudaError_t e = dmalloc(&d_t, static_cast<size_t>(n_samples));
  if (e == cudaSuccess) e = dmalloc(&d_q, n_state ? n_state : 1);
  if (e == cudaSuccess) e = dmalloc(&d_v, n_state ? n_state : 1);
  if (e == cudaSuccess) e = dmalloc(&d_log, count);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_t, t.data(), sizeof(double) * n_samples, cudaMemcpyHostToDevice, s->q);
  if (e == cudaSuccess && n_state) e = cudaMemcpyAsync(d_q, sample_pos, sizeof(double) * n_state, cudaMemcpyDefault, s->q);
  if (e == cudaSuccess && n_state) e = cudaMemcpyAsync(d_v, sample_vel, sizeof(double) * n_state, cudaMemcpyDefault, s->q);
  if (e == cudaSuccess)
    e = launch_interpolate_log(s->d_sys, n_samples, d_t, d_q, d_v, t_first, dt_record, n_records, d_log, s->q);
  s->launches += 1;
  if (e == cudaSuccess) e = cudaMemcpyAsync(log, d_log, count * sizeof(double), cudaMemcpyDefault, s->q);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->q);
  cudaFree(d_t);
  cudaFree(d_q);
  cudaFree(d_v);
  cudaFree(d_log);
  CKS(s, e);
  return GLISSE_OK;
}

int glisse_read(glisse_sim* s, double* const pos[3], double* const vel[3], int* flag, long long* removal_step) {
  if (!s) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  break_chain(s);
  CKS(s, launch_scatter_to_original(scatter_args(s), s->nslots_upper, s->q));
  s->launches += 1;
  const size_t N = static_cast<size_t>(s->n);
  for (int k = 0; k < 3; ++k) {
    if (pos && pos[k]) CKS(s, cudaMemcpyAsync(pos[k], s->fin[k], N * sizeof(double), cudaMemcpyDefault, s->q));
    if (vel && vel[k]) CKS(s, cudaMemcpyAsync(vel[k], s->fin[3 + k], N * sizeof(double), cudaMemcpyDefault, s->q));
  }
  if (flag) CKS(s, cudaMemcpyAsync(flag, s->fin_flag, N * sizeof(int), cudaMemcpyDefault, s->q));
  if (removal_step)
    CKS(s, cudaMemcpyAsync(removal_step, s->fin_rstep, N * sizeof(long long), cudaMemcpyDefault, s->q));
  return sync_all(s);
}

int glisse_snapshot(glisse_sim* s, int kind, double* const out[6], int* flag, long long* removal_step) {
  if (!s || (kind != GLISSE_SNAPSHOT_CARTESIAN && kind != GLISSE_SNAPSHOT_ELEMENTS)) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  return enqueue_sample(s, true, kind, out, flag, removal_step, nullptr, false);
}

int glisse_snapshot_wait(glisse_sim* s) {
  if (!s) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (!s->r) return GLISSE_OK;  // no snapshot was ever taken
  CKS(s, cudaSetDevice(s->device));
  CKS(s, cudaStreamSynchronize(s->r));
  return GLISSE_OK;
}

int glisse_snapshot_ring(glisse_sim* s, int kind, int n_slots, double* data, int* flag, long long* removal_step,
                         long long* slot_step) {
  if (!s || n_slots < 0) return GLISSE_EINVAL;
  if (n_slots > 0 && (!data || (kind != GLISSE_SNAPSHOT_CARTESIAN && kind != GLISSE_SNAPSHOT_ELEMENTS)))
    return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  if (s->r) CKS(s, cudaStreamSynchronize(s->r));   // copies into the ring being replaced are done
  s->ring_kind = kind;
  s->ring_slots = n_slots;
  s->ring_data = n_slots ? data : nullptr;
  s->ring_flag = n_slots ? flag : nullptr;
  s->ring_rstep = n_slots ? removal_step : nullptr;
  s->ring_step = n_slots ? slot_step : nullptr;
  s->ring_emitted = 0;
  return GLISSE_OK;
}

long long glisse_snapshots_emitted(glisse_sim* s) { return s ? s->ring_emitted : GLISSE_EINVAL; }

int glisse_resonance_begin(glisse_sim* s, int planet, int p, int q, double window) {
  if (!s || planet < 0 || planet >= s->np || q < 1 || p <= q || !(window > 0.0)) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  break_chain(s);
  CKS(s, launch_libration_reset(s->lib, s->n, s->q));
  s->launches += 1;
  s->res_planet = planet; s->res_p = p; s->res_q = q;
  s->res_window = window;
  s->res_samples = 0;
  return GLISSE_OK;
}

int glisse_resonance_sample(glisse_sim* s) {
  if (!s || s->res_planet < 0) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (s->planets_stale) return GLISSE_EINVAL;  // the internal planet clock is stale
  CKS(s, cudaSetDevice(s->device));
  return enqueue_sample(s, false, 0, nullptr, nullptr, nullptr, nullptr, true);
}

int glisse_resonance_read(glisse_sim* s, unsigned char* seen0, unsigned char* seen180, double* phi_last,
                          long long* n_samples) {
  if (!s || s->res_planet < 0) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  break_chain(s);
  const size_t N = static_cast<size_t>(s->n);
  if (seen0) CKS(s, cudaMemcpyAsync(seen0, s->lib.seen0, N, cudaMemcpyDefault, s->q));
  if (seen180) CKS(s, cudaMemcpyAsync(seen180, s->lib.seen180, N, cudaMemcpyDefault, s->q));
  if (phi_last) CKS(s, cudaMemcpyAsync(phi_last, s->lib.phi, N * sizeof(double), cudaMemcpyDefault, s->q));
  if (n_samples) *n_samples = s->res_samples;
  return sync_all(s);
}

int glisse_libration_read(glisse_sim* s, double* phi_min, double* phi_max, double* amp_mean, double* amp_max,
                          int* n_amp) {
  if (!s || s->res_planet < 0) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  break_chain(s);
  const size_t N = static_cast<size_t>(s->n);
  if (phi_min) CKS(s, cudaMemcpyAsync(phi_min, s->lib.phi_min, N * sizeof(double), cudaMemcpyDefault, s->q));
  if (phi_max) CKS(s, cudaMemcpyAsync(phi_max, s->lib.phi_max, N * sizeof(double), cudaMemcpyDefault, s->q));
  if (amp_mean) {
    CKS(s, launch_libration_mean(s->lib, s->d_amp_mean, s->n, s->q));
    s->launches += 1;
    CKS(s, cudaMemcpyAsync(amp_mean, s->d_amp_mean, N * sizeof(double), cudaMemcpyDefault, s->q));
  }
  if (amp_max) CKS(s, cudaMemcpyAsync(amp_max, s->lib.amp_max, N * sizeof(double), cudaMemcpyDefault, s->q));
  if (n_amp) CKS(s, cudaMemcpyAsync(n_amp, s->lib.n_amp, N * sizeof(int), cudaMemcpyDefault, s->q));
  return sync_all(s);
}

int glisse_read_planets(glisse_sim* s, double* pos, double* vel) {
  if (!s) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (s->planets_stale) return GLISSE_EINVAL;
  CKS(s, cudaSetDevice(s->device));
  const int np = s->np;
  if (np == 0 || (!pos && !vel)) return sync_all(s);
  break_chain(s);
  double* d_out = s->d_ptmp;
  const int sp = planets_at_current_step(s);
  if (sp != GLISSE_OK) return sp;
  if (pos) CKS(s, cudaMemcpyAsync(pos, d_out, sizeof(double) * 3 * np, cudaMemcpyDefault, s->q));
  if (vel) CKS(s, cudaMemcpyAsync(vel, d_out + 3 * np, sizeof(double) * 3 * np, cudaMemcpyDefault, s->q));
  return sync_all(s);
}

long long glisse_active_count(glisse_sim* s) {
  if (!s) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  if (cudaSetDevice(s->device) != cudaSuccess) return GLISSE_ECUDA;
  break_chain(s);
  unsigned long long c = 0;
  cudaError_t e = cudaMemsetAsync(s->d_counters + 1, 0, sizeof(unsigned long long), s->q);
  if (e == cudaSuccess) e = launch_count_active(s->flag[s->w], s->d_nslots + s->w, s->nslots_upper, s->d_counters + 1, s->q);
  s->launches += 1;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&c, s->d_counters + 1, sizeof(c), cudaMemcpyDeviceToHost, s->q);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->q);
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    s->status = GLISSE_ECUDA;
    return GLISSE_ECUDA;
  }
  const int st = sync_all(s);
  return st == GLISSE_OK ? static_cast<long long>(c) : st;
}

long long glisse_step(glisse_sim* s) { return s ? s->step : GLISSE_EINVAL; }

long long glisse_particle_steps(glisse_sim* s) {
  if (!s) return GLISSE_EINVAL;
  const int st = sync_all(s);
  if (st != GLISSE_OK) return st;
  unsigned long long c = 0;
  if (cudaMemcpy(&c, s->d_counters, sizeof(c), cudaMemcpyDeviceToHost) != cudaSuccess) {
    (void)cudaGetLastError();
    s->status = GLISSE_ECUDA;
    return GLISSE_ECUDA;
  }
  return static_cast<long long>(c);
}

long long glisse_launch_count(glisse_sim* s) { return s ? s->launches : GLISSE_EINVAL; }

int glisse_sync(glisse_sim* s) {
  if (!s) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  return sync_all(s);
}

int glisse_particle_kernel_time(glisse_sim* s, double* ms, long long* launches) {
  if (!s) return GLISSE_EINVAL;
  const int st = glisse_sync(s);
  if (ms) *ms = s->timed_ms;
  if (launches) *launches = s->timed_launches;
  s->timed_ms = 0.0;
  s->timed_launches = 0;
  return st;
}

int glisse_solver_stats_enable(glisse_sim* s, int on) {
  if (!s) return GLISSE_EINVAL;
  if (s->status != GLISSE_OK) return s->status;
  CKS(s, cudaSetDevice(s->device));
  break_chain(s);
  CKS(s, cudaMemsetAsync(s->d_stats, 0, 3 * sizeof(unsigned long long), s->q));
  s->stats_on = on != 0;
  return GLISSE_OK;
}

int glisse_solver_stats(glisse_sim* s, long long* warp_steps, long long* warp_iters, long long* warp_slow) {
  if (!s) return GLISSE_EINVAL;
  const int st = glisse_sync(s);
  if (st != GLISSE_OK) return st;
  unsigned long long c[3] = {};
  CKS(s, cudaMemcpy(c, s->d_stats, sizeof(c), cudaMemcpyDeviceToHost));
  if (warp_steps) *warp_steps = static_cast<long long>(c[0]);
  if (warp_iters) *warp_iters = static_cast<long long>(c[1]);
  if (warp_slow) *warp_slow = static_cast<long long>(c[2]);
  return GLISSE_OK;
}

int glisse_fp64_peak_probe(int device, void* stream, double millis, double* flops) {
  if (!flops || device < 0) return GLISSE_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev) {
    (void)cudaGetLastError();
    return GLISSE_ECUDA;
  }
  CK(cudaSetDevice(device));
  CK(run_fp64_probe(static_cast<cudaStream_t>(stream), millis, flops));
  return GLISSE_OK;
}

int glisse_test_primitive(int which, long long n, const double* in, double* out) {
  if (which < 0 || which > 5 || n < 1 || !in || !out) return GLISSE_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    (void)cudaGetLastError();
    return GLISSE_ECUDA;
  }
  const size_t in_per = (which >= 4) ? 10 : 1, out_per = (which >= 4) ? 7 : (which == 3 ? 2 : 1);
  double *d_in = nullptr, *d_out = nullptr;
  CK(dmalloc(&d_in, static_cast<size_t>(n) * in_per));
  cudaError_t e = dmalloc(&d_out, static_cast<size_t>(n) * out_per);
  if (e == cudaSuccess) e = cudaMemcpy(d_in, in, sizeof(double) * n * in_per, cudaMemcpyDefault);
  if (e == cudaSuccess) e = run_primitive(which, n, d_in, d_out, nullptr);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (e == cudaSuccess) e = cudaMemcpy(out, d_out, sizeof(double) * n * out_per, cudaMemcpyDefault);
  cudaFree(d_in);
  cudaFree(d_out);
  CK(e);
  return GLISSE_OK;
}

void glisse_destroy(glisse_sim* s) { free_sim(s); }

// One-shot run over host (or device) arrays, pipelined over parts (include/glisse.h).  Each part is a sim
// of its own on a contiguous slice of the particles: they never interact, so this is the
// paper's own partition of the particles with the planets replicated — here over time slots of one GPU
// instead of over GPUs.  Part i+1 is created (its upload) and part i read back (its download) while the
// kernels of the other parts run.
int glisse_run(double gm_star, int n_planets, const double* gm_planet, const double* planet_pos,
               const double* planet_vel, const double* planet_rcrit, long long n_particles,
               const double* const pos[3], const double* const vel[3], double dt, const glisse_params* params,
               long long n_steps, int n_parts, double* const out_pos[3], double* const out_vel[3], int* flag,
               long long* removal_step, long long* particle_steps) {
  constexpr int kMaxParts = 64;
  constexpr long long kAutoPart = 1LL << 17;   // automatic: parts of about 2^17 particles, at most 8
  if (n_particles < 1 || n_steps < 0 || n_parts < 0 || n_parts > kMaxParts || !pos || !vel) return GLISSE_EINVAL;
  for (int k = 0; k < 3; ++k)
    if (!pos[k] || !vel[k]) return GLISSE_EINVAL;
  if (n_parts == 0) n_parts = static_cast<int>(std::max<long long>(1, std::min<long long>(8, n_particles / kAutoPart)));
  // cuts at multiples of 256 particles (whole warps, 2 KiB-aligned rows); no part is empty
  long long cut[kMaxParts + 1];
  int parts = 0;
  cut[0] = 0;
  for (int i = 1; i <= n_parts; ++i) {
    long long c = (i == n_parts) ? n_particles : (n_particles * i / n_parts) / 256 * 256;
    if (c > cut[parts]) cut[++parts] = c;
  }
  glisse_sim* sims[kMaxParts] = {};
  int st = GLISSE_OK;
  for (int i = 0; i < parts && st == GLISSE_OK; ++i) {
    const long long lo = cut[i];
    const double* p[3] = {pos[0] + lo, pos[1] + lo, pos[2] + lo};
    const double* v[3] = {vel[0] + lo, vel[1] + lo, vel[2] + lo};
    st = glisse_create(&sims[i], gm_star, n_planets, gm_planet, planet_pos, planet_vel, planet_rcrit, cut[i + 1] - lo, p,
                       v, dt, params);
    if (st == GLISSE_OK) st = glisse_advance(sims[i], n_steps);
  }
  long long psteps = 0;
  for (int i = 0; i < parts && st == GLISSE_OK; ++i) {
    const long long lo = cut[i];
    double* p[3] = {nullptr, nullptr, nullptr};
    double* v[3] = {nullptr, nullptr, nullptr};
    for (int k = 0; k < 3; ++k) {
      if (out_pos && out_pos[k]) p[k] = out_pos[k] + lo;
      if (out_vel && out_vel[k]) v[k] = out_vel[k] + lo;
    }
    st = glisse_read(sims[i], p, v, flag ? flag + lo : nullptr, removal_step ? removal_step + lo : nullptr);
    if (st == GLISSE_OK && particle_steps) {
      const long long c = glisse_particle_steps(sims[i]);
      if (c < 0) st = static_cast<int>(c);
      else psteps += c;
    }
  }
  for (int i = 0; i < parts; ++i) free_sim(sims[i]);
  if (st == GLISSE_OK && particle_steps) *particle_steps = psteps;
  return st;
}

}  // extern "C"
