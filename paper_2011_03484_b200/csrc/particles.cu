// particles.cu — the particle kernel (steps a2–a7 of DESIGN.md; PAPER.md:91-95 step list, 103-113
// kick, 123-127 solver and encounter flags).  Hand-written for sm_100a.
//
// One particle per thread.  The six state doubles live in registers for all steps of the chunk
// (PAPER.md:107, 61), loaded once and stored once, coalesced, from struct-of-arrays storage.
// The planet log (q_j(t_s), h0(t_s)) is staged into shared memory by bulk
// asynchronous copies (cp.async.bulk = TMA 1-D, completion on an mbarrier) into a double-buffered
// ring that is PRIVATE TO EACH WARP: a warp never waits for another warp, a warp whose particles
// are all removed leaves at once, and every log read is a conflict-free shared-memory broadcast.
//
// Step structure (kick ½ – drift – kick ½, O1–O5).  The closing half kick of step s and
// the opening half kick of step s+1 use the same acceleration: it is evaluated once and applied
// as two half kicks, so that a chunk boundary (where the state is stored between them) leaves no
// trace in the bits: results do not depend on K or on how advance() calls are split.
//
// The step loop is the same straight code for all 32 lanes, with no per-lane predicate: a lane whose
// particle is gone runs a copy of a live lane's body (struct Lane below), and everything a removal or a
// hard Kepler solve needs runs in two out-of-line functions entered on one warp vote each
// (removal_at_kick, solve_and_flag).  The FP64 pipe is the roofline; what this layout saves is the
// integer work that existed only because lanes can be dead (DESIGN.md sections 7 and 12).
#include "glisse_internal.cuh"
#include "kepler.cuh"

namespace glisse {
namespace {

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}

// 1-D bulk copy global -> shared, completion signalled on the mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ---- launch chaining: completion lists between back-to-back launches -------------------
__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// programmatic dependent launch: the next launch in the stream (if it asked for programmatic
// serialisation) may become resident once every block of this grid has executed this or exited
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// A warp of a chained launch takes the k-th completed group of the previous launch, k = blockIdx.x.
// Deadlock-free: the previous launch's blocks call pdl_launch_dependents only once they own a group, so
// when this block is resident every block of the previous launch is resident or finished, and those
// never wait on anything later.  The time-out (seconds; never expected) turns a logic error into a
// status instead of a hung device.
__device__ __forceinline__ int acquire_group(const ParticleArgs& a, int lane) {
  int g = static_cast<int>(blockIdx.x);
  if (a.wait_list != nullptr) {
    int v = 0;
    if (lane == 0) {
      int* slot = a.wait_list + blockIdx.x;
      const long long t0 = clock64();
      unsigned ns = 32;
      while ((v = ld_acquire(slot)) == 0) {
        __nanosleep(ns);
        if (ns < 2048) ns <<= 1;
        if (clock64() - t0 > (8LL << 30)) { atomicExch(a.error, 1); v = -1; break; }
      }
      // the entry is this block's alone: free it for the launch after next (an atomic, so that the
      // clearing has been performed at L2 before this block lets dependents launch)
      atomicExch(slot, 0);
    }
    v = __shfl_sync(kFullMask, v, 0);
    g = v - 1;   // -2: gave up
  }
  return g;
}

__device__ __forceinline__ void publish_group(const ParticleArgs& a, int lane, int g) {
  __threadfence();   // this lane's stores of the group's state are visible device-wide ...
  __syncwarp();
  if (lane == 0) {   // ... before the group is handed on
    const unsigned pos = atomicAdd(a.done_ticket, 1u) - a.ticket_base;
    st_release(a.done_list + pos, g + 1);
  }
}

__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// ---- shared-memory reads of the staged log by 32-bit shared address (the record pointer is one
// uniform register that advances by the stride; ordered after the mbarrier wait, both being volatile)
__device__ __forceinline__ double lds_f64(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}

__device__ __forceinline__ void lds_f64x2(uint32_t addr, double& v0, double& v1) {
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v0), "=d"(v1) : "r"(addr));
}

// The per-lane state of the step loop.  A lane whose own particle is gone (removed in an earlier launch,
// past the end of the array, or flagged during this launch) is `dead`: it goes on with a COPY of a live
// lane's body (its donor), so that it computes exactly what the donor computes — never a NaN, a slow
// path or a test hit of its own — and the step loop needs no per-lane predicate at all.  Everything a
// removal needs (flag, removal record, the frozen state written to memory, a new donor for the lane and
// for every lane that was copying it) happens in blocks entered on one warp vote.
struct Lane {
  double x, y, z, vx, vy, vz;
  int flag;     // of the lane's own particle (0 = still integrating); -1 = the lane never had one
  int rs;       // record index (within this launch) at which it was flagged
  bool dead;    // the registers hold a donor's body
};

__device__ __forceinline__ double shfl_f64(double v, int src) { return __shfl_sync(kFullMask, v, src); }

// the frozen state of a particle flagged during this launch goes to memory at once (O5 / S12)
__device__ __forceinline__ void freeze(const ParticleArgs& a, long long i, const Lane& L, int flag, int k) {
  a.st[0][i] = L.x; a.st[1][i] = L.y; a.st[2][i] = L.z;
  a.st[3][i] = L.vx; a.st[4][i] = L.vy; a.st[5][i] = L.vz;
  a.flag[i] = flag;
  a.rstep[i] = a.step0 + k;
}

// ---- the removal blocks: out of line, entered by the whole warp on one vote, so that neither their
// registers nor their branches cost the step loop anything.  The lane's numbers travel through a small
// record in local memory.  Both return true when no lane of the warp has a particle left.
struct KickRecord {
  Lane L;
  double ax, ay, az, r2;
};

// Exact distance tests of O5 at the record at `rec` (the hot path saw a high-word superset pass in some
// lane), lowest planet index first (S11); a particle that is hit is frozen WITHOUT this evaluation's kick.
static __device__ __noinline__ bool removal_at_kick(const ParticleArgs& a, int np, uint32_t rec, int k, long long i,
                                                    KickRecord* io) {
  Lane L = io->L;
  const double r2 = io->r2;
  int hit = 0;
  for (int jj = 0; jj < np; ++jj) {
    const int j = np - 1 - jj;
    const double qx = lds_f64(rec + 24 * j), qy = lds_f64(rec + 24 * j + 8), qz = lds_f64(rec + 24 * j + 16);
    const double dx = L.x - qx, dy = L.y - qy, dz = L.z - qz;
    const double d2 = fma(dx, dx, fma(dy, dy, dz * dz));
    hit = (d2 < a.rc2[j]) ? (GLISSE_FLAG_PLANET0 + j) : hit;
  }
  hit = (r2 > a.rmax2) ? GLISSE_FLAG_RMAX : hit;
  hit = (r2 < a.rmin2) ? GLISSE_FLAG_RMIN : hit;
  if (!__any_sync(kFullMask, hit != 0)) return false;
  if (hit != 0 && !L.dead) {
    freeze(a, i, L, hit, k);
    io->L.flag = hit;
    io->L.rs = k;
  }
  const bool dead = L.dead || hit != 0;
  io->L.dead = dead;
  const unsigned alive = __ballot_sync(kFullMask, !dead);
  if (alive == 0u) return true;
  // every lane that hit — the particle's own lane and the lanes that were copying it — takes a new donor
  const int donor = __ffs(alive) - 1;
  const double tx = shfl_f64(L.x, donor), ty = shfl_f64(L.y, donor), tz = shfl_f64(L.z, donor);
  const double tvx = shfl_f64(L.vx, donor), tvy = shfl_f64(L.vy, donor), tvz = shfl_f64(L.vz, donor);
  const double tax = shfl_f64(io->ax, donor), tay = shfl_f64(io->ay, donor), taz = shfl_f64(io->az, donor);
  const double tr2 = shfl_f64(r2, donor);
  if (hit != 0) {
    io->L.x = tx; io->L.y = ty; io->L.z = tz; io->L.vx = tvx; io->L.vy = tvy; io->L.vz = tvz;
    io->ax = tax; io->ay = tay; io->az = taz; io->r2 = tr2;
  }
  return false;
}

// Force evaluation with the tests (O1/O4/O5) at the record at shared address `rec`, then the kick(s):
// v += acc hdt, and again with hdt2 (hdt for an interior record of KDK — the closing half kick of one step
// and the opening one of the next — and for DKD's full kick; 0 at record 0).  Returns true when no lane of
// the warp has a particle left.  r2 = |r|^2 is handed on to the drift.
template <int NP>
__device__ __forceinline__ bool kick_with_tests(const ParticleArgs& a, int np, uint32_t rec, int k, long long i,
                                                double hdt, double hdt2, Lane& L, double& r2) {
  // The tests compare squared distances (O5).  On the hot path they are taken on the HIGH WORDS in the
  // integer pipe, as a superset (d2 < R2 implies hi(d2) <= hi(R2) for non-negative doubles); the exact
  // fp64 comparisons run only in a warp where some lane passes the superset.
  r2 = fma(L.x, L.x, fma(L.y, L.y, L.z * L.z));
  const int r2h = __double2hiint(r2);
  bool maybe = (r2h >= a.rmax2_hi) | (r2h <= a.rmin2_hi);   // (| not ||: no short-circuit, no predicated loads)
  double ax, ay, az;
  if (NP > 0) {   // the record as 16-byte shared-memory loads (records are 16-byte aligned, stride even)
    constexpr int kD = 3 * (NP > 0 ? NP : 1) + 3;
    double rv[kD + 1];
#pragma unroll
    for (int c = 0; c < kD; c += 2) lds_f64x2(rec + 8 * c, rv[c], rv[c + 1]);
    ax = rv[3 * NP]; ay = rv[3 * NP + 1]; az = rv[3 * NP + 2];  // h0
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      const double dx = L.x - rv[3 * j], dy = L.y - rv[3 * j + 1], dz = L.z - rv[3 * j + 2];
      const double d2 = fma(dx, dx, fma(dy, dy, dz * dz));
      maybe = maybe | (__double2hiint(d2) <= a.rc2_hi[j]);
      const double w = gm_over_r3(a.gm[j], d2);
      ax = fma(-w, dx, ax);
      ay = fma(-w, dy, ay);
      az = fma(-w, dz, az);
    }
  } else {
    ax = lds_f64(rec + 24 * np); ay = lds_f64(rec + 24 * np + 8); az = lds_f64(rec + 24 * np + 16);  // h0
    for (int j = 0; j < np; ++j) {
      const double qx = lds_f64(rec + 24 * j), qy = lds_f64(rec + 24 * j + 8), qz = lds_f64(rec + 24 * j + 16);
      const double dx = L.x - qx, dy = L.y - qy, dz = L.z - qz;
      const double d2 = fma(dx, dx, fma(dy, dy, dz * dz));
      maybe = maybe | (__double2hiint(d2) <= a.rc2_hi[j]);
      const double w = gm_over_r3(a.gm[j], d2);
      ax = fma(-w, dx, ax);
      ay = fma(-w, dy, ay);
      az = fma(-w, dz, az);
    }
  }
  if (__any_sync(kFullMask, maybe)) {  // rare
    KickRecord io;
    io.L = L; io.ax = ax; io.ay = ay; io.az = az; io.r2 = r2;
    const bool finished = removal_at_kick(a, np, rec, k, i, &io);
    L = io.L; ax = io.ax; ay = io.ay; az = io.az; r2 = io.r2;
    if (__any_sync(kFullMask, finished)) return true;   // (the vote tells the compiler that the exit is warp-uniform)
  }
  L.vx = fma(ax, hdt, L.vx); L.vy = fma(ay, hdt, L.vy); L.vz = fma(az, hdt, L.vz);
  L.vx = fma(ax, hdt2, L.vx); L.vy = fma(ay, hdt2, L.vy); L.vz = fma(az, hdt2, L.vz);
  return false;
}

struct DriftRecord {
  Lane L;
  DriftVars v;
  double xk, sm, cm1;     // the solver's state: x, sin x − x, cos x − 1
  int thr;                // acceptance bound of the fast solver for this body
  bool unbound, open, slow;
  int nonconv;            // the body has been through the definition's solver already and did not converge
  unsigned iters, went_slow;   // statistics: fast-solver steps taken here, slow path entered
};

// Everything a drift can need beyond its first fast-solver step: further steps for the bodies that are
// still `open` (exactly as kepler_drift_warp takes them, starting with step number it0), the definition's
// solver for the `slow` ones, flags 3 / 4 with the state on entry to the drift frozen, new donors.
static __device__ __noinline__ bool solve_and_flag(const ParticleArgs& a, int it0, int k, long long i, DriftRecord* io) {
  DriftVars v = io->v;
  double xk = io->xk, sm = io->sm, cm1 = io->cm1;
  const int thr = io->thr;
  const bool unbound = io->unbound;
  bool open = io->open, slow = io->slow;
  // a step of half a revolution or more: dM reduced to (-pi, pi] here (reading S9); the caller counted the
  // body as not open, so the definition's solver takes it
  if (!(hi_abs(v.dM) < kHiPi)) {
    v.dM = reduce_mean_motion(v.dM);
    io->v.dM = v.dM;
  }
  unsigned iters = 0;
  for (int it = it0; it < kFastMaxIters && __any_sync(kFullMask, open); ++it) {
    double xn, smn, cmn, dl;
    fast_step(v, xk, xn, smn, cmn, dl);
    ++iters;
    if (open) {
      sm = smn; cm1 = cmn; xk = xn;
      const bool done = hi_abs(dl) < thr;
      const bool lost = !done && !is_small_angle(xk);
      open = !done && !lost;
      slow = slow || lost;
    }
  }
  slow = slow || open;   // no convergence in kFastMaxIters steps
  int nonconv = io->nonconv;
  io->went_slow = 0;
  if (__any_sync(kFullMask, slow)) {
    io->went_slow = 1;
    const ExactSolve o = kepler_solve_exact(slow, v.ec, v.es, v.q, v.dM, v.invq, v.e2, a.iters, a.tol);
    if (slow) { xk = o.x; sm = o.sm; cm1 = o.cm1; nonconv = o.nonconv; }
  }
  io->iters = iters;
  io->xk = xk; io->sm = sm; io->cm1 = cm1;
  const bool bad = unbound || nonconv != 0;
  if (!__any_sync(kFullMask, bad)) return false;
  const Lane L = io->L;
  if (bad && !L.dead) {
    const int why = unbound ? GLISSE_FLAG_UNBOUND : GLISSE_FLAG_NONCONV;
    freeze(a, i, L, why, k);
    io->L.flag = why;
    io->L.rs = k;
  }
  const bool dead = L.dead || bad;
  io->L.dead = dead;
  const unsigned alive = __ballot_sync(kFullMask, !dead);
  if (alive == 0u) return true;
  const int donor = __ffs(alive) - 1;
  // (one value at a time: the shuffle, then the select)
#define GL_TAKE(field) { const double t_ = shfl_f64(field, donor); if (bad) io->field = t_; }
  GL_TAKE(L.x) GL_TAKE(L.y) GL_TAKE(L.z) GL_TAKE(L.vx) GL_TAKE(L.vy) GL_TAKE(L.vz)
  GL_TAKE(v.rinv) GL_TAKE(v.sqa) GL_TAKE(v.rsa) GL_TAKE(v.q) GL_TAKE(v.ec) GL_TAKE(v.es)
  GL_TAKE(v.dM) GL_TAKE(v.a) GL_TAKE(v.invq)
#undef GL_TAKE
  { const double t_ = shfl_f64(xk, donor); if (bad) io->xk = t_; }
  { const double t_ = shfl_f64(sm, donor); if (bad) io->sm = t_; }
  { const double t_ = shfl_f64(cm1, donor); if (bad) io->cm1 = t_; }
  return false;
}

// Which Kepler solver an instantiation of the kernel carries (chosen once per simulation, api.cu):
// the fast solver from the first-order starting point, the same from the third-order one (REFINE in
// kepler.cuh; include/glisse.h: guess_order), or the definition's solver alone for a run whose kepler_iters /
// kepler_tol keep the fast one out (kepler.cuh: kFastMinIters, kFastMinTol).
enum : int { kSolverFast = 0, kSolverFastRefined = 1, kSolverDefinition = 2 };

// Kepler drift of the warp's 32 bodies (O2): begin, one fast-solver step, finish, with one vote in between
// that sends the warp to solve_and_flag.  In the kSolverFastRefined instantiation (planet-crossing
// populations) a second fast-solver step is common, so it is taken in line before the call; in the
// kSolverDefinition one every body goes straight to kepler_solve_exact and only a flag goes out of line.
// Returns true when no lane of the warp has a particle left.
template <int SOLVER, bool STATS>
__device__ __forceinline__ bool drift_with_flags(const ParticleArgs& a, double two_mu, double inv_mu_dt, double r2, int k,
                                                 long long i, Lane& L, unsigned (&stat)[3]) {
  constexpr bool REFINE = SOLVER == kSolverFastRefined;
  DriftVars v;
  double xk, xn, sm, cm1, dl;
  bool unbound;
  drift_begin<REFINE>(a.mu, two_mu, a.inv_mu, inv_mu_dt, r2, L.x, L.y, L.z, L.vx, L.vy, L.vz, v, xk, unbound);
  if (SOLVER == kSolverDefinition) {
    if (!(hi_abs(v.dM) < kHiPi)) v.dM = reduce_mean_motion(v.dM);
    const ExactSolve o = kepler_solve_exact(!unbound, v.ec, v.es, v.q, v.dM, v.invq, v.e2, a.iters, a.tol);
    xn = o.x; sm = o.sm; cm1 = o.cm1;
    const int nonconv = unbound ? 0 : o.nonconv;
    if (STATS) { stat[0] += 1; stat[2] += 1; }
    if (__any_sync(kFullMask, unbound || nonconv != 0)) {
      DriftRecord io;
      io.L = L; io.v = v; io.xk = xn; io.sm = sm; io.cm1 = cm1; io.thr = 0;
      io.unbound = unbound; io.open = false; io.slow = false; io.nonconv = nonconv;
      const bool finished = solve_and_flag(a, kFastMaxIters, k, i, &io);
      L = io.L; v = io.v; xn = io.xk; sm = io.sm; cm1 = io.cm1;
      if (__any_sync(kFullMask, finished)) return true;
    }
    drift_finish(v, xn, sm, cm1, L.x, L.y, L.z, L.vx, L.vy, L.vz);
    return false;
  }
  const int e2h = hi_word(v.e2);
  // (an unbound body needs no test of its own here: alpha <= 0 makes e^2 a NaN, a denormal alpha makes it 1,
  // and either fails e2h < kHiE2_080; a step of half a revolution or more has one, since dM is not reduced
  // on this path)
  const bool hard = !(e2h < kHiE2_080) | !is_small_angle(xk) | !(hi_abs(v.dM) < kHiPi);
  fast_step(v, xk, xn, sm, cm1, dl);
  const bool done = fast_accepts(hi_abs(dl), e2h);
  if (STATS) { stat[0] += 1; stat[1] += 1; }
  if (__any_sync(kFullMask, hard | !done)) {
    const int thr = fast_threshold(e2h);
    const bool notopen = unbound | hard;
    bool open = !notopen && !done && is_small_angle(xn);
    bool slow = !unbound && (notopen || (!done && !open));
    int it0 = 1;
    bool more = true;
    if (REFINE) {   // the second step in line
      if (__any_sync(kFullMask, open)) {
        double xn2, smn, cmn, dl2;
        fast_step(v, xn, xn2, smn, cmn, dl2);
        if (STATS) stat[1] += 1;
        if (open) {
          sm = smn; cm1 = cmn; xn = xn2;
          const bool done2 = hi_abs(dl2) < thr;
          const bool lost = !done2 && !is_small_angle(xn);
          open = !done2 && !lost;
          slow = slow || lost;
        }
      }
      it0 = 2;
      more = __any_sync(kFullMask, open || slow || unbound);
    }
    if (more) {
      DriftRecord io;
      io.L = L; io.v = v; io.xk = xn; io.sm = sm; io.cm1 = cm1; io.thr = thr;
      io.unbound = unbound; io.open = open; io.slow = slow; io.nonconv = 0;
      const bool finished = solve_and_flag(a, it0, k, i, &io);
      L = io.L; v = io.v; xn = io.xk; sm = io.sm; cm1 = io.cm1;
      if (STATS) { stat[1] += io.iters; stat[2] += io.went_slow; }
      if (__any_sync(kFullMask, finished)) return true;
    }
  }
  drift_finish(v, xn, sm, cm1, L.x, L.y, L.z, L.vx, L.vy, L.vz);
  return false;
}

// NP > 0: compile-time planet count (fully unrolled kick); NP == 0: run-time count a.np.
// STATS: instrumented instantiation (glisse_test.h: glisse_solver_stats); same arithmetic.
// DKD: the drift-kick-drift splitting (GLISSE_SCHEME_DKD): per step a half drift, the force evaluation
// with the tests at the half-step record, a full kick, a half drift; nsteps records are read, not
// nsteps + 1, and the state between launches is synchronised at the integer steps as in KDK.
// SOLVER: kSolverFast / kSolverFastRefined / kSolverDefinition (above).
template <int NP, bool STATS, bool DKD, int SOLVER>
__global__ void __launch_bounds__(kParticleBlock, GL_MIN_BLOCKS) particle_kernel(const __grid_constant__ ParticleArgs a) {
  static_assert(kParticleBlock == 32, "one warp per block: the launch chain hands groups of one warp on");
  static_assert(kParticlesPerThread == 1, "one particle per thread");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31;
  const int np = NP > 0 ? NP : a.np;
  const int stride = a.stride;
  const int nsteps = a.nsteps;
  const int R = a.stage_recs;
  const int stage_doubles = R * stride;

  const int grp = acquire_group(a, lane);
  pdl_launch_dependents();
  if (grp < 0) return;   // gave up waiting (a.error is set): touch nothing
  const int n = *a.n_slots;
  const long long i = static_cast<long long>(grp) * kParticleBlock + threadIdx.x;  // consecutive lanes, consecutive particles

  // ---- a2: load ------------------------------------------------------------------------------
  Lane L;
  L.x = 1.0; L.y = 0.0; L.z = 0.0; L.vx = 0.0; L.vy = 0.0; L.vz = 0.0;
  L.flag = -1;
  L.rs = -1;
  if (i < n) {  // through L2: the group's previous owner may have run on another SM a launch ago
    L.flag = __ldcg(a.flag + i);
    L.x = __ldcg(a.st[0] + i); L.y = __ldcg(a.st[1] + i); L.z = __ldcg(a.st[2] + i);
    L.vx = __ldcg(a.st[3] + i); L.vy = __ldcg(a.st[4] + i); L.vz = __ldcg(a.st[5] + i);
  }
  const bool own = (L.flag == 0);   // the lane has a particle to integrate
  L.dead = !own;
  {
    if (!__any_sync(kFullMask, own)) {  // nothing to do in this warp: leave before any copy
      publish_group(a, lane, grp);
      return;
    }
    const unsigned alive = __ballot_sync(kFullMask, own);
    const int donor = __ffs(alive) - 1;
    const double tx = shfl_f64(L.x, donor), ty = shfl_f64(L.y, donor), tz = shfl_f64(L.z, donor);
    const double tvx = shfl_f64(L.vx, donor), tvy = shfl_f64(L.vy, donor), tvz = shfl_f64(L.vz, donor);
    if (!own) { L.x = tx; L.y = ty; L.z = tz; L.vx = tvx; L.vy = tvy; L.vz = tvz; }
  }

  // ---- warp-private ring ------------------------------------------------------------------------
  double* ring = reinterpret_cast<double*>(smem_raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(ring + static_cast<size_t>(kRingSlots) * stage_doubles);
  const uint32_t ring_addr = smem_u32(ring);
  const uint32_t rec_bytes = static_cast<uint32_t>(stride) * 8u;
  const int nrec = DKD ? nsteps : nsteps + 1;
  const int nstages = (nrec + R - 1) / R;
  if (lane == 0) {
    for (int sl = 0; sl < kRingSlots; ++sl) mbar_init(&bars[sl], 1);
    fence_mbar_init();
    fence_proxy_async();
    for (int st = 0; st < kRingSlots && st < nstages; ++st) {
      const int recs = min(R, nrec - st * R);
      const uint32_t bytes = static_cast<uint32_t>(recs) * stride * 8u;
      mbar_expect_tx(&bars[st], bytes);
      bulk_g2s(ring + st * stage_doubles, a.log + static_cast<size_t>(st) * stage_doubles, bytes, &bars[st]);
    }
  }
  __syncwarp();

  const double hdt = a.hdt;
  const double two_mu = a.two_mu;
  const double inv_mu_dt = DKD ? a.inv_mu_hdt : a.inv_mu_dt;
  unsigned stat[3] = {0u, 0u, 0u};
  double hdt2 = DKD ? hdt : 0.0;   // the second half kick: none at record 0 of KDK
  bool finished = false;           // no lane has a particle left
  int st = 0;
  for (; st < nstages; ++st) {
    const int slot = st & (kRingSlots - 1);
    mbar_wait(&bars[slot], (st / kRingSlots) & 1);
    uint32_t rec = ring_addr + static_cast<uint32_t>(slot * stage_doubles) * 8u;
    const int recs = min(R, nrec - st * R);
    // the steps of this stage; in KDK the very last record of the launch is a kick without a drift
    const int nfull = (!DKD && st == nstages - 1) ? recs - 1 : recs;
    int kk = 0;
    for (; kk < nfull; ++kk, rec += rec_bytes) {
      const int k = st * R + kk;   // record index within the launch (used by the removal blocks only)
      double r2;
      if (DKD) {  // ---- first half drift of step k (D1): flags 3 / 4 freeze the state of t_k
        r2 = fma(L.x, L.x, fma(L.y, L.y, L.z * L.z));
        if (drift_with_flags<SOLVER, STATS>(a, two_mu, inv_mu_dt, r2, k, i, L, stat)) { finished = true; break; }
      }
      // ---- a3/a4: force evaluation with the tests at time t_{step0+k}, kick(s) ------------------------
      if (kick_with_tests<NP>(a, np, rec, k, i, hdt, hdt2, L, r2)) { finished = true; break; }
      // ---- a5/a6: drift (O2; in DKD the second half drift, D4) ---------------------------------------
      if (DKD) r2 = fma(L.x, L.x, fma(L.y, L.y, L.z * L.z));
      if (drift_with_flags<SOLVER, STATS>(a, two_mu, inv_mu_dt, r2, k, i, L, stat)) { finished = true; break; }
      hdt2 = hdt;
    }
    if (finished) break;
    if (kk < recs) {   // KDK: closing half kick of the launch's last step at record nsteps
      double r2;
      if (kick_with_tests<NP>(a, np, rec, st * R + kk, i, hdt, 0.0, L, r2)) { finished = true; break; }
    }
    __syncwarp();
    if (lane == 0 && st + kRingSlots < nstages) {
      const int nx = st + kRingSlots;
      const int recs_n = min(R, nrec - nx * R);
      const uint32_t bytes = static_cast<uint32_t>(recs_n) * stride * 8u;
      fence_proxy_async();
      mbar_expect_tx(&bars[slot], bytes);
      bulk_g2s(ring + slot * stage_doubles, a.log + static_cast<size_t>(nx) * stage_doubles, bytes, &bars[slot]);
    }
  }
  // a warp that leaves early must not retire while a bulk copy into its ring is still in flight
  if (st < nstages) {
    for (int o = st + 1; o < nstages && o < st + kRingSlots; ++o)
      mbar_wait(&bars[o & (kRingSlots - 1)], (o / kRingSlots) & 1);
  }

  // ---- a7: store (particles flagged during this launch were written when they were flagged) ----------
  if (own && L.flag == 0) {
    a.st[0][i] = L.x; a.st[1][i] = L.y; a.st[2][i] = L.z;
    a.st[3][i] = L.vx; a.st[4][i] = L.vy; a.st[5][i] = L.vz;
  }
  // steps started by this thread's particle: all nsteps for a survivor; for a particle flagged at
  // record k, KDK: k if a force-evaluation test caught it and k + 1 if its drift did (flags 3 and 4);
  // DKD: k + 1 whatever caught it (the step had begun with its first half drift)
  unsigned drifts = 0;
  if (own)
    drifts = L.flag == 0 ? static_cast<unsigned>(nsteps)
                         : static_cast<unsigned>(L.rs) +
                               ((DKD || L.flag == GLISSE_FLAG_NONCONV || L.flag == GLISSE_FLAG_UNBOUND) ? 1u : 0u);
  unsigned tot = __reduce_add_sync(kFullMask, drifts);
  if (lane == 0 && tot) atomicAdd(a.pstep_counter, static_cast<unsigned long long>(tot));
  if (STATS && lane == 0) {
    atomicAdd(a.solver_stats, static_cast<unsigned long long>(stat[0]));
    atomicAdd(a.solver_stats + 1, static_cast<unsigned long long>(stat[1]));
    atomicAdd(a.solver_stats + 2, static_cast<unsigned long long>(stat[2]));
  }
  publish_group(a, lane, static_cast<int>((i - threadIdx.x) / kParticleBlock));
}

size_t particle_smem_bytes(const ParticleArgs& a) {
  return static_cast<size_t>(kParticleWarps) * kRingSlots * a.stage_recs * a.stride * 8 +
         static_cast<size_t>(kParticleWarps) * kRingSlots * 8;
}

// The one pass over the particles at create: identity order, flags and removal steps (working and original
// order), the count of non-finite inputs (counts[0]: create refuses them), and the count of bodies that would
// take the third-order starting point at this instant (counts[1]: guess_order = 0 chooses the instantiation
// from their share, bin_iterations = 2 the binning).  Plain arithmetic: off the hot path.
__global__ void __launch_bounds__(256) create_pass_kernel(const double* x, const double* y, const double* z,
                                                           const double* vx, const double* vy, const double* vz,
                                                           long long n, double mu, double dt,
                                                           unsigned long long* counts, int* id, int* flag,
                                                           long long* rstep, int* fin_flag, long long* fin_rstep) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  bool want = false, bad = false;
  if (i < n) {
    id[i] = static_cast<int>(i);
    flag[i] = 0;
    rstep[i] = -1;
    fin_flag[i] = 0;
    fin_rstep[i] = -1;
    bad = !isfinite(x[i]) | !isfinite(y[i]) | !isfinite(z[i]) | !isfinite(vx[i]) | !isfinite(vy[i]) | !isfinite(vz[i]);
    const double r0 = sqrt(x[i] * x[i] + y[i] * y[i] + z[i] * z[i]);
    const double v2 = vx[i] * vx[i] + vy[i] * vy[i] + vz[i] * vz[i];
    const double u = x[i] * vx[i] + y[i] * vy[i] + z[i] * vz[i];
    const double alpha = 2.0 * mu / r0 - v2;
    if (alpha > 0.0) {
      const double q = r0 * alpha / mu;
      const double ec = 1.0 - q, es = u * sqrt(alpha) / mu;
      const double e2 = ec * ec + es * es;
      const double ndt = alpha * sqrt(alpha) * dt / mu;
      const double xk = fma(-rint(ndt * kInvTwoPi), kTwoPi, ndt) / q;
      want = hi_word(e2) < kHiE2_080 && is_small_angle(xk) && wants_refined_guess(hi_word(e2), hi_abs(xk));
    }
  }
  const int cb = __syncthreads_count(bad);
  const int cw = __syncthreads_count(want);
  if (threadIdx.x == 0 && cb) atomicAdd(counts, static_cast<unsigned long long>(cb));
  if (threadIdx.x == 0 && cw) atomicAdd(counts + 1, static_cast<unsigned long long>(cw));
}

template <int NP, bool STATS, bool DKD, int SOLVER>
cudaError_t configure_kernel() {
  return cudaFuncSetAttribute(particle_kernel<NP, STATS, DKD, SOLVER>,
                              cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

// the instantiations that exist: {plain, DKD} x three solvers, and the instrumented plain one for the two fast solvers
template <int NP>
cudaError_t configure_one() {
  cudaError_t e;
  if ((e = configure_kernel<NP, false, false, kSolverFast>())) return e;
  if ((e = configure_kernel<NP, false, false, kSolverFastRefined>())) return e;
  if ((e = configure_kernel<NP, false, false, kSolverDefinition>())) return e;
  if ((e = configure_kernel<NP, false, true, kSolverFast>())) return e;
  if ((e = configure_kernel<NP, false, true, kSolverFastRefined>())) return e;
  if ((e = configure_kernel<NP, false, true, kSolverDefinition>())) return e;
  if ((e = configure_kernel<NP, true, false, kSolverFast>())) return e;
  return configure_kernel<NP, true, false, kSolverFastRefined>();
}

template <int NP, bool STATS, bool DKD, int SOLVER>
cudaError_t launch_one(const ParticleArgs& a, int blocks, size_t smem, bool chained, cudaStream_t s) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(blocks));
  cfg.blockDim = dim3(kParticleBlock);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = chained ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, particle_kernel<NP, STATS, DKD, SOLVER>, a);
}

template <int NP>
cudaError_t launch_np(const ParticleArgs& a, int n_groups, size_t smem, bool chained, bool stats, bool dkd, int solver,
                      cudaStream_t s) {
  // (no instrumented instantiation for DKD or for the definition's solver: their statistics stay zero)
  if (solver == kSolverDefinition)
    return dkd ? launch_one<NP, false, true, kSolverDefinition>(a, n_groups, smem, chained, s)
               : launch_one<NP, false, false, kSolverDefinition>(a, n_groups, smem, chained, s);
  if (solver == kSolverFastRefined) {
    if (dkd) return launch_one<NP, false, true, kSolverFastRefined>(a, n_groups, smem, chained, s);
    return stats ? launch_one<NP, true, false, kSolverFastRefined>(a, n_groups, smem, chained, s)
                 : launch_one<NP, false, false, kSolverFastRefined>(a, n_groups, smem, chained, s);
  }
  if (dkd) return launch_one<NP, false, true, kSolverFast>(a, n_groups, smem, chained, s);
  return stats ? launch_one<NP, true, false, kSolverFast>(a, n_groups, smem, chained, s)
               : launch_one<NP, false, false, kSolverFast>(a, n_groups, smem, chained, s);
}

}  // namespace

cudaError_t configure_particle_kernels() {
  cudaError_t e;
  if ((e = configure_one<0>())) return e;
  if ((e = configure_one<4>())) return e;
  return configure_one<8>();
}

cudaError_t launch_particle_kernel(const ParticleArgs& a, int n_groups, bool chained, bool stats, bool dkd, bool refine,
                                   bool definition_only, cudaStream_t s) {
  if (n_groups < 1) n_groups = 1;
  const size_t smem = particle_smem_bytes(a);
  const int solver = definition_only ? kSolverDefinition : (refine ? kSolverFastRefined : kSolverFast);
  cudaError_t e;
  if (a.np == 4) e = launch_np<4>(a, n_groups, smem, chained, stats, dkd, solver, s);
  else if (a.np == 8) e = launch_np<8>(a, n_groups, smem, chained, stats, dkd, solver, s);
  else e = launch_np<0>(a, n_groups, smem, chained, stats, dkd, solver, s);
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_create_pass(const double* const st[6], long long n, double mu, double dt, unsigned long long* counts,
                               int* id, int* flag, long long* rstep, int* fin_flag, long long* fin_rstep,
                               cudaStream_t s) {
  create_pass_kernel<<<static_cast<int>((n + 255) / 256), 256, 0, s>>>(st[0], st[1], st[2], st[3], st[4], st[5], n, mu, dt,
                                                                        counts, id, flag, rstep, fin_flag, fin_rstep);
  return cudaGetLastError();
}

bool fast_solver_allowed(int kepler_iters, double kepler_tol) {
  return kepler_iters >= kFastMinIters && kepler_tol >= kFastMinTol;
}

// particles per launch group (one warp's worth): the host sizes grids and completion lists with it
int particles_per_group() { return kParticleBlock * kParticlesPerThread; }

}  // namespace glisse
