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

// NP > 0: compile-time planet count (fully unrolled kick); NP == 0: run-time count a.np.
// P = particles per thread (kParticlesPerThread): independent instruction streams, see kepler.cuh.
// STATS: instrumented instantiation (glisse_test.h: glisse_solver_stats); same arithmetic.
// DKD: the drift-kick-drift splitting (GLISSE_SCHEME_DKD): per step a half drift, the force evaluation
// with the tests at the half-step record, a full kick, a half drift; nsteps records are read, not
// nsteps + 1, and the state between launches is synchronised at the integer steps as in KDK.
// REFINE: third-order starting point of the Kepler solve (kepler.cuh; include/glisse.h: guess_order).
template <int NP, int P, bool STATS, bool DKD, bool REFINE>
__global__ void __launch_bounds__(kParticleBlock, GL_MIN_BLOCKS) particle_kernel(const __grid_constant__ ParticleArgs a) {
  static_assert(kParticleBlock == 32, "one warp per block: the launch chain hands groups of one warp on");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31;
  constexpr int warp = 0;
  const int np = NP > 0 ? NP : a.np;
  const int stride = a.stride;
  const int nsteps = a.nsteps;
  const int R = a.stage_recs;
  const int stage_doubles = R * stride;

  const int grp = acquire_group(a, lane);
  pdl_launch_dependents();
  if (grp < 0) return;   // gave up waiting (a.error is set): touch nothing
  const int n = *a.n_slots;
  // particle p of this thread: consecutive threads hold consecutive particles (coalesced), the P
  // particles of a thread lie kParticleBlock apart
  const long long i0 = static_cast<long long>(grp) * (kParticleBlock * P) + threadIdx.x;

  // ---- a2: load ------------------------------------------------------------------------------
  double x[P], y[P], z[P], vx[P], vy[P], vz[P];
  int flag[P];
  bool was_alive[P], alive[P];
  int rs[P];   // record index (within this launch) at which the particle was flagged, −1 = not yet
  bool any_alive_t = false;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    const long long i = i0 + p * kParticleBlock;
    x[p] = 1.0; y[p] = 0.0; z[p] = 0.0; vx[p] = 0.0; vy[p] = 0.0; vz[p] = 0.0;
    flag[p] = -1;
    if (i < n) {  // through L2: the group's previous owner may have run on another SM a launch ago
      flag[p] = __ldcg(a.flag + i);
      x[p] = __ldcg(a.st[0] + i); y[p] = __ldcg(a.st[1] + i); z[p] = __ldcg(a.st[2] + i);
      vx[p] = __ldcg(a.st[3] + i); vy[p] = __ldcg(a.st[4] + i); vz[p] = __ldcg(a.st[5] + i);
    }
    was_alive[p] = (flag[p] == 0);
    alive[p] = was_alive[p];
    any_alive_t = any_alive_t || alive[p];
    rs[p] = -1;
  }
  if (!__any_sync(kFullMask, any_alive_t)) {  // nothing to do in this warp: leave before any copy
    publish_group(a, lane, grp);
    return;
  }

  // ---- warp-private ring ------------------------------------------------------------------------
  double* ring = reinterpret_cast<double*>(smem_raw) + static_cast<size_t>(warp) * kRingSlots * stage_doubles;
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<double*>(smem_raw) +
                                               static_cast<size_t>(kParticleWarps) * kRingSlots * stage_doubles) +
                   warp * kRingSlots;
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
  unsigned stat_calls = 0, stat_iters = 0, stat_slow = 0;
  int k = 0;  // global record index
  int st = 0;
  for (; st < nstages; ++st) {
    const int slot = st & (kRingSlots - 1);
    mbar_wait(&bars[slot], (st / kRingSlots) & 1);
    const double* stage = ring + slot * stage_doubles;
    const int recs = min(R, nrec - st * R);
    bool any_alive = true;
    for (int kk = 0; kk < recs; ++kk, ++k) {
      const double* rec = stage + kk * stride;
      if (DKD) {  // ---- first half drift of step k (D1): flags 3 / 4 freeze the state of t_k
        double r2h[P];
        int st_h[P], fi;
        bool ws;
#pragma unroll
        for (int p = 0; p < P; ++p) r2h[p] = fma(x[p], x[p], fma(y[p], y[p], z[p] * z[p]));
        kepler_drift_warp<P, REFINE>(alive, a.mu, a.inv_mu, a.inv_mu_hdt, a.iters, a.tol, r2h, x, y, z, vx, vy, vz, st_h,
                                     fi, ws);
        if (STATS) { stat_calls += 1; stat_iters += fi; stat_slow += ws ? 1 : 0; }
#pragma unroll
        for (int p = 0; p < P; ++p) {
          if (st_h[p] != 0) {
            flag[p] = st_h[p];
            rs[p] = k;
            alive[p] = false;
          }
        }
      }
      // ---- a3/a4: force evaluation with the tests (O1/O4/O5) at time t_{step0+k} ----------------
      // The tests compare squared distances (O5).  On the hot path they are taken on the HIGH WORDS
      // in the integer pipe, as a superset (d2 < R2 implies hi(d2) <= hi(R2) for non-negative
      // doubles); the exact fp64 comparisons run only in a warp where some lane passes the superset.
      double r2[P], ax[P], ay[P], az[P];
      bool maybe[P];
#pragma unroll
      for (int p = 0; p < P; ++p) {
        r2[p] = fma(x[p], x[p], fma(y[p], y[p], z[p] * z[p]));
        ax[p] = rec[3 * np]; ay[p] = rec[3 * np + 1]; az[p] = rec[3 * np + 2];  // h0
        const int r2h = __double2hiint(r2[p]);
        maybe[p] = (r2h >= a.rmax2_hi) || (r2h <= a.rmin2_hi);
      }
#pragma unroll
      for (int j = 0; j < np; ++j) {
        const double qx = rec[3 * j], qy = rec[3 * j + 1], qz = rec[3 * j + 2];
#pragma unroll
        for (int p = 0; p < P; ++p) {
          const double dx = x[p] - qx, dy = y[p] - qy, dz = z[p] - qz;
          const double d2 = fma(dx, dx, fma(dy, dy, dz * dz));
          maybe[p] = maybe[p] || (__double2hiint(d2) <= a.rc2_hi[j]);
          const double w = gm_over_r3(a.gm[j], d2);
          ax[p] = fma(-w, dx, ax[p]);
          ay[p] = fma(-w, dy, ay[p]);
          az[p] = fma(-w, dz, az[p]);
        }
      }
      int hit[P];
      bool any_maybe = false;
#pragma unroll
      for (int p = 0; p < P; ++p) {
        hit[p] = 0;
        any_maybe = any_maybe || (maybe[p] && alive[p]);
      }
      if (__any_sync(kFullMask, any_maybe)) {  // rare: the exact tests, lowest planet index wins (S11)
        for (int jj = 0; jj < np; ++jj) {
          const int j = np - 1 - jj;
          const double qx = rec[3 * j], qy = rec[3 * j + 1], qz = rec[3 * j + 2];
#pragma unroll
          for (int p = 0; p < P; ++p) {
            const double dx = x[p] - qx, dy = y[p] - qy, dz = z[p] - qz;
            const double d2 = fma(dx, dx, fma(dy, dy, dz * dz));
            hit[p] = (d2 < a.rc2[j]) ? (GLISSE_FLAG_PLANET0 + j) : hit[p];
          }
        }
#pragma unroll
        for (int p = 0; p < P; ++p) {
          hit[p] = (r2[p] > a.rmax2) ? GLISSE_FLAG_RMAX : hit[p];
          hit[p] = (r2[p] < a.rmin2) ? GLISSE_FLAG_RMIN : hit[p];
        }
      }
      bool any_alive_k = false;
#pragma unroll
      for (int p = 0; p < P; ++p) {
        if (alive[p] && hit[p] != 0) {
          flag[p] = hit[p];
          rs[p] = k;
          alive[p] = false;
        }
        if (alive[p]) {
          vx[p] = fma(ax[p], hdt, vx[p]); vy[p] = fma(ay[p], hdt, vy[p]); vz[p] = fma(az[p], hdt, vz[p]);
          // KDK interior: closing half kick of step k-1 and opening of step k; DKD: the one full kick (D3)
          if (DKD || (k > 0 && k < nsteps)) {
            vx[p] = fma(ax[p], hdt, vx[p]); vy[p] = fma(ay[p], hdt, vy[p]); vz[p] = fma(az[p], hdt, vz[p]);
          }
        }
      }
      // ---- a5/a6: drift (O2; in DKD the second half drift, D4) ---------------------------------------
      if (DKD || k < nsteps) {
        int st_d[P];
        int fast_iters;
        bool went_slow;
        kepler_drift_warp<P, REFINE>(alive, a.mu, a.inv_mu, DKD ? a.inv_mu_hdt : a.inv_mu_dt, a.iters, a.tol, r2, x, y,
                                     z, vx, vy, vz, st_d, fast_iters, went_slow);
        if (STATS) {
          stat_calls += 1;
          stat_iters += fast_iters;
          stat_slow += went_slow ? 1 : 0;
        }
#pragma unroll
        for (int p = 0; p < P; ++p) {
          if (st_d[p] != 0) {
            flag[p] = st_d[p];
            rs[p] = k;
            alive[p] = false;
          }
        }
      }
#pragma unroll
      for (int p = 0; p < P; ++p) any_alive_k = any_alive_k || alive[p];
      any_alive = __any_sync(kFullMask, any_alive_k);
      if (!any_alive) break;
    }
    if (!any_alive) break;
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

  // ---- a7: store --------------------------------------------------------------------------------
#pragma unroll
  for (int p = 0; p < P; ++p) {
    if (was_alive[p]) {  // particles that were already removed at load are untouched
      const long long i = i0 + p * kParticleBlock;
      a.st[0][i] = x[p]; a.st[1][i] = y[p]; a.st[2][i] = z[p];
      a.st[3][i] = vx[p]; a.st[4][i] = vy[p]; a.st[5][i] = vz[p];
      if (flag[p] != 0) {
        a.flag[i] = flag[p];
        a.rstep[i] = a.step0 + rs[p];
      }
    }
  }
  // steps started by this thread's particles: all nsteps for a survivor; for a particle flagged at
  // record k, KDK: k if a force-evaluation test caught it and k + 1 if its drift did (flags 3 and 4);
  // DKD: k + 1 whatever caught it (the step had begun with its first half drift)
  unsigned drifts = 0;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    if (was_alive[p])
      drifts += flag[p] == 0 ? static_cast<unsigned>(nsteps)
                             : static_cast<unsigned>(rs[p]) +
                                   ((DKD || flag[p] == GLISSE_FLAG_NONCONV || flag[p] == GLISSE_FLAG_UNBOUND) ? 1u : 0u);
  }
  unsigned tot = __reduce_add_sync(kFullMask, drifts);
  if (lane == 0 && tot) atomicAdd(a.pstep_counter, static_cast<unsigned long long>(tot));
  if (STATS && lane == 0) {
    atomicAdd(a.solver_stats, static_cast<unsigned long long>(stat_calls));
    atomicAdd(a.solver_stats + 1, static_cast<unsigned long long>(stat_iters));
    atomicAdd(a.solver_stats + 2, static_cast<unsigned long long>(stat_slow));
  }
  // (the group index is rebuilt from i0 rather than kept live across the step loop)
  publish_group(a, lane, static_cast<int>((i0 - threadIdx.x) / (kParticleBlock * P)));
}

size_t particle_smem_bytes(const ParticleArgs& a) {
  return static_cast<size_t>(kParticleWarps) * kRingSlots * a.stage_recs * a.stride * 8 +
         static_cast<size_t>(kParticleWarps) * kRingSlots * 8;
}

// Bodies that would take the third-order starting point at this instant (guess_order = 0 chooses the
// instantiation from their share at create).  Plain arithmetic: off the hot path.
__global__ void __launch_bounds__(256) count_refine_kernel(const double* x, const double* y, const double* z,
                                                            const double* vx, const double* vy, const double* vz,
                                                            long long n, double mu, double dt,
                                                            unsigned long long* out) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  bool want = false;
  if (i < n) {
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
  const int c = __syncthreads_count(want);
  if (threadIdx.x == 0 && c) atomicAdd(out, static_cast<unsigned long long>(c));
}

template <int NP, bool STATS, bool DKD, bool REFINE>
cudaError_t configure_kernel() {
  return cudaFuncSetAttribute(particle_kernel<NP, kParticlesPerThread, STATS, DKD, REFINE>,
                              cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

template <int NP>
cudaError_t configure_one() {
  cudaError_t e;
  if ((e = configure_kernel<NP, false, false, false>())) return e;
  if ((e = configure_kernel<NP, false, false, true>())) return e;
  if ((e = configure_kernel<NP, false, true, false>())) return e;
  if ((e = configure_kernel<NP, false, true, true>())) return e;
  if ((e = configure_kernel<NP, true, false, false>())) return e;
  return configure_kernel<NP, true, false, true>();
}

template <int NP, bool STATS, bool DKD, bool REFINE>
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
  return cudaLaunchKernelEx(&cfg, particle_kernel<NP, kParticlesPerThread, STATS, DKD, REFINE>, a);
}

template <int NP, bool REFINE>
cudaError_t launch_np(const ParticleArgs& a, int n_groups, size_t smem, bool chained, bool stats, bool dkd, cudaStream_t s) {
  if (dkd) return launch_one<NP, false, true, REFINE>(a, n_groups, smem, chained, s);   // (no instrumented DKD instantiation)
  return stats ? launch_one<NP, true, false, REFINE>(a, n_groups, smem, chained, s)
               : launch_one<NP, false, false, REFINE>(a, n_groups, smem, chained, s);
}

}  // namespace

cudaError_t configure_particle_kernels() {
  cudaError_t e;
  if ((e = configure_one<0>())) return e;
  if ((e = configure_one<4>())) return e;
  return configure_one<8>();
}

cudaError_t launch_particle_kernel(const ParticleArgs& a, int n_groups, bool chained, bool stats, bool dkd, bool refine,
                                   cudaStream_t s) {
  if (n_groups < 1) n_groups = 1;
  const size_t smem = particle_smem_bytes(a);
  cudaError_t e;
  if (a.np == 4) e = refine ? launch_np<4, true>(a, n_groups, smem, chained, stats, dkd, s) : launch_np<4, false>(a, n_groups, smem, chained, stats, dkd, s);
  else if (a.np == 8) e = refine ? launch_np<8, true>(a, n_groups, smem, chained, stats, dkd, s) : launch_np<8, false>(a, n_groups, smem, chained, stats, dkd, s);
  else e = refine ? launch_np<0, true>(a, n_groups, smem, chained, stats, dkd, s) : launch_np<0, false>(a, n_groups, smem, chained, stats, dkd, s);
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_count_refine(const double* const st[6], long long n, double mu, double dt, unsigned long long* out,
                                cudaStream_t s) {
  count_refine_kernel<<<static_cast<int>((n + 255) / 256), 256, 0, s>>>(st[0], st[1], st[2], st[3], st[4], st[5], n, mu, dt, out);
  return cudaGetLastError();
}

// particles per launch group (one warp's worth): the host sizes grids and completion lists with it
int particles_per_group() { return kParticleBlock * kParticlesPerThread; }

}  // namespace glisse
