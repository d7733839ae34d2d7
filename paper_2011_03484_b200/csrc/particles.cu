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

__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// NP > 0: compile-time planet count (fully unrolled kick); NP == 0: run-time count a.np.
template <int NP>
__global__ void __launch_bounds__(kParticleBlock, GL_MIN_BLOCKS) particle_kernel(const __grid_constant__ ParticleArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const int np = NP > 0 ? NP : a.np;
  const int stride = a.stride;
  const int nsteps = a.nsteps;
  const int R = a.stage_recs;
  const int stage_doubles = R * stride;

  const int n = *a.n_slots;
  const long long i = static_cast<long long>(blockIdx.x) * kParticleBlock + threadIdx.x;
  const bool in_range = i < n;

  // ---- a2: load ------------------------------------------------------------------------------
  double x = 1.0, y = 0.0, z = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
  int flag = -1;
  if (in_range) {
    flag = a.flag[i];
    x = a.st[0][i]; y = a.st[1][i]; z = a.st[2][i];
    vx = a.st[3][i]; vy = a.st[4][i]; vz = a.st[5][i];
  }
  const bool was_alive = (flag == 0);
  bool alive = was_alive;
  if (!__any_sync(kFullMask, alive)) return;  // nothing to do in this warp: leave before any copy
  long long rs = -1;
  unsigned drifts = 0;

  // ---- warp-private ring ------------------------------------------------------------------------
  double* ring = reinterpret_cast<double*>(smem_raw) + static_cast<size_t>(warp) * kRingSlots * stage_doubles;
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<double*>(smem_raw) +
                                               static_cast<size_t>(kParticleWarps) * kRingSlots * stage_doubles) +
                   warp * kRingSlots;
  const int nrec = nsteps + 1;
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
      // ---- a3/a4: force evaluation with the tests (O1/O4/O5) at time t_{step0+k} ----------------
      const double r2 = fma(x, x, fma(y, y, z * z));
      double ax = rec[3 * np], ay = rec[3 * np + 1], az = rec[3 * np + 2];  // h0
      int hit = 0;
#pragma unroll
      for (int jj = 0; jj < np; ++jj) {
        const int j = np - 1 - jj;  // descending, so the lowest index wins (reading S11)
        const double dx = x - rec[3 * j], dy = y - rec[3 * j + 1], dz = z - rec[3 * j + 2];
        const double d2 = fma(dx, dx, fma(dy, dy, dz * dz));
        hit = (d2 < a.rc2[j]) ? (GLISSE_FLAG_PLANET0 + j) : hit;
        const double ri = rsqrt_f64(d2);
        const double w = (a.gm[j] * ri) * (ri * ri);
        ax = fma(-w, dx, ax);
        ay = fma(-w, dy, ay);
        az = fma(-w, dz, az);
      }
      hit = (r2 > a.rmax2) ? GLISSE_FLAG_RMAX : hit;
      hit = (r2 < a.rmin2) ? GLISSE_FLAG_RMIN : hit;
      if (alive && hit != 0) {
        flag = hit;
        rs = a.step0 + k;
        alive = false;
      }
      if (alive) {
        vx = fma(ax, hdt, vx); vy = fma(ay, hdt, vy); vz = fma(az, hdt, vz);
        if (k > 0 && k < nsteps) {  // interior: closing half kick of step k-1 and opening of step k
          vx = fma(ax, hdt, vx); vy = fma(ay, hdt, vy); vz = fma(az, hdt, vz);
        }
      }
      // ---- a5/a6: drift (O2) --------------------------------------------------------------------
      if (k < nsteps) {
        drifts += alive ? 1u : 0u;
        const int st_d = kepler_drift_warp(alive, a.mu, a.inv_mu, a.inv_mu_dt, a.iters, a.tol, r2, x, y, z,
                                           vx, vy, vz);
        if (st_d != 0) {
          flag = st_d;
          rs = a.step0 + k;
          alive = false;
        }
      }
      any_alive = __any_sync(kFullMask, alive);
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
  if (was_alive) {  // particles that were already removed at load are untouched
    a.st[0][i] = x; a.st[1][i] = y; a.st[2][i] = z;
    a.st[3][i] = vx; a.st[4][i] = vy; a.st[5][i] = vz;
    if (flag != 0) {
      a.flag[i] = flag;
      a.rstep[i] = rs;
    }
  }
  unsigned tot = __reduce_add_sync(kFullMask, drifts);
  if (lane == 0 && tot) atomicAdd(a.pstep_counter, static_cast<unsigned long long>(tot));
}

size_t particle_smem_bytes(const ParticleArgs& a) {
  return static_cast<size_t>(kParticleWarps) * kRingSlots * a.stage_recs * a.stride * 8 +
         static_cast<size_t>(kParticleWarps) * kRingSlots * 8;
}

}  // namespace

cudaError_t configure_particle_kernels() {
  cudaError_t e;
  const int carve = cudaSharedmemCarveoutMaxShared;
  if ((e = cudaFuncSetAttribute(particle_kernel<0>, cudaFuncAttributePreferredSharedMemoryCarveout, carve))) return e;
  if ((e = cudaFuncSetAttribute(particle_kernel<4>, cudaFuncAttributePreferredSharedMemoryCarveout, carve))) return e;
  if ((e = cudaFuncSetAttribute(particle_kernel<8>, cudaFuncAttributePreferredSharedMemoryCarveout, carve))) return e;
  return cudaSuccess;
}

cudaError_t launch_particle_kernel(const ParticleArgs& a, int n_slots_upper, cudaStream_t s) {
  if (n_slots_upper < 1) n_slots_upper = 1;
  const int blocks = (n_slots_upper + kParticleBlock - 1) / kParticleBlock;
  const size_t smem = particle_smem_bytes(a);
  if (a.np == 4) particle_kernel<4><<<blocks, kParticleBlock, smem, s>>>(a);
  else if (a.np == 8) particle_kernel<8><<<blocks, kParticleBlock, smem, s>>>(a);
  else particle_kernel<0><<<blocks, kParticleBlock, smem, s>>>(a);
  return cudaGetLastError();
}

}  // namespace glisse
