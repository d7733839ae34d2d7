// compact.cu — survivor compaction ("resync", step a8 of DESIGN.md) and the small
// bookkeeping kernels around it.
//
// The paper runs a stable partition that moves deactivated particles to the array tail so later
// launches cover only active ones, keeping the relative order of the survivors.  Here: a
// warp-ballot + prefix-sum stable partition in three small kernels (per-block count, scan of the
// block counts, scatter).  Survivors go, in order, to the prefix of the other working buffer; a
// removed particle's frozen state goes to its ORIGINAL index in the `fin` arrays, which is where
// glisse_read assembles the result, so compaction is invisible to the caller (reading S16).
//
// Iteration-count binning ("it is desirable to sort the particles by the expected number
// of iterations required to solve Kepler's equation, so that threads in the same block will perform
// similar amounts of work ... the most eccentric group would be launched first"; the paper proposes
// it and did not build it): with bins > 1 the survivors are partitioned by a hardness bin of their
// ORBIT (not of the instant: a chunk spans many revolutions), hardest bin first, particle order kept
// within a bin.  Every survivor is moved by the partition anyway, so the ordering is free; a particle's
// arithmetic never depends on its warp-mates, so results are bit-identical to the unbinned run.
#include "glisse_internal.cuh"
#include "kepler.cuh"

namespace glisse {
namespace {

constexpr int kBlock = 256;
constexpr unsigned kFull = 0xffffffffu;

// Hardness bin of an orbit for the particle kernel's Kepler solver (kepler.cuh): 0 = one quartic step
// is accepted at every phase of the orbit, 1 = some phases need more, 2 = some phase leaves the fast
// solver (e >= 0.8, |x0| > pi/4, unbound).  The fast solver starts from x0 = dM/q, q = 1 - e cos E0,
// and accepts once the Newton update delta = f(x0)/f'(x0) is below an eccentricity-dependent bound.
// With Kepler's equation as  q x + (es/2) x^2 + (ec/6) x^3 - (es/24) x^4 ... = dM  the update left by the
// first-order starting point is ~ [(es/2) x0^2 + (ec/6) x0^3] / q, and by the third-order reversion
// (where the body qualifies for it: kepler.cuh) ~ |5 b2^3 - 5 b2 b3 + b4| y^4 with b2 = es/2q, b3 = ec/6q,
// b4 = -es/24q, y = dM/q.  First a bound: the largest these can be over the phase E0 — every e sin, e cos
// replaced by e, every q by 1 - e — with a safety factor of 2: closed form, a few dozen operations, and it
// clears every body of a quiet population.  A body it does not clear is then looked at phase by phase:
// delta at 12 phases E0, from the starting point the run's instantiation would use.  The key is evaluated
// for every survivor at every resync.  A heuristic: it decides only which particles share a warp,
// never a result.
__device__ int hardness_bin(double mu, double dt, bool refine, double x, double y, double z, double vx, double vy,
                            double vz) {
  const double r = sqrt(x * x + y * y + z * z);
  const double v2 = vx * vx + vy * vy + vz * vz;
  const double u = x * vx + y * vy + z * vz;
  const double alpha = 2.0 * mu / r - v2;
  if (!(alpha > 0.0)) return 2;
  const double ec = 1.0 - r * alpha / mu;
  const double e2 = ec * ec + u * u * alpha / (mu * mu);
  if (!(e2 < 0.64)) return 2;
  const double e = sqrt(e2);
  const double kTwoPi = 6.283185307179586;
  double dM = alpha * sqrt(alpha) * dt / mu;
  dM = fabs(dM - kTwoPi * rint(dM / kTwoPi));
  const double q = 1.0 - e;                       // smallest q of the orbit
  if (dM >= 0.78539816 * q) return 2;
  const double thr = 0.5 * fmin(9e-5, 1.9e-5 * 0.64 / e2);   // kepler.cuh: fast_threshold, with the safety factor
  const double y0 = dM / q;                       // largest starting point of the orbit
  const double b2 = 0.5 * e / q, b3 = e / (6.0 * q), b4 = e / (24.0 * q);
  double worst = (b2 + b3 * y0) * y0 * y0;       // first-order starting point
  if (refine && wants_refined_guess(hi_word(e2), hi_abs(y0)))
    worst = (5.0 * b2 * b2 * b2 + 5.0 * b2 * b3 + b4) * (y0 * y0) * (y0 * y0);
  if (worst < thr) return 0;
  worst = 0.0;
  for (int k = 0; k < 12; ++k) {
    double s0, c0;
    sincos(kTwoPi * k / 12.0, &s0, &c0);
    const double qk = 1.0 - e * c0, es = e * s0;
    double x0 = dM / qk;
    if (refine && wants_refined_guess(hi_word(e2), hi_abs(x0))) {
      const double c2 = 0.5 * es / qk, c3 = e * c0 / (6.0 * qk);
      x0 = x0 + x0 * x0 * (-c2 + (2.0 * c2 * c2 - c3) * x0);
    }
    double sx, cx;
    sincos(x0, &sx, &cx);
    const double f = (x0 - dM) - e * c0 * sx + es * (1.0 - cx);   // Kepler's equation at x0
    const double f1 = 1.0 - e * c0 * cx + es * sx;
    worst = fmax(worst, fabs(f / f1));
  }
  return worst < thr ? 0 : 1;
}

// per block and per bin: number of active slots; also writes every slot's bin
__global__ void __launch_bounds__(kBlock) count_block_actives(const CompactArgs a, int nb) {
  __shared__ int cnt[kCompactBins];
  const int n = *a.n_in;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  const bool act = (i < n) && (a.src_flag[i] == 0);
  if (threadIdx.x < kCompactBins) cnt[threadIdx.x] = 0;
  __syncthreads();
  int b = 0;
  if (act && a.bins > 1)
    b = hardness_bin(a.mu, a.dt, a.refine != 0, a.src[0][i], a.src[1][i], a.src[2][i], a.src[3][i], a.src[4][i],
                     a.src[5][i]);
  if (i < n) a.bin[i] = static_cast<unsigned char>(b);
  for (int k = 0; k < a.bins; ++k) {
    const unsigned m = __ballot_sync(kFull, act && b == k);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(&cnt[k], __popc(m));
  }
  __syncthreads();
  // hardest bin first: output order index = bins - 1 - bin
  if (threadIdx.x < a.bins) a.block_counts[(a.bins - 1 - threadIdx.x) * nb + blockIdx.x] = cnt[threadIdx.x];
}

// exclusive scan of block_counts[0..nb) in place (one block), total -> *n_out
// n_out_host (may be null): mapped pinned word that also receives the total — the host learns the
// survivor count without a device-to-host copy in the particle stream (a copy there would queue behind
// a snapshot's multi-megabyte copies on the same copy engine and hold the next chunk back)
__global__ void __launch_bounds__(1024) scan_block_counts(int* __restrict__ block_counts, int nb,
                                                           int* __restrict__ n_out, volatile int* n_out_host) {
  __shared__ int warp_sums[32];
  __shared__ int carry_s;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < nb; base += 1024) {
    const int i = base + threadIdx.x;
    const int v = (i < nb) ? block_counts[i] : 0;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(kFull, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      int w = warp_sums[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(kFull, w, o);
        if (lane >= o) w += t;
      }
      warp_sums[lane] = w;  // inclusive over warps
    }
    __syncthreads();
    const int carry = carry_s;
    const int warp_off = warp ? warp_sums[warp - 1] : 0;
    if (i < nb) block_counts[i] = carry + warp_off + inc - v;
    __syncthreads();
    if (threadIdx.x == 0) carry_s = carry + warp_sums[31];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    *n_out = carry_s;
    if (n_out_host) {
      *n_out_host = carry_s;
      __threadfence_system();
    }
  }
}

__global__ void __launch_bounds__(kBlock) scatter_partition(const CompactArgs a, int nb) {
  __shared__ int warp_counts[kCompactBins][kBlock / 32];
  const int n = *a.n_in;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool in = i < n;
  const int fl = in ? a.src_flag[i] : -1;
  const bool act = fl == 0;
  const int b = act ? a.bin[i] : 0;
  unsigned m = 0;   // ballot of this thread's own bin
  for (int k = 0; k < a.bins; ++k) {
    const unsigned mk = __ballot_sync(kFull, act && b == k);
    if (lane == 0) warp_counts[k][warp] = __popc(mk);
    if (b == k) m = mk;
  }
  __syncthreads();
  if (!in) return;
  const int id = a.src_id[i];
  if (act) {
    int off = a.block_counts[(a.bins - 1 - b) * nb + blockIdx.x];
    for (int w = 0; w < warp; ++w) off += warp_counts[b][w];
    const int d = off + __popc(m & ((1u << lane) - 1u));
#pragma unroll
    for (int k = 0; k < 6; ++k) a.dst[k][d] = a.src[k][i];
    a.dst_id[d] = id;
    a.dst_flag[d] = 0;
    a.dst_rstep[d] = -1;
  } else {
#pragma unroll
    for (int k = 0; k < 6; ++k) a.fin[k][id] = a.src[k][i];
    a.fin_flag[id] = fl;
    a.fin_rstep[id] = a.src_rstep[i];
  }
}

__global__ void __launch_bounds__(kBlock) scatter_to_original(const ScatterArgs a) {
  const int n = *a.n_slots;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i >= n) return;
  const int id = a.id[i];
#pragma unroll
  for (int k = 0; k < 6; ++k) a.fin[k][id] = a.st[k][i];
  a.fin_flag[id] = a.flag[i];
  a.fin_rstep[id] = a.rstep[i];
}

__global__ void __launch_bounds__(kBlock) count_active_kernel(const int* __restrict__ flag,
                                                               const int* __restrict__ n_slots,
                                                               unsigned long long* __restrict__ out) {
  const int n = *n_slots;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  const bool act = (i < n) && (flag[i] == 0);
  const int c = __syncthreads_count(act);
  if (threadIdx.x == 0 && c) atomicAdd(out, static_cast<unsigned long long>(c));
}

}  // namespace

cudaError_t launch_compaction(const CompactArgs& a, int n_slots_upper, cudaStream_t s, long long* launches) {
  if (n_slots_upper < 1) n_slots_upper = 1;
  const int nb = (n_slots_upper + kBlock - 1) / kBlock;
  count_block_actives<<<nb, kBlock, 0, s>>>(a, nb);
  scan_block_counts<<<1, 1024, 0, s>>>(a.block_counts, a.bins * nb, a.n_out, a.n_out_host);
  scatter_partition<<<nb, kBlock, 0, s>>>(a, nb);
  if (launches) *launches += 3;
  return cudaGetLastError();
}

cudaError_t launch_scatter_to_original(const ScatterArgs& a, int n_slots_upper, cudaStream_t s) {
  if (n_slots_upper < 1) n_slots_upper = 1;
  scatter_to_original<<<(n_slots_upper + kBlock - 1) / kBlock, kBlock, 0, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_count_active(const int* flag, const int* n_slots, int n_slots_upper, unsigned long long* out,
                                cudaStream_t s) {
  if (n_slots_upper < 1) n_slots_upper = 1;
  count_active_kernel<<<(n_slots_upper + kBlock - 1) / kBlock, kBlock, 0, s>>>(flag, n_slots, out);
  return cudaGetLastError();
}

}  // namespace glisse
