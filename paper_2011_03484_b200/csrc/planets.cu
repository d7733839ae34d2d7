// planets.cu — the planet-history kernel (step a1 of DESIGN.md; "standard
// Wisdom-Holman" for the mutually interacting planets, PAPER.md:109-115 planet log and h0).
//
// The paper integrates the planets on the CPU and ships each chunk over PCIe; here
// one warp advances them on the device, lane k = planet k in Jacobi order, and writes the chunk of
// K+1 log records straight to HBM, one chunk ahead of the particle kernel on its own stream.
// The step is serial in time, so what matters is latency: all sums over planets run through
// register shuffles, in the index order of the definition (O3).
//
//   eta_k = gm0 + sum_{i<=k} gm_i ;  Jacobi r'_k = q_k − (sum_{i<k} gm_i q_i)/eta_{k-1}
//   q_k = r'_k + sum_{i<k} (gm_i/eta_i) r'_i
//   kick:  v'_k += h (eta_k/eta_{k-1}) [ gm0 r'_k/|r'_k|^3 + A_k + (1/eta_k) sum_{i>k} gm_i A_i ]
//          A_i = − gm0 q_i/|q_i|^3 − sum_{j != i} gm_j (q_i − q_j)/|q_i − q_j|^3
//   drift: two-body motion of (r'_k, v'_k) about mu_k = gm0 eta_k/eta_{k-1}
#include <mutex>

#include "glisse_internal.cuh"
#include "kepler.cuh"

namespace glisse {
namespace {

constexpr int kPlanetKeplerIters = 10;
constexpr double kPlanetKeplerTol = 1e-13;

struct Lane {
  int np, lane;
  bool live;
  double gm0, gm, eta, eta_prev, wj;  // wj = gm/eta
  double inv_eta, inv_eta_prev, sc;   // 1/eta_k, 1/eta_{k-1}, eta_k/eta_{k-1}
  double mu, inv_mu;
};

__device__ __forceinline__ double shfl(double v, int src) { return __shfl_sync(kFullMask, v, src); }

// NP > 0: compile-time planet count, every sum over planets fully unrolled so that the np
// independent chains (one rsqrt each) overlap: the step is serial in time and latency is all that
// counts.  NP == 0: run-time count.
template <int NP>
__device__ __forceinline__ int count(const Lane& L) { return NP > 0 ? NP : L.np; }

// Partner of this lane in round jj = 0 .. np−2 of an all-pairs exchange: lane+1, lane+2, ... wrapping
// at np.  No lane ever meets itself, so the pair terms need no self test and no branch; partners
// above the lane come first and in increasing order, then those below it in increasing order, so the
// one-sided sums of the definition (over i > k, over i < k) are still added in increasing i.
template <int NP>
__device__ __forceinline__ int partner(const Lane& L, int jj) {
  const int np = count<NP>(L);
  const int j = L.lane + 1 + jj;
  return j >= np ? j - np : j;   // lanes >= np (idle) read some live lane; their results are discarded
}

// s += take ? t : 0, the one-sided sums of the Jacobi maps.  Up to four planets the condition (a function of
// lane and round only) is kept as a weight 1.0 / 0.0 in a register over the step loop and the sum is ONE fma:
// fma(1, t, s) = t + s and fma(0, t, s) = s to the bit (36 selects fewer per step at N_p = 4; measured slower
// from N_p = 8 on, where the weights no longer fit the registers).
template <int NP>
__device__ __forceinline__ void add_if(bool take, double t, double& s) {
  if constexpr (NP > 0 && NP <= 4) s = fma(take ? 1.0 : 0.0, t, s);
  else s += take ? t : 0.0;
}

// q from r' (Jacobi -> heliocentric): q_k = r'_k + sum_{i<k} (gm_i/eta_i) r'_i; the same linear map
// serves velocities
template <int NP>
__device__ __forceinline__ void jacobi_to_helio(const Lane& L, double rx, double ry, double rz, double& qx,
                                                double& qy, double& qz) {
  const int np = count<NP>(L);
  const double cx = L.wj * rx, cy = L.wj * ry, cz = L.wj * rz;
  double sx = 0.0, sy = 0.0, sz = 0.0;
#pragma unroll
  for (int jj = 0; jj + 1 < np; ++jj) {
    const int j = partner<NP>(L, jj);
    const double tx = shfl(cx, j), ty = shfl(cy, j), tz = shfl(cz, j);
    add_if<NP>(j < L.lane, tx, sx); add_if<NP>(j < L.lane, ty, sy); add_if<NP>(j < L.lane, tz, sz);
  }
  qx = rx + sx; qy = ry + sy; qz = rz + sz;
}

// r' from q (heliocentric -> Jacobi): r'_k = q_k − (sum_{i<k} gm_i q_i)/eta_{k−1}
template <int NP>
__device__ __forceinline__ void helio_to_jacobi(const Lane& L, double qx, double qy, double qz, double& rx,
                                                double& ry, double& rz) {
  const int np = count<NP>(L);
  const double cx = L.gm * qx, cy = L.gm * qy, cz = L.gm * qz;
  double sx = 0.0, sy = 0.0, sz = 0.0;
#pragma unroll
  for (int jj = 0; jj + 1 < np; ++jj) {
    const int j = partner<NP>(L, jj);
    const double tx = shfl(cx, j), ty = shfl(cy, j), tz = shfl(cz, j);
    add_if<NP>(j < L.lane, tx, sx); add_if<NP>(j < L.lane, ty, sy); add_if<NP>(j < L.lane, tz, sz);
  }
  rx = qx - sx * L.inv_eta_prev; ry = qy - sy * L.inv_eta_prev; rz = qz - sz * L.inv_eta_prev;
}

// Jacobi acceleration of this lane's planet, and h0 (valid on lane 0, which writes it)
template <int NP>
__device__ __forceinline__ void kick_accel(const Lane& L, double qx, double qy, double qz, double rx, double ry,
                                           double rz, double r2, double& ax, double& ay, double& az, double& hx,
                                           double& hy, double& hz) {
  const int np = count<NP>(L);
  // star term of A_i and this planet's contribution to h0
  const double q2 = fma(qx, qx, fma(qy, qy, qz * qz));
  const double qi3 = gm_over_r3(1.0, q2);
  double Ax = -(L.gm0 * qi3) * qx, Ay = -(L.gm0 * qi3) * qy, Az = -(L.gm0 * qi3) * qz;
  const double tx = (L.gm * qi3) * qx, ty = (L.gm * qi3) * qy, tz = (L.gm * qi3) * qz;
  // the Jacobi two-body term, independent of the sums below
  const double w0 = gm_over_r3(L.gm0, r2);   // r2 = |r'|^2
  hx = -tx; hy = -ty; hz = -tz;   // lane 0: t_0, then t_1, t_2, ... in the rounds below
#pragma unroll
  for (int jj = 0; jj + 1 < np; ++jj) {
    const int j = partner<NP>(L, jj);
    const double gj = shfl(L.gm, j);
    const double qjx = shfl(qx, j), qjy = shfl(qy, j), qjz = shfl(qz, j);
    hx -= shfl(tx, j); hy -= shfl(ty, j); hz -= shfl(tz, j);
    const double dx = qx - qjx, dy = qy - qjy, dz = qz - qjz;
    const double d2 = fma(dx, dx, fma(dy, dy, dz * dz));
    const double w = gm_over_r3(gj, d2);
    Ax = fma(-w, dx, Ax); Ay = fma(-w, dy, Ay); Az = fma(-w, dz, Az);
  }
  // tail_k = sum_{i>k} gm_i A_i, added in increasing i
  const double mx = L.gm * Ax, my = L.gm * Ay, mz = L.gm * Az;
  double Tx = 0.0, Ty = 0.0, Tz = 0.0;
#pragma unroll
  for (int jj = 0; jj + 1 < np; ++jj) {
    const int j = partner<NP>(L, jj);
    const double ux = shfl(mx, j), uy = shfl(my, j), uz = shfl(mz, j);
    add_if<NP>(j > L.lane, ux, Tx); add_if<NP>(j > L.lane, uy, Ty); add_if<NP>(j > L.lane, uz, Tz);
  }
  // idle lanes get a zero kick: their stand-in orbit stays the circle it started as
  const double sc = L.live ? L.sc : 0.0;
  ax = sc * (fma(w0, rx, Ax) + Tx * L.inv_eta);
  ay = sc * (fma(w0, ry, Ay) + Ty * L.inv_eta);
  az = sc * (fma(w0, rz, Az) + Tz * L.inv_eta);
}

__device__ __forceinline__ Lane make_lane(const PlanetSystem* sys) {
  Lane L;
  L.np = sys->np;
  L.lane = threadIdx.x & 31;
  L.live = L.lane < L.np;
  L.gm0 = sys->gm0;
  L.gm = L.live ? sys->gm[L.lane] : 0.0;
  L.eta = L.live ? sys->eta[L.lane] : 1.0;
  L.eta_prev = L.live ? sys->eta_prev[L.lane] : 1.0;
  L.wj = L.gm / L.eta;
  L.inv_eta = 1.0 / L.eta;
  L.inv_eta_prev = 1.0 / L.eta_prev;
  L.sc = L.eta / L.eta_prev;
  L.mu = L.gm0 * L.eta / L.eta_prev;
  L.inv_mu = 1.0 / L.mu;
  return L;
}

template <int NP>
__device__ __forceinline__ void write_record(const Lane& L, double* log, double* jlog, int rec, int stride,
                                             double qx, double qy, double qz, double hx, double hy, double hz,
                                             double rx, double ry, double rz, double vx, double vy, double vz) {
  const int np = count<NP>(L);
  double* r = log + static_cast<size_t>(rec) * stride;
  if (L.live) {
    r[3 * L.lane] = qx; r[3 * L.lane + 1] = qy; r[3 * L.lane + 2] = qz;
    double* js = jlog + static_cast<size_t>(rec) * 6 * np;
    js[3 * L.lane] = rx; js[3 * L.lane + 1] = ry; js[3 * L.lane + 2] = rz;
    js[3 * np + 3 * L.lane] = vx; js[3 * np + 3 * L.lane + 1] = vy; js[3 * np + 3 * L.lane + 2] = vz;
  }
  if (L.lane == 0) {
    r[3 * np] = hx; r[3 * np + 1] = hy; r[3 * np + 2] = hz;
    if ((3 * np + 3) & 1) r[3 * np + 3] = 0.0;   // the one padding word of an odd record (log_stride)
  }
}

template <int NP>
__global__ void __launch_bounds__(32) planet_history_kernel(const PlanetSystem* sys, const double* __restrict__ jin,
                                                             double* __restrict__ log, double* __restrict__ jlog,
                                                             int nsteps, double dt, long long step0,
                                                             long long* fail_step) {
  const Lane L = make_lane(sys);
  const int stride = log_stride(count<NP>(L));
  const double hdt = 0.5 * dt;
  const double inv_mu_dt = L.inv_mu * dt;
  const double two_mu = 2.0 * L.mu;
  // Idle lanes (lane >= np) carry a stand-in: a circular orbit with n dt = 0.01, never kicked, never
  // written.  It takes the same path through the drift as the planets (one quartic step), so the
  // warp does not diverge there; a lane that is merely masked off would.
  // Each idle lane sits at its own phase of that circle: two lanes at the same point would meet at distance
  // zero in the all-pairs exchange, and the NaN of that (discarded) term would reach the lane's velocity
  // through 0 x NaN, and from there send the whole warp through the definition's solver at every step.
  const double r_idle = cbrt(L.gm0 * dt * dt * 1e4);
  double s_idle, c_idle;
  sincospi(L.lane * (1.0 / 16.0), &s_idle, &c_idle);
  const double v_idle = sqrt(L.gm0 / r_idle);
  double rx = r_idle * c_idle, ry = r_idle * s_idle, rz = 0.0, vx = -v_idle * s_idle, vy = v_idle * c_idle, vz = 0.0;
  if (L.live) {
    rx = jin[3 * L.lane]; ry = jin[3 * L.lane + 1]; rz = jin[3 * L.lane + 2];
    vx = jin[3 * L.np + 3 * L.lane]; vy = jin[3 * L.np + 3 * L.lane + 1]; vz = jin[3 * L.np + 3 * L.lane + 2];
  }
  double qx, qy, qz, ax, ay, az, hx, hy, hz;
  // |r'|^2 and its inverse root for the NEXT drift: the kick leaves the positions alone, so both are known
  // as soon as the drift ends and are computed beside the kick, off the dependent chain of the step
  double r2 = fma(rx, rx, fma(ry, ry, rz * rz));
  double rinv = rsqrt_f64(r2);
  jacobi_to_helio<NP>(L, rx, ry, rz, qx, qy, qz);
  kick_accel<NP>(L, qx, qy, qz, rx, ry, rz, r2, ax, ay, az, hx, hy, hz);
  write_record<NP>(L, log, jlog, 0, stride, qx, qy, qz, hx, hy, hz, rx, ry, rz, vx, vy, vz);
  int bad = -1;   // first step (within this launch) whose drift failed
  for (int s = 0; s < nsteps; ++s) {
    vx = fma(ax, hdt, vx); vy = fma(ay, hdt, vy); vz = fma(az, hdt, vz);
    // third-order starting point (kepler.cuh): Jupiter at dt = 180 d needs one quartic step instead of two
    // The drift in the particle kernel's three pieces (kepler.cuh), with no per-lane predicate: begin, ONE
    // fast-solver step, finish.  If any lane (planet or stand-in) is not served by that — not accepted, e >= 0.8,
    // |x| > pi/4, a step of half a revolution or more, unbound — the whole warp takes the general routine
    // instead, from the untouched state; for the lanes the short form does serve, the two are the same
    // arithmetic, bit for bit.
    int st = 0;
    {
      DriftVars dv;
      double xk, xn, sm, cm1, dl;
      bool unbound;
      drift_begin_rinv<true>(L.mu, two_mu, L.inv_mu, inv_mu_dt, r2, rinv, rx, ry, rz, vx, vy, vz, dv, xk, unbound);
      const int e2h = hi_word(dv.e2);
      const int thr = e2h < kHiE2_010 ? kHiThr0 : (e2h < kHiE2_030 ? kHiThr1 : (e2h < kHiE2_050 ? kHiThr2 : kHiThr3));
      const bool hard = !(e2h < kHiE2_080) | !is_small_angle(xk) | !(hi_abs(dv.dM) < kHiPi);
      fast_step(dv, xk, xn, sm, cm1, dl);
      if (__any_sync(kFullMask, hard | !(hi_abs(dl) < thr))) {
        st = kepler_drift_one<true>(true, L.mu, L.inv_mu, inv_mu_dt, kPlanetKeplerIters, kPlanetKeplerTol, r2, rx, ry,
                                    rz, vx, vy, vz);
      } else {
        drift_finish(dv, xn, sm, cm1, rx, ry, rz, vx, vy, vz);
      }
    }
    const unsigned failed = __ballot_sync(kFullMask, st != 0 && L.live);
    if (failed && bad < 0) bad = s;
    r2 = fma(rx, rx, fma(ry, ry, rz * rz));
    rinv = rsqrt_f64(r2);
    jacobi_to_helio<NP>(L, rx, ry, rz, qx, qy, qz);
    kick_accel<NP>(L, qx, qy, qz, rx, ry, rz, r2, ax, ay, az, hx, hy, hz);
    vx = fma(ax, hdt, vx); vy = fma(ay, hdt, vy); vz = fma(az, hdt, vz);
    write_record<NP>(L, log, jlog, s + 1, stride, qx, qy, qz, hx, hy, hz, rx, ry, rz, vx, vy, vz);
  }
  // records up to and including step0 + bad are valid (glisse_internal.cuh: kNoPlanetFailure)
  if (bad >= 0 && L.lane == 0) atomicMin(fail_step, step0 + bad);
}

__global__ void __launch_bounds__(32) planet_init_kernel(const PlanetSystem* sys, const double* q, const double* qd,
                                                          double* jstate) {
  const Lane L = make_lane(sys);
  double qx = 0, qy = 0, qz = 0, wx = 0, wy = 0, wz = 0;
  if (L.live) {
    qx = q[3 * L.lane]; qy = q[3 * L.lane + 1]; qz = q[3 * L.lane + 2];
    wx = qd[3 * L.lane]; wy = qd[3 * L.lane + 1]; wz = qd[3 * L.lane + 2];
  }
  double rx, ry, rz, vx, vy, vz;
  helio_to_jacobi<0>(L, qx, qy, qz, rx, ry, rz);
  helio_to_jacobi<0>(L, wx, wy, wz, vx, vy, vz);
  if (L.live) {
    jstate[3 * L.lane] = rx; jstate[3 * L.lane + 1] = ry; jstate[3 * L.lane + 2] = rz;
    jstate[3 * L.np + 3 * L.lane] = vx; jstate[3 * L.np + 3 * L.lane + 1] = vy;
    jstate[3 * L.np + 3 * L.lane + 2] = vz;
  }
}

__global__ void __launch_bounds__(32) planet_read_kernel(const PlanetSystem* sys, const double* jstate, double* q,
                                                          double* qd) {
  const Lane L = make_lane(sys);
  double rx = 0, ry = 0, rz = 0, vx = 0, vy = 0, vz = 0;
  if (L.live) {
    rx = jstate[3 * L.lane]; ry = jstate[3 * L.lane + 1]; rz = jstate[3 * L.lane + 2];
    vx = jstate[3 * L.np + 3 * L.lane]; vy = jstate[3 * L.np + 3 * L.lane + 1];
    vz = jstate[3 * L.np + 3 * L.lane + 2];
  }
  double qx, qy, qz, wx, wy, wz;
  jacobi_to_helio<0>(L, rx, ry, rz, qx, qy, qz);
  jacobi_to_helio<0>(L, vx, vy, vz, wx, wy, wz);
  if (L.live) {
    if (q) { q[3 * L.lane] = qx; q[3 * L.lane + 1] = qy; q[3 * L.lane + 2] = qz; }
    if (qd) { qd[3 * L.lane] = wx; qd[3 * L.lane + 1] = wy; qd[3 * L.lane + 2] = wz; }
  }
}


// Planet log from a sparse history ("interpolation from a history file"; DESIGN.md reading
// S24): one thread per record.  The cubic that matches positions and velocities at both ends of the interval
// [t_m, t_m+1] that holds t, in powers of tau = (t - t_m)/D:
//   q(t) = q_m + tau { D qd_m + tau [ 3 d - D (2 qd_m + qd_m+1) + tau ( -2 d + D (qd_m + qd_m+1) ) ] },  d = q_m+1 - q_m
// then h0 = -sum_j gm_j q_j/|q_j|^3 of the interpolated positions.  The interval is found by bisection.
__global__ void __launch_bounds__(128) interpolate_log_kernel(const PlanetSystem* sys, long long n_samples,
                                                              const double* __restrict__ st,
                                                              const double* __restrict__ sq,
                                                              const double* __restrict__ sv, double t_first,
                                                              double dt_record, long long n_records,
                                                              double* __restrict__ log) {
  const long long r = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (r >= n_records) return;
  const int np = sys->np;
  const int stride = log_stride(np);
  const double t = t_first + static_cast<double>(r) * dt_record;
  long long lo = 0, hi = n_samples - 1;   // invariant: st[lo] <= t (<= st[hi]); ends with hi = lo + 1
  while (hi - lo > 1) {
    const long long mid = (lo + hi) >> 1;
    if (t >= st[mid]) lo = mid; else hi = mid;
  }
  const double D = st[lo + 1] - st[lo];
  const double tau = (t - st[lo]) / D;
  double* rec = log + r * stride;
  double hx = 0.0, hy = 0.0, hz = 0.0;
  for (int j = 0; j < np; ++j) {
    double q[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const long long i0 = (lo * np + j) * 3 + c, i1 = ((lo + 1) * np + j) * 3 + c;
      const double q0 = sq[i0], d = sq[i1] - q0;
      const double v0 = D * sv[i0], v1 = D * sv[i1];
      const double c2 = 3.0 * d - (2.0 * v0 + v1);
      const double c3 = (v0 + v1) - 2.0 * d;
      q[c] = q0 + tau * (v0 + tau * (c2 + tau * c3));
      rec[3 * j + c] = q[c];
    }
    const double r2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2];
    const double w = sys->gm[j] / (r2 * sqrt(r2));
    hx -= w * q[0]; hy -= w * q[1]; hz -= w * q[2];
  }
  rec[3 * np] = hx; rec[3 * np + 1] = hy; rec[3 * np + 2] = hz;
  for (int c = 3 * np + 3; c < stride; ++c) rec[c] = 0.0;
}

}  // namespace

cudaError_t launch_planet_kernel(const PlanetSystem* sys, int np, const double* jin, double* log, double* jlog,
                                 int nsteps, double dt, long long step0, long long* fail_step, int exclusive_sm_bytes,
                                 cudaStream_t s) {
  // The kernel is one warp whose K steps are serial: all that counts is its latency, and sharing an
  // SM with ~25 particle warps that saturate the FP64 pipe doubles it.  It therefore asks for the
  // whole shared memory of an SM (unused), which keeps every other block off that SM: 1/148 of the
  // device for the ~1.4 ms it runs per chunk.
  const size_t smem = exclusive_sm_bytes > 0 ? static_cast<size_t>(exclusive_sm_bytes) : 0;
  switch (np) {
    case 4: planet_history_kernel<4><<<1, 32, smem, s>>>(sys, jin, log, jlog, nsteps, dt, step0, fail_step); break;
    case 8: planet_history_kernel<8><<<1, 32, smem, s>>>(sys, jin, log, jlog, nsteps, dt, step0, fail_step); break;
    default: planet_history_kernel<0><<<1, 32, smem, s>>>(sys, jin, log, jlog, nsteps, dt, step0, fail_step); break;
  }
  return cudaGetLastError();
}

cudaError_t configure_planet_kernels(int* exclusive_sm_bytes) {
  int dev = 0, optin = 0;
  cudaError_t e;
  if ((e = cudaGetDevice(&dev))) return e;
  if ((e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev))) return e;
  if ((e = cudaFuncSetAttribute(planet_history_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin))) return e;
  if ((e = cudaFuncSetAttribute(planet_history_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin))) return e;
  if ((e = cudaFuncSetAttribute(planet_history_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin))) return e;
  *exclusive_sm_bytes = optin;
  return cudaSuccess;
}

cudaError_t launch_planet_init(const PlanetSystem* sys, const double* q, const double* qd, double* jstate,
                               cudaStream_t s) {
  planet_init_kernel<<<1, 32, 0, s>>>(sys, q, qd, jstate);
  return cudaGetLastError();
}

cudaError_t launch_planet_read(const PlanetSystem* sys, const double* jstate, double* q, double* qd,
                               cudaStream_t s) {
  planet_read_kernel<<<1, 32, 0, s>>>(sys, jstate, q, qd);
  return cudaGetLastError();
}

cudaError_t launch_interpolate_log(const PlanetSystem* sys, long long n_samples, const double* sample_time,
                                   const double* sample_pos, const double* sample_vel, double t_first, double dt_record,
                                   long long n_records, double* log, cudaStream_t s) {
  if (n_records <= 0) return cudaSuccess;
  interpolate_log_kernel<<<static_cast<unsigned>((n_records + 127) / 128), 128, 0, s>>>(
      sys, n_samples, sample_time, sample_pos, sample_vel, t_first, dt_record, n_records, log);
  return cudaGetLastError();
}

// ---- the planet log without any allocation (include/glisse.h: glisse_planet_log_static) --------------------
// The planet-history kernel writes, beside the log, the Jacobi state at every record (so that any step can be
// resumed from): for glisse_planet_log that is scratch, which it gets from cudaMalloc.  Here the scratch is a
// file-scope array in device memory of a fixed size, for callers that may not allocate.  Every GPU that loads
// the library holds these 2 MiB until the process exits; every call on a device shares them.
static __device__ __align__(256) double g_static_jlog[kStaticJlogDoubles];

namespace {
std::mutex g_static_mu;
double* g_static_jlog_addr[64] = {};   // per device: the array's DEVICE address (its name is a host-side stand-in)
}  // namespace

// Device address of the static scratch on the CURRENT device, looked up once per device.
static cudaError_t static_jlog_address(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_jlog_addr[dev]) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_static_jlog);
    if (e != cudaSuccess) return e;
    if (!ptr) return cudaErrorInvalidSymbol;
    g_static_jlog_addr[dev] = ptr;
  }
  *out = g_static_jlog_addr[dev];
  return cudaSuccess;
}

long long static_planet_log_limit(int np) {
  if (np < 0 || np > kMaxPlanets) return -1;
  const long long per_record = np > 0 ? 6LL * np : 1;
  return static_cast<long long>(kStaticJlogDoubles) / per_record - 1;   // records = steps + 1
}

cudaError_t launch_planet_kernel_static(const PlanetSystem* sys, int np, const double* jin, double* log, int nsteps,
                                        double dt, long long step0, long long* fail_step, cudaStream_t s) {
  if (nsteps < 0 || nsteps > static_planet_log_limit(np)) return cudaErrorInvalidValue;   // (the caller checks first)
  double* jlog = nullptr;
  cudaError_t e = static_jlog_address(&jlog);
  if (e != cudaSuccess) return e;
  // Nothing in the scratch has to start at zero: the kernel writes every Jacobi record of this call before
  // anything could read it, and nothing of an earlier call is read.
  return launch_planet_kernel(sys, np, jin, log, jlog, nsteps, dt, step0, fail_step, 0, s);
}

}  // namespace glisse
