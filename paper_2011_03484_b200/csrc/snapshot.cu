// snapshot.cu — periodic output of the particle arrays ("For periodic output of
// particle positions ... the particle arrays are copied back to the CPU after a user-configurable
// number of planetary chunk calculations"; "logged orbital elements at a 2048-year
// interval").  SURVEY.md §8(f) row 1.
//
// One kernel turns the original-order arrays (fin[], filled by scatter_to_original) into a staging
// copy — Cartesian as it is, or osculating heliocentric elements (a, e, i, Omega, omega, M) — that
// a third stream copies to the caller while the particle stream goes on integrating.
// HBM-bound: 64 B read + 64 B written per particle, once per snapshot.  CUDA path only: nothing
// here is used by, or derived from, oracle/.
//
// Elements (Murray & Dermott, Solar System Dynamics, §2.8): h = r x v; 1/a = 2/|r| − |v|^2/mu;
// evec = (v x h)/mu − r/|r|; tan i = |h_xy|/h_z; node n = (−h_y, h_x, 0), Omega = atan2(n_y, n_x);
// omega = angle from n to evec about h; e cos E = 1 − |r|/a, e sin E = r.v/sqrt(mu a),
// M = E − e sin E.  Conventions where an angle is undefined: i = 0: Omega = 0, omega measured from
// x; e = 0: omega = 0 and M = angle from n (or x) to r; 1/a <= 0: M = NaN.  Angles in [0, 2 pi).
#include "glisse_internal.cuh"

namespace glisse {
namespace {

constexpr double kTwoPiS = 6.283185307179586476925286766559;

__device__ __forceinline__ double wrap_2pi(double x) {
  x = fmod(x, kTwoPiS);
  return x < 0.0 ? x + kTwoPiS : x;
}

// angle of w in the orbital plane from the node direction (or from x when the node is undefined)
__device__ __forceinline__ double in_plane_angle(const double (&w)[3], const double (&h)[3], double H, double nx,
                                                 double ny, double N) {
  if (N == 0.0) return atan2(h[2] >= 0.0 ? w[1] : -w[1], w[0]);
  const double ax = nx / N, ay = ny / N;                 // nhat = (ax, ay, 0)
  const double hx = h[0] / H, hy = h[1] / H, hz = h[2] / H;
  const double mx = -hz * ay, my = hz * ax, mz = hx * ay - hy * ax;  // hhat x nhat
  return atan2(w[0] * mx + w[1] * my + w[2] * mz, w[0] * ax + w[1] * ay);
}

// osculating elements of (r, v) about mu -> el[0..5] = a, e, i, Omega, omega, M
__device__ __forceinline__ void elements_of(double mu, const double (&r)[3], const double (&v)[3], double (&el)[6]) {
  const double R = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  const double V2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
  const double rv = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
  const double h[3] = {r[1] * v[2] - r[2] * v[1], r[2] * v[0] - r[0] * v[2], r[0] * v[1] - r[1] * v[0]};
  const double H = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
  const double inv_a = 2.0 / R - V2 / mu;
  const double sma = 1.0 / inv_a;
  const double ev[3] = {(v[1] * h[2] - v[2] * h[1]) / mu - r[0] / R, (v[2] * h[0] - v[0] * h[2]) / mu - r[1] / R,
                        (v[0] * h[1] - v[1] * h[0]) / mu - r[2] / R};
  const double e = sqrt(ev[0] * ev[0] + ev[1] * ev[1] + ev[2] * ev[2]);
  const double nx = -h[1], ny = h[0];
  const double N = sqrt(nx * nx + ny * ny);
  const double inc = atan2(N, h[2]);
  const double Omega = (N == 0.0) ? 0.0 : wrap_2pi(atan2(ny, nx));
  double omega, M;
  if (e == 0.0) {
    omega = 0.0;
    M = wrap_2pi(in_plane_angle(r, h, H, nx, ny, N));
  } else {
    omega = wrap_2pi(in_plane_angle(ev, h, H, nx, ny, N));
    if (inv_a > 0.0) {
      const double ecosE = 1.0 - R / sma;
      const double esinE = rv / sqrt(mu * sma);
      M = wrap_2pi(atan2(esinE, ecosE) - esinE);
    } else {
      M = __longlong_as_double(0x7ff8000000000000LL);
    }
  }
  el[0] = sma; el[1] = e; el[2] = inc; el[3] = Omega; el[4] = omega; el[5] = M;
}

__global__ void __launch_bounds__(256) snapshot_kernel(SnapshotArgs a) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= a.n) return;
  const double r[3] = {a.fin[0][i], a.fin[1][i], a.fin[2][i]};
  const double v[3] = {a.fin[3][i], a.fin[4][i], a.fin[5][i]};
  a.out_flag[i] = a.fin_flag[i];
  a.out_rstep[i] = a.fin_rstep[i];
  if (a.kind == GLISSE_SNAPSHOT_CARTESIAN) {
    a.out[0][i] = r[0]; a.out[1][i] = r[1]; a.out[2][i] = r[2];
    a.out[3][i] = v[0]; a.out[4][i] = v[1]; a.out[5][i] = v[2];
    return;
  }
  double el[6];
  elements_of(a.mu, r, v, el);
#pragma unroll
  for (int k = 0; k < 6; ++k) a.out[k][i] = el[k];
}

// Resonant-argument reduction: phi = p lambda − q lambda_pl − (p − q) varpi with
// lambda = Omega + omega + M, varpi = Omega + omega, for every ACTIVE particle at the current step;
// seen0 / seen180 record whether phi has ever come within `window` of 0 or of pi ("librating
// particles [are] those with a resonant argument that never comes within 10 deg of 0 deg or never
// within 10 deg of 180 deg").  The planet's elements are about gm_star + gm_planet.
__global__ void __launch_bounds__(256) resonance_kernel(ResonanceArgs a) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= a.n || a.fin_flag[i] != 0) return;
  const double rp[3] = {a.planet_q[0], a.planet_q[1], a.planet_q[2]};
  const double vp[3] = {a.planet_qd[0], a.planet_qd[1], a.planet_qd[2]};
  double pl[6], el[6];
  elements_of(a.mu_planet, rp, vp, pl);
  const double r[3] = {a.fin[0][i], a.fin[1][i], a.fin[2][i]};
  const double v[3] = {a.fin[3][i], a.fin[4][i], a.fin[5][i]};
  elements_of(a.mu, r, v, el);
  const double varpi = el[3] + el[4];
  const double lambda = varpi + el[5];
  const double lambda_pl = pl[3] + pl[4] + pl[5];
  const double phi = wrap_2pi(a.p * lambda - a.q * lambda_pl - (a.p - a.q) * varpi);
  a.phi[i] = phi;
  const double d0 = fmin(phi, kTwoPiS - phi);          // angular distance to 0
  const double d180 = fabs(phi - 0.5 * kTwoPiS);       // angular distance to pi
  if (d0 < a.window) a.seen0[i] = 1;
  if (d180 < a.window) a.seen180[i] = 1;
}

}  // namespace

cudaError_t launch_snapshot(const SnapshotArgs& a, cudaStream_t s) {
  const int blocks = static_cast<int>((a.n + 255) / 256);
  snapshot_kernel<<<blocks, 256, 0, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_resonance(const ResonanceArgs& a, cudaStream_t s) {
  const int blocks = static_cast<int>((a.n + 255) / 256);
  resonance_kernel<<<blocks, 256, 0, s>>>(a);
  return cudaGetLastError();
}

}  // namespace glisse
