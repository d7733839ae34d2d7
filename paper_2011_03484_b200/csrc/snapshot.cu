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
// Elements, written from Murray & Dermott, Solar System Dynamics, §2.8 ("the orbit in space", the
// inverse problem at its end): with R = |r|, the specific angular momentum h = r x v and R Rdot = r.v,
//   vis-viva:            1/a = 2/R - v^2/mu
//   conic equation:      e cos f = h^2/(mu R) - 1,   e sin f = h Rdot/mu      (f = true anomaly)
//   orientation of h:    tan I = |h_xy| / h_z,  sin Omega = h_x/|h_xy|,  cos Omega = -h_y/|h_xy|
//   argument of latitude sin(omega + f) = Z / (R sin I),  cos(omega + f) = (X cos Omega + Y sin Omega)/R
//   pericentre:          omega = (omega + f) - f
//   eccentric anomaly:   e cos E = 1 - R/a,  e sin E = R Rdot / sqrt(mu a);  M = E - e sin E.
// Conventions where an angle is undefined (include/glisse.h): orbit in the reference plane (h_xy = 0):
// Omega = 0 and omega + f is the longitude of r from x counted along the motion; e = 0: omega = 0 and
// M = omega + f; 1/a <= 0: M = NaN.  Angles in [0, 2 pi).
#include "glisse_internal.cuh"

namespace glisse {
namespace {

constexpr double kTau = 6.283185307179586476925286766559;
constexpr double kInvTau = 0.15915494309189533576888376337251;

// x mod 2 pi into [0, 2 pi)
__device__ __forceinline__ double to_turn(double x) {
  double y = fma(-kTau, floor(x * kInvTau), x);
  if (y >= kTau) y -= kTau;
  if (y < 0.0) y += kTau;
  return y;
}

struct Osculating {
  double a, e, inc, Omega, omega, M;
};

__device__ __forceinline__ Osculating osculating_elements(double mu, double X, double Y, double Z, double U, double V,
                                                          double W) {
  Osculating o;
  const double R = sqrt(X * X + Y * Y + Z * Z);
  const double speed2 = U * U + V * V + W * W;
  const double RRdot = X * U + Y * V + Z * W;
  const double hx = Y * W - Z * V, hy = Z * U - X * W, hz = X * V - Y * U;
  const double hxy2 = hx * hx + hy * hy;
  const double hh = hxy2 + hz * hz;
  const double hxy = sqrt(hxy2), h = sqrt(hh);
  const double one_over_a = 2.0 / R - speed2 / mu;
  o.a = 1.0 / one_over_a;
  const double ecosf = hh / (mu * R) - 1.0;
  const double esinf = h * RRdot / (mu * R);
  o.e = sqrt(ecosf * ecosf + esinf * esinf);
  o.inc = atan2(hxy, hz);
  double lat;  // omega + f
  if (hxy > 0.0) {
    const double sinO = hx / hxy, cosO = -hy / hxy;
    o.Omega = to_turn(atan2(hx, -hy));
    lat = atan2(Z * (h / hxy), X * cosO + Y * sinO);
  } else {
    o.Omega = 0.0;
    lat = atan2(hz < 0.0 ? -Y : Y, X);
  }
  if (o.e == 0.0) {
    o.omega = 0.0;
    o.M = to_turn(lat);
  } else {
    o.omega = to_turn(lat - atan2(esinf, ecosf));
    if (one_over_a > 0.0) {
      const double esinE = RRdot / sqrt(mu * o.a);
      const double ecosE = 1.0 - R * one_over_a;
      o.M = to_turn(atan2(esinE, ecosE) - esinE);
    } else {
      o.M = __longlong_as_double(0x7ff8000000000000LL);
    }
  }
  return o;
}

// The sample pass: snapshot staging and / or resonant-argument reduction of one instant.
//
// Resonant argument: phi = p lambda - q lambda_pl - (p - q) varpi with
// lambda = Omega + omega + M, varpi = Omega + omega, for every ACTIVE particle; the planet's elements
// are about gm_star + gm_planet.  Libration test: seen0 / seen180 record whether phi
// has ever come within `window` of 0 or of pi.  Amplitude ("successive maxima and minima
// of the resonant angle and ... the difference between them"): turning points of the sampled phi in
// [0, 2 pi), each after the first giving one amplitude sample |ext - previous ext| / 2
// (include/glisse.h: glisse_libration_read).
__global__ void __launch_bounds__(256) sample_kernel(SampleArgs a) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= a.n) return;
  if (i == 0 && a.step_out != nullptr) *a.step_out = a.step;
  const double X = a.fin[0][i], Y = a.fin[1][i], Z = a.fin[2][i];
  const double U = a.fin[3][i], V = a.fin[4][i], W = a.fin[5][i];
  const int fl = a.fin_flag[i];
  const bool want_phi = a.do_resonance && fl == 0;
  const bool want_el = (a.do_snapshot && a.kind == GLISSE_SNAPSHOT_ELEMENTS) || want_phi;
  Osculating o{};
  if (want_el) o = osculating_elements(a.mu, X, Y, Z, U, V, W);
  if (a.do_snapshot) {
    a.out_flag[i] = fl;
    a.out_rstep[i] = a.fin_rstep[i];
    if (a.kind == GLISSE_SNAPSHOT_CARTESIAN) {
      a.out[0][i] = X; a.out[1][i] = Y; a.out[2][i] = Z;
      a.out[3][i] = U; a.out[4][i] = V; a.out[5][i] = W;
    } else {
      a.out[0][i] = o.a; a.out[1][i] = o.e; a.out[2][i] = o.inc;
      a.out[3][i] = o.Omega; a.out[4][i] = o.omega; a.out[5][i] = o.M;
    }
  }
  if (!want_phi) return;
  const Osculating pl = osculating_elements(a.mu_planet, a.planet_q[0], a.planet_q[1], a.planet_q[2], a.planet_qd[0],
                                            a.planet_qd[1], a.planet_qd[2]);
  const double varpi = o.Omega + o.omega;
  const double lambda = varpi + o.M;
  const double lambda_pl = pl.Omega + pl.omega + pl.M;
  const double phi = to_turn(a.p * lambda - a.q * lambda_pl - (a.p - a.q) * varpi);
  const LibrationRecord& L = a.lib;
  // the window test
  if (fmin(phi, kTau - phi) < a.window) L.seen0[i] = 1;
  if (fabs(phi - 0.5 * kTau) < a.window) L.seen180[i] = 1;
  // running extrema
  L.phi_min[i] = fmin(L.phi_min[i], phi);
  L.phi_max[i] = fmax(L.phi_max[i], phi);
  // turning points
  const int seen = L.n_seen[i];
  if (seen > 0) {
    const double prev = L.phi[i];
    const int trend = L.trend[i];
    const int now = phi > prev ? 1 : (phi < prev ? -1 : trend);
    if (trend != 0 && now == -trend) {  // the previous sample was a maximum (trend +1) or a minimum (-1)
      if (L.ext_kind[i] != 0) {
        const double amp = 0.5 * fabs(prev - L.ext_last[i]);
        L.amp_sum[i] += amp;
        L.amp_max[i] = fmax(L.amp_max[i], amp);
        L.n_amp[i] += 1;
      }
      L.ext_last[i] = prev;
      L.ext_kind[i] = static_cast<signed char>(trend);
    }
    L.trend[i] = static_cast<signed char>(now);
  }
  L.phi[i] = phi;
  L.n_seen[i] = seen + 1;
}

__global__ void __launch_bounds__(256) libration_reset_kernel(LibrationRecord L, long long n) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n) return;
  L.phi[i] = 0.0;
  L.seen0[i] = 0; L.seen180[i] = 0;
  L.phi_min[i] = __longlong_as_double(0x7ff0000000000000LL);   // +inf
  L.phi_max[i] = __longlong_as_double(0xfff0000000000000LL);   // -inf
  L.ext_last[i] = 0.0; L.amp_sum[i] = 0.0; L.amp_max[i] = 0.0;
  L.n_amp[i] = 0; L.n_seen[i] = 0;
  L.trend[i] = 0; L.ext_kind[i] = 0;
}

__global__ void __launch_bounds__(256) libration_mean_kernel(LibrationRecord L, double* amp_mean, long long n) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int k = L.n_amp[i];
  amp_mean[i] = k > 0 ? L.amp_sum[i] / k : __longlong_as_double(0x7ff8000000000000LL);
}

}  // namespace

cudaError_t launch_sample(const SampleArgs& a, cudaStream_t s) {
  const int blocks = static_cast<int>((a.n + 255) / 256);
  sample_kernel<<<blocks, 256, 0, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_libration_reset(const LibrationRecord& lib, long long n, cudaStream_t s) {
  libration_reset_kernel<<<static_cast<int>((n + 255) / 256), 256, 0, s>>>(lib, n);
  return cudaGetLastError();
}

cudaError_t launch_libration_mean(const LibrationRecord& lib, double* amp_mean, long long n, cudaStream_t s) {
  libration_mean_kernel<<<static_cast<int>((n + 255) / 256), 256, 0, s>>>(lib, amp_mean, n);
  return cudaGetLastError();
}

}  // namespace glisse
