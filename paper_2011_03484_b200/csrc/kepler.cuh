// kepler.cuh — device-side Kepler drift (step a5 of DESIGN.md) shared by the
// particle kernel and the planet-history kernel.  CUDA path only.
//
// Kepler's equation in differenced form, x = E(t0+dt) − E(t0)  (reading S4):
//     dM = x − ec sin x + es (1 − cos x),   ec = e cos E0 = 1 − r0/a,   es = e sin E0 = r·v / sqrt(mu a)
// solved by Newton's method from the guess of reading S5, at most `iters` updates; a lane stops
// updating at its own convergence (|update| <= kExitEps) and the loop leaves when every live lane
// of the warp has converged (warp-uniform exit, reading S7) — so a lane's arithmetic never depends
// on its warp-mates and results are bit-identical under compaction / re-chunking.
// Then the Gauss f, g functions advance (r, v).
#pragma once
#include <cuda_runtime.h>

#include "sincos_coeffs.inc"

namespace glisse {

constexpr unsigned kFullMask = 0xffffffffu;
constexpr double kPiOver4 = 0.78539816339744830962;
constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr double kInvTwoPi = 0.15915494309189533576888376337251;
// A Newton update below this size means the next one would be < kExitEps^2 * e / (2 (1 − e)),
// i.e. below 1e-17 for every e <= 0.999: x is converged to roundoff.
constexpr double kExitEps = 1e-10;

// sin and cos for |x| <= pi/4 without range reduction (coefficients: gen_sincos_coeffs.py,
// max relative error 2e-17 before rounding).  13 DFMA + 3 DMUL.
__device__ __forceinline__ void sincos_small(double x, double& s, double& c) {
  const double t = x * x;
  double ps = fma(t, GL_S5, GL_S4);
  double pc = fma(t, GL_C5, GL_C4);
  ps = fma(t, ps, GL_S3);
  pc = fma(t, pc, GL_C3);
  ps = fma(t, ps, GL_S2);
  pc = fma(t, pc, GL_C2);
  ps = fma(t, ps, GL_S1);
  pc = fma(t, pc, GL_C1);
  ps = fma(t, ps, GL_S0);
  pc = fma(t, pc, GL_C0);
  const double x3 = t * x;
  const double t2 = t * t;
  s = fma(x3, ps, x);
  c = fma(t2, pc, fma(-0.5, t, 1.0));
}

// sin/cos for any x.  Must be called by all 32 lanes of the warp; `live` lanes with |x| > pi/4 take
// the library sincos (argument reduction), chosen per lane, skipped when no lane needs it.
__device__ __forceinline__ void sincos_warp(bool live, double x, double& s, double& c) {
  sincos_small(x, s, c);
  const bool big = live && !(fabs(x) <= kPiOver4);
  if (__any_sync(kFullMask, big)) {
    if (big) sincos(x, &s, &c);
  }
}

// Kepler drift of one body per lane.  All 32 lanes must call; `live` marks lanes whose body is to
// be advanced.  r2 = |r|^2 on entry.  Returns 0, GLISSE_FLAG_NONCONV (3) or GLISSE_FLAG_UNBOUND (4);
// on a non-zero return (or !live) the state is untouched.
__device__ __forceinline__ int kepler_drift_warp(bool live, double mu, double inv_mu, double dt, int iters,
                                                 double tol, double r2, double& x, double& y, double& z,
                                                 double& vx, double& vy, double& vz) {
  const double v2 = fma(vx, vx, fma(vy, vy, vz * vz));
  const double u = fma(x, vx, fma(y, vy, z * vz));
  const double rinv = rsqrt(r2);
  const double r0 = r2 * rinv;
  const double alpha = fma(2.0 * mu, rinv, -v2);  // mu / a
  const bool live_in = live;
  const bool unbound = !(alpha > 0.0);
  live = live && !unbound;
  const double al = live ? alpha : 1.0;  // keep dead lanes finite so they never trigger slow paths
  const double rsa = rsqrt(al);
  const double sqa = al * rsa;    // sqrt(alpha)
  const double inva = rsa * rsa;  // 1 / alpha
  const double q = r0 * al * inv_mu;  // r0 / a = 1 − ec
  const double ec = 1.0 - q;
  const double es = u * sqa * inv_mu;
  const double ndt = al * sqa * inv_mu * dt;  // n dt
  const double dM = fma(-rint(ndt * kInvTwoPi), kTwoPi, ndt);  // reading S9
  const double invq = mu * rinv * inva;                        // a / r0

  // initial guess (reading S5)
  const double x1 = dM * invq;
  const double e2 = fma(ec, ec, es * es);
  const double x1sq = x1 * x1;
  const bool simple = (fabs(es * x1) < 0.25 * q) && (e2 * x1sq * x1sq < 0.0625 * q * q);
  double xk = x1;
  if (__any_sync(kFullMask, live && !simple)) {
    const double yy = dM - es;
    double sy, cy;
    sincos_warp(live && !simple, yy, sy, cy);
    const double sg = fma(es, cy, ec * sy);
    const double e = sqrt(e2);
    if (!simple) xk = yy + (sg >= 0.0 ? 0.85 : -0.85) * e;
  }
  if (!live) xk = 0.0;

  // Newton updates, warp-uniform exit
  bool conv = !live;
  double s, c;
  for (int it = 0; it < iters; ++it) {
    sincos_warp(!conv, xk, s, c);
    const double f = fma(es, 1.0 - c, fma(-ec, s, xk)) - dM;
    const double fp = fma(es, s, fma(-ec, c, 1.0));
    const double d = f / fp;
    if (!conv) {
      xk -= d;
      conv = fabs(d) <= kExitEps;
    }
    if (__all_sync(kFullMask, conv)) break;
  }
  sincos_warp(live, xk, s, c);
  const double rho = fma(es, 1.0 - c, fma(-ec, s, xk)) - dM;  // residual of Kepler's equation
  const bool nonconv = !(fabs(rho) <= tol);

  // Gauss f, g (PAPER.md:94 step 4): applied as r += (f−1) r + g v, v += fdot r + (gdot−1) v
  const double p = fma(es, s, fma(-ec, c, 1.0));  // r(t)/a
  const double invp = 1.0 / p;
  const double cm1 = c - 1.0;
  const double fm1 = cm1 * invq;
  const double g = ((dM - xk) + s) * (mu * inva * rsa);  // / n
  const double fd = -(s * invp) * (sqa * rinv);
  const double gm1 = cm1 * invp;
  if (live && !nonconv) {
    const double nx = fma(fm1, x, fma(g, vx, x));
    const double ny = fma(fm1, y, fma(g, vy, y));
    const double nz = fma(fm1, z, fma(g, vz, z));
    vx = fma(fd, x, fma(gm1, vx, vx));
    vy = fma(fd, y, fma(gm1, vy, vy));
    vz = fma(fd, z, fma(gm1, vz, vz));
    x = nx; y = ny; z = nz;
  }
  if (!live_in) return 0;
  return unbound ? GLISSE_FLAG_UNBOUND : (nonconv ? GLISSE_FLAG_NONCONV : 0);
}

}  // namespace glisse
