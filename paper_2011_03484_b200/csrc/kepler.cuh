// kepler.cuh — device-side fp64 primitives and the Kepler drift (step a5 of DESIGN.md;
// PAPER.md:92-101, 123) shared by the particle kernel and the planet-history kernel.
// CUDA path only: nothing here is used by, or derived from, oracle/.
//
// Kepler's equation in differenced form, x = E(t0+dt) − E(t0)  (reading S4):
//     dM = x − ec sin x + es (1 − cos x),   ec = e cos E0 = 1 − r0/a,   es = e sin E0 = r·v / sqrt(mu a)
// solved by Newton's method from the guess of reading S5, at most `iters` updates.  A lane stops
// updating at its own convergence (|update| <= kExitEps) and the loop leaves when every live lane
// of the warp has converged (warp-uniform exit, reading S7) — a lane's arithmetic never depends
// on its warp-mates, so results are bit-identical under compaction and re-chunking.
// Then the Gauss f, g functions advance (r, v).
//
// The FP64 pipe is the roofline of the whole path, so every primitive here is
// written to a counted number of FP64-pipe instructions:
//   rsqrt_f64   MUFU.RSQ64H seed + one cubic step          (2 DMUL + 3 DFMA)
//   rcp_f64     MUFU.RCP64H seed + two quadratic steps     (4 DFMA)
//   rcp_f64_1   MUFU.RCP64H seed + one quadratic step      (2 DFMA; 2^-39, Newton updates only)
//   sincosm     sin x − x and cos x − 1 on |x| <= pi/4     (4 DMUL + 12 DFMA), no range reduction
#pragma once
#include <cuda_runtime.h>

#include "../../include/glisse.h"
#include "sincos_coeffs.inc"

namespace glisse {

constexpr unsigned kFullMask = 0xffffffffu;
constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr double kInvTwoPi = 0.15915494309189533576888376337251;
// A Newton update below this size means the next one would be < kExitEps^2 e / (2 (1 − e)), i.e.
// below 1e-15 |x| ulp level for every e <= 0.999: x is converged to roundoff, and sin/cos of the
// updated x follow from the angle-addition formulae truncated after the d^2 terms (error d^3/6).
constexpr double kExitEps = 1e-9;

// ---- seeds from the special-function unit (upper 32 bits of the operand, ~2^-20 relative) --------
__device__ __forceinline__ double mufu_rsq(double a) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
  return y;
}
__device__ __forceinline__ double mufu_rcp(double a) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
  return y;
}

// 1/sqrt(a) for normal positive a.  Seed error e0 <= 2^-19.9; the cubic step leaves (5/16) e0^3.
__device__ __forceinline__ double rsqrt_f64(double a) {
  const double y = mufu_rsq(a);
  const double t = a * y;
  const double e = fma(-t, y, 1.0);  // 1 − a y^2
  const double p = fma(0.375, e, 0.5);
  const double ye = y * e;
  return fma(ye, p, y);  // y (1 + e/2 + 3 e^2/8)
}

// 1/a for normal a, full precision (two Newton steps: 2^-39.8 -> 2^-79).
__device__ __forceinline__ double rcp_f64(double a) {
  double y = mufu_rcp(a);
  double e = fma(-a, y, 1.0);
  y = fma(y, e, y);
  e = fma(-a, y, 1.0);
  return fma(y, e, y);
}

// 1/a to 2^-39 (one Newton step).  Only for the Newton update of Kepler's equation, where a
// relative error of 2^-39 in the update leaves the quadratic convergence untouched.
__device__ __forceinline__ double rcp_f64_1(double a) {
  const double y = mufu_rcp(a);
  const double e = fma(-a, y, 1.0);
  return fma(y, e, y);
}

// The polynomial coefficients live in the constant bank so that every DFMA of the Horner chains takes
// its coefficient as a c[3][..] operand: as 64-bit immediates they cost two UMOV each per use, which
// competes with the FP64 pipe for issue slots (profiles/r01: 54 UMOV per particle-step).
static __constant__ double kSinCoef[6] = {GL_S0, GL_S1, GL_S2, GL_S3, GL_S4, GL_S5};
static __constant__ double kCosCoef[6] = {GL_C0, GL_C1, GL_C2, GL_C3, GL_C4, GL_C5};

__device__ __forceinline__ int hi_word(double x) { return __double2hiint(x); }

// |x| <= pi/4, decided on the high word (integer pipe, not the FP64 pipe).  NaN/Inf -> false.
__device__ __forceinline__ bool is_small_angle(double x) {
  return (hi_word(x) & 0x7fffffff) < 0x3fe921fb;  // high word of pi/4 = 0x3fe921fb54442d18
}

// sm = sin x − x and cm1 = cos x − 1 for |x| <= pi/4 (coefficients: gen_sincos_coeffs.py, max
// relative error 2e-17 before rounding).  Returning the differences keeps full relative accuracy
// in the two places the drift needs them: g ~ dM − x + sin x and f − 1 ~ cos x − 1.
__device__ __forceinline__ void sincosm_small(double x, double& sm, double& cm1) {
  const double t = x * x;
  double ps = fma(t, kSinCoef[5], kSinCoef[4]);
  double pc = fma(t, kCosCoef[5], kCosCoef[4]);
  ps = fma(t, ps, kSinCoef[3]);
  pc = fma(t, pc, kCosCoef[3]);
  ps = fma(t, ps, kSinCoef[2]);
  pc = fma(t, pc, kCosCoef[2]);
  ps = fma(t, ps, kSinCoef[1]);
  pc = fma(t, pc, kCosCoef[1]);
  ps = fma(t, ps, kSinCoef[0]);
  pc = fma(t, pc, kCosCoef[0]);
  const double x3 = t * x;
  const double t2 = t * t;
  const double mh = -0.5 * t;
  sm = x3 * ps;
  cm1 = fma(t2, pc, mh);
}

// sm, cm1 for any x.  Must be called by all 32 lanes; `live` lanes whose |x| > pi/4 take the
// library sincos (full argument reduction), chosen per lane, skipped when no lane needs it.
__device__ __forceinline__ void sincosm_warp(bool live, double x, double& sm, double& cm1) {
  sincosm_small(x, sm, cm1);
  const bool big = live && !is_small_angle(x);
  if (__any_sync(kFullMask, big)) {
    if (big) {
      double s, c;
      sincos(x, &s, &c);
      sm = s - x;
      cm1 = c - 1.0;
    }
  }
}

// Kepler drift of one body per lane about a point mass mu for time dt.  All 32 lanes must call;
// `live` marks lanes whose body is to be advanced.  r2 = |r|^2 on entry; inv_mu = 1/mu and
// inv_mu_dt = dt/mu are passed in because they are constants of the run.  Returns 0,
// GLISSE_FLAG_NONCONV (3) or GLISSE_FLAG_UNBOUND (4); on a non-zero return, or for !live lanes,
// the state is untouched.
__device__ __forceinline__ int kepler_drift_warp(bool live, double mu, double inv_mu, double inv_mu_dt,
                                                 int iters, double tol, double r2, double& x, double& y,
                                                 double& z, double& vx, double& vy, double& vz) {
  const double v2 = fma(vx, vx, fma(vy, vy, vz * vz));
  const double u = fma(x, vx, fma(y, vy, z * vz));
  const double rinv = rsqrt_f64(r2);
  const double r0 = r2 * rinv;
  const double alpha = fma(2.0 * mu, rinv, -v2);  // mu / a
  const bool live_in = live;
  const bool unbound = !(alpha > 0.0);
  live = live && !unbound;
  const double al = live ? alpha : 1.0;  // dead lanes stay finite so they never trigger slow paths
  const double rsa = rsqrt_f64(al);
  const double sqa = al * rsa;        // sqrt(alpha) = n a
  const double inva = rsa * rsa;      // 1 / alpha
  const double q = r0 * (al * inv_mu);  // r0 / a = 1 − ec
  const double ec = 1.0 - q;
  const double es = u * (sqa * inv_mu);
  const double ndt = (al * sqa) * inv_mu_dt;                   // n dt
  const double dM = fma(-rint(ndt * kInvTwoPi), kTwoPi, ndt);  // reading S9
  const double a = mu * inva;
  const double invq = a * rinv;  // a / r0

  // initial guess (reading S5): x1 = dM/q if |es| |x1| < q/4 and e x1^2 < q/4, compared squared
  const double x1 = dM * invq;
  const double e2 = fma(ec, ec, es * es);
  const double t1 = x1 * x1;
  const double q16 = (0.25 * q) * (0.25 * q);
  const bool simple = ((es * es) * t1 < q16) && ((e2 * t1) * t1 < q16);
  double xk = x1;
  if (__any_sync(kFullMask, live && !simple)) {
    const double yy = dM - es;
    double sy, cy;
    sincosm_warp(live && !simple, yy, sy, cy);
    const double sg = fma(es, 1.0 + cy, ec * (yy + sy));
    const double e = sqrt(e2);
    if (!simple) xk = yy + (sg >= 0.0 ? 0.85 : -0.85) * e;
  }
  if (!live) xk = 0.0;

  // Newton updates, warp-uniform exit.  After a lane's last update d (|d| <= eps)
  // its sin/cos at x − d follow from those at x by angle addition instead of a fresh evaluation.
  bool conv = !live;
  double sm = 0.0, cm1 = 0.0;  // sin x − x, cos x − 1 at the current xk
  for (int it = 0; it < iters; ++it) {
    double smk, cmk;
    sincosm_warp(!conv, xk, smk, cmk);
    const double s = xk + smk;
    const double f = fma(-es, cmk, fma(-ec, s, xk - dM));
    const double fp = fma(es, s, fma(-ec, cmk, q));
    const double d = f * rcp_f64_1(fp);
    if (!conv) {
      conv = fabs(d) <= kExitEps;
      // sin(x − d) − (x − d), cos(x − d) − 1 to O(d^3); exact enough only once |d| <= eps
      const double c = 1.0 + cmk;
      const double hd = 0.5 * d;
      sm = fma(-d, fma(hd, s, cmk), smk);
      cm1 = fma(d, fma(-hd, c, s), cmk);
      xk -= d;
    }
    if (__all_sync(kFullMask, conv)) break;
  }
  // lanes that ran out of updates (or iters == 0) need a fresh evaluation at the final x
  if (__any_sync(kFullMask, !conv)) {
    double smk, cmk;
    sincosm_warp(!conv, xk, smk, cmk);
    if (!conv) { sm = smk; cm1 = cmk; }
  }
  const double s = xk + sm;
  const double rho = fma(-es, cm1, fma(-ec, s, xk - dM));  // residual of Kepler's equation
  const bool nonconv = !(fabs(rho) <= tol);

  // Gauss f, g (PAPER.md:94 step 4), applied as r += (f−1) r + g v, v += fdot r + (gdot−1) v
  const double p = fma(es, s, fma(-ec, cm1, q));  // r(t)/a
  const double invp = rcp_f64(p);
  const double fm1 = cm1 * invq;
  const double g = (dM + sm) * (a * rsa);  // (dM − x + sin x) / n
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
