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

// sm, cm1 for any x, P bodies per lane.  Must be called by all 32 lanes; `live` bodies whose |x| > pi/4
// take the library sincos (full argument reduction), chosen per body, skipped when no lane needs it.
template <int P>
__device__ __forceinline__ void sincosm_warp(const bool (&live)[P], const double (&x)[P], double (&sm)[P],
                                             double (&cm1)[P]) {
  bool big[P];
  bool any_big = false;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    sincosm_small(x[p], sm[p], cm1[p]);
    big[p] = live[p] && !is_small_angle(x[p]);
    any_big = any_big || big[p];
  }
  if (__any_sync(kFullMask, any_big)) {
#pragma unroll
    for (int p = 0; p < P; ++p) {
      if (big[p]) {
        double s, c;
        sincos(x[p], &s, &c);
        sm[p] = s - x[p];
        cm1[p] = c - 1.0;
      }
    }
  }
}

// Kepler drift of P bodies per lane about a point mass mu for time dt.  The P bodies of a lane are
// independent instruction streams that the compiler interleaves: the drift of one body is a serial
// chain of dependent FP64 operations (8 cycles each on sm_100), so P = 2 doubles the work in flight
// per warp and halves the per-body share of every warp-wide vote, branch and constant load.
// All 32 lanes must call; `live[p]` marks bodies to be advanced.  r2 = |r|^2 on entry; inv_mu = 1/mu
// and inv_mu_dt = dt/mu are constants of the run.  st[p] returns 0, GLISSE_FLAG_NONCONV (3) or
// GLISSE_FLAG_UNBOUND (4); on a non-zero status, or for !live bodies, the state is untouched.
// A body's arithmetic never depends on the other bodies of its lane or warp.
template <int P>
__device__ __forceinline__ void kepler_drift_warp(const bool (&live_in)[P], double mu, double inv_mu,
                                                  double inv_mu_dt, int iters, double tol, const double (&r2)[P],
                                                  double (&x)[P], double (&y)[P], double (&z)[P], double (&vx)[P],
                                                  double (&vy)[P], double (&vz)[P], int (&st)[P]) {
  bool live[P], unbound[P], simple[P], rough[P];
  double rinv[P], sqa[P], rsa[P], q[P], ec[P], es[P], dM[P], a[P], invq[P], e2[P], xk[P];
  bool any_rough = false;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    const double v2 = fma(vx[p], vx[p], fma(vy[p], vy[p], vz[p] * vz[p]));
    const double u = fma(x[p], vx[p], fma(y[p], vy[p], z[p] * vz[p]));
    rinv[p] = rsqrt_f64(r2[p]);
    const double r0 = r2[p] * rinv[p];
    const double alpha = fma(2.0 * mu, rinv[p], -v2);  // mu / a
    unbound[p] = !(alpha > 0.0);
    live[p] = live_in[p] && !unbound[p];
    const double al = live[p] ? alpha : 1.0;  // dead bodies stay finite so they never trigger slow paths
    rsa[p] = rsqrt_f64(al);
    sqa[p] = al * rsa[p];                    // sqrt(alpha) = n a
    const double inva = rsa[p] * rsa[p];     // 1 / alpha
    q[p] = r0 * (al * inv_mu);               // r0 / a = 1 − ec
    ec[p] = 1.0 - q[p];
    es[p] = u * (sqa[p] * inv_mu);
    const double ndt = (al * sqa[p]) * inv_mu_dt;                   // n dt
    dM[p] = fma(-rint(ndt * kInvTwoPi), kTwoPi, ndt);               // reading S9
    a[p] = mu * inva;
    invq[p] = a[p] * rinv[p];  // a / r0

    // initial guess (reading S5): x1 = dM/q if |es| |x1| < q/4 and e x1^2 < q/4, compared squared
    const double x1 = dM[p] * invq[p];
    e2[p] = fma(ec[p], ec[p], es[p] * es[p]);
    const double t1 = x1 * x1;
    const double q16 = (0.25 * q[p]) * (0.25 * q[p]);
    simple[p] = ((es[p] * es[p]) * t1 < q16) && ((e2[p] * t1) * t1 < q16);
    xk[p] = x1;
    rough[p] = live[p] && !simple[p];
    any_rough = any_rough || rough[p];
  }
  if (__any_sync(kFullMask, any_rough)) {
    double yy[P], sy[P], cy[P];
#pragma unroll
    for (int p = 0; p < P; ++p) yy[p] = dM[p] - es[p];
    sincosm_warp<P>(rough, yy, sy, cy);
#pragma unroll
    for (int p = 0; p < P; ++p) {
      const double sg = fma(es[p], 1.0 + cy[p], ec[p] * (yy[p] + sy[p]));
      const double e = sqrt(e2[p]);
      if (!simple[p]) xk[p] = yy[p] + (sg >= 0.0 ? 0.85 : -0.85) * e;
    }
  }

  // Newton updates, warp-uniform exit.  After a body's last update d (|d| <= eps)
  // its sin/cos at x − d follow from those at x by angle addition instead of a fresh evaluation.
  bool conv[P], open[P];
  double sm[P], cm1[P];  // sin x − x, cos x − 1 at the current xk
#pragma unroll
  for (int p = 0; p < P; ++p) {
    if (!live[p]) xk[p] = 0.0;
    conv[p] = !live[p];
    sm[p] = 0.0;
    cm1[p] = 0.0;
  }
  for (int it = 0; it < iters; ++it) {
    double smk[P], cmk[P];
#pragma unroll
    for (int p = 0; p < P; ++p) open[p] = !conv[p];
    sincosm_warp<P>(open, xk, smk, cmk);
    bool all_conv = true;
#pragma unroll
    for (int p = 0; p < P; ++p) {
      const double s = xk[p] + smk[p];
      const double f = fma(-es[p], cmk[p], fma(-ec[p], s, xk[p] - dM[p]));
      const double fp = fma(es[p], s, fma(-ec[p], cmk[p], q[p]));
      const double d = f * rcp_f64_1(fp);
      if (!conv[p]) {
        conv[p] = fabs(d) <= kExitEps;
        // sin(x − d) − (x − d), cos(x − d) − 1 to O(d^3); exact enough only once |d| <= eps
        const double c = 1.0 + cmk[p];
        const double hd = 0.5 * d;
        sm[p] = fma(-d, fma(hd, s, cmk[p]), smk[p]);
        cm1[p] = fma(d, fma(-hd, c, s), cmk[p]);
        xk[p] -= d;
      }
      all_conv = all_conv && conv[p];
    }
    if (__all_sync(kFullMask, all_conv)) break;
  }
  // bodies that ran out of updates (or iters == 0) need a fresh evaluation at the final x
  bool any_open = false;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    open[p] = !conv[p];
    any_open = any_open || open[p];
  }
  if (__any_sync(kFullMask, any_open)) {
    double smk[P], cmk[P];
    sincosm_warp<P>(open, xk, smk, cmk);
#pragma unroll
    for (int p = 0; p < P; ++p)
      if (open[p]) { sm[p] = smk[p]; cm1[p] = cmk[p]; }
  }
#pragma unroll
  for (int p = 0; p < P; ++p) {
    const double s = xk[p] + sm[p];
    const double rho = fma(-es[p], cm1[p], fma(-ec[p], s, xk[p] - dM[p]));  // residual of Kepler's equation
    const bool nonconv = !(fabs(rho) <= tol);

    // Gauss f, g (PAPER.md:94 step 4), applied as r += (f−1) r + g v, v += fdot r + (gdot−1) v
    const double pr = fma(es[p], s, fma(-ec[p], cm1[p], q[p]));  // r(t)/a
    const double invp = rcp_f64(pr);
    const double fm1 = cm1[p] * invq[p];
    const double g = (dM[p] + sm[p]) * (a[p] * rsa[p]);  // (dM − x + sin x) / n
    const double fd = -(s * invp) * (sqa[p] * rinv[p]);
    const double gm1 = cm1[p] * invp;
    if (live[p] && !nonconv) {
      const double nx = fma(fm1, x[p], fma(g, vx[p], x[p]));
      const double ny = fma(fm1, y[p], fma(g, vy[p], y[p]));
      const double nz = fma(fm1, z[p], fma(g, vz[p], z[p]));
      vx[p] = fma(fd, x[p], fma(gm1, vx[p], vx[p]));
      vy[p] = fma(fd, y[p], fma(gm1, vy[p], vy[p]));
      vz[p] = fma(fd, z[p], fma(gm1, vz[p], vz[p]));
      x[p] = nx; y[p] = ny; z[p] = nz;
    }
    st[p] = !live_in[p] ? 0 : (unbound[p] ? GLISSE_FLAG_UNBOUND : (nonconv ? GLISSE_FLAG_NONCONV : 0));
  }
}

// One body per lane (the planet-history kernel and the primitive test hook).
__device__ __forceinline__ int kepler_drift_warp(bool live, double mu, double inv_mu, double inv_mu_dt, int iters,
                                                 double tol, double r2, double& x, double& y, double& z,
                                                 double& vx, double& vy, double& vz) {
  const bool l1[1] = {live};
  const double r21[1] = {r2};
  double x1[1] = {x}, y1[1] = {y}, z1[1] = {z}, vx1[1] = {vx}, vy1[1] = {vy}, vz1[1] = {vz};
  int st[1];
  kepler_drift_warp<1>(l1, mu, inv_mu, inv_mu_dt, iters, tol, r21, x1, y1, z1, vx1, vy1, vz1, st);
  x = x1[0]; y = y1[0]; z = z1[0]; vx = vx1[0]; vy = vy1[0]; vz = vz1[0];
  return st[0];
}

// single-body sin x − x, cos x − 1 (test hook)
__device__ __forceinline__ void sincosm_warp(bool live, double x, double& sm, double& cm1) {
  const bool l1[1] = {live};
  const double x1[1] = {x};
  double s1[1], c1[1];
  sincosm_warp<1>(l1, x1, s1, c1);
  sm = s1[0];
  cm1 = c1[0];
}

}  // namespace glisse
