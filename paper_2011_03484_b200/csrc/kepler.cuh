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
//   sincosm     sin x − x and cos x − 1 on |x| <= pi/4     (4 DMUL + 11 DFMA), no range reduction
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

// gm / d^3 from d2 = d^2 (the kick's weight), seed y ~ d2^(-1/2):
//   gm y^3 (1 − e)^(-3/2),  e = 1 − d2 y^2,  (1 − e)^(-3/2) = 1 + (3/2) e + (15/8) e^2 + O(e^3)
// |e| <= 2^-18.9 leaves (35/16) e^3 < 2e-17.  4 DMUL + 3 DFMA, one less than rsqrt_f64 and a cube.
__device__ __forceinline__ double gm_over_r3(double gm, double d2) {
  const double y = mufu_rsq(d2);
  const double y2 = y * y;
  const double e = fma(-d2, y2, 1.0);
  const double y3 = (gm * y) * y2;
  const double p = fma(1.875, e, 1.5);
  return fma(y3, p * e, y3);
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
#ifdef GL_SINCOS_IMM
constexpr double kSinCoef[6] = {GL_S0, GL_S1, GL_S2, GL_S3, GL_S4, GL_S5};
constexpr double kCosCoef[6] = {GL_C0, GL_C1, GL_C2, GL_C3, GL_C4, GL_C5};
#else
static __constant__ double kSinCoef[6] = {GL_S0, GL_S1, GL_S2, GL_S3, GL_S4, GL_S5};
static __constant__ double kCosCoef[6] = {GL_C0, GL_C1, GL_C2, GL_C3, GL_C4, GL_C5};
#endif

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
  sm = x3 * ps;
  cm1 = t * fma(t, pc, -0.5);
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

// single-body sin x − x, cos x − 1 (test hook)
__device__ __forceinline__ void sincosm_warp(bool live, double x, double& sm, double& cm1) {
  const bool l1[1] = {live};
  const double x1[1] = {x};
  double s1[1], c1[1];
  sincosm_warp<1>(l1, x1, s1, c1);
  sm = s1[0];
  cm1 = c1[0];
}


// ---- the definition's solver (O2), one body per lane: guess of reading S5, at most `iters`
// Newton updates with a per-lane stop at |update| <= kExitEps and a warp-uniform exit (reading S7),
// residual test against `tol`.  Serves the bodies the fast solver below does not accept (e >= 0.8,
// |x| > pi/4, iters < 5, or no convergence in kFastMaxIters quartic steps), so that the
// non-convergence flag is decided exactly as the definition decides it.  Kept out of
// line: it is off the hot path and must not cost the particle kernel registers.
struct ExactSolve {
  double x, sm, cm1;  // x, sin x − x, cos x − 1 at the final x
  int nonconv;
};

static __device__ __noinline__ ExactSolve kepler_solve_exact(bool live, double ec, double es, double q, double dM,
                                                      double invq, double e2, int iters, double tol) {
  // initial guess (reading S5): x1 = dM/q if |es| |x1| < q/4 and e x1^2 < q/4, compared squared
  const double x1 = dM * invq;
  const double t1 = x1 * x1;
  const double q16 = (0.25 * q) * (0.25 * q);
  const bool simple = ((es * es) * t1 < q16) && ((e2 * t1) * t1 < q16);
  double xk = x1;
  const bool rough = live && !simple;
  if (__any_sync(kFullMask, rough)) {
    const double yy = dM - es;
    double sy, cy;
    sincosm_warp(rough, yy, sy, cy);
    const double sg = fma(es, 1.0 + cy, ec * (yy + sy));
    const double e = sqrt(e2);
    if (!simple) xk = yy + (sg >= 0.0 ? 0.85 : -0.85) * e;
  }
  if (!live) xk = 0.0;
  bool conv = !live;
  double sm = 0.0, cm1 = 0.0;
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
  // bodies that ran out of updates (or iters == 0) need a fresh evaluation at the final x
  if (__any_sync(kFullMask, !conv)) {
    double smk, cmk;
    sincosm_warp(!conv, xk, smk, cmk);
    if (!conv) { sm = smk; cm1 = cmk; }
  }
  const double s = xk + sm;
  const double rho = fma(-es, cm1, fma(-ec, s, xk - dM));  // residual of Kepler's equation
  ExactSolve o;
  o.x = xk; o.sm = sm; o.cm1 = cm1;
  o.nonconv = !(fabs(rho) <= tol) ? 1 : 0;
  return o;
}

// ---- fast solver -------------------------------------------------------------------------------------
// From x0 = dM/q, steps of quartic convergence: with f and its derivatives f1, f2, f3 at x (all from
// one sin/cos evaluation: f3 = 1 − f1) and delta = f/f1, the root of the cubic Taylor model is
//     d = delta (1 + a2 delta + (2 a2^2 − a3) delta^2),   a2 = f2/(2 f1),  a3 = f3/(6 f1),
// leaving an error (5 a2^3 − 5 a2 a3 + a4) delta^4.  A body is converged once |delta| is below a
// bound chosen from its eccentricity so that this error is < 2e-17 (a_k <= e/(k! (1 − e))):
//     e < 0.1: 1e-4     e < 0.3: 9e-5     e < 0.5: 5.5e-5     e < 0.8: 2e-5
// and sin, cos at x − d then follow from those at x by angle addition carried to d^3 (the d^4 terms
// are < 5e-18).  One step suffices wherever e x^2 / 2 is below the bound — every particle of
// BASELINE.json configs 1-4 — against the two Newton updates plus test the definition needs there.
// Kepler's equation has one root (f1 >= 1 − e > 0), so both solvers return the same x to roundoff.
// Thresholds and range tests are taken on the high words (integer pipe): the FP64 pipe is the
// roofline.
// Refined starting point.  x0 = dM/q is the first term of the reversion of
//     q x + (es/2) x^2 + (ec/6) x^3 + ... = dM,
// and the Newton update it leaves is ~ es x0^2 / (2 q): too large for one quartic step once e x0^2
// reaches ~1e-4 (planet-crossing orbits at small a, config 5; Jupiter itself at dt = 180 d).  Those
// bodies start instead from the reversion carried to third order,
//     x = y - b2 y^2 + (2 b2^2 - b3) y^3,   y = dM/q,  b2 = es/(2q),  b3 = ec/(6q)      (9 FP64 operations)
// whose error is O(y^4) (~1e-5 at y = 0.3), so that ONE quartic step is accepted where two were needed.
// Which bodies take it is decided per body from its own numbers (so a body's arithmetic still never
// depends on its warp-mates), in the integer pipe: log2(e^2)/4 + log2|y| = log2(sqrt(e) |y|) read off the
// high words (piecewise-linear in the mantissa, good to 0.15 in log2) against log2(sqrt(6e-5)) = -7.0.
// It is a compile-time variant of the drift (template REFINE): in the kernels of quiet workloads even a
// never-taken branch around these nine operations cost 4 % (measured), so they do not contain it; the
// instantiation is chosen per simulation (include/glisse.h: guess_order), never per launch.
constexpr int kRefineLevel = static_cast<int>((1023.0 * 1.25 - 7.0) * 1048576.0);
__device__ __forceinline__ bool wants_refined_guess(int e2_hi, int x_hi_abs) {
  return (e2_hi >> 2) + x_hi_abs > kRefineLevel;
}

constexpr int kFastMinIters = 5;   // the paper's count; below it the definition may not converge
constexpr int kFastMaxIters = 4;
// The fast solver does not evaluate the residual: what it accepts has a residual below 2e-17 plus the
// rounding of the residual's own evaluation (<= 2e-15 for |dM| <= pi).  A caller whose kepler_tol is
// below that floor is asking the definition's residual test to decide on roundoff, so every body then
// goes through the definition's solver, which does evaluate it.
constexpr double kFastMinTol = 4e-15;

__device__ __forceinline__ int hi_abs(double x) { return hi_word(x) & 0x7fffffff; }

// high words of the constants above (any bound below the stated value is safe)
constexpr int kHiE2_010 = 0x3f847ae1;   // 0.01   = 0x3f847ae147ae147b
constexpr int kHiE2_030 = 0x3fb70a3d;   // 0.09   = 0x3fb70a3d70a3d70a
constexpr int kHiE2_050 = 0x3fd00000;   // 0.25
constexpr int kHiE2_080 = 0x3fe47ae1;   // 0.64   = 0x3fe47ae147ae147b
constexpr int kHiThr0 = 0x3f1a36e2;     // 1e-4   = 0x3f1a36e2eb1c432d
constexpr int kHiThr1 = 0x3f1797cc;     // 9e-5   = 0x3f1797cc39ffd60f
constexpr int kHiThr2 = 0x3f0cd5f9;     // 5.5e-5 = 0x3f0cd5f99c38b04b
constexpr int kHiThr3 = 0x3ef4f8b5;     // 2e-5   = 0x3ef4f8b588e368f1

// Kepler drift of P bodies per lane about a point mass mu for time dt.  The P bodies of a lane are
// independent instruction streams that the compiler interleaves: the drift of one body is a serial
// chain of dependent FP64 operations, so P = 2 doubles the work in flight per warp and halves the
// per-body share of every warp-wide vote, branch and constant load.
// All 32 lanes must call; `live[p]` marks bodies to be advanced.  r2 = |r|^2 on entry; inv_mu = 1/mu
// and inv_mu_dt = dt/mu are constants of the run.  st[p] returns 0, GLISSE_FLAG_NONCONV (3) or
// GLISSE_FLAG_UNBOUND (4); on a non-zero status, or for !live bodies, the state is untouched.
// A body's arithmetic never depends on the other bodies of its lane or warp.
template <int P, bool REFINE = false>
__device__ __forceinline__ void kepler_drift_warp(const bool (&live_in)[P], double mu, double inv_mu,
                                                  double inv_mu_dt, int iters, double tol, const double (&r2)[P],
                                                  double (&x)[P], double (&y)[P], double (&z)[P], double (&vx)[P],
                                                  double (&vy)[P], double (&vz)[P], int (&st)[P], int& fast_iters,
                                                  bool& went_slow) {
  bool live[P], unbound[P], open[P], slow[P];
  double rinv[P], sqa[P], rsa[P], q[P], ec[P], es[P], dM[P], a[P], invq[P], e2[P], xk[P];
  double sm[P], cm1[P];  // sin x − x, cos x − 1 at the final xk
  int thr[P], nonconv[P];
  const bool fast_on = iters >= kFastMinIters && tol >= kFastMinTol;
  // 2 mu, exactly, by an exponent increment in the integer (uniform) pipe: one FP64 instruction less per step
  const double two_mu = __longlong_as_double(__double_as_longlong(mu) + (1LL << 52));
  bool any_open = false;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    const double v2 = fma(vx[p], vx[p], fma(vy[p], vy[p], vz[p] * vz[p]));
    const double u = fma(x[p], vx[p], fma(y[p], vy[p], z[p] * vz[p]));
    rinv[p] = rsqrt_f64(r2[p]);
    const double r0 = r2[p] * rinv[p];
    const double alpha = fma(two_mu, rinv[p], -v2);  // mu / a
    unbound[p] = !(hi_word(alpha) > 0);                // alpha <= 0 (or below 2^-1042: no such orbit)
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
    e2[p] = fma(ec[p], ec[p], es[p] * es[p]);
    xk[p] = live[p] ? dM[p] * invq[p] : 0.0;

    const int e2h = hi_word(e2[p]);
    thr[p] = e2h < kHiE2_010 ? kHiThr0 : (e2h < kHiE2_030 ? kHiThr1 : (e2h < kHiE2_050 ? kHiThr2 : kHiThr3));
    open[p] = live[p] && fast_on && e2h < kHiE2_080 && is_small_angle(xk[p]);
    if (REFINE && open[p] && wants_refined_guess(e2h, hi_abs(xk[p]))) {
      const double yy = xk[p];
      const double hq = 0.5 * invq[p];
      const double b2 = es[p] * hq;
      const double b3 = (ec[p] * hq) * (1.0 / 3.0);
      const double c3 = fma(2.0 * b2, b2, -b3);
      xk[p] = fma(yy * yy, fma(c3, yy, -b2), yy);
    }
    slow[p] = live[p] && !open[p];
    any_open = any_open || open[p];
    sm[p] = 0.0;
    cm1[p] = 0.0;
    nonconv[p] = 0;
  }
  fast_iters = 0;   // warp-uniform: iterations of the fast solver this warp executes (solver statistics)
  // (the first step is taken without asking whether any lane is open: a warp with none — every lane on
  // the slow path or dead — is rare, and the vote and branch cost every other warp 0.9 %)
  for (int it = 0; it < kFastMaxIters && ((it == 0 && fast_on) || __any_sync(kFullMask, any_open)); ++it) {
    any_open = false;
    fast_iters = it + 1;
#pragma unroll
    for (int p = 0; p < P; ++p) {
      double smk, cmk;
      sincosm_small(xk[p], smk, cmk);
      const double s = xk[p] + smk;
      const double c = 1.0 + cmk;
      const double f = fma(-es[p], cmk, fma(-ec[p], s, xk[p] - dM[p]));
      const double f1 = fma(es[p], s, fma(-ec[p], cmk, q[p]));
      const double f2 = fma(ec[p], s, es[p] * c);
      const double inv = rcp_f64_1(f1);
      const double dl = f * inv;        // Newton update
      const double h = dl * inv;
      const double u2 = f2 * h;         // 2 a2 delta
      const double f3 = 1.0 - f1;
      const double v6 = (f3 * h) * dl;  // 6 a3 delta^2
      const double w = fma(u2, fma(0.5, u2, 0.5), v6 * (-1.0 / 6.0));
      const double d = fma(dl, w, dl);
      // sin(x − d) − (x − d) and cos(x − d) − 1 from s, c at x:  sin d = d − d^3/6, cos d = 1 − d^2/2
      const double hd = 0.5 * d;
      const double h2 = hd * d;                  // d^2 / 2
      const double d3 = h2 * (d * (1.0 / 3.0));  // d^3 / 6
      const double smn = fma(c, d3, fma(-h2, s, fma(-d, cmk, smk)));
      const double cmn = fma(-s, d3, fma(-h2, c, fma(d, s, cmk)));
      if (open[p]) {
        sm[p] = smn;
        cm1[p] = cmn;
        xk[p] -= d;
        const bool done = hi_abs(dl) < thr[p];
        const bool lost = !done && !is_small_angle(xk[p]);  // left the polynomial's range (or NaN)
        open[p] = !done && !lost;
        slow[p] = slow[p] || lost;
      }
      any_open = any_open || open[p];
    }
  }
  bool any_slow = false;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    slow[p] = slow[p] || open[p];  // no convergence in kFastMaxIters steps
    any_slow = any_slow || slow[p];
  }
  went_slow = __any_sync(kFullMask, any_slow);
  if (went_slow) {
#pragma unroll
    for (int p = 0; p < P; ++p) {
      if (P == 1 || __any_sync(kFullMask, slow[p])) {   // (P == 1: any_slow above is this very vote)
        const ExactSolve o = kepler_solve_exact(slow[p], ec[p], es[p], q[p], dM[p], invq[p], e2[p], iters, tol);
        if (slow[p]) {
          xk[p] = o.x; sm[p] = o.sm; cm1[p] = o.cm1; nonconv[p] = o.nonconv;
        }
      }
    }
  }
#pragma unroll
  for (int p = 0; p < P; ++p) {
    const double s = xk[p] + sm[p];
    // Gauss f, g (PAPER.md:94 step 4), applied as r += (f−1) r + g v, v += fdot r + (gdot−1) v
    const double pr = fma(es[p], s, fma(-ec[p], cm1[p], q[p]));  // r(t)/a
    const double invp = rcp_f64(pr);
    const double fm1 = cm1[p] * invq[p];
    const double g = (dM[p] + sm[p]) * (a[p] * rsa[p]);  // (dM − x + sin x) / n
    const double fd = -(s * invp) * (sqa[p] * rinv[p]);
    const double gm1 = cm1[p] * invp;
    if (live[p] && !nonconv[p]) {
      // (in this order — inner position sums, velocities in place, positions in place — the loop-carried
      // state needs no register copies at the end of the step: six IMAD.MOV fewer, 1.3 % of the step)
      const double tx = fma(g, vx[p], x[p]), ty = fma(g, vy[p], y[p]), tz = fma(g, vz[p], z[p]);
      vx[p] = fma(fd, x[p], fma(gm1, vx[p], vx[p]));
      vy[p] = fma(fd, y[p], fma(gm1, vy[p], vy[p]));
      vz[p] = fma(fd, z[p], fma(gm1, vz[p], vz[p]));
      x[p] = fma(fm1, x[p], tx); y[p] = fma(fm1, y[p], ty); z[p] = fma(fm1, z[p], tz);
    }
    st[p] = !live_in[p] ? 0 : (unbound[p] ? GLISSE_FLAG_UNBOUND : (nonconv[p] ? GLISSE_FLAG_NONCONV : 0));
  }
}

// ---- the drift in three pieces, for the particle kernel --------------------------------------------
// The same arithmetic as kepler_drift_warp (bit for bit, for every body it advances), cut where the
// particle kernel wants its warp votes: the kernel runs drift_begin, ONE fast-solver step and
// drift_finish for all 32 lanes without any per-lane predicate, and everything a body can need beyond
// that (further fast steps, the definition's solver, the unbound / non-convergence flags) in a block it
// enters on one vote.  A lane that holds no particle of its own runs a copy of a live lane's body there
// (particles.cu), so no lane needs to be kept finite by selects: an unbound body's NaNs stay in its
// own lane and send the warp to that block.
struct DriftVars {
  double rinv, sqa, rsa, q, ec, es, dM, a, invq, e2;
};

// rinv = rsqrt_f64(r2): a caller whose positions are known long before its velocities (the planet-history
// kernel: the kick changes the velocities only) takes it off the dependent chain by computing it early
template <bool REFINE>
__device__ __forceinline__ void drift_begin_rinv(double mu, double two_mu, double inv_mu, double inv_mu_dt, double r2,
                                                 double rinv, double x, double y, double z, double vx, double vy,
                                                 double vz, DriftVars& k, double& xk, bool& unbound) {
  const double v2 = fma(vx, vx, fma(vy, vy, vz * vz));
  const double u = fma(x, vx, fma(y, vy, z * vz));
  k.rinv = rinv;
  const double r0 = r2 * k.rinv;
  const double al = fma(two_mu, k.rinv, -v2);  // mu / a
  unbound = !(hi_word(al) > 0);                 // alpha <= 0 (or below 2^-1042: no such orbit), or NaN
  k.rsa = rsqrt_f64(al);
  k.sqa = al * k.rsa;                    // sqrt(alpha) = n a
  const double inva = k.rsa * k.rsa;     // 1 / alpha
  k.q = r0 * (al * inv_mu);              // r0 / a = 1 − ec
  k.ec = 1.0 - k.q;
  k.es = u * (k.sqa * inv_mu);
  // n dt.  The reduction of reading S9 (dM = n dt - 2 pi rint(n dt / 2 pi)) changes nothing while
  // |n dt| <= pi, i.e. while a step spans less than half a revolution: it is left to reduce_mean_motion,
  // which the caller applies (out of line) to the bodies whose |n dt| is not below kHiPi
  k.dM = (al * k.sqa) * inv_mu_dt;
  k.a = mu * inva;
  k.invq = k.a * k.rinv;  // a / r0
  k.e2 = fma(k.ec, k.ec, k.es * k.es);
  xk = k.dM * k.invq;
  if (REFINE) {
    const int e2h = hi_word(k.e2);
    if (e2h < kHiE2_080 && is_small_angle(xk) && wants_refined_guess(e2h, hi_abs(xk))) {
      const double yy = xk;
      const double hq = 0.5 * k.invq;
      const double b2 = k.es * hq;
      const double b3 = (k.ec * hq) * (1.0 / 3.0);
      const double c3 = fma(2.0 * b2, b2, -b3);
      xk = fma(yy * yy, fma(c3, yy, -b2), yy);
    }
  }
}

template <bool REFINE>
__device__ __forceinline__ void drift_begin(double mu, double two_mu, double inv_mu, double inv_mu_dt, double r2,
                                            double x, double y, double z, double vx, double vy, double vz,
                                            DriftVars& k, double& xk, bool& unbound) {
  drift_begin_rinv<REFINE>(mu, two_mu, inv_mu, inv_mu_dt, r2, rsqrt_f64(r2), x, y, z, vx, vy, vz, k, xk, unbound);
}

// reading S9 for a body whose step spans half a revolution or more (drift_begin)
constexpr int kHiPi = 0x400921fb;   // high word of pi = 0x400921fb54442d18: hi_abs(x) < kHiPi implies |x| < pi
__device__ __forceinline__ double reduce_mean_motion(double ndt) {
  return fma(-rint(ndt * kInvTwoPi), kTwoPi, ndt);
}

// Acceptance bound of the fast solver for this eccentricity (high word of the bound on |delta|), for the
// particle kernel: the same error model as the tiers above — (5 a2^3 + 5 a2 a3 + a4) delta^4 < 2e-17
// with a_k = e / (k! (1 - e)) — as ONE integer instruction instead of seven: in the high words
// (piecewise-linear logarithms) the bound is below  min(9e-5, 1.9e-5 (0.64 / e^2))  for every e < 0.8:
// at most 0.974 of the model's bound (worst at e = 0.36), i.e. an error below 1.8e-17.  It is never
// tighter than the tiers by more than 10 % and up to 2.4 times wider between their steps (e = 0.5),
// which saves planet-crossing bodies a second step.
constexpr int kHiThrLine = kHiE2_080 + kHiThr3 - 0x10000;
__device__ __forceinline__ int fast_threshold(int e2h) { return min(kHiThr1, kHiThrLine - e2h); }
// |delta| (high word, sign cleared) is below fast_threshold(e2h): as two compares and an add, no selects
__device__ __forceinline__ bool fast_accepts(int dl_hi_abs, int e2h) {
  return (dl_hi_abs < kHiThr1) & (dl_hi_abs + e2h < kHiThrLine);
}

// one step of the fast solver from xk: the new x, sin x − x and cos x − 1 there, and the Newton update dl
__device__ __forceinline__ void fast_step(const DriftVars& k, double xk, double& xn, double& smn, double& cmn,
                                          double& dl) {
  double smk, cmk;
  sincosm_small(xk, smk, cmk);
  const double s = xk + smk;
  const double c = 1.0 + cmk;
  const double f = fma(-k.es, cmk, fma(-k.ec, s, xk - k.dM));
  const double f1 = fma(k.es, s, fma(-k.ec, cmk, k.q));
  const double f2 = fma(k.ec, s, k.es * c);
  const double inv = rcp_f64_1(f1);
  dl = f * inv;                     // Newton update
  const double h = dl * inv;
  const double u2 = f2 * h;         // 2 a2 delta
  const double f3 = 1.0 - f1;
  const double v6 = (f3 * h) * dl;  // 6 a3 delta^2
  const double w = fma(u2, fma(0.5, u2, 0.5), v6 * (-1.0 / 6.0));
  const double d = fma(dl, w, dl);
  const double hd = 0.5 * d;
  const double h2 = hd * d;                  // d^2 / 2
  const double d3 = h2 * (d * (1.0 / 3.0));  // d^3 / 6
  smn = fma(c, d3, fma(-h2, s, fma(-d, cmk, smk)));
  cmn = fma(-s, d3, fma(-h2, c, fma(d, s, cmk)));
  xn = xk - d;
}

// Gauss f, g (PAPER.md:94 step 4) from the solved x: r += (f−1) r + g v, v += fdot r + (gdot−1) v
__device__ __forceinline__ void drift_finish(const DriftVars& k, double xk, double sm, double cm1, double& x,
                                             double& y, double& z, double& vx, double& vy, double& vz) {
  const double s = xk + sm;
  const double pr = fma(k.es, s, fma(-k.ec, cm1, k.q));  // r(t)/a
  const double invp = rcp_f64(pr);
  const double fm1 = cm1 * k.invq;
  const double g = (k.dM + sm) * (k.a * k.rsa);  // (dM − x + sin x) / n
  const double fd = -(s * invp) * (k.sqa * k.rinv);
  const double gm1 = cm1 * invp;
  const double tx = fma(g, vx, x), ty = fma(g, vy, y), tz = fma(g, vz, z);
  vx = fma(fd, x, fma(gm1, vx, vx));
  vy = fma(fd, y, fma(gm1, vy, vy));
  vz = fma(fd, z, fma(gm1, vz, vz));
  x = fma(fm1, x, tx); y = fma(fm1, y, ty); z = fma(fm1, z, tz);
}

// One body per lane (the planet-history kernel and the primitive test hook).
template <bool REFINE>
__device__ __forceinline__ int kepler_drift_one(bool live, double mu, double inv_mu, double inv_mu_dt, int iters,
                                                double tol, double r2, double& x, double& y, double& z,
                                                double& vx, double& vy, double& vz) {
  const bool l1[1] = {live};
  const double r21[1] = {r2};
  double x1[1] = {x}, y1[1] = {y}, z1[1] = {z}, vx1[1] = {vx}, vy1[1] = {vy}, vz1[1] = {vz};
  int st[1], fast_iters;
  bool went_slow;
  kepler_drift_warp<1, REFINE>(l1, mu, inv_mu, inv_mu_dt, iters, tol, r21, x1, y1, z1, vx1, vy1, vz1, st, fast_iters,
                               went_slow);
  x = x1[0]; y = y1[0]; z = z1[0]; vx = vx1[0]; vy = vy1[0]; vz = vz1[0];
  return st[0];
}

}  // namespace glisse
