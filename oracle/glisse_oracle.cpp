/*
 * glisse_oracle.cpp — the ORACLE: a plain, slow, single-threaded fp64 CPU implementation of the
 * GLISSE test-particle integrator, written from the paper (Zhang & Gladman 2020, PAPER.md) and
 * the readings listed in DESIGN.md §2.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may build, load or call it.  It shares no code, header, table or helper
 * with the CUDA path under paper_2011_03484_b200/csrc/, and neither side includes the other.
 *
 * Style: the algorithm step by step in the paper's order and notation; no blocking, fusion,
 * reordering, vectorisation or early exit.  Build: g++ -O2 -ffp-contract=off (no FMA
 * contraction), libm sin/cos/sqrt.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): two-body closed form (T1), single-planet
 * Kepler orbit (T2), finite-difference gradient of H_int vs the planet kick (T3), CR3BP Jacobi
 * constant bounded and O(dt^2) (T4), time reversal (T5), order-2 convergence to a brute-force
 * high-order direct integration (T6), the paper's 5-iteration / 1e-14 claim (T7),
 * removal logic on crafted inputs (T8), osculating elements against the textbook perifocal
 * construction (T9), resonant argument against its formula and constant at exact commensurability
 * (T10), libration summary against constructed librators and hand-worked series (T11), the interpolated
 * planet log against exactness on cubics, the Hermite error bound on a circular orbit and h0's formula (T12).
 * Parity unpinned: none of the functions below; the
 * paper's application-level numbers (10.8 % librators …) are unpinned because the authors'
 * initial conditions are not available.
 *
 * Notation: mu0 = G m0 (star); mu_j = G m_j, j = 0..Np-1 in Jacobi order (innermost first,
 * PAPER.md:87); q_j, qd_j heliocentric planet position / velocity; r, v heliocentric particle
 * position / velocity; dt the fixed step.
 */
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <vector>

namespace {

constexpr int kMaxPlanets = 32;
constexpr int kPlanetKeplerIters = 10; /* generous count for planets, O3 */
constexpr double kTwoPi = 6.283185307179586476925286766559;

enum Flag { ACTIVE = 0, RMIN = 1, RMAX = 2, NONCONV = 3, UNBOUND = 4, PLANET0 = 16 };

struct Params {
  double r_min, r_max;
  int kepler_iters;
  double kepler_tol;
  int scheme; /* 0 = kick-drift-kick, 1 = drift-kick-drift (BASELINE.json's wording, reading S20) */
};

/* ---------------------------------------------------------------------------------------------
 * O2. Kepler drift (PAPER.md:92-94 steps 2–4 and the Kepler equation at).
 * Advance (r, v) along the two-body orbit about a point mass mu for time dt.
 * Differenced form of Kepler's equation in x = E(t) − E(t0) (reading S4):
 *     dM = n dt = x − ec sin x + es (1 − cos x),   ec = e cos E0,  es = e sin E0,
 * solved by exactly `iters` Newton updates from the initial guess of reading S5, followed by the
 * Gauss f and g functions.  Returns ACTIVE, UNBOUND (alpha <= 0, reading S8) or NONCONV
 * (|residual| > tol, reading S6).  On a non-zero return r, v are left untouched.
 * ------------------------------------------------------------------------------------------- */
int kepler_drift(double mu, double r[3], double v[3], double dt, int iters, double tol) {
  const double r0 = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
  const double u = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
  const double alpha = 2.0 * mu / r0 - v2; /* = mu / a */
  if (!(alpha > 0.0)) return UNBOUND;
  const double a = mu / alpha;
  const double n = std::sqrt(mu / (a * a * a));
  const double ec = 1.0 - r0 / a;
  const double es = u / (n * a * a);
  const double e = std::sqrt(ec * ec + es * es);
  const double ndt = n * dt;
  const double dM = ndt - kTwoPi * std::nearbyint(ndt / kTwoPi); /* reading S9 */

  /* initial guess, reading S5 */
  const double q = r0 / a; /* = 1 − ec */
  const double x1 = dM / q;
  double x;
  if (std::fabs(es) * std::fabs(x1) < 0.25 * q && e * x1 * x1 < 0.25 * q) {
    x = x1;
  } else {
    const double y = dM - es;
    const double sg = es * std::cos(y) + ec * std::sin(y);
    x = y + (sg >= 0.0 ? 0.85 : -0.85) * e;
  }

  /* fixed number of Newton updates */
  for (int it = 0; it < iters; ++it) {
    const double s = std::sin(x), c = std::cos(x);
    const double f = x - ec * s + es * (1.0 - c) - dM;
    const double fp = 1.0 - ec * c + es * s;
    x = x - f / fp;
  }
  const double s = std::sin(x), c = std::cos(x);
  const double res = x - ec * s + es * (1.0 - c) - dM;
  if (!(std::fabs(res) <= tol)) return NONCONV;

  /* Gauss f, g functions (BASELINE.json north_star; Danby, Fundamentals of Celestial Mechanics §6.7) */
  const double p = 1.0 - ec * c + es * s; /* r(t)/a */
  const double fg_f = 1.0 + (c - 1.0) * a / r0;
  const double fg_g = (dM - x + s) / n; /* = dt + (s − x)/n with dM in place of n dt (S9) */
  const double fg_fd = -n * s * a / (r0 * p);
  const double fg_gd = 1.0 + (c - 1.0) / p;
  for (int k = 0; k < 3; ++k) {
    const double rk = r[k], vk = v[k];
    r[k] = fg_f * rk + fg_g * vk;
    v[k] = fg_fd * rk + fg_gd * vk;
  }
  return ACTIVE;
}

/* ---------------------------------------------------------------------------------------------
 * h0, the common heliocentric term:  h0 = − sum_j mu_j q_j / |q_j|^3 .
 * ------------------------------------------------------------------------------------------- */
void common_term_h0(int np, const double* gm, const double* q, double h0[3]) {
  h0[0] = h0[1] = h0[2] = 0.0;
  for (int j = 0; j < np; ++j) {
    const double* qj = q + 3 * j;
    const double d2 = qj[0] * qj[0] + qj[1] * qj[1] + qj[2] * qj[2];
    const double d = std::sqrt(d2);
    const double w = gm[j] / (d2 * d);
    for (int k = 0; k < 3; ++k) h0[k] -= w * qj[k];
  }
}

/* ---------------------------------------------------------------------------------------------
 * O3. One Wisdom–Holman step of the planets ("standard Wisdom-Holman mixed-variable
 * symplectic algorithm"), Jacobi coordinates, reading S14.
 *   eta_k = m0 + sum_{i<=k} m_i  (eta_{-1} = m0); all masses enter as G m.
 *   Jacobi position  r'_k = q_k − (sum_{i<k} m_i q_i) / eta_{k-1}   (same map for velocities)
 *   inverse          q_k  = r'_k + sum_{i<k} (m_i / eta_i) r'_i
 *   H_int = sum_k G m_k m0 (1/|r'_k| − 1/|q_k|) − sum_{i<j} G m_i m_j / |q_i − q_j|
 *   kick  v'_k += h (eta_k/eta_{k-1}) [ mu0 r'_k/|r'_k|^3 + A_k + (1/eta_k) sum_{i>k} m_i A_i ],
 *         A_i = − mu0 q_i/|q_i|^3 − sum_{j != i} mu_j (q_i − q_j)/|q_i − q_j|^3
 *   drift of planet k: two-body motion in (r'_k, v'_k) with mu = mu0 eta_k / eta_{k-1}.
 * Returns 0, or the 1-based index of the first planet whose drift failed.
 * ------------------------------------------------------------------------------------------- */
void helio_to_jacobi(int np, double gm0, const double* gm, const double* h, double* jac) {
  double sum[3] = {0.0, 0.0, 0.0}; /* sum_{i<k} m_i h_i */
  double eta = gm0;                /* eta_{k-1} */
  for (int k = 0; k < np; ++k) {
    for (int c = 0; c < 3; ++c) jac[3 * k + c] = h[3 * k + c] - sum[c] / eta;
    for (int c = 0; c < 3; ++c) sum[c] += gm[k] * h[3 * k + c];
    eta += gm[k];
  }
}

void jacobi_to_helio(int np, double gm0, const double* gm, const double* jac, double* h) {
  double sum[3] = {0.0, 0.0, 0.0}; /* sum_{i<k} (m_i/eta_i) r'_i */
  double eta = gm0;
  for (int k = 0; k < np; ++k) {
    for (int c = 0; c < 3; ++c) h[3 * k + c] = jac[3 * k + c] + sum[c];
    eta += gm[k]; /* eta_k */
    for (int c = 0; c < 3; ++c) sum[c] += gm[k] / eta * jac[3 * k + c];
  }
}

/* Jacobi accelerations dv'_k/dt = −(1/m'_k) dH_int/dr'_k, m'_k = m_k eta_{k-1}/eta_k. */
void planet_kick_accel(int np, double gm0, const double* gm, const double* q, const double* rj,
                       double* acc) {
  std::vector<double> A(3 * np, 0.0);
  for (int i = 0; i < np; ++i) {
    const double* qi = q + 3 * i;
    const double d2 = qi[0] * qi[0] + qi[1] * qi[1] + qi[2] * qi[2];
    const double d = std::sqrt(d2);
    const double w = gm0 / (d2 * d);
    for (int c = 0; c < 3; ++c) A[3 * i + c] = -w * qi[c];
    for (int j = 0; j < np; ++j) {
      if (j == i) continue;
      const double* qj = q + 3 * j;
      const double dx[3] = {qi[0] - qj[0], qi[1] - qj[1], qi[2] - qj[2]};
      const double s2 = dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2];
      const double s = std::sqrt(s2);
      const double wj = gm[j] / (s2 * s);
      for (int c = 0; c < 3; ++c) A[3 * i + c] -= wj * dx[c];
    }
  }
  double eta_prev = gm0;
  for (int k = 0; k < np; ++k) {
    const double eta = eta_prev + gm[k];
    const double* rk = rj + 3 * k;
    const double d2 = rk[0] * rk[0] + rk[1] * rk[1] + rk[2] * rk[2];
    const double d = std::sqrt(d2);
    const double w = gm0 / (d2 * d);
    double tail[3] = {0.0, 0.0, 0.0}; /* sum_{i>k} m_i A_i */
    for (int i = k + 1; i < np; ++i)
      for (int c = 0; c < 3; ++c) tail[c] += gm[i] * A[3 * i + c];
    for (int c = 0; c < 3; ++c)
      acc[3 * k + c] = (eta / eta_prev) * (w * rk[c] + A[3 * k + c] + tail[c] / eta);
    eta_prev = eta;
  }
}

int planet_step(int np, double gm0, const double* gm, double* q, double* qd, double dt) {
  if (np == 0) return 0;
  std::vector<double> rj(3 * np), vj(3 * np), acc(3 * np);
  helio_to_jacobi(np, gm0, gm, q, rj.data());
  helio_to_jacobi(np, gm0, gm, qd, vj.data());
  /* kick 1/2 */
  planet_kick_accel(np, gm0, gm, q, rj.data(), acc.data());
  for (int i = 0; i < 3 * np; ++i) vj[i] += 0.5 * dt * acc[i];
  /* drift 1 */
  double eta_prev = gm0;
  for (int k = 0; k < np; ++k) {
    const double eta = eta_prev + gm[k];
    const double mu = gm0 * eta / eta_prev;
    const int st = kepler_drift(mu, &rj[3 * k], &vj[3 * k], dt, kPlanetKeplerIters, 1e-13);
    if (st != ACTIVE) return k + 1;
    eta_prev = eta;
  }
  /* kick 1/2 at the new positions */
  jacobi_to_helio(np, gm0, gm, rj.data(), q);
  planet_kick_accel(np, gm0, gm, q, rj.data(), acc.data());
  for (int i = 0; i < 3 * np; ++i) vj[i] += 0.5 * dt * acc[i];
  jacobi_to_helio(np, gm0, gm, vj.data(), qd);
  return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O1/O4/O5. One force evaluation on a particle with the tests of PAPER.md:125-127 ("while
 * computing the acceleration").  Returns the flag that fires (priority: r_min, r_max, lowest
 * planet index; reading S11) or ACTIVE with the acceleration
 *     a = h0 − sum_j mu_j (r − q_j)/|r − q_j|^3
 * ------------------------------------------------------------------------------------------- */
int particle_accel(int np, const double* gm, const double* q, const double h0[3],
                   const double* rcrit2, const Params& P, const double r[3], double a[3]) {
  const double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
  if (P.r_min > 0.0 && r2 < P.r_min * P.r_min) return RMIN;
  if (P.r_max > 0.0 && r2 > P.r_max * P.r_max) return RMAX;
  a[0] = h0[0]; a[1] = h0[1]; a[2] = h0[2];
  int hit = ACTIVE;
  for (int j = 0; j < np; ++j) {
    const double d[3] = {r[0] - q[3 * j], r[1] - q[3 * j + 1], r[2] - q[3 * j + 2]};
    const double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (hit == ACTIVE && d2 < rcrit2[j]) hit = PLANET0 + j;
    const double dd = std::sqrt(d2);
    const double w = gm[j] / (d2 * dd);
    for (int k = 0; k < 3; ++k) a[k] -= w * d[k];
  }
  return hit;
}

struct Sim {
  double gm0 = 0.0;
  int np = 0;
  std::vector<double> gm, q, qd, rcrit2;
  long long n = 0;
  std::vector<double> x[3], v[3];
  std::vector<int> flag;
  std::vector<long long> rstep;
  double dt = 0.0;
  Params P{};
  long long step = 0;
  long long particle_steps = 0;
  /* drift-kick-drift only: q, qd above hold the planets at t_{step - 1/2} once step > 0 (the instants
   * at which the scheme samples them); q0, qd0 keep the state at t_0 */
  std::vector<double> q_half, qd_half;
  bool half_started = false;
};

/* kick every active particle by h·a evaluated with planets (q, h0); `completed` = number of
 * completed steps to record on a hit (reading S12) */
void kick_particles(Sim& S, const double* q, const double h0[3], double h, long long completed) {
  for (long long i = 0; i < S.n; ++i) {
    if (S.flag[i] != ACTIVE) continue;
    const double r[3] = {S.x[0][i], S.x[1][i], S.x[2][i]};
    double a[3];
    const int hit = particle_accel(S.np, S.gm.data(), q, h0, S.rcrit2.data(), S.P, r, a);
    if (hit != ACTIVE) {
      S.flag[i] = hit;
      S.rstep[i] = completed;
      continue; /* frozen: the kick of this evaluation is NOT applied (O5) */
    }
    for (int k = 0; k < 3; ++k) S.v[k][i] += h * a[k];
  }
}

void drift_particles(Sim& S, double dt) {
  for (long long i = 0; i < S.n; ++i) {
    if (S.flag[i] != ACTIVE) continue;
    double r[3] = {S.x[0][i], S.x[1][i], S.x[2][i]};
    double v[3] = {S.v[0][i], S.v[1][i], S.v[2][i]};
    const int st = kepler_drift(S.gm0, r, v, dt, S.P.kepler_iters, S.P.kepler_tol);
    if (st != ACTIVE) {
      S.flag[i] = st;
      S.rstep[i] = S.step; /* flagged during step `step`: that many steps were completed */
      continue;
    }
    for (int k = 0; k < 3; ++k) { S.x[k][i] = r[k]; S.v[k][i] = v[k]; }
  }
}

long long count_active(const Sim& S) {
  long long c = 0;
  for (long long i = 0; i < S.n; ++i) c += (S.flag[i] == ACTIVE);
  return c;
}

int log_stride(int np) { return (3 * (np + 1) + 1) & ~1; }

bool all_finite(const double* p, long long n) {
  for (long long i = 0; i < n; ++i)
    if (!std::isfinite(p[i])) return false;
  return true;
}

}  // namespace

extern "C" {

struct oracle_sim;

typedef struct {
  double r_min, r_max;
  int kepler_iters;
  double kepler_tol;
  int scheme; /* 0 kick-drift-kick (default), 1 drift-kick-drift */
} oracle_params;

void oracle_default_params(oracle_params* p) {
  if (!p) return;
  p->r_min = 0.0;
  p->r_max = std::numeric_limits<double>::infinity();
  p->kepler_iters = 5;
  p->kepler_tol = 1e-14;
  p->scheme = 0;
}

int oracle_log_stride(int n_planets) {
  return (n_planets < 0 || n_planets > kMaxPlanets) ? 0 : log_stride(n_planets);
}

int oracle_create(oracle_sim** out, double gm_star, int n_planets, const double* gm_planet,
                  const double* planet_pos, const double* planet_vel, const double* planet_rcrit,
                  long long n_particles, const double* const pos[3], const double* const vel[3],
                  double dt, const oracle_params* params) {
  if (!out) return -1;
  *out = nullptr;
  if (n_planets < 0 || n_planets > kMaxPlanets || n_particles < 1 || !pos || !vel) return -1;
  if (!(gm_star > 0.0) || !std::isfinite(gm_star) || dt == 0.0 || !std::isfinite(dt)) return -1;
  if (n_planets > 0 && (!gm_planet || !planet_pos || !planet_vel)) return -1;
  for (int k = 0; k < 3; ++k)
    if (!pos[k] || !vel[k] || !all_finite(pos[k], n_particles) || !all_finite(vel[k], n_particles))
      return -1;
  if (n_planets > 0 && (!all_finite(gm_planet, n_planets) || !all_finite(planet_pos, 3 * n_planets) ||
                        !all_finite(planet_vel, 3 * n_planets)))
    return -1;
  Sim* S = new (std::nothrow) Sim;
  if (!S) return -3;
  S->gm0 = gm_star;
  S->np = n_planets;
  S->gm.assign(gm_planet, gm_planet + n_planets);
  for (int j = 0; j < n_planets; ++j)
    if (!(S->gm[j] > 0.0)) { delete S; return -1; }
  S->q.assign(planet_pos, planet_pos + 3 * n_planets);
  S->qd.assign(planet_vel, planet_vel + 3 * n_planets);
  S->rcrit2.assign(n_planets, 0.0);
  if (planet_rcrit)
    for (int j = 0; j < n_planets; ++j) S->rcrit2[j] = planet_rcrit[j] * planet_rcrit[j];
  S->n = n_particles;
  for (int k = 0; k < 3; ++k) {
    S->x[k].assign(pos[k], pos[k] + n_particles);
    S->v[k].assign(vel[k], vel[k] + n_particles);
  }
  S->flag.assign(n_particles, ACTIVE);
  S->rstep.assign(n_particles, -1);
  S->dt = dt;
  oracle_params d;
  oracle_default_params(&d);
  if (params) d = *params;
  if (d.kepler_iters < 0 || !(d.kepler_tol > 0.0) || d.scheme < 0 || d.scheme > 1) { delete S; return -1; }
  S->P.scheme = d.scheme;
  S->P.r_min = d.r_min;
  S->P.r_max = (std::isfinite(d.r_max) ? d.r_max : 0.0);
  S->P.kepler_iters = d.kepler_iters;
  S->P.kepler_tol = d.kepler_tol;
  *out = reinterpret_cast<oracle_sim*>(S);
  return 0;
}

/* Drift-kick-drift variant (BASELINE.json north_star's wording; reading S20 of DESIGN.md §2): the same
 * second-order splitting with the roles exchanged,
 *   D1. drift every active particle for dt/2 (O2's routine);
 *   D2. planets at the half step t_{s+1/2}: the planets are carried by the same Wisdom-Holman step as in
 *       the kick-drift-kick scheme, started with ONE step of size dt/2 (t_0 -> t_{1/2}) and continued with
 *       steps of size dt (t_{s-1/2} -> t_{s+1/2}), so that they are sampled where the kick needs them
 *       (the log may hold the planets at whatever instants the scheme asks for);
 *   D3. kick every active particle by dt a(r, q(t_{s+1/2})), tests O5 on this evaluation; a hit records
 *       `step` completed steps and freezes the state of that instant (after D1, without this kick);
 *   D4. drift for dt/2.
 * A particle flagged in D1 or D4 keeps the state it had on entry to that drift. */
static int advance_dkd(Sim& S, long long n_steps) {
  const double hdt = 0.5 * S.dt;
  double h0[3];
  for (long long s = 0; s < n_steps; ++s) {
    S.particle_steps += count_active(S);
    drift_particles(S, hdt);                                                     /* D1 */
    if (!S.half_started) {                                                       /* D2 */
      S.q_half = S.q; S.qd_half = S.qd;
      if (planet_step(S.np, S.gm0, S.gm.data(), S.q_half.data(), S.qd_half.data(), hdt)) return -4;
      S.half_started = true;
    } else {
      if (planet_step(S.np, S.gm0, S.gm.data(), S.q_half.data(), S.qd_half.data(), S.dt)) return -4;
    }
    common_term_h0(S.np, S.gm.data(), S.q_half.data(), h0);
    kick_particles(S, S.q_half.data(), h0, S.dt, S.step);                        /* D3 */
    drift_particles(S, hdt);                                                     /* D4 */
    S.step += 1;
    /* planets at the integer time t_step, for oracle_read_planets: half a step on from t_{step-1/2} */
    S.q = S.q_half; S.qd = S.qd_half;
    if (planet_step(S.np, S.gm0, S.gm.data(), S.q.data(), S.qd.data(), hdt)) return -4;
  }
  return 0;
}

/* One full step s -> s+1 for everything, in the order O1, O2, O3, O4 of DESIGN.md §2. */
int oracle_advance(oracle_sim* sim, long long n_steps) {
  if (!sim || n_steps < 0) return -1;
  Sim& S = *reinterpret_cast<Sim*>(sim);
  if (S.P.scheme == 1) return advance_dkd(S, n_steps);
  const double h = 0.5 * S.dt;
  double h0[3];
  for (long long s = 0; s < n_steps; ++s) {
    /* O1: opening half kick, planets at t_s */
    common_term_h0(S.np, S.gm.data(), S.q.data(), h0);
    kick_particles(S, S.q.data(), h0, h, S.step);
    S.particle_steps += count_active(S);
    /* O2: drift */
    drift_particles(S, S.dt);
    /* O3: planets t_s -> t_{s+1} */
    const int bad = planet_step(S.np, S.gm0, S.gm.data(), S.q.data(), S.qd.data(), S.dt);
    if (bad) return -4;
    /* O4: closing half kick, planets at t_{s+1} */
    common_term_h0(S.np, S.gm.data(), S.q.data(), h0);
    kick_particles(S, S.q.data(), h0, h, S.step + 1);
    S.step += 1;
  }
  return 0;
}

/* Planet log for the next n_steps steps: n_steps+1 records of oracle_log_stride(np) doubles
 * [q_0 … q_{Np-1}, h0, pad] at times t_s … t_{s+n}.  The simulation is not
 * changed. */
int oracle_planet_log(oracle_sim* sim, long long n_steps, double* log) {
  if (!sim || n_steps < 0 || !log) return -1;
  const Sim& S = *reinterpret_cast<Sim*>(sim);
  std::vector<double> q = S.q, qd = S.qd;
  const int st = log_stride(S.np);
  if (S.P.scheme == 1) {
    /* drift-kick-drift: record k = planets at t_{step + k + 1/2}, k = 0 .. n_steps (D2) */
    if (S.half_started) {
      q = S.q_half; qd = S.qd_half;
      if (planet_step(S.np, S.gm0, S.gm.data(), q.data(), qd.data(), S.dt)) return -4;
    } else {
      if (planet_step(S.np, S.gm0, S.gm.data(), q.data(), qd.data(), 0.5 * S.dt)) return -4;
    }
    for (long long s = 0; s <= n_steps; ++s) {
      double* rec = log + s * st;
      for (int i = 0; i < st; ++i) rec[i] = 0.0;
      for (int i = 0; i < 3 * S.np; ++i) rec[i] = q[i];
      common_term_h0(S.np, S.gm.data(), q.data(), rec + 3 * S.np);
      if (s < n_steps && planet_step(S.np, S.gm0, S.gm.data(), q.data(), qd.data(), S.dt)) return -4;
    }
    return 0;
  }
  for (long long s = 0; s <= n_steps; ++s) {
    double* rec = log + s * st;
    for (int i = 0; i < st; ++i) rec[i] = 0.0;
    for (int i = 0; i < 3 * S.np; ++i) rec[i] = q[i];
    common_term_h0(S.np, S.gm.data(), q.data(), rec + 3 * S.np);
    if (s < n_steps) {
      const int bad = planet_step(S.np, S.gm0, S.gm.data(), q.data(), qd.data(), S.dt);
      if (bad) return -4;
    }
  }
  return 0;
}

/* Planet log from a SPARSE history by interpolation ("these planetary positions could be
 * supplied using any method, such as interpolation from a history file"; reading S24): the
 * history holds n_samples instants t_m (strictly increasing) with the heliocentric positions q_j(t_m) and
 * velocities qd_j(t_m) of the np planets, [n_samples][np][3] each.  Record r = 0 .. n_records-1 of the log
 * is taken at t = t_first + r dt_record by cubic Hermite interpolation on the interval [t_m, t_m+1] that
 * holds t (the last interval includes its right end), component by component:
 *   tau = (t - t_m)/D,  D = t_m+1 - t_m
 *   q(t) = h00 q_m + h10 D qd_m + h01 q_m+1 + h11 D qd_m+1
 *   h00 = 2 tau^3 - 3 tau^2 + 1, h10 = tau^3 - 2 tau^2 + tau, h01 = -2 tau^3 + 3 tau^2, h11 = tau^3 - tau^2
 * and h0 = -sum_j mu_j q_j/|q_j|^3 of the interpolated positions.  Layout of a record as in
 * oracle_planet_log.  Returns -1 for bad arguments or a time outside the history. */
int oracle_interpolate_log(int np, const double* gm, long long n_samples, const double* sample_time,
                           const double* sample_pos, const double* sample_vel, double t_first, double dt_record,
                           long long n_records, double* log) {
  if (np < 0 || np > kMaxPlanets || n_samples < 2 || n_records < 0 || !sample_time || !log) return -1;
  if (np > 0 && (!gm || !sample_pos || !sample_vel)) return -1;
  for (long long m = 0; m + 1 < n_samples; ++m)
    if (!(sample_time[m + 1] > sample_time[m])) return -1;
  const int st = log_stride(np);
  for (long long r = 0; r < n_records; ++r) {
    const double t = t_first + static_cast<double>(r) * dt_record;
    if (!(t >= sample_time[0]) || !(t <= sample_time[n_samples - 1])) return -1;
    long long m = 0;
    while (m + 2 < n_samples && t >= sample_time[m + 1]) ++m;
    const double D = sample_time[m + 1] - sample_time[m];
    const double tau = (t - sample_time[m]) / D;
    const double tau2 = tau * tau, tau3 = tau2 * tau;
    const double h00 = 2.0 * tau3 - 3.0 * tau2 + 1.0;
    const double h10 = tau3 - 2.0 * tau2 + tau;
    const double h01 = -2.0 * tau3 + 3.0 * tau2;
    const double h11 = tau3 - tau2;
    double* rec = log + r * st;
    for (int i = 0; i < st; ++i) rec[i] = 0.0;
    for (int i = 0; i < 3 * np; ++i) {
      const double q0 = sample_pos[m * 3 * np + i], q1 = sample_pos[(m + 1) * 3 * np + i];
      const double v0 = sample_vel[m * 3 * np + i], v1 = sample_vel[(m + 1) * 3 * np + i];
      rec[i] = h00 * q0 + h10 * D * v0 + h01 * q1 + h11 * D * v1;
    }
    common_term_h0(np, gm, rec, rec + 3 * np);
  }
  return 0;
}

/* Particles only, planets taken from a caller-supplied log; planet state unchanged. */
int oracle_advance_with_log(oracle_sim* sim, long long n_steps, const double* log) {
  if (!sim || n_steps < 0 || !log) return -1;
  Sim& S = *reinterpret_cast<Sim*>(sim);
  const double h = 0.5 * S.dt;
  const int st = log_stride(S.np);
  if (S.P.scheme == 1) { /* drift-kick-drift: record s = planets at the half step of step s */
    for (long long s = 0; s < n_steps; ++s) {
      const double* rec = log + s * st;
      S.particle_steps += count_active(S);
      drift_particles(S, h);
      kick_particles(S, rec, rec + 3 * S.np, S.dt, S.step);
      drift_particles(S, h);
      S.step += 1;
    }
    return 0;
  }
  for (long long s = 0; s < n_steps; ++s) {
    const double* r0 = log + s * st;
    const double* r1 = log + (s + 1) * st;
    kick_particles(S, r0, r0 + 3 * S.np, h, S.step);
    S.particle_steps += count_active(S);
    drift_particles(S, S.dt);
    kick_particles(S, r1, r1 + 3 * S.np, h, S.step + 1);
    S.step += 1;
  }
  return 0;
}

int oracle_read(oracle_sim* sim, double* const pos[3], double* const vel[3], int* flag,
                long long* removal_step) {
  if (!sim) return -1;
  const Sim& S = *reinterpret_cast<Sim*>(sim);
  for (int k = 0; k < 3; ++k) {
    if (pos && pos[k]) std::memcpy(pos[k], S.x[k].data(), sizeof(double) * S.n);
    if (vel && vel[k]) std::memcpy(vel[k], S.v[k].data(), sizeof(double) * S.n);
  }
  if (flag) std::memcpy(flag, S.flag.data(), sizeof(int) * S.n);
  if (removal_step) std::memcpy(removal_step, S.rstep.data(), sizeof(long long) * S.n);
  return 0;
}

int oracle_read_planets(oracle_sim* sim, double* pos, double* vel) {
  if (!sim) return -1;
  const Sim& S = *reinterpret_cast<Sim*>(sim);
  if (pos) std::memcpy(pos, S.q.data(), sizeof(double) * 3 * S.np);
  if (vel) std::memcpy(vel, S.qd.data(), sizeof(double) * 3 * S.np);
  return 0;
}

long long oracle_active_count(oracle_sim* sim) {
  return sim ? count_active(*reinterpret_cast<Sim*>(sim)) : -1;
}
long long oracle_step(oracle_sim* sim) { return sim ? reinterpret_cast<Sim*>(sim)->step : -1; }
long long oracle_particle_steps(oracle_sim* sim) {
  return sim ? reinterpret_cast<Sim*>(sim)->particle_steps : -1;
}
void oracle_destroy(oracle_sim* sim) { delete reinterpret_cast<Sim*>(sim); }

/* ---- single functions exposed so the pins can test each part on its own -------------------- */

/* O2 on one body; returns the flag (0, 3 or 4). */
int oracle_kepler_drift(double mu, double* r, double* v, double dt, int iters, double tol) {
  return kepler_drift(mu, r, v, dt, iters, tol);
}

/* O3 kick accelerations in Jacobi coordinates for heliocentric positions q [np][3]. */
int oracle_planet_kick_accel(int np, double gm0, const double* gm, const double* q, double* acc) {
  if (np < 0 || np > kMaxPlanets) return -1;
  std::vector<double> rj(3 * np);
  helio_to_jacobi(np, gm0, gm, q, rj.data());
  planet_kick_accel(np, gm0, gm, q, rj.data(), acc);
  return 0;
}

void oracle_helio_to_jacobi(int np, double gm0, const double* gm, const double* h, double* jac) {
  helio_to_jacobi(np, gm0, gm, h, jac);
}
void oracle_jacobi_to_helio(int np, double gm0, const double* gm, const double* jac, double* h) {
  jacobi_to_helio(np, gm0, gm, jac, h);
}

/* One O3 step on caller arrays. */
int oracle_planet_step(int np, double gm0, const double* gm, double* q, double* qd, double dt) {
  return planet_step(np, gm0, gm, q, qd, dt);
}

/* O1/O5 on one particle: returns the flag, fills a[3] when it is 0. */
int oracle_particle_accel(int np, const double* gm, const double* q, const double* rcrit,
                          double r_min, double r_max, const double* r, double* a) {
  Params P{r_min, std::isfinite(r_max) ? r_max : 0.0, 5, 1e-14, 0};
  std::vector<double> rc2(np);
  for (int j = 0; j < np; ++j) rc2[j] = rcrit ? rcrit[j] * rcrit[j] : 0.0;
  double h0[3];
  common_term_h0(np, gm, q, h0);
  return particle_accel(np, gm, q, h0, rc2.data(), P, r, a);
}

/* Osculating heliocentric elements (a, e, i, Omega, omega, M) of a massless body from (r, v): the
 * quantities the paper logs ("logged orbital elements at a 2048-year interval", PAPER.md:268;
 * periodic output).  Textbook definition (Murray & Dermott, Solar System Dynamics,
 * §2.8): h = r x v, a from the vis-viva integral, the eccentricity vector
 * evec = (v x h)/mu − r/|r|, tan i = |h_xy|/h_z, node vector n = z x h = (−h_y, h_x, 0),
 * Omega = atan2(n_y, n_x), omega = angle from n to evec measured in the orbital plane about h,
 * e cos E = 1 − |r|/a, e sin E = r.v / sqrt(mu a), M = E − e sin E.  Conventions where an angle is
 * undefined: i = 0 (n = 0): Omega = 0 and omega = atan2(evec_y, evec_x); e = 0: omega = 0 and M is
 * the angle from n (or from x when i = 0) to r; unbound (1/a <= 0): M = NaN.  Angles in [0, 2 pi). */
void oracle_elements(double mu, const double* r, const double* v, double* out) {
  const double two_pi = 2.0 * M_PI;
  const double R = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  const double V2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
  const double rv = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
  const double h[3] = {r[1] * v[2] - r[2] * v[1], r[2] * v[0] - r[0] * v[2], r[0] * v[1] - r[1] * v[0]};
  const double H = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
  const double inv_a = 2.0 / R - V2 / mu;
  const double a = 1.0 / inv_a;
  const double ev[3] = {(v[1] * h[2] - v[2] * h[1]) / mu - r[0] / R, (v[2] * h[0] - v[0] * h[2]) / mu - r[1] / R,
                        (v[0] * h[1] - v[1] * h[0]) / mu - r[2] / R};
  const double e = std::sqrt(ev[0] * ev[0] + ev[1] * ev[1] + ev[2] * ev[2]);
  const double n[2] = {-h[1], h[0]};
  const double N = std::sqrt(n[0] * n[0] + n[1] * n[1]);
  const double inc = std::atan2(N, h[2]);  /* tan i = |h_xy| / h_z: acos(h_z/|h|) has no digits left near i = 0 */
  auto wrap = [&](double x) { x = std::fmod(x, two_pi); return x < 0.0 ? x + two_pi : x; };
  /* angle of a vector w in the orbital plane, measured from the node (or from x when i = 0) about h:
   * components along nhat and along hhat x nhat */
  auto in_plane_angle = [&](const double* w) {
    if (N == 0.0) return std::atan2(h[2] >= 0.0 ? w[1] : -w[1], w[0]);
    const double nh[3] = {n[0] / N, n[1] / N, 0.0};
    const double hh[3] = {h[0] / H, h[1] / H, h[2] / H};
    const double m[3] = {hh[1] * nh[2] - hh[2] * nh[1], hh[2] * nh[0] - hh[0] * nh[2], hh[0] * nh[1] - hh[1] * nh[0]};
    return std::atan2(w[0] * m[0] + w[1] * m[1] + w[2] * m[2], w[0] * nh[0] + w[1] * nh[1] + w[2] * nh[2]);
  };
  const double Omega = (N == 0.0) ? 0.0 : wrap(std::atan2(n[1], n[0]));
  double omega, M;
  if (e == 0.0) {
    omega = 0.0;
    M = wrap(in_plane_angle(r));
  } else {
    omega = wrap(in_plane_angle(ev));
    if (inv_a > 0.0) {
      const double ecosE = 1.0 - R / a;
      const double esinE = rv / std::sqrt(mu * a);
      const double E = std::atan2(esinE, ecosE);
      M = wrap(E - esinE);
    } else {
      M = std::numeric_limits<double>::quiet_NaN();
    }
  }
  out[0] = a; out[1] = e; out[2] = inc; out[3] = Omega; out[4] = omega; out[5] = M;
}

/* Resonant argument of the p:q mean-motion resonance with a planet:
 * phi = p lambda − q lambda_pl − (p − q) varpi, lambda = Omega + omega + M, varpi = Omega + omega, from
 * the osculating elements above (the particle's about mu, the planet's about mu_pl = G(m0 + m_pl));
 * returned in [0, 2 pi). */
double oracle_resonant_argument(double mu, const double* r, const double* v, double mu_pl, const double* rp,
                                const double* vp, int p, int q) {
  double el[6], pl[6];
  oracle_elements(mu, r, v, el);
  oracle_elements(mu_pl, rp, vp, pl);
  const double varpi = el[3] + el[4];
  const double lambda = varpi + el[5];
  const double lambda_pl = pl[3] + pl[4] + pl[5];
  double phi = std::fmod(p * lambda - q * lambda_pl - (p - q) * varpi, 2.0 * M_PI);
  if (phi < 0.0) phi += 2.0 * M_PI;
  return phi;
}

/* Libration summary of one particle's sampled resonant argument.
 * phi[0..n) are the samples in [0, 2 pi), in time order.
 *   - window test ("never comes within 10 deg of 0 deg or never within 10 deg of 180 deg"):
 *     seen0 = some sample lies within `window` of 0 (or 2 pi), seen180 = within `window` of pi;
 *   - running extrema: the smallest and largest sample;
 *   - amplitude ("a running window that diagnosed successive maxima and minima of the
 *     resonant angle and measured the difference between them"): sample k (0 < k < n-1) is a turning
 *     point if the series rose into it and falls out of it (a maximum) or fell into it and rises out of
 *     it (a minimum), where "rose / fell into it" looks back past equal neighbours to the last change;
 *     every turning point after the first gives one amplitude sample, half its distance to the turning
 *     point before it.  out = { seen0, seen180, phi_min, phi_max, amp_mean (NaN if none), amp_max (0 if
 *     none), number of amplitude samples }. */
void oracle_libration_summary(const double* phi, long long n, double window, double* out) {
  const double two_pi = 2.0 * M_PI;
  double seen0 = 0.0, seen180 = 0.0;
  double lo = std::numeric_limits<double>::infinity(), hi = -std::numeric_limits<double>::infinity();
  for (long long k = 0; k < n; ++k) {
    const double to_zero = std::min(phi[k], two_pi - phi[k]);
    const double to_pi = std::fabs(phi[k] - M_PI);
    if (to_zero < window) seen0 = 1.0;
    if (to_pi < window) seen180 = 1.0;
    lo = std::min(lo, phi[k]);
    hi = std::max(hi, phi[k]);
  }
  std::vector<double> turning; /* values of the turning points, in time order */
  for (long long k = 1; k + 1 < n; ++k) {
    /* direction of the last change before sample k (0 if the series has been flat so far) */
    int into = 0;
    for (long long j = k; j >= 1 && into == 0; --j) {
      if (phi[j] > phi[j - 1]) into = 1;
      if (phi[j] < phi[j - 1]) into = -1;
    }
    int out_of = 0;
    if (phi[k + 1] > phi[k]) out_of = 1;
    if (phi[k + 1] < phi[k]) out_of = -1;
    if (into != 0 && out_of == -into) turning.push_back(phi[k]);
  }
  double sum = 0.0, largest = 0.0;
  long long count = 0;
  for (size_t t = 1; t < turning.size(); ++t) {
    const double amp = 0.5 * std::fabs(turning[t] - turning[t - 1]);
    sum += amp;
    largest = std::max(largest, amp);
    count += 1;
  }
  out[0] = seen0; out[1] = seen180; out[2] = lo; out[3] = hi;
  out[4] = count > 0 ? sum / static_cast<double>(count) : std::numeric_limits<double>::quiet_NaN();
  out[5] = largest;
  out[6] = static_cast<double>(count);
}

}  // extern "C"
