"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json `configs`).

This module is the ONLY code shared by the oracle side (tests, cpu_baseline) and the CUDA side
(binding, bench).  It holds none of the integrator's arithmetic: it draws orbital elements from
the distributions BASELINE.json states and turns them into heliocentric Cartesian vectors with
the textbook two-body element -> state map.  It imports neither `oracle/` nor the CUDA binding.

The paper's own initial conditions are not available (PAPER.md:183, 262-268 describe them but
give no files); these inputs stand in for them.  Recipe:
  rng = numpy.random.default_rng([201103484, c, k])   c = config 1..5, k = 0 planets, 1 particles
  whole vectors drawn in the order a, e, i, Omega, omega, M;  angles ~ U[0, 2pi)
  planets:  mu = G (m0 + m_p);   particles:  mu = G m0;   G = k^2 (Gaussian constant), m0 = 1.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

#: Gaussian gravitational constant squared, AU^3 Msun^-1 day^-2 (the paper never states units;
#: DESIGN.md reading S2).
G = 0.01720209895 ** 2

SEED = 201103484

GIANT_MASS = (9.5479e-4, 2.8589e-4, 4.3662e-5, 5.1514e-5)      # BASELINE.json configs[0]
GIANT_A = (5.20, 9.55, 19.2, 30.1)
# BASELINE.json configs[3] gives only the ends of the 8-planet system; the fill is DESIGN.md §3.
EIGHT_MASS = (1.66e-7, 2.45e-6, 3.00e-6, 3.23e-7) + GIANT_MASS
EIGHT_A = (0.39, 0.72, 1.00, 1.52) + GIANT_A


@dataclasses.dataclass
class Workload:
    """One seeded problem instance; arrays are float64, C-contiguous."""
    name: str
    gm_star: float
    gm_planet: np.ndarray      # [Np]
    planet_pos: np.ndarray     # [Np,3] heliocentric
    planet_vel: np.ndarray     # [Np,3]
    planet_rcrit: np.ndarray   # [Np] absolute encounter radii (1 Hill radius at nominal a)
    pos: np.ndarray            # [3,N]  struct-of-arrays
    vel: np.ndarray            # [3,N]
    dt: float
    steps: int                 # BASELINE.json's step count for the config
    r_min: float
    r_max: float
    chunk_steps: int = 1024

    @property
    def n_particles(self) -> int:
        return self.pos.shape[1]

    @property
    def n_planets(self) -> int:
        return self.gm_planet.shape[0]

    def subset(self, n: int) -> "Workload":
        """The first n particles with the full planet system (particles are independent)."""
        return dataclasses.replace(self, pos=np.ascontiguousarray(self.pos[:, :n]),
                                   vel=np.ascontiguousarray(self.vel[:, :n]))


def solve_kepler_elliptic(M: np.ndarray, e: np.ndarray) -> np.ndarray:
    """Eccentric anomaly E with E - e sin E = M, by bisection-safeguarded Newton (input prep only)."""
    M = np.mod(M, 2.0 * np.pi)
    E = np.where(e < 0.8, M, np.pi * np.ones_like(M))
    lo = np.zeros_like(M)
    hi = 2.0 * np.pi * np.ones_like(M)
    for _ in range(80):
        f = E - e * np.sin(E) - M
        lo = np.where(f < 0, E, lo)
        hi = np.where(f > 0, E, hi)
        En = E - f / (1.0 - e * np.cos(E))
        bad = (En <= lo) | (En >= hi)
        En = np.where(bad, 0.5 * (lo + hi), En)
        if np.all(np.abs(En - E) <= 1e-16 * np.maximum(1.0, np.abs(E))):
            E = En
            break
        E = En
    return E


def elements_to_cartesian(mu, a, e, inc, Omega, omega, M):
    """Heliocentric position/velocity [n,3] from osculating elements (Murray & Dermott §2.8)."""
    a, e, inc, Omega, omega, M = (np.asarray(t, dtype=np.float64) for t in (a, e, inc, Omega, omega, M))
    E = solve_kepler_elliptic(M, e)
    cE, sE = np.cos(E), np.sin(E)
    b = a * np.sqrt(1.0 - e * e)
    n = np.sqrt(mu / a ** 3)
    # in-plane coordinates, pericentre along +x
    xp = a * (cE - e)
    yp = b * sE
    rr = a * (1.0 - e * cE)
    vxp = -a * a * n * sE / rr
    vyp = a * b * n * cE / rr
    cO, sO = np.cos(Omega), np.sin(Omega)
    co, so = np.cos(omega), np.sin(omega)
    ci, si = np.cos(inc), np.sin(inc)
    # rotation R_z(Omega) R_x(i) R_z(omega)
    r11 = cO * co - sO * so * ci
    r12 = -cO * so - sO * co * ci
    r21 = sO * co + cO * so * ci
    r22 = -sO * so + cO * co * ci
    r31 = so * si
    r32 = co * si
    pos = np.stack([r11 * xp + r12 * yp, r21 * xp + r22 * yp, r31 * xp + r32 * yp], axis=-1)
    vel = np.stack([r11 * vxp + r12 * vyp, r21 * vxp + r22 * vyp, r31 * vxp + r32 * vyp], axis=-1)
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel)


def hill_radius(a_p, m_p, m_0=1.0, k=1.0):
    """R_H = a_p (m_p / 3 m_0)^(1/3); k = multiplier."""
    return k * np.asarray(a_p) * (np.asarray(m_p) / (3.0 * m_0)) ** (1.0 / 3.0)


def _planets(c: int, masses, a_nom, e_max: float, i_max_deg: float, m0: float = 1.0):
    rng = np.random.default_rng([SEED, c, 0])
    npl = len(masses)
    m = np.asarray(masses, dtype=np.float64)
    a = np.asarray(a_nom, dtype=np.float64)
    e = rng.uniform(0.0, e_max, npl)
    inc = rng.uniform(0.0, math.radians(i_max_deg), npl)
    Om = rng.uniform(0.0, 2 * np.pi, npl)
    om = rng.uniform(0.0, 2 * np.pi, npl)
    M = rng.uniform(0.0, 2 * np.pi, npl)
    pos, vel = elements_to_cartesian(G * (m0 + m), a, e, inc, Om, om, M)
    return G * m, pos, vel, hill_radius(a, m, m0)


def _particles(c: int, n: int, a_lo, a_hi, e_max, i_max_deg, m0: float = 1.0):
    rng = np.random.default_rng([SEED, c, 1])
    a = rng.uniform(a_lo, a_hi, n)
    e = rng.uniform(0.0, e_max, n)
    inc = rng.uniform(0.0, math.radians(i_max_deg), n)
    Om = rng.uniform(0.0, 2 * np.pi, n)
    om = rng.uniform(0.0, 2 * np.pi, n)
    M = rng.uniform(0.0, 2 * np.pi, n)
    pos, vel = elements_to_cartesian(G * m0, a, e, inc, Om, om, M)
    return np.ascontiguousarray(pos.T), np.ascontiguousarray(vel.T)


#: (name, planets(masses, a, e_max, i_max), particles(N, a_lo, a_hi, e_max, i_max), dt, steps)
_CONFIGS = {
    1: ("c1: 4 giants, 1,024 particles a~U[20,28]", (GIANT_MASS, GIANT_A, 0.05, 1.0),
        (1024, 20.0, 28.0, 0.05, 2.0), 180.0, 10_000),
    2: ("c2: 4 giants, 131,072 particles a~U[20,28]", (GIANT_MASS, GIANT_A, 0.05, 1.0),
        (131_072, 20.0, 28.0, 0.02, 1.0), 180.0, 100_000),
    3: ("c3: 4 giants, 262,144 resonant-TNO-like particles a~U[53,65]", (GIANT_MASS, GIANT_A, 0.05, 1.0),
        (262_144, 53.0, 65.0, 0.4, 20.0), 180.0, 100_000),
    4: ("c4: 8 planets, 1,048,576 particles a~U[2,50], dt=4d", (EIGHT_MASS, EIGHT_A, 0.1, 1.0),
        (1_048_576, 2.0, 50.0, 0.2, 10.0), 4.0, 20_000),
    5: ("c5: 4 giants, 4,194,304 planet-crossing particles a~U[5,35]", (GIANT_MASS, GIANT_A, 0.05, 1.0),
        (4_194_304, 5.0, 35.0, 0.5, 30.0), 180.0, 50_000),
}


def config(c: int, n_particles: int | None = None) -> Workload:
    """BASELINE.json configs[c-1] (c = 1..5).  n_particles overrides N (same seed, so the first
    particles of a smaller draw are NOT a prefix of a larger one; use Workload.subset for that)."""
    name, (pm, pa, pe, pi_), (n, alo, ahi, emax, imax), dt, steps = _CONFIGS[c]
    if n_particles is not None:
        n = int(n_particles)
    gm, ppos, pvel, rcrit = _planets(c, pm, pa, pe, pi_)
    pos, vel = _particles(c, n, alo, ahi, emax, imax)
    return Workload(name=name, gm_star=G * 1.0, gm_planet=gm, planet_pos=ppos, planet_vel=pvel,
                    planet_rcrit=rcrit, pos=pos, vel=vel, dt=dt, steps=steps, r_min=1.0, r_max=1000.0)


def one_m_four_planets(n_particles: int = 1_048_576) -> Workload:
    """BASELINE.json north_star's target workload: '1M particles x 4 planets' — the 4-giant system
    with config 2's particle distribution (the paper's Fig. 2 benchmark shape),
    at N = 2^20."""
    name, (pm, pa, pe, pi_), (_, alo, ahi, emax, imax), dt, steps = _CONFIGS[2]
    gm, ppos, pvel, rcrit = _planets(2, pm, pa, pe, pi_)
    pos, vel = _particles(2, n_particles, alo, ahi, emax, imax)
    return Workload(name=f"1M x 4 planets: 4 giants, {n_particles:,} particles a~U[20,28]",
                    gm_star=G, gm_planet=gm, planet_pos=ppos, planet_vel=pvel, planet_rcrit=rcrit,
                    pos=pos, vel=vel, dt=dt, steps=steps, r_min=1.0, r_max=1000.0)


def chain_system(n_planets: int, n_particles: int = 2048, dt: float = 5.0) -> Workload:
    """A seeded system with ANY planet count 0..32, for the code paths BASELINE.json's two planet
    counts (4 and 8) do not reach: planets on a geometric ladder a_k = 1.5 rho^k AU out to 40 AU (rho
    capped at 1.35), equal masses chosen so that neighbours sit 12 mutual Hill radii apart
    (m = 1.5 ((rho - 1) / 12)^3, capped at 1e-4), e ~ U[0, 0.02], i ~ U[0, 1 deg]; particles
    a ~ U[1.2, 1.2 a_last], e ~ U[0, 0.1], i ~ U[0, 5 deg], angles uniform; dt = 5 d (134 steps per
    orbit of the innermost planet, so that the 1,000-step parity horizon is 7 of its orbits and the
    roundoff sensitivity of most particles stays below 1e-12); removal at r < 0.3 AU, r > 1000 AU, 1 Hill radius."""
    npl = int(n_planets)
    rho = min(1.35, (40.0 / 1.5) ** (1.0 / max(npl - 1, 1)))
    mass = min(1e-4, 1.5 * ((rho - 1.0) / 12.0) ** 3)
    a_nom = 1.5 * rho ** np.arange(npl)
    c = 100 + npl
    gm, ppos, pvel, rcrit = _planets(c, [mass] * npl, a_nom, 0.02, 1.0)
    a_hi = 1.2 * (a_nom[-1] if npl else 40.0)
    pos, vel = _particles(c, n_particles, 1.2, a_hi, 0.1, 5.0)
    return Workload(name=f"chain: {npl} planets a = 1.5 x {rho:.4f}^k AU, m = {mass:.3g}, {n_particles} particles",
                    gm_star=G, gm_planet=gm.reshape(npl), planet_pos=ppos.reshape(npl, 3),
                    planet_vel=pvel.reshape(npl, 3), planet_rcrit=np.asarray(rcrit, dtype=np.float64).reshape(npl),
                    pos=pos, vel=vel, dt=dt, steps=1000, r_min=0.3, r_max=1000.0)


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous particle slice [lo, hi) of rank `rank` out of `world` (particles never interact,
    PAPER.md:27,35: planets are replicated, particles partitioned, no exchange)."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
