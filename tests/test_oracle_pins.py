"""Pins for the oracle (oracle/glisse_oracle.cpp) against what the paper and the mathematics fix.

Nothing here retypes the oracle's formulas: each pin is a closed form, an invariant, a brute-force
computation or a claim printed in the paper (DESIGN.md §4 lists which oracle function each pins).
All run without a GPU.
"""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

from paper_2011_03484_b200 import inputs
from tests.orbital import angle_diff, cartesian_to_elements
from tests.orbital import state_from_elements as _state_from_elements

G = inputs.G


def _random_particles(seed, n, a_lo, a_hi, e_max, i_max_deg):
    rng = np.random.default_rng(seed)
    a = rng.uniform(a_lo, a_hi, n)
    e = rng.uniform(0, e_max, n)
    inc = rng.uniform(0, np.radians(i_max_deg), n)
    Om, om, M = (rng.uniform(0, 2 * np.pi, n) for _ in range(3))
    pos, vel = inputs.elements_to_cartesian(G, a, e, inc, Om, om, M)
    return dict(a=a, e=e, inc=inc, Omega=Om, omega=om, M=M), pos, vel


# ---------------------------------------------------------------------------------------------
# T1  two-body closed form: no planets -> the step is a pure Kepler drift (pins O2 entirely)
# ---------------------------------------------------------------------------------------------
def test_T1_two_body_elements_preserved_and_closed_form_position(oracle_mod):
    el, pos, vel = _random_particles(11, 256, 2.0, 70.0, 0.8, 40.0)
    dt, steps = 180.0, 10_000
    S = oracle_mod.OracleSim(G, [], np.zeros((0, 3)), np.zeros((0, 3)), None, pos.T, vel.T, dt)
    S.advance(steps)
    p, v, flag, _ = S.read()
    assert np.all(flag == 0)
    out = cartesian_to_elements(G, p.T, v.T)
    # BASELINE.json north_star: orbital elements preserved to 1e-12 relative over 1e4 steps
    assert np.max(np.abs(out["a"] / el["a"] - 1)) < 1e-12
    assert np.max(np.abs(out["e"] - el["e"])) < 1e-12
    assert np.max(np.abs(out["inc"] - el["inc"])) < 1e-12
    assert np.max(angle_diff(out["Omega"], el["Omega"]) * np.sin(el["inc"])) < 1e-12
    # closed form: M advances by n dt per step, everything else fixed -> position known analytically
    n = np.sqrt(G / el["a"] ** 3)
    pos_ref, vel_ref = inputs.elements_to_cartesian(G, el["a"], el["e"], el["inc"], el["Omega"], el["omega"],
                                                    el["M"] + n * dt * steps)
    # the only error left is along-track: a relative roundoff da/a ~ 1e-13 accumulates a phase error
    # 1.5 (da/a) (n dt steps), seen in position amplified by up to 1/(1-e)^2 near pericentre
    phase = n * dt * steps
    bound = 3e-13 * phase / (1 - el["e"]) ** 2
    err = np.linalg.norm(p.T - pos_ref, axis=1) / np.linalg.norm(pos_ref, axis=1)
    errv = np.linalg.norm(v.T - vel_ref, axis=1) / np.linalg.norm(vel_ref, axis=1)
    assert np.all(err < bound) and np.all(errv < bound)
    far = (el["a"] > 20.0) & (el["e"] < 0.5)  # the paper's regime: < 1e-10 outright
    assert far.sum() > 50 and np.max(err[far]) < 1e-10 and np.max(errv[far]) < 1e-10


def test_T1_single_drift_matches_closed_form_large_steps(oracle_mod):
    """One drift with dM anywhere in (-pi, pi] and beyond 2 pi (reading S9), high e included."""
    rng = np.random.default_rng(5)
    n = 2000
    a = rng.uniform(0.3, 70.0, n)
    e = rng.uniform(0.0, 0.8, n)
    inc = rng.uniform(0, np.pi / 3, n)
    Om, om, M = (rng.uniform(0, 2 * np.pi, n) for _ in range(3))
    pos, vel = inputs.elements_to_cartesian(G, a, e, inc, Om, om, M)
    dt = 180.0
    nn = np.sqrt(G / a ** 3)
    for sign in (+1.0, -1.0):
        pref, vref = inputs.elements_to_cartesian(G, a, e, inc, Om, om, M + sign * nn * dt)
        worst = 0.0
        for i in range(n):
            fl, r1, v1 = oracle_mod.kepler_drift(G, pos[i], vel[i], sign * dt, iters=8, tol=1e-13)
            assert fl == 0
            worst = max(worst, np.linalg.norm(r1 - pref[i]) / np.linalg.norm(pref[i]),
                        np.linalg.norm(v1 - vref[i]) / np.linalg.norm(vref[i]))
        # the closed form itself carries ~ (n dt) eps of phase roundoff (n dt up to ~2e3 rad here)
        assert worst < 5e-12


def test_T1_drift_conserves_energy_and_angular_momentum(oracle_mod):
    _, pos, vel = _random_particles(3, 200, 5.0, 40.0, 0.7, 30.0)
    for i in range(pos.shape[0]):
        fl, r1, v1 = oracle_mod.kepler_drift(G, pos[i], vel[i], 180.0)
        assert fl == 0
        E0 = 0.5 * vel[i] @ vel[i] - G / np.linalg.norm(pos[i])
        E1 = 0.5 * v1 @ v1 - G / np.linalg.norm(r1)
        assert abs(E1 / E0 - 1) < 1e-13
        h0, h1 = np.cross(pos[i], vel[i]), np.cross(r1, v1)
        assert np.linalg.norm(h1 - h0) / np.linalg.norm(h0) < 1e-14


# ---------------------------------------------------------------------------------------------
# T2  single planet: H_int == 0, the planet follows an exact Kepler orbit with mu = G(m0+m1)
# ---------------------------------------------------------------------------------------------
def test_T2_single_planet_is_exact_two_body(oracle_mod):
    m1 = 9.5479e-4
    mu = G * (1 + m1)
    el = dict(a=5.2, e=0.3, inc=0.2, Omega=1.0, omega=2.0, M=0.5)
    q, qd = inputs.elements_to_cartesian(mu, *[np.array([el[k]]) for k in ("a", "e", "inc", "Omega", "omega", "M")])
    acc = oracle_mod.planet_kick_accel(G, [G * m1], q)
    assert np.max(np.abs(acc)) < 1e-20  # the bracket vanishes identically for Np = 1
    dt, steps = 30.0, 5000
    _, pos, vel = _random_particles(1, 1, 20, 21, 0.01, 1)
    S = oracle_mod.OracleSim(G, [G * m1], q, qd, None, pos.T, vel.T, dt)
    S.advance(steps)
    q1, qd1 = S.read_planets()
    n = np.sqrt(mu / el["a"] ** 3)
    qr, qdr = inputs.elements_to_cartesian(mu, [el["a"]], [el["e"]], [el["inc"]], [el["Omega"]], [el["omega"]],
                                           [el["M"] + n * dt * steps])
    assert np.linalg.norm(q1 - qr) / np.linalg.norm(qr) < 1e-10
    assert np.linalg.norm(qd1 - qdr) / np.linalg.norm(qdr) < 1e-10
    out = cartesian_to_elements(mu, q1, qd1)
    assert abs(out["a"][0] / el["a"] - 1) < 1e-12 and abs(out["e"][0] - el["e"]) < 1e-12


# ---------------------------------------------------------------------------------------------
# T3  planet kick = -(1/m'_k) dH_int/dr'_k, by central finite differences of H_int written out here
# ---------------------------------------------------------------------------------------------
def _jacobi_to_helio_np(m0, m, rj):
    eta = m0 + np.cumsum(m)
    q = np.zeros_like(rj)
    for k in range(len(m)):
        q[k] = rj[k] + sum((m[i] / eta[i]) * rj[i] for i in range(k))
    return q


def _H_int(m0, m, rj):
    """H_int / G (masses, not G m) in Jacobi coordinates, O3 / SURVEY S14."""
    q = _jacobi_to_helio_np(m0, m, rj)
    H = 0.0
    for k in range(len(m)):
        H += m[k] * m0 * (1.0 / np.linalg.norm(rj[k]) - 1.0 / np.linalg.norm(q[k]))
    for i in range(len(m)):
        for j in range(i + 1, len(m)):
            H -= m[i] * m[j] / np.linalg.norm(q[i] - q[j])
    return H


@pytest.mark.parametrize("npl", [2, 4, 8])
def test_T3_planet_kick_is_gradient_of_H_int(oracle_mod, npl):
    rng = np.random.default_rng(100 + npl)
    m0 = 1.0
    m = rng.uniform(1e-4, 3e-3, npl)
    a = np.sort(rng.uniform(1.0, 30.0, npl))
    ang = rng.uniform(0, 2 * np.pi, npl)
    q = np.stack([a * np.cos(ang), a * np.sin(ang), rng.uniform(-0.5, 0.5, npl)], axis=1)
    rj = oracle_mod.helio_to_jacobi(m0, m, q)
    # the two coordinate maps are inverse to each other, and agree with the map written out above
    assert np.max(np.abs(oracle_mod.jacobi_to_helio(m0, m, rj) - q)) < 1e-14
    assert np.max(np.abs(_jacobi_to_helio_np(m0, m, rj) - q)) < 1e-14
    # Jacobi position = position relative to the centre of mass of the star and all interior planets
    for k in range(npl):
        com = (m[:k, None] * q[:k]).sum(axis=0) / (m0 + m[:k].sum())
        assert np.max(np.abs(rj[k] - (q[k] - com))) < 1e-14
    acc = oracle_mod.planet_kick_accel(m0, m, q)  # G = 1 units
    eta = m0 + np.cumsum(m)
    eta_prev = np.concatenate([[m0], eta[:-1]])
    mjac = m * eta_prev / eta
    h = 1e-5
    for k in range(npl):
        for c in range(3):
            rp, rm = rj.copy(), rj.copy()
            rp[k, c] += h
            rm[k, c] -= h
            grad = (_H_int(m0, m, rp) - _H_int(m0, m, rm)) / (2 * h)
            ref = -grad / mjac[k]
            assert abs(acc[k, c] - ref) <= 2e-6 * np.max(np.abs(acc[k])) + 1e-13, (k, c, acc[k, c], ref)


# ---------------------------------------------------------------------------------------------
# T4  circular restricted three-body problem: Jacobi constant bounded, error O(dt^2)
# ---------------------------------------------------------------------------------------------
def _jacobi_constant(mu0, mu1, n1, r, v, q1, qd1):
    f = mu1 / (mu0 + mu1)
    rb = r - f * q1
    vb = v - f * qd1
    return (0.5 * np.sum(vb * vb, axis=-1) - mu0 / np.linalg.norm(r, axis=-1)
            - mu1 / np.linalg.norm(r - q1, axis=-1) - n1 * (rb[..., 0] * vb[..., 1] - rb[..., 1] * vb[..., 0]))


def _cr3bp_max_error(oracle_mod, dt, total_days, pos, vel, sample_every, scheme="kdk"):
    m1 = 9.5479e-4
    mu0, mu1 = G, G * m1
    a1 = 5.2
    n1 = np.sqrt((mu0 + mu1) / a1 ** 3)
    q = np.array([[a1, 0.0, 0.0]])
    qd = np.array([[0.0, a1 * n1, 0.0]])
    S = oracle_mod.OracleSim(mu0, [mu1], q, qd, None, pos.T, vel.T, dt, scheme=scheme)
    C0 = _jacobi_constant(mu0, mu1, n1, pos, vel, q[0], qd[0])
    nblocks = int(round(total_days / dt / sample_every))
    errs = []
    for _ in range(nblocks):
        S.advance(sample_every)
        p, v, flag, _ = S.read()
        assert np.all(flag == 0)
        qq, qqd = S.read_planets()
        C = _jacobi_constant(mu0, mu1, n1, p.T, v.T, qq[0], qqd[0])
        errs.append(np.abs(C / C0 - 1))
    return np.array(errs)  # [nblocks, N]


@pytest.mark.parametrize("scheme", ["kdk", "dkd"])
def test_T4_cr3bp_jacobi_constant_bounded_and_second_order(oracle_mod, scheme):
    """Both splittings (kick-drift-kick of PAPER.md:91-95; drift-kick-drift, reading S20) are symplectic
    and of order 2: the same pin holds for each."""
    _, pos, vel = _random_particles(21, 48, 7.5, 12.0, 0.05, 0.0)  # planar, outside the planet
    total = 180.0 * 4000
    e180 = _cr3bp_max_error(oracle_mod, 180.0, total, pos, vel, 100, scheme)
    e90 = _cr3bp_max_error(oracle_mod, 90.0, total, pos, vel, 200, scheme)
    e45 = _cr3bp_max_error(oracle_mod, 45.0, total, pos, vel, 400, scheme)
    m180, m90, m45 = (np.median(e.max(axis=0)) for e in (e180, e90, e45))
    # symplectic: no secular drift -> the maximum over the second half is not larger than ~ the first half's
    half = e180.shape[0] // 2
    first, second = e180[:half].max(axis=0), e180[half:].max(axis=0)
    assert np.median(second / first) < 1.5
    assert m180 < 5e-5
    # second order: error falls by 4 per halving of dt
    assert 3.5 < m180 / m90 < 4.5, (m180, m90)
    assert 3.5 < m90 / m45 < 4.5, (m90, m45)


# ---------------------------------------------------------------------------------------------
# T5  time reversal of the whole map (planets and particles)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", ["kdk", "dkd"])
def test_T5_time_reversal(oracle_mod, scheme):
    w = inputs.config(1)
    _, pos, vel = _random_particles(31, 512, 23.0, 26.0, 0.02, 1.0)  # quiet band between Uranus and Neptune
    n = 1000
    S = oracle_mod.OracleSim(w.gm_star, w.gm_planet, w.planet_pos, w.planet_vel, None, pos.T, vel.T, w.dt,
                             scheme=scheme)
    S.advance(n)
    p1, v1, flag, _ = S.read()
    q1, qd1 = S.read_planets()
    assert np.all(flag == 0)
    B = oracle_mod.OracleSim(w.gm_star, w.gm_planet, q1, qd1, None, p1, v1, -w.dt, scheme=scheme)
    B.advance(n)
    p2, v2, flag2, _ = B.read()
    q2, qd2 = B.read_planets()
    assert np.all(flag2 == 0)
    rel = lambda x, y: np.max(np.linalg.norm(x - y, axis=-1) / np.linalg.norm(y, axis=-1))
    assert rel(q2, w.planet_pos) < 1e-11 and rel(qd2, w.planet_vel) < 1e-11
    # BASELINE.json north_star: recovers the initial state to 1e-11 relative
    assert rel(p2.T, pos) < 1e-11 and rel(v2.T, vel) < 1e-11


# ---------------------------------------------------------------------------------------------
# T6  brute-force direct integration of the heliocentric N-body equations (DOP853, rtol 1e-13):
#     the WH map converges to it at second order, for planets and particles
# ---------------------------------------------------------------------------------------------
def _direct_rhs(gm0, gm, npl, npart):
    def rhs(t, y):
        y = y.reshape(-1, 6)
        q, qd = y[:npl, :3], y[:npl, 3:]
        r, v = y[npl:, :3], y[npl:, 3:]
        out = np.zeros_like(y)
        out[:, :3] = y[:, 3:]
        qn3 = np.linalg.norm(q, axis=1) ** 3
        indirect = -(gm[:, None] * q / qn3[:, None]).sum(axis=0)  # acceleration of the frame (star)
        for i in range(npl):
            acc = -(gm0 + gm[i]) * q[i] / qn3[i] + indirect + gm[i] * q[i] / qn3[i]
            for j in range(npl):
                if j != i:
                    d = q[j] - q[i]
                    acc = acc + gm[j] * d / np.linalg.norm(d) ** 3
            out[i, 3:] = acc
        for k in range(npart):
            acc = -gm0 * r[k] / np.linalg.norm(r[k]) ** 3 + indirect
            for j in range(npl):
                d = q[j] - r[k]
                acc = acc + gm[j] * d / np.linalg.norm(d) ** 3
            out[npl + k, 3:] = acc
        return out.ravel()
    return rhs


@pytest.mark.parametrize("scheme", ["kdk", "dkd"])
def test_T6_second_order_convergence_to_direct_integration(oracle_mod, scheme):
    w = inputs.config(1)
    _, pos, vel = _random_particles(41, 6, 12.0, 27.0, 0.1, 3.0)
    T = 7200.0
    npl, npart = w.n_planets, pos.shape[0]
    y0 = np.concatenate([np.concatenate([w.planet_pos, w.planet_vel], axis=1),
                         np.concatenate([pos, vel], axis=1)], axis=0).ravel()
    sol = solve_ivp(_direct_rhs(w.gm_star, w.gm_planet, npl, npart), (0.0, T), y0, method="DOP853",
                    rtol=1e-13, atol=1e-15)
    yT = sol.y[:, -1].reshape(-1, 6)
    errs_pl, errs_pa = [], []
    for dt in (180.0, 90.0, 45.0, 22.5):
        S = oracle_mod.OracleSim(w.gm_star, w.gm_planet, w.planet_pos, w.planet_vel, None, pos.T, vel.T, dt,
                                 scheme=scheme)
        S.advance(int(round(T / dt)))
        p, v, flag, _ = S.read()
        q, _qd = S.read_planets()
        assert np.all(flag == 0)
        errs_pl.append(np.max(np.linalg.norm(q - yT[:npl, :3], axis=1)))
        errs_pa.append(np.max(np.linalg.norm(p.T - yT[npl:, :3], axis=1)))
    for errs in (errs_pl, errs_pa):
        ratios = [errs[i] / errs[i + 1] for i in range(3)]
        if scheme == "kdk":
            assert all(3.6 < r < 4.4 for r in ratios), (errs, ratios)
        else:
            # drift-kick-drift carries the planets as S(dt/2) S(dt)^(n-1) S(dt/2): still second order, but
            # at dt = 180 d (24 steps per Jupiter orbit) the next term of the error expansion is still
            # visible in the PLANETS' error; its ratio climbs to 4 as dt falls (measured 3.42, 3.77, 3.90; the
            # particles' is 4.00 throughout)
            assert 3.3 < ratios[0] < 4.4 and 3.6 < ratios[1] < 4.4 and 3.8 < ratios[2] < 4.2, (errs, ratios)
    assert errs_pl[-1] < 1e-4 and errs_pa[-1] < 1e-4


# ---------------------------------------------------------------------------------------------
# T7  the paper's solver claim: "5 iterations were sufficient for convergence within
#     1e-14 for ... e < 0.8, 20 au < a < 70 au, dt <= 120 days"
# ---------------------------------------------------------------------------------------------
def test_T7_five_newton_iterations_converge_in_paper_range(oracle_mod):
    rng = np.random.default_rng(7)
    n = 4000
    a = rng.uniform(20.0, 70.0, n)
    e = rng.uniform(0.0, 0.8, n)
    inc = rng.uniform(0, 0.5, n)
    Om, om, M = (rng.uniform(0, 2 * np.pi, n) for _ in range(3))
    pos, vel = inputs.elements_to_cartesian(G, a, e, inc, Om, om, M)
    nn = np.sqrt(G / a ** 3)
    pref, _ = inputs.elements_to_cartesian(G, a, e, inc, Om, om, M + nn * 120.0)
    for i in range(n):
        fl5, r5, _ = oracle_mod.kepler_drift(G, pos[i], vel[i], 120.0, iters=5, tol=1e-14)
        assert fl5 == 0
        fl3, r3, _ = oracle_mod.kepler_drift(G, pos[i], vel[i], 120.0, iters=3, tol=1e-14)
        assert fl3 == 0  # with the guess of reading S5 three already suffice in this range
        assert np.linalg.norm(r5 - pref[i]) / np.linalg.norm(pref[i]) < 2e-14 * max(1.0, 1.0 / (1 - e[i]))
    # and a single update is NOT enough at high eccentricity near pericentre (the count matters)
    p, v = inputs.elements_to_cartesian(G, [30.0], [0.79], [0.1], [0.3], [0.4], [0.01])
    fl1, _, _ = oracle_mod.kepler_drift(G, p[0], v[0], 120.0, iters=1, tol=1e-14)
    assert fl1 == 3


# ---------------------------------------------------------------------------------------------
# T8  removal logic on crafted inputs (O5, readings S8, S11, S12)
# ---------------------------------------------------------------------------------------------
def test_T8_removal_logic(oracle_mod):
    w = inputs.config(1)
    q = w.planet_pos
    rc = w.planet_rcrit
    vcirc = lambda r: np.cross([0, 0, 1.0], r) / np.linalg.norm(r) * np.sqrt(G / np.linalg.norm(r))
    P, V = [], []
    # 0: inside planet 2's sphere at t0
    P.append(q[2] + np.array([0.1, 0.0, 0.0]) * rc[2]); V.append(vcirc(P[-1]))
    # 1: quiet particle
    P.append(np.array([24.5, 0.0, 0.0])); V.append(vcirc(P[-1]))
    # 2: inside r_min (beats everything)
    P.append(np.array([0.005, 0.0, 0.0])); V.append(vcirc(P[-1]))
    # 3: outside r_max
    P.append(np.array([0.0, 1200.0, 0.0])); V.append(vcirc(P[-1]))
    # 4: hyperbolic -> unbound at the first drift
    P.append(np.array([40.0, 0.0, 0.0])); V.append(3.0 * vcirc(P[-1]))
    # 5: e = 0.999 at pericentre, one Newton update -> not converged
    p5, v5 = inputs.elements_to_cartesian(G, [60.0], [0.999], [0.1], [0.3], [0.4], [0.0])
    P.append(p5[0]); V.append(v5[0])
    pos, vel = np.array(P), np.array(V)
    S = oracle_mod.OracleSim(w.gm_star, w.gm_planet, w.planet_pos, w.planet_vel, rc, pos.T, vel.T, w.dt,
                             r_min=0.01, r_max=1000.0, kepler_iters=1)
    # the pericentre distance 0.06 AU of particle 5 must not trip r_min
    S.advance(3)
    p, v, flag, rstep = S.read()
    assert list(flag) == [18, 0, 1, 2, 4, 3]
    assert flag[0] == 16 + 2 and rstep[0] == 0
    assert np.array_equal(p[:, 0], pos[0]) and np.array_equal(v[:, 0], vel[0])  # state untouched (S12)
    assert flag[1] == 0 and rstep[1] == -1
    assert flag[2] == 1 and rstep[2] == 0 and np.array_equal(v[:, 2], vel[2])
    assert flag[3] == 2 and rstep[3] == 0 and np.array_equal(v[:, 3], vel[3])
    assert flag[4] == 4 and rstep[4] == 0
    assert np.array_equal(p[:, 4], pos[4])       # frozen at entry to the drift: position unchanged,
    assert not np.array_equal(v[:, 4], vel[4])   # velocity carries the opening half kick
    assert flag[5] == 3 and rstep[5] == 0
    assert S.active_count() == 1 and S.step() == 3

    # r_min beats an encounter; two overlapping spheres -> lowest planet index (S11)
    fl, _ = oracle_mod.particle_accel(w.gm_planet, q, rc, 50.0, 1000.0, q[1] + 0.01)
    assert fl == 1
    big = rc.copy(); big[1] = 100.0; big[3] = 100.0
    fl, _ = oracle_mod.particle_accel(w.gm_planet, q, big, 0.0, np.inf, q[3] + 0.01)
    assert fl == 16 + 1
    # strict inequality, test on squared distances: exactly on the sphere is not a hit
    q1 = np.array([[3.0, 4.0, 0.0]])
    fl, _ = oracle_mod.particle_accel([1e-3 * G], q1, [5.0], 0.0, np.inf, np.array([6.0, 8.0, 0.0]))
    assert fl == 0
    fl, _ = oracle_mod.particle_accel([1e-3 * G], q1, [5.0], 0.0, np.inf, np.array([6.0, 7.999999, 0.0]))
    assert fl == 16


def test_T8_removal_step_counts_completed_steps(oracle_mod):
    """A particle on a collision course with a planet sphere is flagged at the first force evaluation
    inside it; removal_step = completed steps at that evaluation, position = position at that time."""
    m1 = 1e-3
    mu1 = G * m1
    a1 = 5.0
    n1 = np.sqrt(G * (1 + m1) / a1 ** 3)
    q = np.array([[a1, 0.0, 0.0]])
    qd = np.array([[0.0, a1 * n1, 0.0]])
    # particle on a retrograde circular orbit at the planet's distance, a quarter turn ahead: a head-on
    # approach at 2 n1, sampled every 0.31 AU of relative motion, so the 0.5 AU sphere cannot be missed
    r = a1
    phi = np.pi / 2
    pos = np.array([[r * np.cos(phi), r * np.sin(phi), 0.0]])
    vel = -np.array([[-np.sin(phi), np.cos(phi), 0.0]]) * np.sqrt(G / r)
    rc = np.array([0.5])
    dt = 20.0
    S = oracle_mod.OracleSim(G, [mu1], q, qd, rc, pos.T, vel.T, dt)
    # reference trajectory without the test
    F = oracle_mod.OracleSim(G, [mu1], q, qd, None, pos.T, vel.T, dt)
    hit_step = None
    for s in range(1, 2000):
        F.advance(1)
        p, _, _, _ = F.read()
        qq, _ = F.read_planets()
        if np.linalg.norm(p[:, 0] - qq[0]) < rc[0]:
            hit_step = s
            p_hit = p[:, 0].copy()
            break
    assert hit_step is not None and hit_step > 3
    S.advance(hit_step + 5)
    p, v, flag, rstep = S.read()
    assert flag[0] == 16 and rstep[0] == hit_step
    assert np.array_equal(p[:, 0], p_hit)
    assert S.particle_steps() == hit_step


def test_advance_split_equals_single_advance(oracle_mod):
    w = inputs.config(1).subset(64)
    A = oracle_mod.OracleSim.from_workload(w)
    B = oracle_mod.OracleSim.from_workload(w)
    A.advance(300)
    B.advance(100); B.advance(1); B.advance(199)
    for x, y in zip(A.read(), B.read()):
        assert np.array_equal(x, y)


def test_advance_with_own_log_is_identical(oracle_mod):
    """The planet log carries everything the particles need: feeding the oracle's
    own log back reproduces advance() bit for bit; record layout [q_j..., h0, pad]."""
    w = inputs.config(1).subset(64)
    A = oracle_mod.OracleSim.from_workload(w)
    B = oracle_mod.OracleSim.from_workload(w)
    log = B.planet_log(200)
    assert log.shape == (201, 16)
    assert np.array_equal(log[0, :12].reshape(4, 3), w.planet_pos)
    h0 = -(w.gm_planet[:, None] * w.planet_pos / np.linalg.norm(w.planet_pos, axis=1)[:, None] ** 3).sum(axis=0)
    assert np.allclose(log[0, 12:15], h0, rtol=1e-14, atol=0)
    A.advance(200)
    B.advance_with_log(200, log)
    for x, y in zip(A.read(), B.read()):
        assert np.array_equal(x, y)
    qa, _ = A.read_planets()
    assert np.array_equal(log[200, :12].reshape(4, 3), qa)


def test_dkd_removal_semantics_split_invariance_and_own_log(oracle_mod):
    """Drift-kick-drift (reading S20): hand-worked removal cases, split-advance identity, and
    advance_with_log on the scheme's own half-step planet log."""
    w = inputs.config(1)
    q, rc = w.planet_pos, w.planet_rcrit
    pos, vel = w.pos[:, :8].copy(), w.vel[:, :8].copy()
    # particle 0: unbound at t0 -> the first half drift refuses it: flag 4, step 0, state untouched
    vel[:, 0] *= 1.2 * np.sqrt(2.0 * w.gm_star / np.linalg.norm(pos[:, 0])) / np.linalg.norm(vel[:, 0])
    # particle 1: far outside r_max -> caught at the first force evaluation (after half a drift): flag 2,
    # step 0, frozen at t_{1/2}: position moved, the velocity of a pure Kepler half drift (no kick)
    pos[:, 1] = [900.0, 500.0, 0.0]
    vel[:, 1] = np.sqrt(w.gm_star / np.hypot(900.0, 500.0)) * np.array([-500.0, 900.0, 0.0]) / np.hypot(900.0, 500.0)
    S = oracle_mod.OracleSim(w.gm_star, w.gm_planet, q, w.planet_vel, rc, pos, vel, w.dt, r_min=1.0, r_max=1000.0,
                             scheme="dkd")
    S.advance(3)
    p, v, f, r = S.read()
    assert f[0] == 4 and r[0] == 0 and np.array_equal(p[:, 0], pos[:, 0]) and np.array_equal(v[:, 0], vel[:, 0])
    fl, r_half, v_half = oracle_mod.kepler_drift(w.gm_star, pos[:, 1], vel[:, 1], 0.5 * w.dt)
    assert fl == 0 and f[1] == 2 and r[1] == 0
    assert np.array_equal(p[:, 1], r_half) and np.array_equal(v[:, 1], v_half)
    assert (f[2:] == 0).all() and S.particle_steps() == 2 + 6 * 3     # two particles started one step each
    # split advances and the scheme's own log
    A = oracle_mod.OracleSim.from_workload(w, scheme="dkd")
    A.advance(150)
    B = oracle_mod.OracleSim.from_workload(w, scheme="dkd")
    B.advance(70); B.advance(0); B.advance(80)
    C = oracle_mod.OracleSim.from_workload(w, scheme="dkd")
    log = C.planet_log(150)
    C.advance_with_log(150, log)
    for x, y, z in zip(A.read(), B.read(), C.read()):
        assert np.array_equal(x, y) and np.array_equal(x, z)
    qa, qda = A.read_planets()
    qb, qdb = B.read_planets()
    assert np.array_equal(qa, qb) and np.array_equal(qda, qdb)
    # the log's records are the planets at the half steps: record 0 = one Wisdom-Holman step of dt/2
    st, q_half, _ = oracle_mod.planet_step(w.gm_star, w.gm_planet, w.planet_pos, w.planet_vel, 0.5 * w.dt)
    assert st == 0 and np.array_equal(log[0, :12].reshape(4, 3), q_half)
    # no planets at all: D(dt/2) D(dt/2) is the same Kepler flow as D(dt) to roundoff, so both schemes agree
    K = oracle_mod.OracleSim(w.gm_star, [], np.zeros((0, 3)), np.zeros((0, 3)), None, w.pos, w.vel, w.dt)
    D = oracle_mod.OracleSim(w.gm_star, [], np.zeros((0, 3)), np.zeros((0, 3)), None, w.pos, w.vel, w.dt, scheme="dkd")
    K.advance(100); D.advance(100)
    pk, pd = K.read()[0], D.read()[0]
    assert np.max(np.linalg.norm(pk - pd, axis=0) / np.linalg.norm(pk, axis=0)) < 1e-12


# ---------------------------------------------------------------------------------------------------
# T9  osculating elements (snapshot output) against the textbook construction
# ---------------------------------------------------------------------------------------------------
def test_T9_elements_match_textbook_construction(oracle_mod):
    mu = inputs.G
    rng = np.random.default_rng(9)
    worst = 0.0
    for _ in range(400):
        a, e = rng.uniform(0.5, 80.0), rng.uniform(0.01, 0.9)
        inc, Om, om, f = rng.uniform(0.05, 3.0), *rng.uniform(0.0, 2.0 * np.pi, 3)
        r, v, M = _state_from_elements(mu, a, e, inc, Om, om, f)
        el = oracle_mod.elements(mu, r[:, None], v[:, None])[:, 0]
        worst = max(worst, abs(el[0] / a - 1.0), abs(el[1] - e), abs(el[2] - inc),
                    abs(angle_diff(el[3], Om)) * np.sin(inc), abs(angle_diff(el[4], om)) * e * np.sin(inc),
                    abs(angle_diff(el[5], M)) * e)
    assert worst < 5e-13, worst


def test_T9_elements_special_cases_and_drift_invariance(oracle_mod):
    mu = inputs.G
    a, e = 30.0, 0.25
    # pericentre on the x axis of an equatorial orbit: (a, e, 0, 0, 0, 0)
    r = np.array([a * (1 - e), 0.0, 0.0])
    v = np.array([0.0, np.sqrt(mu * (1 + e) / (a * (1 - e))), 0.0])
    el = oracle_mod.elements(mu, r[:, None], v[:, None])[:, 0]
    assert abs(el[0] - a) < 1e-12 and abs(el[1] - e) < 1e-14 and el[2] == 0.0 and el[3] == 0.0
    assert min(el[4], 2 * np.pi - el[4]) < 1e-14 and min(el[5], 2 * np.pi - el[5]) < 1e-14
    # circular equatorial orbit a quarter turn on: omega = 0 by convention, M = the longitude
    r = np.array([0.0, 7.0, 0.0])
    v = np.array([-np.sqrt(mu / 7.0), 0.0, 0.0])
    el = oracle_mod.elements(mu, r[:, None], v[:, None])[:, 0]
    assert abs(el[0] - 7.0) < 1e-12 and el[1] < 1e-15 and el[2] == 0.0 and el[3] == 0.0
    assert abs(el[4] + el[5] - np.pi / 2) < 1e-12 or abs(el[4] + el[5] - np.pi / 2 - 2 * np.pi) < 1e-12
    # retrograde: i = pi
    el = oracle_mod.elements(mu, r[:, None], -v[:, None])[:, 0]
    assert abs(el[2] - np.pi) < 1e-15
    # hyperbolic: a < 0, e > 1, M undefined
    el = oracle_mod.elements(mu, r[:, None], 2.0 * v[:, None])[:, 0]
    assert el[0] < 0 and el[1] > 1 and np.isnan(el[5])
    # under the oracle's own two-body drift a, e, i, Omega, omega stay and M advances by n dt
    r0, v0, M0 = _state_from_elements(mu, 25.0, 0.3, 0.4, 1.0, 2.0, 0.7)
    fl, r1, v1 = oracle_mod.kepler_drift(mu, r0, v0, 180.0)
    assert fl == 0
    e0 = oracle_mod.elements(mu, r0[:, None], v0[:, None])[:, 0]
    e1 = oracle_mod.elements(mu, r1[:, None], v1[:, None])[:, 0]
    assert np.allclose(e0[:5], e1[:5], rtol=0, atol=2e-13)
    n = np.sqrt(mu / 25.0 ** 3)
    assert abs(angle_diff(e1[5], e0[5] + n * 180.0)) < 1e-12


# ---------------------------------------------------------------------------------------------------
# T10  resonant argument against its formula on constructed states, and constant
#      at exact commensurability
# ---------------------------------------------------------------------------------------------------
def test_T10_resonant_argument(oracle_mod):
    mu, mu_pl = inputs.G, inputs.G * (1.0 + 5.1514e-5)
    rng = np.random.default_rng(10)
    for p, q in ((3, 1), (5, 2), (3, 2)):
        for _ in range(100):
            e, inc, Om, om, f = rng.uniform(0.05, 0.6), rng.uniform(0.1, 1.0), *rng.uniform(0, 2 * np.pi, 3)
            r, v, M = _state_from_elements(mu, 62.6, e, inc, Om, om, f)
            ep, ip, Op, wp, fp = 0.01, 0.03, *rng.uniform(0, 2 * np.pi, 3)
            rp, vp, Mp = _state_from_elements(mu_pl, 30.1, ep, ip, Op, wp, fp)
            phi = oracle_mod.resonant_argument(mu, r[:, None], v[:, None], mu_pl, rp, vp, p, q)[0]
            want = (p * (Om + om + M) - q * (Op + wp + Mp) - (p - q) * (Om + om)) % (2 * np.pi)
            assert angle_diff(phi, want) < 1e-10 / ep, (p, q)
    # exact 3:1 commensurability, no interaction: phi-dot = 3 n − n_pl = 0, so phi stays put while both
    # bodies run round their Kepler orbits under the oracle's drift
    a_pl = 30.1
    a = a_pl * (3.0 ** 2 * mu / mu_pl) ** (1.0 / 3.0)      # 3 sqrt(mu/a^3) = sqrt(mu_pl/a_pl^3)
    r, v, _ = _state_from_elements(mu, a, 0.3, 0.2, 1.0, 2.0, 0.5)
    rp, vp, _ = _state_from_elements(mu_pl, a_pl, 0.01, 0.03, 0.3, 0.7, 4.0)
    phi0 = oracle_mod.resonant_argument(mu, r[:, None], v[:, None], mu_pl, rp, vp, 3, 1)[0]
    for _ in range(200):
        _, r, v = oracle_mod.kepler_drift(mu, r, v, 180.0)
        _, rp, vp = oracle_mod.kepler_drift(mu_pl, rp, vp, 180.0)
    phi1 = oracle_mod.resonant_argument(mu, r[:, None], v[:, None], mu_pl, rp, vp, 3, 1)[0]
    assert angle_diff(phi1, phi0) < 1e-9


# ---------------------------------------------------------------------------------------------------
# T11  libration summary (PAPER.md:264 window test, PAPER.md:288 amplitude from successive extrema)
#      against constructed librators (closed form) and hand-worked series
# ---------------------------------------------------------------------------------------------------
def test_T11_libration_summary_on_constructed_series(oracle_mod):
    window = np.deg2rad(10.0)
    # phi(t) = pi + A sin(w t), m samples per period: the turning points are the samples nearest the
    # true extrema, at most half a sample away, so every amplitude sample lies in [A cos(pi/m), A]
    for A, m, periods in ((1.0, 40, 6.3), (0.3, 25, 11.5), (2.9, 64, 4.2)):
        k = np.arange(int(m * periods))
        phi = np.pi + A * np.sin(2.0 * np.pi * k / m + 0.4)
        r = oracle_mod.libration_summary(phi, window)
        shrink = np.cos(np.pi / m)
        assert A * shrink <= r["amp_mean"] <= A and A * shrink <= r["amp_max"] <= A
        assert np.pi - A <= r["phi_min"] <= np.pi - A * shrink and np.pi + A * shrink <= r["phi_max"] <= np.pi + A
        # one turning point per half period (phase 0.4: the first lies (pi/2 - 0.4)/(2 pi) of a period in)
        n_turn = int(np.floor(2.0 * (periods - 1.0 / m - (np.pi / 2 - 0.4) / (2 * np.pi)))) + 1
        assert r["n_amp"] == n_turn - 1
        assert bool(r["seen180"]) and bool(r["seen0"]) == (A > np.pi - window)
    # hand-worked: rises to 3 (max), falls to 1 (min), rises through a plateau to 3 (max), falls
    r = oracle_mod.libration_summary(np.array([1.0, 2.0, 3.0, 2.0, 1.0, 2.0, 2.0, 3.0, 1.0]), 0.05)
    assert r["n_amp"] == 2 and r["amp_mean"] == 1.0 and r["amp_max"] == 1.0
    assert r["phi_min"] == 1.0 and r["phi_max"] == 3.0 and not r["seen0"] and not r["seen180"]
    # a plateau at the top counts once, with the plateau's value; unequal swings average
    r = oracle_mod.libration_summary(np.array([1.0, 3.0, 3.0, 0.5, 2.5, 2.0]), 0.05)
    assert r["n_amp"] == 2 and r["amp_mean"] == 0.5 * (1.25 + 1.0) and r["amp_max"] == 1.25
    # monotonic: no turning point, no amplitude
    r = oracle_mod.libration_summary(np.linspace(0.5, 3.0, 30), 0.05)
    assert r["n_amp"] == 0 and np.isnan(r["amp_mean"]) and r["amp_max"] == 0.0
    # circulation: phi = 0.3 k mod 2 pi wraps every ~21 samples; each wrap is a maximum just below 2 pi
    # followed at once by a minimum just above 0, so every amplitude sample is close to pi
    phi = np.mod(0.3 * np.arange(200), 2 * np.pi)
    r = oracle_mod.libration_summary(phi, window)
    assert r["seen0"] and r["seen180"] and r["n_amp"] >= 15
    assert np.pi - 0.3 <= r["amp_mean"] <= np.pi and r["amp_max"] <= np.pi
    # window edges are strict: a sample exactly `window` from pi does not count
    r = oracle_mod.libration_summary(np.array([np.pi + 0.25, np.pi - 0.25]), 0.25)
    assert not r["seen180"]
    r = oracle_mod.libration_summary(np.array([np.pi + 0.2499]), 0.25)
    assert r["seen180"] and not r["seen0"]
    r = oracle_mod.libration_summary(np.array([2 * np.pi - 0.1]), 0.25)
    assert r["seen0"]


# ---------------------------------------------------------------------------------------------------
# T12  planet log interpolated from a sparse history (reading S24):
#      exact on cubics, the Hermite error bound on a circular orbit, the samples themselves, h0's formula
# ---------------------------------------------------------------------------------------------------
def test_T12_interpolated_planet_log(oracle_mod):
    rng = np.random.default_rng(12)
    npl = 3
    gm = np.array([3e-7, 1e-6, 2.5e-7])
    stride = 3 * (npl + 1) + ((3 * (npl + 1)) & 1)

    def h0_of(q):   # PAPER.md:111, typed out
        return -sum(gm[j] * q[j] / np.linalg.norm(q[j]) ** 3 for j in range(npl))

    # (a) cubic Hermite interpolation reproduces any cubic exactly: q_j(t) = c0 + c1 t + c2 t^2 + c3 t^3
    c = rng.uniform(-1.0, 1.0, (4, npl, 3)) + np.array([3.0, 0.0, 0.0, 0.0])[:, None, None]
    ts = np.array([0.0, 0.7, 1.1, 2.5, 2.9, 4.0])          # unequal spacing
    poly = lambda t: c[0] + c[1] * t + c[2] * t ** 2 + c[3] * t ** 3
    dpoly = lambda t: c[1] + 2 * c[2] * t + 3 * c[3] * t ** 2
    q = np.array([poly(t) for t in ts]); v = np.array([dpoly(t) for t in ts])
    t_first, dtr, n = 0.05, 0.0393, 100
    log = oracle_mod.interpolate_log(gm, ts, q, v, t_first, dtr, n)
    assert log.shape == (n, stride)
    for r in range(n):
        t = t_first + r * dtr
        want = poly(t)
        assert np.max(np.abs(log[r, :3 * npl].reshape(npl, 3) - want)) <= 2e-14 * np.max(np.abs(want))
        assert np.allclose(log[r, 3 * npl:3 * npl + 3], h0_of(log[r, :3 * npl].reshape(npl, 3)), rtol=1e-14, atol=0)
        assert np.all(log[r, 3 * npl + 3:] == 0.0)
    # (b) at the sample instants it returns the samples (both ends of the history included)
    log = oracle_mod.interpolate_log(gm, ts[[0, 3, 5]], q[[0, 3, 5]], v[[0, 3, 5]], 0.0, 2.5, 2)
    assert np.array_equal(log[0, :3 * npl], q[0].ravel()) and np.allclose(log[1, :3 * npl], q[3].ravel(), rtol=1e-15)
    log = oracle_mod.interpolate_log(gm, ts, q, v, 4.0, 1.0, 1)
    assert np.allclose(log[0, :3 * npl], q[5].ravel(), rtol=1e-15)
    # (c) a circular orbit of radius a and mean motion w sampled every D: the error of cubic Hermite
    # interpolation is bounded by D^4 max|q''''| / 384 = a (w D)^4 / 384, and is not far below it
    a, w = 5.2, 2 * np.pi / 4332.6
    for D in (120.0, 240.0, 480.0):
        ts = np.arange(0.0, 4000.0, D)
        circ = lambda t: np.array([[a * np.cos(w * t), a * np.sin(w * t), 0.0]])
        dcirc = lambda t: np.array([[-a * w * np.sin(w * t), a * w * np.cos(w * t), 0.0]])
        q = np.array([circ(t) for t in ts]); v = np.array([dcirc(t) for t in ts])
        tt = np.arange(0.0, ts[-1], 7.3)
        log = oracle_mod.interpolate_log(gm[:1], ts, q, v, 0.0, 7.3, len(tt))
        err = max(np.linalg.norm(log[r, :3] - circ(t)[0]) for r, t in enumerate(tt))
        bound = a * (w * D) ** 4 / 384.0
        assert 0.3 * bound <= err <= 1.0001 * bound * np.sqrt(2.0), (D, err, bound)   # two components, each bounded
    # (d) refusals: a time outside the history, samples out of order
    for bad in (dict(t_first=-0.1), dict(t_first=3999.0, n=200)):
        with pytest.raises(ValueError):
            oracle_mod.interpolate_log(gm[:1], ts, q, v, bad.get("t_first", 0.0), 7.3, bad.get("n", 3))
    with pytest.raises(ValueError):
        oracle_mod.interpolate_log(gm[:1], ts[::-1], q, v, 0.0, 7.3, 3)
