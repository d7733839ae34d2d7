"""Host-side checks of the seeded workload generators (no GPU, no oracle)."""
import numpy as np

from paper_2011_03484_b200 import inputs
from tests.orbital import angle_diff, cartesian_to_elements


def test_elements_roundtrip():
    rng = np.random.default_rng(0)
    n = 500
    a = rng.uniform(0.4, 70, n)
    e = rng.uniform(0.01, 0.9, n)
    inc = rng.uniform(0.01, 3.0, n)
    Om, om, M = (rng.uniform(0, 2 * np.pi, n) for _ in range(3))
    pos, vel = inputs.elements_to_cartesian(inputs.G, a, e, inc, Om, om, M)
    out = cartesian_to_elements(inputs.G, pos, vel)
    assert np.max(np.abs(out["a"] / a - 1)) < 1e-12
    assert np.max(np.abs(out["e"] - e)) < 1e-12
    assert np.max(np.abs(out["inc"] - inc)) < 1e-10
    assert np.max(angle_diff(out["Omega"], Om)) < 1e-9
    assert np.max(angle_diff(out["omega"], om)) < 1e-8
    assert np.max(angle_diff(out["M"], M)) < 1e-8


def test_hill_radii_formula():
    # R_H = a_p (m_p / 3 m_0)^(1/3); values for the four giants at the nominal a of
    # BASELINE.json configs[0], worked by hand from the formula
    rh = inputs.hill_radius(inputs.GIANT_A, inputs.GIANT_MASS)
    assert np.allclose(rh, [0.355030, 0.436210, 0.468772, 0.776547], atol=5e-7)


def test_configs_shapes_and_distributions():
    for c, (n, alo, ahi, emax, np_) in {1: (1024, 20, 28, 0.05, 4), 2: (131072, 20, 28, 0.02, 4),
                                        4: (4096, 2, 50, 0.2, 8)}.items():
        w = inputs.config(c, n_particles=n)
        assert w.pos.shape == (3, n) and w.vel.shape == (3, n) and w.n_planets == np_
        assert w.pos.flags.c_contiguous and w.pos.dtype == np.float64
        el = cartesian_to_elements(w.gm_star, w.pos.T, w.vel.T)
        assert alo - 1e-9 <= el["a"].min() and el["a"].max() <= ahi + 1e-9
        assert el["e"].max() <= emax + 1e-9
        # planets are in Jacobi order (increasing distance)
        assert np.all(np.diff(np.linalg.norm(w.planet_pos, axis=1)) > 0)
    # seeded: same call, same bits
    a, b = inputs.config(1), inputs.config(1)
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.planet_vel, b.planet_vel)


def test_shard_range_partitions_exactly():
    for n in (1, 7, 1024, 1_048_577):
        for world in (1, 2, 3, 8):
            spans = [inputs.shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
