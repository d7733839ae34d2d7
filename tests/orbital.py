"""Textbook two-body helpers used by the pins (independent of oracle/ and of the CUDA path)."""
import numpy as np


def cartesian_to_elements(mu, r, v):
    """r, v: [...,3] -> dict of a, e, inc, Omega, omega, M (Murray & Dermott §2.8)."""
    r = np.asarray(r, dtype=np.float64)
    v = np.asarray(v, dtype=np.float64)
    rn = np.linalg.norm(r, axis=-1)
    v2 = np.sum(v * v, axis=-1)
    h = np.cross(r, v)
    hn = np.linalg.norm(h, axis=-1)
    a = 1.0 / (2.0 / rn - v2 / mu)
    evec = np.cross(v, h) / mu - r / rn[..., None]
    e = np.linalg.norm(evec, axis=-1)
    # atan2 form: arccos(h_z/h) loses all precision for the near-planar orbits of the configs
    inc = np.arctan2(np.hypot(h[..., 0], h[..., 1]), h[..., 2])
    Omega = np.arctan2(h[..., 0], -h[..., 1])
    node = np.stack([np.cos(Omega), np.sin(Omega), np.zeros_like(Omega)], axis=-1)
    # argument of latitude of pericentre measured in the orbital plane
    m = np.cross(h / hn[..., None], node)
    omega = np.arctan2(np.sum(evec * m, axis=-1), np.sum(evec * node, axis=-1))
    # eccentric anomaly from e cos E = 1 - r/a, e sin E = r.v / sqrt(mu a)
    ecE = 1.0 - rn / a
    esE = np.sum(r * v, axis=-1) / np.sqrt(mu * a)
    E = np.arctan2(esE, ecE)
    M = E - esE
    return dict(a=a, e=e, inc=inc, Omega=np.mod(Omega, 2 * np.pi), omega=np.mod(omega, 2 * np.pi),
                M=np.mod(M, 2 * np.pi))


def angle_diff(a, b):
    return np.abs((a - b + np.pi) % (2 * np.pi) - np.pi)


def state_from_elements(mu, a, e, inc, Om, om, f):
    """Perifocal state at true anomaly f rotated by R_z(Om) R_x(inc) R_z(om), written out here
    (Murray & Dermott eq. 2.119-2.122); returns r, v and the mean anomaly of f."""
    p = a * (1.0 - e * e)
    r = p / (1.0 + e * np.cos(f))
    rp = np.array([r * np.cos(f), r * np.sin(f), 0.0])
    vp = np.sqrt(mu / p) * np.array([-np.sin(f), e + np.cos(f), 0.0])

    def rz(t):
        return np.array([[np.cos(t), -np.sin(t), 0], [np.sin(t), np.cos(t), 0], [0, 0, 1.0]])

    def rx(t):
        return np.array([[1.0, 0, 0], [0, np.cos(t), -np.sin(t)], [0, np.sin(t), np.cos(t)]])

    R = rz(Om) @ rx(inc) @ rz(om)
    E = 2.0 * np.arctan2(np.sqrt(1.0 - e) * np.sin(f / 2.0), np.sqrt(1.0 + e) * np.cos(f / 2.0))
    M = (E - e * np.sin(E)) % (2.0 * np.pi)
    return R @ rp, R @ vp, M
