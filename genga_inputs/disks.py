"""Planetesimal-disk generators for the five BASELINE.json configs.

Units: AU, day, Msun; G = k^2 with the Gaussian constant k = 0.01720209895.
Every random number comes from ``splitmix.uniforms(seed, ...)``: body n draws the eight
uniforms 8n .. 8n+7 (a, e, i, Omega, omega, M, mass, spare) of its population's stream, so a
body's draw does not depend on N.  Body order = generation order (random in a, NOT sorted).
"""
from dataclasses import dataclass, field
import numpy as np

from .splitmix import uniforms

K_GAUSS = 0.01720209895
G_AU_DAY_MSUN = K_GAUSS * K_GAUSS
# Constants the paper does not print: fixed here, recorded in KickInputs.meta.
M_EARTH = 1.0 / 332946.0487          # Msun
M_JUPITER = 1.0 / 1047.3486          # Msun
M_SUN_GRAM = 1.98847e33
AU_CM = 1.495978707e13
DT_DAYS = 6.0
N1_HILL = 3.0                         # eq. 5
N2_VEL = 0.4                          # eq. 5

CONFIG_NAMES = (
    "cfg0_n2048_L0",
    "cfg1_n8192_L0_100kicks",
    "cfg2_n32768_giants_L1",
    "cfg3_n65536_L1",
    "cfg4_tp_2048m_1048576t_L0",
)


@dataclass
class KickInputs:
    """Inputs of one kick call (layout of SURVEY.md 8(b)): SoA float64, C-contiguous."""
    pos: np.ndarray            # [3, N] heliocentric positions, AU
    vel: np.ndarray            # [3, N] heliocentric velocities, AU/day
    mass: np.ndarray           # [N] Msun
    rcrit: np.ndarray          # [level+1, N] r_crit_i at dt / s^k, AU
    n_massive: int
    n_test: int
    level: int
    dt: float
    G: float = G_AU_DAY_MSUN
    enc_factor: float = 1.0
    substeps: int = 2
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return self.n_massive + self.n_test


def _solve_kepler(M, e):
    """Eccentric anomaly from M = E - e sin E (Newton, fixed 12 sweeps; e << 1 here)."""
    E = M + e * np.sin(M)
    for _ in range(12):
        E = E - (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E))
    return E


def elements_to_cartesian(a, e, inc, Omega, omega, M, mu):
    """Heliocentric Cartesian state from Keplerian elements (two-body, gravitational parameter mu)."""
    E = _solve_kepler(M, e)
    cE, sE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    n = np.sqrt(mu / (a * a * a))
    xp = a * (cE - e)
    yp = a * b * sE
    rfac = 1.0 / (1.0 - e * cE)
    vxp = -a * n * sE * rfac
    vyp = a * n * b * cE * rfac
    cO, sO = np.cos(Omega), np.sin(Omega)
    co, so = np.cos(omega), np.sin(omega)
    ci, si = np.cos(inc), np.sin(inc)
    # rotation matrix columns for the orbital-plane x' and y' axes
    px = cO * co - sO * so * ci
    py = sO * co + cO * so * ci
    pz = so * si
    qx = -cO * so - sO * co * ci
    qy = -sO * so + cO * co * ci
    qz = co * si
    pos = np.stack([px * xp + qx * yp, py * xp + qy * yp, pz * xp + qz * yp])
    vel = np.stack([px * vxp + qx * vyp, py * vxp + qy * vyp, pz * vxp + qz * vyp])
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel)


def semi_major_axis(pos, vel, mu):
    """a from the vis-viva equation; used to recompute Hill radii of evolving states (config 1)."""
    r = np.sqrt((pos * pos).sum(axis=0))
    v2 = (vel * vel).sum(axis=0)
    return 1.0 / (2.0 / r - v2 / mu)


def rcrit_rows(a, vel, mass, dt, substeps, nrows, m_star=1.0):
    """Rows k = 0..nrows-1 of r_crit_i = max(n1 R_H,i , n2 (dt / s^k) |v_i|)   (eq. 5 + PAPER.md:638).

    R_H,i = a_i (m_i / (3 m_star))^(1/3); v_i = heliocentric speed."""
    hill = a * np.cbrt(mass / (3.0 * m_star))
    speed = np.sqrt((vel * vel).sum(axis=0))
    rows = [np.maximum(N1_HILL * hill, N2_VEL * (dt / float(substeps) ** k) * speed) for k in range(nrows)]
    return np.ascontiguousarray(np.stack(rows))


def _rayleigh(sigma, u):
    return sigma * np.sqrt(-2.0 * np.log1p(-u))


def _population(n, seed, a_lo, a_hi, sigma_e, sigma_i, a_law="uniform", first=0):
    """Elements of bodies first..first+n-1 of the stream ``seed``; returns dict of arrays."""
    u = uniforms(seed, 8 * first, 8 * n).reshape(n, 8)
    if a_law == "uniform":
        a = a_lo + (a_hi - a_lo) * u[:, 0]
    elif a_law == "sigma_a^-1.5":
        # surface density ~ a^-1.5  =>  dN/da ~ a^-0.5  =>  sqrt(a) uniform
        a = (np.sqrt(a_lo) + u[:, 0] * (np.sqrt(a_hi) - np.sqrt(a_lo))) ** 2
    else:
        raise ValueError(a_law)
    two_pi = 2.0 * np.pi
    return dict(a=a, e=_rayleigh(sigma_e, u[:, 1]), inc=_rayleigh(sigma_i, u[:, 2]),
                Omega=two_pi * u[:, 3], omega=two_pi * u[:, 4], M=two_pi * u[:, 5], umass=u[:, 6])


def _radius_au(mass, density_g_cm3=2.0):
    return np.cbrt(3.0 * mass * M_SUN_GRAM / (4.0 * np.pi * density_g_cm3)) / AU_CM


def make_disk(n, seed, total_mass=2.5 * M_EARTH, a_lo=0.5, a_hi=4.0, sigma_e=0.01, sigma_i=0.005,
              a_law="uniform", mass_law="equal", level=0, substeps=2, dt=DT_DAYS,
              n_test=0, tp_seed=None, tp_a=(1.8, 3.5), tp_sigma_e=0.05, tp_sigma_i=0.05,
              giants=False):
    """General recipe; the five configs are thin presets of this (see make_config)."""
    G = G_AU_DAY_MSUN
    el = _population(n, seed, a_lo, a_hi, sigma_e, sigma_i, a_law)
    if mass_law == "equal":
        mass = np.full(n, total_mass / max(n, 1))
    elif mass_law == "loguniform_1e-4_1e-2_mearth":
        mass = M_EARTH * 10.0 ** (-4.0 + 2.0 * el["umass"])
    else:
        raise ValueError(mass_law)
    a = el["a"]
    pos, vel = elements_to_cartesian(a, el["e"], el["inc"], el["Omega"], el["omega"], el["M"], G * (1.0 + mass))
    if giants:
        ug = uniforms(seed ^ 0x5A5A5A5A, 0, 2)
        ga = np.array([5.2, 9.5])
        gm = np.array([1.0, 0.3]) * M_JUPITER
        z = np.zeros(2)
        gp, gv = elements_to_cartesian(ga, z, z, z, z, 2.0 * np.pi * ug, G * (1.0 + gm))
        pos, vel = np.concatenate([pos, gp], axis=1), np.concatenate([vel, gv], axis=1)
        mass, a = np.concatenate([mass, gm]), np.concatenate([a, ga])
    n_massive = pos.shape[1]
    if n_test:
        tel = _population(n_test, seed + 7777 if tp_seed is None else tp_seed, tp_a[0], tp_a[1],
                          tp_sigma_e, tp_sigma_i, "uniform")
        tm = np.zeros(n_test)
        tpos, tvel = elements_to_cartesian(tel["a"], tel["e"], tel["inc"], tel["Omega"], tel["omega"],
                                           tel["M"], G * np.ones(n_test))
        pos, vel = np.concatenate([pos, tpos], axis=1), np.concatenate([vel, tvel], axis=1)
        mass, a = np.concatenate([mass, tm]), np.concatenate([a, tel["a"]])
    rc = rcrit_rows(a, vel, mass, dt, substeps, level + 1)
    meta = dict(seed=seed, M_EARTH=M_EARTH, M_JUPITER=M_JUPITER, density_g_cm3=2.0, a_law=a_law,
                mass_law=mass_law, radius_au_first=float(_radius_au(mass[:1])[0]) if n else 0.0)
    return KickInputs(pos=np.ascontiguousarray(pos), vel=np.ascontiguousarray(vel),
                      mass=np.ascontiguousarray(mass), rcrit=rc, n_massive=n_massive, n_test=n_test,
                      level=level, dt=dt, substeps=substeps, meta=meta)


def make_config(idx, n=None, n_test=None, level=None):
    """BASELINE.json config ``idx`` (0..4); ``n`` / ``n_test`` / ``level`` shrink or re-level it for tests."""
    seed = 1000 + idx
    if idx == 0:
        ki = make_disk(2048 if n is None else n, seed, level=0 if level is None else level)
    elif idx == 1:
        ki = make_disk(8192 if n is None else n, seed, level=0 if level is None else level)
    elif idx == 2:
        ki = make_disk(32768 if n is None else n, seed, total_mass=5.0 * M_EARTH, giants=True,
                       level=1 if level is None else level)
    elif idx == 3:
        ki = make_disk(65536 if n is None else n, seed, a_law="sigma_a^-1.5",
                       mass_law="loguniform_1e-4_1e-2_mearth", level=1 if level is None else level)
    elif idx == 4:
        ki = make_disk(2048 if n is None else n, seed, n_test=1048576 if n_test is None else n_test,
                       level=0 if level is None else level)
    else:
        raise ValueError("config index must be 0..4")
    ki.meta["config"] = CONFIG_NAMES[idx]
    return ki


def make_ring(n, radius=1.0, mass=1e-9, partners=8):
    """Fig. 7 geometry: n equal bodies on a ring, r_crit between the chord to the
    (partners/2)-th and (partners/2 + 1)-th neighbour, so every body has exactly ``partners`` partners."""
    G = G_AU_DAY_MSUN
    phi = 2.0 * np.pi * np.arange(n) / n
    pos = np.stack([radius * np.cos(phi), radius * np.sin(phi), np.zeros(n)])
    vc = np.sqrt(G / radius)
    vel = np.stack([-vc * np.sin(phi), vc * np.cos(phi), np.zeros(n)])
    h = partners // 2
    chord = lambda k: 2.0 * radius * np.sin(np.pi * k / n)
    rc = 0.5 * (chord(h) + chord(h + 1))
    return KickInputs(pos=np.ascontiguousarray(pos), vel=np.ascontiguousarray(vel), mass=np.full(n, mass),
                      rcrit=np.full((1, n), rc), n_massive=n, n_test=0, level=0, dt=DT_DAYS,
                      meta=dict(ring=True, partners=partners))
