"""Test-harness pieces AROUND the kick (not product code, not oracle code): the Sun part HC (eq. 4,
PAPER.md:68) and the Kepler drift FG (eq. 2) of the democratic-heliocentric
leapfrog of App. A, in numpy, so that pin P8 and config 1 can advance a state
between kicks.  Democratic coordinates: heliocentric positions q, barycentric velocities v."""
import numpy as np


def kepler_drift(q, v, mu, dt):
    """Advance each body on its two-body orbit about the central mass (gravitational parameter mu)
    by dt with Gauss f and g functions in the eccentric-anomaly difference (elliptic orbits)."""
    r0 = np.sqrt((q * q).sum(axis=0))
    v2 = (v * v).sum(axis=0)
    u = (q * v).sum(axis=0)
    a = 1.0 / (2.0 / r0 - v2 / mu)
    if np.any(a <= 0):
        raise ValueError("harness Kepler drift handles bound orbits only")
    n = np.sqrt(mu / (a * a * a))
    ec = 1.0 - r0 / a                      # e cos E0
    es = u / (n * a * a)                   # e sin E0
    dM = n * dt
    # solve  dE - ec sin dE + es (1 - cos dE) = dM
    dE = dM.copy()
    for _ in range(20):
        s, c = np.sin(dE), np.cos(dE)
        fn = dE - ec * s + es * (1.0 - c) - dM
        fp = 1.0 - ec * c + es * s
        dE = dE - fn / fp
    s, c = np.sin(dE), np.cos(dE)
    f = 1.0 - (a / r0) * (1.0 - c)
    g = dt + (s - dE) / n
    r = a * (1.0 - ec * c + es * s)
    fd = -(a * a * n / (r0 * r)) * s
    gd = 1.0 - (a / r) * (1.0 - c)
    return f * q + g * v, fd * q + gd * v


def sun_drift(q, v, mass, m_star, dt):
    """HC: q_i += dt * (sum_j m_j v_j) / m_star   (eq. 4)."""
    p = (mass * v).sum(axis=1, keepdims=True)
    return q + dt * p / m_star


def energy(q, v, mass, m_star, G):
    """Total energy in democratic heliocentric variables (eq. 1-4 with K-terms recombined)."""
    p = mass * v
    kin = 0.5 * (mass * (v * v).sum(axis=0)).sum() + 0.5 * (p.sum(axis=1) ** 2).sum() / m_star
    r = np.sqrt((q * q).sum(axis=0))
    pot = -(G * m_star * mass / r).sum()
    n = q.shape[1]
    for i in range(n):
        for j in range(i + 1, n):
            d = np.sqrt(((q[:, i] - q[:, j]) ** 2).sum())
            pot -= G * mass[i] * mass[j] / d
    return kin + pot


def leapfrog_step(q, v, mass, m_star, G, dt, kick_acc):
    """One step of App. A: Kick(dt/2) HC(dt/2) FG(dt) HC(dt/2) Kick(dt/2).
    ``kick_acc(q)`` returns the interaction acceleration [3, N] (the path under test)."""
    v = v + 0.5 * dt * kick_acc(q)
    q = sun_drift(q, v, mass, m_star, 0.5 * dt)
    q, v = kepler_drift(q, v, G * m_star, dt)
    q = sun_drift(q, v, mass, m_star, 0.5 * dt)
    v = v + 0.5 * dt * kick_acc(q)
    return q, v
