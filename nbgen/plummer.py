"""Plummer-sphere sampler (the paper only cites Plummer [14]; the procedure is
the standard inverse-mass-profile + von Neumann rejection construction).

Input synthesis only: no pair sums live here.  `mean_field` is the closed-form smooth field of the
Plummer model, used to give block-time-step test states a physically shaped (acc, jerk) to
predict from; it is never used as an expected value.
"""
import numpy as np

from .rng import Streams

HENON_A = 3.0 * np.pi / 16.0  # Plummer scale length for which W = -1/2 at M = G = 1
MASS_CUT = 0.999              # mass-fraction cut: r <= 38.7 a


def _unit_vectors(u_cos, u_phi):
    c = 2.0 * u_cos - 1.0
    s = np.sqrt(np.maximum(0.0, 1.0 - c * c))
    phi = 2.0 * np.pi * u_phi
    return np.stack([s * np.cos(phi), s * np.sin(phi), c])


def plummer(n, seed, a=HENON_A, mass=1.0, recentre=True):
    """n equal-mass stars of total mass `mass`, scale length a, G = 1.

    Returns m (n,), x (3, n), v (3, n), all float64.  Per-star draws, in order:
    u1 (radius; redrawn until 0 < u1 <= 0.999), u2, u3 (position direction), then pairs
    (u4, u5) until 0.1*u5 < u4^2 (1-u4^2)^3.5 (speed as a fraction of escape speed),
    then u6, u7 (velocity direction).  Centre of mass and its velocity are subtracted last.
    No energy rescale."""
    st = Streams(seed, n)
    u1 = st.uniform()
    bad = np.flatnonzero(~((u1 > 0.0) & (u1 <= MASS_CUT)))
    while bad.size:
        u1[bad] = st.uniform(bad)
        bad = bad[~((u1[bad] > 0.0) & (u1[bad] <= MASS_CUT))]
    r = a / np.sqrt(u1 ** (-2.0 / 3.0) - 1.0)
    x = r * _unit_vectors(st.uniform(), st.uniform())

    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        u4 = st.uniform(todo)
        u5 = st.uniform(todo)
        ok = 0.1 * u5 < u4 * u4 * (1.0 - u4 * u4) ** 3.5
        q[todo[ok]] = u4[ok]
        todo = todo[~ok]
    speed = q * np.sqrt(2.0 * mass / a) * (1.0 + (r / a) ** 2) ** -0.25
    v = speed * _unit_vectors(st.uniform(), st.uniform())

    m = np.full(n, mass / n)
    if recentre:
        x -= (x @ m / mass)[:, None]
        v -= (v @ m / mass)[:, None]
    return m, np.ascontiguousarray(x), np.ascontiguousarray(v)


def mean_field(x, v, a=HENON_A, mass=1.0):
    """Smooth Plummer field at positions x (3, n) for velocities v: acc = -M x / (r^2+a^2)^1.5 and
    its time derivative along v.  Input synthesis for block-step states (config 3)."""
    s = (x * x).sum(0) + a * a
    s15 = s ** -1.5
    rv = (x * v).sum(0)
    acc = -mass * x * s15
    jrk = -mass * (v * s15 - 3.0 * rv * x * s ** -2.5)
    return acc, jrk
