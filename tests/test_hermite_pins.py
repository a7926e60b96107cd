"""Pins of oracle/hermite.py (corrector, interpolated derivatives, time-step criterion, block rule,
scheduler: DESIGN.md R12, R18..R21) against things the mathematics fixes -- CPU only."""
import numpy as np
import pytest

import oracle
from oracle import hermite as H


def _poly_state(c, tau):
    """x(tau) = sum c_k tau^k / k!  (c: (K, 3)) and its first three derivatives + a', a''."""
    from math import factorial
    out = []
    for d in range(6):
        s = np.zeros(3)
        for k in range(d, c.shape[0]):
            s = s + c[k] * tau ** (k - d) / factorial(k - d)
        out.append(s.reshape(3, 1))
    return out     # x, v, a, j, a2, a3


def test_corrector_exact_on_quartic_orbit():
    """R12 is the Hermite quadrature: exact when the acceleration is a quadratic in time (x a
    quartic).  A wrong sign or a coefficient other than 1/2, 1/12 breaks exactness."""
    rng = np.random.default_rng(5)
    c = rng.uniform(-1, 1, (5, 3))
    x0, v0, a0, j0, _, _ = _poly_state(c, 0.0)
    for dt in (0.5, 0.125):
        x1, v1, a1, j1, _, _ = _poly_state(c, dt)
        gx, gv = H.correct(x0, v0, a0, j0, a1, j1, dt)
        assert np.abs(gx - x1).max() < 1e-15 and np.abs(gv - v1).max() < 1e-15
    # a quintic is NOT integrated exactly: v stays exact (a is a cubic) and the local error of x is
    # dt^5 v''''/720, so it falls 32x per halving
    c = rng.uniform(-1, 1, (6, 3))
    errs = []
    for dt in (0.5, 0.25, 0.125):
        x0, v0, a0, j0, _, _ = _poly_state(c, 0.0)
        x1, v1, a1, j1, _, _ = _poly_state(c, dt)
        gx, gv = H.correct(x0, v0, a0, j0, a1, j1, dt)
        errs.append(np.abs(gx - x1).max())
    assert 28 < errs[0] / errs[1] < 36 and 28 < errs[1] / errs[2] < 36


def test_derivatives_exact_for_cubic_acceleration():
    """R18: with a(tau) a cubic, the interpolation returns a''(t1) and a''' exactly."""
    rng = np.random.default_rng(6)
    c = rng.uniform(-1, 1, (6, 3))          # x of degree 5 -> a of degree 3
    dt = 0.25
    _, _, a0, j0, _, _ = _poly_state(c, 0.0)
    _, _, a1, j1, a2, a3 = _poly_state(c, dt)
    g2, g3 = H.derivatives(a0, j0, a1, j1, dt)
    assert np.abs(g2 - a2).max() < 1e-12 and np.abs(g3 - a3).max() < 1e-11


def test_aarseth_criterion_on_circular_orbit():
    """R19 closed form: on a circular orbit of angular frequency w every derivative has norm
    w^(k+2) R, so dt = sqrt(eta) / w exactly."""
    w, R, eta = 1.7, 2.5, 0.02
    e1, e2 = np.array([[1.0], [0.0], [0.0]]), np.array([[0.0], [1.0], [0.0]])
    a, j, a2, a3 = -w ** 2 * R * e1, -w ** 3 * R * e2, w ** 4 * R * e1, w ** 5 * R * e2
    assert abs(H.aarseth_dt(a, j, a2, a3, eta)[0] - np.sqrt(eta) / w) < 1e-15
    assert abs(H.initial_dt(a, j, 0.01)[0] - 0.01 / w) < 1e-15
    # force-free particle: no finite step is asked for
    z = np.zeros((3, 1))
    assert np.isinf(H.aarseth_dt(z, z, z, z, eta)[0]) and np.isinf(H.initial_dt(z, z, 0.01)[0])
    # and with the interpolated derivatives (R18) the same value is approached as dt^2
    errs = []
    for dt in (0.1, 0.05):
        th = w * dt
        a1 = -w ** 2 * R * (np.cos(th) * e1 + np.sin(th) * e2)
        j1 = -w ** 3 * R * (-np.sin(th) * e1 + np.cos(th) * e2)
        g2, g3 = H.derivatives(a, j, a1, j1, dt)
        errs.append(abs(H.aarseth_dt(a1, j1, g2, g3, eta)[0] - np.sqrt(eta) / w))
    assert errs[1] < errs[0] / 3.0


def test_block_rule_cases():
    """R20, case by case (dt_min = 2^-10, dt_max = 2^-2)."""
    lo, hi = 2.0 ** -10, 2.0 ** -2
    f = lambda d, w, t1: float(H.block_dt(np.array([d]), np.array([w]), t1, lo, hi)[0])
    assert f(2.0 ** -4, 0.05, 0.25) == 2.0 ** -5            # shrink once: 1/32 <= 0.05
    assert f(2.0 ** -4, 0.009, 0.25) == 2.0 ** -7           # shrink repeatedly: 1/128 <= 0.009
    assert f(2.0 ** -4, 1e-9, 0.25) == lo                   # never below dt_min
    assert f(2.0 ** -4, 0.1, 0.25) == 2.0 ** -4             # wants < 2 dt: keep
    assert f(2.0 ** -4, 0.2, 0.25) == 2.0 ** -3             # may double: 0.25 is a multiple of 1/8
    assert f(2.0 ** -4, 0.2, 0.3125) == 2.0 ** -4           # 5/16 is not a multiple of 1/8: keep
    assert f(2.0 ** -4, 10.0, 0.25) == 2.0 ** -3            # doubles at most once
    assert f(hi, np.inf, 1.0) == hi                         # never above dt_max
    q = H.quantise_dt(np.array([0.3, 0.05, 1e-9, np.inf, 2.0 ** -6]), lo, hi)
    assert q.tolist() == [hi, 2.0 ** -5, lo, hi, 2.0 ** -6]


def test_next_block():
    t = np.array([0.0, 0.25, 0.125, 0.25, 0.0])
    dt = np.array([0.5, 0.125, 0.25, 0.25, 0.375])
    t_next, idx = H.next_block(t, dt)
    assert t_next == 0.375 and idx.tolist() == [1, 2, 4]


def _two_body(e):
    """Equal masses 1/2, G = 1, semi-major axis 1, at pericentre.  Returns m, x, v, period."""
    m = np.array([0.5, 0.5])
    rp, vp = 1.0 - e, np.sqrt((1.0 + e) / (1.0 - e))
    x = np.array([[-rp / 2, rp / 2], [0.0, 0.0], [0.0, 0.0]])
    v = np.array([[0.0, 0.0], [-vp / 2, vp / 2], [0.0, 0.0]])
    return m, x, v, 2.0 * np.pi


def _energy(m, x, v):
    _, _, p = oracle.force(m, x, v, np.arange(m.shape[0], dtype=np.int32), 0.0)
    return 0.5 * (m * (v * v).sum(0)).sum() + 0.5 * (m * p).sum()


@pytest.mark.parametrize("e", [0.3, 0.5])
def test_p11_shared_step_scheme_is_fourth_order(e):
    """P11: predictor (oracle_predict) + force (oracle_force) + corrector (R12) with a shared step:
    the energy error after a fixed time falls ~16x per halving of dt (eccentric orbits; on the
    circular orbit the leading term cancels and it falls 32x)."""
    errs = []
    for steps in (64, 128, 256):
        m, x, v, T = _two_body(e)
        il = np.arange(2, dtype=np.int32)
        dt = T / 4 / steps
        a, j, _ = oracle.force(m, x, v, il, 0.0)
        e0 = _energy(m, x, v)
        t = np.zeros(2)
        for s in range(steps):
            xp, vp = oracle.predict(t[0] + dt, x, v, a, j, t)
            a1, j1, _ = oracle.force(m, xp, vp, il, 0.0)
            x, v = H.correct(x, v, a, j, a1, j1, dt)
            a, j, t = a1, j1, t + dt
        errs.append(abs(_energy(m, x, v) - e0))
    assert 10 < errs[0] / errs[1] < 24 and 10 < errs[1] / errs[2] < 24


def test_block_step_integration_conserves_energy():
    """Whole scheme (R12, R18..R21) on a small Plummer sphere: individual block steps, the energy
    drift over 1/8 time unit stays small and steps are powers of two on a commensurate grid."""
    import nbgen
    m, x, v = nbgen.plummer(64, 77)
    n, eps2, eta = 64, 1e-4, 0.01
    lo, hi = 2.0 ** -16, 2.0 ** -4
    il = np.arange(n, dtype=np.int32)
    a, j, p = oracle.force(m, x, v, il, eps2)
    e0 = 0.5 * (m * (v * v).sum(0)).sum() + 0.5 * (m * p).sum()
    t = np.zeros(n)
    dt = H.quantise_dt(H.initial_dt(a, j, eta), lo, hi)
    nsteps = 0
    while True:
        t1, idx = H.next_block(t, dt)
        if t1 > 0.125:
            break
        xp, vp = oracle.predict(t1, x, v, a, j, t)
        a1, j1, _ = oracle.force(m, xp, vp, idx, eps2)
        H.corrector_step(x, v, a, j, t, dt, idx, t1, a1, j1, eta, lo, hi)
        assert np.all(np.fmod(t[idx], dt[idx]) == 0.0)          # commensurate block grid
        nsteps += 1
    xp, vp = oracle.predict(0.125, x, v, a, j, t)
    _, _, p = oracle.force(m, xp, vp, il, eps2)
    e1 = 0.5 * (m * (vp * vp).sum(0)).sum() + 0.5 * (m * p).sum()
    assert nsteps > 8 and abs(e1 - e0) < 1e-6 * abs(e0)
    assert np.all(np.log2(dt) == np.round(np.log2(dt)))
