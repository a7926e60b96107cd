"""-m "not gpu": pins of the 6th-order oracle (oracle_force6: acc, jerk, snap, pot; reading R22 of
DESIGN.md; "high >= 4th order integrators").  The paper prints no formula, so every pin
is something the mathematics fixes independently of the closed form the oracle types in:

  P13  rigid rotation: ANY configuration turning rigidly with angular velocity W has acc(t) =
       R(t) acc(0), hence jerk = W x acc and snap = W x (W x acc) -- exact, any masses, any eps
  P14  snap = d(jerk)/dt = d2(acc)/dt2 along x + v tau + a tau^2/2, by central differences of the
       ALREADY PINNED oracle.force, with the h^2 convergence of the stencil
  P15  a 50-digit numerical second derivative (mpmath) of the plain acceleration sum, small N,
       with a flagged pair, a coincident pair and duplicates in the i-list
  P16  sum_i m_i snap_i = 0; acc, jerk, pot bit-identical to oracle.force; predicted acceleration
"""
import numpy as np
import pytest

import nbgen
import oracle


def _rigid(n, seed, omega):
    rng = np.random.default_rng(seed)
    x = rng.normal(size=(3, n))
    m = rng.uniform(0.1, 10.0, n)
    w = np.array(omega, dtype=np.float64)[:, None]
    v = np.cross(w, x, axis=0)
    a = np.cross(w, v, axis=0)
    return m, x, v, a, w


@pytest.mark.parametrize("eps2", [0.0, 0.37])
def test_p13_rigid_rotation_closed_form(eps2):
    n = 23
    m, x, v, a, w = _rigid(n, 7, (0.3, -0.2, 0.5))
    il = np.arange(n, dtype=np.int32)
    acc, jrk, snp, pot = oracle.force6(m, x, v, a, il, eps2)
    jr = np.cross(w, acc, axis=0)
    sr = np.cross(w, jr, axis=0)
    assert np.abs(jrk - jr).max() <= 1e-13 * np.abs(jr).max()
    assert np.abs(snp - sr).max() <= 1e-12 * np.abs(sr).max()
    # a boost and a uniform extra acceleration change nothing (only differences enter)
    acc2, jrk2, snp2, _ = oracle.force6(m, x, v + 3.0, a - 7.0, il, eps2)
    assert np.abs(snp2 - snp).max() <= 1e-12 * np.abs(snp).max()
    assert np.abs(jrk2 - jrk).max() <= 1e-12 * np.abs(jrk).max()


def test_p13_ring_values():
    """The ring of tests/golden/ring_k7.txt (K = 7, R = 2, m = 1/7, omega = 0.3 about z): the snap of
    the particle at (R, 0, 0) is -omega^2 acc_x = +0.09 x 0.0823130311058..."""
    k, rad, om = 7, 2.0, 0.3
    ang = 2 * np.pi * np.arange(k) / k
    x = np.stack([rad * np.cos(ang), rad * np.sin(ang), np.zeros(k)])
    v = om * np.stack([-x[1], x[0], np.zeros(k)])
    a = -om * om * x
    acc, jrk, snp, pot = oracle.force6(np.full(k, 1.0 / k), x, v, a, np.arange(k, dtype=np.int32), 0.0)
    assert acc[0, 0] == pytest.approx(-0.0823130311058, rel=1e-11)
    assert snp[0, 0] == pytest.approx(0.09 * 0.0823130311058, rel=1e-11)
    assert abs(snp[1, 0]) < 1e-15 and abs(snp[2, 0]) < 1e-15


def test_p14_finite_differences_of_pinned_force():
    n, eps2 = 400, 1e-3
    m, x, v = nbgen.plummer(n, 31)
    m = m * (0.5 + nbgen.Streams(32, n).uniform())
    a = 0.3 * np.random.default_rng(33).normal(size=(3, n))
    il = np.arange(n, dtype=np.int32)
    _, _, snp, _ = oracle.force6(m, x, v, a, il, eps2)
    scale = np.sqrt((snp ** 2).sum(0))
    err = []
    for h in (2e-3, 1e-3, 5e-4):
        fp = oracle.force(m, x + v * h + a * (h * h / 2), v + a * h, il, eps2)
        fm = oracle.force(m, x - v * h + a * (h * h / 2), v - a * h, il, eps2)
        f0 = oracle.force(m, x, v, il, eps2)
        d_jerk = (fp[1] - fm[1]) / (2 * h)                       # d(jerk)/dt
        d2_acc = (fp[0] - 2 * f0[0] + fm[0]) / (h * h)            # d2(acc)/dt2
        e1 = np.sqrt(((d_jerk - snp) ** 2).sum(0)) / scale
        e2 = np.sqrt(((d2_acc - snp) ** 2).sum(0)) / scale
        err.append((np.median(e1), np.median(e2)))
    err = np.array(err)
    assert (err[2] < 2e-4).all(), err
    ratio = err[:-1] / err[1:]
    assert (ratio > 3.3).all() and (ratio < 4.7).all(), ratio       # h^2 stencils


def test_p15_mpmath_second_derivative():
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 50
    rng = np.random.default_rng(41)
    n = 7
    m = rng.uniform(0.1, 10.0, n)
    x, v, a = rng.normal(size=(3, n)), rng.normal(size=(3, n)), rng.normal(size=(3, n))
    x[:, 5] = x[:, 4]                                             # coincident, moving apart
    flags = np.zeros(n, np.uint8)
    flags[[1, 2]] = 1
    eps2 = 0.05
    il = np.array([0, 1, 4, 1, 6], np.int32)
    acc, jrk, snp, pot = oracle.force6(m, x, v, a, il, eps2, flags)

    def acc_of(i, c, tau):
        s = mp.mpf(0)
        for j in range(n):
            if j == i:
                continue
            r = [mp.mpf(x[q, j]) - mp.mpf(x[q, i]) + (mp.mpf(v[q, j]) - mp.mpf(v[q, i])) * tau +
                 (mp.mpf(a[q, j]) - mp.mpf(a[q, i])) * tau * tau / 2 for q in range(3)]
            e2 = mp.mpf(0) if (flags[i] and flags[j]) else mp.mpf(eps2)
            s2 = r[0] ** 2 + r[1] ** 2 + r[2] ** 2 + e2
            s += mp.mpf(m[j]) * r[c] / s2 ** mp.mpf(1.5)
        return s

    for k, i in enumerate(il):
        for c in range(3):
            ref2 = mp.diff(lambda tau: acc_of(int(i), c, tau), 0, 2)
            ref1 = mp.diff(lambda tau: acc_of(int(i), c, tau), 0, 1)
            assert abs(mp.mpf(snp[c, k]) - ref2) <= mp.mpf(1e-12) * max(1, abs(ref2)), (i, c)
            assert abs(mp.mpf(jrk[c, k]) - ref1) <= mp.mpf(1e-12) * max(1, abs(ref1)), (i, c)


def test_p16_momentum_identity_and_predicted_acceleration():
    n, eps2 = 300, 2e-3
    m, x, v = nbgen.plummer(n, 51)
    m = m * (0.5 + nbgen.Streams(52, n).uniform())
    rng = np.random.default_rng(53)
    a = rng.normal(size=(3, n))
    flags = (rng.uniform(size=n) < 0.05).astype(np.uint8)
    il = np.arange(n, dtype=np.int32)
    acc, jrk, snp, pot = oracle.force6(m, x, v, a, il, eps2, flags)
    ref = oracle.force(m, x, v, il, eps2, flags)
    assert np.array_equal(acc, ref[0]) and np.array_equal(jrk, ref[1]) and np.array_equal(pot, ref[2])
    assert np.abs((m * snp).sum(1)).max() <= 1e-9 * np.abs(m * snp).sum(1).max()
    # massless others, N = 1, s = 0 with eps2 = 0
    z = np.zeros((3, 1))
    out = oracle.force6(np.ones(1), z, z, z, np.zeros(1, np.int32), 0.0)
    assert all((q == 0).all() for q in out)
    x2 = np.zeros((3, 2))
    out = oracle.force6(np.ones(2), x2, x2, x2, np.array([0, 1], np.int32), 0.0)
    assert all((q == 0).all() for q in out)
    # R22: ap = a + jerk dt, exactly
    ap = oracle.predict_acc(0.5, np.full((3, 2), 3.0), np.full((3, 2), 6.0), np.array([0.0, 0.25]))
    assert (ap[:, 0] == 6.0).all() and (ap[:, 1] == 4.5).all()
