"""Pins of the fp64 oracle against things other than itself (P1..P12).

The paper prints no formula and no number for the direct path, so the pins are: exact rationals
worked by hand (P1), conservation laws (P2), the Plummer model's known energies (P3), finite
differences (P4, P5), an independent 50-digit brute force (P6), symmetries (P7), a closed-form
many-body sum (P8), the predictor's exact values and convergence order on a Kepler orbit (P9) and
degenerate inputs (P12).  A dropped term, wrong sign, wrong index or transposed operand in
oracle/nb_oracle.c fails at least one of them.
"""
import math
import os
from fractions import Fraction

import mpmath
import numpy as np
import pytest

import nbgen
import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def all_force(m, x, v, eps2, flags=None):
    return oracle.force(m, x, v, np.arange(m.shape[0], dtype=np.int32), eps2, flags)


# ------------------------------------------------------------------ P1 exact two-body example
@pytest.mark.parametrize("row", _rows("two_body_exact.txt"))
def test_p1_two_body_exact(row):
    eps2, who = float(row[0]), int(row[1])
    want = np.array([float(Fraction(s)) for s in row[2:]])
    m = np.array([3.0, 2.0])
    x = np.array([[0.0, 3.0], [0.0, 4.0], [0.0, 0.0]])
    v = np.array([[0.0, 1.0], [0.0, -2.0], [0.0, 0.5]])
    acc, jrk, pot = all_force(m, x, v, eps2)
    got = np.concatenate([acc[:, who], jrk[:, who], [pot[who]]])
    np.testing.assert_allclose(got, want, rtol=8 * np.finfo(float).eps, atol=1e-18)   # a handful of roundings
    # momentum and energy of the pair, exactly representable cases
    assert abs((m * acc).sum(1)).max() < 1e-16
    w_tot = 0.5 * (m * pot).sum()
    assert w_tot == pytest.approx(-1.0 if eps2 == 11 else -1.2, rel=1e-15)


# ------------------------------------------------------------------ P2 momentum
@pytest.mark.parametrize("n,eps2", [(1024, 1e-4), (4096, 0.0)])
def test_p2_momentum(n, eps2):
    m, x, v = nbgen.plummer(n, 7)
    m = m * (0.5 + nbgen.Streams(8, n).uniform())          # unequal masses
    flags = (nbgen.Streams(9, n).uniform() < 0.01).astype(np.uint8)
    acc, jrk, pot = all_force(m, x, v, eps2, flags)
    assert abs((m * acc).sum(1)).max() < 1e-12
    assert abs((m * jrk).sum(1)).max() < 1e-12


# ------------------------------------------------------------------ P3 Plummer energies
def test_p3_plummer_energy():
    n = 16384
    m, x, v = nbgen.plummer(n, 12)
    acc, jrk, pot = all_force(m, x, v, 2.0 ** -20)
    w = 0.5 * (m * pot).sum()
    k = 0.5 * (m * (v * v).sum(0)).sum()
    assert abs(w + 0.5) < 0.01       # Henon units: W = -1/2
    assert abs(k - 0.25) < 0.01      # virial: K = 1/4
    assert (pot < 0).all()
    # virial of the sampled forces: sum m x.a = W exactly for eps = 0; close for small eps
    assert (m * (x * acc).sum(0)).sum() == pytest.approx(w, rel=2e-3)


# ------------------------------------------------------------------ P4 finite-difference jerk
def test_p4_finite_difference_jerk():
    n, eps2 = 1024, 1e-4
    m, x, v = nbgen.plummer(n, 21)
    _, jrk, _ = all_force(m, x, v, eps2)
    errs = []
    for h in (1e-4, 5e-5):
        ap, _, _ = all_force(m, x + h * v, v, eps2)
        am, _, _ = all_force(m, x - h * v, v, eps2)
        fd = (ap - am) / (2 * h)
        errs.append(np.sqrt(((fd - jrk) ** 2).sum(0)) / np.sqrt((jrk ** 2).sum(0)))
    assert np.median(errs[1]) < 1e-6 and errs[1].max() < 2e-3
    ratio = np.median(errs[0]) / np.median(errs[1])
    assert 3.5 < ratio < 4.5          # central difference: error ~ h^2


# ------------------------------------------------------------------ P5 acc = -d pot_i / d x_i
def test_p5_acc_is_minus_gradient_of_pot():
    n, eps2, h = 256, 1e-3, 1e-6
    m, x, v = nbgen.plummer(n, 22)
    acc, _, _ = all_force(m, x, v, eps2)
    for i in (0, 17, 255):
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[c, i] += h
            xm[c, i] -= h
            pp = oracle.force(m, xp, v, [i], eps2)[2][0]
            pm = oracle.force(m, xm, v, [i], eps2)[2][0]
            assert -(pp - pm) / (2 * h) == pytest.approx(acc[c, i], rel=1e-6, abs=1e-9)


# ------------------------------------------------------------------ P6 50-digit brute force
def _mp_force(m, x, v, flags, ilist, eps2):
    mpmath.mp.dps = 50
    M = [mpmath.mpf(float(q)) for q in m]
    X = [[mpmath.mpf(float(q)) for q in x[:, p]] for p in range(len(m))]
    V = [[mpmath.mpf(float(q)) for q in v[:, p]] for p in range(len(m))]
    out = []
    for i in ilist:
        a = [mpmath.mpf(0)] * 3
        jk = [mpmath.mpf(0)] * 3
        pot = mpmath.mpf(0)
        for j in range(len(m)):
            if j == i:
                continue
            r = [X[j][c] - X[i][c] for c in range(3)]
            w = [V[j][c] - V[i][c] for c in range(3)]
            e2 = 0 if (flags[i] & flags[j] & 1) else mpmath.mpf(eps2)
            s = sum(q * q for q in r) + e2
            if s == 0:
                continue
            rv = sum(p * q for p, q in zip(r, w))
            pot -= M[j] / mpmath.sqrt(s)
            for c in range(3):
                a[c] += M[j] * r[c] / s ** mpmath.mpf(1.5)
                jk[c] += M[j] * (w[c] / s ** mpmath.mpf(1.5) - 3 * rv * r[c] / s ** mpmath.mpf(2.5))
        out.append([float(q) for q in a] + [float(q) for q in jk] + [float(pot)])
    return np.array(out).T


@pytest.mark.parametrize("n,seed,eps2", [(2, 1, 0.0), (17, 2, 0.25), (64, 3, 1e-4), (33, 4, 0.0)])
def test_p6_brute_force_50_digits(n, seed, eps2):
    st = nbgen.Streams(1000 + seed, n)
    m = 0.1 + 9.9 * st.uniform()
    x = np.stack([st.uniform() * 4 - 2 for _ in range(3)])
    v = np.stack([st.uniform() * 2 - 1 for _ in range(3)])
    flags = (st.uniform() < 0.3).astype(np.uint8)
    if n >= 17:                      # coincident pairs: one flagged-flagged, one plain
        x[:, 5] = x[:, 3]
        x[:, 9] = x[:, 8]
        flags[3] = flags[5] = 1
        flags[8] = flags[9] = 0
    ilist = list(range(n)) + [0, n - 1]                     # duplicates are legal
    acc, jrk, pot = oracle.force(m, x, v, ilist, eps2, flags)
    ref = _mp_force(m, x, v, flags, ilist, eps2)
    got = np.concatenate([acc, jrk, pot[None]])
    scale = np.abs(ref).max(1, keepdims=True)
    assert np.isfinite(got).all()
    assert (np.abs(got - ref) / scale).max() < 1e-13


def test_p6_predictor_50_digits():
    n = 40
    st = nbgen.Streams(77, n)
    arr = [np.stack([st.uniform() * 2 - 1 for _ in range(3)]) for _ in range(4)]
    tj = st.uniform() * 0.5
    t = 0.3125
    xp, vp = oracle.predict(t, *arr, tj)
    mpmath.mp.dps = 50
    for p in range(n):
        dt = mpmath.mpf(t) - mpmath.mpf(float(tj[p]))
        for c in range(3):
            x, v, a, j = (mpmath.mpf(float(q[c, p])) for q in arr)
            ex = x + v * dt + a * dt ** 2 / 2 + j * dt ** 3 / 6
            ev = v + a * dt + j * dt ** 2 / 2
            assert abs(xp[c, p] - float(ex)) <= 4e-16 * max(1.0, abs(float(ex)))
            assert abs(vp[c, p] - float(ev)) <= 4e-16 * max(1.0, abs(float(ev)))


# ------------------------------------------------------------------ P7 invariances
def _case(n=512, seed=31):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    return m, x, v


def _close(a, b, tol):
    for p, q in zip(a, b):
        s = np.abs(q).max()
        assert np.abs(p - q).max() <= tol * s


def test_p7_translation_and_boost():
    m, x, v = _case()
    ref = all_force(m, x, v, 1e-4)
    _close(all_force(m, x + np.array([[1e3], [-2e3], [5e2]]), v, 1e-4), ref, 1e-9)
    _close(all_force(m, x, v + np.array([[3.0], [-1.0], [0.5]]), 1e-4), ref, 1e-12)


def test_p7_rotation():
    m, x, v = _case()
    th, ph = 0.7, -1.1
    r1 = np.array([[math.cos(th), -math.sin(th), 0], [math.sin(th), math.cos(th), 0], [0, 0, 1]])
    r2 = np.array([[1, 0, 0], [0, math.cos(ph), -math.sin(ph)], [0, math.sin(ph), math.cos(ph)]])
    rot = r1 @ r2
    a, j, p = all_force(m, x, v, 1e-4)
    a2, j2, p2 = all_force(m, rot @ x, rot @ v, 1e-4)
    _close((a2, j2, p2), (rot @ a, rot @ j, p), 1e-12)


def test_p7_scaling():
    m, x, v = _case()
    lam, eps2 = 3.0, 1e-4
    a, j, p = all_force(m, x, v, eps2)
    a2, j2, p2 = all_force(m, lam * x, v / math.sqrt(lam), lam * lam * eps2)
    _close((a2, j2, p2), (a / lam ** 2, j / lam ** 3.5, p / lam), 1e-12)


def test_p7_permutation_and_j_split():
    m, x, v = _case()
    n = m.shape[0]
    il = np.arange(0, n, 3, dtype=np.int32)
    ref = oracle.force(m, x, v, il, 1e-4)
    perm = nbgen.permutation(5, n)
    inv = np.empty(n, np.int32)
    inv[perm] = np.arange(n, dtype=np.int32)
    _close(oracle.force(m[perm], x[:, perm], v[:, perm], inv[il], 1e-4), ref, 1e-12)
    # partial forces over j-subsets add up
    ma, mb = m.copy(), m.copy()
    ma[n // 3:] = 0.0
    mb[:n // 3] = 0.0
    fa = oracle.force(ma, x, v, il, 1e-4)
    fb = oracle.force(mb, x, v, il, 1e-4)
    _close([p + q for p, q in zip(fa, fb)], ref, 1e-12)


def test_p7_i_independence_and_duplicates():
    m, x, v = _case()
    a, j, p = all_force(m, x, v, 1e-4)
    il = np.array([5, 500, 5, 0, 511, 500], np.int32)            # i's independent
    a2, j2, p2 = oracle.force(m, x, v, il, 1e-4)
    assert (a2 == a[:, il]).all() and (j2 == j[:, il]).all() and (p2 == p[il]).all()


def test_p7_flags_only_change_flagged_pairs():
    m, x, v = _case(64)
    flags = np.zeros(64, np.uint8)
    flags[[3, 40]] = 1
    base = all_force(m, x, v, 0.04)
    got = all_force(m, x, v, 0.04, flags)
    keep = np.setdiff1d(np.arange(64), [3, 40])
    assert all((g[..., keep] == b[..., keep]).all() for g, b in zip(got, base))
    # the pair (3, 40) is exactly the unsoftened two-body term swapped for the softened one
    pair = oracle.force(m[[3, 40]], x[:, [3, 40]], v[:, [3, 40]], [0, 1], 0.0)
    soft = oracle.force(m[[3, 40]], x[:, [3, 40]], v[:, [3, 40]], [0, 1], 0.04)
    for g, b, u, s in zip(got, base, pair, soft):
        np.testing.assert_allclose(g[..., [3, 40]], b[..., [3, 40]] - s + u, rtol=1e-12, atol=1e-15)


# ------------------------------------------------------------------ P8 ring closed form
def test_p8_ring_closed_form():
    k, rad, om = 7, 2.0, 0.3
    mass = 1.0 / k
    ang = 2 * math.pi * np.arange(k) / k
    x = np.stack([rad * np.cos(ang), rad * np.sin(ang), np.zeros(k)])
    v = om * np.stack([-x[1], x[0], np.zeros(k)])
    acc, jrk, pot = all_force(np.full(k, mass), x, v, 0.0)
    s = sum(1.0 / math.sin(math.pi * q / k) for q in range(1, k))
    gold = [float(q) for q in _rows("ring_k7.txt")[0]]
    assert -mass * s / (4 * rad * rad) == pytest.approx(gold[0], abs=2e-13)
    assert acc[0, 0] == pytest.approx(gold[0], abs=2e-13)
    assert pot[0] == pytest.approx(gold[1], abs=2e-13)
    assert jrk[1, 0] == pytest.approx(gold[2], abs=2e-13)
    for p in range(k):
        rhat = x[:, p] / rad
        np.testing.assert_allclose(acc[:, p], -mass * s / (4 * rad * rad) * rhat, atol=1e-15)
        np.testing.assert_allclose(jrk[:, p], om * np.array([-acc[1, p], acc[0, p], 0]), atol=1e-15)
        assert pot[p] == pytest.approx(-mass * s / (2 * rad), rel=1e-14)


# ------------------------------------------------------------------ P9 predictor
def test_p9_predictor_exact_values():
    one = np.ones((3, 1))
    xp, vp = oracle.predict(0.5, 1 * one, 2 * one, 3 * one, 6 * one, np.zeros(1))
    assert (xp == 2.5).all() and (vp == 4.25).all()
    xp, vp = oracle.predict(0.25, 1 * one, 2 * one, 3 * one, 6 * one, np.full(1, 0.75))  # dt = -1/2
    assert (xp == 0.25).all() and (vp == 1.25).all()
    st = nbgen.Streams(3, 9)
    q = [np.stack([st.uniform() for _ in range(3)]) for _ in range(4)]
    tj = st.uniform()
    xp, vp = oracle.predict(0.0, q[0], q[1], q[2], q[3], np.zeros(9))
    assert (xp == q[0]).all() and (vp == q[1]).all()            # dt = 0 is the identity
    xp, vp = oracle.predict(2.0, q[0], q[1], 0 * q[2], 0 * q[3], tj)
    np.testing.assert_allclose(xp, q[0] + q[1] * (2.0 - tj), rtol=1e-15)   # straight line
    assert (vp == q[1]).all()


def _kepler(t, ecc=0.5):
    """Unit-mass test particle around a fixed unit mass, a = 1, pericentre at t = 0."""
    big_e = t
    for _ in range(50):
        big_e -= (big_e - ecc * math.sin(big_e) - t) / (1 - ecc * math.cos(big_e))
    b = math.sqrt(1 - ecc * ecc)
    x = np.array([math.cos(big_e) - ecc, b * math.sin(big_e), 0.0])
    edot = 1.0 / (1 - ecc * math.cos(big_e))
    v = np.array([-math.sin(big_e) * edot, b * math.cos(big_e) * edot, 0.0])
    r = math.sqrt(x @ x)
    a = -x / r ** 3
    j = -(v / r ** 3 - 3 * (x @ v) * x / r ** 5)
    return x, v, a, j


def test_p9_predictor_order_on_kepler_orbit():
    t0 = 0.4
    s0 = [q[:, None].copy() for q in _kepler(t0)]
    ex, ev = [], []
    for dt in (0.04, 0.02, 0.01):
        xp, vp = oracle.predict(t0 + dt, *s0, np.full(1, t0))
        xt, vt, _, _ = _kepler(t0 + dt)
        ex.append(np.abs(xp[:, 0] - xt).max())
        ev.append(np.abs(vp[:, 0] - vt).max())
    assert 14 < ex[0] / ex[1] < 18 and 14 < ex[1] / ex[2] < 18      # x error ~ dt^4
    assert 7 < ev[0] / ev[1] < 9 and 7 < ev[1] / ev[2] < 9          # v error ~ dt^3


# ------------------------------------------------------------------ P12 degenerate inputs
def test_p12_degenerate():
    one = np.ones((3, 1))
    a, j, p = oracle.force(np.ones(1), one, one, [0], 0.01)
    assert (a == 0).all() and (j == 0).all() and (p == 0).all()         # N = 1
    m, x, v = nbgen.plummer(33, 4)
    a, j, p = oracle.force(m, x, v, np.zeros(0, np.int32), 0.01)
    assert a.shape == (3, 0) and p.shape == (0,)                        # N_i = 0
    m0 = np.zeros(33)
    m0[7] = 1.0
    a, j, p = oracle.force(m0, x, v, [7], 0.0)
    assert (a == 0).all() and (j == 0).all() and (p == 0).all()         # only massless others
    x[:, 1] = x[:, 0]
    a, j, p = oracle.force(m, x, v, [0, 1], 0.0)                        # R6: coincident, eps = 0
    assert np.isfinite(a).all() and np.isfinite(j).all() and np.isfinite(p).all()
    m2 = np.array([2.0, 5.0])                                           # R5: eps > 0 interacts
    x2 = np.ones((3, 2))
    v2 = np.array([[0.0, 1.0], [0.0, 2.0], [0.0, -1.0]])
    a2, j2, p2 = oracle.force(m2, x2, v2, [0, 1], 1e-2)
    assert (a2 == 0).all()
    np.testing.assert_allclose(p2, [-5.0 / 0.1, -2.0 / 0.1], rtol=1e-15)
    np.testing.assert_allclose(j2[:, 0], 5.0 * v2[:, 1] / 1e-3, rtol=1e-14)
    np.testing.assert_allclose(j2[:, 1], -2.0 * v2[:, 1] / 1e-3, rtol=1e-14)
