"""fp64 CPU oracle of the Hermite block-time-step machinery around the force call -- TEST
INFRASTRUCTURE (only tests/, smoke() and bench.py's CPU-baseline legs may import it; it shares no
code with paper_1409_5474_b200/).

What it follows.  The paper only NAMES these pieces: "4th order Hermite predictor-corrector"
(PAPER.md:129), "high >= 4th order integrators with individual time stepping [3]",
"block time steps", "only the particles are updated that require a force update at a
certain time".  It prints no formula, so the formulas are DESIGN.md's readings R12
(corrector) and R18..R21 (interpolated derivatives, time-step criterion, block rule, scheduler),
which are the textbook forms of the scheme the paper cites as [3].  Plain numpy, fp64, one
statement per formula, in the order of the readings.
"""
import numpy as np


def derivatives(a0, j0, a1, j1, dt):
    """R18: second and third time derivative of the acceleration from the Hermite interpolation
    of (a0, j0) at t0 and (a1, j1) at t1 = t0 + dt.  Returns (a2 at t1, a3), each like a0."""
    a2_0 = (-6.0 * (a0 - a1) - dt * (4.0 * j0 + 2.0 * j1)) / (dt * dt)
    a3 = (12.0 * (a0 - a1) + 6.0 * dt * (j0 + j1)) / (dt * dt * dt)
    return a2_0 + dt * a3, a3


def correct(x0, v0, a0, j0, a1, j1, dt):
    """R12: one P(EC) pass.  dt may be an array (one step per particle)."""
    v1 = v0 + (a0 + a1) * (dt / 2.0) + (j0 - j1) * (dt * dt / 12.0)
    x1 = x0 + (v0 + v1) * (dt / 2.0) + (a0 - a1) * (dt * dt / 12.0)
    return x1, v1


def _norm(q):
    return np.sqrt((q * q).sum(axis=0))


def aarseth_dt(a1, j1, a2, a3, eta):
    """R19: dt = sqrt( eta (|a||a2| + |j|^2) / (|j||a3| + |a2|^2) ), all at t1.  A vanishing
    denominator (force-free particle) gives +inf: the block rule then caps it."""
    na, nj, n2, n3 = _norm(a1), _norm(j1), _norm(a2), _norm(a3)
    num = eta * (na * n2 + nj * nj)
    den = nj * n3 + n2 * n2
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(den > 0.0, np.sqrt(num / den), np.inf)


def initial_dt(a, j, eta_s):
    """R19 (start): dt = eta_s |a| / |j|; +inf where |j| = 0."""
    na, nj = _norm(a), _norm(j)
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(nj > 0.0, eta_s * na / nj, np.inf)


def block_dt(dt_old, dt_want, t1, dt_min, dt_max):
    """R20: the new power-of-two step of a particle that has just been advanced to t1 with step
    dt_old, given the step dt_want the criterion asks for:
        shrink: halve while dt > dt_want (never below dt_min);
        grow:   double once if dt_want >= 2 dt_old, t1 is a multiple of 2 dt_old and 2 dt_old <= dt_max;
        else keep."""
    dt_old = np.asarray(dt_old, dtype=np.float64)
    dt_want = np.broadcast_to(np.asarray(dt_want, dtype=np.float64), dt_old.shape)
    out = np.empty_like(dt_old)
    for k in range(dt_old.size):
        d, w = float(dt_old.flat[k]), float(dt_want.flat[k])
        if w < d:
            while d > w and d * 0.5 >= dt_min:
                d *= 0.5
        elif w >= 2.0 * d and 2.0 * d <= dt_max and np.fmod(t1, 2.0 * d) == 0.0:
            d *= 2.0
        out.flat[k] = d
    return out


def quantise_dt(dt_want, dt_min, dt_max):
    """R20 (start): the largest power of two <= dt_want, clamped to [dt_min, dt_max]."""
    dt_want = np.asarray(dt_want, dtype=np.float64)
    out = np.empty_like(dt_want)
    for k in range(dt_want.size):
        w = float(dt_want.flat[k])
        d = dt_max
        while d > w and d * 0.5 >= dt_min:
            d *= 0.5
        out.flat[k] = d
    return out


def next_block(t, dt):
    """R21: the next block time min_j (t_j + dt_j) and the particles due then, ascending index."""
    due = t + dt
    t_next = due.min()
    return float(t_next), np.flatnonzero(due == t_next).astype(np.int32)


def corrector_step(x, v, a, j, t, dt, idx, t1, a1, j1, eta, dt_min, dt_max):
    """One corrector pass on the particles idx (R12, R18..R20), in place on the SoA state
    x, v, a, j (3, n), t, dt (n,).  a1, j1 (3, ni) are the forces at t1 in idx order."""
    h = t1 - t[idx]
    x1, v1 = correct(x[:, idx], v[:, idx], a[:, idx], j[:, idx], a1, j1, h)
    a2, a3 = derivatives(a[:, idx], j[:, idx], a1, j1, h)
    want = aarseth_dt(a1, j1, a2, a3, eta)
    new_dt = block_dt(dt[idx], want, t1, dt_min, dt_max)
    x[:, idx], v[:, idx], a[:, idx], j[:, idx] = x1, v1, a1, j1
    t[idx] = t1
    dt[idx] = new_dt
    return want
