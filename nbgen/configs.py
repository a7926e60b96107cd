"""The five BASELINE.json configs as seeded synthetic particle sets (recipe: DESIGN.md "Input
recipe", after SURVEY.md §8(d)).  They stand in for the paper's own initial conditions
("see [15] for details"), which are not available.  Every builder takes an optional
size so that tests can run the same recipe at sizes the oracle finishes in seconds.

No force arithmetic here: only sampling, placement and bookkeeping.
"""
from dataclasses import dataclass, field

import numpy as np

from .plummer import HENON_A, mean_field, plummer
from .rng import Streams, integers, permutation

SEED0 = 140954740  # config c uses SEED0 + c


@dataclass
class Case:
    """j-particle state in SoA fp64 plus what one benchmark/parity case needs around it."""
    name: str
    m: np.ndarray            # (N,)
    x: np.ndarray            # (3, N)
    v: np.ndarray            # (3, N)
    a: np.ndarray            # (3, N)  stored acceleration at t (predictor input)
    j: np.ndarray            # (3, N)  stored jerk at t
    t: np.ndarray            # (N,)    time each particle's state refers to
    flags: np.ndarray        # (N,) uint8; bit 0 = pairs among flagged particles are unsoftened
    eps2: float
    t_now: float = 0.0
    i_lists: list = field(default_factory=list)   # int32 arrays, one per force call
    dt: float = 0.0          # shared step of config 2
    steps: int = 0

    @property
    def n(self):
        return self.m.shape[0]


def _rest(name, m, x, v, eps2, **kw):
    n = m.shape[0]
    z = np.zeros((3, n))
    return Case(name, m, x, v, z.copy(), z.copy(), np.zeros(n), np.zeros(n, np.uint8), eps2, **kw)


def config1(n=1024):
    """Plummer sphere, Henon units, eps = 0.01, all active: once in index order, once shuffled."""
    s = SEED0 + 1
    m, x, v = plummer(n, s)
    c = _rest("cfg1_plummer", m, x, v, 1.0e-4)
    c.i_lists = [np.arange(n, dtype=np.int32), permutation(s * 100 + 99, n)]
    return c


def config2(n=65536, steps=10):
    """Plummer sphere, eps = 1/256, all active, predictor + force over `steps` shared steps of
    dt = 1/256 (the harness runs the corrector, R12)."""
    s = SEED0 + 2
    m, x, v = plummer(n, s)
    c = _rest("cfg2_hermite", m, x, v, 2.0 ** -16, dt=2.0 ** -8, steps=steps)
    c.i_lists = [np.arange(n, dtype=np.int32)]
    return c


def config3(n=1 << 20, sizes=(1, 1024, 16384, 262144, 1 << 20)):
    """Plummer sphere in a synthetic block-time-step state: particle j sits at level k_j in
    {4..12}, dt_j = 2^-k_j, t_j = floor(t_now/dt_j) dt_j with t_now = 1707/4096; stored (a, jerk)
    are the smooth Plummer field at the stored (x, v).  Active subsets are nested prefixes of one
    seeded permutation, passed unsorted."""
    s = SEED0 + 3
    m, x, v = plummer(n, s)
    c = _rest("cfg3_blockstep", m, x, v, 2.0 ** -20)
    c.a, c.j = mean_field(x, v, HENON_A, 1.0)
    c.t_now = 1707.0 * 2.0 ** -12          # 0b011010101011: a different t_j at every level
    dtj = 2.0 ** -integers(s * 100 + 98, n, 4, 12).astype(np.float64)
    c.t = np.floor(c.t_now / dtj) * dtj
    perm = permutation(s * 100 + 99, n)
    c.i_lists = [perm[:k].copy() for k in sizes if k <= n]
    return c


def config4(n_gal=1 << 19, sep=10.0, peri=1.0, m_bh=1.0e-3):
    """Two Plummer spheres (scale 1, galaxy mass = n_gal * 2^-20 at full size -> 1/2), a flagged
    black hole at each centre, on a parabolic approach with pericentre `peri` for two point
    masses; order: stars A, BH A, stars B, BH B.  eps2 = 1e-6, BH-BH pair unsoftened."""
    s = SEED0 + 4
    m_gal = 0.5
    parts = []
    m_pt = m_gal + m_bh
    vt = np.sqrt(2.0 * (2.0 * m_pt) * peri) / sep           # angular momentum of a parabola
    vr = -np.sqrt(2.0 * (2.0 * m_pt) / sep - vt * vt)       # inward
    dx = np.array([sep, 0.0, 0.0])
    dv = np.array([vr, vt, 0.0])
    for g, sign in ((0, -0.5), (1, +0.5)):
        m, x, v = plummer(n_gal, s * 100 + g, a=1.0, mass=m_gal)
        m = np.append(m, m_bh)
        x = np.concatenate([x, np.zeros((3, 1))], 1) + (sign * dx)[:, None]
        v = np.concatenate([v, np.zeros((3, 1))], 1) + (sign * dv)[:, None]
        parts.append((m, x, v))
    m = np.concatenate([p[0] for p in parts])
    x = np.ascontiguousarray(np.concatenate([p[1] for p in parts], 1))
    v = np.ascontiguousarray(np.concatenate([p[2] for p in parts], 1))
    c = _rest("cfg4_merger", m, x, v, 1.0e-6)
    c.flags[n_gal] = 1
    c.flags[2 * n_gal + 1] = 1
    c.i_lists = [np.arange(c.n, dtype=np.int32)]
    return c


def config5(n_stars=1 << 22, n_active=1 << 20, n_gal=11, radius=20.0):
    """Group of 11 Plummer spheres: sizes log-uniform in [2^17, 2^20] rescaled to n_stars, star
    mass 1/n_stars, scale a_g = (n_g / max n)^(1/3), centres uniform in a sphere of radius 20,
    cold (no bulk velocity), one BH of 1 % of its galaxy's mass at each centre; order: stars g,
    BH g.  One softening for all pairs (flags stay clear).  Active: n_active entries of a seeded
    permutation."""
    s = SEED0 + 5
    w = 2.0 ** (17.0 + 3.0 * Streams(s * 100 + 96, n_gal).uniform())
    ng = np.rint(n_stars * w / w.sum()).astype(np.int64)
    ng[np.argmax(ng)] += n_stars - ng.sum()
    cs = Streams(s * 100 + 97, n_gal)
    rc = radius * cs.uniform() ** (1.0 / 3.0)
    cz = 2.0 * cs.uniform() - 1.0
    ph = 2.0 * np.pi * cs.uniform()
    sz = np.sqrt(1.0 - cz * cz)
    centres = rc * np.stack([sz * np.cos(ph), sz * np.sin(ph), cz])
    ms, xs, vs = [], [], []
    for g in range(n_gal):
        mg = ng[g] / n_stars
        m, x, v = plummer(int(ng[g]), s * 100 + g, a=(ng[g] / ng.max()) ** (1.0 / 3.0), mass=mg)
        ms += [m, [0.01 * mg]]
        xs += [x + centres[:, g:g + 1], centres[:, g:g + 1]]
        vs += [v, np.zeros((3, 1))]
    m = np.concatenate(ms)
    x = np.ascontiguousarray(np.concatenate(xs, 1))
    v = np.ascontiguousarray(np.concatenate(vs, 1))
    c = _rest("cfg5_group", m, x, v, 1.0e-6)
    c.i_lists = [permutation(s * 100 + 99, c.n)[:min(n_active, c.n)].copy()]
    return c


def sample_positions(seed, n_list, n_sample):
    """Seed-sampled positions k into an i_list of length n_list (sorted, unique)."""
    if n_sample >= n_list:
        return np.arange(n_list, dtype=np.int64)
    return np.sort(permutation(seed, n_list)[:n_sample].astype(np.int64))
