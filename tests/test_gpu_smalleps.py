"""-m gpu: small NON-ZERO softening, where the self pair would dominate an fp32 sum.

With eps2 > 0 the pair (i, i) has r = 0 exactly, so a pair loop that leaves it in adds m_i/eps to
the potential of particle i; at eps -> 0 that term is orders of magnitude above the real terms
(|pot_i| ~ 1) and an fp32 partial sum that holds it rounds them away.  R5 excludes the
self pair by index, the kernel must do the same *before* the fp32 sum.  PAPER.md:53 (precision of
the distance, extreme mass ratios) and PAPER.md:141 (runs at 50 / 5 / 0.5 pc softening) are the
settings this guards: ordinary stars at eps = 1e-5 .. 1e-8, one heavy unflagged particle (black
hole with a small softening) at the centre, and eps2 = 1e-32, where m eps^-3 overflows fp32.

Every threads-per-i variant of the pair kernel (N_i <= 8: 32 threads per i; <= 64: 4; else 1), a
forced j-split and both reduce modes are covered.  Tolerances: BASELINE.json's 1e-5 / 1e-4.
"""
import numpy as np
import pytest

import nbgen
import oracle
from util import check_parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

N = 8192


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _case(eps, heavy=None):
    m, x, v = nbgen.plummer(N, 4242)
    if heavy is not None:                       # one heavy, UNFLAGGED particle at rest at the centre
        m[0] = heavy
        x[:, 0] = 0.0
        v[:, 0] = 0.0
    return nbgen.configs._rest("smalleps", m, x, v, eps * eps)


def _lists():
    perm = nbgen.permutation(77, N)
    few = np.concatenate([[0], perm[:4]]).astype(np.int32)           # 5 i: 32 threads per i
    mid = np.concatenate([[0], perm[:39]]).astype(np.int32)          # 40 i: 4 threads per i
    return [("all", np.arange(N, dtype=np.int32)), ("mid", mid), ("few", few)]


def _run(nbm, c, il, splits, mode):
    with nbm.Context(c.n, len(il)) as ctx:
        ctx.load_case(c)
        ctx.predict(0.0)
        ctx.tuning(splits, mode)
        out = [q.cpu().numpy() for q in ctx.force(il, c.eps2)]
        ctx.sync()
    return out


@pytest.mark.parametrize("eps", [1e-5, 1e-6, 1e-8, 1e-16])
@pytest.mark.parametrize("heavy", [None, 2.5e-3, 1e-2])
def test_small_softening_pot(nbmod, eps, heavy):
    """eps = 1e-16 is eps2 = 1e-32: m_i eps^-3 = 1e44 overflows fp32 (inf * 0 = NaN if the self
    pair is evaluated)."""
    c = _case(eps, heavy)
    xp, vp = oracle.predict(0.0, c.x, c.v, c.a, c.j, c.t)
    worst = [0.0, 0.0, 0.0]
    for name, il in _lists():
        ref = oracle.force(c.m, xp, vp, il, c.eps2)
        for splits, mode in [(0, 0), (3, 0), (0, 1)]:
            got = _run(nbmod, c, il, splits, mode)
            assert all(np.isfinite(g).all() for g in got), (name, splits, mode)
            e = check_parity(got, ref)
            worst = [max(a, b) for a, b in zip(worst, e)]
    print("eps %.0e heavy %s: max e_acc %.2e e_jerk %.2e e_pot %.2e  (m_i/eps up to %.1e)" % (
        eps, heavy, worst[0], worst[1], worst[2], (heavy or 1.0 / N) / eps))


def test_small_softening_by_value_and_coincident(nbmod):
    """nb_force_ext has no self pair: an i-particle on top of a j-particle interacts with it
    (pot -m/eps, R5); and two distinct members of the j-set at one place do the same in nb_force."""
    c = _case(1e-6)
    c.x[:, 9] = c.x[:, 8]
    c.v[:, 9] = c.v[:, 8]
    il = np.array([8, 9, 100, 4097], np.int32)
    xp, vp = oracle.predict(0.0, c.x, c.v, c.a, c.j, c.t)
    ref = oracle.force(c.m, xp, vp, il, c.eps2)
    got = _run(nbmod, c, il, 0, 0)
    check_parity(got, ref)
    assert ref[2][0] < -0.5 * c.m[9] / 1e-6            # the coincident partner dominates pot
    # by value: append the probes as massless particles for the oracle (tests/test_gpu_ext.py)
    xi = np.ascontiguousarray(c.x[:, [8, 200]])
    vi = np.ascontiguousarray(c.v[:, [8, 200]])
    m2 = np.concatenate([c.m, np.zeros(2)])
    x2, v2 = np.concatenate([c.x, xi], 1), np.concatenate([c.v, vi], 1)
    ref2 = oracle.force(m2, x2, v2, np.array([N, N + 1], np.int32), c.eps2)
    with nbmod.Context(c.n, 2) as ctx:
        ctx.load_case(c)
        ctx.predict(0.0)
        got2 = [q.cpu().numpy() for q in ctx.force_ext(xi, vi, c.eps2)]
        ctx.sync()
    check_parity(got2, ref2)
