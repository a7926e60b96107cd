"""-m gpu: the full-double pair loop (nb_set_precision(ctx, 1), force64.cu) against the
fp64 oracle.  Tolerance 1e-12 (metric R10): both sides are fp64, they differ by the order of the
additions (R9), FMA contraction and the Newton-refined reciprocal square root."""
import numpy as np
import pytest

import nbgen
import oracle
from util import rel_err_scalar, rel_err_vec

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL64 = 1.0e-12


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _case(n, seed, eps2):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    c = nbgen.configs._rest("rand", m, x, v, eps2)
    c.a, c.j = nbgen.mean_field(x, v)
    c.t = 0.25 * nbgen.Streams(seed + 2, n).uniform()
    return c


def _errs(got, ref):
    return (rel_err_vec(got[0], ref[0]).max(), rel_err_vec(got[1], ref[1]).max(),
            rel_err_scalar(got[2], ref[2]).max())


@pytest.mark.parametrize("eps2", [2.0 ** -14, 0.0])
@pytest.mark.parametrize("n,ni", [(1, 1), (130, 130), (6000, 6000), (6000, 77)])
def test_fp64_force_matches_oracle(nbmod, n, ni, eps2):
    c = _case(n, 900 + n, eps2)
    if n >= 130:
        c.flags[[11, n - 3, n // 2]] = 1                        # unsoftened among themselves (R7)
        c.x[:, 5] = c.x[:, 6]                                   # two distinct particles at one place
        c.v[:, 5] = c.v[:, 6]
        c.a[:, 5], c.j[:, 5], c.t[5] = c.a[:, 6], c.j[:, 6], c.t[6]
    il = nbgen.permutation(901, n)[:ni].astype(np.int32)
    if n >= 130:
        il[:3] = [11, 5, n - 3]
    t = 0.3
    xp, vp = oracle.predict(t, c.x, c.v, c.a, c.j, c.t)
    ref = oracle.force(c.m, xp, vp, il, eps2, c.flags if c.flags.any() else None)
    with nbmod.Context(n, max(ni, 1)) as ctx:
        ctx.precision(1)
        ctx.load_case(c)
        ctx.predict(t)
        for splits in (0, 1, 3):
            ctx.tuning(splits, 0)
            got = [q.cpu().numpy() for q in ctx.force(il, eps2)]
            if n == 1:
                assert all((g == 0).all() for g in got)
                continue
            ea, ej, ep = _errs(got, ref)
            assert ea <= TOL64 and ej <= TOL64 and ep <= TOL64, (splits, ea, ej, ep)
        again = [q.cpu().numpy() for q in ctx.force(il, eps2)]
        assert all((p == q).all() for p, q in zip(again, got))
        ctx.sync()


def test_precision_switch_needs_a_new_predict(nbmod):
    c = _case(300, 33, 1e-4)
    nb = nbmod.binding
    with nbmod.Context(c.n) as ctx:
        ctx.load_case(c)
        ctx.predict(0.0)
        ctx.precision(1)
        with pytest.raises(nb.NBError) as e:
            ctx.force(np.arange(4, dtype=np.int32), 1e-4)
        assert e.value.status == nb.NB_ERR_STATE
        with pytest.raises(nb.NBError):
            ctx.precision(2)
        ctx.predict(0.0)
        ctx.force(np.arange(4, dtype=np.int32), 1e-4)
        ctx.precision(0)
        ctx.predict(0.0)
        ctx.force(np.arange(4, dtype=np.int32), 1e-4)
        ctx.sync()


@pytest.mark.parametrize("with_jerk", [True, False])
def test_fp64_force_ext(nbmod, with_jerk):
    n, ni, eps2, t = 5000, 333, 2.0 ** -12, 0.2
    c = _case(n, 950, eps2)
    _, xi, vi = nbgen.plummer(ni, 951)
    xi = np.ascontiguousarray(xi + 0.3)
    xp, vp = oracle.predict(t, c.x, c.v, c.a, c.j, c.t)
    mm = np.concatenate([c.m, np.zeros(ni)])
    ref = oracle.force(mm, np.concatenate([xp, xi], 1), np.concatenate([vp, vi if with_jerk else 0 * vi], 1),
                       np.arange(n, n + ni, dtype=np.int32), eps2)
    with nbmod.Context(n, ni) as ctx:
        ctx.precision(1)
        ctx.load_case(c)
        ctx.predict(t)
        acc, jrk, pot = ctx.force_ext(xi, vi if with_jerk else None, eps2)
        ga, gp = acc.cpu().numpy(), pot.cpu().numpy()
        assert rel_err_vec(ga, ref[0]).max() <= TOL64 and rel_err_scalar(gp, ref[2]).max() <= TOL64
        if with_jerk:
            assert rel_err_vec(jrk.cpu().numpy(), ref[1]).max() <= TOL64
        else:
            assert jrk is None
        ctx.sync()


def test_extreme_mass_ratio_needs_fp64(nbmod):
    """PAPER.md:53's case: planetesimals (m = 1e-12) around a black hole (m = 1).  The mutual
    perturbation of the planetesimals is what an integration is after; it is 1e-9 of the force.
    Measured as the force with the black hole's exact two-body term subtracted: the fp64 loop
    keeps it to 1e-4, the mixed-precision loop (fp32 pair terms) cannot."""
    n = 4097
    s = nbgen.Streams(77, n)
    r = 1.0 + 0.1 * s.uniform()
    ph = 2.0 * np.pi * s.uniform()
    x = np.stack([r * np.cos(ph), r * np.sin(ph), 0.01 * (s.uniform() - 0.5)])
    v = np.stack([-np.sin(ph), np.cos(ph), 0.0 * ph]) / np.sqrt(r)
    m = np.full(n, 1.0e-12)
    x[:, 0], v[:, 0], m[0] = 0.0, 0.0, 1.0
    eps2 = 1e-8
    il = np.arange(1, n, dtype=np.int32)
    ref = oracle.force(m, x, v, il, eps2)
    m0 = m.copy()
    m0[0] = 0.0
    pert = oracle.force(m0, x, v, il, eps2)[0]                 # planetesimals only
    out = {}
    for mode in (0, 1):
        with nbmod.Context(n) as ctx:
            ctx.precision(mode)
            ctx.set_j(m, x, v)
            ctx.predict(0.0)
            acc = ctx.force(il, eps2)[0].cpu().numpy()
            ctx.sync()
        bh = ref[0] - pert                                      # the black hole's term (oracle)
        out[mode] = np.sqrt(((acc - bh - pert) ** 2).sum(0)) / np.sqrt((pert ** 2).sum(0))
    assert np.median(out[1]) < 1e-4 and out[1].max() < 1e-2
    assert np.median(out[0]) > 1.0                              # fp32 pair terms: perturbation lost


def test_config3_full_size_fp64_sampled(nbmod):
    c = nbgen.config3()
    il = c.i_lists[2]                                           # 16384 active i
    with nbmod.Context(c.n, len(il)) as ctx:
        ctx.precision(1)
        ctx.load_case(c)
        ctx.predict(c.t_now)
        got = [q.cpu().numpy() for q in ctx.force(il, c.eps2)]
        ctx.sync()
    pos = nbgen.sample_positions(nbgen.SEED0 * 100 + 64, len(il), 512)
    xp, vp = oracle.predict(c.t_now, c.x, c.v, c.a, c.j, c.t)
    ref = oracle.force(c.m, xp, vp, il[pos], c.eps2)
    ea, ej, ep = _errs([got[0][:, pos], got[1][:, pos], got[2][pos]], ref)
    print("cfg3 fp64 sampled", ea, ej, ep)
    assert ea <= TOL64 and ej <= 10 * TOL64 and ep <= TOL64
