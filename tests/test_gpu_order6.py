"""-m gpu: the 6th-order variant (nb_set_order 6 + nb_force6: acc, jerk, snap, pot) against
oracle.force6 on the predicted state (positions and velocities by R1, accelerations by R22).
Tolerances: 1e-5 acc and pot, 1e-4 jerk (BASELINE.json), 1e-3 snap (DESIGN.md
derives it: snap is a sum of terms ~ s^-5/2 with heavier cancellation than jerk).  PAPER.md:35."""
import numpy as np
import pytest

import nbgen
import oracle
from util import check_parity, rel_err_vec

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL_SNP = 1.0e-3


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _case(n, seed, eps2):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    c = nbgen.configs._rest("o6", m, x, v, eps2)
    c.a, c.j = nbgen.mean_field(x, v)
    c.t = 0.125 * nbgen.Streams(seed + 2, n).uniform()
    return c


def _ref(c, t, il, eps2):
    xp, vp = oracle.predict(t, c.x, c.v, c.a, c.j, c.t)
    ap = oracle.predict_acc(t, c.a, c.j, c.t)
    return oracle.force6(c.m, xp, vp, ap, il, eps2, c.flags if c.flags.any() else None)


def _gpu(nbm, c, t, il, eps2, splits=0):
    with nbm.Context(c.n, max(1, len(il))) as ctx:
        ctx.order(6)
        ctx.load_case(c)
        ctx.predict(t)
        ctx.tuning(splits, 0)
        out = [q.cpu().numpy() for q in ctx.force6(il, eps2)]
        # the 4th-order call still works beside it and agrees on acc, jerk, pot
        f4 = [q.cpu().numpy() for q in ctx.force(il, eps2)]
        ctx.sync()
    return out, f4


def _check(got, ref):
    e = check_parity([got[0], got[1], got[3]], [ref[0], ref[1], ref[3]])
    es = rel_err_vec(got[2], ref[2]).max() if ref[3].size else 0.0
    assert es <= TOL_SNP, ("snap", es)
    return e + (es,)


@pytest.mark.parametrize("n", [2, 33, 257, 1025, 3000])
@pytest.mark.parametrize("eps2", [2.0 ** -12, 0.0])
def test_force6_matches_oracle(nbmod, n, eps2):
    c = _case(n, 600 + n, eps2)
    if n >= 257:
        c.flags[[3, 130, n - 1]] = 1
        c.x[:, 130] = c.x[:, 3] + np.array([1e-3, 2e-3, -1e-3])       # a tight flagged pair
        c.x[:, 7] = c.x[:, 6]                                          # coincident, distinct
    il = np.arange(n, dtype=np.int32)
    got, f4 = _gpu(nbmod, c, 0.2, il, eps2)
    ref = _ref(c, 0.2, il, eps2)
    print("order 6, n=%d eps2=%g:" % (n, eps2), _check(got, ref))
    check_parity(f4, [ref[0], ref[1], ref[3]])


def test_force6_subsets_splits_and_errors(nbmod):
    nb = nbmod.binding
    c = _case(5000, 650, 2.0 ** -14)
    il = nbgen.permutation(651, c.n)[:700].astype(np.int32)
    il[5] = il[6]                                                     # duplicate
    ref = _ref(c, 0.3, il, c.eps2)
    outs = []
    for splits in (0, 1, 7):
        got, _ = _gpu(nbmod, c, 0.3, il, c.eps2, splits)
        _check(got, ref)
        outs.append(got)
    assert all(np.array_equal(p, q) for p, q in zip(outs[1], _gpu(nbmod, c, 0.3, il, c.eps2, 1)[0]))   # deterministic
    with nbmod.Context(c.n) as ctx:
        ctx.load_case(c)
        ctx.predict(0.3)
        with pytest.raises(nb.NBError) as e:                          # order 4: no such records
            ctx.force6(il, c.eps2)
        assert e.value.status == nb.NB_ERR_STATE
        ctx.order(6)
        with pytest.raises(nb.NBError) as e:                          # order changed: predict first
            ctx.force6(il, c.eps2)
        assert e.value.status == nb.NB_ERR_STATE
        ctx.predict(0.3)
        bad = il.copy()
        bad[2] = c.n
        a, j, s, p = [q.cpu().numpy() for q in ctx.force6(bad, c.eps2)]
        with pytest.raises(nb.NBError) as e:
            ctx.sync()
        assert e.value.status == nb.NB_ERR_INDEX
        assert np.isnan(s[:, 2]).all() and np.isnan(p[2])
        keep = np.arange(len(il)) != 2
        _check([a[:, keep], j[:, keep], s[:, keep], p[keep]], [q[..., keep] for q in ref])


def test_force6_rigid_rotation_on_gpu(nbmod):
    """P13 on the GPU: a rigidly rotating configuration has snap = W x (W x acc)."""
    n = 300
    rng = np.random.default_rng(77)
    x = rng.normal(size=(3, n))
    m = rng.uniform(0.1, 1.0, n) / n
    w = np.array([0.3, -0.2, 0.5])[:, None]
    v = np.cross(w, x, axis=0)
    a = np.cross(w, v, axis=0)
    c = nbgen.configs._rest("rot", m, x, v, 1e-2)
    c.a = a
    il = np.arange(n, dtype=np.int32)
    got, _ = _gpu(nbmod, c, 0.0, il, c.eps2)
    sr = np.cross(w, np.cross(w, got[0], axis=0), axis=0)
    assert rel_err_vec(got[2], sr).max() <= TOL_SNP
