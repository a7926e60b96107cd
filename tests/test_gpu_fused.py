"""-m gpu: nb_force_fused (predictor inside the pair loop, one pass over the j-store, <= 8 active
particles, fp64 throughout; fused.cu) against oracle.predict + oracle.force, tolerance 1e-12."""
import numpy as np
import pytest

import nbgen
import oracle
from oracle import hermite as H
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
    m, x, v = nbgen.plummer(max(n, 2), seed)
    m, x, v = m[:n].copy(), np.ascontiguousarray(x[:, :n]), np.ascontiguousarray(v[:, :n])
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    c = nbgen.configs._rest("rand", m, x, v, eps2)
    c.a, c.j = nbgen.mean_field(x, v)
    c.t = 0.25 * nbgen.Streams(seed + 2, n).uniform()
    return c


@pytest.mark.parametrize("eps2", [2.0 ** -14, 0.0])
@pytest.mark.parametrize("n,ni", [(1, 1), (3, 2), (1001, 1), (1001, 3), (1001, 4), (100003, 5), (100003, 8)])
def test_fused_force_matches_oracle(nbmod, n, ni, eps2):
    c = _case(n, 1200 + n + ni, eps2)
    il = nbgen.permutation(1201, n)[:ni].astype(np.int32)
    if n > 1000:
        c.flags[[7, n - 2, int(il[0])]] = 1                    # one active particle is flagged (R7)
        c.x[:, 5], c.v[:, 5] = c.x[:, 6], c.v[:, 6]            # coincident pair
        c.a[:, 5], c.j[:, 5], c.t[5] = c.a[:, 6], c.j[:, 6], c.t[6]
        if ni >= 3:
            il[1], il[2] = 5, 7
    t = 0.3
    xp, vp = oracle.predict(t, c.x, c.v, c.a, c.j, c.t)
    ref = oracle.force(c.m, xp, vp, il, eps2, c.flags if c.flags.any() else None)
    with nbmod.Context(n, 8) as ctx:
        ctx.load_case(c)                                       # note: no nb_predict
        got = [q.cpu().numpy() for q in ctx.force_fused(t, il, eps2)]
        again = [q.cpu().numpy() for q in ctx.force_fused(t, il, eps2)]
        ctx.sync()
    assert all((p == q).all() for p, q in zip(again, got))     # deterministic (R9)
    if n == 1:
        assert all((g == 0).all() for g in got)
        return
    assert rel_err_vec(got[0], ref[0]).max() <= TOL64
    assert rel_err_vec(got[1], ref[1]).max() <= TOL64
    assert rel_err_scalar(got[2], ref[2]).max() <= TOL64


def test_fused_argument_errors(nbmod):
    nb = nbmod.binding
    c = _case(100, 5, 1e-4)
    with nbmod.Context(100, 16) as ctx:
        ctx.load_case(c)
        z = torch.zeros((3, 9), dtype=torch.float64, device=ctx.device)
        p = torch.zeros(9, dtype=torch.float64, device=ctx.device)
        il = torch.arange(9, dtype=torch.int32, device=ctx.device)
        with pytest.raises(nb.NBError) as e:
            nb.nb_force_fused(ctx.h, 0.0, il, 9, 1e-4, z, z, p)             # more than NB_FUSED_MAX
        assert e.value.status == nb.NB_ERR_ARG
        with pytest.raises(nb.NBError):
            nb.nb_force_fused(ctx.h, float("nan"), il, 2, 1e-4, z, z, p)
        nb.nb_force_fused(ctx.h, 0.0, il, 0, 1e-4, None, None, None)        # ni = 0: no-op
        bad = torch.tensor([3, 100], dtype=torch.int32, device=ctx.device)  # index out of range
        nb.nb_force_fused(ctx.h, 0.0, bad, 2, 1e-4, z, z, p)
        with pytest.raises(nb.NBError) as e:
            ctx.sync()
        assert e.value.status == nb.NB_ERR_INDEX
        assert torch.isnan(p[1]).item() and torch.isfinite(p[0]).item()


def test_nb_step_with_and_without_the_fused_path(nbmod):
    """The same block steps taken through nb_force_fused (blocks of <= 8) and through predict +
    mixed-precision force agree to the mixed path's tolerance, and both follow the oracle's schedule."""
    n, eps2, eta = 1024, 1e-4, 0.02
    lo, hi = 2.0 ** -18, 2.0 ** -5
    m, x, v = nbgen.plummer(n, 606)
    il = np.arange(n, dtype=np.int32)
    a, j, _ = oracle.force(m, x, v, il, eps2)
    dt = H.quantise_dt(H.initial_dt(a, j, eta), lo, hi)
    out = {}
    for fused in (True, False):
        with nbmod.Context(n) as ctx:
            ctx.fused(fused)
            ctx.set_j(m, x, v, a, j, np.zeros(n))
            ctx.set_dt(dt)
            sizes, small = [], 0
            for step in range(40):
                t1, ni = ctx.step(eps2, eta, lo, hi)
                sizes.append((t1, ni))
                small += ni <= 8
            out[fused] = (ctx.state().cpu().numpy(), sizes)
            ctx.sync()
        assert small >= 5                                       # the fused path was really taken
    sa, sb = out[True], out[False]
    same = [p == q for p, q in zip(sa[1], sb[1])]
    k = same.index(False) if False in same else len(same)       # schedules may part late (step choice)
    assert k >= 20
    if k == len(same):
        assert np.abs(sa[0][1:7] - sb[0][1:7]).max() < 1e-7
