"""-m gpu: the HOST-buffer entry points -- the path bench.py's `e2e` number times -- against the oracle,
and the small boundary calls no other test touches (nb_set_stream on a non-default stream,
nb_block_forces, the state rules after nb_correct / nb_init_steps, by-value forces on an empty
j-set, a zero step).  SURVEY.md 8(b) "host-pointer convenience"; PAPER.md:83 (the host link)."""
import numpy as np
import pytest

import nbgen
import oracle
from oracle import hermite as H
from util import check_parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _case(n, seed, eps2=2.0 ** -14):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    c = nbgen.configs._rest("host", m, x, v, eps2)
    c.a, c.j = nbgen.mean_field(x, v)
    c.t = 0.125 * nbgen.Streams(seed + 2, n).uniform()
    return c


def _host(a, pinned):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return t.pin_memory() if pinned else t


@pytest.mark.parametrize("pinned", [True, False])
def test_host_path_matches_oracle(nbmod, pinned):
    """nb_set_j_host -> nb_update_j_host -> nb_predict -> nb_force_host, exactly bench.py's e2e step,
    on 6000 particles (47 j-tiles, 24 i-tiles, ragged tails), every particle checked."""
    nb = nbmod.binding
    n, t1 = 6000, 0.25
    c, c2 = _case(n, 301), _case(n, 302)
    idx = nbgen.permutation(303, n)[:2500].astype(np.int32)
    il = nbgen.permutation(304, n)[:5555].astype(np.int32)
    with nbmod.Context(n) as ctx:
        keep = [_host(q, pinned) for q in (c.m, c.x, c.v, c.a, c.j, c.t)]
        nb.nb_set_j_host(ctx.h, 0, n, *keep)
        upd = [_host(getattr(c2, f)[..., idx], pinned) for f in ("m", "x", "v", "a", "j", "t")]
        h_idx, h_il = _host(idx, pinned), _host(il, pinned)
        nb.nb_update_j_host(ctx.h, h_idx, len(idx), *upd)
        nb.nb_predict(ctx.h, t1)
        acc, jrk, pot = (_host(np.empty((3, len(il))), pinned), _host(np.empty((3, len(il))), pinned),
                         _host(np.empty(len(il)), pinned))
        nb.nb_force_host(ctx.h, h_il, len(il), c.eps2, acc, jrk, pot)      # returns synchronised
        got = [acc.numpy().copy(), jrk.numpy().copy(), pot.numpy().copy()]
        # the same call with device-resident buffers gives the same bits (deterministic reduce)
        dev = [q.cpu().numpy() for q in ctx.force(il, c.eps2)]
        ctx.sync()
    for f in ("m", "x", "v", "a", "j", "t"):
        getattr(c, f)[..., idx] = getattr(c2, f)[..., idx]
    xp, vp = oracle.predict(t1, c.x, c.v, c.a, c.j, c.t)
    ref = oracle.force(c.m, xp, vp, il, c.eps2)
    print("host path (pinned=%s):" % pinned, check_parity(got, ref))
    assert all(np.array_equal(g, d) for g, d in zip(got, dev))


def test_set_stream_non_default(nbmod):
    nb = nbmod.binding
    c = _case(3000, 311)
    il = np.arange(c.n, dtype=np.int32)
    side = torch.cuda.Stream()
    with nbmod.Context(c.n) as ctx:
        ctx.load_case(c)
        ctx.sync()
        nb.nb_set_stream(ctx.h, side.cuda_stream)
        with torch.cuda.stream(side):
            ctx.predict(0.1)
            got = ctx.force(il, c.eps2)
        ctx.sync()                                    # synchronises the context's (side) stream
        got = [q.cpu().numpy() for q in got]
    xp, vp = oracle.predict(0.1, c.x, c.v, c.a, c.j, c.t)
    check_parity(got, oracle.force(c.m, xp, vp, il, c.eps2))


def test_block_forces_and_state_rules(nbmod):
    """nb_block_forces returns the forces nb_step used; after nb_correct / nb_init_steps / nb_step
    the packed predicted state is stale whatever the block size (NB_ERR_STATE until nb_predict)."""
    nb = nbmod.binding
    n, eps2, eta, lo, hi = 1500, 2.0 ** -12, 0.02, 2.0 ** -18, 2.0 ** -5
    m, x, v = nbgen.plummer(n, 321)
    il = np.arange(n, dtype=np.int32)
    with nbmod.Context(n) as ctx:
        with pytest.raises(nb.NBError) as e:
            nb.nb_block_forces(ctx.h)
        assert e.value.status == nb.NB_ERR_STATE
        ctx.set_j(m, x, v)
        ctx.predict(0.0)
        ga, gj, gp = ctx.force(il, eps2)
        ctx.init_steps(il, ga, gj, eta, lo, hi)
        with pytest.raises(nb.NBError) as e:           # stored (a, jerk) changed
            ctx.force(il[:300], eps2)
        assert e.value.status == nb.NB_ERR_STATE
        for fused in (True, False):
            ctx.fused(fused)
            st = ctx.state().cpu().numpy()
            t1, ni = ctx.step(eps2, eta, lo, hi)
            pa, pj, pp = nb.nb_block_forces(ctx.h)
            rt1, idx = H.next_block(st[13], st[14])
            assert t1 == rt1 and ni == len(idx)
            view = nbmod.context._DeviceView
            a1 = torch.as_tensor(view(pa, 3 * ni, "<f8"), device=ctx.device).cpu().numpy().reshape(3, ni)
            j1 = torch.as_tensor(view(pj, 3 * ni, "<f8"), device=ctx.device).cpu().numpy().reshape(3, ni)
            p1 = torch.as_tensor(view(pp, ni, "<f8"), device=ctx.device).cpu().numpy()
            xp, vp = oracle.predict(t1, st[1:4], st[4:7], st[7:10], st[10:13], st[13])
            check_parity([a1, j1, p1], oracle.force(st[0], xp, vp, idx, eps2))
            with pytest.raises(nb.NBError) as e:       # whatever the block size was
                ctx.force(il[:300], eps2)
            assert e.value.status == nb.NB_ERR_STATE
        ctx.predict(t1)
        ctx.force(il[:300], eps2)
        z = torch.zeros((3, 2), dtype=torch.float64, device=ctx.device)
        ctx.correct(np.array([3, 4], np.int32), t1 + lo, z, z, eta, lo, hi)
        with pytest.raises(nb.NBError) as e:
            ctx.force(il[:300], eps2)
        assert e.value.status == nb.NB_ERR_STATE
        ctx.sync()


def test_zero_step_is_reported(nbmod):
    """Steps never set (dt = 0): the scheduler returns t = min t_j, the corrector must not divide by
    h = 0 -- the particle is left alone and nb_sync reports NB_ERR_STATE."""
    nb = nbmod.binding
    n = 300
    m, x, v = nbgen.plummer(n, 331)
    with nbmod.Context(n) as ctx:
        ctx.set_j(m, x, v)
        before = ctx.state().cpu().numpy()
        t1, ni = ctx.step(1e-4, 0.02, 2.0 ** -10, 2.0 ** -4)
        assert t1 == 0.0 and ni == n
        with pytest.raises(nb.NBError) as e:
            ctx.sync()
        assert e.value.status == nb.NB_ERR_STATE
        after = ctx.state().cpu().numpy()
        assert np.array_equal(before[:7], after[:7]) and np.isfinite(after).all()
        ctx.sync()                                     # latch cleared


def test_by_value_on_empty_j_set(nbmod):
    """n = 0: nb_force_ext sums over nothing and must write zeros (not NaN)."""
    xi = np.random.default_rng(5).normal(size=(3, 40))
    with nbmod.Context(64, 64) as ctx:
        ctx.predict(0.0)
        a, j, p = ctx.force_ext(xi, xi, 1e-4)
        ctx.sync()
        assert all((q.cpu().numpy() == 0.0).all() for q in (a, j, p))
