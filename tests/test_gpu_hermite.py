"""-m gpu: the device block-step layer (nb_next_block, nb_init_steps, nb_correct, nb_step) against
oracle/hermite.py (R12, R18..R21), through the C-ABI."""
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


def _state(n, seed, levels=(4, 12)):
    """Random block-step state: dyadic steps 2^-k, particle times on their own step grid."""
    s = nbgen.Streams(seed, n)
    m = 0.5 + s.uniform()
    x = np.stack([s.uniform() - 0.5 for _ in range(3)])
    v = np.stack([s.uniform() - 0.5 for _ in range(3)])
    a = np.stack([s.uniform() - 0.5 for _ in range(3)])
    j = np.stack([s.uniform() - 0.5 for _ in range(3)]) * 4.0
    k = levels[0] + np.floor(s.uniform() * (levels[1] - levels[0] + 1)).astype(np.int64)
    dt = 2.0 ** -k.astype(np.float64)
    t = np.floor(s.uniform() * 37.0) * dt
    return m, x, v, a, j, t, dt


def _load(ctx, m, x, v, a, j, t, dt):
    ctx.set_j(m, x, v, a, j, t)
    ctx.set_dt(dt)


def _list(ctx, view, ni):
    """The context-owned device list (int32 tensor view) on the host."""
    assert view.shape[0] == ni
    return view.cpu().numpy()


@pytest.mark.parametrize("n", [1, 255, 1000, 100003])
def test_next_block_matches_oracle(nbmod, n):
    m, x, v, a, j, t, dt = _state(n, 401 + n)
    with nbmod.Context(n) as ctx:
        _load(ctx, m, x, v, a, j, t, dt)
        t1, ni, addr = ctx.next_block()
        rt, ridx = H.next_block(t, dt)
        assert t1 == rt and ni == len(ridx)                      # bit-exact (R21)
        assert np.array_equal(_list(ctx, addr, ni), ridx)
        # everything due at once, and a negative time
        t2 = np.full(n, -3.0)
        d2 = np.full(n, 0.25)
        _load(ctx, m, x, v, a, j, t2, d2)
        t1, ni, addr = ctx.next_block()
        assert t1 == -2.75 and ni == n
        assert np.array_equal(_list(ctx, addr, ni), np.arange(n, dtype=np.int32))


def test_next_block_overflow_is_reported(nbmod):
    n = 4096
    m, x, v, a, j, t, dt = _state(n, 77)
    with nbmod.Context(n, 16) as ctx:
        _load(ctx, m, x, v, a, j, np.zeros(n), np.full(n, 0.5))
        with pytest.raises(nbmod.binding.NBError) as e:
            ctx.next_block()
        assert e.value.status == nbmod.binding.NB_ERR_ARG


def _compare_state(got, ref, tol_xv, tol_aj):
    m, x, v, a, j, t, dt = ref
    g = got.cpu().numpy()
    assert np.array_equal(g[0], m) and np.array_equal(g[13], t)
    for lo, q, tol in ((1, x, tol_xv), (4, v, tol_xv), (7, a, tol_aj), (10, j, tol_aj)):
        d = np.abs(g[lo:lo + 3] - q).max()
        assert d <= tol * max(1.0, np.abs(q).max()), (lo, d)
    return g[14]


def test_correct_and_init_match_oracle(nbmod):
    n, ni = 5000, 1777
    m, x, v, a, j, t, dt = _state(n, 91)
    idx = nbgen.permutation(92, n)[:ni].astype(np.int32)
    idx = idx[np.argsort(t[idx] + dt[idx], kind="stable")]
    t1 = 40.0 * 2.0 ** -4                                        # ahead of every particle time
    s = nbgen.Streams(93, ni)
    a1 = np.stack([s.uniform() - 0.5 for _ in range(3)])
    j1 = np.stack([s.uniform() - 0.5 for _ in range(3)]) * 4.0
    eta, lo, hi = 0.02, 2.0 ** -14, 2.0 ** -3
    # the step taken is h = t1 - t_i; the stored step enters the block rule only
    with nbmod.Context(n) as ctx:
        _load(ctx, m, x, v, a, j, t, dt)
        d_a1 = torch.from_numpy(a1).to(ctx.device)
        d_j1 = torch.from_numpy(j1).to(ctx.device)
        ctx.correct(idx, t1, d_a1, d_j1, eta, lo, hi)
        got = ctx.state()
        ctx.sync()
        rx, rv, ra, rj, rt, rdt = x.copy(), v.copy(), a.copy(), j.copy(), t.copy(), dt.copy()
        want = H.corrector_step(rx, rv, ra, rj, rt, rdt, idx, t1, a1, j1, eta, lo, hi)
        gdt = _compare_state(got, (m, rx, rv, ra, rj, rt, rdt), 1e-14, 0.0)
        # the power-of-two decision: equal, except where the wanted step sits within rounding of a
        # decision threshold (both sides decide in fp64; FMA contraction moves `want` by ~1e-16)
        diff = np.flatnonzero(gdt != rdt)
        for i in diff:
            k = int(np.flatnonzero(idx == i)[0])
            r = want[k] / rdt[i]
            assert min(abs(r - 1.0), abs(r - 2.0), abs(r - 0.5)) < 1e-12
        assert len(diff) <= 2

        # start: a, j stored and first steps quantised (R19, R20)
        ctx.init_steps(idx, d_a1, d_j1, 0.01, lo, hi)
        g = ctx.state().cpu().numpy()
        ref = H.quantise_dt(H.initial_dt(a1, j1, 0.01), lo, hi)
        assert np.array_equal(g[7:10][:, idx], a1) and np.array_equal(g[10:13][:, idx], j1)
        assert np.array_equal(g[14][idx], ref)
        others = np.setdiff1d(np.arange(n), idx)
        assert np.array_equal(g[14][others], gdt[others])


def test_bad_step_bounds_are_rejected(nbmod):
    with nbmod.Context(16) as ctx:
        z = torch.zeros((3, 1), dtype=torch.float64, device=ctx.device)
        il = np.zeros(1, np.int32)
        for lo, hi in ((0.3, 0.5), (0.5, 0.25), (0.0, 0.5), (0.25, 0.75)):
            with pytest.raises(nbmod.binding.NBError):
                ctx.correct(il, 1.0, z, z, 0.01, lo, hi)


def test_nb_step_lockstep_with_oracle(nbmod):
    """Whole block steps.  The oracle drives the trajectory; before every step the GPU context is
    given the oracle's stored state, so nothing the oracle consumes ever comes from the GPU."""
    n, eps2, eta = 2048, 2.0 ** -12, 0.02
    lo, hi = 2.0 ** -18, 2.0 ** -5
    m, x, v = nbgen.plummer(n, 555)
    il = np.arange(n, dtype=np.int32)
    a, j, _ = oracle.force(m, x, v, il, eps2)
    t = np.zeros(n)
    dt = H.quantise_dt(H.initial_dt(a, j, eta), lo, hi)
    with nbmod.Context(n) as ctx:
        # start on the device: forces at t = 0, first steps
        ctx.set_j(m, x, v)
        ctx.predict(0.0)
        ga, gj, gp = ctx.force(il, eps2)
        ctx.init_steps(il, ga, gj, eta, lo, hi)
        g = ctx.state().cpu().numpy()
        near = np.abs(np.log2(H.initial_dt(a, j, eta)) % 1.0)
        off = np.flatnonzero(g[14] != dt)
        assert all(min(near[i], 1.0 - near[i]) < 1e-4 for i in off) and len(off) <= 4
        sizes = []
        for step in range(24):
            _load(ctx, m, x, v, a, j, t, dt)
            t1, ni = ctx.step(eps2, eta, lo, hi)
            got = ctx.state()
            rt1, idx = H.next_block(t, dt)
            assert t1 == rt1 and ni == len(idx)
            xp, vp = oracle.predict(t1, x, v, a, j, t)
            a1, j1, _ = oracle.force(m, xp, vp, idx, eps2)
            want = H.corrector_step(x, v, a, j, t, dt, idx, t1, a1, j1, eta, lo, hi)
            # forces carry the pair kernel's 1e-5 / 1e-4 tolerance; x, v feel them times h^2/12, h/2
            g = got.cpu().numpy()
            check_parity([g[7:10][:, idx], g[10:13][:, idx], np.ones(len(idx))], (a1, j1, np.ones(len(idx))))
            assert np.array_equal(g[13], t)
            assert np.abs(g[1:4] - x).max() < 1e-8 and np.abs(g[4:7] - v).max() < 1e-6
            bad = np.flatnonzero(g[14] != dt)
            for i in bad:
                k = int(np.flatnonzero(idx == i)[0])
                r = want[k] / dt[i]
                # a2, a3 are differences of forces: the pair kernel's 1e-6 moves `want` by up to
                # a few percent, so only particles near a decision threshold may decide differently
                assert min(abs(r - 1.0), abs(r - 2.0), abs(r - 0.5)) < 0.1
            assert len(bad) <= max(2, ni // 10)
            sizes.append(ni)
        assert min(sizes) < n // 4                                # genuinely individual steps


def test_free_running_device_integration_conserves_energy(nbmod):
    """nb_step alone drives a Plummer sphere for 1/16 time unit; energy is conserved to the level
    a 4th-order Hermite scheme with eta = 0.01 gives (oracle run: < 1e-6)."""
    n, eps2, eta = 1024, 1e-4, 0.01
    lo, hi = 2.0 ** -20, 2.0 ** -5
    m, x, v = nbgen.plummer(n, 808)
    il = np.arange(n, dtype=np.int32)
    _, _, p0 = oracle.force(m, x, v, il, eps2)
    e0 = 0.5 * (m * (v * v).sum(0)).sum() + 0.5 * (m * p0).sum()
    with nbmod.Context(n) as ctx:
        ctx.set_j(m, x, v)
        ctx.predict(0.0)
        ga, gj, gp = ctx.force(il, eps2)
        ctx.init_steps(il, ga, gj, eta, lo, hi)
        steps = 0
        while True:
            t1, ni, _ = ctx.next_block()
            if t1 > 0.0625:
                break
            ctx.step(eps2, eta, lo, hi)
            steps += 1
            assert steps < 100000
        ctx.predict(0.0625)
        xp, vp = (q.cpu().numpy() for q in ctx.predicted())
        ctx.sync()
    _, _, p1 = oracle.force(m, xp, vp, il, eps2)
    e1 = 0.5 * (m * (vp * vp).sum(0)).sum() + 0.5 * (m * p1).sum()
    print("device block-step run: %d steps, dE/E = %.2e" % (steps, (e1 - e0) / abs(e0)))
    assert steps > 16 and abs(e1 - e0) < 2e-6 * abs(e0)
