"""-m gpu: mid-size calls whose last i-tile is at most half full (N_i = 256 q + rem, 1 <= rem <= 128): the
dispatcher hands that tile to the few-i kernel as a segment of its own (nb_api.cu force_impl, DESIGN.md
7.3) when the j-set is large enough for a 256-slot pass to cost more than a launch.  Two pair-kernel
launches of DIFFERENT variants (thread per i; 2 .. 32 threads per i) write two partial buffers that one
reduction reads.  Checked element by element against the oracle: by index (own pair, flagged pairs, a bad
index in either segment), by value with ids, acc + pot only, eps2 = 0; and that calls just outside the
rule (rem = 0, rem > 128, more than 16384 particles, small N) keep one segment."""
import numpy as np
import pytest

import nbgen
import oracle
from util import check_parity, rel_err_scalar, rel_err_vec

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

N = 160000 + 77           # large enough for every rem <= 128 to take the tail (the rule needs N >= ~150000)


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


@pytest.fixture(scope="module")
def world(nbmod):
    m, x, v = nbgen.plummer(N, 7300)
    m = m * (0.5 + nbgen.Streams(7301, N).uniform())
    a, j = nbgen.mean_field(x, v)
    tj = 0.25 * nbgen.Streams(7302, N).uniform()
    t = 0.2
    flags = np.zeros(N, np.uint8)
    flags[[40, 1100, 90000, N - 3]] = 1
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    ctx = nbmod.Context(N, 16500)
    ctx.set_j(m, x, v, a, j, tj)
    fl = np.flatnonzero(flags).astype(np.int32)
    ctx.set_flags(fl, np.ones(len(fl), np.uint8))
    ctx.predict(t)
    yield ctx, m, xp, vp, flags
    ctx.close()


def _i_list(ni, seed):
    il = nbgen.permutation(seed, N)[:ni].astype(np.int32)
    il[0], il[ni // 2], il[ni - 1], il[ni - 2] = 40, 1100, 90000, N - 3     # flagged ones in both segments
    return il


@pytest.mark.parametrize("ni,eps2", [(256 + 1, 2.0 ** -14), (256 + 8, 0.0), (256 + 40, 2.0 ** -14), (512 + 64, 1e-12),
                                     (768 + 100, 2.0 ** -14), (1024 + 128, 2.0 ** -14), (2048 + 17, 0.0),
                                     # above 4096 particles the reduction is one thread per i, but one warp per i
                                     # of the tail (its hundreds of j-subsets)
                                     (4096 + 20, 2.0 ** -14), (8192 + 60, 0.0)])
def test_tail_segment_by_index(nbmod, world, ni, eps2):
    ctx, m, xp, vp, flags = world
    il = _i_list(ni, 7310 + ni)
    got = [q.cpu().numpy() for q in ctx.force(il, eps2)]
    info = ctx.last_launch()
    ctx.sync()
    assert info["kernels"] == 3                      # full tiles + tail + one reduction
    check_parity(got, oracle.force(m, xp, vp, il, eps2, flags))
    again = [q.cpu().numpy() for q in ctx.force(il, eps2)]
    assert all(np.array_equal(p, q) for p, q in zip(got, again))     # deterministic (R9)


def test_tail_segment_by_value_and_kick(nbmod, world):
    ctx, m, xp, vp, flags = world
    ni, eps2 = 512 + 30, 2.0 ** -14
    il = _i_list(ni, 7400)
    ref = oracle.force(m, xp, vp, il, eps2, flags)
    got = [q.cpu().numpy() for q in ctx.force_ext_ids(xp[:, il], vp[:, il], il, flags[il], eps2)]
    assert ctx.last_launch()["kernels"] == 3
    check_parity(got, ref)
    # particles from outside the j-set; with jerk, and acc + pot only (the kick)
    _, xo, vo = nbgen.plummer(ni, 7401)
    xo, vo = np.ascontiguousarray(xo + 0.3), np.ascontiguousarray(vo)
    ref = oracle.force(np.concatenate([m, np.zeros(ni)]), np.concatenate([xp, xo], 1), np.concatenate([vp, vo], 1),
                       np.arange(N, N + ni, dtype=np.int32), eps2)
    got = [q.cpu().numpy() for q in ctx.force_ext(xo, vo, eps2)]
    assert ctx.last_launch()["kernels"] == 3
    check_parity(got, ref)
    acc, none, pot = ctx.force_ext(xo, None, eps2)
    assert none is None and ctx.last_launch()["kernels"] == 3
    assert rel_err_vec(acc.cpu().numpy(), ref[0]).max() <= 1e-5
    assert rel_err_scalar(pot.cpu().numpy(), ref[2]).max() <= 1e-5
    ctx.sync()


def test_tail_segment_bad_index_in_either_segment(nbmod, world):
    ctx, m, xp, vp, flags = world
    nb = nbmod.binding
    ni, eps2 = 256 + 20, 2.0 ** -14
    il = _i_list(ni, 7500)
    il[100], il[256 + 5] = -7, N                       # one in the full tile, one in the tail
    got = [q.cpu().numpy() for q in ctx.force(il, eps2)]
    with pytest.raises(nb.NBError) as e:
        ctx.sync()
    assert e.value.status == nb.NB_ERR_INDEX
    bad = np.zeros(ni, bool)
    bad[[100, 256 + 5]] = True
    assert np.isnan(got[0][:, bad]).all() and np.isnan(got[2][bad]).all()
    ok = ~bad
    ref = oracle.force(m, xp, vp, il[ok], eps2, flags)
    check_parity([got[0][:, ok], got[1][:, ok], got[2][ok]], ref)


def test_calls_outside_the_rule_keep_one_segment(nbmod, world):
    ctx, m, xp, vp, flags = world
    for ni in (256, 512, 256 + 129, 1024 + 255, 130, 4096 + 129, 16384 + 20):
        ctx.force(_i_list(ni, 7600 + ni), 1e-6)
        assert ctx.last_launch()["kernels"] == 2, ni
    ctx.tuning(3, 0)                                   # forced j-split: one segment
    ctx.force(_i_list(300, 7601), 1e-6)
    assert ctx.last_launch()["kernels"] == 2
    ctx.tuning(0, 0)
    ctx.sync()
    # a small j-set: a launch costs more than the 256-slot pass
    n = 5000
    m2, x2, v2 = nbgen.plummer(n, 7602)
    z = np.zeros((3, n))
    with nbmod.Context(n, 512) as small:
        small.set_j(m2, x2, v2, z, z, np.zeros(n))
        small.predict(0.0)
        il = nbgen.permutation(7603, n)[:300].astype(np.int32)
        got = [q.cpu().numpy() for q in small.force(il, 1e-4)]
        assert small.last_launch()["kernels"] == 2
        small.sync()
    check_parity(got, oracle.force(m2, x2, v2, il, 1e-4))


@pytest.mark.parametrize("queue", [2, 1, 0])
def test_tail_segment_in_a_block_step(nbmod, queue):
    """nb_steps: a block of 256 q + rem particles that the persistent kernel hands over is planned on the
    device (steps.cu plan_block: queue modes 2 and 1) or goes through nb_step (mode 0); both cut the tail
    off.  The steps are set by hand so that the first block is exactly the chosen particles; forces of the
    block and the corrected state are checked against the oracle's step."""
    from oracle import hermite as H
    eps2, eta, lo, hi = 2.0 ** -14, 0.02, 2.0 ** -20, 2.0 ** -4
    m, x, v = nbgen.plummer(N, 7700)
    a, j = nbgen.mean_field(x, v)
    view = nbmod.context._DeviceView
    with nbmod.Context(N, 8192) as ctx:
        ctx.steps_queue(queue)
        for ni in (256 + 40, 1024 + 100, 4096 + 20):
            idx = np.sort(nbgen.permutation(7701 + ni, N)[:ni]).astype(np.int32)
            t = np.zeros(N)
            dt = np.full(N, 2.0 ** -6)
            dt[idx] = 2.0 ** -10
            ctx.set_j(m, x, v, a, j, t)
            ctx.set_dt(dt)
            done, gt, gni = ctx.steps(1, eps2, eta, lo, hi)[:3]
            assert done == 1 and gt[0] == 2.0 ** -10 and gni[0] == ni
            xs, vs, as_, js, ts, dts = x.copy(), v.copy(), a.copy(), j.copy(), t.copy(), dt.copy()
            t1, due = H.next_block(ts, dts)
            assert np.array_equal(due, idx)
            xp, vp = oracle.predict(t1, xs, vs, as_, js, ts)
            a1, j1, p1 = oracle.force(m, xp, vp, idx, eps2)
            pa, pj, pp = nbmod.binding.nb_block_forces(ctx.h)
            ga = torch.as_tensor(view(pa, 3 * ni, "<f8"), device=ctx.device).cpu().numpy().reshape(3, ni)
            gj = torch.as_tensor(view(pj, 3 * ni, "<f8"), device=ctx.device).cpu().numpy().reshape(3, ni)
            gp = torch.as_tensor(view(pp, ni, "<f8"), device=ctx.device).cpu().numpy()
            check_parity([ga, gj, gp], [a1, j1, p1])
            H.corrector_step(xs, vs, as_, js, ts, dts, idx, t1, a1, j1, eta, lo, hi)
            g = ctx.state().cpu().numpy()
            assert np.abs(g[1:4] - xs).max() < 1e-9 and np.abs(g[4:7] - vs).max() < 1e-7
            assert np.array_equal(g[13], ts) and (g[14] != dts).sum() <= max(2, ni // 100)
        ctx.sync()


def test_random_midsize_shapes(nbmod):
    """Seeded random (N, N_i) around the rule's edges -- rem = 1, 128, 129, 255, 0; N on both sides of the
    threshold; by index and by value; eps2 = 0 now and then -- each against the oracle."""
    rng = np.random.RandomState(7800)
    rems = [1, 2, 7, 8, 9, 16, 17, 31, 32, 33, 63, 64, 65, 127, 128, 129, 200, 255, 0]
    for case in range(19):
        n = int(rng.choice([60000, 70001, 90000, 149000, 152000, 200003, 300000]))
        q = int(rng.choice([1, 1, 2, 3, 5, 8, 15, 16, 17, 33]))
        ni = 256 * q + rems[case]
        eps2 = float(rng.choice([0.0, 2.0 ** -14, 1e-12]))
        m, x, v = nbgen.plummer(n, 7801 + case)
        zero = np.zeros((3, n))
        flags = np.zeros(n, np.uint8)
        il = nbgen.permutation(7900 + case, n)[:ni].astype(np.int32)
        if case % 3 == 0:
            flags[il[[0, ni - 1]]] = 1
            flags[il[ni // 2]] = 1
        with nbmod.Context(n, ni) as ctx:
            ctx.set_j(m, x, v, zero, zero, np.zeros(n))
            fl = np.flatnonzero(flags).astype(np.int32)
            if len(fl):
                ctx.set_flags(fl, np.ones(len(fl), np.uint8))
            ctx.predict(0.0)
            if case % 2 == 0:
                got = [g.cpu().numpy() for g in ctx.force(il, eps2)]
            else:
                got = [g.cpu().numpy() for g in ctx.force_ext_ids(x[:, il], v[:, il], il, flags[il], eps2)]
            kernels = ctx.last_launch()["kernels"]
            ctx.sync()
        rem = ni % 256
        if rem == 0 or rem > 128 or ni > 16384:
            assert kernels == 2, (case, n, ni)
        check_parity(got, oracle.force(m, x, v, il, eps2, flags if flags.any() else None))


def test_tail_segment_under_the_peer_exchange(nbmod, world):
    """nb_xforce (world of one: the whole window / flag / sum path) on a call with a tail segment returns
    nb_force_ext_ids' forces bit for bit: the exchange kernels run after the one reduction of both segments."""
    ctx, m, xp, vp, flags = world
    ctx.xchg_create(0, 1, 2048)
    try:
        for ni in (256 + 40, 1024 + 7):
            il = _i_list(ni, 8000 + ni)
            args = (xp[:, il], vp[:, il], il, flags[il], 2.0 ** -14)
            want = [q.cpu().numpy() for q in ctx.force_ext_ids(*args)]
            assert ctx.last_launch()["kernels"] == 3
            got = [q.cpu().numpy() for q in ctx.xforce(*args)]
            assert ctx.last_launch()["kernels"] == 5           # + push + sum
            ctx.sync()
            assert all(np.array_equal(g, w) for g, w in zip(got, want))
    finally:
        ctx.xchg_destroy()


def test_predict_and_force_captured_into_a_cuda_graph(nbmod):
    """nb_predict + nb_force recorded into a CUDA graph on the context's stream and replayed: the chains of
    dependent launches (csrc/pdl.h), the one-launch kernels, the few-i kernel and a call with a tail segment
    all give the bits of the eager call."""
    n = 150000
    m, x, v = nbgen.plummer(n, 8100)
    zero = np.zeros((3, n))
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        with nbmod.Context(n, 4096, stream=s.cuda_stream) as ctx:
            ctx.set_j(m, x, v, zero, zero, np.zeros(n))
            ctx.predict(0.0)
            for ni in (1, 12, 100, 300, 1024):
                il = torch.as_tensor(nbgen.permutation(8101, n)[:ni].astype(np.int32)).to(ctx.device)
                eager = [q.clone() for q in ctx.force(il, 1e-6)]
                s.synchronize()
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=s):
                    ctx.predict(0.0)
                    out = ctx.force(il, 1e-6)
                for _ in range(3):
                    graph.replay()
                torch.cuda.synchronize()
                assert all(torch.equal(a, b) for a, b in zip(eager, out)), ni
            ctx.sync()
