"""-m gpu: the CUDA path (through the C-ABI binding) against the fp64 oracle, element by element on
the same seeded inputs.  Tolerances are BASELINE.json's: max per-particle relative error 1e-5
(acc, pot), 1e-4 (jerk), metric R10 (tests/util.py).  Small cases span several j-tiles (TJ = 128),
i-tiles (256) and ragged tails; the full-size configs are checked on sampled i."""
import numpy as np
import pytest

import nbgen
import oracle
from util import TOL_ACC, TOL_JRK, TOL_POT, check_parity, rel_err_scalar, rel_err_vec

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _np(ts):
    return [q.cpu().numpy() for q in ts]


def _gpu_force(nbm, case, t, i_list, eps2=None, splits=0, mode=0):
    with nbm.Context(case.n, max(1, len(i_list))) as ctx:
        ctx.load_case(case)
        ctx.predict(t)
        ctx.tuning(splits, mode)
        out = _np(ctx.force(i_list, case.eps2 if eps2 is None else eps2))
        info = ctx.last_launch()
        ctx.sync()
    return out, info


def _oracle_force(case, t, i_list, eps2=None):
    xp, vp = oracle.predict(t, case.x, case.v, case.a, case.j, case.t)
    fl = case.flags if case.flags.any() else None
    return oracle.force(case.m, xp, vp, i_list, case.eps2 if eps2 is None else eps2, fl)


def _random_case(n, seed, eps2=1e-4, with_state=True):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    c = nbgen.configs._rest("rand", m, x, v, eps2)
    if with_state:
        c.a, c.j = nbgen.mean_field(x, v)
        c.t = 0.25 * nbgen.Streams(seed + 2, n).uniform()
    return c


# ------------------------------------------------------------------ a1 predictor
@pytest.mark.parametrize("n", [1, 2, 127, 129, 1000, 4099])
def test_predictor_matches_oracle(nbmod, n):
    c = _random_case(n, 50 + n)
    t = 0.3
    with nbmod.Context(n) as ctx:
        ctx.load_case(c)
        ctx.predict(t)
        xp, vp = _np(ctx.predicted())
        ctx.sync()
    rx, rv = oracle.predict(t, c.x, c.v, c.a, c.j, c.t)
    # FMA/Horner vs the oracle's plain polynomial: a few ulp of the largest term (R1)
    assert (np.abs(xp - rx) <= 4e-16 * np.maximum(1.0, np.abs(rx))).all()
    assert (np.abs(vp - rv) <= 4e-16 * np.maximum(1.0, np.abs(rv))).all()


def test_predictor_exact_values(nbmod):
    one = np.ones((3, 1))
    with nbmod.Context(4) as ctx:
        ctx.set_j(np.ones(1), 1 * one, 2 * one, 3 * one, 6 * one, np.zeros(1))
        ctx.predict(0.5)
        xp, vp = _np(ctx.predicted())
        assert (xp == 2.5).all() and (vp == 4.25).all()          # P9
        ctx.predict(0.0)
        xp, vp = _np(ctx.predicted())
        assert (xp == 1.0).all() and (vp == 2.0).all()           # dt = 0 is the identity


# ------------------------------------------------------------------ config 1 and small pins
def test_config1_all_active(nbmod):
    c = nbgen.config1()
    for il in c.i_lists:
        got, info = _gpu_force(nbmod, c, 0.0, il)
        ref = _oracle_force(c, 0.0, il)
        print("cfg1", check_parity(got, ref), info)
    # P2 on the GPU result: momentum; P3: W agrees with the oracle's
    got, _ = _gpu_force(nbmod, c, 0.0, c.i_lists[0])
    ref = _oracle_force(c, 0.0, c.i_lists[0])
    assert abs((c.m * got[0]).sum(1)).max() < 1e-7
    assert abs((c.m * got[1]).sum(1)).max() < 1e-6
    assert 0.5 * (c.m * got[2]).sum() == pytest.approx(0.5 * (c.m * ref[2]).sum(), rel=1e-7)


@pytest.mark.parametrize("eps2", [11.0, 0.0])
def test_p1_two_body_on_gpu(nbmod, eps2):
    m = np.array([3.0, 2.0])
    x = np.array([[0.0, 3.0], [0.0, 4.0], [0.0, 0.0]])
    v = np.array([[0.0, 1.0], [0.0, -2.0], [0.0, 0.5]])
    c = nbgen.configs._rest("two", m, x, v, eps2)
    got, _ = _gpu_force(nbmod, c, 0.0, [0, 1])
    ref = _oracle_force(c, 0.0, [0, 1])
    check_parity(got, ref, scale=0.1)          # <= 1e-6 relative


def test_p8_ring_unsoftened(nbmod):
    k, rad, om = 7, 2.0, 0.3
    ang = 2 * np.pi * np.arange(k) / k
    x = np.stack([rad * np.cos(ang), rad * np.sin(ang), np.zeros(k)])
    v = om * np.stack([-x[1], x[0], np.zeros(k)])
    c = nbgen.configs._rest("ring", np.full(k, 1.0 / k), x, v, 0.0)
    got, _ = _gpu_force(nbmod, c, 0.0, np.arange(k))
    check_parity(got, _oracle_force(c, 0.0, np.arange(k)), scale=0.1)
    assert got[0][0, 0] == pytest.approx(-0.0823130311058, rel=1e-6)
    assert got[2][0] == pytest.approx(-0.3292521244232, rel=1e-6)
    assert got[1][1, 0] == pytest.approx(-0.0246939093317, rel=1e-6)


@pytest.mark.parametrize("n", [1, 2, 33, 257, 1025])
def test_p12_sizes_and_tails(nbmod, n):
    c = _random_case(n, 70 + n)
    il = np.arange(n, dtype=np.int32)
    got, _ = _gpu_force(nbmod, c, 0.1, il)
    ref = _oracle_force(c, 0.1, il)
    if n == 1:
        assert all((g == 0).all() for g in got)
    else:
        check_parity(got, ref)


def test_degenerate_inputs(nbmod):
    c = _random_case(300, 5)
    with nbmod.Context(300, 300) as ctx:
        ctx.load_case(c)
        ctx.predict(0.0)
        a, j, p = ctx.force(np.zeros(0, np.int32), 1e-4)            # N_i = 0: no-op
        assert a.shape == (3, 0) and p.shape == (0,)
        ctx.sync()
    # everything else massless: exact zeros; coincident particles: finite (R5/R6)
    c.m[:] = 0.0
    c.m[7] = 1.0
    got, _ = _gpu_force(nbmod, c, 0.0, [7])
    assert all((g == 0).all() for g in got)
    c = _random_case(300, 6)
    c.x[:, 1] = c.x[:, 0]
    for eps2 in (0.0, 1e-4):
        got, _ = _gpu_force(nbmod, c, 0.0, [0, 1, 2], eps2=eps2)
        ref = _oracle_force(c, 0.0, [0, 1, 2], eps2=eps2)
        assert all(np.isfinite(g).all() for g in got)
        check_parity(got, ref)


# ------------------------------------------------------------------ a4: j-split, reduce, atomics
def test_j_split_variants_agree(nbmod):
    c = _random_case(5000, 90, eps2=2.0 ** -16)
    il = nbgen.permutation(91, c.n)[:777]
    ref = _oracle_force(c, 0.2, il)
    outs = []
    for splits, mode in [(1, 0), (3, 0), (7, 0), (40, 0), (0, 0), (5, 1), (0, 1)]:
        got, info = _gpu_force(nbmod, c, 0.2, il, splits=splits, mode=mode)
        check_parity(got, ref)
        assert splits == 0 or info["j_splits"] == splits
        outs.append(got)
    for g in outs[1:]:                                   # variants differ by rounding only
        assert rel_err_vec(g[0], outs[0][0]).max() < 2 * TOL_ACC
        assert rel_err_vec(g[1], outs[0][1]).max() < 2 * TOL_JRK
    again, _ = _gpu_force(nbmod, c, 0.2, il, splits=7, mode=0)
    assert all((p == q).all() for p, q in zip(again, outs[2]))    # deterministic (R9)


@pytest.mark.parametrize("ni", [1, 3, 8, 9, 16, 17, 32, 33, 64, 65, 128, 129, 200])
def test_few_active_i_share_threads(nbmod, ni):
    """few i active -> 32, 16, .. 2 threads per i split the j-quads of a tile (the 256
    slots of a CTA hold the next power of two >= N_i particles), shuffle butterfly; up to 16 i the
    pair kernel's last CTA also reduces (one launch).  Includes a flagged i, its own tile, and the
    self pair of every i."""
    c = _random_case(6000, 94, eps2=2.0 ** -14)
    c.flags[[11, 4000]] = 1
    il = nbgen.permutation(95, c.n)[:ni].astype(np.int32)
    il[0] = 11
    ref = _oracle_force(c, 0.3, il)
    for splits, mode in [(0, 0), (1, 0), (5, 0), (0, 1)]:
        got, info = _gpu_force(nbmod, c, 0.3, il, splits=splits, mode=mode)
        check_parity(got, ref)
    got0, _ = _gpu_force(nbmod, c, 0.3, il, eps2=0.0)
    check_parity(got0, _oracle_force(c, 0.3, il, eps2=0.0))


def test_whole_wave_segment_plus_remainder(nbmod):
    """Four waves of i-tiles and more: the dispatcher runs whole waves with one j-subset and the
    remainder with a split j (two pair-kernel launches, one reduction); below four waves the whole call
    is split.  Duplicates keep N small."""
    c = _random_case(3000, 92, eps2=2.0 ** -18)
    c.flags[[7, 2999]] = 1
    ni = 4 * 148 * 4 * 256 + 1234                                 # > 4 x 592 full i-tiles + a ragged one
    il = (nbgen.permutation(93, ni) % c.n).astype(np.int32)
    got, info = _gpu_force(nbmod, c, 0.1, il)
    # whether 3 or 4 CTAs are resident per SM, a whole-wave segment and a split remainder exist
    assert info["kernels"] >= 3 and info["ctas"] > (ni + 255) // 256
    ref_all = _oracle_force(c, 0.1, np.arange(c.n, dtype=np.int32))
    ref = [ref_all[0][:, il], ref_all[1][:, il], ref_all[2][il]]
    check_parity(got, ref)
    atom, _ = _gpu_force(nbmod, c, 0.1, il, mode=1)
    check_parity(atom, ref)


def test_i_subsets_duplicates_and_order(nbmod):
    c = _random_case(2048, 95)
    full, _ = _gpu_force(nbmod, c, 0.0, np.arange(c.n))
    il = np.array([5, 2047, 5, 0, 1000, 129, 128, 127, 2047], np.int32)
    got, _ = _gpu_force(nbmod, c, 0.0, il)
    check_parity(got, _oracle_force(c, 0.0, il))
    assert rel_err_vec(got[0], full[0][:, il]).max() < 2 * TOL_ACC   # i's independent
    assert rel_err_vec(got[1], full[1][:, il]).max() < 2 * TOL_JRK
    assert rel_err_scalar(got[2], full[2][il]).max() < 2 * TOL_POT
    assert (got[2][0] == got[2][2]) and (got[0][:, 1] == got[0][:, 8]).all()


def test_translation_stress(nbmod):
    """the distance is where single precision fails; shift everything by 1e3."""
    c = _random_case(3000, 97, eps2=2.0 ** -20)
    c.x += np.array([[1e3], [-2e3], [5e2]])
    il = np.arange(c.n)
    got, _ = _gpu_force(nbmod, c, 0.0, il)
    check_parity(got, _oracle_force(c, 0.0, il))


# ------------------------------------------------------------------ R7 flags, a0 updates
def test_flagged_pairs_unsoftened(nbmod):
    c = _random_case(700, 101, eps2=1e-2)
    c.flags[[3, 130, 699]] = 1
    c.x[:, 130] = c.x[:, 3] + np.array([1e-3, 2e-3, -1e-3])       # a tight flagged pair
    il = np.arange(c.n)
    got, _ = _gpu_force(nbmod, c, 0.05, il)
    ref = _oracle_force(c, 0.05, il)
    check_parity(got, ref)
    soft = oracle.force(c.m, *oracle.predict(0.05, c.x, c.v, c.a, c.j, c.t), il, c.eps2)
    assert rel_err_vec(ref[0][:, [3]], soft[0][:, [3]]).max() > 0.5   # the flags matter here
    # clearing the flags gives the plain softened answer again
    with nbmod.Context(c.n) as ctx:
        ctx.load_case(c)
        ctx.set_flags(np.array([3, 130, 699], np.int32), np.zeros(3, np.uint8))
        ctx.predict(0.05)
        check_parity(_np(ctx.force(il, c.eps2)), soft)
        ctx.sync()


def test_update_j_scatter(nbmod):
    c = _random_case(1500, 103)
    c2 = _random_case(1500, 104)
    idx = nbgen.permutation(7, c.n)[:400]
    with nbmod.Context(c.n) as ctx:
        ctx.load_case(c)
        ctx.update_j(idx, c2.m[idx], c2.x[:, idx], c2.v[:, idx], c2.a[:, idx], c2.j[:, idx], c2.t[idx])
        ctx.predict(0.3)
        got = _np(ctx.force(np.arange(c.n), c.eps2))
        xp, vp = _np(ctx.predicted())
        ctx.sync()
    for f in ("m", "x", "v", "a", "j", "t"):
        getattr(c, f)[..., idx] = getattr(c2, f)[..., idx]
    rx, rv = oracle.predict(0.3, c.x, c.v, c.a, c.j, c.t)
    assert np.abs(xp - rx).max() < 1e-14 and np.abs(vp - rv).max() < 1e-14
    check_parity(got, _oracle_force(c, 0.3, np.arange(c.n)))


# ------------------------------------------------------------------ boundary behaviour
def test_errors_and_host_variants(nbmod):
    nb = nbmod.binding
    c = _random_case(600, 110)
    with pytest.raises(nb.NBError) as e:
        nb.nb_create(0, 1, 0, None)
    assert e.value.status == nb.NB_ERR_ARG
    h = nb.nb_create(c.n, c.n, 0, torch.cuda.current_stream().cuda_stream)
    try:
        acc, jrk, pot = np.empty((3, 4)), np.empty((3, 4)), np.empty(4)
        il = np.array([0, 5, 599, 7], np.int32)
        with pytest.raises(nb.NBError) as e:                       # force before predict
            nb.nb_force_host(h, il, 4, 1e-4, acc, jrk, pot)
        assert e.value.status == nb.NB_ERR_STATE
        nb.nb_set_j_host(h, 0, c.n, c.m, c.x, c.v, c.a, c.j, c.t)
        assert nb.nb_count(h) == c.n
        nb.nb_predict(h, 0.1)
        with pytest.raises(nb.NBError) as e:
            nb.nb_force_host(h, il, 4, -1.0, acc, jrk, pot)
        assert e.value.status == nb.NB_ERR_ARG
        with pytest.raises(nb.NBError) as e:
            nb.nb_force_host(h, il, c.n + 1, 1e-4, acc, jrk, pot)
        assert e.value.status == nb.NB_ERR_ARG
        nb.nb_force_host(h, il, 4, c.eps2, acc, jrk, pot)
        check_parity((acc, jrk, pot), _oracle_force(c, 0.1, il))
        bad = np.array([0, 600, -1, 7], np.int32)                  # out-of-range entries
        with pytest.raises(nb.NBError) as e:
            nb.nb_force_host(h, bad, 4, c.eps2, acc, jrk, pot)
        assert e.value.status == nb.NB_ERR_INDEX
        assert np.isnan(pot[1]) and np.isnan(pot[2]) and np.isnan(acc[:, 1]).all()
        check_parity((acc[:, [0, 3]], jrk[:, [0, 3]], pot[[0, 3]]), _oracle_force(c, 0.1, [0, 7]))
        nb.nb_sync(h)                                              # latch was cleared
        nb.nb_clear(h)
        assert nb.nb_count(h) == 0
    finally:
        nb.nb_destroy(h)


def test_lent_workspace(nbmod):
    nb = nbmod.binding
    c = _random_case(900, 111)
    nbytes = nb.nb_workspace_bytes(c.n, c.n)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    ctx = nbmod.Context(c.n)
    nb.nb_set_workspace(ctx.h, ws.data_ptr() + off, nbytes)
    ctx.load_case(c)
    ctx.predict(0.0)
    got = _np(ctx.force(np.arange(c.n), c.eps2))
    ctx.sync()
    with pytest.raises(nb.NBError):
        nb.nb_set_workspace(ctx.h, ws.data_ptr() + off, nbytes)     # too late
    ctx.close()
    check_parity(got, _oracle_force(c, 0.0, np.arange(c.n)))


def test_bitwise_repeatability_of_every_kernel_path(nbmod):
    """compute-sanitizer is closed on this GPU pool (profiles/r2_sanitizer.md), so races in the tile
    ring (release counter, refill by the last warp out, mbarrier phases), in the ticket reduction and
    in the persistent kernel's slots are hunted the other way round: every path is deterministic by
    construction (R9), so 12 back-to-back repeats under different timing (a second stream keeps the
    chip busy for half of them) must give bit-identical results -- and the first of them matches the
    oracle."""
    c = _random_case(20000, 130, eps2=2.0 ** -16)
    c.flags[[17, 9000]] = 1
    perm = nbgen.permutation(131, c.n)
    side = torch.cuda.Stream()
    noise = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    for ni in (3, 8, 12, 100, 300, 20000):             # direct, few-i (in-kernel and separate reduce), all-i
        il = perm[:ni].astype(np.int32)
        il[0] = 17
        ref = _oracle_force(c, 0.1, il)
        with nbmod.Context(c.n, ni) as ctx:
            ctx.load_case(c)
            ctx.predict(0.1)
            first = None
            for rep in range(12):
                if rep % 2:
                    with torch.cuda.stream(side):
                        noise.fill_(rep)
                got = _np(ctx.force(il, c.eps2))
                if first is None:
                    first = got
                    check_parity(got, ref)
                else:
                    assert all(np.array_equal(p, q) for p, q in zip(first, got)), (ni, rep)
            ctx.sync()
        side.synchronize()


def test_sixteen_million_particles(nbmod):
    """Largest size exercised: N = 2^24 + 5 (1.9 GB of j-store, 131073 tiles with a ragged last one),
    four times config 5.  Active subsets of 3, 40 and 600 particles (the first and the last particle
    among them) against ALL j: the handful falls back from the direct kernel to the tile kernel here
    (its per-thread fp32 sums would exceed R17's 64 terms), the others take the threads-per-i and the
    all-i mapping.  Oracle: every checked particle against all 16.8 M."""
    n, eps2 = (1 << 24) + 5, 1e-6
    m, x, v = nbgen.plummer(n, 4242)
    a, j = nbgen.mean_field(x, v)
    tj = 0.01 * nbgen.Streams(4243, n).uniform()
    t = 0.01
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    with nbmod.Context(n, 1024) as ctx:
        ctx.set_j(m, x, v, a, j, tj)
        ctx.predict(t)
        for ni in (3, 40, 600):
            il = nbgen.permutation(7 + ni, n)[:ni].astype(np.int32)
            il[0], il[1] = n - 1, 0
            got = [q.cpu().numpy() for q in ctx.force(il, eps2)]
            ctx.sync()
            print("N=2^24+5 ni=%d" % ni, check_parity(got, oracle.force(m, xp, vp, il, eps2)), ctx.last_launch())
        px, _ = ctx.predicted(n - 4099, 4099)
        assert rel_err_vec(px.cpu().numpy(), xp[:, n - 4099:]).max() <= 1e-14
