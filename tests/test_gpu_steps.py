"""-m gpu: nb_steps -- many block steps inside one persistent kernel -- against the fp64 oracle
(oracle/hermite.py R12, R18..R21 around oracle.predict / oracle.force).

The oracle drives its own trajectory from the same start; the GPU is given the oracle's stored state
before every nb_steps call and then runs k = 1, 7 or 64 steps on its own.  Blocks the persistent
kernel takes itself are computed in IEEE double (forces agree with the oracle to ~1e-13), so block
times, block sizes and the power-of-two step decisions must come out IDENTICAL and the state equal
to rounding; blocks handed to the host path (nb_step's packed fp32 kernel) carry that kernel's 1e-5 /
1e-4 tolerance, as in tests/test_gpu_hermite.py.  PAPER.md:41, :49, :83, :129."""
import numpy as np
import pytest

import nbgen
import oracle
from oracle import hermite as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _load(ctx, m, x, v, a, j, t, dt):
    ctx.set_j(m, x, v, a, j, t)
    ctx.set_dt(dt)


def _start(n, seed, eps2, eta, lo, hi, flags=None):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    il = np.arange(n, dtype=np.int32)
    a, j, _ = oracle.force(m, x, v, il, eps2, flags)
    t = np.zeros(n)
    dt = H.quantise_dt(H.initial_dt(a, j, eta), lo, hi)
    return m, x, v, a, j, t, dt


def _oracle_steps(k, m, x, v, a, j, t, dt, eps2, eta, lo, hi, flags=None):
    """k block steps of the oracle, in place; returns the (t1, ni) log and the last block's forces."""
    log_t, log_ni, last = [], [], None
    for _ in range(k):
        t1, idx = H.next_block(t, dt)
        xp, vp = oracle.predict(t1, x, v, a, j, t)
        a1, j1, p1 = oracle.force(m, xp, vp, idx, eps2, flags)
        H.corrector_step(x, v, a, j, t, dt, idx, t1, a1, j1, eta, lo, hi)
        log_t.append(t1)
        log_ni.append(len(idx))
        last = (idx, a1, j1, p1)
    return np.array(log_t), np.array(log_ni), last


@pytest.mark.parametrize("n", [1, 2, 200, 512])
def test_steps_all_in_kernel_match_oracle(nbmod, n):
    """Every block fits the persistent kernel (bound lifted, n <= 512).  The 80 steps pass t = 2^-6,
    where every particle is due at once (a block of n: one thread per due particle at n = 512)."""
    eps2, eta, lo, hi = 2.0 ** -10, 0.02, 2.0 ** -12, 2.0 ** -6
    m, x, v, a, j, t, dt = _start(n, 900 + n, eps2, eta, lo, hi)
    if n == 1:
        a[:] = 0.0
        j[:] = 0.0
        dt[:] = hi
    with nbmod.Context(n) as ctx:
        ctx.steps_bound(1 << 40)
        total = 0
        for k in (1, 7, 64, 7, 1):
            _load(ctx, m, x, v, a, j, t, dt)
            done, gt, gni = ctx.steps(k, eps2, eta, lo, hi)
            rt, rni, last = _oracle_steps(k, m, x, v, a, j, t, dt, eps2, eta, lo, hi)
            assert done == k
            assert np.array_equal(gt, rt), (gt, rt)
            assert np.array_equal(gni, rni), (gni, rni)
            g = ctx.state().cpu().numpy()
            small = rni.max() <= 512
            tol = 1e-11 if small else 1e-7
            assert np.array_equal(g[13], t)
            assert np.abs(g[1:4] - x).max() <= tol and np.abs(g[4:7] - v).max() <= tol * 10
            if small:
                scale = np.abs(a).max()
                assert np.abs(g[7:10] - a).max() <= 1e-11 * scale
                assert np.abs(g[10:13] - j).max() <= 1e-10 * np.abs(j).max()
                assert np.array_equal(g[14], dt)
                # nb_block_forces: the last block's forces, in ascending index order
                pa, pj, pp = nbmod.binding.nb_block_forces(ctx.h)
                ni = len(last[0])
                view = nbmod.context._DeviceView
                ga = torch.as_tensor(view(pa, 3 * ni, "<f8"), device=ctx.device).cpu().numpy().reshape(3, ni)
                gp = torch.as_tensor(view(pp, ni, "<f8"), device=ctx.device).cpu().numpy()
                assert np.abs(ga - last[1]).max() <= 1e-11 * scale
                assert np.abs(gp - last[3]).max() <= 1e-11 * np.abs(last[3]).max()
            else:
                assert (g[14] != dt).sum() <= max(2, n // 50)
            total += k
        ctx.sync()


def test_steps_flags_eps0_and_t_end(nbmod):
    """Unsoftened flagged pairs and eps2 = 0 inside the persistent kernel; t_end stops the run before
    the first block beyond it; k = 0 and a second call continue cleanly."""
    n, eta, lo, hi = 150, 0.02, 2.0 ** -18, 2.0 ** -6
    flags = np.zeros(n, np.uint8)
    flags[[3, 77, 149]] = 1
    for eps2 in (2.0 ** -8, 0.0):
        m, x, v, a, j, t, dt = _start(n, 950, eps2, eta, lo, hi, flags)
        with nbmod.Context(n) as ctx:
            ctx.steps_bound(1 << 40)
            _load(ctx, m, x, v, a, j, t, dt)
            ctx.set_flags(np.flatnonzero(flags).astype(np.int32), np.ones(3, np.uint8))
            assert ctx.steps(0, eps2, eta, lo, hi)[0] == 0
            rt, rni, _ = _oracle_steps(40, m, x, v, a, j, t, dt, eps2, eta, lo, hi, flags)
            t_end = rt[24]
            n_before = int((rt <= t_end).sum())
            done, gt, gni = ctx.steps(1000, eps2, eta, lo, hi, t_end=t_end)
            assert done == n_before and np.array_equal(gt, rt[:done]) and np.array_equal(gni, rni[:done])
            done2, gt2, gni2 = ctx.steps(40 - done, eps2, eta, lo, hi)
            assert done2 == 40 - done and np.array_equal(gt2, rt[done:]) and np.array_equal(gni2, rni[done:])
            g = ctx.state().cpu().numpy()
            assert np.array_equal(g[13], t) and np.array_equal(g[14], dt)
            assert np.abs(g[1:4] - x).max() <= 1e-11 and np.abs(g[4:7] - v).max() <= 1e-10
            ctx.sync()


@pytest.mark.parametrize("queue", [2, 1, 0])
def test_steps_host_path_and_mixed(nbmod, queue):
    """Bound 0: every block is handed over (the seam itself); default bound at N = 3000: a mix.
    queue = 2: handed-over blocks are planned on the device and their kernels run as the body of a
    WHILE node of one CUDA graph; 1: the same rounds queued on the stream ahead of time; 0: the host
    takes them through nb_step's launches.  The oracle is
    stepped in lock-step with the GPU's own log here, because fp32 forces may move a step decision
    near a threshold (tests/test_gpu_hermite.py)."""
    n, eps2, eta, lo, hi = 3000, 2.0 ** -12, 0.02, 2.0 ** -18, 2.0 ** -5
    m, x, v, a, j, t, dt = _start(n, 970, eps2, eta, lo, hi)
    with nbmod.Context(n) as ctx:
        ctx.steps_queue(queue)
        for bound, k in ((0, 12), (30000000, 48)):
            ctx.steps_bound(bound)
            _load(ctx, m, x, v, a, j, t, dt)
            l0 = ctx.launch_count()
            done, gt, gni, us = ctx.steps(k, eps2, eta, lo, hi, times=True)
            launches = ctx.launch_count() - l0
            rt, rni, last = _oracle_steps(k, m, x, v, a, j, t, dt, eps2, eta, lo, hi)
            assert done == k and np.array_equal(gt, rt)
            assert (gni != rni).sum() <= 2 and np.abs(gni - rni).max() <= 2
            assert (us > 0).all() and us.sum() < 1e6
            g = ctx.state().cpu().numpy()
            assert np.abs(g[1:4] - x).max() < 1e-7 and np.abs(g[4:7] - v).max() < 1e-5
            assert (g[14] != dt).sum() <= max(2, n // 100)
            if gni[-1] == rni[-1]:
                # nb_block_forces after a handed-over block: the packed fp32 kernel's tolerances
                pa, pj, pp = nbmod.binding.nb_block_forces(ctx.h)
                ni = len(last[0])
                view = nbmod.context._DeviceView
                ga = torch.as_tensor(view(pa, 3 * ni, "<f8"), device=ctx.device).cpu().numpy().reshape(3, ni)
                gp = torch.as_tensor(view(pp, ni, "<f8"), device=ctx.device).cpu().numpy()
                tol = 1e-5          # the trajectory went through fp32 blocks, whichever kernel took the last one
                assert (np.linalg.norm(ga - last[1], axis=0) <= tol * np.linalg.norm(last[1], axis=0)).all()
                assert (np.abs(gp - last[3]) <= tol * np.abs(last[3])).all()
            if bound == 0:
                assert launches >= 4 * k            # every block through launches of its own
            else:
                small = int(((gni <= 512) & (gni * n <= bound)).sum())
                print("mixed run (queue %d): %d of %d blocks in the persistent kernel, %d launches"
                      % (queue, small, k, launches))
                assert small > 0
                if queue != 1:              # mode 1 may queue rounds beyond the end of the run
                    assert launches < 6 * (k - small) + 2 * (k - small) + 8
        ctx.sync()


def test_steps_queue_modes_accepted(nbmod):
    nb = nbmod.binding
    with nbmod.Context(64) as ctx:
        for mode in (-1, 0, 1, 2, -1):
            ctx.steps_queue(mode)
        for mode in (-2, 3):
            with pytest.raises(nb.NBError) as e:
                ctx.steps_queue(mode)
            assert e.value.status == nb.NB_ERR_ARG


def test_steps_queued_flags_eps0_t_end_and_overflow(nbmod):
    """The device-planned path for handed-over blocks (bound 0: every block): unsoftened flagged
    pairs, eps2 = 0 (the guarded pair kernels), t_end, k larger than what is left, and a block above
    ni_max (NB_ERR_ARG, nothing advanced past it)."""
    n, eta, lo, hi = 700, 0.02, 2.0 ** -18, 2.0 ** -6
    flags = np.zeros(n, np.uint8)
    flags[[3, 77, 649]] = 1
    for eps2 in (2.0 ** -8, 0.0):
        m, x, v, a, j, t, dt = _start(n, 960, eps2, eta, lo, hi, flags)
        with nbmod.Context(n) as ctx:
            ctx.steps_bound(0)
            _load(ctx, m, x, v, a, j, t, dt)
            ctx.set_flags(np.flatnonzero(flags).astype(np.int32), np.ones(3, np.uint8))
            rt, rni, _ = _oracle_steps(30, m, x, v, a, j, t, dt, eps2, eta, lo, hi, flags)
            t_end = rt[17]
            n_before = int((rt <= t_end).sum())
            done, gt, gni = ctx.steps(1000, eps2, eta, lo, hi, t_end=t_end)
            assert done == n_before and np.array_equal(gt, rt[:done])
            assert (gni != rni[:done]).sum() <= 1
            done2, gt2, gni2 = ctx.steps(30 - done, eps2, eta, lo, hi)
            assert done2 == 30 - done and np.array_equal(gt2, rt[done:])
            g = ctx.state().cpu().numpy()
            assert np.array_equal(g[13], t)
            assert np.abs(g[1:4] - x).max() <= 1e-7 and np.abs(g[4:7] - v).max() <= 1e-5
            ctx.sync()
    # a block larger than ni_max: every particle due at once, ni_max = 256
    m, x, v, a, j, t, dt = _start(n, 961, 2.0 ** -8, eta, lo, hi)
    dt[:] = hi
    with nbmod.Context(n, ni_max=256) as ctx:
        _load(ctx, m, x, v, a, j, t, dt)
        with pytest.raises(nbmod.binding.NBError):
            ctx.steps(5, 2.0 ** -8, eta, lo, hi)
        g = ctx.state().cpu().numpy()
        assert np.array_equal(g[13], t) and np.array_equal(g[1:4], x)


@pytest.mark.parametrize("queue", [2, 1, 0])
def test_steps_slice_overflow_goes_to_host_path(nbmod, queue):
    """More than 128 due particles inside ONE slice of the persistent kernel (N = 30000: 148 slices of
    203): the slice cannot publish them all, the block must be handed to the host path, not truncated.
    And the device time log adds up."""
    n, eps2, eta, lo, hi = 30000, 2.0 ** -12, 0.02, 2.0 ** -16, 2.0 ** -6
    m, x, v = nbgen.plummer(n, 990)
    il = np.arange(n, dtype=np.int32)
    a, j, _ = oracle.force(m, x, v, il, eps2)
    t = np.zeros(n)
    dt = np.full(n, hi)
    dt[1000:1150] = lo                      # 150 consecutive particles due first, in one slice
    dt[20000] = 2 * lo
    with nbmod.Context(n) as ctx:
        ctx.steps_queue(queue)
        _load(ctx, m, x, v, a, j, t, dt)
        done, gt, gni, us = ctx.steps(3, eps2, eta, lo, hi, times=True)
        rt, rni, _ = _oracle_steps(3, m, x, v, a, j, t, dt, eps2, eta, lo, hi)
        assert done == 3 and np.array_equal(gt, rt) and np.array_equal(gni, rni), (gt, gni, rt, rni)
        assert rni[0] == 150
        g = ctx.state().cpu().numpy()
        assert np.array_equal(g[13], t)
        assert np.abs(g[1:4] - x).max() < 1e-9 and np.abs(g[4:7] - v).max() < 1e-7
        assert (us > 0).all() and us.sum() < 1e6
        print("device time per step (us):", us)
        ctx.sync()
