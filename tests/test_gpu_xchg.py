"""-m gpu: nb_xforce -- the j-sharded scheme of PAPER.md:55 with the exchange of the partial forces done
by the kernels themselves over peer memory (csrc/xchg.h), checked on ONE GPU:

* world 1: the complete path (window, push to oneself, flag, wait, sum) must return nb_force_ext_ids'
  forces bit for bit (x + nothing = x), in the one-launch form (ni <= 16) and with the two exchange
  kernels (ni > 16);
* two ranks as two contexts of one process, each holding half of the particles and the other's window
  attached by address.  Kernels of one rank never wait for kernels of the other here: both ranks push
  first (phase 1), then both sum (phase 2) -- or one rank pushes and the other then runs the one-launch
  form, whose wait finds the flag already raised.  Both ranks must get the same bits, the oracle's
  forces within the mixed-precision tolerances, and the unsharded nb_force result to fp32 summation
  order; repeated
  calls walk through both buffers of the windows."""
import numpy as np
import pytest

import nbgen
import oracle
from util import check_parity, rel_err_scalar, rel_err_vec

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _j_set(n, seed):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    a, j = nbgen.mean_field(x, v)
    t = 0.25 * nbgen.Streams(seed + 2, n).uniform()
    return m, x, v, a, j, t


def _load_slice(ctx, lo, hi, m, x, v, a, j, tj, flags, t):
    ctx.set_j(m[lo:hi], x[:, lo:hi], v[:, lo:hi], a[:, lo:hi], j[:, lo:hi], tj[lo:hi])
    fl = np.flatnonzero(flags[lo:hi]).astype(np.int32)
    if len(fl):
        ctx.set_flags(fl, np.ones(len(fl), np.uint8))
    ctx.predict(t)


def test_world_of_one_is_the_by_value_call(nbmod):
    n, t = 3000, 0.2
    m, x, v, a, j, tj = _j_set(n, 910)
    flags = np.zeros(n, np.uint8)
    flags[[40, 1100]] = 1
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    with nbmod.Context(n, 512) as ctx:
        _load_slice(ctx, 0, n, m, x, v, a, j, tj, flags, t)
        ctx.xchg_create(0, 1, 512)
        handle, ptr = ctx.xchg_export()
        assert len(handle) == nbmod.binding.NB_XCHG_HANDLE_BYTES and ptr != 0
        ctx.xchg_attach(0, same_process_ptr=ptr)               # own rank: accepted and ignored
        for ni, eps2 in ((5, 2.0 ** -14), (16, 0.0), (17, 1e-12), (300, 2.0 ** -14), (5, 1e-12)):
            il = nbgen.permutation(911 + ni, n)[:ni].astype(np.int32)
            il[:2] = [40, 1100]
            args = (xp[:, il], vp[:, il], il, flags[il], eps2)
            want = [q.cpu().numpy() for q in ctx.force_ext_ids(*args)]
            k0 = ctx.launch_count()
            got = [q.cpu().numpy() for q in ctx.xforce(*args)]
            launches = ctx.launch_count() - k0
            ctx.sync()
            for g, w in zip(got, want):
                assert np.array_equal(g, w)
            assert launches == (1 if ni <= 16 else 4)          # pair + reduce + push + sum when not fused
            check_parity(got, oracle.force(m, xp, vp, il, eps2, flags))
        # split form
        part = ctx.xforce(*args, phase=1)
        got = [q.cpu().numpy() for q in ctx.xforce(None, None, None, None, eps2, phase=2, out=part)]
        ctx.sync()
        for g, w in zip(got, want):
            assert np.array_equal(g, w)
        ctx.xchg_destroy()
        with pytest.raises(nbmod.binding.NBError) as e:
            ctx.xforce(*args)
        assert e.value.status == nbmod.binding.NB_ERR_STATE


def test_two_ranks_in_one_process(nbmod):
    n, cut, t = 4096, 2048, 0.2
    m, x, v, a, j, tj = _j_set(n, 920)
    flags = np.zeros(n, np.uint8)
    flags[[40, 1100, 2105, 3900]] = 1
    x[:, 2105] = x[:, 40] + 2e-3                              # a close flagged pair across the cut
    v[:, 2105], a[:, 2105], j[:, 2105], tj[2105] = v[:, 40], a[:, 40], j[:, 40], tj[40]
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    bounds = ((0, cut), (cut, n))
    with nbmod.Context(n, 512) as full, nbmod.Context(cut, 512) as c0, nbmod.Context(n - cut, 512) as c1:
        ranks = (c0, c1)
        _load_slice(full, 0, n, m, x, v, a, j, tj, flags, t)
        for r, c in enumerate(ranks):
            _load_slice(c, bounds[r][0], bounds[r][1], m, x, v, a, j, tj, flags, t)
            c.xchg_create(r, 2, 400)
        # a rank whose peer is not attached refuses
        with pytest.raises(nbmod.binding.NBError) as e:
            c0.xforce(xp[:, :3], vp[:, :3], np.array([0, 1, 2], np.int32), None, 1e-4)
        assert e.value.status == nbmod.binding.NB_ERR_STATE
        ptrs = [c.xchg_export()[1] for c in ranks]
        c0.xchg_attach(1, same_process_ptr=ptrs[1])
        c1.xchg_attach(0, same_process_ptr=ptrs[0])

        call = 0
        for ni, eps2 in ((5, 2.0 ** -14), (12, 1e-12), (300, 2.0 ** -14), (8, 0.0), (16, 2.0 ** -14), (300, 0.0),
                         (1, 1e-12)):
            il = nbgen.permutation(921 + call, n)[:ni].astype(np.int32)
            il[:min(ni, 4)] = [40, 1100, 2105, 3900][:min(ni, 4)]
            ref = oracle.force(m, xp, vp, il, eps2, flags)
            unsharded = [q.cpu().numpy() for q in full.force(il, eps2)]
            args = []
            for r in range(2):
                lo, hi = bounds[r]
                self_idx = np.where((il >= lo) & (il < hi), il - lo, -1).astype(np.int32)
                args.append((xp[:, il], vp[:, il], self_idx, flags[il], eps2))
            if call % 2 == 0:
                # both push, then both sum
                parts = [ranks[r].xforce(*args[r], phase=1) for r in range(2)]
                for c in ranks:
                    c.sync()
                outs = [ranks[r].xforce(None, None, None, None, eps2, phase=2, out=parts[r]) for r in range(2)]
            else:
                # rank 1 pushes; rank 0 runs the whole call (one launch for ni <= 16: its wait finds rank
                # 1's flag raised); rank 1 sums afterwards
                p1 = c1.xforce(*args[1], phase=1)
                c1.sync()
                k0 = c0.launch_count()
                o0 = c0.xforce(*args[0], phase=0)
                assert c0.launch_count() - k0 == (1 if ni <= 16 else 4)
                c0.sync()
                outs = [o0, c1.xforce(None, None, None, None, eps2, phase=2, out=p1)]
            for c in ranks:
                c.sync()
            got = [[q.cpu().numpy() for q in o] for o in outs]
            for q0, q1 in zip(got[0], got[1]):
                assert np.array_equal(q0, q1)                  # same bits on both ranks
            check_parity(got[0], ref)
            # the unsharded by-index call groups its fp32 partial sums differently (another mapping)
            assert rel_err_vec(got[0][0], unsharded[0]).max() <= 2e-6
            assert rel_err_vec(got[0][1], unsharded[1]).max() <= 4e-5
            assert rel_err_scalar(got[0][2], unsharded[2]).max() <= 2e-6
            call += 1
        with pytest.raises(nbmod.binding.NBError) as e:       # above the window's capacity
            c0.xforce(xp[:, :401], vp[:, :401], np.full(401, -1, np.int32), None, 1e-4)
        assert e.value.status == nbmod.binding.NB_ERR_ARG


def _ipc_worker(rank, world, port, out_q):
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    sys.path.insert(0, os.path.join(root, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import sharding
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, t = 4096, 0.2
        m, x, v, a, j, tj = _j_set(n, 930)
        flags = np.zeros(n, np.uint8)
        flags[[40, 3900]] = 1
        xp, vp = oracle.predict(t, x, v, a, j, tj)
        lo, hi = sharding.shard_bounds(n, rank, world)
        worst, bits = 0.0, []
        with nbm.Context(hi - lo, 512) as ctx:
            _load_slice(ctx, lo, hi, m, x, v, a, j, tj, flags, t)
            assert sharding.xchg_connect(ctx, 400) == (rank, world)     # IPC handles over all_gather_object
            for call, (ni, eps2) in enumerate(((5, 2.0 ** -14), (300, 1e-12), (16, 0.0))):
                il = nbgen.permutation(931 + call, n)[:ni].astype(np.int32)
                il[:2] = [40, 3900]
                self_idx = np.where((il >= lo) & (il < hi), il - lo, -1).astype(np.int32)
                part = ctx.xforce(xp[:, il], vp[:, il], self_idx, flags[il], eps2, phase=1)
                ctx.sync()
                dist.barrier()                                          # every rank has pushed: nobody waits on the GPU
                got = [q.cpu().numpy() for q in ctx.xforce(None, None, None, None, eps2, phase=2, out=part)]
                ctx.sync()
                ref = oracle.force(m, xp, vp, il, eps2, flags)
                worst = max(worst, rel_err_vec(got[0], ref[0]).max() / 1e-5, rel_err_vec(got[1], ref[1]).max() / 1e-4,
                            rel_err_scalar(got[2], ref[2]).max() / 1e-5)
                bits.append(b"".join(q.tobytes() for q in got))
                dist.barrier()
            both = [None] * world
            dist.all_gather_object(both, bits)
            same = all(b == both[0] for b in both)
            dist.barrier()                                              # peers stay alive until everybody is done
        out_q.put((rank, float(worst), bool(same)))
    finally:
        dist.destroy_process_group()


def test_two_processes_share_windows_by_ipc_handle(nbmod):
    """Two PROCESSES on the one GPU, each a rank with half of the particles: sharding.xchg_connect
    exchanges real CUDA IPC handles, pushes land in the other process's window.  The halves of the call
    are separated by a host barrier, so no kernel of one process waits for the other's."""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_ipc_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=300) for _ in procs]
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == [0, 1]
    assert all(r[1] <= 1.0 for r in res), res          # within the north_star tolerances of the oracle
    assert all(r[2] for r in res), res                 # identical bits in both processes


def test_a_silent_peer_is_reported_not_waited_for_forever(nbmod):
    """Rank 0 of 2 whose peer never pushes: the wait gives up after the time limit, latches NB_ERR_PEER
    (nb_sync) and the context stays usable."""
    n, t = 2048, 0.1
    m, x, v, a, j, tj = _j_set(n, 940)
    flags = np.zeros(n, np.uint8)
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    with nbmod.Context(n, 64) as c0, nbmod.Context(n, 64) as c1:
        for r, c in enumerate((c0, c1)):
            _load_slice(c, 0, n, m, x, v, a, j, tj, flags, t)
            c.xchg_create(r, 2, 64)
        c0.xchg_attach(1, same_process_ptr=c1.xchg_export()[1])
        c0.xchg_timeout(0.05)
        il = np.arange(5, dtype=np.int32)
        for ni in (5, 40):                                     # in the pair kernel's last CTA; in xchg_sum_kernel
            c0.xforce(xp[:, :ni], vp[:, :ni], np.arange(ni, dtype=np.int32), None, 1e-4)
            with pytest.raises(nbmod.binding.NBError) as e:
                c0.sync()
            assert e.value.status == nbmod.binding.NB_ERR_PEER
        c0.sync()                                              # the latch is cleared
        got = [q.cpu().numpy() for q in c0.force(il, 1e-4)]
        c0.sync()
        check_parity(got, oracle.force(m, xp, vp, il, 1e-4))
        with pytest.raises(nbmod.binding.NBError):
            c0.xchg_timeout(0.0)


def test_a_rank_with_an_empty_slice(nbmod):
    """World of two where rank 1 holds no particle at all: its partial forces are zeros, the sum is rank
    0's force (bit for bit), in both exchange forms."""
    n, t = 2000, 0.1
    m, x, v, a, j, tj = _j_set(n, 950)
    flags = np.zeros(n, np.uint8)
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    with nbmod.Context(n, 64) as c0, nbmod.Context(16, 64) as c1:
        _load_slice(c0, 0, n, m, x, v, a, j, tj, flags, t)
        c1.predict(t)                                          # nothing loaded: n = 0
        for r, c in enumerate((c0, c1)):
            c.xchg_create(r, 2, 64)
        c0.xchg_attach(1, same_process_ptr=c1.xchg_export()[1])
        c1.xchg_attach(0, same_process_ptr=c0.xchg_export()[1])
        for ni in (3, 40):
            il = nbgen.permutation(951 + ni, n)[:ni].astype(np.int32)
            none = np.full(ni, -1, np.int32)
            want = [q.cpu().numpy() for q in c0.force_ext_ids(xp[:, il], vp[:, il], il, None, 1e-4)]
            p1 = c1.xforce(xp[:, il], vp[:, il], none, None, 1e-4, phase=1)
            c1.sync()
            assert all(float(q.abs().max()) == 0.0 for q in p1)
            got = [q.cpu().numpy() for q in c0.xforce(xp[:, il], vp[:, il], il, None, 1e-4)]
            o1 = [q.cpu().numpy() for q in c1.xforce(None, None, None, None, 1e-4, phase=2, out=p1)]
            c0.sync()
            c1.sync()
            for g, w, o in zip(got, want, o1):
                assert np.array_equal(g, w) and np.array_equal(o, w)


def _step_worker(rank, world, port, out_q):
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    sys.path.insert(0, os.path.join(root, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    from oracle import hermite as H
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import sharding
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, eps2, eta, dmin, dmax, steps = 1024, 2.0 ** -12, 0.02, 2.0 ** -14, 2.0 ** -6, 14
        m, x, v = nbgen.plummer(n, 960)
        m = m * (0.5 + nbgen.Streams(961, n).uniform())
        flags = np.zeros(n, np.uint8)
        flags[[10, 900]] = 1
        il = np.arange(n, dtype=np.int32)
        a, j, _ = oracle.force(m, x, v, il, eps2, flags)
        t = np.zeros(n)
        dt = H.quantise_dt(H.initial_dt(a, j, eta), dmin, dmax)
        lo, hi = sharding.shard_bounds(n, rank, world)
        sl = slice(lo, hi)
        dev = torch.device("cuda", 0)
        with nbm.Context(hi - lo, n) as ctx:
            ctx.set_j(m[sl], x[:, sl], v[:, sl], a[:, sl], j[:, sl], t[sl])
            fl = np.flatnonzero(flags[sl]).astype(np.int32)
            if len(fl):
                ctx.set_flags(fl, np.ones(len(fl), np.uint8))
            ctx.set_dt(dt[sl])
            sharding.xchg_connect(ctx, n)
            fdev = torch.from_numpy(flags[sl].copy()).to(dev)
            log = [sharding.step_j_sharded(ctx, lo, hi, fdev, eps2, eta, dmin, dmax, exchange="xchg_split")
                   for _ in range(steps)]
            ctx.sync()
            mine = ctx.state().cpu().numpy()
            dist.barrier()
        # the same steps by ONE context holding all particles (nb_step), on this rank's own
        with nbm.Context(n) as full:
            full.set_j(m, x, v, a, j, t)
            full.set_flags(np.array([10, 900], np.int32), np.ones(2, np.uint8))
            full.set_dt(dt)
            ref = [full.step(eps2, eta, dmin, dmax) for _ in range(steps)]
            full.sync()
            want = full.state().cpu().numpy()[:, sl]
        same_log = [(float(q[0]), int(q[1])) for q in log] == [(float(q[0]), int(q[1])) for q in ref]
        err_x = float(np.abs(mine[1:4] - want[1:4]).max())
        err_v = float(np.abs(mine[4:7] - want[4:7]).max())
        same_dt = bool(np.array_equal(mine[13], want[13]) and np.array_equal(mine[14], want[14]))
        out_q.put((rank, same_log, err_x, err_v, same_dt, int(max(q[1] for q in ref))))
    finally:
        dist.destroy_process_group()


def test_block_steps_of_two_ranks_equal_one_context(nbmod):
    """sharding.step_j_sharded with real contexts: two processes on the one GPU, each scheduling,
    predicting and correcting half of 1024 particles, forces through nb_xforce (split halves: no kernel
    waits for another process's kernel).  14 block steps give the block times, block sizes, particle
    times and power-of-two steps of ONE context running nb_step on all particles, and its positions to
    fp32-summation order."""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_step_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=300) for _ in procs]
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == [0, 1]
    assert all(r[1] for r in res), res
    assert all(r[2] < 1e-9 and r[3] < 1e-7 for r in res), res
    assert all(r[4] for r in res), res
