"""-m "not gpu": host logic of the multi-GPU decomposition (paper_1409_5474_b200/sharding.py),
world_size 2 over gloo on the CPU.  Each rank's "force call" here is the ORACLE on its i-slice
(tests may call the oracle); what is tested is the slicing and the assembly in i_list order, i.e.
that sharded == unsharded exactly (the i-particles are independent)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

torch = pytest.importorskip("torch")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_bounds_cover_without_overlap():
    import __graft_entry__ as g
    g.build()
    from paper_1409_5474_b200 import sharding
    for ni in (0, 1, 2, 7, 256, 1000, 1 << 20):
        for world in (1, 2, 3, 8):
            cuts = [sharding.shard_bounds(ni, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == ni
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_bounds(10, 2, 2)


def _worker(rank, world, port, ni, out_q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    import nbgen
    import oracle
    from paper_1409_5474_b200 import sharding
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = nbgen.config1(512)
        il = nbgen.permutation(5, c.n)[:ni]
        mine = sharding.shard_i_list(il, rank, world)
        a, j, p = oracle.force(c.m, c.x, c.v, mine, c.eps2)
        acc, jrk, pot = sharding.gather_forces(torch.from_numpy(a), torch.from_numpy(j),
                                               torch.from_numpy(p), len(il))
        ra, rj, rp = oracle.force(c.m, c.x, c.v, il, c.eps2)
        ok = (acc.numpy() == ra).all() and (jrk.numpy() == rj).all() and (pot.numpy() == rp).all()
        out_q.put((rank, bool(ok), tuple(acc.shape)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("ni", [301, 2, 1])
def test_gather_forces_world2_gloo(ni):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, ni, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == [0, 1]
    assert all(r[1] for r in res)
    assert all(r[2] == (3, ni) for r in res)


def _worker_j(rank, world, port, ni, eps2, out_q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    import nbgen
    import oracle
    from paper_1409_5474_b200 import sharding
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = nbgen.config1(777)
        c.m = c.m * (0.5 + nbgen.Streams(9, c.n).uniform())
        c.flags[[5, 300, 390, 776]] = 1                              # flagged on both sides of the cut
        c.x[:, 390] = c.x[:, 5] + 1e-3                               # a tight flagged pair ACROSS ranks
        il = nbgen.permutation(6, c.n)[:ni].copy()
        il[:min(ni, 4)] = [5, 390, 300, 776][:min(ni, 4)]
        lo, hi = sharding.shard_bounds(c.n, rank, world)             # this rank's j-slice
        pos = sharding.owned(il, lo, hi)
        mine = il[pos.numpy()]
        state = torch.from_numpy(np.concatenate([c.x[:, mine], c.v[:, mine], c.flags[None, mine].astype(np.float64),
                                                 mine[None].astype(np.float64)], 0))

        def by_value_ids(x, v, self_idx, iflags):
            # the rank's "nb_force_ext_ids": the oracle on its j-slice with the i-particles appended
            # massless; an i-particle that IS a member of the slice is evaluated in place (by index)
            xi, vi, sidx, ifl = x.numpy(), v.numpy(), self_idx.numpy(), iflags.numpy()
            k = xi.shape[1]
            mm = np.concatenate([c.m[lo:hi], np.zeros(k)])
            xx = np.concatenate([c.x[:, lo:hi], xi], 1)
            vv = np.concatenate([c.v[:, lo:hi], vi], 1)
            ff = np.concatenate([c.flags[lo:hi], ifl]).astype(np.uint8)
            who = np.where(sidx >= 0, sidx, hi - lo + np.arange(k)).astype(np.int32)
            a, j, p = oracle.force(mm, xx, vv, who, eps2, ff)
            return torch.from_numpy(a), torch.from_numpy(j), torch.from_numpy(p)

        acc, jrk, pot = sharding.force_j_sharded(by_value_ids, state, pos, len(il), lo, hi)
        ra, rj, rp = oracle.force(c.m, c.x, c.v, il, eps2, c.flags)
        ea = np.abs(acc.numpy() - ra).max() / np.abs(ra).max()
        ej = np.abs(jrk.numpy() - rj).max() / np.abs(rj).max()
        ep = np.abs(pot.numpy() - rp).max() / np.abs(rp).max()
        soft = oracle.force(c.m, c.x, c.v, il, eps2)                 # the flags must matter in this case
        differs = bool(np.abs(soft[0] - ra).max() > 1e-3 * np.abs(ra).max()) or eps2 != 1e-4
        out_q.put((rank, float(max(ea, ej, ep)), differs))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("ni,eps2", [(301, 1e-4), (5, 1e-4), (64, 0.0), (301, 1e-12)])
def test_force_j_sharded_world2_gloo(ni, eps2):
    """j distributed over the ranks, partial forces summed.  Equal to the unsharded
    sum up to the order of the fp64 additions, including unsoftened flagged pairs across the cut
    and a softening small enough that a self pair left in would dominate pot."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_j, args=(r, 2, port, ni, eps2, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == [0, 1]
    assert all(r[1] < 1e-12 for r in res), res
    assert all(r[2] for r in res), res


def _worker_x(rank, world, port, ni, eps2, out_q):
    """Host logic of the peer-memory exchange (sharding.xchg_connect / force_j_sharded_xchg).  The
    stand-in context does on the CPU what csrc/xchg.h does on the device -- every rank has a window of
    `world` slots, a push writes a rank's partial forces into slot [rank] of EVERY window, the sum adds
    the slots of one's own window in rank order -- with files under a shared directory as the
    "peer memory" and the oracle as each rank's pair kernel."""
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import tempfile
    import time
    import torch.distributed as dist
    import nbgen
    import oracle
    from paper_1409_5474_b200 import sharding
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = nbgen.config1(777)
        c.m = c.m * (0.5 + nbgen.Streams(9, c.n).uniform())
        c.flags[[5, 300, 390, 776]] = 1
        c.x[:, 390] = c.x[:, 5] + 1e-3
        lo, hi = sharding.shard_bounds(c.n, rank, world)
        shared = [tempfile.mkdtemp(prefix="nbx%d_" % rank)]

        class Window:
            def __init__(self):
                self.rank = self.world = None
                self.cap = 0
                self.peers = {}
                self.epoch = 0
                self.log = []

            def xchg_create(self, r, w, ni_cap):
                self.rank, self.world, self.cap = r, w, ni_cap
                self.peers = {r: shared[0]}
                self.log.append(("create", r, w))

            def xchg_export(self):
                return ("%-64s" % shared[0]).encode()[:64], 0

            def xchg_attach(self, peer, handle=None, same_process_ptr=None):
                assert handle is not None and len(handle) == 64 and peer != self.rank
                self.peers[peer] = handle.decode().strip()
                self.log.append(("attach", peer))

            def xforce(self, x, v, self_idx, iflags, eps2_):
                assert sorted(self.peers) == list(range(self.world)) and x.shape[1] <= self.cap
                self.epoch += 1
                xi, vi, sidx, ifl = x.numpy(), v.numpy(), self_idx.numpy(), iflags.numpy()
                k = xi.shape[1]
                mm = np.concatenate([c.m[lo:hi], np.zeros(k)])
                xx = np.concatenate([c.x[:, lo:hi], xi], 1)
                vv = np.concatenate([c.v[:, lo:hi], vi], 1)
                ff = np.concatenate([c.flags[lo:hi], ifl]).astype(np.uint8)
                who = np.where(sidx >= 0, sidx, hi - lo + np.arange(k)).astype(np.int32)
                a, j, p = oracle.force(mm, xx, vv, who, eps2_, ff)
                part = np.concatenate([a, j, p[None]], 0)
                buf = self.epoch & 1
                for peer, d in self.peers.items():                      # push: data, then the flag
                    np.save(os.path.join(d, "slot%d_%d.npy" % (buf, self.rank)), part)
                    with open(os.path.join(d, "flag%d_%d.tmp" % (buf, self.rank)), "w") as f:
                        f.write(str(self.epoch))
                    os.replace(os.path.join(d, "flag%d_%d.tmp" % (buf, self.rank)),
                               os.path.join(d, "flag%d_%d" % (buf, self.rank)))
                total = None
                for r in range(self.world):                             # wait and sum, rank 0 first
                    fn = os.path.join(shared[0], "flag%d_%d" % (buf, r))
                    t0 = time.time()
                    while True:
                        try:
                            if int(open(fn).read() or -1) == self.epoch:
                                break
                        except (OSError, ValueError):
                            pass
                        assert time.time() - t0 < 60
                        time.sleep(0.001)
                    s = np.load(os.path.join(shared[0], "slot%d_%d.npy" % (buf, r)))
                    total = s if total is None else total + s
                t = torch.from_numpy(total)
                return t[0:3], t[3:6], t[6]

        w = Window()
        assert sharding.xchg_connect(w, 512) == (rank, world)
        assert w.log == [("create", rank, world)] + [("attach", r) for r in range(world) if r != rank]
        worst, same = 0.0, True
        for call in range(3):                                           # walks through both buffers
            il = nbgen.permutation(6 + call, c.n)[:ni].copy()
            il[:min(ni, 4)] = [5, 390, 300, 776][:min(ni, 4)]
            pos = sharding.owned(il, lo, hi)
            mine = il[pos.numpy()]
            state = torch.from_numpy(np.concatenate([c.x[:, mine], c.v[:, mine],
                                                     c.flags[None, mine].astype(np.float64),
                                                     mine[None].astype(np.float64)], 0))
            acc, jrk, pot = sharding.force_j_sharded_xchg(w, state, pos, len(il), lo, hi, eps2)
            ra, rj, rp = oracle.force(c.m, c.x, c.v, il, eps2, c.flags)
            worst = max(worst, np.abs(acc.numpy() - ra).max() / np.abs(ra).max(),
                        np.abs(jrk.numpy() - rj).max() / np.abs(rj).max(),
                        np.abs(pot.numpy() - rp).max() / np.abs(rp).max())
            both = [None] * world
            dist.all_gather_object(both, (acc.numpy().tobytes(), jrk.numpy().tobytes(), pot.numpy().tobytes()))
            same = same and all(b == both[0] for b in both)             # identical bits on every rank
        out_q.put((rank, float(worst), bool(same)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("ni,eps2,world", [(301, 1e-4, 2), (5, 1e-12, 2), (64, 1e-4, 3)])
def test_xchg_host_logic_world2_gloo(ni, eps2, world):
    """sharding.xchg_connect wires every rank to every peer's window (handles travel by
    all_gather_object, own rank skipped, barrier before the first push) and force_j_sharded_xchg returns
    the unsharded force on every rank, bit-identical across ranks (rank-order sum); two and three ranks."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_x, args=(r, world, port, ni, eps2, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == list(range(world))
    assert all(r[1] < 1e-12 for r in res), res
    assert all(r[2] for r in res), res


def _worker_step(rank, world, port, steps, out_q):
    """sharding.step_j_sharded over gloo: every rank's context is a stand-in that keeps a slice of the
    particles and answers next_block / predict / predicted / force_ext_ids / correct with the oracle
    (oracle/hermite.py, oracle.predict, oracle.force).  The sharded run must reproduce the oracle's
    unsharded block-step integration: same block times and sizes, same state."""
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    import nbgen
    import oracle
    from oracle import hermite as H
    from paper_1409_5474_b200 import sharding
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, eps2, eta, dmin, dmax = 200, 2.0 ** -10, 0.02, 2.0 ** -12, 2.0 ** -6
        m, x, v = nbgen.plummer(n, 977)
        m = m * (0.5 + nbgen.Streams(978, n).uniform())
        flags = np.zeros(n, np.uint8)
        flags[[3, 150]] = 1
        il = np.arange(n, dtype=np.int32)
        a, j, _ = oracle.force(m, x, v, il, eps2, flags)
        t = np.zeros(n)
        dt = H.quantise_dt(H.initial_dt(a, j, eta), dmin, dmax)
        lo, hi = sharding.shard_bounds(n, rank, world)

        class Slice:
            """particles [lo, hi) of the set, with the oracle as every kernel"""
            def __init__(self):
                sl = slice(lo, hi)
                self.m, self.x, self.v = m[sl].copy(), x[:, sl].copy(), v[:, sl].copy()
                self.a, self.j, self.t, self.dt = a[:, sl].copy(), j[:, sl].copy(), t[sl].copy(), dt[sl].copy()
                self.f = flags[sl].copy()

            def next_block(self):
                t1, idx = H.next_block(self.t, self.dt)
                return t1, len(idx), torch.from_numpy(idx)

            def predict(self, tp):
                self.xp, self.vp = oracle.predict(tp, self.x, self.v, self.a, self.j, self.t)

            def predicted(self):
                return torch.from_numpy(self.xp), torch.from_numpy(self.vp)

            def force_ext_ids(self, xi, vi, sidx, ifl, e2):
                xi, vi, sidx, ifl = xi.numpy(), vi.numpy(), sidx.numpy(), ifl.numpy()
                k = xi.shape[1]
                mm = np.concatenate([self.m, np.zeros(k)])
                xx = np.concatenate([self.xp, xi], 1)
                vv = np.concatenate([self.vp, vi], 1)
                ff = np.concatenate([self.f, ifl]).astype(np.uint8)
                who = np.where(sidx >= 0, sidx, hi - lo + np.arange(k)).astype(np.int32)
                fa, fj, fp = oracle.force(mm, xx, vv, who, e2, ff)
                return torch.from_numpy(fa), torch.from_numpy(fj), torch.from_numpy(fp)

            def correct(self, idx, t1, a1, j1, eta_, dmin_, dmax_):
                H.corrector_step(self.x, self.v, self.a, self.j, self.t, self.dt, idx.numpy().astype(np.int64), t1,
                                 a1.numpy(), j1.numpy(), eta_, dmin_, dmax_)

        me = Slice()
        fl = torch.from_numpy(me.f)
        log = [sharding.step_j_sharded(me, lo, hi, fl, eps2, eta, dmin, dmax, exchange="nccl") for _ in range(steps)]
        # the unsharded oracle run from the same start
        ref = []
        for _ in range(steps):
            t1, idx = H.next_block(t, dt)
            xp, vp = oracle.predict(t1, x, v, a, j, t)
            a1, j1, _ = oracle.force(m, xp, vp, idx, eps2, flags)
            H.corrector_step(x, v, a, j, t, dt, idx, t1, a1, j1, eta, dmin, dmax)
            ref.append((t1, len(idx)))
        sl = slice(lo, hi)
        same_log = [(float(q[0]), int(q[1])) for q in log] == [(float(q[0]), int(q[1])) for q in ref]
        err = max(np.abs(me.x - x[:, sl]).max(), np.abs(me.v - v[:, sl]).max(), np.abs(me.a - a[:, sl]).max() * 1e-3)
        same_dt = bool(np.array_equal(me.dt, dt[sl]) and np.array_equal(me.t, t[sl]))
        out_q.put((rank, same_log, float(err), same_dt, max(q[1] for q in ref)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_step_j_sharded_world2_gloo(world):
    """PAPER.md:41/:49 on the j-sharded layout of PAPER.md:55: 40 block steps (past t = 2^-6, where
    every particle is due at once) with two ranks equal the unsharded oracle integration."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_step, args=(r, world, port, 40, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == list(range(world))
    assert all(r[1] for r in res), res                 # block times and sizes identical to the unsharded run
    assert all(r[2] < 1e-11 for r in res), res         # state equal up to the order of the fp64 additions
    assert all(r[3] for r in res), res                 # every particle's time and power-of-two step identical
    assert res[0][4] == 200                            # the run contains the all-particles block
