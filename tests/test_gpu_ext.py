"""-m gpu: nb_force_ext (i-particles by value, "a completely different set"; with jerk,
or acc + pot only) against the fp64 oracle.  The oracle needs no new code for this: the i-particles
are appended to the j-set as MASSLESS particles and addressed by index -- massless particles exert
nothing on each other and the self pair of an appended particle is skipped by index (R5), so
oracle.force on the joined set is exactly the by-value sum."""
import numpy as np
import pytest

import nbgen
import oracle
from util import check_parity, rel_err_scalar, rel_err_vec, TOL_ACC, TOL_POT

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


def _i_set(ni, seed, shift):
    """A second Plummer sphere, displaced so that the two systems overlap partly."""
    _, x, v = nbgen.plummer(max(ni, 2), seed)
    x, v = x[:, :ni].copy(), v[:, :ni].copy()
    x[0] += shift
    return x, v


def _oracle_ext(m, xp, vp, xi, vi, eps2):
    n, ni = m.shape[0], xi.shape[1]
    mm = np.concatenate([m, np.zeros(ni)])
    xx = np.concatenate([xp, xi], axis=1)
    vv = np.concatenate([vp, vi], axis=1)
    return oracle.force(mm, xx, vv, np.arange(n, n + ni, dtype=np.int32), eps2)


@pytest.mark.parametrize("ni", [1, 7, 64, 300, 2049])
@pytest.mark.parametrize("eps2", [2.0 ** -14, 0.0])
def test_force_ext_with_jerk(nbmod, ni, eps2):
    n, t = 6000, 0.3
    m, x, v, a, j, tj = _j_set(n, 700)
    xi, vi = _i_set(ni, 800 + ni, 0.7)
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    if ni >= 7:
        # an i-particle exactly on top of a j-particle: -m/eps in pot when softened, nothing when not (R6)
        xi[:, 3], vi[:, 3] = xp[:, 1234], vp[:, 1234]
    ref = _oracle_ext(m, xp, vp, xi, vi, eps2)
    with nbmod.Context(n, max(ni, 1)) as ctx:
        ctx.set_j(m, x, v, a, j, tj)
        ctx.predict(t)
        for splits in (0, 1, 5):
            ctx.tuning(splits, 0)
            got = [q.cpu().numpy() for q in ctx.force_ext(xi, vi, eps2)]
            check_parity(got, ref)
        again = [q.cpu().numpy() for q in ctx.force_ext(xi, vi, eps2)]
        assert all((p == q).all() for p, q in zip(again, got))          # deterministic (R9)
        ctx.sync()


@pytest.mark.parametrize("ni", [1, 9, 300, 2049])
def test_force_ext_acc_pot_only(nbmod, ni):
    n, t, eps2 = 6000, 0.3, 2.0 ** -14
    m, x, v, a, j, tj = _j_set(n, 710)
    xi, vi = _i_set(ni, 810 + ni, -0.4)
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    ra, _, rp = _oracle_ext(m, xp, vp, xi, np.zeros_like(xi), eps2)
    with nbmod.Context(n, max(ni, 1)) as ctx:
        ctx.set_j(m, x, v, a, j, tj)
        ctx.predict(t)
        acc, jrk, pot = ctx.force_ext(xi, None, eps2)
        assert jrk is None
        ga, gp = acc.cpu().numpy(), pot.cpu().numpy()
        ctx.sync()
    assert rel_err_vec(ga, ra).max() <= TOL_ACC and rel_err_scalar(gp, rp).max() <= TOL_POT


def test_force_ext_argument_errors(nbmod):
    nb = nbmod.binding
    with nbmod.Context(64, 8) as ctx:
        z = torch.zeros((3, 4), dtype=torch.float64, device=ctx.device)
        p = torch.zeros(4, dtype=torch.float64, device=ctx.device)
        with pytest.raises(nb.NBError) as e:                     # before any nb_predict
            nb.nb_force_ext(ctx.h, 4, z, z, 1e-4, z, z, p)
        assert e.value.status == nb.NB_ERR_STATE
        m, x, v = nbgen.plummer(64, 5)
        ctx.set_j(m, x, v)
        ctx.predict(0.0)
        for args in ((4, z, None, 1e-4, z, z, p),                # jerk asked for without velocities
                     (4, z, z, 1e-4, z, None, p),                # velocities given, no jerk buffer
                     (9, z, z, 1e-4, z, z, p),                   # ni > ni_max
                     (4, z, z, -1.0, z, z, p)):                  # negative eps2
            with pytest.raises(nb.NBError) as e:
                nb.nb_force_ext(ctx.h, *args)
            assert e.value.status == nb.NB_ERR_ARG
        nb.nb_force_ext(ctx.h, 0, None, None, 1e-4, None, None, None)   # ni = 0: no-op
        ctx.sync()


def test_bridge_kick_two_galaxies(nbmod):
    """The use NEXT-2 names: the kick galaxy B's stars receive from galaxy A (config 4's two
    spheres at a quarter of the size), acc + pot only, checked on 1024 sampled stars of B; and the
    momentum the two mutual kicks exchange cancels (sum m a over B = - sum m a over A)."""
    c = nbgen.config4(n_gal=1 << 17)
    na = (1 << 17) + 1
    eps2 = c.eps2
    A = (c.m[:na].copy(), np.ascontiguousarray(c.x[:, :na]), np.ascontiguousarray(c.v[:, :na]))
    B = (c.m[na:].copy(), np.ascontiguousarray(c.x[:, na:]), np.ascontiguousarray(c.v[:, na:]))
    with nbmod.Context(na) as ctx:
        ctx.set_j(*A)
        ctx.predict(0.0)
        acc_b, _, pot_b = ctx.force_ext(B[1], None, eps2)
        acc_b, pot_b = acc_b.cpu().numpy(), pot_b.cpu().numpy()
        ctx.set_j(*B)
        ctx.predict(0.0)
        acc_a = ctx.force_ext(A[1], None, eps2)[0].cpu().numpy()
        ctx.sync()
    pos = nbgen.sample_positions(nbgen.SEED0 * 100 + 42, B[0].shape[0], 1024)
    ra, _, rp = _oracle_ext(A[0], A[1], A[2], B[1][:, pos], np.zeros((3, len(pos))), eps2)
    assert rel_err_vec(acc_b[:, pos], ra).max() <= TOL_ACC
    assert rel_err_scalar(pot_b[pos], rp).max() <= TOL_POT
    pa, pb = (A[0] * acc_a).sum(1), (B[0] * acc_b).sum(1)
    assert np.abs(pa + pb).max() <= 1e-7 * np.abs(pa).max()


def test_by_value_members_of_a_j_slice(nbmod):
    """nb_force_ext_ids: the call one GPU makes in the j-sharded scheme.  The context holds
    a SLICE of the particles; the active particles come by value, some of them members of the slice
    (self pair excluded by index, also at a softening where it would swamp pot), some flagged
    (unsoftened pairs with the flagged members of the slice, R7).  Oracle: the full set with the
    masses outside the slice zeroed."""
    n, lo, hi, t = 3000, 1000, 2500, 0.2
    m, x, v, a, j, tj = _j_set(n, 730)
    flags = np.zeros(n, np.uint8)
    flags[[40, 1100, 1105, 2400, 2900]] = 1
    x[:, 1105] = x[:, 40] + 2e-3                       # flagged i outside the slice, flagged j inside, close
    v[:, 1105], a[:, 1105], j[:, 1105], tj[1105] = v[:, 40], a[:, 40], j[:, 40], tj[40]    # and staying close
    xp, vp = oracle.predict(t, x, v, a, j, tj)
    mm = m.copy()
    mm[:lo] = 0.0
    mm[hi:] = 0.0
    for ni, eps2 in ((300, 2.0 ** -14), (12, 1e-12), (5, 0.0), (300, 1e-12)):
        il = nbgen.permutation(731, n)[:ni].astype(np.int32)
        il[:5] = [40, 1100, 1105, 2400, 2900]
        ref = oracle.force(mm, xp, vp, il, eps2, flags)
        self_idx = np.where((il >= lo) & (il < hi), il - lo, -1).astype(np.int32)
        with nbmod.Context(hi - lo, ni) as ctx:
            ctx.set_j(m[lo:hi], x[:, lo:hi], v[:, lo:hi], a[:, lo:hi], j[:, lo:hi], tj[lo:hi])
            fl = np.flatnonzero(flags[lo:hi]).astype(np.int32)
            ctx.set_flags(fl, np.ones(len(fl), np.uint8))
            ctx.predict(t)
            got = [q.cpu().numpy() for q in ctx.force_ext_ids(xp[:, il], vp[:, il], self_idx, flags[il], eps2)]
            ctx.sync()
        print("ids ni=%d eps2=%g" % (ni, eps2), check_parity(got, ref))
    soft = oracle.force(mm, xp, vp, il, 2.0 ** -14)
    hard = oracle.force(mm, xp, vp, il, 2.0 ** -14, flags)
    assert rel_err_vec(soft[0][:, [0]], hard[0][:, [0]]).max() > 0.5       # the flags matter here


def test_j_sharded_path_on_one_gpu(nbmod):
    """sharding.force_j_sharded with the real kernel behind it (world size 1 over NCCL): by-value
    partial forces with member indices and flags reproduce the by-index force call."""
    import socket
    import torch.distributed as dist
    from paper_1409_5474_b200 import sharding
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % port, rank=0, world_size=1)
    try:
        n, ni, t, eps2 = 5000, 700, 0.3, 2.0 ** -14
        m, x, v, a, j, tj = _j_set(n, 720)
        flags = np.zeros(n, np.uint8)
        flags[[7, 4000]] = 1
        il = nbgen.permutation(721, n)[:ni].astype(np.int32)
        il[:2] = [7, 4000]
        xp, vp = oracle.predict(t, x, v, a, j, tj)
        ref = oracle.force(m, xp, vp, il, eps2, flags)
        with nbmod.Context(n, ni) as ctx:
            ctx.set_j(m, x, v, a, j, tj)
            ctx.set_flags(np.array([7, 4000], np.int32), np.ones(2, np.uint8))
            ctx.predict(t)
            px, pv = ctx.predicted()
            pos = sharding.owned(il, 0, n).to(ctx.device)
            idx = torch.from_numpy(il.astype(np.int64)).to(ctx.device)
            fl = torch.from_numpy(flags.astype(np.float64)).to(ctx.device)
            state = torch.cat([px[:, idx], pv[:, idx], fl[None, idx], idx[None].to(torch.float64)], 0)
            got = sharding.force_j_sharded(lambda xi, vi, si, fi: ctx.force_ext_ids(xi, vi, si, fi, eps2),
                                           state, pos, ni, 0, n)
            got = [q.cpu().numpy() for q in got]
            ctx.sync()
        check_parity(got, ref)
    finally:
        dist.destroy_process_group()


def test_bench_shard_j_runs_on_one_gpu():
    """bench.py --shard j (the arm a multi-GPU scaling run of the paper's scheme would use) on one GPU:
    world size 1 goes through the same all_gather / nb_force_ext_ids / all_reduce path."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--shard", "j", "--workload", "small",
                          "--steps", "2", "--warmup", "3"], capture_output=True, text=True, timeout=600, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["n_gpus"] == 1 and line["value"] > 1e10
    assert "j-sharded" in line["config"]["parallelism"]
