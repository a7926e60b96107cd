"""nb_force_static (include/nb.h, csrc/static_force.cu): the force call that allocates nothing -- no
context, scratch memory in a static device array of the library.  Collected last on purpose (zz): the
suite runs with pytest -x.

-m gpu: its output against the existing by-value / by-index paths (the mixed-precision default within
the north_star tolerances, the IEEE-double mode to rounding) and against the oracle, on calls issued back
to back on one stream (the second must not see the first's tickets or partial sums), with sizes that
change from call to call; that the calls leave the device's free memory where it was; the call captured
into a CUDA graph and replayed.
not gpu: the size limits are refused before any device work."""
import numpy as np
import pytest

import nbgen
import oracle
from util import TOL_ACC, TOL_JRK, TOL_POT, check_parity, rel_err_scalar, rel_err_vec

torch = pytest.importorskip("torch")

TOL64 = 1.0e-12


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _j_set(n, seed):
    m, x, v = nbgen.plummer(n, seed)
    m = m * (0.5 + nbgen.Streams(seed + 1, n).uniform())
    return m, np.ascontiguousarray(x), np.ascontiguousarray(v)


def _close(got, want, ta, tj, tp):
    assert rel_err_vec(got[0], want[0]).max() <= ta
    assert rel_err_vec(got[1], want[1]).max() <= tj
    assert rel_err_scalar(got[2], want[2]).max() <= tp


class _Call:
    """Inputs and outputs of one nb_force_static call, all allocated BEFORE the calls are issued."""

    def __init__(self, nbm, dev, jset, xi, vi, self_idx, eps2):
        self.nb = nbm.binding
        self.n = jset[0].shape[0]
        self.m, self.x, self.v = jset
        self.ni = xi.shape[1]
        self.xi = torch.as_tensor(np.ascontiguousarray(xi)).to(dev)
        self.vi = torch.as_tensor(np.ascontiguousarray(vi)).to(dev)
        self.self_idx = None if self_idx is None else torch.as_tensor(self_idx.astype(np.int32)).to(dev)
        self.eps2 = eps2
        self.acc = torch.full((3, self.ni), float("nan"), dtype=torch.float64, device=dev)
        self.jrk = torch.full((3, self.ni), float("nan"), dtype=torch.float64, device=dev)
        self.pot = torch.full((self.ni,), float("nan"), dtype=torch.float64, device=dev)

    def issue(self, stream=None):
        s = torch.cuda.current_stream().cuda_stream if stream is None else stream
        self.nb.nb_force_static(s, self.n, self.m, self.x, self.v, self.ni, self.xi, self.vi, self.self_idx,
                                self.eps2, self.acc, self.jrk, self.pot)

    def result(self):
        return [q.cpu().numpy() for q in (self.acc, self.jrk, self.pot)]


@pytest.mark.gpu
def test_static_force_matches_the_context_paths_on_calls_in_a_row(nbmod):
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    n, eps2 = 6000 + 37, 2.0 ** -14                             # 48 j-tiles, the last one ragged
    m, x, v = _j_set(n, 4100)
    x[:, 5], v[:, 5] = x[:, 6], v[:, 6]                         # two distinct particles at one place (R6)
    zero = np.zeros((3, n))
    jset = tuple(torch.as_tensor(q).to(dev) for q in (m, x, v))

    # members of the j-set (own pair skipped by index) and particles from outside it, several sizes: one
    # i-tile, several, two per thread (ni > 1024); a one-particle call last
    cases = []
    for ni, kind in ((300, "members"), (5, "members"), (1500, "members"), (333, "outside"), (1, "members"),
                     (2500, "outside")):
        if kind == "members":
            il = nbgen.permutation(4200 + ni, n)[:ni].astype(np.int32)
            il[0] = 5 if ni > 1 else 6
            cases.append((kind, il, x[:, il], v[:, il], il))
        else:
            _, xo, vo = nbgen.plummer(ni, 4300 + ni)
            cases.append((kind, None, np.ascontiguousarray(xo + 0.3), np.ascontiguousarray(vo), None))

    with nbmod.Context(n, 4096) as ctx:
        # the existing paths, on the same particles: t = t_j = 0, so the predicted state IS (x, v)
        want = {}
        for mode in (0, 1):
            ctx.precision(mode)
            ctx.set_j(m, x, v, zero, zero, np.zeros(n))
            ctx.predict(0.0)
            for c, (kind, il, xi, vi, _) in enumerate(cases):
                if kind == "outside":
                    out = ctx.force_ext(xi, vi, eps2)
                elif mode == 0:
                    out = ctx.force_ext_ids(xi, vi, il, None, eps2)
                else:
                    out = ctx.force(il, eps2)
                want[mode, c] = [q.cpu().numpy() for q in out]
        ctx.sync()

        calls = [_Call(nbmod, dev, jset, xi, vi, sidx, eps2) for (_, _, xi, vi, sidx) in cases]
        for call in calls:                                      # first use on this device: set-up, and both
            call.issue()                                        # kernel variants loaded
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info(dev)[0]
        for _ in range(2):                                      # every call twice, all back to back, no sync
            for call in calls:
                call.issue()
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info(dev)[0] >= free0         # nothing was allocated

    for c, (call, (kind, il, xi, vi, _)) in enumerate(zip(calls, cases)):
        got = call.result()
        assert all(np.isfinite(g).all() for g in got)
        _close(got, want[0, c], TOL_ACC, TOL_JRK, TOL_POT)      # the mixed-precision default path
        _close(got, want[1, c], TOL64, TOL64, TOL64)            # the IEEE-double path
        if kind == "members":
            ref = oracle.force(m, x, v, il, eps2)
        else:
            ni = xi.shape[1]
            ref = oracle.force(np.concatenate([m, np.zeros(ni)]), np.concatenate([x, xi], 1),
                               np.concatenate([v, vi], 1), np.arange(n, n + ni, dtype=np.int32), eps2)
        check_parity(got, ref)
        _close(got, ref, TOL64, TOL64, TOL64)

    # the same call again gives the same bits (fixed summation order), whatever ran in between
    before = calls[2].result()
    calls[4].issue()
    calls[2].issue()
    torch.cuda.synchronize()
    assert all(np.array_equal(p, q) for p, q in zip(before, calls[2].result()))


@pytest.mark.gpu
def test_static_force_degenerate_sizes_and_no_jerk(nbmod):
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    nb = nbmod.binding
    n = 130
    m, x, v = _j_set(n, 4400)
    jset = tuple(torch.as_tensor(q).to(dev) for q in (m, x, v))
    il = np.arange(0, n, 7, dtype=np.int32)
    s = torch.cuda.current_stream().cuda_stream
    # eps2 = 0, jrk = NULL
    call = _Call(nbmod, dev, jset, x[:, il], v[:, il], il, 0.0)
    nb.nb_force_static(s, n, *jset, call.ni, call.xi, call.vi, call.self_idx, 0.0, call.acc, None, call.pot)
    torch.cuda.synchronize()
    ref = oracle.force(m, x, v, il, 0.0)
    assert rel_err_vec(call.acc.cpu().numpy(), ref[0]).max() <= TOL64
    assert rel_err_scalar(call.pot.cpu().numpy(), ref[2]).max() <= TOL64
    assert torch.isnan(call.jrk).all()                          # untouched
    # n = 0: zeros; ni = 0: nothing happens
    call = _Call(nbmod, dev, jset, x[:, il], v[:, il], None, 1e-4)
    nb.nb_force_static(s, 0, None, None, None, call.ni, call.xi, call.vi, None, 1e-4, call.acc, call.jrk, call.pot)
    nb.nb_force_static(s, n, *jset, 0, None, None, None, 1e-4, None, None, None)
    torch.cuda.synchronize()
    assert all((g == 0).all() for g in call.result())
    # one particle alone feels nothing
    one = tuple(q[..., :1].contiguous() for q in jset)
    call = _Call(nbmod, dev, one, x[:, :1], v[:, :1], np.zeros(1, np.int32), 1e-4)
    call.issue()
    torch.cuda.synchronize()
    assert all((g == 0).all() for g in call.result())


@pytest.mark.gpu
def test_static_force_under_stream_capture(nbmod):
    """What the entry point is for: the call recorded into a CUDA graph (where cudaMalloc is not allowed)
    and replayed on new inputs in the same buffers."""
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    n, ni, eps2 = 2000, 200, 2.0 ** -12
    m, x, v = _j_set(n, 4500)
    jset = tuple(torch.as_tensor(q).to(dev) for q in (m, x, v))
    il = nbgen.permutation(4501, n)[:ni].astype(np.int32)
    call = _Call(nbmod, dev, jset, x[:, il], v[:, il], il, eps2)
    call.issue()                                                # set-up happens outside the capture
    torch.cuda.synchronize()
    first = call.result()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        call.issue()                                            # torch's capture stream is current here
    il2 = nbgen.permutation(4502, n)[:ni].astype(np.int32)
    call.xi.copy_(torch.as_tensor(np.ascontiguousarray(x[:, il2])))
    call.vi.copy_(torch.as_tensor(np.ascontiguousarray(v[:, il2])))
    call.self_idx.copy_(torch.as_tensor(il2))
    for _ in range(2):
        graph.replay()
    torch.cuda.synchronize()
    got = call.result()
    _close(got, oracle.force(m, x, v, il2, eps2), TOL64, TOL64, TOL64)
    _close(first, oracle.force(m, x, v, il, eps2), TOL64, TOL64, TOL64)


def test_static_force_refuses_sizes_beyond_its_limits(nbmod):
    """Before any device work (this runs without a GPU too): NB_ERR_ARG, "invalid argument"."""
    nb = nbmod.binding
    assert nb.NB_STATIC_NI_MAX == 4096 and nb.NB_STATIC_SCRATCH_BYTES == 4 << 20
    dummy = 256                                                 # never dereferenced: the sizes are checked first
    for n, ni in ((100, nb.NB_STATIC_NI_MAX + 1), (1 << 31, 4), (-1, 4), (100, -1)):
        with pytest.raises(nb.NBError) as e:
            nb.nb_force_static(None, n, dummy, dummy, dummy, ni, dummy, dummy, None, 1e-4, dummy, dummy, dummy)
        assert e.value.status == nb.NB_ERR_ARG and "invalid argument" in str(e.value)
    for eps2 in (-1.0, float("nan")):
        with pytest.raises(nb.NBError) as e:
            nb.nb_force_static(None, 100, dummy, dummy, dummy, 4, dummy, dummy, None, eps2, dummy, dummy, dummy)
        assert e.value.status == nb.NB_ERR_ARG
    with pytest.raises(nb.NBError) as e:                       # a required pointer is NULL
        nb.nb_force_static(None, 100, dummy, dummy, dummy, 4, None, dummy, None, 1e-4, dummy, dummy, dummy)
    assert e.value.status == nb.NB_ERR_ARG
