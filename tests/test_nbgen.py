"""The seeded generators: determinism, order independence, and the shapes the configs promise."""
import numpy as np

import nbgen


def test_streams_are_order_independent():
    a = nbgen.Streams(42, 100)
    b = nbgen.Streams(42, 40, first=60)
    ua = [a.uniform() for _ in range(3)]
    ub = [b.uniform() for _ in range(3)]
    for p, q in zip(ua, ub):
        assert (p[60:] == q).all()
        assert (p >= 0).all() and (p < 1).all()
    # selective advance touches only the selected streams
    c = nbgen.Streams(42, 100)
    c.uniform(np.array([3, 5]))
    u = c.uniform()
    assert u[3] == ua[1][3] and u[4] == ua[0][4]


def test_splitmix64_reference_value():
    # splitmix64 from state 0: first outputs of the published algorithm
    s = nbgen.Streams.__new__(nbgen.Streams)
    s.state = np.zeros(1, np.uint64)
    assert int(s.bits()[0]) == 0xE220A8397B1DCDAF
    assert int(s.bits()[0]) == 0x6E789E6AA1B965F4


def test_permutation_and_integers():
    p = nbgen.permutation(7, 1000)
    assert sorted(p.tolist()) == list(range(1000)) and p.dtype == np.int32
    assert (nbgen.permutation(7, 1000) == p).all() and (nbgen.permutation(8, 1000) != p).any()
    k = nbgen.integers(3, 5000, 4, 12)
    assert k.min() == 4 and k.max() == 12 and len(np.unique(k)) == 9


def test_plummer_is_centred_and_reproducible():
    m, x, v = nbgen.plummer(4096, 5)
    m2, x2, v2 = nbgen.plummer(4096, 5)
    assert (x == x2).all() and (v == v2).all()
    assert abs(x @ m).max() < 1e-15 and abs(v @ m).max() < 1e-15
    r = np.sqrt((x * x).sum(0))
    assert r.max() < 39 * nbgen.HENON_A
    assert abs(np.median(r) - 0.7686) < 0.03            # half-mass radius of the Henon-unit model
    # every star is bound in the smooth potential: v < v_esc (before the tiny recentring shift)
    vesc2 = 2.0 / np.sqrt(r * r + nbgen.HENON_A ** 2)
    assert ((v * v).sum(0) < vesc2 * 1.001).all()


def test_config_shapes_small():
    c3 = nbgen.config3(n=4096, sizes=(1, 1024, 4096))
    assert [len(i) for i in c3.i_lists] == [1, 1024, 4096]
    assert (c3.i_lists[1] == c3.i_lists[2][:1024]).all()
    assert ((c3.t <= c3.t_now) & (c3.t_now - c3.t < 2.0 ** -4)).all() and len(np.unique(c3.t)) > 4
    c4 = nbgen.config4(n_gal=512)
    assert c4.n == 1026 and np.flatnonzero(c4.flags).tolist() == [512, 1025]
    assert c4.m[512] == 1e-3 and c4.m[1025] == 1e-3
    # the two black holes are on a parabola for point masses of (galaxy + BH) each: E = 0, q = 1
    dx, dv = c4.x[:, 1025] - c4.x[:, 512], c4.v[:, 1025] - c4.v[:, 512]
    mt = 2 * 0.501
    assert abs(0.5 * dv @ dv - mt / np.sqrt(dx @ dx)) < 1e-12
    lz = dx[0] * dv[1] - dx[1] * dv[0]
    assert abs(lz * lz / (2 * mt) - 1.0) < 1e-12
    c5 = nbgen.config5(n_stars=1 << 14, n_active=1 << 10)
    assert c5.n == (1 << 14) + 11 and len(c5.i_lists[0]) == 1024 and not c5.flags.any()
    assert abs(c5.m.sum() - 1.01) < 1e-12
    assert np.sqrt((c5.x ** 2).sum(0)).max() < 20 + 39


def test_config_full_sizes():
    assert nbgen.config1().n == 1024 and nbgen.config2().n == 65536
    c4 = nbgen.config4()
    assert c4.n == (1 << 20) + 2
    dv = c4.v[:, -1] - c4.v[:, 1 << 19]
    np.testing.assert_allclose(dv, [-0.4246881208604733, 0.1415627069534911, 0.0], rtol=1e-14)
