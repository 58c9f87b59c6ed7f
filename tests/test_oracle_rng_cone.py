"""Pins P-1 .. P-3 for the oracle: Philox4x32-10, the (0,1) uniforms and the cone trial move.

None of these tests needs a GPU.  Each pin is chosen so that a plausible mistake (wrong round constant,
swapped counter words, 24-bit instead of 23-bit mantissa, full-angle instead of half-angle cone, uniform in
polar angle instead of solid angle, a non-orthogonal frame) fails it.
"""
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _kat_rows():
    rows = []
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_p1_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, want in rows:
        got = oracle.philox4x32_10(ctr, key)
        assert [int(g) for g in got] == want


def test_p1_philox_is_a_bijection_on_counters_and_sensitive_to_every_word():
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    seen = {tuple(int(v) for v in base)}
    for w in range(4):
        c = [1, 2, 3, 4]; c[w] ^= 1
        out = tuple(int(v) for v in oracle.philox4x32_10(c, [5, 6]))
        assert out not in seen; seen.add(out)
    for w in range(2):
        k = [5, 6]; k[w] ^= 1
        out = tuple(int(v) for v in oracle.philox4x32_10([1, 2, 3, 4], k))
        assert out not in seen; seen.add(out)


def test_p2_uniforms_open_interval_and_exact_in_fp32():
    rs = [0, 1, 0x1FF, 0x200, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF, 0xFFFFFE00, 0xDEADBEEF]
    rng = np.random.default_rng(0)
    rs += [int(v) for v in rng.integers(0, 2**32, size=2000, dtype=np.uint64)]
    for r in rs:
        u = oracle.uniform(r)
        assert 0.0 < u < 1.0
        assert u == ((r >> 9) + 0.5) / 2**23            # the definition (reading C-8)
        assert float(np.float32(u)) == u                 # bit-identical after the fp32 round trip
    assert oracle.uniform(0) == 2.0**-24 and oracle.uniform(0xFFFFFFFF) == 1.0 - 2.0**-24
    # a 24-bit variant ((r>>8)+0.5)*2^-24 would NOT survive the round trip: make sure the pin can tell
    bad = ((0xFFFFFFFF >> 8) + 0.5) / 2**24
    assert float(np.float32(bad)) != bad


def test_p2_uniform_moments():
    key = [42, 0]
    us = np.array([oracle.uniform(int(oracle.philox4x32_10([i, 0, 0, 0], key)[k])) for i in range(4000) for k in range(4)])
    n = len(us)
    assert abs(us.mean() - 0.5) < 4 * np.sqrt(1 / 12 / n)
    assert abs(us.var() - 1 / 12) < 4 * np.sqrt(1 / 180 / n)


def test_p2_site_uniforms_use_every_bit_of_their_two_words_once():
    """Reading C-26: u0 <- bits 31..9 of w0, u2 <- bits 31..9 of w1, u1 <- bits 8..0 of w0 then bits 8..0 of w1."""
    rng = np.random.default_rng(1)
    for _ in range(300):
        w0, w1 = (int(v) for v in rng.integers(0, 2**32, size=2, dtype=np.uint64))
        u1 = oracle.uniform_azimuth(w0, w1)
        assert 0.0 <= u1 < 1.0 and float(np.float32(u1)) == u1 and float(np.float32(1.0 + u1)) == 1.0 + u1
        assert u1 == (((w0 & 511) << 9) | (w1 & 511)) / 2**18
        bit = int(rng.integers(0, 32))
        for which in (0, 1):
            v0, v1 = (w0 ^ (1 << bit), w1) if which == 0 else (w0, w1 ^ (1 << bit))
            changed = [oracle.uniform(v0) != oracle.uniform(w0), oracle.uniform_azimuth(v0, v1) != u1, oracle.uniform(v1) != oracle.uniform(w1)]
            expect = [which == 0 and bit >= 9, bit < 9, which == 1 and bit >= 9]
            assert changed == expect
    assert oracle.uniform_azimuth(0, 0) == 0.0 and oracle.uniform_azimuth(0x1FF, 0x1FF) == 1.0 - 2.0**-18


def test_p2_site_uniforms_pair_sharing_and_moments():
    """Sites x and x^2 of a row read the two halves of one block; different rows, colours and sweeps read other blocks;
    all three uniforms of a site are flat and mutually uncorrelated over the lattice."""
    o = oracle.Oracle(16, 8, 8, seed=99)
    key = [99, 0]
    u = {}
    for z in range(8):
        for y in range(8):
            for x in range(16):
                u[(x, y, z)] = o.site_uniforms(x, y, z, (x + y + z) & 1, 7)
    for (x, y, z), got in list(u.items())[::17]:
        first = (x & ~2) + 16 * (y + 8 * z)
        r = [int(v) for v in oracle.philox4x32_10([first, ((x + y + z) & 1) << 8, 7, 0], key)]
        w0, w1 = (r[2], r[3]) if x & 2 else (r[0], r[1])
        assert got == (oracle.uniform(w0), oracle.uniform_azimuth(w0, w1), oracle.uniform(w1))
    assert len({v for v in u.values()}) == len(u)                      # no two sites share their numbers
    assert o.site_uniforms(0, 0, 0, 0, 8) != u[(0, 0, 0)]             # the sweep moves the stream
    a = np.array(list(u.values())); n = len(a)
    for k in range(3):
        assert abs(a[:, k].mean() - 0.5) < 4 * np.sqrt(1 / 12 / n)
        assert abs(a[:, k].var() - 1 / 12) < 5 * np.sqrt(1 / 180 / n)
    c = np.corrcoef(a.T)
    assert np.abs(c - np.eye(3)).max() < 4 / np.sqrt(n)


def test_pair_move_uniforms_share_blocks_like_the_site_uniforms_in_their_own_stream():
    """Constrained pair move (stream tag 1, keyed on the leader): same 64-bit split as C-26, different stream."""
    o = oracle.Oracle(16, 8, 8, seed=99)
    for (x, y, z) in ((0, 0, 0), (2, 0, 0), (5, 3, 2), (7, 3, 2), (14, 7, 7)):
        c = (x + y + z) & 1
        first = (x & ~2) + 16 * (y + 8 * z)
        r = [int(v) for v in oracle.philox4x32_10([first, 1 | (c << 8), 12, 0], [99, 0])]
        w0, w1 = (r[2], r[3]) if x & 2 else (r[0], r[1])
        want = (((w0 >> 9) + 0.5) / 2**23, (((w0 & 511) << 9) | (w1 & 511)) / 2**18, ((w1 >> 9) + 0.5) / 2**23)
        assert o.pair_uniforms(x, y, z, c, 12) == want
        assert o.pair_uniforms(x, y, z, c, 12) != o.site_uniforms(x, y, z, c, 12)


def test_random_start_is_uniform_on_the_sphere_and_seeded():
    o = oracle.Oracle(24, 20, 16, seed=7); o.init_random(); S = o.get_spins()
    n = len(S)
    assert np.abs(np.linalg.norm(S, axis=1) - 1).max() < 1e-15
    assert np.abs(S.mean(axis=0)).max() < 4 * np.sqrt(1 / 3 / n)                       # <S> = 0
    assert np.abs((S ** 2).mean(axis=0) - 1 / 3).max() < 4 * np.sqrt(4 / 45 / n)      # <S_a^2> = 1/3, var = 4/45
    hist, _ = np.histogram(S[:, 2], bins=10, range=(-1, 1))                           # z flat (Archimedes)
    assert np.abs(hist - n / 10).max() < 5 * np.sqrt(n / 10)
    phi = np.arctan2(S[:, 1], S[:, 0]); hist, _ = np.histogram(phi, bins=8, range=(-np.pi, np.pi))
    assert np.abs(hist - n / 8).max() < 5 * np.sqrt(n / 8)
    r = oracle.philox4x32_10([5, 3, 0, 0], [7, 0])                                      # the wiring: site 5, tag 3
    z = 2 * oracle.uniform(int(r[0])) - 1; ph = 2 * np.pi * oracle.uniform(int(r[1]))
    assert np.allclose(S[5], [np.sqrt(1 - z * z) * np.cos(ph), np.sqrt(1 - z * z) * np.sin(ph), z], atol=1e-15)
    o2 = oracle.Oracle(24, 20, 16, seed=7); o2.init_random(); assert (o2.get_spins() == S).all()
    o3 = oracle.Oracle(24, 20, 16, seed=8); o3.init_random(); assert not (o3.get_spins() == S).all()


# ---------------------------------------------------------------------------------------- P-3 cone move
def _spins():
    rng = np.random.default_rng(5)
    v = rng.standard_normal((40, 3)); v /= np.linalg.norm(v, axis=1, keepdims=True)
    special = np.array([[0, 0, 1.0], [0, 0, -1.0], [1.0, 0, 0], [0, 1.0, 0], [0.6, 0.8, 0.0], [1e-9, 0, -1.0]])
    special /= np.linalg.norm(special, axis=1, keepdims=True)
    return np.vstack([v, special])


@pytest.mark.parametrize("theta", [np.pi / 180, 0.5, np.pi / 2, 2.5, np.pi])
def test_p3_cone_unit_norm_inside_cone_and_closed_form_polar_angle(theta):
    rng = np.random.default_rng(11)
    for S in _spins():
        for _ in range(20):
            u0, u1 = rng.random(2)
            Sn = oracle.cone_move(S, theta, u0, u1)
            assert abs(np.linalg.norm(Sn) - 1.0) < 1e-12
            c = float(S @ Sn)
            assert c >= np.cos(theta) - 1e-12                           # theta is the HALF-angle (C-6)
            assert abs(c - (1.0 - u0 * (1.0 - np.cos(theta)))) < 1e-12   # uniform in solid angle (C-7)


def test_p3_cone_azimuth_is_uniform_and_frame_orthonormal():
    # for fixed polar deviation, the displacement d = S' - S integrated over u1 must have no transverse mean,
    # and S' traced over u1 must be a circle of constant radius about S.
    n = 360
    for S in _spins():
        for u0 in (0.1, 0.7):
            pts = np.array([oracle.cone_move(S, 1.0, u0, (k + 0.5) / n) for k in range(n)])
            centre = pts.mean(axis=0)
            c = 1.0 - u0 * (1.0 - np.cos(1.0))
            assert np.allclose(centre, c * S, atol=1e-12)
            r = np.linalg.norm(pts - centre, axis=1)
            assert np.allclose(r, np.sqrt(1 - c * c), atol=1e-12)
            # consecutive points are equally spaced in azimuth (chord lengths equal)
            chord = np.linalg.norm(np.roll(pts, -1, axis=0) - pts, axis=1)
            assert chord.std() < 1e-12


def test_p3_cone_at_pi_is_the_uniform_sphere_draw():
    # stratified (u0,u1) grid = midpoint quadrature of the sphere average: <S'> = 0, <S'_a^2> = 1/3, any S
    n0, n1 = 60, 120
    for S in _spins()[:8]:
        acc1 = np.zeros(3); acc2 = np.zeros(3)
        for i in range(n0):
            for j in range(n1):
                Sn = oracle.cone_move(S, np.pi, (i + 0.5) / n0, (j + 0.5) / n1)
                acc1 += Sn; acc2 += Sn * Sn
        acc1 /= n0 * n1; acc2 /= n0 * n1
        assert np.abs(acc1).max() < 1e-10
        assert np.abs(acc2 - 1 / 3).max() < 2e-4


def test_p3_cone_mean_cosine():
    # E[S.S'] = (1 + cos theta)/2 for a cap that is uniform in solid angle (polar-angle-uniform would give sin(theta)/theta)
    theta = 1.2
    n = 2000
    S = np.array([0.36, -0.48, 0.8])
    vals = [float(S @ oracle.cone_move(S, theta, (i + 0.5) / n, 0.37)) for i in range(n)]
    assert abs(np.mean(vals) - (1 + np.cos(theta)) / 2) < 1e-9
    assert abs(np.mean(vals) - np.sin(theta) / theta) > 1e-2
