"""Pins of the oracle's RNG (R1, R2) and model (Eq. 1) -- CPU only."""
import math
import os

import numpy as np
import pytest
from scipy import stats

from oracle import oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = O.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_counter_sensitivity():
    base = O.philox([1, 2, 3, 4], [5, 6])
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] += 1
        assert not np.array_equal(O.philox(c, [5, 6]), base)
    assert not np.array_equal(O.philox([1, 2, 3, 4], [6, 6]), base)
    assert not np.array_equal(O.philox([1, 2, 3, 4], [5, 7]), base)


def test_stream_layout_R1():
    # seed -> key = (lo32, hi32); counter = (q, slot, t, tag)
    seed = (0xDEADBEEF << 32) | 0x01234567
    w = O.philox([0, 7, 11, O.TAG_ACC], [0x01234567, 0xDEADBEEF])
    assert O.word0(seed, O.TAG_ACC, 11, 7) == int(w[0])
    assert O.uniform(seed, O.TAG_ACC, 11, 7) == ((int(w[0]) >> 8) + 1) / 2.0 ** 24
    # quad q=2 of a V=12 draw: Box-Muller of words (0,1) and (2,3)
    z = O.normals(seed, O.TAG_PROP, 11, 7, 12)
    w = [int(x) for x in O.philox([2, 7, 11, O.TAG_PROP], [0x01234567, 0xDEADBEEF])]
    for j, (a, b) in enumerate([(w[0], w[1]), (w[2], w[3])]):
        r = math.sqrt(-2.0 * math.log(((a >> 8) + 1) / 2.0 ** 24))
        th = 2.0 * math.pi * (b >> 8) / 2.0 ** 24
        assert z[8 + 2 * j] == pytest.approx(r * math.cos(th), abs=1e-14)
        assert z[9 + 2 * j] == pytest.approx(r * math.sin(th), abs=1e-14)


def test_ragged_quad_is_truncation():
    z8 = O.normals(3, O.TAG_INIT, 0, 5, 8)
    for V in (1, 2, 3, 5, 7):
        assert np.array_equal(O.normals(3, O.TAG_INIT, 0, 5, V), z8[:V])


def test_normals_are_standard_normal():
    z = np.concatenate([O.normals(42, O.TAG_PROP, t, i, 400) for t in range(5) for i in range(50)])
    n = z.size
    assert abs(z.mean()) < 4.0 / math.sqrt(n)
    assert abs(z.var() - 1.0) < 4.0 * math.sqrt(2.0 / n)
    assert abs(stats.skew(z)) < 4.0 * math.sqrt(6.0 / n)
    assert abs(stats.kurtosis(z)) < 4.0 * math.sqrt(24.0 / n)
    assert stats.kstest(z, "norm").pvalue > 1e-3
    assert np.abs(z).max() <= math.sqrt(2 * 24 * math.log(2)) + 1e-12   # R2: |z| <= 5.77
    # adjacent sites (cos/sin partners and different word pairs) are uncorrelated
    zz = z.reshape(-1, 4)
    c = np.corrcoef(zz.T)
    assert np.abs(c - np.eye(4)).max() < 4.0 / math.sqrt(zz.shape[0])


def test_uniform_range_and_mean():
    u = np.array([O.uniform(9, O.TAG_ACC, t, i) for t in range(40) for i in range(500)])
    assert u.min() > 0.0 and u.max() <= 1.0
    assert abs(u.mean() - 0.5) < 4.0 / math.sqrt(12 * u.size)
    assert np.all(u * 2 ** 24 == np.round(u * 2 ** 24))


def test_init_particles_layout():
    phi = O.init_particles(5, 7, 10)
    for i in range(7):
        assert np.array_equal(phi[:, i], O.normals(5, O.TAG_INIT, 0, i, 10))


# ---------------------------------------------------------------- Eq. 1 ----
def _rand_field(L, seed=0, scale=1.0):
    return np.random.default_rng(seed).normal(size=(L, L)) * scale


@pytest.mark.parametrize("L", [1, 2, 3, 4, 10])
def test_z2_and_translation_invariance(L):
    f = _rand_field(L, L)
    s = O.action_field(f, L, -4.0, 1.0)
    assert O.action_field(-f, L, -4.0, 1.0) == pytest.approx(s, rel=1e-14)
    assert O.u0_field(-f) == O.u0_field(f)
    for sh in [(1, 0), (0, 1), (2, 3)]:
        g = np.roll(f, sh, axis=(0, 1))
        assert O.action_field(g, L, -4.0, 1.0) == pytest.approx(s, rel=1e-12, abs=1e-12)
    # the two lattice directions are equivalent
    assert O.action_field(f.T.copy(), L, -4.0, 1.0) == pytest.approx(s, rel=1e-12, abs=1e-12)


@pytest.mark.parametrize("L", [1, 2, 4, 7])
def test_constant_field(L):
    c, m0sq, lam = 0.7, -4.0, 1.3
    f = np.full((L, L), c)
    V = L * L
    s, a = O.action_field(f, L, m0sq, lam, with_abs=True)
    assert s == pytest.approx(V * (0.5 * m0sq * c * c + lam * c ** 4), rel=1e-13)
    assert a == pytest.approx(V * (0.5 * abs(m0sq) * c * c + lam * c ** 4), rel=1e-13)
    assert O.u0_field(f) == pytest.approx(0.5 * V * c * c, rel=1e-14)


@pytest.mark.parametrize("L", [2, 3, 4, 10])
def test_plane_wave_eigenvalues(L):
    """lambda = 0: S = 1/2 (m0^2 + khat^2) |phi|^2 on a lattice plane wave, khat^2 =
    sum_mu 4 sin^2(pi k_mu / L); at L = 2 this pins the doubled periodic bond (A2)."""
    m0sq = 0.5
    r, c = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    for k1 in range(L):
        for k2 in range(L):
            f = np.cos(2 * np.pi * (k1 * r + k2 * c) / L) + 0.3 * np.sin(2 * np.pi * (k1 * r + k2 * c) / L)
            kh = 4 * np.sin(np.pi * k1 / L) ** 2 + 4 * np.sin(np.pi * k2 / L) ** 2
            want = 0.5 * (m0sq + kh) * np.sum(f * f)
            assert O.action_field(f, L, m0sq, 0.0) == pytest.approx(want, rel=1e-12, abs=1e-12)


def test_direction_weights_are_separately_half():
    """A field varying along one axis only: S = L * (1-D chain action); catches a dropped or
    doubled direction."""
    L = 5
    g = np.random.default_rng(1).normal(size=L)
    chain = sum(0.5 * (g[(i + 1) % L] - g[i]) ** 2 for i in range(L))
    pot = sum(0.5 * -4.0 * x * x + 1.0 * x ** 4 for x in g)
    rows = np.tile(g, (L, 1))           # varies with column c
    cols = rows.T.copy()                # varies with row r
    for f in (rows, cols):
        assert O.action_field(f, L, -4.0, 1.0) == pytest.approx(L * (chain + pot), rel=1e-13)


@pytest.mark.parametrize("L", [1, 2, 3, 6])
def test_gradient_matches_finite_differences(L):
    m0sq, lam = -4.0, 1.0
    f = _rand_field(L, 10 + L)
    g = O.action_grad_field(f, L, m0sq, lam).reshape(L, L)
    h = 1e-5
    for r in range(L):
        for c in range(L):
            fp, fm = f.copy(), f.copy()
            fp[r, c] += h
            fm[r, c] -= h
            fd = (O.action_field(fp, L, m0sq, lam) - O.action_field(fm, L, m0sq, lam)) / (2 * h)
            assert g[r, c] == pytest.approx(fd, rel=1e-6, abs=1e-7)
    # first-order change for a small random displacement
    d = _rand_field(L, 99) * 1e-6
    ds = O.action_field(f + d, L, m0sq, lam) - O.action_field(f, L, m0sq, lam)
    assert ds == pytest.approx(np.sum(g * d), rel=1e-4, abs=1e-12)


def test_action_batch_layout():
    L, N = 4, 9
    rng = np.random.default_rng(3)
    phi = rng.normal(size=(L * L, N))
    S, U0, A = O.action_batch(phi, L, -4.0, 1.0, with_abs=True)
    for i in range(N):
        s, a = O.action_field(phi[:, i].copy(), L, -4.0, 1.0, with_abs=True)
        assert S[i] == s and A[i] == a
        assert U0[i] == pytest.approx(0.5 * np.sum(phi[:, i] ** 2), rel=1e-15)
    assert np.all(A >= np.abs(S))
