"""Pins of the oracle's population step (P1-P4, C1, C2; readings R3, R5, R6, A4) -- CPU only."""
import math
from fractions import Fraction

import numpy as np
import pytest
from scipy.optimize import brentq
from scipy.special import logsumexp

from oracle import oracle as O


def gauss_a(L, m0sq):
    k = np.arange(L)
    kh = 4 * np.sin(np.pi * k / L) ** 2
    return (m0sq + kh[:, None] + kh[None, :]).reshape(-1)


# ------------------------------------------------------------------ P1/P2 ---
def test_ess_invariants():
    S = np.random.default_rng(0).normal(size=1000) * 3
    assert O.ess_frac(S, 0.0) == pytest.approx(1.0, rel=1e-14)
    prev = 1.0
    for d in [0.01, 0.1, 0.5, 1.0, 5.0, 50.0]:
        e = O.ess_frac(S, d)
        assert 1.0 / S.size - 1e-15 <= e <= prev + 1e-15
        prev = e
    assert O.ess_frac(S, 1e4) == pytest.approx(1.0 / S.size, rel=1e-6)
    assert O.ess_frac(np.full(10, 2.5), 3.0) == pytest.approx(1.0, rel=1e-14)
    # shift invariance of the weights
    assert O.ess_frac(S + 123.0, 0.7) == pytest.approx(O.ess_frac(S, 0.7), rel=1e-11)


def test_ess_two_point_closed_form():
    # N/2 particles at S=0, N/2 at S=c: ESS/N = (1+e)^2 / (2 (1+e^2)), e = exp(-delta c)
    S = np.array([0.0, 2.0] * 8)
    for d in (0.1, 0.9):
        e = math.exp(-d * 2.0)
        assert O.ess_frac(S, d) == pytest.approx((1 + e) ** 2 / (2 * (1 + e * e)), rel=1e-14)


def test_reweight_matches_library_logsumexp():
    rng = np.random.default_rng(1)
    S = rng.normal(size=5000) * 10 - 30
    w, dlz = O.reweight(S, 0.37)
    assert dlz == pytest.approx(logsumexp(-0.37 * S) - math.log(S.size), rel=1e-13)
    assert w.dtype == np.float32 and w.max() == np.float32(1.0)
    assert np.argmax(w) == np.argmin(S)
    ref = np.exp(-0.37 * (S - S.min()))
    assert np.allclose(w, ref, rtol=1e-6, atol=0)
    assert O.lib().orc_lse_neg(S, S.size, 0.37) == pytest.approx(logsumexp(-0.37 * S), rel=1e-13)


def test_next_delta_is_the_root_and_final_rule():
    rng = np.random.default_rng(2)
    S = rng.normal(size=4000) * 5
    d, fin = O.next_delta(S, 0.2, 0.5)
    assert not fin and 0 < d < 0.8
    assert O.ess_frac(S, d) == pytest.approx(0.5, abs=1e-9)
    root = brentq(lambda x: O.ess_frac(S, x) - 0.5, 1e-12, 0.8, xtol=1e-15, rtol=1e-14)
    assert d == pytest.approx(root, rel=1e-9)
    # final step: whole remaining interval is affordable
    d, fin = O.next_delta(S * 1e-3, 0.25, 0.5)
    assert fin and d == 0.75


def test_bisection_gaussian_schedule_closed_form():
    """lambda=0: large-N ESS/N = prod_k sqrt(1+2 d c_k)/(1+d c_k), c_k = a_k/(1+beta a_k).
    L=4, m0^2=1, target 0.5: first delta from beta=0 on N(0,I) particles."""
    a = gauss_a(4, 1.0)

    def f(d, beta):
        c = a / (1 + beta * a)
        return np.prod(np.sqrt(1 + 2 * d * c) / (1 + d * c)) - 0.5

    want = brentq(lambda d: f(d, 0.0), 1e-9, 1.0)
    assert want == pytest.approx(0.078920, abs=2e-6)          # SURVEY 8(c) closed-form schedule
    phi = O.init_particles(11, 200000, 16)
    S, _ = O.action_batch(phi, 4, 1.0, 0.0)
    d, fin = O.next_delta(S, 0.0, 0.5)
    assert not fin
    assert d == pytest.approx(want, rel=0.03)
    # E[S_E] at beta=0 is 1/2 sum a_k = 40
    assert S.mean() == pytest.approx(0.5 * a.sum(), rel=0.01)


# --------------------------------------------------------------------- P3 ---
def textbook_systematic(q, U):
    """Textbook systematic resampling in exact rational arithmetic on integer masses q:
    position p_j = (j + U/2^32)/N; ancestor = first i whose normalised CDF strictly exceeds p_j."""
    N = len(q)
    T = sum(q)
    cdf, run = [], 0
    for x in q:
        run += x
        cdf.append(Fraction(run, T))
    anc = []
    for j in range(N):
        p = (Fraction(j) + Fraction(U, 2 ** 32)) / N
        i = 0
        while i < N - 1 and cdf[i] <= p:
            i += 1
        anc.append(i)
    return anc


@pytest.mark.parametrize("N", [1, 2, 3, 5, 8, 13])
def test_resampling_brute_force(N):
    rng = np.random.default_rng(N)
    for trial in range(30):
        w = rng.random(N).astype(np.float32) ** (1 + trial % 4)
        if trial % 5 == 0 and N > 2:
            w[rng.integers(N)] = 0.0
        w /= w.max()
        q = [int(math.floor(float(x) * 2 ** 40)) for x in w]
        Us = [0, 1, 2 ** 31, 2 ** 32 - 1] + [int(u) for u in rng.integers(0, 2 ** 32, 6)]
        for U in Us:
            assert list(O.resample_systematic(w, U)) == textbook_systematic(q, U)


def test_resampling_invariants():
    rng = np.random.default_rng(7)
    N = 5000                                                 # not a power of two
    w = np.exp(-rng.normal(size=N) * 2).astype(np.float32)
    w /= w.max()
    q = np.floor(w.astype(np.float64) * 2 ** 40)
    for U in (0, 12345, 2 ** 32 - 1):
        a = O.resample_systematic(w, U)
        assert np.all(np.diff(a) >= 0) and a.min() >= 0 and a.max() < N
        counts = np.bincount(a, minlength=N)
        assert counts.sum() == N
        expect = N * q / q.sum()
        assert np.all(counts >= np.floor(expect) - 1e-9) and np.all(counts <= np.ceil(expect) + 1e-9)
    for U in (0, 999, 2 ** 32 - 1):
        assert np.array_equal(O.resample_systematic(np.ones(64, np.float32), U), np.arange(64))
    one = np.zeros(10, np.float32)
    one[3] = 1.0
    assert np.all(O.resample_systematic(one, 777) == 3)
    with pytest.raises(ValueError):
        O.resample_systematic(np.zeros(4, np.float32), 1)


def test_gather():
    rng = np.random.default_rng(8)
    a = rng.normal(size=(6, 11))
    anc = np.sort(rng.integers(0, 11, 11)).astype(np.int32)
    assert np.array_equal(O.gather(a, anc), a[:, anc])
    assert np.array_equal(O.gather(a[0].copy(), anc), a[0, anc])


# ------------------------------------------------------------------ C1/C2 ---
def test_covariance_and_cholesky_match_library():
    rng = np.random.default_rng(9)
    V, N = 12, 400
    mix = rng.normal(size=(V, V))
    phi = mix @ rng.normal(size=(V, N)) + rng.normal(size=(V, 1)) * 5
    mu, Sig = O.covariance(phi)
    assert np.allclose(mu, phi.mean(axis=1), rtol=1e-13)
    assert np.allclose(Sig, np.cov(phi), rtol=1e-11, atol=1e-12)          # 1/(N-1), centred
    Lc, st = O.cholesky(Sig)
    assert st == 0
    assert np.allclose(Lc, np.linalg.cholesky(Sig), rtol=1e-10, atol=1e-12)
    assert np.all(np.triu(Lc, 1) == 0) and np.all(np.diag(Lc) > 0)
    Sig2, Lc2, st2 = O.cov_chol(phi)
    assert st2 == 0 and np.array_equal(Sig2, Sig) and np.array_equal(Lc2, Lc)


def test_cholesky_jitter_and_failure():
    # rank-deficient: N < V particles -> pivot <= 0 -> jitter eps = 1e-6 tr/V once (A4)
    rng = np.random.default_rng(10)
    V = 6
    x = rng.normal(size=(V, 1))
    Sig = x @ x.T
    Lc, st = O.cholesky(Sig)
    assert st == 1
    eps = 1e-6 * np.trace(Sig) / V
    assert np.allclose(Lc @ Lc.T, Sig + eps * np.eye(V), rtol=1e-9, atol=1e-12)
    _, st = O.cholesky(-np.eye(3))
    assert st == -1


def test_covariance_of_gaussian_field_is_circulant():
    """Gaussian case at beta: exact Sigma = F diag(1/(1+beta a_k)) F^T; at beta=0 it is I."""
    phi = O.init_particles(3, 100000, 16)
    _, Sig = O.covariance(phi)
    assert np.abs(Sig - np.eye(16)).max() < 5.0 / math.sqrt(100000)
