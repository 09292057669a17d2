"""Pins of the oracle's slice-sampling inner kernel for nested sampling (NEXT row f3;
PAPER.md:53(iv), :174; reading A16)."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

from oracle import oracle as O


def gauss_a(L, m0sq):
    k = np.arange(L)
    kh = 4 * np.sin(np.pi * k / L) ** 2
    return (m0sq + kh[:, None] + kh[None, :]).reshape(-1)


def test_every_move_obeys_slice_and_constraint_and_replays_from_the_streams():
    L, V, N, k = 3, 9, 400, 4
    rng = np.random.default_rng(0)
    phi = rng.normal(size=(V, N)) * 0.6
    S, U0 = O.action_batch(phi, L, -4.0, 1.0)
    S_star = np.quantile(S, 0.7)
    keep = S < S_star
    phi, S, U0 = phi[:, keep], S[keep], U0[keep]
    N = phi.shape[1]
    _, Sig = O.covariance(phi)
    Lc, _ = O.cholesky(Sig)
    p, S2, U2, t, nexp, nshr, amb = O.slice_walk(phi, S, U0, L, -4.0, 1.0, Lc, S_star, 7, 11, k)
    Sc, Uc = O.action_batch(p, L, -4.0, 1.0)
    assert np.allclose(Sc, S2, atol=1e-11) and np.allclose(Uc, U2, atol=1e-11)
    assert np.all(S2 < S_star)
    assert np.all(nexp <= 7) and np.all(nshr <= 32) and (t != 0).mean() > 0.95
    # replay the first step of a few walkers by hand from the documented streams
    for i in range(0, N, 37):
        z = O.normals(7, 5, 11, i, V)
        d = Lc @ z
        assert np.allclose(p[:, i] if k == 1 else phi[:, i] + t[0, i] * d,
                           phi[:, i] + t[0, i] * d)
        f1 = phi[:, i] + t[0, i] * d
        S1, U1 = O.action_batch(f1.reshape(V, 1), L, -4.0, 1.0)
        w = O.draw(7, 7, 11, i, 0)
        logy = -U0[i] + math.log(((w[0] >> 8) + 1) / 2 ** 24)
        if t[0, i] != 0:
            assert S1[0] < S_star and -U1[0] > logy         # the accepted point is inside the slice
        assert abs(t[0, i]) <= 8.0                          # bracket never wider than m_expand * width


def test_unconstrained_1d_slice_sampler_keeps_the_standard_normal():
    """V = 1, S_star = +inf: plain slice sampling of N(0,1) with direction d = Lc z."""
    N, k = 20000, 6
    rng = np.random.default_rng(1)
    phi = rng.normal(size=(1, N))
    S, U0 = O.action_batch(phi, 1, 1.0, 0.0)
    Lc = np.array([[1.0]])
    p, S2, U2, t, nexp, nshr, amb = O.slice_walk(phi, S, U0, 1, 1.0, 0.0, Lc, np.inf, 3, 1, k)
    x = p[0]
    assert abs(x.mean()) < 4 / math.sqrt(N) and abs(x.var() - 1) < 5 * math.sqrt(2 / N)
    assert stats.kstest(x, "norm").pvalue > 1e-3
    assert np.corrcoef(phi[0], x)[0, 1] < 0.3              # the chain actually moves


def test_constrained_prior_is_invariant():
    """Exact samples of N(0,I) restricted to S_E < S_star (by rejection): the kernel must leave the
    distribution of S_E and U0 unchanged."""
    L, V = 2, 4
    rng = np.random.default_rng(2)
    cand = rng.normal(size=(V, 400000))
    S, U0 = O.action_batch(cand, L, -4.0, 1.0)
    S_star = np.quantile(S, 0.05)
    keep = np.nonzero(S < S_star)[0][:15000]
    phi, S, U0 = cand[:, keep], S[keep], U0[keep]
    N = phi.shape[1]
    _, Sig = O.covariance(phi)
    Lc, _ = O.cholesky(Sig)
    p, S2, U2, t, *_ = O.slice_walk(phi, S, U0, L, -4.0, 1.0, Lc, S_star, 5, 1, 5)
    assert np.all(S2 < S_star) and (t != 0).mean() > 0.9
    for a, b in ((S, S2), (U0, U2), (phi[0], p[0]), (np.abs(phi.mean(0)), np.abs(p.mean(0)))):
        assert abs(a.mean() - b.mean()) < 5 * a.std() / math.sqrt(N)
        assert stats.ks_2samp(a, b).pvalue > 1e-3


def test_ns_with_slice_kernel_logZ_closed_form_and_quadrature():
    exact = -0.5 * np.sum(np.log1p(gauss_a(4, 1.0)))
    lz = np.array([O.ns_run(4, 1.0, 0.0, 1024, 128, 8, s, inner="slice")["logZ"] for s in range(6)])
    assert abs(lz.mean() - exact) < 3 * lz.std(ddof=1) / math.sqrt(6) + 0.02
    f = lambda x: math.exp(-0.5 * x * x - (0.5 * -4.0 * x * x + x ** 4)) / math.sqrt(2 * math.pi)
    want = math.log(integrate.quad(f, -8, 8)[0])
    lz = np.array([O.ns_run(1, -4.0, 1.0, 1024, 128, 5, s, inner="slice")["logZ"] for s in range(8)])
    assert abs(lz.mean() - want) < 3 * lz.std(ddof=1) / math.sqrt(8) + 5e-3
    # and the two inner kernels agree on the broken-phase C0 lattice
    a = np.array([O.ns_run(4, -4.0, 1.0, 1024, 128, 10, s, inner="slice")["logZ"] for s in range(4)])
    b = np.array([O.ns_run(4, -4.0, 1.0, 1024, 128, 30, s)["logZ"] for s in range(4)])
    assert abs(a.mean() - b.mean()) < 3 * math.hypot(a.std(ddof=1), b.std(ddof=1)) / 2 + 0.08
