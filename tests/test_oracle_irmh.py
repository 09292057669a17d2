"""Pins of the oracle's SMC-IRMH rejuvenation (NEXT row f2; PAPER.md:53(ii), :200; reading A15)."""
import math

import numpy as np
import pytest
from scipy import integrate
from scipy.stats import multivariate_normal

from oracle import oracle as O


def gauss_K(L, m0sq):
    """Matrix of the quadratic action S_E = 1/2 phi^T K phi (lambda = 0) on the periodic lattice."""
    V = L * L
    K = np.zeros((V, V))
    for r in range(L):
        for c in range(L):
            x = r * L + c
            K[x, x] += 4 + m0sq
            for y in (r * L + (c + 1) % L, r * L + (c - 1) % L, ((r + 1) % L) * L + c,
                      ((r - 1) % L) * L + c):
                K[x, y] -= 1
    return K


def test_proposal_equal_to_target_is_always_accepted():
    """Gaussian target p_beta = N(0, (I + beta K)^-1) and the proposal fitted to it exactly: the MH
    ratio is 1 for every proposal, so g = -ln u to rounding and every step accepts."""
    L, V, N, beta = 3, 9, 500, 0.7
    Sig = np.linalg.inv(np.eye(V) + beta * gauss_K(L, 0.8))
    Lc = np.linalg.cholesky(Sig)
    rng = np.random.default_rng(0)
    phi = Lc @ rng.normal(size=(V, N))
    S, U0 = O.action_batch(phi, L, 0.8, 0.0)
    p, S2, U2, acc, mar = O.irmh_mutate(phi, S, U0, L, 0.8, 0.0, np.zeros(V), Lc, beta, 11, 1, 4)
    assert acc.all()
    u = np.array([[O.uniform(11, 2, 1 + j, i) for i in range(N)] for j in range(4)])
    assert np.allclose(mar, -np.log(u), atol=1e-9)
    # the new state is the proposal mu + Lc z of the last step
    z = np.stack([O.normals(11, 1, 4, i, V) for i in range(N)], axis=1)
    assert np.allclose(p, Lc @ z, atol=1e-12)


def test_margin_against_library_densities():
    """g + ln u = log[p(phi') q(phi)] - log[p(phi) q(phi')] with q from scipy's multivariate normal."""
    L, V, N, beta = 2, 4, 40, 0.45
    rng = np.random.default_rng(3)
    A = rng.normal(size=(V, V))
    Sig = A @ A.T / V + 0.3 * np.eye(V)
    mu = rng.normal(size=V) * 0.3
    Lc = np.linalg.cholesky(Sig)
    phi = rng.normal(size=(V, N))
    S, U0 = O.action_batch(phi, L, -4.0, 1.0)
    p, S2, U2, acc, mar = O.irmh_mutate(phi, S, U0, L, -4.0, 1.0, mu, Lc, beta, 5, 7, 1)
    q = multivariate_normal(mean=mu, cov=Sig)
    for i in range(N):
        z = O.normals(5, 1, 7, i, V)
        fp = mu + Lc @ z
        Sp, Up = O.action_batch(fp.reshape(V, 1), L, -4.0, 1.0)
        want = (-(Up[0] + beta * Sp[0]) + q.logpdf(phi[:, i])) - (-(U0[i] + beta * S[i]) + q.logpdf(fp))
        u = O.uniform(5, 2, 7, i)
        assert mar[0, i] == pytest.approx(want - math.log(u), abs=1e-9)
        assert np.allclose(p[:, i], fp if acc[0, i] else phi[:, i])


def test_whitened_norm_is_carried_correctly_over_steps():
    """k steps in one call == k calls of one step (the carried |w|^2 = |z|^2 after an accept equals
    the forward substitution of the accepted state)."""
    L, V, N, beta = 3, 9, 300, 0.6
    rng = np.random.default_rng(8)
    phi = rng.normal(size=(V, N)) * 0.7
    mu, Sig = O.covariance(phi)
    Lc, st = O.cholesky(Sig)
    S, U0 = O.action_batch(phi, L, -4.0, 1.0)
    pa, Sa, Ua, acca, mara = O.irmh_mutate(phi, S, U0, L, -4.0, 1.0, mu, Lc, beta, 2, 1, 5)
    pb, Sb, Ub = phi, S, U0
    for j in range(5):
        pb, Sb, Ub, accb, marb = O.irmh_mutate(pb, Sb, Ub, L, -4.0, 1.0, mu, Lc, beta, 2, 1 + j, 1)
        assert np.array_equal(accb[0], acca[j]) and np.allclose(marb[0], mara[j], atol=1e-9)
    assert np.allclose(pa, pb) and 0.02 < acca.mean() < 0.98


def test_irmh_leaves_target_invariant_with_a_mismatched_proposal():
    L, V, N, beta = 3, 9, 40000, 1.0
    K = gauss_K(L, 1.0)
    Sig_t = np.linalg.inv(np.eye(V) + beta * K)
    rng = np.random.default_rng(4)
    phi = np.linalg.cholesky(Sig_t) @ rng.normal(size=(V, N))
    S, U0 = O.action_batch(phi, L, 1.0, 0.0)
    mu = np.full(V, 0.05)
    Lc = np.linalg.cholesky(1.4 * Sig_t + 0.02 * np.eye(V))
    p, S2, U2, acc, mar = O.irmh_mutate(phi, S, U0, L, 1.0, 0.0, mu, Lc, beta, 9, 1, 3)
    assert 0.2 < acc.mean() < 0.95
    Sc, Uc = O.action_batch(p, L, 1.0, 0.0)
    assert np.allclose(Sc, S2) and np.allclose(Uc, U2)
    assert abs(S2.mean() - S.mean()) < 5 * S.std() / math.sqrt(N)
    assert abs(U2.mean() - U0.mean()) < 5 * U0.std() / math.sqrt(N)
    assert abs(p.mean()) < 5 * math.sqrt(Sig_t.trace() / V / (V * N)) * 3


def test_smc_irmh_logZ_gaussian_and_L1():
    exact = -0.5 * np.linalg.slogdet(np.eye(16) + gauss_K(4, 1.0))[1]
    lz = np.array([O.smc_irmh_run(4, 1.0, 0.0, 2048, 50 + s, 3, 0.7)["logZ"] for s in range(12)])
    assert abs(lz.mean() - exact) < 3 * lz.std(ddof=1) / math.sqrt(12) + 5e-3
    # L = 1 phi^4 (both neighbours are the site itself: no kinetic term), bimodal: 1-D quadrature
    f = lambda x: math.exp(-0.5 * x * x - (0.5 * -4.0 * x * x + x ** 4)) / math.sqrt(2 * math.pi)
    want = math.log(integrate.quad(f, -8, 8)[0])
    lz = np.array([O.smc_irmh_run(1, -4.0, 1.0, 4096, 80 + s, 3, 0.7)["logZ"] for s in range(12)])
    assert abs(lz.mean() - want) < 3 * lz.std(ddof=1) / math.sqrt(12) + 5e-3
