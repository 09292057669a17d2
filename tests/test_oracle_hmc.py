"""Pins of the oracle's SMC-HMC rejuvenation (NEXT row f1; PAPER.md:53(iii), :172; reading A14)."""
import math

import numpy as np
import pytest

from oracle import oracle as O


def gauss_a(L, m0sq):
    k = np.arange(L)
    kh = 4 * np.sin(np.pi * k / L) ** 2
    return (m0sq + kh[:, None] + kh[None, :]).reshape(-1)


def test_leapfrog_is_reversible_and_volume_free():
    L, V = 4, 16
    rng = np.random.default_rng(0)
    q0, p0 = rng.normal(size=V), rng.normal(size=V)
    var = rng.uniform(0.5, 2.0, V)
    q1, p1, dH = O.leapfrog(q0, p0, L, -4.0, 1.0, var, 0.05, 20, 0.7)
    q2, p2, dH2 = O.leapfrog(q1, -p1, L, -4.0, 1.0, var, 0.05, 20, 0.7)      # flip and run back
    assert np.allclose(q2, q0, atol=1e-11) and np.allclose(-p2, p0, atol=1e-11)
    assert dH2 == pytest.approx(-dH, abs=1e-10)


def test_energy_error_is_second_order():
    L, V = 4, 16
    rng = np.random.default_rng(1)
    q0, p0 = rng.normal(size=V) * 0.5, rng.normal(size=V)
    var = np.ones(V)
    T = 1.0                                            # fixed trajectory length
    errs = [abs(O.leapfrog(q0, p0, L, -4.0, 1.0, var, T / n, n, 1.0)[2]) for n in (40, 80, 160)]
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.2)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.2)


def test_free_harmonic_mode_closed_form():
    """L = 1, lambda = 0: U = 1/2 (1 + beta m0^2) phi^2, a 1-D oscillator: with many small steps the
    trajectory matches cos/sin with frequency sqrt(var (1 + beta m0^2))."""
    m0sq, beta, var = 1.0, 0.5, np.array([2.0])
    w2 = var[0] * (1 + beta * m0sq)
    q, p, dH = O.leapfrog(np.array([0.8]), np.array([0.3]), 1, m0sq, 0.0, var, 1e-3, 1000, beta)
    t, w = 1.0, math.sqrt(w2)
    want_q = 0.8 * math.cos(w * t) + 0.3 * var[0] / w * math.sin(w * t)
    assert q[0] == pytest.approx(want_q, abs=1e-5) and abs(dH) < 1e-6


def test_hmc_kernel_leaves_gaussian_target_invariant():
    L, V, N, beta = 4, 16, 20000, 0.6
    a = gauss_a(L, 1.0)
    rng = np.random.default_rng(5)
    fk = np.fft.fft2(rng.normal(size=(N, L, L))) / np.sqrt(1 + beta * a.reshape(L, L))
    phi = np.real(np.fft.ifft2(fk)).reshape(N, V).T.copy()
    S, U0 = O.action_batch(phi, L, 1.0, 0.0)
    var = phi.var(axis=1, ddof=1)
    p2, S2, U2, acc, mar = O.hmc_mutate(phi, S, U0, L, 1.0, 0.0, var, 0.3, 10, beta, seed=3, t0=1, k=3)
    assert np.array_equal(acc.astype(bool), mar > 0)
    assert 0.6 < acc.mean() <= 1.0
    Sc, Uc = O.action_batch(p2, L, 1.0, 0.0)
    assert np.allclose(Sc, S2, rtol=1e-12, atol=1e-12) and np.allclose(Uc, U2, rtol=1e-12)
    assert abs(S2.mean() - S.mean()) < 5 * S.std() / math.sqrt(N)
    M2a, M2b = O.magnetisation(phi) ** 2, O.magnetisation(p2) ** 2
    assert abs(M2b.mean() - M2a.mean()) < 5 * M2a.std() / math.sqrt(N)
    moved = np.abs(p2 - phi).max(axis=0) > 0.1
    assert moved.mean() > 0.6                          # trajectories actually move the particles


def test_smc_hmc_logZ_gaussian_and_L1():
    exact = -0.5 * np.sum(np.log1p(gauss_a(4, 1.0)))
    v = [O.smc_hmc_run(4, 1.0, 0.0, 2048, s, 4, ess_target=0.9, eps=0.25, nfrog=10)["logZ"] for s in range(8)]
    m, se = np.mean(v), np.std(v, ddof=1) / math.sqrt(8)
    assert abs(m - exact) < 3 * se + 0.01, (m, se, exact)
    from tests.test_oracle_runs import quad_L1
    v = [O.smc_hmc_run(1, -4.0, 1.0, 4096, s, 3, ess_target=0.9, eps=0.2, nfrog=10)["logZ"] for s in range(12)]
    m, se = np.mean(v), np.std(v, ddof=1) / math.sqrt(12)
    assert abs(m - quad_L1()[0]) < 3 * se + 1e-3, (m, se)
