"""Pins of the kappa-lambda parameterisation (Appendix G, Eqs. 2-5; reading A18)
in the oracle -- CPU only.  Expected values are written out here from the paper's equations, never
taken from the oracle."""
import math

import numpy as np
import pytest

from oracle import oracle as O


def _field(L, seed):
    return np.random.default_rng(seed).normal(size=(L, L))


def eq5(f, kappa, lam):
    """Eq. 5: -kappa sum_{x,mu} phi_x phi_{x+mu} + (kappa D + 1 - 2 lambda) sum phi^2
    + lambda sum phi^4, D = 2, constant dropped."""
    nb = np.roll(f, -1, axis=0) + np.roll(f, -1, axis=1)
    return -kappa * np.sum(f * nb) + (2 * kappa + 1 - 2 * lam) * np.sum(f ** 2) + lam * np.sum(f ** 4)


@pytest.mark.parametrize("L", [1, 2, 3, 6])
@pytest.mark.parametrize("kappa,lam", [(0.3, 0.5), (1.0, 0.02), (2.5, 1.7)])
def test_eq2_eq5_and_the_eq1_stencil_agree(L, kappa, lam):
    f = _field(L, 7 * L)
    V = L * L
    kin, m0sq, l4, const = O.kl_to_eq1(kappa, lam)
    with O.kinetic(kin):
        s1 = O.action_field(f, L, m0sq, l4)
    assert O.kinetic  # context restored below
    assert O.lib().orc_get_kinetic() == 1.0
    s2 = O.action_eq2_field(f, L, kappa, lam)
    assert s2 == pytest.approx(eq5(f, kappa, lam) + V * lam, rel=1e-12, abs=1e-12)   # Eqs. 3-5
    assert s1 == pytest.approx(s2 - V * const, rel=1e-12, abs=1e-12)                 # Eq. 4 remap
    assert s1 == pytest.approx(eq5(f, kappa, lam), rel=1e-12, abs=1e-12)


def test_kappa_scales_only_the_kinetic_term():
    L, m0sq, lam = 5, -4.0, 1.0
    f = _field(L, 3)
    s_pot = O.action_field(np.full((L, L), 0.0), L, m0sq, lam)
    assert s_pot == 0.0
    with O.kinetic(0.0):
        pot = O.action_field(f, L, m0sq, lam)
    assert pot == pytest.approx(np.sum(0.5 * m0sq * f ** 2 + lam * f ** 4), rel=1e-13)
    base = O.action_field(f, L, m0sq, lam)
    for kappa in (0.25, 2.0, 3.5):
        with O.kinetic(kappa):
            assert O.action_field(f, L, m0sq, lam) == pytest.approx(pot + kappa * (base - pot), rel=1e-12)
    c = np.full((L, L), 0.7)                         # constant field: kinetic term vanishes
    with O.kinetic(9.0):
        assert O.action_field(c, L, m0sq, lam) == pytest.approx(L * L * (0.5 * m0sq * 0.49 + lam * 0.7 ** 4), rel=1e-13)


@pytest.mark.parametrize("L", [2, 3, 4])
def test_plane_wave_eigenvalues_with_kappa(L):
    """lambda = 0: S = 1/2 (m0^2 + kappa khat^2) |phi|^2 on a lattice plane wave."""
    m0sq, kappa = 0.5, 1.7
    r, c = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    for k1 in range(L):
        for k2 in range(L):
            f = np.cos(2 * np.pi * (k1 * r + k2 * c) / L)
            kh = 4 * np.sin(np.pi * k1 / L) ** 2 + 4 * np.sin(np.pi * k2 / L) ** 2
            with O.kinetic(kappa):
                got = O.action_field(f, L, m0sq, 0.0)
            assert got == pytest.approx(0.5 * (m0sq + kappa * kh) * np.sum(f * f), rel=1e-12, abs=1e-12)


@pytest.mark.parametrize("L", [1, 2, 3, 6])
def test_gradient_with_kappa_matches_finite_differences(L):
    kappa, m0sq, lam = 0.6, -1.5, 0.8
    f = _field(L, 10 + L)
    with O.kinetic(kappa):
        g = O.action_grad_field(f, L, m0sq, lam).reshape(L, L)
        h = 1e-5
        for r in range(L):
            for c in range(L):
                fp, fm = f.copy(), f.copy()
                fp[r, c] += h
                fm[r, c] -= h
                fd = (O.action_field(fp, L, m0sq, lam) - O.action_field(fm, L, m0sq, lam)) / (2 * h)
                assert g[r, c] == pytest.approx(fd, rel=1e-6, abs=1e-7)


def logZ_gauss_kappa(L, kappa, m0sq):
    """lambda = 0: log int N(phi;0,I) exp(-S) dphi = -1/2 sum_k ln(1 + m0^2 + kappa khat_k^2)."""
    k = np.arange(L)
    kh = 4 * np.sin(np.pi * k / L) ** 2
    return -0.5 * np.sum(np.log1p(m0sq + kappa * (kh[:, None] + kh[None, :])))


def _mean_se(v):
    v = np.asarray(v)
    return v.mean(), v.std(ddof=1) / math.sqrt(v.size)


def test_smc_logZ_gaussian_eq2_L4():
    """Eq. 2 at lambda = 0: S = kappa/2 sum (dphi)^2 + sum phi^2, i.e. m0^2 = 2 -- Gaussian, so
    log Z is the closed form above; the SMC-RW, SMC-HMC runs must reproduce it."""
    kappa = 0.5
    kin, m0sq, lam, _ = O.kl_to_eq1(kappa, 0.0)
    want = logZ_gauss_kappa(4, kappa, m0sq)
    assert want == pytest.approx(-0.5 * sum(math.log(3 + 0.5 * (a + b)) for a in (0, 2, 4, 2) for b in (0, 2, 4, 2)), rel=1e-13)
    with O.kinetic(kin):
        runs = [O.smc_run(4, m0sq, lam, 2048, s, 48, ess_target=0.9) for s in range(8)]
        hruns = [O.smc_hmc_run(4, m0sq, lam, 1024, s, 2, ess_target=0.9, eps=0.15, nfrog=10) for s in range(8)]
    m, se = _mean_se([r["logZ"] for r in runs])
    assert abs(m - want) < 3 * se + 0.01, (m, se, want)
    assert abs(m - logZ_gauss_kappa(4, 1.0, m0sq)) > 10 * se        # kappa = 1 would be caught
    m, se = _mean_se([r["logZ"] for r in hruns])
    assert abs(m - want) < 3 * se + 0.01, (m, se, want)
    # <M^2> at beta = 1: the zero mode has variance 1/(1 + m0^2) whatever kappa
    m2, s2 = _mean_se([O.observables(r["phi"], r["S"])["M2"] for r in runs])
    assert abs(m2 - 1.0 / (16 * (1 + m0sq))) < 4 * s2


def quad_L2_kappa(kappa, m0sq, lam, n=81, lim=4.0):
    """4-D trapezoid at L = 2 with the kinetic term scaled by kappa (every bond of the 2x2 torus
    doubled, A2): S = kappa sum over the 4 distinct bonds of (dphi)^2 + sum_x pot(phi_x)."""
    x = np.linspace(-lim, lim, n)
    h = x[1] - x[0]
    g = np.exp(-0.5 * x * x - (0.5 * m0sq * x * x + lam * x ** 4)) / math.sqrt(2 * math.pi)
    T = np.exp(-kappa * (x[:, None] - x[None, :]) ** 2)
    K = (T * g[None, :]) @ T * h
    return math.log(np.sum(g[:, None] * g[None, :] * K * K) * h * h)


def test_smc_phi4_eq2_L2_quadrature():
    """Broken-phase Eq. 2 point (kappa = 0.8, lambda = 1.5: m0^2 = -4) on the 2x2 torus against 4-D
    quadrature; also an NS run (hard-constraint kernel) at the same point."""
    kappa, lam2 = 0.8, 1.5
    kin, m0sq, lam, _ = O.kl_to_eq1(kappa, lam2)
    assert m0sq == -4.0
    want = quad_L2_kappa(kappa, m0sq, lam)
    assert abs(want - quad_L2_kappa(1.0, m0sq, lam)) > 0.05
    with O.kinetic(kin):
        runs = [O.smc_run(2, m0sq, lam, 4096, s, 20, ess_target=0.9) for s in range(12)]
        ns = [O.ns_run(2, m0sq, lam, 1024, 128, 20, s) for s in range(6)]
    m, se = _mean_se([r["logZ"] for r in runs])
    assert abs(m - want) < 3 * se + 2e-3, (m, se, want)
    m, se = _mean_se([r["logZ"] for r in ns])
    assert abs(m - want) < 3 * se + 0.02, (m, se, want)
