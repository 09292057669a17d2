"""End-to-end pins of the oracle's SMC-RW and nested-sampling runs (O-2, O-3) against closed forms
and quadrature -- CPU only.  Expected values are computed here, never by the oracle."""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import oracle as O


def gauss_a(L, m0sq):
    k = np.arange(L)
    kh = 4 * np.sin(np.pi * k / L) ** 2
    return (m0sq + kh[:, None] + kh[None, :]).reshape(-1)


def logZ_gauss(L, m0sq):
    """log int N(phi;0,I) exp(-S_E) dphi for lambda=0: -1/2 sum_k ln(1 + a_k) (reading A1)."""
    return -0.5 * np.sum(np.log1p(gauss_a(L, m0sq)))


def quad_L1(beta=1.0, m0sq=-4.0, lam=1.0):
    """1-D quadrature at L=1 (kinetic term vanishes, A2): Z, <M^2>, <|M|>, <S_E> under
    N(phi;0,1) exp(-beta S_E)."""
    s = lambda p: 0.5 * m0sq * p * p + lam * p ** 4
    dens = lambda p: math.exp(-0.5 * p * p - beta * s(p)) / math.sqrt(2 * math.pi)
    I = lambda g: integrate.quad(lambda p: g(p) * dens(p), -8, 8, epsabs=1e-13, epsrel=1e-13)[0]
    Z = I(lambda p: 1.0)
    return math.log(Z), I(lambda p: p * p) / Z, I(abs) / Z, I(s) / Z


def quad_L2(m0sq=-4.0, lam=1.0, n=81, lim=4.0):
    """4-D trapezoid at L=2, V=4; every bond of the 2x2 torus is doubled (A2):
    S = sum over the 4 distinct bonds of (dphi)^2 + sum_x pot(phi_x)."""
    x = np.linspace(-lim, lim, n)
    h = x[1] - x[0]
    g = np.exp(-0.5 * x * x - (0.5 * m0sq * x * x + lam * x ** 4)) / math.sqrt(2 * math.pi)
    T = np.exp(-(x[:, None] - x[None, :]) ** 2)              # one doubled bond
    # sites a b / c d ; bonds a-b, c-d, a-c, b-d.  Z = sum_{a,d} g_a g_d (sum_b g_b T_ab T_bd)^2
    K = (T * g[None, :]) @ T * h                             # K[a,d] = sum_b T_ab g_b T_bd
    Z = np.sum(g[:, None] * g[None, :] * K * K) * h * h
    return math.log(Z)


def test_quadrature_reference_values():
    # SURVEY 8(c) [quadrature] values -- recomputed here, not read from the oracle
    lz, m2, am, se = quad_L1()
    assert lz == pytest.approx(0.389979211603, abs=1e-10)
    assert m2 == pytest.approx(0.657861312140, abs=1e-9)
    assert am == pytest.approx(0.718901424834, abs=1e-9)
    assert se == pytest.approx(-0.572326640175, abs=1e-9)
    assert quad_L2() == pytest.approx(-0.917325395297, abs=1e-8)
    assert logZ_gauss(4, 1.0) == pytest.approx(-13.804616350061, abs=1e-10)
    assert logZ_gauss(2, 1.0) == pytest.approx(-3.289625606005, abs=1e-10)


def _mean_se(v):
    v = np.asarray(v)
    return v.mean(), v.std(ddof=1) / math.sqrt(v.size)


def test_smc_logZ_gaussian_L4():
    """lambda=0, m0^2=1, L=4: exact log Z = -13.8046 (BJ north_star's closed form)."""
    runs = [O.smc_run(4, 1.0, 0.0, 2048, s, 48, ess_target=0.9) for s in range(8)]
    m, se = _mean_se([r["logZ"] for r in runs])
    assert abs(m - logZ_gauss(4, 1.0)) < 3 * se + 0.01, (m, se)
    assert se < 0.03
    # observables at beta=1: <M^2> = 1/(V (1+m0^2)), E[S_E] = 1/2 sum a/(1+a)
    a = gauss_a(4, 1.0)
    m2 = [O.observables(r["phi"], r["S"])["M2"] for r in runs]
    ms, ses = _mean_se(m2)
    assert abs(ms - 1.0 / (16 * 2.0)) < 4 * ses
    sm, sse = _mean_se([r["S"].mean() for r in runs])
    assert abs(sm - 0.5 * np.sum(a / (1 + a))) < 4 * sse
    for r in runs:
        b = r["info"][:, 0]
        assert np.all(np.diff(b) > 0) and b[-1] == 1.0
        assert np.all(r["info"][:-1, 2] == pytest.approx(0.9, abs=1e-6))
        assert r["logZ"] == pytest.approx(r["info"][:, 3].sum(), rel=1e-12)
        S, U0 = O.action_batch(r["phi"], 4, 1.0, 0.0)
        assert np.allclose(S, r["S"], rtol=1e-12, atol=1e-12)
        assert np.allclose(U0, r["U0"], rtol=1e-12, atol=1e-12)


def test_smc_schedule_gaussian_L4_target_half():
    # closed-form large-N schedule at ESS 0.5: 0.0789, 0.1938, 0.3589, 0.5940, 0.9274, 1 (6 temps)
    r = O.smc_run(4, 1.0, 0.0, 8192, 1, 32, ess_target=0.5)
    want = [0.078920, 0.193823, 0.358873, 0.594047, 0.927425, 1.0]
    assert r["T"] == 6
    assert np.allclose(r["info"][:, 0], want, rtol=0.08)


def test_smc_phi4_L1_quadrature():
    lz, m2, am, se_ = quad_L1()
    runs = [O.smc_run(1, -4.0, 1.0, 4096, s, 10, ess_target=0.9) for s in range(16)]
    m, se = _mean_se([r["logZ"] for r in runs])
    assert abs(m - lz) < 3 * se + 1e-3, (m, se)
    obs = [O.observables(r["phi"], r["S"]) for r in runs]
    for key, want in (("M2", m2), ("absM", am), ("mean_SE", se_)):
        mm, ss = _mean_se([o[key] for o in obs])
        assert abs(mm - want) < 4 * ss, (key, mm, ss, want)
    # histogram is a normalised density over 80 bins, symmetric target
    h = np.mean([o["hist"] for o in obs], axis=0)
    assert h.sum() == pytest.approx(1.0, abs=1e-12)
    assert abs(h[:40].sum() - 0.5) < 0.03


def test_smc_phi4_L2_quadrature():
    runs = [O.smc_run(2, -4.0, 1.0, 4096, s, 20, ess_target=0.9) for s in range(12)]
    m, se = _mean_se([r["logZ"] for r in runs])
    assert abs(m - quad_L2()) < 3 * se + 2e-3, (m, se)


def test_mutation_leaves_gaussian_target_invariant_and_is_consistent():
    """RW-Metropolis kernel: start from exact samples of the Gaussian p_beta, k steps leave the
    moments unchanged; accept == (margin > 0); rejected particles untouched; cached S, U0 exact."""
    L, V, N, beta = 4, 16, 20000, 0.6
    a = gauss_a(L, 1.0)
    rng = np.random.default_rng(5)
    # exact sampling in Fourier space: real field with spectrum 1/(1+beta a_k)
    white = rng.normal(size=(N, L, L))
    fk = np.fft.fft2(white) / np.sqrt(1 + beta * a.reshape(L, L))
    phi = np.real(np.fft.ifft2(fk)).reshape(N, V).T.copy()
    S, U0 = O.action_batch(phi, L, 1.0, 0.0)
    assert S.mean() == pytest.approx(0.5 * np.sum(a / (1 + beta * a)), rel=0.02)
    _, Lc, st = O.cov_chol(phi)
    assert st == 0
    s = 2.38 / math.sqrt(V)
    p2, S2, U2, acc, mar, _ = O.mutate(phi, S, U0, L, 1.0, 0.0, Lc, s, beta, seed=3, t0=1, k=8)
    assert np.array_equal(acc.astype(bool), mar > 0)
    assert 0.15 < acc.mean() < 0.45                       # 2.38/sqrt(V) scaling
    never = acc.sum(axis=0) == 0
    assert never.any() and np.array_equal(p2[:, never], phi[:, never])
    Sc, Uc = O.action_batch(p2, L, 1.0, 0.0)
    assert np.allclose(Sc, S2, rtol=1e-12, atol=1e-12) and np.allclose(Uc, U2, rtol=1e-12)
    se = S.std() / math.sqrt(N)
    assert abs(S2.mean() - S.mean()) < 5 * se
    M2a, M2b = O.magnetisation(phi) ** 2, O.magnetisation(p2) ** 2
    assert abs(M2b.mean() - M2a.mean()) < 5 * M2a.std() / math.sqrt(N)
    assert M2b.mean() == pytest.approx(1.0 / (V * (1 + beta * 1.0)), rel=0.05)
    # first-step margin, retyped once from R4 for one particle with its own streams
    i = 17
    z = O.normals(3, O.TAG_PROP, 1, i, V)
    fp = phi[:, i] + s * (Lc @ z)
    g = -((O.u0_field(fp) - U0[i]) + beta * (O.action_field(fp, L, 1.0, 0.0) - S[i])) \
        - math.log(O.uniform(3, O.TAG_ACC, 1, i))
    assert mar[0, i] == pytest.approx(g, rel=1e-10, abs=1e-12)


def test_mutate_ns_mode_constraint():
    L, V, N = 3, 9, 4000
    phi = O.init_particles(2, N, V)
    S, U0 = O.action_batch(phi, L, -4.0, 1.0)
    S_star = np.median(S)
    keep = S < S_star
    phi, S, U0 = phi[:, keep].copy(), S[keep].copy(), U0[keep].copy()
    _, Lc, _ = O.cov_chol(phi)
    p2, S2, U2, acc, mar, cmar = O.mutate(phi, S, U0, L, -4.0, 1.0, Lc, 2.38 / 3, 0.0, seed=2,
                                          t0=1, k=5, mode=O.MODE_NS, S_star=S_star)
    assert np.all(S2 < S_star)
    assert np.array_equal(acc.astype(bool), (mar > 0) & (cmar > 0))
    assert ((mar > 0) & (cmar <= 0)).any()                 # the constraint did reject something
    Sc, _ = O.action_batch(p2, L, -4.0, 1.0)
    assert np.allclose(Sc, S2, rtol=1e-12, atol=1e-12)


# --------------------------------------------------------------------- NS ---
def test_ns_select_order():
    rng = np.random.default_rng(4)
    S = rng.normal(size=300).round(1)                     # many ties
    dead = O.ns_select(S, 40)
    order = np.lexsort((np.arange(300), -S))              # S descending, ties by index ascending
    assert np.array_equal(dead, order[:40])


def test_ns_logZ_gaussian_L4_and_volume_bookkeeping():
    n, kd = 1024, 128
    runs = [O.ns_run(4, 1.0, 0.0, n, kd, 20, s) for s in range(6)]
    lz = [r["logZ"] for r in runs]
    m, se = _mean_se(lz)
    assert abs(m - logZ_gauss(4, 1.0)) < 3 * se + 0.02, (m, se)
    r = runs[0]
    # A6: deterministic shrinkage per iteration = -sum_{j=1..k} 1/(n-j+1)
    per = -sum(1.0 / (n - j + 1) for j in range(1, kd + 1))
    assert np.allclose(np.diff(r["info"][:, 0]), per, rtol=1e-12)
    assert r["info"][0, 0] == pytest.approx(per, rel=1e-12)
    assert r["logX"] == pytest.approx(per * r["iters"], rel=1e-12)
    # dead weights tile the unit volume: sum w_j + X_final = 1
    assert np.exp(r["dead_logw"]).sum() + math.exp(r["logX"]) == pytest.approx(1.0, rel=1e-12)
    # thresholds tighten monotonically, live points obey the last one, termination rule fired
    assert np.all(np.diff(r["info"][:, 2]) < 0)
    assert np.all(r["S"] < r["info"][-1, 2])
    assert r["info"][-1, 4] < 1e-3 and np.all(r["info"][:-1, 4] >= 1e-3)
    # within an iteration dead points are in increasing likelihood
    dS = r["dead_S"].reshape(r["iters"], kd)
    assert np.all(np.diff(dS, axis=1) <= 0)
    # posterior <M^2> from dead + live points vs 1/(V(1+m0^2))
    vals = []
    for r in runs:
        M = np.concatenate([r["dead_M"], O.magnetisation(r["phi"])])
        lw = np.concatenate([r["dead_logw"] - r["dead_S"],
                             np.full(n, r["logX"] - math.log(n)) - r["S"]])
        vals.append(O.observables_from_M(M, None, lw, 16)["M2"])
    mm, ss = _mean_se(vals)
    assert abs(mm - 1 / 32.0) < 4 * ss + 5e-4, (mm, ss)


def test_ns_phi4_L1_and_agreement_with_smc_on_C0():
    lz1 = quad_L1()[0]
    v = [O.ns_run(1, -4.0, 1.0, 1024, 128, 10, s)["logZ"] for s in range(8)]
    m, se = _mean_se(v)
    assert abs(m - lz1) < 3 * se + 5e-3, (m, se)
    ns = [O.ns_run(4, -4.0, 1.0, 2048, 256, 30, s)["logZ"] for s in range(4)]
    smc = [O.smc_run(4, -4.0, 1.0, 2048, s, 48, ess_target=0.9)["logZ"] for s in range(4)]
    (a, sa), (b, sb) = _mean_se(ns), _mean_se(smc)
    assert abs(a - b) < 3 * math.hypot(sa, sb) + 0.05, (a, sa, b, sb)
