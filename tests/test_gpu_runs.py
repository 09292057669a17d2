"""GPU end-to-end parity: whole SMC-RW and nested-sampling runs through the C ABI against closed
forms (pins the CUDA path directly) and against oracle runs of the same configuration."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2511_15196_b200 import binding as B
from paper_2511_15196_b200 import build, inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    B.load()


def gauss_a(L, m0sq):
    k = np.arange(L)
    kh = 4 * np.sin(np.pi * k / L) ** 2
    return (m0sq + kh[:, None] + kh[None, :]).reshape(-1)


def logZ_gauss(L, m0sq):
    return -0.5 * np.sum(np.log1p(gauss_a(L, m0sq)))


def mean_se(v):
    v = np.asarray(v, float)
    return v.mean(), v.std(ddof=1) / math.sqrt(v.size)


def gpu_smc(L, N, seed, k, ess, m0sq=-4.0, lam=1.0, path=0):
    h = B.smc_init(L, m0sq, lam, N, seed)
    B.smc_set_params(h, k_steps=k, ess_target=ess, mutation_path=path)
    T = B.smc_run(h)
    out = {"T": T, "logZ": B.log_Z(h), "obs": B.observables(h), "hist": B.smc_get_history(h),
           "state": B.smc_get_state(h)}
    h.close()
    return out


def test_first_temperature_matches_oracle_stepwise():
    """One smc_step on C0 from the shared initial state: delta, dlogZ, ancestors-derived unique
    count and the post-resampling covariance agree with the oracle's first temperature."""
    c = inputs.CONFIGS["C0"]
    h = B.smc_init(c["L"], c["m0sq"], c["lam"], c["N"], 0)
    B.smc_set_params(h, k_steps=c["k"], ess_target=c["ess"])
    info = B.smc_step(h)
    ref = O.smc_run(c["L"], c["m0sq"], c["lam"], c["N"], 0, c["k"], ess_target=c["ess"], max_temps=1)
    r0 = ref["info"][0]
    assert info["temp_index"] == 0 and not info["done"]
    assert info["delta"] == pytest.approx(r0[1], rel=1e-4)
    assert info["ess_frac"] == pytest.approx(0.5, abs=1e-4)
    assert info["dlogZ"] == pytest.approx(r0[3], abs=2e-5)
    assert abs(info["n_unique"] - r0[5]) <= 2
    assert info["accept_rate"] == pytest.approx(r0[4], abs=0.03)
    assert info["chol_status"] == 0
    st = B.smc_get_state(h)
    assert st["step"] == c["k"] and st["beta"] == info["beta"]
    S, U0, A = O.action_batch(st["phi"].astype(np.float64), c["L"], c["m0sq"], c["lam"], with_abs=True)
    assert np.all(np.abs(st["S"] - S) <= 2e-5 * A)
    h.close()


def test_smc_gaussian_L4_closed_form_and_oracle():
    """lambda=0, m0^2=1 (BASELINE configs[0] Gaussian variant, stronger settings so the estimator
    bias is below the SE): GPU log Z vs the closed form -13.8046 and vs oracle runs."""
    exact = logZ_gauss(4, 1.0)
    g = [gpu_smc(4, 2048, s, 48, 0.9, m0sq=1.0, lam=0.0) for s in range(16)]
    m, se = mean_se([r["logZ"] for r in g])
    assert abs(m - exact) < 3 * se + 0.01, (m, se, exact)
    o = [O.smc_run(4, 1.0, 0.0, 2048, s, 48, ess_target=0.9)["logZ"] for s in range(16)]
    mo, so = mean_se(o)
    assert abs(m - mo) < 3 * math.hypot(se, so), (m, se, mo, so)
    m2, s2 = mean_se([r["obs"]["M2"] for r in g])
    assert abs(m2 - 1 / 32.0) < 4 * s2
    a = gauss_a(4, 1.0)
    ms, ss = mean_se([r["obs"]["mean_SE"] for r in g])
    assert abs(ms - 0.5 * np.sum(a / (1 + a))) < 4 * ss
    for r in g:
        betas = [x["beta"] for x in r["hist"]]
        assert len(betas) == r["T"] and betas[-1] == 1.0 and np.all(np.diff(betas) > 0)
        assert r["logZ"] == pytest.approx(sum(x["dlogZ"] for x in r["hist"]), rel=1e-9)
        assert all(abs(x["ess_frac"] - 0.9) < 1e-3 for x in r["hist"][:-1])


@pytest.mark.parametrize("name", ["C0", "C0g", "C1"])
def test_smc_statistical_parity_16_seeds(name):
    """BASELINE configs[0], its Gaussian variant and configs[1] (L=10, N=16384, k=20; also chi): <|M|>,
    <M^2>, histogram and log Z of 16 GPU runs vs 16 oracle runs within 3 combined standard errors."""
    c = inputs.CONFIGS[name]
    g = [gpu_smc(c["L"], c["N"], s, c["k"], c["ess"], c["m0sq"], c["lam"]) for s in range(16)]
    o = [O.smc_run(c["L"], c["m0sq"], c["lam"], c["N"], s, c["k"], ess_target=c["ess"]) for s in range(16)]
    oobs = [O.observables(r["phi"], r["S"]) for r in o]
    pairs = {"logZ": ([r["logZ"] for r in g], [r["logZ"] for r in o]),
             "absM": ([r["obs"]["absM"] for r in g], [x["absM"] for x in oobs]),
             "M2": ([r["obs"]["M2"] for r in g], [x["M2"] for x in oobs]),
             "chi": ([r["obs"]["chi"] for r in g], [x["chi"] for x in oobs]),
             "mean_SE": ([r["obs"]["mean_SE"] for r in g], [x["mean_SE"] for x in oobs])}
    for key, (a, b) in pairs.items():
        (ma, sa), (mb, sb) = mean_se(a), mean_se(b)
        assert abs(ma - mb) < 3 * math.hypot(sa, sb), (key, ma, sa, mb, sb)
    hg = np.array([r["obs"]["hist"] for r in g])
    ho = np.array([x["hist"] for x in oobs])
    # coarse 10-bin version of the 80-bin histogram, each within 3 combined SE (+ a small floor)
    cg, co = hg.reshape(16, 10, 8).sum(2), ho.reshape(16, 10, 8).sum(2)
    se = np.sqrt(cg.var(0, ddof=1) / 16 + co.var(0, ddof=1) / 16)
    assert np.all(np.abs(cg.mean(0) - co.mean(0)) < 3 * se + 2e-3)
    assert abs(np.mean([r["T"] for r in g]) - np.mean([r["T"] for r in o])) < 1.0
    if name == "C0g":
        m, se_ = mean_se([r["logZ"] for r in g])
        assert abs(m - logZ_gauss(4, 1.0)) < 4 * se_ + 0.12     # k=10 estimator is biased high (H7)


def test_smc_phi4_L1_L2_quadrature():
    """GPU log Z against 1-D / 4-D quadrature values (computed in tests/test_oracle_runs.py's
    helpers, independent of both implementations)."""
    from tests.test_oracle_runs import quad_L1, quad_L2
    g = [gpu_smc(1, 4096, s, 10, 0.9)["logZ"] for s in range(16)]
    m, se = mean_se(g)
    assert abs(m - quad_L1()[0]) < 3 * se + 1e-3, (m, se)
    g = [gpu_smc(2, 4096, s, 20, 0.9)["logZ"] for s in range(12)]
    m, se = mean_se(g)
    assert abs(m - quad_L2()) < 3 * se + 2e-3, (m, se)


def test_smc_run_is_deterministic_and_resumable():
    a = gpu_smc(4, 1024, 5, 10, 0.5)
    b = gpu_smc(4, 1024, 5, 10, 0.5)
    assert a["logZ"] == b["logZ"] and np.array_equal(a["state"]["phi"], b["state"]["phi"])
    # step-by-step == run
    h = B.smc_init(4, -4.0, 1.0, 1024, 5)
    B.smc_set_params(h, k_steps=10, ess_target=0.5)
    n = 0
    while True:
        info = B.smc_step(h)
        n += 1
        if info["done"]:
            break
    assert n == a["T"] and B.log_Z(h) == a["logZ"]
    assert np.array_equal(B.smc_get_state(h)["phi"], a["state"]["phi"])
    again = B.smc_step(h)                                   # no-op once done
    assert again["done"] and B.log_Z(h) == a["logZ"]
    h.close()


# ------------------------------------------------------------------ nested sampling -----------
def test_ns_first_iteration_lockstep():
    c = inputs.CONFIGS["C2"]
    L, n, kd, nw = c["L"], c["n_live"], c["k_del"], c["n_walk"]
    seed = 11
    h = B.ns_init(L, c["m0sq"], c["lam"], n, kd, nw, seed, max_iters=64)
    st0 = B.smc_get_state(h)
    info = B.ns_step(h)
    S0 = st0["S"].astype(np.float64)
    dead = B.ns_get_dead(h)
    ref_dead = O.ns_select(S0, kd)
    assert np.array_equal(dead["last_dead"], ref_dead)                       # N1 exact
    assert info["S_star"] == S0[ref_dead[-1]]
    per = -sum(1.0 / (n - j + 1) for j in range(1, kd + 1))                  # A6
    assert info["logX"] == pytest.approx(per, rel=1e-12)
    lw = np.array([-sum(1.0 / (n - m + 1) for m in range(1, j)) +
                   math.log1p(-math.exp(-1.0 / (n - j + 1))) for j in range(1, kd + 1)])
    assert np.allclose(dead["dead_logw"], lw, rtol=1e-12, atol=1e-14)
    assert np.array_equal(dead["dead_S"], st0["S"][ref_dead])
    Mref = st0["phi"][:, ref_dead].astype(np.float64).mean(axis=0)
    assert np.allclose(dead["dead_M"], Mref, atol=1e-6)
    from scipy.special import logsumexp
    assert info["logZ"] == pytest.approx(logsumexp(lw - S0[ref_dead]), rel=1e-10)
    # N3: replay the constrained walks in the oracle from the GPU's own start state / factor
    Lc = B.smc_get_chol(h)
    surv = np.setdiff1d(np.arange(n), ref_dead)
    start = np.array([surv[O.word0(seed, O.TAG_NS_START, 0, j) % (n - kd)] for j in range(kd)])
    p, S, U0, acc, mar, cmar = O.mutate(st0["phi"][:, start], st0["S"][start], st0["U0"][start], L,
                                        c["m0sq"], c["lam"], Lc, np.float32(2.38 / L), 0.0, seed, 1,
                                        nw, mode=O.MODE_NS, S_star=info["S_star"])
    st1 = B.smc_get_state(h)
    amb = (np.abs(mar) < 1e-4) | (np.abs(cmar) < 1e-4 * np.maximum(1.0, abs(info["S_star"])))
    clean = ~amb.any(axis=0)
    assert clean.mean() > 0.9
    got = st1["phi"][:, ref_dead]
    assert np.abs(got[:, clean] - p[:, clean]).max() < 2e-5
    assert np.all(st1["S"] < info["S_star"] + 1e-3)
    keep = np.setdiff1d(np.arange(n), ref_dead)
    assert np.array_equal(st1["phi"][:, keep], st0["phi"][:, keep])          # survivors untouched
    assert info["accept_rate"] == pytest.approx(acc.mean(), abs=0.01)
    # N4
    log_live = info["logX"] + logsumexp(-st1["S"].astype(np.float64)) - math.log(n)
    rem = math.exp(log_live - np.logaddexp(info["logZ"], log_live))
    assert info["remaining_frac"] == pytest.approx(rem, rel=1e-6)
    h.close()


def gpu_ns(L, n, kd, nw, seed, m0sq=-4.0, lam=1.0, max_iters=2048):
    h = B.ns_init(L, m0sq, lam, n, kd, nw, seed, max_iters=max_iters)
    it = B.ns_run(h, max_iters)
    out = {"iters": it, "logZ": B.log_Z(h), "obs": B.observables(h)}
    h.close()
    return out


def test_ns_gaussian_L4_closed_form_and_oracle():
    g = [gpu_ns(4, 1024, 128, 20, s, m0sq=1.0, lam=0.0) for s in range(8)]
    m, se = mean_se([r["logZ"] for r in g])
    assert abs(m - logZ_gauss(4, 1.0)) < 3 * se + 0.02, (m, se)
    o = [O.ns_run(4, 1.0, 0.0, 1024, 128, 20, s) for s in range(8)]
    mo, so = mean_se([r["logZ"] for r in o])
    assert abs(m - mo) < 3 * math.hypot(se, so) + 0.01
    assert abs(np.mean([r["iters"] for r in g]) - np.mean([r["iters"] for r in o])) < 2.0
    m2, s2 = mean_se([r["obs"]["M2"] for r in g])
    assert abs(m2 - 1 / 32.0) < 4 * s2 + 5e-4


def ns_oracle_observables(r, n, V):
    """NS-weighted observables from an oracle run: dead points with weight w_j e^{-S_j}, live points
    with weight X / n e^{-S_i} (Skilling 2006; reading A6)."""
    M = np.concatenate([r["dead_M"], O.magnetisation(r["phi"])])
    S = np.concatenate([r["dead_S"], r["S"]])
    logw = np.concatenate([r["dead_logw"] - r["dead_S"], r["logX"] - math.log(n) - r["S"]])
    return O.observables_from_M(M, S, logw, V)


def test_ns_C2_statistical_parity_16_seeds():
    """BASELINE configs[2] (L=10, 4096 live points, 512 deleted per iteration, 25-step walks, stop at
    1e-3) over 16 seeds: log Z, iteration count and the NS-weighted <|M|>, <M^2>, chi, <S_E> and
    10-bin histogram of `observables()` against the oracle's dead + live points, each within 3
    combined standard errors (north_star; PAPER.md:53(iv), :293-295)."""
    c = inputs.CONFIGS["C2"]
    L, n, V, ns = c["L"], c["n_live"], c["L"] ** 2, 16
    g = [gpu_ns(L, n, c["k_del"], c["n_walk"], s) for s in range(ns)]
    o = [O.ns_run(L, c["m0sq"], c["lam"], n, c["k_del"], c["n_walk"], s) for s in range(ns)]
    oobs = [ns_oracle_observables(r, n, V) for r in o]
    pairs = {"logZ": ([r["logZ"] for r in g], [r["logZ"] for r in o]),
             "iters": ([r["iters"] for r in g], [r["iters"] for r in o])}
    for key in ("absM", "M2", "chi", "mean_SE"):
        pairs[key] = ([r["obs"][key] for r in g], [x[key] for x in oobs])
    for key, (a, b) in pairs.items():
        (ma, sa), (mb, sb) = mean_se(a), mean_se(b)
        print("C2 %-8s gpu %.5g +- %.2g   oracle %.5g +- %.2g   (%.2f combined SE)"
              % (key, ma, sa, mb, sb, abs(ma - mb) / math.hypot(sa, sb)))
        assert abs(ma - mb) < 3 * math.hypot(sa, sb), (key, ma, sa, mb, sb)
    hg = np.array([r["obs"]["hist"] for r in g]).reshape(ns, 10, 8).sum(2)
    ho = np.array([x["hist"] for x in oobs]).reshape(ns, 10, 8).sum(2)
    se = np.sqrt(hg.var(0, ddof=1) / ns + ho.var(0, ddof=1) / ns)
    assert np.all(np.abs(hg.mean(0) - ho.mean(0)) < 3 * se + 2e-3)
    # the weighted mode balance is finite and of order one in the broken phase with both modes
    mb_g = np.array([r["obs"]["mode_balance"] for r in g])
    assert np.all(np.isfinite(mb_g)) and np.all(mb_g > 0)
