"""GPU parity for the SMC-HMC row (PAPER.md:53(iii), :172; reading A14): the CUDA
HMC kernel through the C ABI against the FP64 oracle on the same seeded inputs.

Tolerance.  An HMC proposal is a whole trajectory, not a small perturbation, so H_new is a full
fp32 evaluation of S_E, U0 and the kinetic energy: the margin g = (H_old - H_new) - ln u carries
the 2e-5 * A error of reading A12 (A = sum of the absolute terms of S_E, a few hundred at V = 100)
plus the fp32 rounding of nfrog leapfrog steps.  Decisions are therefore compared outside
|g| < BAND_HMC = 6e-4 and margins within BAND_HMC / 2 + 1e-5 |g| (measured: 3e-5 at C1's
shape, 1.1e-4 worst case over the twelve lock-step shapes in round 2 -- profiles/r02_parity_margins.md --
and 2.3e-4 on unit-normal fields at L = 4; the band was 1e-3 in round 1)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2511_15196_b200 import binding as B
from paper_2511_15196_b200 import build, inputs

pytestmark = pytest.mark.gpu

BAND_HMC = 6e-4


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    B.load()


def hmc_lockstep(L, N, k, beta, seed, eps, nfrog, m0sq=-4.0, lam=1.0, t_start=0, fields="smooth"):
    h = B.smc_init(L, m0sq, lam, N, seed)
    B.smc_set_params(h, k_steps=k, kernel=1, hmc_eps=eps, hmc_leapfrog=nfrog)
    if fields == "smooth":
        B.smc_set_state(h, inputs.smooth_fields(L, N, seed=seed + 1), beta, t_start)
    else:
        B.smc_set_state(h, B.smc_get_state(h)["phi"], beta, t_start)
    B.estimate_cov_chol(h)
    st0 = B.smc_get_state(h)
    acc, mar = B.smc_mutate(h, k)
    st1 = B.smc_get_state(h)
    assert st1["step"] == t_start + k
    f0 = st0["phi"].astype(np.float64)
    S0, U00 = O.action_batch(f0, L, m0sq, lam)
    _, Sig = O.covariance(f0)
    p, S, U0, oacc, omar = O.hmc_mutate(f0, S0, U00, L, m0sq, lam, np.diag(Sig).copy(),
                                        float(np.float32(eps)), nfrog, beta, seed, t_start + 1, k)
    amb = np.abs(omar) < BAND_HMC
    first = np.where(amb.any(axis=0), amb.argmax(axis=0), k)
    valid = np.arange(k)[:, None] < first[None, :]
    assert valid.mean() > 0.9
    assert np.array_equal(acc[valid], oacc[valid]), "HMC accept decisions differ outside the band"
    assert np.all(np.isfinite(st1["phi"]))
    # a diverging trajectory (|g| beyond any acceptable energy error) amplifies rounding along the
    # way: relative 1e-3 there; the decision (reject) is exact either way
    d, go = np.abs(mar[valid] - omar[valid]), np.abs(omar[valid])
    sane = go < 20.0
    print("hmc L=%d N=%d: worst |dg| %.2e on |g| < 20 (band %.0e), valid fraction %.3f"
          % (L, N, d[sane].max() if sane.any() else 0.0, BAND_HMC, valid.mean()))
    assert np.all(d < np.where(go < 20.0, 0.5 * BAND_HMC + 1e-5 * go, 1e-3 * go))
    clean = first == k
    assert np.abs(st1["phi"][:, clean] - p[:, clean]).max() < 1e-4
    Sx, Ux, A = O.action_batch(st1["phi"].astype(np.float64), L, m0sq, lam, with_abs=True)
    assert np.all(np.abs(st1["S"] - Sx) <= 2e-5 * A + 2e-5)
    assert np.all(np.abs(st1["U0"] - Ux) <= 2e-5 * Ux + 2e-5)
    h.close()
    return acc.mean(), np.abs(mar[valid] - omar[valid]).max()


@pytest.mark.parametrize("L,N,k,beta,eps,nfrog,fields", [
    (10, 4096, 3, 0.3, 0.15, 20, "smooth"), (10, 1000, 2, 1.0, 0.1, 20, "smooth"),
    (4, 1024, 4, 0.5, 0.1, 10, "init"), (5, 333, 3, 0.7, 0.15, 7, "smooth"),
    (1, 200, 5, 1.0, 0.1, 5, "init"), (2, 129, 4, 0.5, 0.1, 8, "init"),
    (9, 640, 2, 0.6, 0.1, 20, "smooth"), (16, 2048, 2, 0.2, 0.1, 20, "smooth"),
    (22, 500, 1, 0.4, 0.05, 12, "smooth"), (11, 31, 2, 0.0, 0.1, 6, "init"),
    # L > 22: position and momentum in HBM scratch, one launch per leapfrog half-step
    (23, 300, 2, 0.4, 0.05, 10, "smooth"), (32, 200, 1, 0.3, 0.04, 8, "smooth")])
def test_hmc_lockstep(L, N, k, beta, eps, nfrog, fields):
    rate, _ = hmc_lockstep(L, N, k, beta, seed=31 + L, eps=eps, nfrog=nfrog, fields=fields,
                           t_start=5 * k)
    assert 0.0 < rate <= 1.0


def test_hmc_rejects_bad_parameters():
    h = B.smc_init(10, -4.0, 1.0, 256, 1)
    for bad in (dict(hmc_eps=0.0), dict(hmc_leapfrog=0), dict(kernel=3)):
        with pytest.raises(B.Phi4Error):
            B.smc_set_params(h, **{"kernel": 1, **bad})
    h.close()


def smc_hmc_gpu(L, m0sq, lam, N, seed, k, ess, eps, nfrog):
    h = B.smc_init(L, m0sq, lam, N, seed)
    B.smc_set_params(h, k_steps=k, ess_target=ess, kernel=1, hmc_eps=eps, hmc_leapfrog=nfrog)
    T = B.smc_run(h)
    hist = B.smc_get_history(h)
    lz = B.log_Z(h)
    obs = B.observables(h)
    h.close()
    return T, lz, hist, obs


def test_smc_hmc_first_temperature_matches_oracle():
    """Temperature 0 has no earlier decision to diverge on: beta_1, dlogZ and ESS agree to fp32
    rounding, the acceptance rate to the band fraction."""
    L, N, k = 6, 2048, 2
    T, lz, hist, _ = smc_hmc_gpu(L, -4.0, 1.0, N, 5, k, 0.5, 0.15, 10)
    ref = O.smc_hmc_run(L, -4.0, 1.0, N, 5, k, 0.5, float(np.float32(0.15)), 10)
    assert abs(hist[0]["beta"] - ref["info"][0, 0]) < 1e-5 * ref["info"][0, 0] + 1e-7
    assert abs(hist[0]["dlogZ"] - ref["info"][0, 3]) < 1e-4
    assert abs(hist[0]["accept_rate"] - ref["info"][0, 4]) < 0.01
    assert abs(T - ref["T"]) <= 2


def test_smc_hmc_gaussian_closed_form():
    """lambda = 0, m0^2 > 0: log Z = -1/2 log det(I + K) (reading A1); SMC-HMC estimates over seeds
    must agree with it within 3 SE, and with the oracle's SMC-HMC estimates within 3 combined SE."""
    L, N, k, m0sq = 4, 2048, 2, 0.5
    V = L * L
    K = np.zeros((V, V))
    for r in range(L):
        for c in range(L):
            x = r * L + c
            K[x, x] += 4 + m0sq
            for y in (r * L + (c + 1) % L, r * L + (c - 1) % L, ((r + 1) % L) * L + c,
                      ((r - 1) % L) * L + c):
                K[x, y] -= 1
    exact = -0.5 * np.linalg.slogdet(np.eye(V) + K)[1]
    g = np.array([smc_hmc_gpu(L, m0sq, 0.0, N, 100 + s, k, 0.7, 0.2, 10)[1] for s in range(16)])
    o = np.array([O.smc_hmc_run(L, m0sq, 0.0, N, 100 + s, k, 0.7, float(np.float32(0.2)), 10)["logZ"]
                  for s in range(16)])
    se_g, se_o = g.std(ddof=1) / 4, o.std(ddof=1) / 4
    assert abs(g.mean() - exact) < 3 * se_g + 0.01
    assert abs(g.mean() - o.mean()) < 3 * np.hypot(se_g, se_o) + 1e-3


def test_smc_hmc_broken_phase_statistics():
    """C0-sized broken-phase run: SMC-HMC and the oracle's SMC-HMC agree on log Z and <|M|> within
    3 combined SE over 16 seeds, and HMC agrees with the RW kernel's log Z."""
    L, N, k = 4, 1024, 3
    g, gm, o, om, rw = [], [], [], [], []
    for s in range(16):
        _, lz, _, obs = smc_hmc_gpu(L, -4.0, 1.0, N, 700 + s, k, 0.5, 0.15, 10)
        g.append(lz); gm.append(obs["absM"])
        r = O.smc_hmc_run(L, -4.0, 1.0, N, 700 + s, k, 0.5, float(np.float32(0.15)), 10)
        o.append(r["logZ"]); om.append(np.abs(r["phi"].mean(axis=0)).mean())
        h = B.smc_init(L, -4.0, 1.0, N, 700 + s)
        B.smc_set_params(h, k_steps=10, ess_target=0.5)
        B.smc_run(h)
        rw.append(B.log_Z(h))
        h.close()
    g, gm, o, om, rw = map(np.array, (g, gm, o, om, rw))
    se = lambda a: a.std(ddof=1) / 4
    assert abs(g.mean() - o.mean()) < 3 * np.hypot(se(g), se(o))
    assert abs(gm.mean() - om.mean()) < 3 * np.hypot(se(gm), se(om))
    assert abs(g.mean() - rw.mean()) < 3 * np.hypot(se(g), se(rw)) + 0.02
