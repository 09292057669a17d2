"""GPU parity for the SMC-IRMH row (PAPER.md:53(ii), :200; reading A15): the CUDA
independent-MH path through the C ABI against the FP64 oracle on the same seeded inputs.

Tolerance.  An independent proposal is not a small perturbation: dS_E and dU0 are differences of
two full fp32 sums (2e-5 * A, reading A12) and the proposal-density terms 1/2 |z|^2, 1/2 |w|^2 are
O(V / 2).  Decisions are compared outside |g| < BAND_IRMH = 1e-3, margins within BAND_IRMH / 2 +
2e-5 |g| (an independent proposal far in the tail has |g| in the hundreds)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2511_15196_b200 import binding as B
from paper_2511_15196_b200 import build, inputs

pytestmark = pytest.mark.gpu

BAND_IRMH = 1e-3


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    B.load()


def irmh_lockstep(L, N, k, beta, seed, m0sq=-4.0, lam=1.0, t_start=0, fields="smooth"):
    h = B.smc_init(L, m0sq, lam, N, seed)
    B.smc_set_params(h, k_steps=k, kernel=2)
    if fields == "smooth":
        B.smc_set_state(h, inputs.smooth_fields(L, N, seed=seed + 1), beta, t_start)
    else:
        B.smc_set_state(h, B.smc_get_state(h)["phi"], beta, t_start)
    B.estimate_cov_chol(h)
    Lc, mu = B.smc_get_chol(h), B.smc_get_mean(h)
    st0 = B.smc_get_state(h)
    acc, mar = B.smc_mutate(h, k)
    st1 = B.smc_get_state(h)
    assert st1["step"] == t_start + k
    f0 = st0["phi"].astype(np.float64)
    S0, U00 = O.action_batch(f0, L, m0sq, lam)
    # the oracle is fed the GPU's factor and mean (reading R6: factor-level rounding must not leak
    # into decision parity); the mean itself is checked against the oracle's
    assert np.abs(mu - O.covariance(f0)[0]).max() < 1e-6
    p, S, U0, oacc, omar = O.irmh_mutate(f0, S0, U00, L, m0sq, lam, mu, Lc, beta, seed, t_start + 1, k)
    amb = np.abs(omar) < BAND_IRMH
    first = np.where(amb.any(axis=0), amb.argmax(axis=0), k)
    valid = np.arange(k)[:, None] < first[None, :]
    assert valid.mean() > 0.95
    assert np.array_equal(acc[valid], oacc[valid]), "IRMH accept decisions differ outside the band"
    d, go = np.abs(mar[valid] - omar[valid]), np.abs(omar[valid])
    assert np.all(d < 0.5 * BAND_IRMH + 2e-5 * go)
    clean = first == k
    assert np.abs(st1["phi"][:, clean] - p[:, clean]).max() < 2e-5
    Sx, Ux, A = O.action_batch(st1["phi"].astype(np.float64), L, m0sq, lam, with_abs=True)
    assert np.all(np.abs(st1["S"] - Sx) <= 4e-5 * A + 2e-5)
    assert np.all(np.abs(st1["U0"] - Ux) <= 4e-5 * Ux + 2e-5)
    h.close()
    return acc.mean()


@pytest.mark.parametrize("L,N,k,beta,fields", [
    (4, 1024, 6, 0.4, "init"), (10, 4096, 4, 0.3, "smooth"), (10, 1000, 3, 1.0, "smooth"),
    (5, 333, 5, 0.7, "smooth"), (1, 200, 6, 1.0, "init"), (2, 129, 6, 0.5, "init"),
    (9, 640, 3, 0.6, "smooth"), (16, 2048, 2, 0.2, "smooth"), (12, 700, 2, 0.1, "init"),
    (10, 16384, 2, 0.5, "smooth"), (3, 77, 4, 0.3, "init"), (7, 500, 3, 0.8, "smooth")])
def test_irmh_lockstep(L, N, k, beta, fields):
    rate = irmh_lockstep(L, N, k, beta, seed=53 + L, fields=fields, t_start=2 * k)
    assert 0.05 < rate < 1.0


def test_irmh_rejects_unsupported():
    h = B.smc_init(29, -4.0, 1.0, 256, 1)           # V = 841 > 800
    with pytest.raises(B.Phi4Error):
        B.smc_set_params(h, kernel=2)
    h.close()


def smc_irmh_gpu(L, m0sq, lam, N, seed, k, ess):
    h = B.smc_init(L, m0sq, lam, N, seed)
    B.smc_set_params(h, k_steps=k, ess_target=ess, kernel=2)
    T = B.smc_run(h)
    hist = B.smc_get_history(h)
    lz = B.log_Z(h)
    obs = B.observables(h)
    h.close()
    return T, lz, hist, obs


def test_smc_irmh_first_temperature_matches_oracle():
    L, N, k = 6, 2048, 3
    T, lz, hist, _ = smc_irmh_gpu(L, -4.0, 1.0, N, 5, k, 0.5)
    ref = O.smc_irmh_run(L, -4.0, 1.0, N, 5, k, 0.5)
    assert abs(hist[0]["beta"] - ref["info"][0, 0]) < 1e-5 * ref["info"][0, 0] + 1e-7
    assert abs(hist[0]["dlogZ"] - ref["info"][0, 3]) < 1e-4
    assert abs(hist[0]["accept_rate"] - ref["info"][0, 4]) < 0.01
    assert abs(T - ref["T"]) <= 2


def test_smc_irmh_gaussian_closed_form():
    """lambda = 0: log Z = -1/2 log det(I + K) (reading A1).  The fitted Gaussian is then the target
    itself up to estimation noise, so acceptance is high and the estimate tight."""
    L, N, k, m0sq = 4, 2048, 3, 0.5
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
    runs = [smc_irmh_gpu(L, m0sq, 0.0, N, 100 + s, k, 0.7) for s in range(16)]
    g = np.array([r[1] for r in runs])
    assert min(h["accept_rate"] for r in runs for h in r[2]) > 0.6
    o = np.array([O.smc_irmh_run(L, m0sq, 0.0, N, 100 + s, k, 0.7)["logZ"] for s in range(16)])
    se_g, se_o = g.std(ddof=1) / 4, o.std(ddof=1) / 4
    assert abs(g.mean() - exact) < 3 * se_g + 0.01
    assert abs(g.mean() - o.mean()) < 3 * np.hypot(se_g, se_o) + 1e-3


def test_smc_irmh_broken_phase_statistics():
    L, N, k = 4, 1024, 5
    g, gm, o, om = [], [], [], []
    for s in range(16):
        _, lz, _, obs = smc_irmh_gpu(L, -4.0, 1.0, N, 900 + s, k, 0.5)
        g.append(lz); gm.append(obs["absM"])
        r = O.smc_irmh_run(L, -4.0, 1.0, N, 900 + s, k, 0.5)
        o.append(r["logZ"]); om.append(np.abs(r["phi"].mean(axis=0)).mean())
    g, gm, o, om = map(np.array, (g, gm, o, om))
    se = lambda a: a.std(ddof=1) / 4
    assert abs(g.mean() - o.mean()) < 3 * np.hypot(se(g), se(o))
    assert abs(gm.mean() - om.mean()) < 3 * np.hypot(se(gm), se(om))
