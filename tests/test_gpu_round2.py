"""GPU parity cases added in round 2: a strongly correlated factor at full size (paired-tile GEMM,
several accumulation chains), the cached S_E after whole runs, checkpoint / resume bit for bit,
the nested-sampling truncation status, host counters taken from the device, argument limits."""
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


# ---------------------------------------------------------------- correlated L_c at full size ---
@pytest.mark.parametrize("L,N,k,n_sub,path", [(32, 65536, 2, 192, 0), (40, 8192, 2, 128, 0), (64, 16384, 1, 64, 0),
                                              (40, 8192, 2, 128, 3), (64, 16384, 1, 64, 3)])
def test_full_size_correlated_factor(L, N, k, n_sub, path):
    """C3's and R40's launch shapes (more tiles than SMs: paired site tiles; K > 1024 at V = 1600
    and 4096: several TMEM accumulation chains) with a factor far from the identity: the particles
    are spatially correlated fields with a magnetisation component, so L_c is dense."""
    V, seed, m0sq, lam, beta = L * L, 3, -4.0, 1.0, 0.3
    rng = np.random.default_rng(77)
    # corr = 0.3: the smoothing filter's spectrum stays in [0.4, 1] (at the default 0.6 it crosses
    # zero between lattice momenta and the covariance is singular in fp32 for L >= 32)
    phi0 = inputs.smooth_fields(L, N, seed=5, corr=0.3)
    h = B.smc_init(L, m0sq, lam, N, seed)
    B.smc_set_params(h, k_steps=k, ess_target=0.5, mutation_path=path)   # 0: scaled 3xFP16, 3: 3xTF32
    B.smc_set_state(h, phi0, beta, 0)
    B.estimate_cov_chol(h)
    Sig, Lc = B.smc_get_cov(h), B.smc_get_chol(h)
    Ld = Lc.astype(np.float64)
    off = np.linalg.norm(Ld - np.diag(np.diag(Ld))) / np.linalg.norm(Ld)
    assert off > 0.5, off                                          # far from diagonal
    xs = np.sort(rng.choice(V, 40, replace=False))
    _, Sref = O.covariance(phi0[xs].astype(np.float64))
    assert np.linalg.norm(Sig[np.ix_(xs, xs)] - Sref) / np.linalg.norm(Sref) < 1e-5
    assert np.linalg.norm(Ld @ Ld.T - Sig) / np.linalg.norm(Sig) < 1e-5            # R6
    sub = np.sort(rng.choice(N, n_sub, replace=False)).astype(np.int32)
    acc, mar = B.smc_mutate(h, k)
    st1 = B.smc_get_state(h)
    S0, U0 = O.action_batch(phi0[:, sub].astype(np.float64), L, m0sq, lam)
    p, S_o, U_o, oacc, omar, _ = O.mutate(phi0[:, sub], S0, U0, L, m0sq, lam, Lc,
                                          np.float32(2.38 / math.sqrt(V)), beta, seed, 1, k, slots=sub)
    amb = np.abs(omar) < 1e-4
    first = np.where(amb.any(axis=0), amb.argmax(axis=0), k)
    valid = np.arange(k)[:, None] < first[None, :]
    assert valid.mean() > 0.97
    assert np.array_equal(acc[:, sub][valid], oacc[valid])
    err = np.abs(mar[:, sub][valid] - omar[valid]) - 1e-5 * np.abs(omar[valid])
    print("correlated L=%d path %d: worst margin error %.3g (band 1e-4), off-diagonal weight %.2f, accept %.3f"
          % (L, path, err.max(), off, acc.mean()))
    assert err.max() < 1e-4 * max(1.0, math.sqrt(V / 100.0))
    clean = first == k
    assert np.abs(st1["phi"][:, sub][:, clean] - p[:, clean]).max() < 2e-5
    assert 0.0 < acc.mean() < 1.0
    h.close()


# ---------------------------------------------------------------- cached S_E after whole runs ---
@pytest.mark.parametrize("name,max_temps,n_sub", [("C1", 4096, 16384), ("C3", 24, 512)])
def test_cached_action_after_whole_run(name, max_temps, n_sub):
    """The weights of P1 / P2 are formed from the cached S_E, which is updated incrementally
    (S += dS) k times per temperature and carried through every gather.  After a whole C1 run
    (14 temperatures x 20 steps) and after 24 temperatures x 20 steps at C3 it must still agree
    with the FP64 action of the particles within reading A12's 2e-5 A + 2e-5."""
    c = inputs.CONFIGS[name]
    L, N = c["L"], c["N"]
    h = B.smc_init(L, c["m0sq"], c["lam"], N, 2)
    B.smc_set_params(h, k_steps=c["k"], ess_target=c["ess"])
    T = B.smc_run(h, max_temps)
    st = B.smc_get_state(h)
    sub = np.sort(np.random.default_rng(1).choice(N, n_sub, replace=False))
    S, U, A = O.action_batch(st["phi"][:, sub].astype(np.float64), L, c["m0sq"], c["lam"], with_abs=True)
    eS = np.abs(st["S"][sub] - S)
    eU = np.abs(st["U0"][sub] - U)
    print("%s after %d temperatures: worst |S_cached - S| = %.3g (%.3g of 2e-5 A + 2e-5), worst |U0| error %.3g"
          % (name, T, eS.max(), (eS / (2e-5 * A + 2e-5)).max(), eU.max()))
    assert np.all(eS <= 2e-5 * A + 2e-5)
    assert np.all(eU <= 2e-5 * U + 2e-5)
    assert st["step"] == T * c["k"]
    h.close()


# ---------------------------------------------------------------- checkpoint / resume -----------
def test_smc_checkpoint_resume_is_bit_exact():
    L, N, k, seed = 6, 2000, 8, 9
    ref = B.smc_init(L, -4.0, 1.0, N, seed)
    B.smc_set_params(ref, k_steps=k, ess_target=0.5, z2_flip=1)
    B.smc_run(ref, 3)
    st, rs = B.smc_get_state(ref), B.smc_get_run_state(ref)
    assert rs["index"] == 3 and rs["step_counter"] == 3 * k and rs["beta"] == st["beta"]
    T_rest = B.smc_run(ref)
    want = B.smc_get_state(ref)
    # a fresh handle with another seed's particles, restored from the checkpoint
    h = B.smc_init(L, -4.0, 1.0, N, seed)
    B.smc_set_params(h, k_steps=k, ess_target=0.5, z2_flip=1)
    B.smc_run(h, 1)
    B.smc_restore(h, st["phi"], st["S"], st["U0"], rs)
    assert B.smc_get_run_state(h) == rs
    assert B.smc_run(h) == T_rest
    got = B.smc_get_state(h)
    assert np.array_equal(got["phi"], want["phi"]) and np.array_equal(got["S"], want["S"])
    assert B.log_Z(h) == B.log_Z(ref) and got["step"] == want["step"]
    assert [x["beta"] for x in B.smc_get_history(h)][3:] == [x["beta"] for x in B.smc_get_history(ref)][3:]
    h.close()
    ref.close()


def test_ns_checkpoint_resume_is_bit_exact():
    L, n, kd, nw, seed = 4, 512, 64, 6, 4
    ref = B.ns_init(L, -4.0, 1.0, n, kd, nw, seed, max_iters=512)
    B.ns_run(ref, 5)
    st, rs, dead = B.smc_get_state(ref), B.smc_get_run_state(ref), B.ns_get_dead(ref)
    assert rs["index"] == 5 and rs["step_counter"] == 5 * nw
    it_rest = B.ns_run(ref)
    assert not ref.truncated
    h = B.ns_init(L, -4.0, 1.0, n, kd, nw, seed, max_iters=512)
    B.smc_restore(h, st["phi"], st["S"], st["U0"], rs)
    B.ns_set_dead(h, dead["dead_S"], dead["dead_M"], dead["dead_logw"])
    assert B.ns_run(h) == it_rest
    assert B.log_Z(h) == B.log_Z(ref)
    assert np.array_equal(B.smc_get_state(h)["phi"], B.smc_get_state(ref)["phi"])
    oa, ob = B.observables(h), B.observables(ref)
    # (the histogram is accumulated with shared-memory atomics: its sums are order-dependent at 1e-17)
    assert oa["absM"] == ob["absM"] and np.allclose(oa["hist"], ob["hist"], rtol=0, atol=1e-14)
    h.close()
    ref.close()


# ---------------------------------------------------------------- NS truncation ------------------
def test_ns_truncation_is_reported():
    """max_iters smaller than the natural iteration count: the run stops with PHI4_ETRUNC, done = 2,
    and log_Z() is the dead-point evidence alone -- exactly what the oracle returns at its cap."""
    L, n, kd, nw, seed, cap = 4, 512, 64, 6, 1, 7
    h = B.ns_init(L, -4.0, 1.0, n, kd, nw, seed, max_iters=cap)
    it = B.ns_run(h)
    assert it == cap and h.truncated
    info = B.ns_step(h)                                   # no-op; reports the state
    assert info["done"] == 2 and info["iter_index"] == cap - 1
    dead = B.ns_get_dead(h)
    from scipy.special import logsumexp
    lz_dead = logsumexp(dead["dead_logw"] - dead["dead_S"].astype(np.float64))
    assert B.log_Z(h) == pytest.approx(lz_dead, rel=1e-10)
    assert info["remaining_frac"] > 1e-3
    o = O.ns_run(L, -4.0, 1.0, n, kd, nw, seed, max_iter=cap)
    assert o["iters"] == cap and abs(o["logZ"] - B.log_Z(h)) < 0.5      # same estimator, own walks
    h.close()
    # a run that converges inside its cap is not truncated
    h = B.ns_init(L, -4.0, 1.0, n, kd, nw, seed, max_iters=512)
    B.ns_run(h)
    assert not h.truncated and B.ns_step(h)["done"] == 1
    h.close()


# ---------------------------------------------------------------- host counters -----------------
def test_enqueue_only_steps_past_the_end_do_not_inflate_the_counter():
    L, N, k = 4, 1024, 10
    ref = B.smc_init(L, -4.0, 1.0, N, 5)
    B.smc_set_params(ref, k_steps=k, ess_target=0.5)
    T = B.smc_run(ref)
    h = B.smc_init(L, -4.0, 1.0, N, 5)
    B.smc_set_params(h, k_steps=k, ess_target=0.5)
    for _ in range(T + 6):                                 # enqueue only, six steps past beta = 1
        B.smc_step(h, want_info=False)
    st = B.smc_get_state(h)
    assert st["beta"] == 1.0 and st["step"] == T * k
    assert np.array_equal(st["phi"], B.smc_get_state(ref)["phi"])
    info = B.smc_step(h)
    assert info["done"] and info["temp_index"] == T - 1
    acc, _ = B.smc_mutate(h, 2)                            # continues at T k + 1
    assert B.smc_get_state(h, want_phi=False)["step"] == T * k + 2
    h.close()
    ref.close()


def test_argument_limits():
    assert B.smc_workspace_bytes(256, 1024) == 0 and B.smc_workspace_bytes(255, 1024) > 0
    assert B.ns_workspace_bytes(256, 1024, 128, 8) == 0
    with pytest.raises(B.Phi4Error):
        B.smc_init(4, float("inf"), 1.0, 256, 0)
    with pytest.raises(B.Phi4Error):
        B.smc_init(4, -4.0, float("nan"), 256, 0)
    with pytest.raises(B.Phi4Error):
        B.smc_init_kl(4, float("inf"), 0.5, 256, 0)
    with pytest.raises(B.Phi4Error):
        B.ns_init_kl(4, float("inf"), 0.5, 256, 32, 4, 0)


# ---------------------------------------------------------------- NS at the paper's settings ----
def test_ns_paper_setting_first_iteration_lockstep():
    """N = 5000 live points, delete fraction 0.5 (2500 deletions per iteration,
    more dead points than one CTA has threads), slice-sampling inner kernel (reading A16)."""
    c = inputs.CONFIGS["PNS10"]
    L, n, kd, nw, seed = c["L"], c["n_live"], c["k_del"], 4, 17
    h = B.ns_init(L, c["m0sq"], c["lam"], n, kd, nw, seed, max_iters=8)
    B.ns_set_params(h, inner=1)
    st0 = B.smc_get_state(h)
    info = B.ns_step(h)
    S0 = st0["S"].astype(np.float64)
    dead = O.ns_select(S0, kd)
    got = B.ns_get_dead(h)
    assert np.array_equal(got["last_dead"], dead)                             # N1 exact
    assert info["S_star"] == S0[dead[-1]]
    lw = np.array([-sum(1.0 / (n - m + 1) for m in range(1, j)) +
                   math.log1p(-math.exp(-1.0 / (n - j + 1))) for j in range(1, kd + 1)])
    assert np.allclose(got["dead_logw"], lw, rtol=1e-12, atol=1e-14)          # N2, reading A6
    from scipy.special import logsumexp
    assert info["logZ"] == pytest.approx(logsumexp(lw - S0[dead]), rel=1e-10)
    assert info["logX"] == pytest.approx(-sum(1.0 / (n - j + 1) for j in range(1, kd + 1)), rel=1e-12)
    # N3: slice walks replayed by the oracle from the GPU's start state and factor
    Lc = B.smc_get_chol(h)
    surv = np.setdiff1d(np.arange(n), dead)
    start = np.array([surv[O.word0(seed, O.TAG_NS_START, 0, j) % (n - kd)] for j in range(kd)])
    f0 = st0["phi"][:, start].astype(np.float64)
    Ss, Us = O.action_batch(f0, L, c["m0sq"], c["lam"])
    p, S, U0, t, nexp, nshr, amb = O.slice_walk(f0, Ss, Us, L, c["m0sq"], c["lam"], Lc, info["S_star"],
                                                seed, 1, nw, width=np.float32(1.0), m_expand=8)
    st1 = B.smc_get_state(h)
    clean = amb.min(axis=0) > 2e-3
    assert clean.mean() > 0.6
    assert np.abs(st1["phi"][:, dead][:, clean] - p[:, clean]).max() < 1e-4
    assert np.array_equal(st1["phi"][:, surv], st0["phi"][:, surv])           # survivors untouched
    assert np.all(st1["S"] < info["S_star"] + 1e-3)
    h.close()


@pytest.mark.parametrize("L,n,kd,nw", [(16, 32768, 16384, 3), (12, 2048, 1024, 4)])
def test_ns_large_v_walk_lockstep(L, n, kd, nw):
    """Constrained RW walks at V > 112: the walkers go through the tcgen05 proposal GEMM (FP16 operands), and
    with 16384 walkers x 256 sites the GEMM of a step also draws the next step's normals (NS tags, walker
    slots); the second case takes a kernel of its own for them.  First iteration against the oracle."""
    seed, m0sq, lam = 23, -4.0, 1.0
    h = B.ns_init(L, m0sq, lam, n, kd, nw, seed, max_iters=4)
    st0 = B.smc_get_state(h)
    info = B.ns_step(h)
    S0 = st0["S"].astype(np.float64)
    dead = O.ns_select(S0, kd)
    assert np.array_equal(B.ns_get_dead(h)["last_dead"], dead)
    Lc = B.smc_get_chol(h)
    surv = np.setdiff1d(np.arange(n), dead)
    start = np.array([surv[O.word0(seed, O.TAG_NS_START, 0, j) % (n - kd)] for j in range(kd)])
    sub = np.sort(np.random.default_rng(5).choice(kd, 256, replace=False)).astype(np.int32)
    f0 = st0["phi"][:, start[sub]].astype(np.float64)
    Ss, Us = O.action_batch(f0, L, m0sq, lam)
    p, S, U0, oacc, omar, cmar = O.mutate(f0, Ss, Us, L, m0sq, lam, Lc, np.float32(2.38 / math.sqrt(L * L)), 0.0,
                                          seed, 1, nw, mode=O.MODE_NS, S_star=info["S_star"], slots=sub)
    amb = np.minimum(np.abs(omar), np.abs(cmar)) < 1e-4
    clean = ~amb.any(axis=0)
    assert clean.mean() > 0.9
    st1 = B.smc_get_state(h)
    got = st1["phi"][:, dead[sub]]
    assert np.abs(got[:, clean] - p[:, clean]).max() < 2e-5
    assert np.array_equal(st1["phi"][:, surv], st0["phi"][:, surv])
    assert np.all(st1["S"] < info["S_star"] + 1e-3) and 0.0 < oacc.mean() < 1.0
    h.close()


def test_ns_paper_setting_statistical_parity():
    """N = 5000, delete fraction 0.5, slice kernel (10 slice steps per replacement instead of 3 V,
    so that eight oracle runs stay affordable): log Z and iterations within 3 combined SE."""
    c = inputs.CONFIGS["PNS10"]
    L, n, kd, nw = c["L"], c["n_live"], c["k_del"], 10

    def gpu(seed):
        h = B.ns_init(L, c["m0sq"], c["lam"], n, kd, nw, seed, max_iters=512)
        B.ns_set_params(h, inner=1)
        it = B.ns_run(h)
        out = (B.log_Z(h), it, B.observables(h)["absM"])
        h.close()
        return out
    g = [gpu(s) for s in range(8)]
    o = [O.ns_run(L, c["m0sq"], c["lam"], n, kd, nw, s, inner="slice") for s in range(8)]
    for key, a, b in (("logZ", [x[0] for x in g], [r["logZ"] for r in o]),
                      ("iters", [x[1] for x in g], [r["iters"] for r in o])):
        a, b = np.asarray(a, float), np.asarray(b, float)
        se = math.hypot(a.std(ddof=1), b.std(ddof=1)) / math.sqrt(8)
        print("PNS10 %s: gpu %.4f oracle %.4f (%.2f combined SE)" % (key, a.mean(), b.mean(),
                                                                    abs(a.mean() - b.mean()) / max(se, 1e-12)))
        assert abs(a.mean() - b.mean()) < 3 * se + (0.5 if key == "iters" else 0.0)


@pytest.mark.parametrize("n,kd", [(40000, 20000), (70000, 1000)])
def test_ns_select_beyond_one_cta(n, kd):
    """More than 16384 live points: the multi-block bitonic network orders the keys; dead list,
    threshold, evidence and start points are still exact."""
    L, nw, seed = 4, 2, 3
    h = B.ns_init(L, -4.0, 1.0, n, kd, nw, seed, max_iters=4)
    st0 = B.smc_get_state(h)
    info = B.ns_step(h)
    S0 = st0["S"].astype(np.float64)
    dead = O.ns_select(S0, kd)
    got = B.ns_get_dead(h)
    assert np.array_equal(got["last_dead"], dead)
    assert info["S_star"] == S0[dead[-1]]
    assert np.array_equal(got["dead_S"], st0["S"][dead])
    st1 = B.smc_get_state(h)
    surv = np.setdiff1d(np.arange(n), dead)
    assert np.array_equal(st1["phi"][:, surv], st0["phi"][:, surv])
    assert np.all(st1["S"] < info["S_star"] + 1e-3)
    # walkers that did not move (2 steps only) sit exactly on their start points: the rule of R1
    start = np.array([surv[O.word0(seed, O.TAG_NS_START, 0, j) % (n - kd)] for j in range(0, kd, 97)])
    moved = 0
    for j, s in zip(range(0, kd, 97), start):
        if not np.array_equal(st1["phi"][:, dead[j]], st0["phi"][:, s]):
            moved += 1
    assert moved < len(start)                     # some walkers stay; the others have moved off
    h.close()
