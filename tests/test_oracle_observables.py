"""CPU pins of the oracle's observables (row O) and of the NS start-point rule (row N3).

Every expected value below is worked out by hand from the definitions the paper gives
(PAPER.md:37 magnetisation / susceptibility, :293 mode balance, :295 80-bin histogram) and
DESIGN.md readings A13 (fixed range [-1.6, 1.6], clamped) and A19 (weighted mode balance),
never from the oracle itself.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O

W = 3.2 / 80            # bin width of reading A13


def obs(M, S=None, logw=None, V=16):
    M = np.asarray(M, float)
    return O.observables_from_M(M, None if S is None else np.asarray(S, float),
                                None if logw is None else np.asarray(logw, float), V)


# ------------------------------------------------------------------ mode balance
def test_mode_balance_counts_positive_over_negative_and_ignores_zeros():
    assert obs([0.5, 0.2, -0.1, 0.0, 0.0])["mode_balance"] == pytest.approx(2.0, abs=1e-15)
    assert obs([0.3, -0.2, -0.9, -1.1, 0.0])["mode_balance"] == pytest.approx(1.0 / 3.0, abs=1e-15)


def test_mode_balance_no_negatives_is_inf_no_positives_is_zero():
    assert obs([0.5, 0.1, 0.0])["mode_balance"] == math.inf        # "+inf (all mass on the positive side)"
    assert obs([-0.5, -0.1, 0.0])["mode_balance"] == 0.0           # "0 (all mass on the negative side)"
    assert obs([0.0, 0.0])["mode_balance"] == math.inf             # no negative samples at all


def test_mode_balance_weighted_is_the_weight_mass_ratio():
    """Reading A19: with log-weights the count of a side is its weight mass.  Weights 3 : 1 : 2 on
    (+, -, +) give (3 + 2) / 1; a common shift of the log-weights changes nothing."""
    M = [0.4, -0.7, 1.0, 0.0]
    lw = np.log([3.0, 1.0, 2.0, 50.0])          # the zero sample is ignored whatever its weight
    assert obs(M, logw=lw)["mode_balance"] == pytest.approx(5.0, rel=1e-14)
    assert obs(M, logw=lw + 1234.5)["mode_balance"] == pytest.approx(5.0, rel=1e-12)
    # equal log-weights reproduce the unweighted count
    assert obs(M, logw=np.full(4, -7.0))["mode_balance"] == pytest.approx(2.0, rel=1e-14)


# ------------------------------------------------------------------ histogram (A13)
def test_histogram_bin_placement_every_bin_centre():
    """One sample at the centre of bin j, for every j: a shifted, mirrored or mis-scaled binning
    moves at least one of them."""
    for j in range(80):
        h = obs([-1.6 + W * (j + 0.5)])["hist"]
        want = np.zeros(80)
        want[j] = 1.0
        assert np.array_equal(h, want), j


def test_histogram_edges_zero_split_and_clamping():
    eps = 1e-9
    cases = [(-1.6, 0), (-1.6 + eps, 0), (-1.6 + W - eps, 0), (-1.6 + W + eps, 1),
             (-eps, 39), (eps, 40),                      # the bins split at zero magnetisation
             (1.6 - eps, 79), (1.6, 79), (1.6 + eps, 79),
             (-5.0, 0), (5.0, 79), (-1.6 - eps, 0)]      # out of range: clamped (A13)
    for m, b in cases:
        h = obs([m])["hist"]
        assert h[b] == 1.0 and h.sum() == 1.0, (m, b, int(np.argmax(h)))


def test_histogram_is_normalised_weight_mass_per_bin():
    M = [-1.0, -1.0, 0.5, 0.5, 0.5, 1.2]
    h = obs(M)["hist"]
    b = lambda m: int(math.floor((m + 1.6) / W))
    assert h[b(-1.0)] == pytest.approx(2 / 6) and h[b(0.5)] == pytest.approx(3 / 6)
    assert h[b(1.2)] == pytest.approx(1 / 6) and h.sum() == pytest.approx(1.0)
    # weighted: two distinct log-weights, shifted far from 0 (log-domain accumulation)
    lw = np.array([math.log(0.25), math.log(0.75)]) + 900.0
    h = obs([0.41, -0.79], logw=lw)["hist"]
    assert h[b(0.41)] == pytest.approx(0.25, rel=1e-12) and h[b(-0.79)] == pytest.approx(0.75, rel=1e-12)
    assert b(0.41) == 50 and b(-0.79) == 20


# ------------------------------------------------------------------ moments and chi
def test_moments_and_susceptibility_from_the_definition():
    """M = (1, -1, 1/2, -1/2): <|M|> = 3/4, <M^2> = 5/8, chi = V (<M^2> - <|M|>^2) = V / 16."""
    o = obs([1.0, -1.0, 0.5, -0.5], S=[1.0, 2.0, 3.0, 6.0], V=16)
    assert o["absM"] == pytest.approx(0.75, abs=1e-15)
    assert o["M2"] == pytest.approx(0.625, abs=1e-15)
    assert o["chi"] == pytest.approx(1.0, abs=1e-14)
    assert o["mean_SE"] == pytest.approx(3.0, abs=1e-15)
    assert obs([1.0, -1.0, 0.5, -0.5], V=100)["chi"] == pytest.approx(6.25, abs=1e-13)
    # a constant |M| has no fluctuation
    assert obs([0.3, -0.3, 0.3], V=49)["chi"] == pytest.approx(0.0, abs=1e-14)


def test_weighted_moments_two_log_weights():
    lw = np.array([math.log(0.25), math.log(0.75)]) - 300.0
    o = obs([0.4, -0.8], S=[2.0, 4.0], logw=lw, V=4)
    assert o["absM"] == pytest.approx(0.25 * 0.4 + 0.75 * 0.8, rel=1e-13)
    assert o["M2"] == pytest.approx(0.25 * 0.16 + 0.75 * 0.64, rel=1e-13)
    assert o["chi"] == pytest.approx(4 * (0.52 - 0.7 ** 2), rel=1e-12)
    assert o["mean_SE"] == pytest.approx(3.5, rel=1e-13)


def test_magnetisation_is_the_site_mean():
    phi = np.arange(12, dtype=float).reshape(4, 3)          # (V, N) site-major
    assert np.allclose(O.magnetisation(phi), [4.5, 5.5, 6.5], atol=1e-15)
    o = O.observables(phi - 5.5)                            # M = (-1, 0, 1)
    assert o["absM"] == pytest.approx(2 / 3) and o["mode_balance"] == pytest.approx(1.0)


# ------------------------------------------------------------------ NS start-point rule (R1, N3)
@pytest.mark.parametrize("seed", [0, 7])
def test_ns_start_points_replay_the_stream(seed):
    """First iteration of the oracle's NS run with a step scale so small that the walkers cannot
    leave their start points: the replacement of dead[j] must be the survivor number
    (word0 mod (n - k_del)) in index order, word0 from the draw (tag 4, t = iteration, slot j) --
    R1, PAPER.md:53(iv).  The stream itself is pinned by the published Philox vectors."""
    L, n, k = 3, 64, 16
    V = L * L
    phi0 = O.init_particles(seed, n, V)
    S0, _ = O.action_batch(phi0, L, -4.0, 1.0)
    # the k largest actions, S descending, ties by index (N1; the order is pinned in test_oracle_runs)
    order = sorted(range(n), key=lambda i: (-S0[i], i))
    dead = order[:k]
    surv = [i for i in range(n) if i not in set(dead)]
    r = O.ns_run(L, -4.0, 1.0, n, k, 3, seed, step_scale=1e-13, max_iter=1)
    assert r["iters"] == 1
    for j, d in enumerate(dead):
        src = surv[O.word0(seed, O.TAG_NS_START, 0, j) % (n - k)]
        assert np.abs(r["phi"][:, d] - phi0[:, src]).max() < 1e-10, (j, d, src)
    for i in surv:                                          # survivors are untouched
        assert np.array_equal(r["phi"][:, i], phi0[:, i])
    # and the dead log holds the deleted points in that order
    assert np.allclose(r["dead_S"], S0[dead], rtol=0, atol=1e-12)
    assert np.allclose(r["dead_M"], phi0[:, dead].mean(0), rtol=0, atol=1e-12)
