"""Pins of the oracle's Z2 flip move (NEXT row f4; reading A17)."""
import math

import numpy as np

from oracle import oracle as O


def test_flip_is_a_symmetry_and_a_fair_coin_from_the_documented_stream():
    L, V, N = 4, 16, 4000
    rng = np.random.default_rng(0)
    phi = rng.normal(size=(V, N))
    S, U0 = O.action_batch(phi, L, -4.0, 1.0)
    p, fl = O.z2_flip(phi, 9, 3)
    sign = np.where(fl.astype(bool), -1.0, 1.0)
    assert np.array_equal(p, phi * sign[None, :])
    S2, U2 = O.action_batch(p, L, -4.0, 1.0)
    assert np.array_equal(S2, S) and np.array_equal(U2, U0)       # even in phi, term by term
    assert abs(fl.mean() - 0.5) < 4 * 0.5 / math.sqrt(N)
    for j in (0, 17, 3999):
        assert fl[j] == O.word0(9, 8, 3, j) >> 31
    _, fl2 = O.z2_flip(phi, 9, 4)
    assert 0.4 < (fl != fl2).mean() < 0.6                         # a fresh coin every temperature


def test_smc_with_flips_balances_the_modes_and_keeps_logZ():
    L, N, k = 4, 2048, 10
    a = [O.smc_run(L, -4.0, 1.0, N, s, k) for s in range(8)]
    b = [O.smc_run(L, -4.0, 1.0, N, s, k, z2_flip=True) for s in range(8)]
    la, lb = np.array([r["logZ"] for r in a]), np.array([r["logZ"] for r in b])
    assert abs(la.mean() - lb.mean()) < 3 * math.hypot(la.std(ddof=1), lb.std(ddof=1)) / math.sqrt(8) + 0.02
    def imbalance(r):
        M = r["phi"].mean(axis=0)
        return abs((M > 0).mean() - 0.5)
    # binomial noise of a fair coin over N particles is 0.011; without flips the imbalance is
    # inherited from the resampling history and is several times larger on average
    assert np.mean([imbalance(r) for r in b]) < 0.03
    assert np.mean([imbalance(r) for r in b]) < np.mean([imbalance(r) for r in a])
    ma = np.mean([np.abs(r["phi"].mean(axis=0)).mean() for r in a])
    mb = np.mean([np.abs(r["phi"].mean(axis=0)).mean() for r in b])
    assert abs(ma - mb) < 0.02                                    # <|M|> is flip-invariant
