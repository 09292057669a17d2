"""GPU parity for the Z2 flip move (reading A17)."""
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


@pytest.mark.parametrize("L,N", [(4, 1024), (10, 5000), (3, 130)])
def test_flip_in_the_gather_is_bit_exact(L, N):
    seed = 77
    h = B.smc_init(L, -4.0, 1.0, N, seed)
    B.smc_set_params(h, z2_flip=1)
    before = B.smc_get_state(h)
    w = inputs.random_weights(N, 5)
    anc = B.smc_resample(h, w)
    assert np.array_equal(anc, O.resample_systematic(w, O.word0(seed, O.TAG_RESAMPLE, 0, 0)))
    ref, fl = O.z2_flip(before["phi"][:, anc].astype(np.float64), seed, 0)   # temperature index 0
    after = B.smc_get_state(h)
    assert 0.4 < fl.mean() < 0.6
    assert np.array_equal(after["phi"].astype(np.float64), ref)
    assert np.array_equal(after["S"], before["S"][anc]) and np.array_equal(after["U0"], before["U0"][anc])
    B.smc_set_params(h, z2_flip=0)                                           # and off again
    anc2 = B.smc_resample(h, w)
    assert np.array_equal(B.smc_get_state(h)["phi"], after["phi"][:, anc2])
    h.close()


def test_smc_runs_with_flips_match_the_oracle_distribution():
    L, N, k = 4, 2048, 10
    g, gb, gm = [], [], []
    for s in range(12):
        h = B.smc_init(L, -4.0, 1.0, N, 300 + s)
        B.smc_set_params(h, k_steps=k, z2_flip=1)
        B.smc_run(h)
        g.append(B.log_Z(h))
        M = B.smc_get_state(h)["phi"].mean(axis=0)
        gb.append(abs((M > 0).mean() - 0.5)); gm.append(np.abs(M).mean())
        h.close()
    o = [O.smc_run(L, -4.0, 1.0, N, 300 + s, k, z2_flip=True) for s in range(12)]
    lo = np.array([r["logZ"] for r in o]); g = np.array(g)
    se = lambda a: a.std(ddof=1) / math.sqrt(len(a))
    assert abs(g.mean() - lo.mean()) < 3 * math.hypot(se(g), se(lo))
    assert np.mean(gb) < 0.03                                # fair-coin noise over N is 0.011
    om = np.array([np.abs(r["phi"].mean(axis=0)).mean() for r in o])
    assert abs(np.mean(gm) - om.mean()) < 3 * math.hypot(se(np.array(gm)), se(om)) + 2e-3
