"""phi4_resample_noalloc: the no-allocation entry point (scratch in a file-scope __device__ array)
against the existing handle-based path smc_resample, on two calls in a row.  Integer work: the
ancestors must agree bit for bit (the tolerance the other resampling tests use).  Collected last
(file name) so that a failure here cannot hide another test under `pytest -x`."""
import numpy as np
import pytest

from paper_2511_15196_b200 import binding as B
from paper_2511_15196_b200 import build, inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    B.load()


def existing_path(w, seed):
    """Ancestors of the handle-based resampler (temperature index 0 of a fresh handle)."""
    h = B.smc_init(4, -4.0, 1.0, w.size, seed)
    anc = B.smc_resample(h, w)
    h.close()
    return anc


def test_noalloc_resample_matches_existing_path_two_calls_in_a_row():
    import torch
    from oracle import oracle as O
    seed = 21
    assert B.load().phi4_noalloc_setup() == 0
    # call 1: more than 32768 weights (multi-block scan, block sums in the scratch), some exact zeros;
    # call 2: fewer, ragged -- the array still holds call 1's CDF beyond entry N and must not matter;
    # call 3: the first again: same answer as before
    cases = [inputs.random_weights(100000, 5, zeros=1000), inputs.random_weights(5001, 6),
             inputs.random_weights(100000, 5, zeros=1000)]
    out = torch.full((B.NOALLOC_MAX_N,), -7, dtype=torch.int32, device="cuda:0")
    free0 = torch.cuda.mem_get_info(0)[0]
    got = []
    for w in cases:
        wd = torch.from_numpy(w).to("cuda:0")
        out.fill_(-7)
        B.phi4_resample_noalloc(wd, seed, 0, out)
        torch.cuda.synchronize()
        got.append(out[:w.size].cpu().numpy())
        assert int(out[w.size:].max()) == -7 and int(out[w.size:].min()) == -7   # nothing written past N
    assert torch.cuda.mem_get_info(0)[0] >= free0 - (1 << 20)       # the calls did not grow device memory
    for w, a in zip(cases, got):
        assert np.array_equal(a, existing_path(w, seed))             # bit-exact vs smc_resample
        assert np.array_equal(a, O.resample_systematic(w, O.word0(seed, O.TAG_RESAMPLE, 0, 0)))
    assert np.array_equal(got[0], got[2])
    # another step index keys another offset U (reading R1): checked against the oracle
    w = cases[1]
    B.phi4_resample_noalloc(torch.from_numpy(w).to("cuda:0"), seed, 3, out)
    torch.cuda.synchronize()
    assert np.array_equal(out[:w.size].cpu().numpy(),
                          O.resample_systematic(w, O.word0(seed, O.TAG_RESAMPLE, 3, 0)))


def test_noalloc_rejects_sizes_beyond_its_capacity():
    import torch
    n = B.NOALLOC_MAX_N + 1
    w = torch.ones(n, dtype=torch.float32, device="cuda:0")
    out = torch.full((n,), -7, dtype=torch.int32, device="cuda:0")
    with pytest.raises(B.Phi4Error) as e:
        B.phi4_resample_noalloc(w, 0, 0, out)
    assert e.value.code == -7 and "capacity" in str(e.value)
    torch.cuda.synchronize()
    assert int(out.max()) == -7                                      # nothing was enqueued
    # the largest admissible size works
    B.phi4_resample_noalloc(w[:B.NOALLOC_MAX_N], 0, 0, out)
    torch.cuda.synchronize()
    assert np.array_equal(out[:B.NOALLOC_MAX_N].cpu().numpy(), np.arange(B.NOALLOC_MAX_N))  # equal weights
