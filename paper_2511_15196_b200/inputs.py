"""Seeded synthetic workloads of the paper's shape (BASELINE.json configs) and input generators.

Holds none of the method's arithmetic: only parameter tables and plain numpy random draws that
both the CUDA path and the CPU oracle are fed with ("Input recipe").  The paper's
workload is itself synthetic -- a lattice model with parameters, no dataset.
"""
import numpy as np

# BASELINE.json configs[0..4]; all m0^2=-4, lambda=1, ESS target 0.5, s = 2.38/sqrt(V), fp32
CONFIGS = {
    "C0": dict(kind="smc", L=4, N=1024, k=10, m0sq=-4.0, lam=1.0, ess=0.5),
    "C0g": dict(kind="smc", L=4, N=1024, k=10, m0sq=1.0, lam=0.0, ess=0.5),   # Gaussian variant
    "C1": dict(kind="smc", L=10, N=16384, k=20, m0sq=-4.0, lam=1.0, ess=0.5),
    "C2": dict(kind="ns", L=10, n_live=4096, k_del=512, n_walk=25, m0sq=-4.0, lam=1.0,
               stop_frac=1e-3),
    "C3": dict(kind="smc", L=32, N=65536, k=20, m0sq=-4.0, lam=1.0, ess=0.5),
    "C4": dict(kind="smc", L=64, N=131072, k=10, m0sq=-4.0, lam=1.0, ess=0.5),
    # paper-scale settings (N = 5000, n_MCMC = 3V, ESS target 0.9; L in {10,15,18}
    # of :208, :236-242) -- a second workload whose wall-clock can be set beside Tables 1-3
    "P10": dict(kind="smc", L=10, N=5000, k=300, m0sq=-4.0, lam=1.0, ess=0.9),
    "P15": dict(kind="smc", L=15, N=5000, k=675, m0sq=-4.0, lam=1.0, ess=0.9),
    "P18": dict(kind="smc", L=18, N=5000, k=972, m0sq=-4.0, lam=1.0, ess=0.9),
    # the paper's ESS sweep (Table 3: ESS 0.90 / 0.99 / 0.999 with 5 V inner steps)
    "P10e99": dict(kind="smc", L=10, N=5000, k=500, m0sq=-4.0, lam=1.0, ess=0.99),
    "P10e999": dict(kind="smc", L=10, N=5000, k=500, m0sq=-4.0, lam=1.0, ess=0.999),
    # the paper's own nested-sampling setting: N = 5000 live points, delete
    # fraction 0.5, slice-sampling inner kernel, n_MCMC = 3 V slice steps per replacement
    "PNS10": dict(kind="ns", L=10, n_live=5000, k_del=2500, n_walk=300, inner="slice", m0sq=-4.0,
                  lam=1.0, stop_frac=1e-3),
}


def random_fields(V, N, seed, scale=1.0):
    """(V, N) fp32 site-major fields ~ N(0, scale^2): a stand-in particle cloud."""
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((V, N)) * scale).astype(np.float32)


def smooth_fields(L, N, seed, corr=0.6, scale=0.8):
    """Spatially correlated fields (nearest-neighbour averaging of white noise), closer to a
    mid-schedule particle cloud than white noise: non-trivial covariance for C1/C2 tests."""
    rng = np.random.default_rng(seed)
    f = rng.standard_normal((N, L, L))
    for _ in range(2):
        f = (1 - corr) * f + corr * 0.25 * (np.roll(f, 1, 1) + np.roll(f, -1, 1) +
                                            np.roll(f, 1, 2) + np.roll(f, -1, 2))
    f += rng.standard_normal((N, 1, 1)) * 0.5          # a magnetisation component
    return (scale * f.reshape(N, L * L).T).astype(np.float32).copy()


def synthetic_actions(N, seed, mean=0.0, std=1.0):
    """S_i ~ N(mean, std^2): with delta = 0.8326/std the weights have ESS/N = 0.5 in expectation
     -- realistic ancestor vectors for isolated resample / gather timing."""
    rng = np.random.default_rng(seed)
    return (mean + std * rng.standard_normal(N)).astype(np.float32)


def random_weights(N, seed, spread=2.0, zeros=0):
    """fp32 weights in [0,1] with max exactly 1 (the resampler's input contract, R5)."""
    rng = np.random.default_rng(seed)
    w = np.exp(-spread * rng.random(N) ** 2 * rng.exponential(1.0, N)).astype(np.float32)
    if zeros:
        w[rng.choice(N, zeros, replace=False)] = 0.0
    w[rng.integers(N)] = 1.0
    w = (w / w.max()).astype(np.float32)
    return w
