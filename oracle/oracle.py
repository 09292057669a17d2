"""ctypes binding of the FP64 CPU oracle (oracle_phi4.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
shares nothing with paper_2511_15196_b200 and never imports it.

All arrays are numpy float64, particles site-major ``phi[x, i]`` (shape (V, N),
C-contiguous), exactly the layout of oracle_phi4.c.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_phi4.c")
_LIB = os.path.join(_HERE, "liboracle_phi4.so")

TAG_INIT, TAG_PROP, TAG_ACC, TAG_RESAMPLE, TAG_NS_START, TAG_NS_PROP, TAG_NS_ACC = range(7)
MODE_SMC, MODE_NS = 0, 1


def build(force=False):
    """gcc -O2 -fopenmp oracle_phi4.c -> liboracle_phi4.so (in oracle/)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".%d.tmp" % os.getpid()
    subprocess.check_call(["gcc", "-O2", "-std=gnu99", "-fopenmp", "-fPIC", "-shared",
                           "-o", tmp, _SRC, "-lm"])
    os.replace(tmp, _LIB)
    return _LIB


_lib = None
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_fp = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_u8p = np.ctypeslib.ndpointer(dtype=np.uint8, flags="C_CONTIGUOUS")
_u32p = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    vp = C.c_void_p
    sig = {
        "orc_num_threads": (C.c_int, []),
        "orc_philox4x32_10": (None, [_u32p, _u32p, _u32p]),
        "orc_normals": (None, [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_int, _dp]),
        "orc_uniform": (C.c_double, [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]),
        "orc_word0": (C.c_uint32, [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]),
        "orc_action_field": (C.c_double, [_dp, C.c_int, C.c_double, C.c_double, vp]),
        "orc_set_kinetic": (None, [C.c_double]),
        "orc_get_kinetic": (C.c_double, []),
        "orc_action_eq2_field": (C.c_double, [_dp, C.c_int, C.c_double, C.c_double]),
        "orc_u0_field": (C.c_double, [_dp, C.c_int]),
        "orc_action_grad_field": (None, [_dp, C.c_int, C.c_double, C.c_double, _dp]),
        "orc_action_batch": (None, [_dp, C.c_int, C.c_int, C.c_double, C.c_double, _dp, _dp, vp]),
        "orc_init_particles": (None, [C.c_uint64, C.c_int, C.c_int, _dp]),
        "orc_mutate": (None, [_dp, _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, _dp,
                              C.c_double, C.c_double, C.c_int, C.c_double, C.c_uint64,
                              C.c_uint32, C.c_uint32, C.c_uint32, C.c_int, vp, vp, vp, vp]),
        "orc_lse_neg": (C.c_double, [_dp, C.c_int, C.c_double]),
        "orc_ess_frac": (C.c_double, [_dp, C.c_int, C.c_double]),
        "orc_next_delta": (C.c_double, [_dp, C.c_int, C.c_double, C.c_double, C.POINTER(C.c_int)]),
        "orc_reweight": (C.c_double, [_dp, C.c_int, C.c_double, vp]),
        "orc_resample_systematic": (C.c_int, [_fp, C.c_int, C.c_uint32, _ip]),
        "orc_gather": (None, [_dp, C.c_int, C.c_int, _ip, _dp]),
        "orc_covariance": (None, [_dp, C.c_int, C.c_int, _dp, _dp]),
        "orc_cholesky": (C.c_int, [_dp, C.c_int, _dp]),
        "orc_cov_chol": (C.c_int, [_dp, C.c_int, C.c_int, _dp, _dp]),
        "orc_magnetisation": (None, [_dp, C.c_int, C.c_int, _dp]),
        "orc_observables_from_M": (None, [_dp, vp, vp, C.c_int, C.c_int, _dp]),
        "orc_observables": (None, [_dp, vp, C.c_int, C.c_int, _dp]),
        "orc_smc_run": (C.c_int, [C.c_int, C.c_double, C.c_double, C.c_int, C.c_uint64, C.c_int,
                                  C.c_double, C.c_double, C.c_int, _dp, _dp, _dp,
                                  C.POINTER(C.c_double), vp]),
        "orc_hmc_mutate": (None, [_dp, _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, _dp,
                                  C.c_double, C.c_int, C.c_double, C.c_uint64, C.c_uint32, C.c_int,
                                  vp, vp, vp]),
        "orc_leapfrog": (C.c_double, [_dp, _dp, C.c_int, C.c_double, C.c_double, _dp, C.c_double,
                                      C.c_int, C.c_double]),
        "orc_smc_hmc_run": (C.c_int, [C.c_int, C.c_double, C.c_double, C.c_int, C.c_uint64, C.c_int,
                                      C.c_double, C.c_double, C.c_int, C.c_int, _dp, _dp, _dp,
                                      C.POINTER(C.c_double), vp]),
        "orc_ns_run_inner": (C.c_int, [C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int,
                                       C.c_uint64, C.c_double, C.c_double, C.c_int, C.c_int,
                                       C.c_double, C.c_int, C.c_int, _dp, _dp, _dp,
                                       C.POINTER(C.c_double), C.POINTER(C.c_double), vp, vp, vp, vp]),
        "orc_slice_walk": (None, [_dp, _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, _dp,
                                  C.c_double, C.c_int, C.c_int, C.c_double, C.c_uint64, C.c_uint32,
                                  C.c_int, vp, vp, vp, vp, vp]),
        "orc_z2_flip": (None, [_dp, C.c_int, C.c_int, C.c_uint64, C.c_uint32, vp]),
        "orc_smc_run_z2": (C.c_int, [C.c_int, C.c_double, C.c_double, C.c_int, C.c_uint64, C.c_int,
                                     C.c_double, C.c_double, C.c_int, _dp, _dp, _dp,
                                     C.POINTER(C.c_double), vp]),
        "orc_irmh_mutate": (None, [_dp, _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, _dp, _dp,
                                   C.c_double, C.c_uint64, C.c_uint32, C.c_int, vp, vp, vp]),
        "orc_smc_irmh_run": (C.c_int, [C.c_int, C.c_double, C.c_double, C.c_int, C.c_uint64, C.c_int,
                                       C.c_double, C.c_int, _dp, _dp, _dp, C.POINTER(C.c_double), vp]),
        "orc_ns_select": (None, [_dp, C.c_int, C.c_int, _ip]),
        "orc_ns_run": (C.c_int, [C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int,
                                 C.c_uint64, C.c_double, C.c_double, C.c_int, _dp, _dp, _dp,
                                 C.POINTER(C.c_double), C.POINTER(C.c_double), vp, vp, vp, vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype = res
        f.argtypes = args
    _lib = L
    return L


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads():
    return lib().orc_num_threads()


def philox(ctr, key):
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(np.asarray(ctr, np.uint32), np.asarray(key, np.uint32), out)
    return out


def draw(seed, tag, t, i, q):
    """The four raw words of the R1 draw (c0, c1, c2, c3) = (q, i, t, tag) under key seed."""
    return [int(v) for v in philox([q, i, t, tag], [seed & 0xFFFFFFFF, seed >> 32])]


def normals(seed, tag, t, i, V):
    z = np.zeros(V)
    lib().orc_normals(seed, tag, t, i, V, z)
    return z


def uniform(seed, tag, t, i):
    return lib().orc_uniform(seed, tag, t, i)


def word0(seed, tag, t, i):
    return lib().orc_word0(seed, tag, t, i)


def action_field(f, L, m0sq, lam, with_abs=False):
    f = _f64(f).reshape(-1)
    a = C.c_double(0.0)
    s = lib().orc_action_field(f, L, m0sq, lam, C.cast(C.byref(a), C.c_void_p))
    return (s, a.value) if with_abs else s


class kinetic:
    """`with kinetic(kappa):` -- every oracle call inside evaluates Eq. 1 with its kinetic term
    multiplied by kappa (Eq. 2; reading A18).  Restores the previous value."""

    def __init__(self, kappa):
        self.kappa = float(kappa)

    def __enter__(self):
        self.prev = lib().orc_get_kinetic()
        lib().orc_set_kinetic(self.kappa)
        return self

    def __exit__(self, *exc):
        lib().orc_set_kinetic(self.prev)
        return False


def kl_to_eq1(kappa, lam):
    """Eq. 2's (kappa, lambda) as Eq. 1 coefficients (Eq. 4): (kinetic, m0sq, lambda) and the
    constant V*lambda per site that Eq. 5 drops (returned per site)."""
    return float(kappa), 2.0 * (1.0 - 2.0 * lam), float(lam), float(lam)


def action_eq2_field(f, L, kappa, lam):
    """Eq. 2 verbatim, constant included."""
    f = _f64(f).reshape(-1)
    return lib().orc_action_eq2_field(f, L, kappa, lam)


def u0_field(f):
    f = _f64(f).reshape(-1)
    return lib().orc_u0_field(f, f.size)


def action_grad_field(f, L, m0sq, lam):
    f = _f64(f).reshape(-1)
    g = np.zeros_like(f)
    lib().orc_action_grad_field(f, L, m0sq, lam, g)
    return g


def action_batch(phi, L, m0sq, lam, with_abs=False):
    phi = _f64(phi)
    V, N = phi.shape
    assert V == L * L
    S, U0 = np.zeros(N), np.zeros(N)
    A = np.zeros(N) if with_abs else None
    lib().orc_action_batch(phi, N, L, m0sq, lam, S, U0, _ptr(A))
    return (S, U0, A) if with_abs else (S, U0)


def init_particles(seed, N, V):
    phi = np.zeros((V, N))
    lib().orc_init_particles(seed, N, V, phi)
    return phi


def mutate(phi, S, U0, L, m0sq, lam, Lc, s, beta, seed, t0, k, mode=MODE_SMC, S_star=0.0,
           tag_prop=None, tag_acc=None, slots=None):
    """k RW-Metropolis steps in place on copies; returns (phi, S, U0, accept[k,N], margin[k,N],
    cmargin[k,N]).  slots: optional Philox slot of each column (default: column index)."""
    phi, S, U0 = _f64(phi).copy(), _f64(S).copy(), _f64(U0).copy()
    V, N = phi.shape
    if tag_prop is None:
        tag_prop = TAG_PROP if mode == MODE_SMC else TAG_NS_PROP
    if tag_acc is None:
        tag_acc = TAG_ACC if mode == MODE_SMC else TAG_NS_ACC
    if slots is not None:
        slots = np.ascontiguousarray(slots, np.int32)
        assert slots.shape == (N,)
    acc = np.zeros((k, N), np.uint8)
    mar = np.zeros((k, N))
    cmar = np.zeros((k, N))
    lib().orc_mutate(phi, S, U0, N, L, m0sq, lam, _f64(Lc), s, beta, mode, S_star, seed,
                     tag_prop, tag_acc, t0, k, _ptr(acc), _ptr(mar), _ptr(cmar), _ptr(slots))
    return phi, S, U0, acc, mar, cmar


def ess_frac(S, delta):
    S = _f64(S)
    return lib().orc_ess_frac(S, S.size, delta)


def next_delta(S, beta, target):
    S = _f64(S)
    fin = C.c_int(0)
    d = lib().orc_next_delta(S, S.size, beta, target, C.byref(fin))
    return d, bool(fin.value)


def reweight(S, delta):
    S = _f64(S)
    w = np.zeros(S.size, np.float32)
    dlz = lib().orc_reweight(S, S.size, delta, _ptr(w))
    return w, dlz


def resample_systematic(w, U):
    w = np.ascontiguousarray(w, np.float32)
    anc = np.zeros(w.size, np.int32)
    rc = lib().orc_resample_systematic(w, w.size, int(U), anc)
    if rc != 0:
        raise ValueError("all weights quantise to zero")
    return anc


def gather(a, anc):
    a = _f64(a)
    a2 = a.reshape(-1, a.shape[-1])
    out = np.zeros_like(a2)
    lib().orc_gather(a2, a2.shape[1], a2.shape[0], np.ascontiguousarray(anc, np.int32), out)
    return out.reshape(a.shape)


def covariance(phi):
    phi = _f64(phi)
    V, N = phi.shape
    mu, Sig = np.zeros(V), np.zeros((V, V))
    lib().orc_covariance(phi, N, V, mu, Sig)
    return mu, Sig


def cholesky(Sigma):
    Sigma = _f64(Sigma)
    V = Sigma.shape[0]
    Lc = np.zeros((V, V))
    st = lib().orc_cholesky(Sigma, V, Lc)
    return Lc, st


def cov_chol(phi):
    phi = _f64(phi)
    V, N = phi.shape
    Sig, Lc = np.zeros((V, V)), np.zeros((V, V))
    st = lib().orc_cov_chol(phi, N, V, Sig, Lc)
    return Sig, Lc, st


def magnetisation(phi):
    phi = _f64(phi)
    V, N = phi.shape
    M = np.zeros(N)
    lib().orc_magnetisation(phi, N, V, M)
    return M


OBS_FIELDS = ("absM", "M2", "chi", "mean_SE", "mode_balance")


def _obs_dict(out):
    d = {k: out[i] for i, k in enumerate(OBS_FIELDS)}
    d["hist"] = out[5:85].copy()
    return d


def observables(phi, S=None):
    phi = _f64(phi)
    V, N = phi.shape
    out = np.zeros(85)
    S = None if S is None else _f64(S)
    lib().orc_observables(phi, _ptr(S), N, V, out)
    return _obs_dict(out)


def observables_from_M(M, S, logw, V):
    M = _f64(M)
    out = np.zeros(85)
    S = None if S is None else _f64(S)
    logw = None if logw is None else _f64(logw)
    lib().orc_observables_from_M(M, _ptr(S), _ptr(logw), M.size, V, out)
    return _obs_dict(out)


SMC_INFO = ("beta", "delta", "ess_frac", "dlogZ", "accept_rate", "n_unique", "chol_status", "_")


def smc_run(L, m0sq, lam, N, seed, k, ess_target=0.5, step_scale=0.0, max_temps=4096, z2_flip=False):
    """z2_flip: flip each particle with probability 1/2 after every resampling (reading A17)."""
    V = L * L
    phi, S, U0 = np.zeros((V, N)), np.zeros(N), np.zeros(N)
    info = np.zeros((max_temps, 8))
    logZ = C.c_double(0.0)
    T = (lib().orc_smc_run_z2 if z2_flip else lib().orc_smc_run)(L, m0sq, lam, N, seed, k, ess_target, step_scale, max_temps, phi, S,
                          U0, C.byref(logZ), _ptr(info))
    if T < 0:
        raise RuntimeError("oracle SMC: covariance not positive definite")
    return {"T": T, "logZ": logZ.value, "phi": phi, "S": S, "U0": U0, "info": info[:T]}


def ns_select(S, k_del):
    S = _f64(S)
    dead = np.zeros(k_del, np.int32)
    lib().orc_ns_select(S, S.size, k_del, dead)
    return dead


NS_INFO = ("logX", "logZ", "S_star", "accept_rate", "remaining_frac", "chol_status")


def ns_run(L, m0sq, lam, n_live, k_del, n_walk, seed, step_scale=0.0, stop_frac=1e-3,
           max_iter=100000, inner="rw", slice_w=1.0, m_expand=8, max_shrink=32):
    """inner = "rw": constrained random walk (reading A5); "slice": slice sampling (reading A16)."""
    V = L * L
    phi, S, U0 = np.zeros((V, n_live)), np.zeros(n_live), np.zeros(n_live)
    info = np.zeros((max_iter, 6))
    dS, dM, dW = (np.zeros(max_iter * k_del) for _ in range(3))
    logZ, logX = C.c_double(0.0), C.c_double(0.0)
    it = lib().orc_ns_run_inner(L, m0sq, lam, n_live, k_del, n_walk, seed, step_scale, stop_frac,
                                max_iter, {"rw": 0, "slice": 1}[inner], slice_w, m_expand,
                                max_shrink, phi, S, U0, C.byref(logZ), C.byref(logX), _ptr(dS),
                                _ptr(dM), _ptr(dW), _ptr(info))
    if it < 0:
        raise RuntimeError("oracle NS: covariance not positive definite")
    n = it * k_del
    return {"iters": it, "logZ": logZ.value, "logX": logX.value, "phi": phi, "S": S, "U0": U0,
            "dead_S": dS[:n], "dead_M": dM[:n], "dead_logw": dW[:n], "info": info[:it]}


# ---------------------------------------------------------------- NEXT row f1: SMC-HMC ----
def hmc_mutate(phi, S, U0, L, m0sq, lam, var, eps, nfrog, beta, seed, t0, k, slots=None):
    """k HMC transitions (reading A14) on copies; returns (phi, S, U0, accept[k,N], margin[k,N])."""
    phi, S, U0 = _f64(phi).copy(), _f64(S).copy(), _f64(U0).copy()
    V, N = phi.shape
    if slots is not None:
        slots = np.ascontiguousarray(slots, np.int32)
    acc = np.zeros((k, N), np.uint8)
    mar = np.zeros((k, N))
    lib().orc_hmc_mutate(phi, S, U0, N, L, m0sq, lam, _f64(var), eps, nfrog, beta, seed, t0, k,
                         _ptr(acc), _ptr(mar), _ptr(slots))
    return phi, S, U0, acc, mar


def leapfrog(q, p, L, m0sq, lam, var, eps, nfrog, beta):
    """One trajectory of a single field; returns (q_new, p_new, H_new - H_old)."""
    q, p = _f64(q).reshape(-1).copy(), _f64(p).reshape(-1).copy()
    dH = lib().orc_leapfrog(q, p, L, m0sq, lam, _f64(var), eps, nfrog, beta)
    return q, p, dH


def smc_hmc_run(L, m0sq, lam, N, seed, k, ess_target=0.5, eps=0.1, nfrog=20, max_temps=4096):
    V = L * L
    phi, S, U0 = np.zeros((V, N)), np.zeros(N), np.zeros(N)
    info = np.zeros((max_temps, 8))
    logZ = C.c_double(0.0)
    T = lib().orc_smc_hmc_run(L, m0sq, lam, N, seed, k, ess_target, eps, nfrog, max_temps, phi, S,
                              U0, C.byref(logZ), _ptr(info))
    return {"T": T, "logZ": logZ.value, "phi": phi, "S": S, "U0": U0, "info": info[:T]}


def irmh_mutate(phi, S, U0, L, m0sq, lam, mu, Lc, beta, seed, t0, k, slots=None):
    """k independent-MH steps from N(mu, Lc Lc^T) (reading A15) on copies; returns
    (phi, S, U0, accept[k,N], margin[k,N])."""
    phi, S, U0 = _f64(phi).copy(), _f64(S).copy(), _f64(U0).copy()
    V, N = phi.shape
    if slots is not None:
        slots = np.ascontiguousarray(slots, np.int32)
    acc = np.zeros((k, N), np.uint8)
    mar = np.zeros((k, N))
    lib().orc_irmh_mutate(phi, S, U0, N, L, m0sq, lam, _f64(mu), _f64(Lc), beta, seed, t0, k,
                          _ptr(acc), _ptr(mar), _ptr(slots))
    return phi, S, U0, acc, mar


def smc_irmh_run(L, m0sq, lam, N, seed, k, ess_target=0.5, max_temps=4096):
    V = L * L
    phi, S, U0 = np.zeros((V, N)), np.zeros(N), np.zeros(N)
    info = np.zeros((max_temps, 8))
    logZ = C.c_double(0.0)
    T = lib().orc_smc_irmh_run(L, m0sq, lam, N, seed, k, ess_target, max_temps, phi, S, U0,
                               C.byref(logZ), _ptr(info))
    if T < 0:
        raise RuntimeError("oracle SMC-IRMH: covariance not positive definite")
    return {"T": T, "logZ": logZ.value, "phi": phi, "S": S, "U0": U0, "info": info[:T]}


# ---------------------------------------------------------------- NEXT row f3: NS slice ----
def slice_walk(phi, S, U0, L, m0sq, lam, Lc, S_star, seed, t0, k, width=1.0, m_expand=8,
               max_shrink=32, slots=None):
    """k constrained slice-sampling steps (reading A16) on copies; returns
    (phi, S, U0, t[k,N], n_expand[k,N], n_shrink[k,N], amb[k,N])."""
    phi, S, U0 = _f64(phi).copy(), _f64(S).copy(), _f64(U0).copy()
    V, N = phi.shape
    if slots is not None:
        slots = np.ascontiguousarray(slots, np.int32)
    t = np.zeros((k, N))
    nexp, nshr = np.zeros((k, N), np.int32), np.zeros((k, N), np.int32)
    amb = np.zeros((k, N))
    lib().orc_slice_walk(phi, S, U0, N, L, m0sq, lam, _f64(Lc), width, m_expand, max_shrink,
                         S_star, seed, t0, k, _ptr(t), _ptr(nexp), _ptr(nshr), _ptr(amb),
                         _ptr(slots))
    return phi, S, U0, t, nexp, nshr, amb


# ---------------------------------------------------------------- NEXT row f4: Z2 flips ----
def z2_flip(phi, seed, T):
    """Flips of reading A17 on a copy; returns (phi, flipped[N])."""
    phi = _f64(phi).copy()
    V, N = phi.shape
    fl = np.zeros(N, np.uint8)
    lib().orc_z2_flip(phi, N, V, seed, T, _ptr(fl))
    return phi, fl
