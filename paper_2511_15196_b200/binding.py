"""Thin ctypes binding of libphi4smc.so (include/phi4smc.h): argument marshalling only.

Every step of the path runs in the CUDA library; torch is used for device memory (the workspace
tensor) and for the current CUDA stream.  There is no CPU fallback: if the library is missing or
no CUDA device is present the calls raise.
"""
import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libphi4smc.so")
HIST_BINS = 80
MAX_HOOK_STEPS = 64

ERRORS = {0: "PHI4_OK", -1: "PHI4_EINVAL", -2: "PHI4_ENOMEM", -3: "PHI4_ENOTPD", -4: "PHI4_ENAN",
          -5: "PHI4_ECUDA", -6: "PHI4_ETRUNC", -7: "PHI4_ETOOBIG"}
NOALLOC_MAX_N = 131072
ETRUNC = -6


class Phi4Error(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        super().__init__("%s failed: %s (%d) %s" % (where, ERRORS.get(code, "?"), code, detail))


class smc_params(C.Structure):
    _fields_ = [("k_steps", C.c_int), ("ess_target", C.c_float), ("step_scale", C.c_float),
                ("mutation_path", C.c_int), ("kernel", C.c_int), ("hmc_eps", C.c_float),
                ("hmc_leapfrog", C.c_int), ("z2_flip", C.c_int)]


class ns_params(C.Structure):
    _fields_ = [("inner", C.c_int), ("slice_width", C.c_float), ("max_expand", C.c_int),
                ("max_shrink", C.c_int)]


class smc_step_info(C.Structure):
    _fields_ = [("beta", C.c_double), ("delta", C.c_double), ("ess_frac", C.c_double),
                ("dlogZ", C.c_double), ("logZ", C.c_double), ("accept_rate", C.c_double),
                ("n_unique", C.c_int), ("chol_status", C.c_int), ("temp_index", C.c_int),
                ("done", C.c_int)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class ns_step_info(C.Structure):
    _fields_ = [("logX", C.c_double), ("logZ", C.c_double), ("S_star", C.c_double),
                ("accept_rate", C.c_double), ("remaining_frac", C.c_double),
                ("chol_status", C.c_int), ("iter_index", C.c_int), ("done", C.c_int)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class phi4_run_state(C.Structure):
    _fields_ = [("beta", C.c_double), ("delta", C.c_double), ("logZ", C.c_double),
                ("logX", C.c_double), ("S_star", C.c_double), ("remaining_frac", C.c_double),
                ("index", C.c_int32), ("done", C.c_int32), ("step_counter", C.c_uint64)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class phi4_peaks(C.Structure):
    _fields_ = [("tf32_tflops_burst", C.c_double), ("tf32_tflops_sustained", C.c_double),
                ("ffma_tlaneops", C.c_double), ("imad_wide_tlaneops", C.c_double),
                ("sms", C.c_int32), ("reserved", C.c_int32), ("dfma_tlaneops", C.c_double),
                ("f16_tflops_burst", C.c_double), ("f16_tflops_sustained", C.c_double)]


class phi4_observables(C.Structure):
    _fields_ = [("absM", C.c_double), ("M2", C.c_double), ("chi", C.c_double),
                ("mean_SE", C.c_double), ("mode_balance", C.c_double),
                ("hist", C.c_double * HIST_BINS)]

    def asdict(self):
        d = {k: getattr(self, k) for k in ("absM", "M2", "chi", "mean_SE", "mode_balance")}
        d["hist"] = np.array(self.hist[:])
        return d


# name -> (restype, argtypes): every symbol include/phi4smc.h declares
_vp, _i, _f, _d, _u64, _sz = C.c_void_p, C.c_int, C.c_float, C.c_double, C.c_uint64, C.c_size_t
SIGNATURES = {
    "phi4_strerror": (C.c_char_p, [_i]),
    "phi4_last_cuda_error": (C.c_char_p, [_vp]),
    "phi4_kernel_launches": (_u64, []),
    "phi4_measure_peaks": (_i, [_d, C.POINTER(phi4_peaks), _vp, _sz, _vp]),
    "phi4_noalloc_setup": (_i, []),
    "phi4_resample_noalloc": (_i, [_vp, _i, _u64, C.c_uint32, _vp, _vp]),
    "smc_workspace_bytes": (_sz, [_i, _i]),
    "smc_init": (_i, [C.POINTER(_vp), _i, _f, _f, _i, _u64, _vp, _sz, _vp]),
    "smc_init_kl": (_i, [C.POINTER(_vp), _i, _f, _f, _i, _u64, _vp, _sz, _vp]),
    "smc_reset": (_i, [_vp, _u64]),
    "smc_destroy": (_i, [_vp]),
    "smc_set_params": (_i, [_vp, C.POINTER(smc_params)]),
    "smc_step": (_i, [_vp, C.POINTER(smc_step_info)]),
    "smc_run": (_i, [_vp, _i, C.POINTER(_i)]),
    "smc_get_history": (_i, [_vp, C.POINTER(smc_step_info), _i, C.POINTER(_i)]),
    "estimate_cov_chol": (_i, [_vp]),
    "observables": (_i, [_vp, C.POINTER(phi4_observables)]),
    "log_Z": (_d, [_vp]),
    "ns_workspace_bytes": (_sz, [_i, _i, _i, _i]),
    "ns_init": (_i, [C.POINTER(_vp), _i, _f, _f, _i, _i, _i, _u64, _d, _i, _vp, _sz, _vp]),
    "ns_init_kl": (_i, [C.POINTER(_vp), _i, _f, _f, _i, _i, _i, _u64, _d, _i, _vp, _sz, _vp]),
    "ns_set_params": (_i, [_vp, C.POINTER(ns_params)]),
    "ns_step": (_i, [_vp, C.POINTER(ns_step_info)]),
    "ns_run": (_i, [_vp, _i, C.POINTER(_i)]),
    "smc_get_state": (_i, [_vp, _vp, _vp, _vp, C.POINTER(_d), C.POINTER(_u64)]),
    "smc_set_state": (_i, [_vp, _vp, _d, _u64]),
    "smc_get_chol": (_i, [_vp, _vp]),
    "smc_set_chol": (_i, [_vp, _vp]),
    "smc_get_cov": (_i, [_vp, _vp]),
    "smc_get_mean": (_i, [_vp, _vp]),
    "smc_mutate": (_i, [_vp, _i, _vp, _vp]),
    "smc_time_mutation": (_i, [_vp, _i, _i, C.POINTER(_f)]),
    "smc_time_phase": (_i, [_vp, _i, _i, C.POINTER(_f)]),
    "smc_reweight": (_i, [_vp, _d, _vp, C.POINTER(smc_step_info)]),
    "smc_resample": (_i, [_vp, _vp, _vp]),
    "ns_get_dead": (_i, [_vp, _vp, _vp, _vp, _vp, _i, C.POINTER(_i)]),
    "ns_set_dead": (_i, [_vp, _vp, _vp, _vp, _i]),
    "smc_get_run_state": (_i, [_vp, C.POINTER(phi4_run_state)]),
    "smc_restore": (_i, [_vp, _vp, _vp, _vp, C.POINTER(phi4_run_state)]),
}

_lib = None


def load():
    """dlopen libphi4smc.so and declare every signature.  Raises if the library is not built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libphi4smc.so is not built: run `python -m paper_2511_15196_b200.build`"
                               " (there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _np_ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Handle:
    """Owns the opaque phi4smc* and the torch workspace tensor it lives in."""

    def __init__(self, ptr, workspace, kind, L, N, **kw):
        self.ptr, self.workspace, self.kind, self.L, self.V, self.N = ptr, workspace, kind, L, L * L, N
        self.__dict__.update(kw)

    def _check(self, rc, where):
        if rc != 0:
            detail = load().phi4_last_cuda_error(self.ptr).decode() if rc == -5 else ""
            raise Phi4Error(rc, where, detail)

    def close(self):
        if self.ptr:
            load().smc_destroy(self.ptr)
            self.ptr = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _device_workspace(nbytes, device):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: the phi4smc path has no CPU fallback")
    return torch.empty(nbytes + 256, dtype=torch.uint8, device=device)


def _stream_ptr(device):
    import torch
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _aligned(ws):
    p = ws.data_ptr()
    return (p + 255) // 256 * 256


def phi4_kernel_launches():
    return load().phi4_kernel_launches()


def phi4_measure_peaks(seconds=2.0, device="cuda:0"):
    ws = _device_workspace(1 << 16, device)
    out = phi4_peaks()
    rc = load().phi4_measure_peaks(seconds, C.byref(out), C.c_void_p(_aligned(ws)), 1 << 16, _stream_ptr(device))
    if rc != 0:
        raise Phi4Error(rc, "phi4_measure_peaks")
    return {k: getattr(out, k) for k, _ in phi4_peaks._fields_ if k != "reserved"}


def phi4_resample_noalloc(w, seed, t, out):
    """w: CUDA float32 tensor (N,), out: CUDA int32 tensor (N,) on the same device; enqueues on
    torch's current stream of that device, allocates nothing.  Raises Phi4Error(-7) if N > NOALLOC_MAX_N."""
    import torch
    assert w.is_cuda and out.is_cuda and w.device == out.device
    assert w.dtype == torch.float32 and out.dtype == torch.int32 and w.is_contiguous() and out.is_contiguous()
    assert out.numel() >= w.numel()
    with torch.cuda.device(w.device):
        rc = load().phi4_resample_noalloc(C.c_void_p(w.data_ptr()), w.numel(), seed, t,
                                          C.c_void_p(out.data_ptr()), _stream_ptr(w.device))
    if rc != 0:
        raise Phi4Error(rc, "phi4_resample_noalloc", load().phi4_strerror(rc).decode())


def smc_workspace_bytes(L, N):
    return load().smc_workspace_bytes(L, N)


def ns_workspace_bytes(L, n_live, k_delete, max_iters):
    return load().ns_workspace_bytes(L, n_live, k_delete, max_iters)


def smc_init(L, m0sq, lam, N, seed, device="cuda:0", _entry="smc_init"):
    lib = load()
    nbytes = lib.smc_workspace_bytes(L, N)
    if nbytes == 0:
        raise Phi4Error(-1, "smc_workspace_bytes")
    ws = _device_workspace(nbytes, device)
    base = _aligned(ws)
    ptr = C.c_void_p()
    rc = getattr(lib, _entry)(C.byref(ptr), L, m0sq, lam, N, seed, C.c_void_p(base),
                              nbytes, _stream_ptr(device))
    if rc != 0:
        detail = lib.phi4_last_cuda_error(ptr if ptr else None).decode()
        if ptr:
            lib.smc_destroy(ptr)
        raise Phi4Error(rc, _entry, detail)
    return Handle(ptr, ws, "smc", L, N)


def smc_init_kl(L, kappa, lam, N, seed, device="cuda:0"):
    """Eq. 2's (kappa, lambda) parameterisation (include/phi4smc.h: smc_init_kl)."""
    return smc_init(L, kappa, lam, N, seed, device, _entry="smc_init_kl")


def ns_init(L, m0sq, lam, n_live, k_delete, n_walk, seed, stop_frac=1e-3, max_iters=4096,
            device="cuda:0", _entry="ns_init"):
    lib = load()
    nbytes = lib.ns_workspace_bytes(L, n_live, k_delete, max_iters)
    if nbytes == 0:
        raise Phi4Error(-1, "ns_workspace_bytes")
    ws = _device_workspace(nbytes, device)
    base = _aligned(ws)
    ptr = C.c_void_p()
    rc = getattr(lib, _entry)(C.byref(ptr), L, m0sq, lam, n_live, k_delete, n_walk, seed, stop_frac,
                              max_iters, C.c_void_p(base), nbytes, _stream_ptr(device))
    if rc != 0:
        detail = lib.phi4_last_cuda_error(ptr if ptr else None).decode()
        if ptr:
            lib.smc_destroy(ptr)
        raise Phi4Error(rc, _entry, detail)
    return Handle(ptr, ws, "ns", L, n_live, k_delete=k_delete, n_walk=n_walk, max_iters=max_iters)


def ns_init_kl(L, kappa, lam, n_live, k_delete, n_walk, seed, stop_frac=1e-3, max_iters=4096,
               device="cuda:0"):
    """Eq. 2's (kappa, lambda) parameterisation (include/phi4smc.h: ns_init_kl)."""
    return ns_init(L, kappa, lam, n_live, k_delete, n_walk, seed, stop_frac, max_iters, device,
                   _entry="ns_init_kl")


def smc_reset(h, seed):
    h._check(load().smc_reset(h.ptr, seed), "smc_reset")


def smc_destroy(h):
    h.close()


def smc_set_params(h, k_steps=10, ess_target=0.5, step_scale=0.0, mutation_path=0, kernel=0,
                   hmc_eps=0.1, hmc_leapfrog=20, z2_flip=0):
    p = smc_params(k_steps, ess_target, step_scale, mutation_path, kernel, hmc_eps, hmc_leapfrog,
                   z2_flip)
    h._check(load().smc_set_params(h.ptr, C.byref(p)), "smc_set_params")


def smc_step(h, want_info=True):
    if not want_info:
        h._check(load().smc_step(h.ptr, None), "smc_step")
        return None
    info = smc_step_info()
    h._check(load().smc_step(h.ptr, C.byref(info)), "smc_step")
    return info.asdict()


def smc_run(h, max_temps=4096):
    n = C.c_int(0)
    h._check(load().smc_run(h.ptr, max_temps, C.byref(n)), "smc_run")
    return n.value


def smc_get_history(h, cap=4096):
    arr = (smc_step_info * cap)()
    n = C.c_int(0)
    h._check(load().smc_get_history(h.ptr, arr, cap, C.byref(n)), "smc_get_history")
    return [arr[i].asdict() for i in range(min(n.value, cap))]


def estimate_cov_chol(h):
    h._check(load().estimate_cov_chol(h.ptr), "estimate_cov_chol")


def observables(h):
    o = phi4_observables()
    h._check(load().observables(h.ptr, C.byref(o)), "observables")
    return o.asdict()


def log_Z(h):
    v = load().log_Z(h.ptr)
    if math.isnan(v):
        raise Phi4Error(-5, "log_Z")
    return v


def ns_set_params(h, inner=0, slice_width=1.0, max_expand=8, max_shrink=32):
    p = ns_params(inner, slice_width, max_expand, max_shrink)
    h._check(load().ns_set_params(h.ptr, C.byref(p)), "ns_set_params")


def ns_step(h, want_info=True):
    """PHI4_ETRUNC (dead-point log full) is not raised: the info then carries done = 2."""
    if not want_info:
        h._check(load().ns_step(h.ptr, None), "ns_step")
        return None
    info = ns_step_info()
    rc = load().ns_step(h.ptr, C.byref(info))
    if rc != ETRUNC:
        h._check(rc, "ns_step")
    return info.asdict()


def ns_run(h, max_iters=4096):
    """Returns the iterations made; h.truncated says whether the run ended with PHI4_ETRUNC."""
    n = C.c_int(0)
    rc = load().ns_run(h.ptr, max_iters, C.byref(n))
    h.truncated = rc == ETRUNC
    if rc != ETRUNC:
        h._check(rc, "ns_run")
    return n.value


def smc_get_state(h, want_phi=True, out=None):
    """out: optional dict of caller-owned C-contiguous fp32 arrays "phi" (V, N), "S" (N,), "U0" (N,)
    to receive the copies (e.g. views of pinned host memory: the device-to-host copies then run at
    full PCIe rate instead of through the driver's staging of pageable memory)."""
    if out is not None:
        phi, S, U0 = (out["phi"] if want_phi else None), out["S"], out["U0"]
        for a, shp in ((phi, (h.V, h.N)), (S, (h.N,)), (U0, (h.N,))):
            assert a is None or (a.dtype == np.float32 and a.shape == shp and a.flags["C_CONTIGUOUS"])
    else:
        phi = np.empty((h.V, h.N), np.float32) if want_phi else None
        S, U0 = np.empty(h.N, np.float32), np.empty(h.N, np.float32)
    beta, t = C.c_double(0), C.c_uint64(0)
    h._check(load().smc_get_state(h.ptr, _np_ptr(phi), _np_ptr(S), _np_ptr(U0), C.byref(beta),
                                  C.byref(t)), "smc_get_state")
    return {"phi": phi, "S": S, "U0": U0, "beta": beta.value, "step": t.value}


def smc_set_state(h, phi, beta, step):
    phi = np.ascontiguousarray(phi, np.float32)
    assert phi.shape == (h.V, h.N)
    h._check(load().smc_set_state(h.ptr, _np_ptr(phi), beta, step), "smc_set_state")


def smc_get_run_state(h):
    rs = phi4_run_state()
    h._check(load().smc_get_run_state(h.ptr, C.byref(rs)), "smc_get_run_state")
    return rs.asdict()


def smc_restore(h, phi, S, U0, run_state):
    phi = np.ascontiguousarray(phi, np.float32)
    assert phi.shape == (h.V, h.N)
    S = None if S is None else np.ascontiguousarray(S, np.float32)
    U0 = None if U0 is None else np.ascontiguousarray(U0, np.float32)
    rs = phi4_run_state(**run_state)
    h._check(load().smc_restore(h.ptr, _np_ptr(phi), _np_ptr(S), _np_ptr(U0), C.byref(rs)), "smc_restore")


def ns_set_dead(h, dead_S, dead_M, dead_logw):
    dS, dM = np.ascontiguousarray(dead_S, np.float32), np.ascontiguousarray(dead_M, np.float32)
    dW = np.ascontiguousarray(dead_logw, np.float64)
    h._check(load().ns_set_dead(h.ptr, _np_ptr(dS), _np_ptr(dM), _np_ptr(dW), dS.size), "ns_set_dead")


def smc_get_chol(h):
    Lc = np.empty((h.V, h.V), np.float32)
    h._check(load().smc_get_chol(h.ptr, _np_ptr(Lc)), "smc_get_chol")
    return Lc


def smc_set_chol(h, Lc):
    Lc = np.ascontiguousarray(Lc, np.float32)
    assert Lc.shape == (h.V, h.V)
    h._check(load().smc_set_chol(h.ptr, _np_ptr(Lc)), "smc_set_chol")


def smc_get_cov(h):
    Sig = np.empty((h.V, h.V), np.float32)
    h._check(load().smc_get_cov(h.ptr, _np_ptr(Sig)), "smc_get_cov")
    return Sig


def smc_get_mean(h):
    mu = np.zeros(h.V, np.float32)
    h._check(load().smc_get_mean(h.ptr, _np_ptr(mu)), "smc_get_mean")
    return mu


def smc_mutate(h, k, want=True):
    acc = np.empty((k, h.N), np.uint8) if want else None
    mar = np.empty((k, h.N), np.float32) if want else None
    h._check(load().smc_mutate(h.ptr, k, _np_ptr(acc), _np_ptr(mar)), "smc_mutate")
    return acc, mar


def smc_time_mutation(h, k, reps=5):
    ms = C.c_float(0.0)
    h._check(load().smc_time_mutation(h.ptr, k, reps, C.byref(ms)), "smc_time_mutation")
    return ms.value


PHASES = {"mutation": 0, "proposal": 1, "normals": 2, "accept": 3, "resample": 4, "gather": 5,
          "covchol": 6, "reweight": 7}


def smc_time_phase(h, phase, reps=5):
    ms = C.c_float(0.0)
    h._check(load().smc_time_phase(h.ptr, PHASES[phase], reps, C.byref(ms)), "smc_time_phase")
    return ms.value


def smc_reweight(h, delta=-1.0):
    w = np.empty(h.N, np.float32)
    info = smc_step_info()
    h._check(load().smc_reweight(h.ptr, delta, _np_ptr(w), C.byref(info)), "smc_reweight")
    return w, info.asdict()


def smc_resample(h, w=None, want=True):
    w = None if w is None else np.ascontiguousarray(w, np.float32)
    anc = np.empty(h.N, np.int32) if want else None
    h._check(load().smc_resample(h.ptr, _np_ptr(w), _np_ptr(anc)), "smc_resample")
    return anc


def ns_get_dead(h):
    cap = h.max_iters * h.k_delete
    idx = np.empty(h.k_delete, np.int32)
    dS, dM, dW = np.empty(cap, np.float32), np.empty(cap, np.float32), np.empty(cap, np.float64)
    n = C.c_int(0)
    h._check(load().ns_get_dead(h.ptr, _np_ptr(idx), _np_ptr(dS), _np_ptr(dM), _np_ptr(dW), cap,
                                C.byref(n)), "ns_get_dead")
    return {"last_dead": idx, "dead_S": dS[:n.value], "dead_M": dM[:n.value],
            "dead_logw": dW[:n.value]}
