"""Thin ctypes binding of libbest.so (include/best.h) — argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C-ABI; torch is used by callers for
device memory and streams.  There is no CPU fallback: if the shared library is missing or fails
to load, importing `lib()` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbest.so")

BEST_OK, BEST_ERR_ARG, BEST_ERR_CUDA, BEST_ERR_NOT_SPD, BEST_ERR_UNSUPPORTED, BEST_ERR_ALLOC = 0, -1, -2, -3, -4, -5
ACT_TANH, ACT_SILU = 0, 1
PREC_FP32, PREC_BF16, PREC_FP32_TC = 0, 1, 2
METHOD_MH, METHOD_MALA, METHOD_HMC = 0, 1, 2

EXPORTS = [
    "best_create", "best_destroy", "best_logp_grad", "best_state_create", "best_state_destroy",
    "best_step_mh", "best_step_mala", "best_step_hmc", "best_step_aies", "best_set_adaptation",
    "best_adapt_stats", "best_get_whitening", "best_set_whitening", "best_state_get",
    "best_state_get_f64", "best_state_last_log_alpha", "best_state_set", "best_launch_count",
    "best_last_error", "best_version", "best_set_step_scale", "best_set_hard_box", "best_burn_in", "best_step_aies_de", "best_rminus1", "best_probe_l2_read",
    "best_state_set_chain_offset", "best_rminus1_noalloc", "best_rminus1_noalloc_max_doubles",
    "best_set_adaptation_exchange", "best_set_aies_exchange",
]

# int fn(const double* send_dev, double* recv_dev, int64_t count, void* stream, void* user)
EXCHANGE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p)


class BestError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libbest error {code}: {msg}")
        self.code = code


class best_config(C.Structure):
    _fields_ = [
        ("d", C.c_int32), ("n_affine", C.c_int32),
        ("widths", C.POINTER(C.c_int32)),
        ("W_flat", C.POINTER(C.c_float)), ("b_flat", C.POINTER(C.c_float)),
        ("activation", C.c_int32), ("mlp_scale", C.c_float),
        ("mu", C.POINTER(C.c_double)), ("Sigma_inv", C.POINTER(C.c_double)),
        ("lo", C.POINTER(C.c_double)), ("hi", C.POINTER(C.c_double)),
        ("pen_kappa", C.c_float), ("pen_gamma", C.c_float),
        ("banana_i", C.c_int32), ("banana_j", C.c_int32), ("banana_sigma", C.c_float),
        ("L", C.POINTER(C.c_double)),
        ("precision", C.c_int32),
    ]


_LIB = None


def lib():
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_04895_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, u64, i32, f32 = C.c_void_p, C.c_int64, C.c_uint64, C.c_int32, C.c_float
    L.best_create.argtypes = [C.POINTER(best_config), C.POINTER(vp)]
    L.best_destroy.argtypes = [vp]
    L.best_destroy.restype = None
    L.best_logp_grad.argtypes = [vp, vp, i64, vp, vp, vp]
    L.best_state_create.argtypes = [vp, i64, vp, vp, C.POINTER(vp)]
    L.best_state_destroy.argtypes = [vp]
    L.best_state_destroy.restype = None
    L.best_step_mh.argtypes = [vp, vp, i64, u64, f32, vp, i32, vp]
    L.best_step_mala.argtypes = [vp, vp, i64, u64, f32, vp, i32, vp]
    L.best_step_hmc.argtypes = [vp, vp, i64, u64, f32, i32, vp, i32, vp]
    L.best_step_aies.argtypes = [vp, vp, i64, u64, f32, vp, i32, vp]
    L.best_step_aies_de.argtypes = [vp, vp, i64, u64, f32, vp, i32, vp]
    L.best_set_adaptation.argtypes = [vp, vp, i32, C.c_double]
    L.best_adapt_stats.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
    L.best_get_whitening.argtypes = [vp, vp]
    L.best_set_whitening.argtypes = [vp, vp]
    L.best_set_step_scale.argtypes = [vp, vp]
    L.best_set_hard_box.argtypes = [vp, i32]
    L.best_rminus1.argtypes = [vp, i64, i64, i32, C.POINTER(C.c_double), vp]
    L.best_probe_l2_read.argtypes = [i64, i32, C.POINTER(C.c_double), vp]
    L.best_rminus1_noalloc.argtypes = [vp, i64, i64, i32, C.POINTER(C.c_double), vp]
    L.best_rminus1_noalloc_max_doubles.argtypes = []
    L.best_rminus1_noalloc_max_doubles.restype = i64
    L.best_burn_in.argtypes = [vp, vp, i32, i32, i64, i64, i64, u64, C.POINTER(C.c_float), C.c_float, i32,
                               C.c_double, vp, C.POINTER(C.c_double), vp, vp]
    L.best_state_get.argtypes = [vp, vp, vp, vp, C.POINTER(u64), vp, C.POINTER(u64), vp]
    L.best_state_get_f64.argtypes = [vp, vp, vp, vp, vp]
    L.best_state_last_log_alpha.argtypes = [vp, vp, vp]
    L.best_state_set.argtypes = [vp, vp, u64, vp]
    L.best_state_set_chain_offset.argtypes = [vp, u64]
    L.best_set_adaptation_exchange.argtypes = [vp, EXCHANGE_FN, vp, i32]
    L.best_set_aies_exchange.argtypes = [vp, EXCHANGE_FN, vp, i32, i32]
    L.best_launch_count.restype = u64
    L.best_last_error.restype = C.c_char_p
    L.best_version.restype = C.c_char_p
    _LIB = L
    return L


def _check(rc):
    if rc != 0:
        raise BestError(rc, lib().best_last_error().decode())


def _ptr(x):
    """numpy array → host pointer; torch tensor → data_ptr(); int/None pass through."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    return int(x)


def launch_count() -> int:
    return int(lib().best_launch_count())


def version() -> str:
    return lib().best_version().decode()


class Context:
    """best_create / best_destroy + the calls that take a best_ctx*."""

    def __init__(self, w, precision: int = PREC_FP32):
        self.d = int(w.d)
        self.precision = precision
        keep = []
        cfg = best_config()
        cfg.d = self.d
        n_affine = max(len(w.widths) - 1, 0)
        cfg.n_affine = n_affine
        if n_affine:
            widths = np.asarray(w.widths, dtype=np.int32)
            Wf = np.concatenate([np.ascontiguousarray(x, dtype=np.float32).ravel() for x in w.W])
            bf = np.concatenate([np.ascontiguousarray(x, dtype=np.float32).ravel() for x in w.b])
            keep += [widths, Wf, bf]
            cfg.widths = widths.ctypes.data_as(C.POINTER(C.c_int32))
            cfg.W_flat = Wf.ctypes.data_as(C.POINTER(C.c_float))
            cfg.b_flat = bf.ctypes.data_as(C.POINTER(C.c_float))
        cfg.activation = int(w.activation)
        cfg.mlp_scale = float(w.mlp_scale)
        for name in ("mu", "Sigma_inv", "lo", "hi", "L"):
            arr = getattr(w, name)
            if arr is not None:
                arr = np.ascontiguousarray(arr, dtype=np.float64)
                keep.append(arr)
                setattr(cfg, name, arr.ctypes.data_as(C.POINTER(C.c_double)))
        cfg.pen_kappa, cfg.pen_gamma = float(w.pen_kappa), float(w.pen_gamma)
        cfg.banana_i, cfg.banana_j = int(w.banana_i), int(w.banana_j)
        cfg.banana_sigma = float(w.banana_sigma)
        cfg.precision = int(precision)
        h = C.c_void_p()
        self._h = None
        _check(lib().best_create(C.byref(cfg), C.byref(h)))
        self._h = h
        del keep

    def close(self):
        if getattr(self, "_h", None):
            try:
                lib().best_destroy(self._h)
            except TypeError:      # interpreter shutdown: the module globals are already gone
                pass
            self._h = None

    def __del__(self):
        self.close()

    def logp_grad(self, theta, n, logp, grad=None, stream=0):
        """theta/logp/grad: numpy (host) or torch cuda tensors (device), float32."""
        _check(lib().best_logp_grad(self._h, _ptr(theta), int(n), _ptr(logp), _ptr(grad), stream or None))

    def new_state(self, theta0, n_chains=None, stream=0):
        return State(self, theta0, n_chains, stream)

    def get_whitening(self):
        L = np.zeros((self.d, self.d))
        _check(lib().best_get_whitening(self._h, L.ctypes.data))
        return L

    def set_whitening(self, L):
        L = np.ascontiguousarray(L, dtype=np.float64)
        _check(lib().best_set_whitening(self._h, L.ctypes.data))

    def set_step_scale(self, s):
        if s is None:
            _check(lib().best_set_step_scale(self._h, None))
            return
        s = np.ascontiguousarray(s, dtype=np.float64)
        if s.shape != (self.d,):
            raise ValueError("step scale must have shape (d,)")
        _check(lib().best_set_step_scale(self._h, s.ctypes.data))

    def set_hard_box(self, on: bool):
        _check(lib().best_set_hard_box(self._h, 1 if on else 0))

    def adapt_stats(self):
        a, b = C.c_int64(), C.c_int64()
        _check(lib().best_adapt_stats(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value


def rminus1(trace, stream=0) -> float:
    """best_rminus1 on a torch cuda float32 trace [n][B][d] (eq 4.1-4.2)."""
    n, nb, d = trace.shape
    if not trace.is_contiguous():
        raise ValueError("trace must be contiguous")
    out = C.c_double()
    _check(lib().best_rminus1(_ptr(trace), n, nb, d, C.byref(out), stream or None))
    return out.value


def rminus1_noalloc(trace, stream=0) -> float:
    """best_rminus1_noalloc: best_rminus1 with its scratch in a static device array (no allocation; size limit)."""
    n, nb, d = trace.shape
    if not trace.is_contiguous():
        raise ValueError("trace must be contiguous")
    out = C.c_double()
    _check(lib().best_rminus1_noalloc(_ptr(trace), n, nb, d, C.byref(out), stream or None))
    return out.value


def rminus1_noalloc_max_doubles() -> int:
    return int(lib().best_rminus1_noalloc_max_doubles())


def probe_l2_read(n_bytes=32 << 20, passes=20, stream=0) -> float:
    """best_probe_l2_read: GB/s of all SMs re-reading an L2-resident buffer."""
    out = C.c_double()
    _check(lib().best_probe_l2_read(n_bytes, passes, C.byref(out), stream or None))
    return out.value


class State:
    """best_state_* + best_step_*."""

    def __init__(self, ctx: Context, theta0, n_chains=None, stream=0):
        self.ctx = ctx
        if isinstance(theta0, np.ndarray):
            theta0 = np.ascontiguousarray(theta0, dtype=np.float32)
            n_chains = theta0.shape[0] if n_chains is None else n_chains
        elif n_chains is None:
            n_chains = theta0.shape[0]
        self.B = int(n_chains)
        h = C.c_void_p()
        self._h = None
        _check(lib().best_state_create(ctx._h, self.B, _ptr(theta0), stream or None, C.byref(h)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            try:
                lib().best_state_destroy(self._h)
            except TypeError:      # interpreter shutdown: the module globals are already gone
                pass
            self._h = None

    def __del__(self):
        self.close()

    def step_mh(self, n_steps, seed, eps, trace=None, thin=0, stream=0):
        _check(lib().best_step_mh(self.ctx._h, self._h, n_steps, seed, eps, _ptr(trace), thin, stream or None))

    def step_mala(self, n_steps, seed, eps, trace=None, thin=0, stream=0):
        _check(lib().best_step_mala(self.ctx._h, self._h, n_steps, seed, eps, _ptr(trace), thin, stream or None))

    def step_hmc(self, n_traj, seed, eps, n_leapfrog, trace=None, thin=0, stream=0):
        _check(lib().best_step_hmc(self.ctx._h, self._h, n_traj, seed, eps, n_leapfrog, _ptr(trace), thin,
                                   stream or None))

    def step_aies(self, n_steps, seed, a=2.0, trace=None, thin=0, stream=0):
        _check(lib().best_step_aies(self.ctx._h, self._h, n_steps, seed, a, _ptr(trace), thin, stream or None))

    def step_aies_de(self, n_steps, seed, sigma_gamma=1e-5, trace=None, thin=0, stream=0):
        _check(lib().best_step_aies_de(self.ctx._h, self._h, n_steps, seed, sigma_gamma, _ptr(trace), thin,
                                       stream or None))

    def set_adaptation(self, adapt_every, jitter=1e-6):
        _check(lib().best_set_adaptation(self.ctx._h, self._h, adapt_every, jitter))

    def set_adaptation_exchange(self, fn, world_size):
        """best_set_adaptation_exchange: fn(send_ptr, recv_ptr, count, stream) -> None / 0 enqueues an all-gather of
        `count` doubles per rank on `stream` (see distributed.allgather_exchange); fn = None switches it off."""
        if fn is None:
            self._xchg = None
            _check(lib().best_set_adaptation_exchange(self._h, C.cast(None, EXCHANGE_FN), None, world_size))
            return

        def tramp(send, recv, count, stream, _user):
            try:
                rc = fn(send or 0, recv or 0, count, stream or 0)
                return int(rc or 0)
            except Exception:          # an exception must not unwind through the C frames
                import traceback
                traceback.print_exc()
                return 1
        self._xchg = EXCHANGE_FN(tramp)          # keep the trampoline alive as long as the state uses it
        _check(lib().best_set_adaptation_exchange(self._h, self._xchg, None, world_size))

    def set_aies_exchange(self, fn, rank, world_size):
        """best_set_aies_exchange: the ensemble moves of this state update the rank's slice of each half-ensemble and
        all-gather it through fn (same signature as in set_adaptation_exchange); fn = None switches it off."""
        if fn is None:
            self._aies_xchg = None
            _check(lib().best_set_aies_exchange(self._h, C.cast(None, EXCHANGE_FN), None, rank, world_size))
            return

        def tramp(send, recv, count, stream, _user):
            try:
                return int(fn(send or 0, recv or 0, count, stream or 0) or 0)
            except Exception:
                import traceback
                traceback.print_exc()
                return 1
        self._aies_xchg = EXCHANGE_FN(tramp)
        _check(lib().best_set_aies_exchange(self._h, self._aies_xchg, None, rank, world_size))

    def burn_in(self, method, n_iter, n_steps, n_adapt, block, seed, eps0, target_accept, n_leapfrog=1,
                jitter=1e-6, stream=0):
        """best_burn_in: returns (eps, best_theta [d] float32, best_logp, eps used in every adaptation block)."""
        m = {"mh": METHOD_MH, "mala": METHOD_MALA, "hmc": METHOD_HMC}.get(method, method)
        eps = C.c_float(eps0)
        best_lp = C.c_double()
        best_th = np.zeros(self.ctx.d, dtype=np.float32)
        nblk = n_iter * (-(-n_adapt // block) if n_adapt > 0 and block > 0 else 0)
        hist = np.zeros(max(nblk, 1), dtype=np.float32)
        _check(lib().best_burn_in(self.ctx._h, self._h, m, n_iter, n_steps, n_adapt, block, seed, C.byref(eps),
                                  target_accept, n_leapfrog, jitter, best_th.ctypes.data, C.byref(best_lp),
                                  hist.ctypes.data, stream or None))
        return eps.value, best_th, best_lp.value, hist[:nblk]

    def get(self, want_grad=True, stream=0):
        d, B = self.ctx.d, self.B
        theta = np.zeros((B, d), dtype=np.float32)
        logp = np.zeros(B, dtype=np.float32)
        grad = np.zeros((B, d), dtype=np.float32) if want_grad else None
        n_accept = np.zeros(B, dtype=np.uint64)
        step, n_evals = C.c_uint64(), C.c_uint64()
        _check(lib().best_state_get(self._h, theta.ctypes.data, logp.ctypes.data, _ptr(grad), C.byref(step),
                                    n_accept.ctypes.data, C.byref(n_evals), stream or None))
        return dict(theta=theta, logp=logp, grad=grad, step=step.value, n_accept=n_accept,
                    n_evals=n_evals.value)

    def get_f64(self, want_grad=True, stream=0):
        d, B = self.ctx.d, self.B
        theta, logp = np.zeros((B, d)), np.zeros(B)
        grad = np.zeros((B, d)) if want_grad else None
        _check(lib().best_state_get_f64(self._h, theta.ctypes.data, logp.ctypes.data, _ptr(grad), stream or None))
        return theta, logp, grad

    def set_chain_offset(self, chain0: int):
        _check(lib().best_state_set_chain_offset(self._h, chain0))

    def last_log_alpha(self, stream=0):
        la = np.zeros(self.B)
        _check(lib().best_state_last_log_alpha(self._h, la.ctypes.data, stream or None))
        return la

    def set(self, theta, step=0, stream=0):
        if isinstance(theta, np.ndarray):
            theta = np.ascontiguousarray(theta, dtype=np.float32)
        _check(lib().best_state_set(self._h, _ptr(theta), step, stream or None))
