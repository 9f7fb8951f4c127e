"""ctypes harness around oracle/liboracle.so — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package except nothing: the `Workload`
objects it accepts are plain data (duck-typed), produced by the shared input generators.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_LIB = None


class _Config(C.Structure):
    _fields_ = [
        ("d", C.c_int32), ("n_affine", C.c_int32),
        ("widths", C.POINTER(C.c_int32)),
        ("W_flat", C.POINTER(C.c_float)), ("b_flat", C.POINTER(C.c_float)),
        ("activation", C.c_int32), ("mlp_scale", C.c_double),
        ("mu", C.POINTER(C.c_double)), ("Sigma_inv", C.POINTER(C.c_double)),
        ("lo", C.POINTER(C.c_double)), ("hi", C.POINTER(C.c_double)),
        ("pen_kappa", C.c_double), ("pen_gamma", C.c_double),
        ("banana_i", C.c_int32), ("banana_j", C.c_int32), ("banana_sigma", C.c_double),
        ("L", C.POINTER(C.c_double)),
    ]


def lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        L = C.CDLL(path)
        dp, u64, i64, i32 = C.POINTER(C.c_double), C.c_uint64, C.c_int64, C.c_int32
        u64p, u32p, vp = C.POINTER(C.c_uint64), C.POINTER(C.c_uint32), C.c_void_p
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_u01.restype = C.c_double
        L.oracle_u01.argtypes = [C.c_uint32]
        L.oracle_normals.argtypes = [u64, u64, u64, i32, dp]
        L.oracle_control.argtypes = [u64, u64, u64, dp, dp, u32p]
        L.oracle_stretch_z.restype = C.c_double
        L.oracle_stretch_z.argtypes = [C.c_double, C.c_double]
        L.oracle_accept.restype = i32
        L.oracle_accept.argtypes = [C.c_double, C.c_double]
        L.oracle_num_threads.restype = i32
        L.oracle_create.restype = vp
        L.oracle_create.argtypes = [C.POINTER(_Config)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_set_whitening.argtypes = [vp, dp]
        L.oracle_get_whitening.argtypes = [vp, dp]
        L.oracle_log_det_L.restype = C.c_double
        L.oracle_log_det_L.argtypes = [vp]
        L.oracle_set_step_scale.argtypes = [vp, dp]
        L.oracle_set_hard_box.argtypes = [vp, i32]
        L.oracle_set_adaptation.argtypes = [vp, i64, C.c_double]
        L.oracle_set_chain_offset.argtypes = [vp, u64]
        L.oracle_adapt_stats.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
        L.oracle_cov_chol.restype = i32
        L.oracle_cov_chol.argtypes = [vp, dp, i64, C.c_double, dp, dp]
        L.oracle_logp_grad.argtypes = [vp, dp, i64, dp, dp]
        L.oracle_mlp.argtypes = [vp, dp, i64, dp, dp]
        L.oracle_pen_f.restype = C.c_double
        L.oracle_pen_f.argtypes = [C.c_double, dp]
        L.oracle_mh_map.argtypes = [vp, dp, C.c_double, dp, C.c_double, dp, dp, dp]
        L.oracle_mala_map.argtypes = [vp, dp, C.c_double, dp, dp, C.c_double, dp, dp, dp, dp]
        L.oracle_hmc_map.argtypes = [vp, dp, C.c_double, dp, dp, C.c_double, i32, dp, dp, dp, dp, dp]
        L.oracle_aies_map.argtypes = [vp, dp, C.c_double, dp, C.c_double, dp, dp, dp]
        L.oracle_step_mh.argtypes = [vp, i64, dp, dp, u64, i64, u64, C.c_double, u64p, dp, dp, i32]
        L.oracle_step_mala.argtypes = [vp, i64, dp, dp, dp, u64, i64, u64, C.c_double, u64p, dp, dp, i32]
        L.oracle_step_hmc.argtypes = [vp, i64, dp, dp, dp, u64, i64, u64, C.c_double, i32, u64p, dp, dp, i32]
        L.oracle_de_map.argtypes = [vp, dp, C.c_double, dp, dp, C.c_double, dp, dp, dp]
        L.oracle_step_aies_de.restype = i32
        L.oracle_step_aies_de.argtypes = [vp, i64, dp, dp, u64, i64, u64, C.c_double, u64p, dp, dp, i32]
        L.oracle_step_aies.restype = i32
        L.oracle_step_aies.argtypes = [vp, i64, dp, dp, u64, i64, u64, C.c_double, u64p, dp, dp, i32]
        _LIB = L
    return _LIB


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def u01(x: int) -> float:
    return lib().oracle_u01(int(x) & 0xFFFFFFFF)


def normals(seed: int, chain: int, step: int, d: int) -> np.ndarray:
    out = np.zeros(d)
    lib().oracle_normals(seed, chain, step, d, _dp(out))
    return out


def control(seed: int, chain: int, step: int):
    u, uz, raw = C.c_double(), C.c_double(), C.c_uint32()
    lib().oracle_control(seed, chain, step, C.byref(u), C.byref(uz), C.byref(raw))
    return u.value, uz.value, raw.value


def stretch_z(u: float, a: float) -> float:
    return lib().oracle_stretch_z(u, a)


def accept(u: float, log_alpha: float) -> bool:
    return bool(lib().oracle_accept(u, log_alpha))


def pen_f(t: float):
    df = C.c_double()
    f = lib().oracle_pen_f(t, C.byref(df))
    return f, df.value


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def rminus1(trace) -> float:
    """Gelman-Rubin type statistic R − 1 of eq (4.1)-(4.2), written out from the
    text: trace [n][B][d] (n samples of each of B chains).  B = covariance of the chain means (unbiased,
    over chains), W = mean over chains of the within-chain covariances (unbiased, over samples),
    d_i = sqrt(B_ii), B~ = D^-1 B D^-1, W~ = D^-1 W D^-1, R − 1 = max_i |lambda_i(W~^-1 B~)|."""
    x = np.asarray(trace, dtype=np.float64)
    n, nb, d = x.shape
    means = x.mean(axis=0)                                        # [B][d]
    Bm = np.atleast_2d(np.cov(means, rowvar=False, ddof=1))
    W = np.zeros((d, d))
    for c in range(nb):
        W += np.atleast_2d(np.cov(x[:, c, :], rowvar=False, ddof=1))
    W /= nb
    dd = np.sqrt(np.diag(Bm))
    Bt = Bm / np.outer(dd, dd)
    Wt = W / np.outer(dd, dd)
    lam = np.linalg.eigvals(np.linalg.inv(Wt) @ Bt)
    return float(np.max(np.abs(lam)))


class Oracle:
    """One target (emulator + Gaussian + banana + box + whitening L) and the sampler steps."""

    def __init__(self, w):
        self.d = int(w.d)
        self._keep = []
        cfg = _Config()
        cfg.d = self.d
        n_affine = max(len(w.widths) - 1, 0)
        cfg.n_affine = n_affine
        if n_affine > 0:
            widths = np.asarray(w.widths, dtype=np.int32)
            Wf = np.concatenate([np.ascontiguousarray(x, dtype=np.float32).ravel() for x in w.W])
            bf = np.concatenate([np.ascontiguousarray(x, dtype=np.float32).ravel() for x in w.b])
            self._keep += [widths, Wf, bf]
            cfg.widths = widths.ctypes.data_as(C.POINTER(C.c_int32))
            cfg.W_flat = Wf.ctypes.data_as(C.POINTER(C.c_float))
            cfg.b_flat = bf.ctypes.data_as(C.POINTER(C.c_float))
        cfg.activation = int(w.activation)
        cfg.mlp_scale = float(w.mlp_scale)
        for name in ("mu", "Sigma_inv", "lo", "hi", "L"):
            arr = _f64(getattr(w, name))
            self._keep.append(arr)
            setattr(cfg, name, _dp(arr))
        cfg.pen_kappa, cfg.pen_gamma = float(w.pen_kappa), float(w.pen_gamma)
        cfg.banana_i, cfg.banana_j = int(w.banana_i), int(w.banana_j)
        cfg.banana_sigma = float(w.banana_sigma)
        self._h = lib().oracle_create(C.byref(cfg))
        if not self._h:
            raise RuntimeError("oracle_create failed")

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            lib().oracle_destroy(h)

    # ---- target -------------------------------------------------------------------------------
    def logp_grad(self, theta, want_grad=True):
        th = _f64(theta).reshape(-1, self.d)
        n = th.shape[0]
        logp = np.zeros(n)
        grad = np.zeros((n, self.d)) if want_grad else None
        lib().oracle_logp_grad(self._h, _dp(th), n, _dp(logp), _dp(grad))
        return logp, grad

    def mlp(self, theta, want_grad=True):
        th = _f64(theta).reshape(-1, self.d)
        n = th.shape[0]
        out = np.zeros(n)
        grad = np.zeros((n, self.d)) if want_grad else None
        lib().oracle_mlp(self._h, _dp(th), n, _dp(out), _dp(grad))
        return out, grad

    # ---- whitening / adaptation ---------------------------------------------------------------
    def set_whitening(self, L):
        lib().oracle_set_whitening(self._h, _dp(_f64(L)))

    def get_whitening(self):
        L = np.zeros((self.d, self.d))
        lib().oracle_get_whitening(self._h, _dp(L))
        return L

    def log_det_L(self):
        return lib().oracle_log_det_L(self._h)

    # ---- per-dimension step factors (R20), hard box (R21) -----------------------
    def set_step_scale(self, s):
        lib().oracle_set_step_scale(self._h, None if s is None else _dp(_f64(s)))

    def set_hard_box(self, on: bool):
        lib().oracle_set_hard_box(self._h, 1 if on else 0)

    def set_chain_offset(self, chain0: int):
        """local chain c draws the Philox stream of global chain id chain0 + c."""
        lib().oracle_set_chain_offset(self._h, int(chain0))

    def set_adaptation(self, adapt_every: int, jitter: float = 1e-6):
        lib().oracle_set_adaptation(self._h, adapt_every, jitter)

    def adapt_stats(self):
        a, b = C.c_int64(), C.c_int64()
        lib().oracle_adapt_stats(self._h, C.byref(a), C.byref(b))
        return a.value, b.value

    def cov_chol(self, samples, jitter=1e-6):
        s = _f64(samples).reshape(-1, self.d)
        Cm = np.zeros((self.d, self.d))
        L = np.zeros((self.d, self.d))
        rc = lib().oracle_cov_chol(self._h, _dp(s), s.shape[0], jitter, _dp(Cm), _dp(L))
        return rc, Cm, L

    # ---- deterministic maps -------------------------------------------------------------------
    def mh_map(self, theta, logp, xi, eps):
        thp, lpp, la = np.zeros(self.d), C.c_double(), C.c_double()
        lib().oracle_mh_map(self._h, _dp(_f64(theta)), logp, _dp(_f64(xi)), eps, _dp(thp),
                            C.byref(lpp), C.byref(la))
        return thp, lpp.value, la.value

    def mala_map(self, theta, logp, grad, xi, eps):
        thp, gp, lpp, la = np.zeros(self.d), np.zeros(self.d), C.c_double(), C.c_double()
        lib().oracle_mala_map(self._h, _dp(_f64(theta)), logp, _dp(_f64(grad)), _dp(_f64(xi)), eps,
                              _dp(thp), C.byref(lpp), _dp(gp), C.byref(la))
        return thp, lpp.value, gp, la.value

    def hmc_map(self, theta, logp, grad, q0, eps, n_leapfrog):
        thp, gp, qp = np.zeros(self.d), np.zeros(self.d), np.zeros(self.d)
        lpp, la = C.c_double(), C.c_double()
        lib().oracle_hmc_map(self._h, _dp(_f64(theta)), logp, _dp(_f64(grad)), _dp(_f64(q0)), eps,
                             n_leapfrog, _dp(thp), C.byref(lpp), _dp(gp), _dp(qp), C.byref(la))
        return thp, lpp.value, gp, qp, la.value

    def aies_map(self, theta_i, logp_i, theta_j, z):
        thp, lpp, la = np.zeros(self.d), C.c_double(), C.c_double()
        lib().oracle_aies_map(self._h, _dp(_f64(theta_i)), logp_i, _dp(_f64(theta_j)), z, _dp(thp),
                              C.byref(lpp), C.byref(la))
        return thp, lpp.value, la.value

    def de_map(self, theta_i, logp_i, theta_j, theta_k, gamma):
        thp = np.zeros(self.d)
        lpp, la = C.c_double(), C.c_double()
        lib().oracle_de_map(self._h, _dp(_f64(theta_i)), logp_i, _dp(_f64(theta_j)), _dp(_f64(theta_k)), gamma,
                            _dp(thp), C.byref(lpp), C.byref(la))
        return thp, lpp.value, la.value

    # ---- chains -------------------------------------------------------------------------------
    def new_state(self, theta0):
        return OracleState(self, theta0)


class OracleState:
    """Chain state (θ, cached log π and ∇θ log π, global step counter, accept counters)."""

    def __init__(self, oracle: Oracle, theta0):
        self.o = oracle
        self.theta = _f64(theta0).reshape(-1, oracle.d).copy()
        self.B = self.theta.shape[0]
        self.logp, self.grad = oracle.logp_grad(self.theta)
        self.step = 0
        self.n_accept = np.zeros(self.B, dtype=np.uint64)
        self.n_evals = self.B
        self.last_log_alpha = np.zeros(self.B)

    def _trace(self, n, thin):
        if not thin:
            return None
        return np.zeros((n // thin, self.B, self.o.d))

    def _u64p(self):
        return self.n_accept.ctypes.data_as(C.POINTER(C.c_uint64))

    def step_mh(self, n_steps, seed, eps, thin=0):
        tr = self._trace(n_steps, thin)
        lib().oracle_step_mh(self.o._h, self.B, _dp(self.theta), _dp(self.logp), self.step, n_steps,
                             seed, eps, self._u64p(), _dp(self.last_log_alpha), _dp(tr), thin)
        self.step += n_steps
        self.n_evals += self.B * n_steps
        return tr

    def step_mala(self, n_steps, seed, eps, thin=0):
        tr = self._trace(n_steps, thin)
        lib().oracle_step_mala(self.o._h, self.B, _dp(self.theta), _dp(self.logp), _dp(self.grad),
                               self.step, n_steps, seed, eps, self._u64p(),
                               _dp(self.last_log_alpha), _dp(tr), thin)
        self.step += n_steps
        self.n_evals += self.B * n_steps
        return tr

    def step_hmc(self, n_traj, seed, eps, n_leapfrog, thin=0):
        tr = self._trace(n_traj, thin)
        lib().oracle_step_hmc(self.o._h, self.B, _dp(self.theta), _dp(self.logp), _dp(self.grad),
                              self.step, n_traj, seed, eps, n_leapfrog, self._u64p(),
                              _dp(self.last_log_alpha), _dp(tr), thin)
        self.step += n_traj
        self.n_evals += self.B * n_traj * n_leapfrog
        return tr

    # ---- burn-in loop (reading R22) ----------------------
    def _step(self, method, n, seed, eps, n_leapfrog):
        if method == "mh":
            self.step_mh(n, seed, eps)
        elif method == "mala":
            self.step_mala(n, seed, eps)
        elif method == "hmc":
            self.step_hmc(n, seed, eps, n_leapfrog)
        else:
            raise ValueError("burn-in loop: mh, mala or hmc (the paper runs none for AIES, P:L260)")

    def burn_in(self, method, n_iter, n_steps, n_adapt, block, seed, eps0, target_accept,
                n_leapfrog=1, jitter=1e-6):
        """n_iter burn-in iterations of n_steps steps each.  In every iteration the first
        n_adapt steps adapt the step size and are then discarded; the covariance of all chains
        over the remaining n_steps − n_adapt steps replaces the whitening factor (O6), and
        the best-fit point (largest log π over the ensemble, kept over iterations) is updated.
        The paper gives no adaptation rule: reading R22 = Nesterov dual averaging as in Hoffman & Gelman
        (2014, Alg. 5; γ = 0.05, t₀ = 10, κ = 0.75, μ = log 10ε) on the acceptance FRACTION of the whole
        ensemble over blocks of `block` steps, restarted in each iteration from the current ε.
        ε crosses the sampler interface as float32, like on the C-ABI.  Returns (ε, θ_best, log π_best,
        [ε used in each block])."""
        GAMMA, T0, KAPPA = 0.05, 10.0, 0.75
        import math
        eps = float(np.float32(eps0))
        best_lp, best_th, hist = -math.inf, None, []
        for _ in range(n_iter):
            if n_adapt > 0:
                mu, hbar, logeps_bar, m, cur, done = math.log(10.0 * eps), 0.0, 0.0, 0, eps, 0
                while done < n_adapt:
                    nb = min(block, n_adapt - done)
                    a0 = int(self.n_accept.sum())
                    cur32 = float(np.float32(cur))
                    hist.append(cur32)
                    self._step(method, nb, seed, cur32, n_leapfrog)
                    alpha = (int(self.n_accept.sum()) - a0) / float(self.B * nb)
                    m += 1
                    hbar = (1.0 - 1.0 / (m + T0)) * hbar + (target_accept - alpha) / (m + T0)
                    logeps = mu - math.sqrt(m) / GAMMA * hbar
                    eta = math.pow(m, -KAPPA)
                    logeps_bar = eta * logeps + (1.0 - eta) * logeps_bar
                    cur = math.exp(logeps)
                    done += nb
                eps = float(np.float32(math.exp(logeps_bar)))
            win = n_steps - n_adapt
            if win > 0:
                self.o.set_adaptation(win, jitter)
                self._step(method, win, seed, eps, n_leapfrog)
                self.o.set_adaptation(0, jitter)
            i = int(np.argmax(self.logp))
            if self.logp[i] > best_lp:
                best_lp, best_th = float(self.logp[i]), self.theta[i].copy()
        return eps, best_th, best_lp, hist

    def step_aies(self, n_steps, seed, a=2.0, thin=0):
        tr = self._trace(n_steps, thin)
        rc = lib().oracle_step_aies(self.o._h, self.B, _dp(self.theta), _dp(self.logp), self.step,
                                    n_steps, seed, a, self._u64p(), _dp(self.last_log_alpha),
                                    _dp(tr), thin)
        if rc != 0:
            raise ValueError("oracle_step_aies: bad arguments")
        self.step += n_steps
        self.n_evals += self.B * n_steps
        return tr

    def step_aies_de(self, n_steps, seed, sigma_gamma=1e-5, thin=0):
        """Differential-evolution move, eq (2.16) (reading R23)."""
        tr = self._trace(n_steps, thin)
        rc = lib().oracle_step_aies_de(self.o._h, self.B, _dp(self.theta), _dp(self.logp), self.step,
                                       n_steps, seed, sigma_gamma, self._u64p(), _dp(self.last_log_alpha),
                                       _dp(tr), thin)
        if rc != 0:
            raise ValueError("oracle_step_aies_de: bad arguments")
        self.step += n_steps
        self.n_evals += self.B * n_steps
        return tr
