"""Seeded synthetic workload generators (inputs only — none of the method's arithmetic lives here).

Both the CPU oracle (``oracle/``) and the CUDA library (``libbest.so``) are fed the arrays
produced here.  The recipes follow SURVEY.md §8(d) / BASELINE.json ``configs`` and stand in for
the paper's trained CLiENT emulators (27-d ΛCDM, 29-d sterile-ν), which are
not available.  Everything is generated in fp64 with ``numpy.random.default_rng(seed)`` and the
MLP arrays are rounded to fp32 (the type of the C-ABI boundary).

Only library routines used to *construct inputs* appear here (QR, Cholesky, inverse).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

ACT_TANH = 0
ACT_SILU = 1
PREC_FP32 = 0
PREC_BF16 = 1


@dataclass
class Workload:
    name: str
    d: int
    widths: List[int]                 # [d, n1, ..., nK, 1]; [] => no MLP
    W: List[np.ndarray]               # W[k]: float32 [widths[k+1], widths[k]]
    b: List[np.ndarray]               # b[k]: float32 [widths[k+1]]
    activation: int
    mlp_scale: float
    mu: Optional[np.ndarray]          # float64 [d] or None
    Sigma: Optional[np.ndarray]       # float64 [d,d] (what Sigma_inv inverts; for tests)
    Sigma_inv: Optional[np.ndarray]   # float64 [d,d] or None
    lo: Optional[np.ndarray]
    hi: Optional[np.ndarray]
    pen_kappa: float = 1.0
    pen_gamma: float = 100.0
    banana_i: int = -1
    banana_j: int = -1
    banana_sigma: float = 0.1
    L: Optional[np.ndarray] = None    # float64 [d,d] lower-triangular whitening factor
    n_chains: int = 0
    theta0: Optional[np.ndarray] = None  # float32 [n_chains, d]
    params: dict = field(default_factory=dict)

    @property
    def macs(self) -> int:
        return int(sum(self.widths[k] * self.widths[k + 1] for k in range(len(self.widths) - 1)))

    def with_chains(self, n_chains: int, seed: int) -> "Workload":
        """Same target, a different number of chains (θ₀ redrawn from ``seed``)."""
        import copy
        w = copy.copy(self)
        w.n_chains = n_chains
        w.theta0 = _theta0(np.random.default_rng(seed), self, n_chains)
        return w


def make_mlp(rng: np.random.Generator, widths: List[int]):
    """Xavier-normal weights N(0, 2/(fan_in+fan_out)), biases N(0, 0.1²)."""
    W, b = [], []
    for k in range(len(widths) - 1):
        fan_in, fan_out = widths[k], widths[k + 1]
        std = np.sqrt(2.0 / (fan_in + fan_out))
        W.append((rng.standard_normal((fan_out, fan_in)) * std).astype(np.float32))
        b.append((rng.standard_normal(fan_out) * 0.1).astype(np.float32))
    return W, b


def _sigma_cond(rng: np.random.Generator, d: int, lam_min: float, lam_max: float) -> np.ndarray:
    """Σ = Q diag(λ) Qᵀ, λ log-uniform in [lam_min, lam_max] with both ends pinned."""
    lam = np.exp(rng.uniform(np.log(lam_min), np.log(lam_max), size=d))
    lam[0], lam[-1] = lam_min, lam_max
    Q, _ = np.linalg.qr(rng.standard_normal((d, d)))
    S = (Q * lam) @ Q.T
    return 0.5 * (S + S.T)


def _theta0(rng: np.random.Generator, w: Workload, n: int) -> np.ndarray:
    Lc = np.linalg.cholesky(w.Sigma)
    th = w.mu[None, :] + rng.standard_normal((n, w.d)) @ Lc.T
    if w.banana_i >= 0:
        th[:, w.banana_j] = th[:, w.banana_i] ** 2 + w.banana_sigma * rng.standard_normal(n)
    return th.astype(np.float32)


def tiny(n_chains: int = 64, seed: int = 1001, activation: int = ACT_TANH,
         mlp_scale: float = 0.1, d: int = 6, hidden=(64, 64)) -> Workload:
    """BASELINE configs[0]: d=6, Σ = GᵀG/(d+2), MLP 6→64→64→1 tanh, s=0.1, box μ ± 10σ."""
    rng = np.random.default_rng(seed)
    mu = rng.standard_normal(d)
    G = rng.standard_normal((d + 2, d))
    Sigma = G.T @ G / (d + 2)
    widths = [d, *hidden, 1]
    W, b = make_mlp(rng, widths)
    sig = np.sqrt(np.diag(Sigma))
    w = Workload("tiny", d, widths, W, b, activation, mlp_scale, mu, Sigma, np.linalg.inv(Sigma),
                 mu - 10 * sig, mu + 10 * sig, L=np.linalg.cholesky(Sigma), n_chains=n_chains,
                 params=dict(eps_mh=0.3, eps_mala=0.3, n_steps=1000))
    w.theta0 = _theta0(rng, w, n_chains)
    return w


def lcdm(n_chains: int = 4096, seed: int = 1002, mlp_scale: float = 1.0, hidden: int = 512,
         n_hidden: int = 4, d: int = 27) -> Workload:
    """BASELINE configs[1]/[2]: d=27, cond(Σ)=1e4, MLP 27→512⁴→1 SiLU (s=1 MALA, s=3 HMC)."""
    rng = np.random.default_rng(seed)
    mu = rng.standard_normal(d)
    Sigma = _sigma_cond(rng, d, 1e-2, 1e2)
    widths = [d] + [hidden] * n_hidden + [1]
    W, b = make_mlp(rng, widths)
    sig = np.sqrt(np.diag(Sigma))
    w = Workload("lcdm", d, widths, W, b, ACT_SILU, mlp_scale, mu, Sigma, np.linalg.inv(Sigma),
                 mu - 10 * sig, mu + 10 * sig, L=np.linalg.cholesky(Sigma), n_chains=n_chains,
                 params=dict(eps_mh=0.3, eps_mala=0.3, eps_hmc=0.1, n_leapfrog=16))
    w.theta0 = _theta0(rng, w, n_chains)
    return w


def sterile(n_chains: int = 32768, seed: int = 1004, mlp_scale: float = 1.0, hidden: int = 1024,
            n_hidden: int = 4) -> Workload:
    """BASELINE configs[3]/[4]: d=29 = 27 + 2 banana-coupled dims, MLP 29→1024⁴→1 SiLU."""
    rng = np.random.default_rng(seed)
    d27, d = 27, 29
    mu = rng.standard_normal(d)
    Sigma = np.eye(d)
    Sigma[:d27, :d27] = _sigma_cond(rng, d27, 1e-2, 1e2)
    widths = [d] + [hidden] * n_hidden + [1]
    W, b = make_mlp(rng, widths)
    sig = np.sqrt(np.diag(Sigma))
    lo, hi = mu - 10 * sig, mu + 10 * sig
    # the banana ridge θ28 ≈ θ27² reaches beyond μ28+10: widen that face so θ₀ starts inside
    hi[28] = max(hi[28], (abs(mu[27]) + 10.0) ** 2)
    w = Workload("sterile", d, widths, W, b, ACT_SILU, mlp_scale, mu, Sigma, np.linalg.inv(Sigma),
                 lo, hi, banana_i=27, banana_j=28, banana_sigma=0.1,
                 L=np.linalg.cholesky(Sigma), n_chains=n_chains,
                 params=dict(a=2.0, eps_mh=0.3, eps_mala=0.01, eps_hmc=0.03, n_leapfrog=8,
                             adapt_every=500))
    w.theta0 = _theta0(rng, w, n_chains)
    return w


def gaussian(d: int, n_chains: int, seed: int, cond: float = 100.0) -> Workload:
    """Closed-form target: s=0, no MLP, no banana, box ±10σ ⇒ posterior N(μ, Σ) (north_star)."""
    rng = np.random.default_rng(seed)
    mu = rng.standard_normal(d)
    Sigma = _sigma_cond(rng, d, 1.0 / np.sqrt(cond), np.sqrt(cond)) if d > 1 else np.array([[1.7]])
    sig = np.sqrt(np.diag(Sigma))
    w = Workload("gaussian", d, [], [], [], ACT_TANH, 0.0, mu, Sigma, np.linalg.inv(Sigma),
                 mu - 10 * sig, mu + 10 * sig, L=np.linalg.cholesky(Sigma), n_chains=n_chains)
    w.theta0 = _theta0(rng, w, n_chains)
    return w


def mlp_only(base: Workload) -> Workload:
    """Same MLP, s=1, no Gaussian/box/banana terms (exposes emulator errors)."""
    import copy
    w = copy.copy(base)
    w.name = base.name + "_mlp_only"
    w.mlp_scale = 1.0
    w.mu = None
    w.Sigma_inv = None
    w.lo = w.hi = None
    w.banana_i = w.banana_j = -1
    return w


def gaussian_only(base: Workload) -> Workload:
    import copy
    w = copy.copy(base)
    w.name = base.name + "_gauss_only"
    w.widths, w.W, w.b = [], [], []
    w.mlp_scale = 0.0
    return w


def probe_points(w: Workload, n: int, seed: int) -> np.ndarray:
    """T1 evaluation points: posterior-like draws, box-face / just-outside points, ±20σ outliers,
    and (banana targets) on/off-ridge points.  float32 [n, d]."""
    rng = np.random.default_rng(seed)
    Lc = np.linalg.cholesky(w.Sigma)
    sig = np.sqrt(np.diag(w.Sigma))
    th = w.mu[None, :] + rng.standard_normal((n, w.d)) @ Lc.T
    if w.banana_i >= 0:
        on = rng.random(n) < 0.5
        ridge = th[:, w.banana_i] ** 2 + w.banana_sigma * rng.standard_normal(n)
        th[:, w.banana_j] = np.where(on, ridge, th[:, w.banana_j])
    q = n // 8
    if w.lo is not None and q > 0:
        # on the faces, and 0.5% / 3% of the box width outside them
        for blk, frac in enumerate((0.0, 0.005, 0.03)):
            rows = slice(blk * q // 2, (blk + 1) * q // 2)
            nrow = th[rows].shape[0]
            dims = rng.integers(0, w.d, size=nrow)
            side = rng.integers(0, 2, size=nrow)
            width = (w.hi - w.lo)[dims]
            val = np.where(side == 0, w.lo[dims] - frac * width, w.hi[dims] + frac * width)
            th[np.arange(rows.start, rows.start + nrow), dims] = val
    if q > 0:
        rows = slice(n - q // 2, n)
        nrow = th[rows].shape[0]
        th[rows] = w.mu[None, :] + 20.0 * sig[None, :] * rng.choice([-1.0, 1.0], size=(nrow, w.d)) \
            * (rng.random((nrow, w.d)) < 0.15)
    return th.astype(np.float32)
