"""Tolerance definitions shared by the GPU parity tests (reading R17/R8)."""
import numpy as np

TOL = {0: 1e-5, 1: 2e-2}   # precision enum → relative tolerance (north_star)


def check_logp_grad(lp, g, lp_ref, g_ref, tol, what=""):
    """logp: |Δ| ≤ tol·max_batch|logp_ref|; gradient: per point ‖Δg‖₂ ≤ tol·‖g_ref‖₂ (no floor)."""
    S = np.abs(lp_ref).max()
    err_lp = np.abs(lp.astype(np.float64) - lp_ref).max()
    # the boundary is fp32: allow its rounding of the value itself (half an ulp of S) on top
    assert err_lp <= tol * S + 6e-8 * S, f"{what}: logp err {err_lp:.3e} vs scale {S:.3e}"
    if g is not None:
        num = np.linalg.norm(g.astype(np.float64) - g_ref, axis=1)
        den = np.linalg.norm(g_ref, axis=1)
        ok = den > 0
        ratio = (num[ok] / den[ok]).max() if ok.any() else 0.0
        assert ratio <= tol + 2e-7, f"{what}: grad norm ratio {ratio:.3e}"
        return err_lp / S, ratio
    return err_lp / S, 0.0


def accept_margins(O, seed, step, B, log_alpha_ref, chains=None):
    """m = |log u − log α_oracle| for every chain (reading R8)."""
    idx = range(B) if chains is None else chains
    u = np.array([O.control(seed, int(c), step)[0] for c in idx])
    return np.abs(np.log(u) - log_alpha_ref)


def log_alpha_bound(O, orc, w, method, theta0, grad0, seed, step, kw, chain0=0, step_scale=None):
    """Upper bound on |log α_gpu − log α_oracle| of ONE bf16-path step, derived from north_star's tolerances
    (DESIGN.md §2 "bound on Δ log α"), from oracle-side quantities only:

      e_lp = TOL · s · max|MLP(θ₀)|   error scale of one log π evaluation (R17: the tolerance applies to the
                                      MLP-only target; the Gaussian / banana / box algebra is fp32-exact to `slack`)
      e_g  = TOL · s · max‖∇MLP(θ₀)‖₂ error scale of one gradient, θ space;  λ = ‖L diag(s)‖₂ maps it to z space

      MH, stretch, DE:  log α = log π(θ′) − log π(θ) (+ exact terms)            ⇒ 2 e_lp
      MALA:  + Hastings term −‖r‖²/(4ε) + …, r = ε(g_z + g_z′) + √(2ε) ξ;  ∂/∂g_z = −r/2 each
                                                                              ⇒ + ρ λ e_g,  ρ = max ‖r‖
      HMC:   every one of the L kicks adds ε δg_z to q, every later drift carries it on:
             |δq| ≤ L ε λ e_g,  |δz| ≤ (L ε)² λ e_g / 2;  δ(½‖q‖²) ≤ ‖q‖ |δq|,  δ log π ≤ ‖g_z‖ |δz|
                                                                              ⇒ + ρ (Lε + (Lε)²/2) λ e_g
    ρ is taken over the batch from the oracle's start gradients and normals, with ‖g_z′‖ ≤ 1.5 max‖g_z‖.
    `slack` = 3e-5 · max|log π| covers the fp32 algebra around the emulator (measured ≤ 2e-6 · S on the exact path)."""
    tol = TOL[1]
    n = theta0.shape[0]
    out, g = orc.mlp(theta0, want_grad=True)
    s = abs(float(w.mlp_scale))
    e_lp = tol * s * float(np.abs(out).max())
    e_g = tol * s * float(np.linalg.norm(g, axis=1).max())
    Ls = orc.get_whitening()
    if step_scale is not None:                            # R20: the step maps use L diag(s)
        Ls = Ls * np.asarray(step_scale)[None, :]
    lam = float(np.linalg.norm(Ls, 2))
    lp0, _ = orc.logp_grad(theta0, want_grad=False)
    fin = np.isfinite(lp0)
    slack = 3e-5 * float(np.abs(lp0[fin]).max()) if fin.any() else 0.0
    bound = 2.0 * e_lp + slack
    if method in ("mala", "hmc"):
        eps = float(kw["eps"])
        gz = grad0 @ Ls                                   # rows: (Lᵀ g)ᵀ
        gzn = float(np.linalg.norm(gz, axis=1).max())
        xin = max(float(np.linalg.norm(O.normals(seed, chain0 + c, step, w.d))) for c in range(0, n, max(1, n // 512)))
        if method == "mala":
            rho = 2.5 * eps * gzn + np.sqrt(2.0 * eps) * 1.25 * xin      # 1.25: max over all chains vs the sampled ones
            bound += rho * lam * e_g
        else:
            nl = int(kw["n_leapfrog"])
            le = nl * eps
            rho = max(1.25 * xin + le * 1.5 * gzn, 1.5 * gzn)
            bound += rho * (le + 0.5 * le * le) * lam * e_g
    return bound, dict(e_lp=e_lp, e_g=e_g, lam=lam, slack=slack)


def expected_mismatches(la_gpu, la_ref):
    """A chain accepts iff u < exp(log α) with u uniform (R7: NaN ⇒ reject), and both sides hold the same u, so the
    decisions differ iff u lies between the two acceptance probabilities:
    E[#mismatches] = Σ_i |min(1, e^{log α_gpu,i}) − min(1, e^{log α_ref,i})|  (exact)."""
    def p(la):
        la = np.where(np.isnan(la), -np.inf, la)
        with np.errstate(over="ignore"):
            return np.minimum(1.0, np.exp(np.minimum(la, 0.0)))
    return float(np.abs(p(np.asarray(la_gpu, dtype=np.float64)) - p(np.asarray(la_ref, dtype=np.float64))).sum())
