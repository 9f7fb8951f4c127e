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
