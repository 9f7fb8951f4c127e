"""Pins for SURVEY §8(f)#1 in the oracle: per-dimension step factors (reading R20) and the hard box
(reading R21).  Closed forms on an exactly whitened Gaussian (every coordinate of z is an independent
standard normal, so each formula factorises per dimension with its own step), the 1-d reduction to a
scalar step on a non-Gaussian target, and the uniform law inside a hard box."""
import math

import numpy as np
import pytest

from paper_2606_04895_b200 import workloads as WL


def _whitened_gaussian(oracle_mod, d, seed, s):
    w = WL.gaussian(d, 4, seed=seed)
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    o.set_step_scale(s)
    return w, o


def test_mh_per_dimension_step_closed_form(oracle_mod):
    """θ' = θ + L(ε s⊙ξ); on the whitened Gaussian log α = ½(‖z‖² − ‖z'‖²), z' = z + ε s⊙ξ."""
    d = 5
    s = np.array([1.0, 10.0, 0.3, 2.5, 0.05])
    w, o = _whitened_gaussian(oracle_mod, d, 21, s)
    rng = np.random.default_rng(4)
    Linv = np.linalg.inv(w.L)
    for eps in (0.05, 0.3):
        for _ in range(5):
            x = w.mu + w.L @ rng.standard_normal(d)
            xi = rng.standard_normal(d)
            lp = o.logp_grad(x[None, :], want_grad=False)[0][0]
            xp, lpp, la = o.mh_map(x, lp, xi, eps)
            z = Linv @ (x - w.mu)
            zp = z + eps * s * xi
            np.testing.assert_allclose(xp, w.mu + w.L @ zp, rtol=0, atol=1e-11)
            assert la == pytest.approx(0.5 * (z @ z - zp @ zp), abs=1e-10)


def test_mala_per_dimension_step_closed_form(oracle_mod):
    """g_z = −z: z'_i = (1 − ε_i) z_i + √(2ε_i) ξ_i with ε_i = ε s_i², log α = Σ_i (ε_i/4)(z_i² − z'_i²)."""
    d = 5
    s = np.array([1.0, 3.0, 0.3, 1.7, 0.1])
    w, o = _whitened_gaussian(oracle_mod, d, 22, s)
    rng = np.random.default_rng(6)
    Linv = np.linalg.inv(w.L)
    for eps in (0.02, 0.1):
        ei = eps * s * s
        for _ in range(5):
            x = w.mu + w.L @ rng.standard_normal(d)
            xi = rng.standard_normal(d)
            lp, g = o.logp_grad(x[None, :])
            xp, lpp, gp, la = o.mala_map(x, lp[0], g[0], xi, eps)
            z = Linv @ (x - w.mu)
            zp = (1.0 - ei) * z + np.sqrt(2.0 * ei) * xi
            np.testing.assert_allclose(xp, w.mu + w.L @ zp, rtol=0, atol=1e-11)
            assert la == pytest.approx(float(np.sum(ei / 4.0 * (z * z - zp * zp))), abs=1e-10)


def test_hmc_per_dimension_step_linear_map(oracle_mod):
    """Standard normal: coordinate i is a harmonic oscillator stepped with h_i = ε s_i; one KDK step is
    [[1−h²/2, h],[−h(1−h²/4), 1−h²/2]] on (z_i, q_i); log α = H0 − H1 with H = ½‖z‖² + ½‖q‖²."""
    d = 4
    w = WL.gaussian(d, 1, seed=2)
    w.mu, w.Sigma, w.Sigma_inv, w.L = np.zeros(d), np.eye(d), np.eye(d), np.eye(d)
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    s = np.array([1.0, 4.0, 0.25, 2.0])
    o.set_step_scale(s)
    rng = np.random.default_rng(8)
    for eps, nl in ((0.1, 1), (0.2, 8), (0.05, 16)):
        x, q = rng.standard_normal(d), rng.standard_normal(d)
        lp, g = o.logp_grad(x[None, :])
        xp, lpp, gp, qp, la = o.hmc_map(x, lp[0], g[0], q, eps, nl)
        for i in range(d):
            h = eps * s[i]
            M = np.array([[1 - h ** 2 / 2, h], [-h * (1 - h ** 2 / 4), 1 - h ** 2 / 2]])
            ref = np.linalg.matrix_power(M, nl) @ np.array([x[i], q[i]])
            assert xp[i] == pytest.approx(ref[0], abs=1e-13)
            assert qp[i] == pytest.approx(ref[1], abs=1e-13)
        H0 = 0.5 * x @ x + 0.5 * q @ q
        H1 = 0.5 * xp @ xp + 0.5 * qp @ qp
        assert la == pytest.approx(H0 - H1, abs=1e-12)


def test_scalar_factor_reduces_to_scaled_eps_on_nongaussian_target(oracle_mod):
    """d = 1, non-Gaussian target, L ≠ 1: factor s ≡ step ε s (MH, HMC) and ε s² (MALA)."""
    w = WL.tiny(n_chains=1, seed=77, d=1, hidden=(8, 8), mlp_scale=1.5)
    w.lo = w.hi = None
    w.L = np.array([[0.7]])
    o1, os_ = oracle_mod.Oracle(w), oracle_mod.Oracle(w)
    s, eps = 2.5, 0.11
    os_.set_step_scale(np.array([s]))
    x = w.theta0[0].astype(np.float64)
    lp, g = o1.logp_grad(x[None, :])
    xi = np.array([0.37])
    a, b = os_.mh_map(x, lp[0], xi, eps), o1.mh_map(x, lp[0], xi, eps * s)
    for u, v in zip(a, b):
        np.testing.assert_allclose(u, v, rtol=0, atol=1e-13)
    a, b = os_.mala_map(x, lp[0], g[0], xi, eps), o1.mala_map(x, lp[0], g[0], xi, eps * s * s)
    for u, v in zip(a, b):
        np.testing.assert_allclose(u, v, rtol=0, atol=1e-12)
    a, b = os_.hmc_map(x, lp[0], g[0], xi, eps, 5), o1.hmc_map(x, lp[0], g[0], xi, eps * s, 5)
    for u, v in zip(a, b):
        np.testing.assert_allclose(u, v, rtol=0, atol=1e-12)


@pytest.mark.parametrize("method", ["mh", "mala", "hmc"])
def test_moments_with_unmatched_step_factors(oracle_mod, method):
    """Any positive s leaves the target invariant: closed-form Gaussian moments within 4 MC standard errors."""
    d = 3
    w = WL.gaussian(d, 256, seed=33, cond=30.0)
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    o.set_step_scale(np.array([0.5, 1.0, 1.8]))
    st = o.new_state(w.theta0)
    kw = dict(mh=dict(eps=0.9), mala=dict(eps=0.35), hmc=dict(eps=0.45, n_leapfrog=4))[method]
    getattr(st, "step_" + method)(300, 11, **kw)
    tr = getattr(st, "step_" + method)(400, 11, thin=4, **kw)
    x = tr.reshape(-1, d)
    # effective sample size: chains are independent, thinned draws are not -> use per-chain means
    cm = tr.mean(axis=0)                      # [B, d]
    se = cm.std(axis=0, ddof=1) / math.sqrt(cm.shape[0])
    assert np.all(np.abs(cm.mean(axis=0) - w.mu) < 4.0 * se + 1e-12)
    var = ((tr - w.mu) ** 2).mean(axis=0)     # [B, d] per-chain second moments
    se_v = var.std(axis=0, ddof=1) / math.sqrt(var.shape[0])
    assert np.all(np.abs(var.mean(axis=0) - np.diag(w.Sigma)) < 4.0 * se_v)
    assert x.shape[0] == 100 * 256


def test_hard_box_value_and_uniform_law(oracle_mod):
    """Inside the box the hard-box target equals the box-free one; outside it is −∞ (rejected).  A flat
    target in a hard box is the uniform law: mean (lo+hi)/2, variance (hi−lo)²/12, never outside."""
    w = WL.tiny(n_chains=64, seed=5, d=3, hidden=(8, 8), mlp_scale=0.7)
    wf = WL.tiny(n_chains=64, seed=5, d=3, hidden=(8, 8), mlp_scale=0.7)
    wf.lo = wf.hi = None
    o_free = oracle_mod.Oracle(wf)
    o = oracle_mod.Oracle(w)
    o.set_hard_box(True)
    mid = 0.5 * (w.lo + w.hi)
    pts = np.stack([mid, mid + 0.49 * (w.hi - w.lo), w.lo.copy(), w.hi.copy()])
    lp, g = o.logp_grad(pts)
    lpf, gf = o_free.logp_grad(pts)
    np.testing.assert_array_equal(lp, lpf)            # the boundary belongs to the box
    np.testing.assert_array_equal(g, gf)
    out = np.stack([mid + np.array([0.0, 0.51, 0.0]) * (w.hi - w.lo), w.lo - 1e-9])
    lpo, _ = o.logp_grad(out)
    assert np.all(np.isneginf(lpo))
    # a proposal outside is rejected whatever u is
    x = mid.copy()
    xi = np.array([0.0, 1.0, 0.0])
    w.L = np.eye(3)
    o.set_whitening(np.eye(3))
    thp, lpp, la = o.mh_map(x, lp[0], xi, float(w.hi[1] - w.lo[1]))
    assert la == -math.inf and not oracle_mod.accept(1e-300, la)
    # uniform law
    d = 2
    wu = WL.gaussian(d, 512, seed=9)
    wu.mu = wu.Sigma = wu.Sigma_inv = None
    wu.lo, wu.hi = np.array([-1.0, 2.0]), np.array([1.0, 2.5])
    wu.L = np.diag([1.0, 0.25])
    rng = np.random.default_rng(2)
    wu.theta0 = (wu.lo + (wu.hi - wu.lo) * rng.random((512, d))).astype(np.float32)
    ou = oracle_mod.Oracle(wu)
    ou.set_hard_box(True)
    st = ou.new_state(wu.theta0)
    st.step_mh(100, 3, eps=0.8)
    tr = st.step_mh(400, 3, eps=0.8, thin=4)
    assert np.all(tr >= wu.lo) and np.all(tr <= wu.hi)
    cm = tr.mean(axis=0)
    se = cm.std(axis=0, ddof=1) / math.sqrt(cm.shape[0])
    assert np.all(np.abs(cm.mean(axis=0) - 0.5 * (wu.lo + wu.hi)) < 4.0 * se)
    v = ((tr - 0.5 * (wu.lo + wu.hi)) ** 2).mean(axis=0)
    se_v = v.std(axis=0, ddof=1) / math.sqrt(v.shape[0])
    assert np.all(np.abs(v.mean(axis=0) - (wu.hi - wu.lo) ** 2 / 12.0) < 4.0 * se_v)
