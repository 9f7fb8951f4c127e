"""Brute-force detailed-balance and closed-form pins for the oracle's single-step maps
(SURVEY §8(c) "What pins each part": MH lattice, MALA pairs + whitened-Gaussian closed form,
HMC linear map / reversibility / volume / phase-space balance)."""
import math

import numpy as np
import pytest

from paper_2606_04895_b200 import workloads as WL


def _target_1d(oracle_mod, L=1.0, scale=1.5):
    """d=1 non-Gaussian target: Gaussian term + tanh MLP 1→8→8→1."""
    w = WL.tiny(n_chains=1, seed=77, d=1, hidden=(8, 8), mlp_scale=scale)
    w.lo = w.hi = None
    w.L = np.array([[L]])
    return w, oracle_mod.Oracle(w)


def _acc_prob(log_alpha):
    """P(log u < log α) for u ~ U(0,1) (the accept rule R7)."""
    return 1.0 if log_alpha >= 0 else math.exp(log_alpha)


def test_mh_detailed_balance_lattice(oracle_mod):
    w, o = _target_1d(oracle_mod, L=0.7)
    n, h = 41, 0.15
    xs = w.mu[0] + (np.arange(n) - n // 2) * h
    logp = np.array([o.logp_grad(np.array([[x]]), want_grad=False)[0][0] for x in xs])
    assert np.ptp(logp) > 1.0
    pi = np.exp(logp - logp.max())
    pi /= pi.sum()
    offsets = {-3: 0.1, -2: 0.15, -1: 0.25, 1: 0.25, 2: 0.15, 3: 0.1}   # symmetric weights
    eps = 0.3
    P = np.zeros((n, n))
    for i in range(n):
        for m, wgt in offsets.items():
            j = i + m
            if not 0 <= j < n:
                continue                                   # proposal off the lattice ⇒ rejected
            xi = np.array([m * h / (eps * 0.7)])           # θ' = θ + ε L ξ lands on lattice point j
            thp, lpp, la = o.mh_map(np.array([xs[i]]), logp[i], xi, eps)
            assert thp[0] == pytest.approx(xs[j], abs=1e-13)
            assert lpp == pytest.approx(logp[j], abs=1e-13)
            P[i, j] = wgt * _acc_prob(la)
        P[i, i] = 1.0 - P[i].sum()
    F = pi[:, None] * P
    assert np.abs(F - F.T).max() < 1e-14
    assert np.abs(pi @ P - pi).max() < 1e-14


def test_mala_closed_form_whitened_gaussian(oracle_mod):
    """Exactly whitened Gaussian: g_z = −z ⇒ log α = (ε/4)(‖z‖² − ‖z'‖²)."""
    w = WL.gaussian(5, 4, seed=21)
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    rng = np.random.default_rng(3)
    Linv = np.linalg.inv(w.L)
    for eps in (0.05, 0.3, 0.9):
        for _ in range(5):
            th = w.mu + w.L @ rng.standard_normal(5) * 1.3
            xi = rng.standard_normal(5)
            lp, g = o.logp_grad(th[None, :])
            thp, lpp, gp, la = o.mala_map(th, lp[0], g[0], xi, eps)
            z, zp = Linv @ (th - w.mu), Linv @ (thp - w.mu)
            # proposal eq (2.3) in z:  z' = z + ε(−z) + sqrt(2ε) ξ
            np.testing.assert_allclose(zp, z - eps * z + math.sqrt(2 * eps) * xi, atol=1e-12)
            assert la == pytest.approx(0.25 * eps * (z @ z - zp @ zp), abs=1e-11)


def test_mala_map_uses_L_and_LT_correctly(oracle_mod):
    """θ' = θ + L(ε Lᵀ∇ + sqrt(2ε) ξ) with numpy matmuls (catches a transposed operand)."""
    w = WL.lcdm(n_chains=2, hidden=16, n_hidden=2)
    o = oracle_mod.Oracle(w)
    rng = np.random.default_rng(8)
    th = w.theta0[0].astype(np.float64)
    xi = rng.standard_normal(w.d)
    lp, g = o.logp_grad(th[None, :])
    eps = 0.2
    thp, lpp, gp, la = o.mala_map(th, lp[0], g[0], xi, eps)
    np.testing.assert_allclose(thp, th + w.L @ (eps * (w.L.T @ g[0]) + math.sqrt(2 * eps) * xi),
                               rtol=1e-12, atol=1e-12)
    lp2, g2 = o.logp_grad(thp[None, :])
    assert lpp == lp2[0] and np.array_equal(gp, g2[0])
    # Hastings ratio from the Gaussian proposal densities N(z + ε g_z, 2ε·1) written with scipy
    from scipy import stats
    Linv = np.linalg.inv(w.L)
    z, zp = Linv @ th, Linv @ thp
    gz, gzp = w.L.T @ g[0], w.L.T @ g2[0]
    fwd = stats.multivariate_normal(z + eps * gz, 2 * eps * np.eye(w.d)).logpdf(zp)
    bwd = stats.multivariate_normal(zp + eps * gzp, 2 * eps * np.eye(w.d)).logpdf(z)
    assert la == pytest.approx(lp2[0] - lp[0] + bwd - fwd, abs=1e-9)
    thm, _, lam = o.mh_map(th, lp[0], xi, eps)
    np.testing.assert_allclose(thm, th + eps * (w.L @ xi), rtol=1e-12, atol=1e-12)


def test_mala_detailed_balance_pairs(oracle_mod):
    w, o = _target_1d(oracle_mod, L=0.8)
    Lv, eps = 0.8, 0.25
    xs = w.mu[0] + np.linspace(-1.5, 1.5, 13)
    lp, g = o.logp_grad(xs[:, None])
    worst = 0.0
    for i in range(len(xs)):
        for j in range(len(xs)):
            if i == j:
                continue
            # whitened coordinate z = x/L; choose ξ so the proposal from i lands on x_j
            gz = Lv * g[i, 0]
            xi = ((xs[j] - xs[i]) / Lv - eps * gz) / math.sqrt(2 * eps)
            thp, lpp, gp, la = o.mala_map(xs[i:i + 1], lp[i], g[i], np.array([xi]), eps)
            assert thp[0] == pytest.approx(xs[j], abs=1e-12)
            qf = math.exp(-xi * xi / 2)                     # ∝ N(z_j; z_i + ε g_z, 2ε)
            flow_ij = math.exp(lp[i]) * qf * _acc_prob(la)
            gzj = Lv * g[j, 0]
            xj = ((xs[i] - xs[j]) / Lv - eps * gzj) / math.sqrt(2 * eps)
            _, _, _, la_b = o.mala_map(xs[j:j + 1], lp[j], g[j], np.array([xj]), eps)
            flow_ji = math.exp(lp[j]) * math.exp(-xj * xj / 2) * _acc_prob(la_b)
            worst = max(worst, abs(flow_ij - flow_ji) / max(flow_ij, flow_ji))
    assert worst < 1e-12


def test_hmc_linear_map_standard_normal(oracle_mod):
    """Standard normal: one KDK step is [[1−ε²/2, ε],[−ε(1−ε²/4), 1−ε²/2]] per coordinate."""
    d = 3
    w = WL.gaussian(d, 1, seed=2)
    w.mu, w.Sigma, w.Sigma_inv, w.L = np.zeros(d), np.eye(d), np.eye(d), np.eye(d)
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    rng = np.random.default_rng(5)
    for eps, nl in ((0.1, 1), (0.3, 8), (0.05, 16)):
        M = np.array([[1 - eps ** 2 / 2, eps], [-eps * (1 - eps ** 2 / 4), 1 - eps ** 2 / 2]])
        assert np.linalg.det(M) == pytest.approx(1.0, abs=1e-14)
        Mn = np.linalg.matrix_power(M, nl)
        x, q = rng.standard_normal(d), rng.standard_normal(d)
        lp, g = o.logp_grad(x[None, :])
        xp, lpp, gp, qp, la = o.hmc_map(x, lp[0], g[0], q, eps, nl)
        ref = Mn @ np.stack([x, q])
        np.testing.assert_allclose(xp, ref[0], atol=1e-13)
        np.testing.assert_allclose(qp, ref[1], atol=1e-13)
        H0 = 0.5 * x @ x + 0.5 * q @ q
        H1 = 0.5 * xp @ xp + 0.5 * qp @ qp
        assert la == pytest.approx(H0 - H1, abs=1e-12)


def test_hmc_reversible_volume_preserving_and_energy_scaling(oracle_mod):
    w = WL.tiny(n_chains=1, seed=31, d=2, hidden=(8, 8), mlp_scale=1.0)
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    rng = np.random.default_rng(1)
    x, q = w.theta0[0].astype(np.float64), rng.standard_normal(2)
    eps, nl = 0.2, 8

    def phi(v):
        lp, g = o.logp_grad(v[None, :2])
        xp, lpp, gp, qp, la = o.hmc_map(v[:2], lp[0], g[0], v[2:], eps, nl)
        return np.concatenate([xp, qp]), la

    v0 = np.concatenate([x, q])
    v1, la = phi(v0)
    back, la_b = phi(np.concatenate([v1[:2], -v1[2:]]))       # Φ∘flip∘Φ = flip
    np.testing.assert_allclose(back[:2], x, atol=1e-12)
    np.testing.assert_allclose(-back[2:], q, atol=1e-12)
    assert la_b == pytest.approx(-la, abs=1e-11)
    J = np.zeros((4, 4))
    for k in range(4):
        hh = 1e-5
        e = np.zeros(4)
        e[k] = hh
        J[:, k] = (phi(v0 + e)[0] - phi(v0 - e)[0]) / (2 * hh)
    assert abs(abs(np.linalg.det(J)) - 1.0) < 1e-7
    # ΔH = O(ε²) at fixed trajectory length
    dH = []
    for e_, n_ in ((0.2, 4), (0.1, 8), (0.05, 16)):
        lp, g = o.logp_grad(x[None, :])
        dH.append(abs(o.hmc_map(x, lp[0], g[0], q, e_, n_)[4]))
    assert dH[0] / dH[1] == pytest.approx(4.0, rel=0.25)
    assert dH[1] / dH[2] == pytest.approx(4.0, rel=0.25)


def test_hmc_detailed_balance_phase_space(oracle_mod):
    """π(x)N(q)α((x,q)→(x',q')) = π(x')N(q')α((x',−q')→(x,−q)) on a 1-D phase-space grid."""
    w, o = _target_1d(oracle_mod, L=0.9)
    eps, nl = 0.25, 5
    worst = 0.0
    for x0 in w.mu[0] + np.linspace(-1.2, 1.2, 7):
        for q0 in np.linspace(-2.0, 2.0, 9):
            lp, g = o.logp_grad(np.array([[x0]]))
            xp, lpp, gp, qp, la = o.hmc_map(np.array([x0]), lp[0], g[0], np.array([q0]), eps, nl)
            f_fwd = math.exp(lp[0] - 0.5 * q0 * q0) * _acc_prob(la)
            xb, lpb, gb, qb, la_b = o.hmc_map(xp, lpp, gp, -qp, eps, nl)
            assert xb[0] == pytest.approx(x0, abs=1e-12) and -qb[0] == pytest.approx(q0, abs=1e-12)
            f_bwd = math.exp(lpp - 0.5 * qp[0] ** 2) * _acc_prob(la_b)
            worst = max(worst, abs(f_fwd - f_bwd) / max(f_fwd, f_bwd))
    assert worst < 1e-11
