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


# ---- burn-in loop (reading R22) -------------------------------------------------------
class _FakeState:
    """Feeds the dual-averaging recursion a prescribed acceptance fraction per block."""

    def __init__(self, oracle_mod, alphas, B=1000):
        self._alphas, self.B, self.k = list(alphas), B, 0
        self.n_accept = np.zeros(B, dtype=np.uint64)
        self.logp, self.theta = np.zeros(B), np.zeros((B, 1))
        self.eps_seen = []
        self.o = type("O", (), {"set_adaptation": lambda self, *a: None})()
        self._burn = oracle_mod.OracleState.burn_in.__get__(self)

    def _step(self, method, n, seed, eps, nl):
        self.eps_seen.append(eps)
        k = int(round(self._alphas[self.k] * self.B * n))
        self.n_accept[0] += np.uint64(k)
        self.k += 1


def test_dual_averaging_closed_form(oracle_mod):
    """Constant acceptance α: H̄_m = (δ−α)·m/(m+t₀) ⇒ log ε_m = μ − √m/γ·(δ−α)·m/(m+t₀), μ = log 10ε₀;
    α ≡ δ ⇒ every ε_m = 10 ε₀ (Hoffman & Gelman 2014, Alg. 5)."""
    eps0, delta, nblk = 0.25, 0.574, 12
    for alpha in (0.574, 0.2, 0.9):
        fs = _FakeState(oracle_mod, [alpha] * nblk)
        eps, _, _, hist = fs._burn("mala", 1, 10 * nblk, 10 * nblk, 10, 1, eps0, delta)
        assert len(hist) == nblk and hist[0] == float(np.float32(eps0))
        m = np.arange(1, nblk)
        ref = np.log(10 * eps0) - np.sqrt(m) / 0.05 * (delta - alpha) * m / (m + 10.0)
        np.testing.assert_allclose(np.log(hist[1:]), ref, rtol=0, atol=2e-6)     # float32 ε at the interface
        # the returned ε is the weighted average log ε̄ = Σ-recursion with weights m^-0.75
        m_all = np.arange(1, nblk + 1)
        le = np.log(10 * eps0) - np.sqrt(m_all) / 0.05 * (delta - alpha) * m_all / (m_all + 10.0)
        bar = 0.0
        for mm, l in zip(m_all, le):
            bar = mm ** -0.75 * l + (1 - mm ** -0.75) * bar
        assert math.log(eps) == pytest.approx(bar, abs=2e-6)


def test_burn_in_finds_optimal_mh_scale_and_covariance(oracle_mod):
    """Anisotropic Gaussian, diagonal initial whitening: after 3 iterations L Lᵀ ≈ Σ, the MH step adapted
    toward acceptance 0.234 is the textbook optimal 2.38/√d (Roberts, Gelman & Gilks 1997; asymptotic in d: ±15 % at d = 30),
    the acceptance of a fresh run sits at the target, and the best-fit point is near μ."""
    d = 30
    w = WL.gaussian(d, 512, seed=44, cond=50.0)
    w.lo = w.hi = None
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
    o = oracle_mod.Oracle(w)
    st = o.new_state(w.theta0)
    eps, th_best, lp_best, hist = st.burn_in("mh", 3, 390, 240, 4, 5, 0.05, 0.234)   # 60 blocks per iteration: ε̄ forgets the 10 ε₀ start
    C = o.get_whitening() @ o.get_whitening().T
    dscale = np.sqrt(np.outer(np.diag(w.Sigma), np.diag(w.Sigma)))
    assert np.abs(C - w.Sigma).max() / dscale.max() < 0.08          # 512 chains x 150 steps per window
    assert 0.85 * 2.38 / math.sqrt(d) < eps < 1.15 * 2.38 / math.sqrt(d), eps
    a0 = st.n_accept.sum()
    st.step_mh(100, 5, eps)
    rate = (st.n_accept.sum() - a0) / (512 * 100)
    assert abs(rate - 0.234) < 0.05, rate
    z = np.linalg.solve(np.linalg.cholesky(w.Sigma), th_best - w.mu)
    assert lp_best == pytest.approx(-0.5 * z @ z, abs=1e-9) and z @ z < 0.5 * d   # the best of 512 chains lies well inside the typical set (E z.z = d)
    assert o.adapt_stats() == (3, 0)


# ---- differential-evolution move, eq (2.16) (reading R23) -------------------------------
def test_de_map_is_eq_2_16(oracle_mod):
    w = WL.tiny(n_chains=8, seed=3, d=3, hidden=(8, 8), mlp_scale=0.7)
    o = oracle_mod.Oracle(w)
    xi, xj, xk = (w.theta0[n].astype(np.float64) for n in range(3))
    lp = o.logp_grad(np.stack([xi]), want_grad=False)[0][0]
    g = 0.61
    thp, lpp, la = o.de_map(xi, lp, xj, xk, g)
    np.testing.assert_allclose(thp, xi + g * (xj - xk), rtol=0, atol=1e-15)
    assert lpp == pytest.approx(o.logp_grad(thp[None, :], want_grad=False)[0][0], abs=1e-13)
    assert la == pytest.approx(lpp - lp, abs=1e-13)                       # symmetric proposal: no extra factor
    # swapping j and k proposes the mirror image
    thm, _, _ = o.de_map(xi, lp, xk, xj, g)
    np.testing.assert_allclose(thm - xi, -(thp - xi), rtol=0, atol=1e-15)


def test_de_partners_distinct_uniform_from_other_half(oracle_mod):
    """σ_γ = 0 ⇒ x' − x_i = 2.38/√(2d)·(x_j − x_k) exactly: recover (j, k) of every walker by brute force over
    all ordered pairs of the ensemble; they must be two different walkers of the complementary half, uniform."""
    d, B = 2, 24
    w = WL.gaussian(d, B, seed=6)
    w.lo = w.hi = None
    w.mu = w.Sigma_inv = None                      # flat target: every proposal is accepted
    o = oracle_mod.Oracle(w)
    g0 = 2.38 / math.sqrt(2 * d)
    half = B // 2
    counts = np.zeros((half, half), dtype=np.int64)
    n_steps = 400
    for step in range(n_steps):
        st = o.new_state(w.theta0)
        st.step = step
        before = st.theta.copy()
        st.step_aies_de(1, 99, sigma_gamma=0.0)
        # half 0 moved against the untouched half 1
        D = before[:, None, :] - before[None, :, :]                       # all ordered pairs x_j − x_k
        for i in range(half):
            disp = (st.theta[i] - before[i]) / g0
            hit = np.abs(D - disp).max(axis=-1) < 1e-12
            np.fill_diagonal(hit, False)
            hits = np.argwhere(hit)
            assert len(hits) == 1, (step, i, hits)
            j, k = hits[0]
            assert j >= half and k >= half
            counts[j - half, k - half] += 1
    assert np.all(np.diag(counts) == 0)
    off = counts[~np.eye(half, dtype=bool)]
    expect = n_steps * half / (half * (half - 1))
    chi2 = float(((off - expect) ** 2 / expect).sum())
    dof = half * (half - 1) - 1
    assert abs(chi2 - dof) < 5.0 * math.sqrt(2.0 * dof), (chi2, dof)


def test_de_gamma_distribution(oracle_mod):
    """γ = (1 + η)·2.38/√(2d), η ~ N(0, σ_γ): ratio of the displacement to (x_j − x_k) has that mean and sd."""
    d, B = 3, 8
    w = WL.gaussian(d, B, seed=7)
    w.lo = w.hi = None
    w.mu = w.Sigma_inv = None
    o = oracle_mod.Oracle(w)
    g0, sg = 2.38 / math.sqrt(2 * d), 0.3
    gam = []
    for step in range(1500):
        a, b = o.new_state(w.theta0), o.new_state(w.theta0)
        a.step = b.step = step
        a.step_aies_de(1, 5, sigma_gamma=0.0)
        b.step_aies_de(1, 5, sigma_gamma=sg)
        da, db = a.theta[:B // 2] - w.theta0[:B // 2], b.theta[:B // 2] - w.theta0[:B // 2]
        gam.append(g0 * (db * da).sum(axis=1) / (da * da).sum(axis=1))      # same (j, k), different γ
    gam = np.concatenate(gam)
    n = gam.size
    assert abs(gam.mean() - g0) < 4.0 * g0 * sg / math.sqrt(n)
    assert abs(gam.std() - g0 * sg) < 4.0 * g0 * sg / math.sqrt(2 * n)


def test_de_moments_anisotropic_gaussian(oracle_mod):
    """Stationarity: closed-form Gaussian moments within 4 MC standard errors (a spurious Jacobian factor in
    log α, or j = k allowed, biases the variance)."""
    d, B = 4, 512
    w = WL.gaussian(d, B, seed=15, cond=100.0)
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    st = o.new_state(w.theta0)
    st.step_aies_de(200, 8, sigma_gamma=0.1)
    tr = st.step_aies_de(600, 8, sigma_gamma=0.1, thin=6)          # [100, B, d]
    acc = st.n_accept.mean() / 800
    assert 0.1 < acc < 0.7, acc
    # walkers of one ensemble are not independent: blocks of time as the replicates
    blocks = tr.reshape(10, 10 * B, d)
    m = blocks.mean(axis=1)
    se = m.std(axis=0, ddof=1) / math.sqrt(10)
    assert np.all(np.abs(m.mean(axis=0) - w.mu) < 4.0 * se + 1e-12)
    v = ((blocks - w.mu) ** 2).mean(axis=1)
    se_v = v.std(axis=0, ddof=1) / math.sqrt(10)
    assert np.all(np.abs(v.mean(axis=0) - np.diag(w.Sigma)) < 4.0 * se_v)


# ---- R − 1 of eq (4.1)-(4.2) --------------------------------------------------------
def _exact_chains(rng, n, nb, d, W0, c):
    """Chains whose within-chain covariance is EXACTLY W0 each and whose means have covariance EXACTLY c·W0."""
    def exact(m, C):
        z = rng.standard_normal((m, d))
        z -= z.mean(axis=0)
        z = z @ np.linalg.inv(np.linalg.cholesky(np.cov(z, rowvar=False, ddof=1)).T)     # sample cov = I
        return z @ np.linalg.cholesky(C).T
    means = exact(nb, c * W0)
    return np.stack([exact(n, W0) + means[k] for k in range(nb)], axis=1)                # [n][B][d]


def test_rminus1_closed_forms(oracle_mod):
    rng = np.random.default_rng(12)
    d, n, nb = 4, 40, 12
    A = rng.standard_normal((d, d))
    W0 = A @ A.T + 0.5 * np.eye(d)
    for c in (0.01, 0.3, 2.0):
        tr = _exact_chains(rng, n, nb, d, W0, c)
        assert oracle_mod.rminus1(tr) == pytest.approx(c, rel=1e-9)                      # B = c W ⇒ every λ = c
        # affine reparametrisation leaves eig(W⁻¹B) unchanged (the D scaling is a similarity)
        T = rng.standard_normal((d, d)) + 2.0 * np.eye(d)
        assert oracle_mod.rminus1(tr @ T.T + rng.standard_normal(d)) == pytest.approx(c, rel=1e-8)
    # d = 1: var(chain means) / mean(chain variances)
    x = rng.standard_normal((50, 7, 1)) * np.linspace(0.5, 2.0, 7)[None, :, None] + rng.standard_normal((1, 7, 1))
    ref = x.mean(axis=0)[:, 0].var(ddof=1) / x[:, :, 0].var(axis=0, ddof=1).mean()
    assert oracle_mod.rminus1(x) == pytest.approx(ref, rel=1e-12)
    # B and W diagonal in the same basis with different ratios: the largest ratio
    ratios = np.array([0.05, 0.7, 0.2])
    nb2 = 9
    m = rng.standard_normal((nb2, 3)); m -= m.mean(axis=0)
    m = m @ np.linalg.inv(np.linalg.cholesky(np.cov(m, rowvar=False, ddof=1)).T) * np.sqrt(ratios)
    z = rng.standard_normal((30, 3)); z -= z.mean(axis=0)
    z = z @ np.linalg.inv(np.linalg.cholesky(np.cov(z, rowvar=False, ddof=1)).T)
    tr = np.stack([z + m[k] for k in range(nb2)], axis=1)
    assert oracle_mod.rminus1(tr) == pytest.approx(ratios.max(), rel=1e-9)


def test_rminus1_mixed_chains_small_unmixed_large(oracle_mod):
    rng = np.random.default_rng(3)
    iid = rng.standard_normal((2000, 16, 5))
    assert oracle_mod.rminus1(iid) < 0.02                         # ~ (d + few)/n for independent draws
    stuck = iid * 0.1 + 3.0 * rng.standard_normal((1, 16, 5))    # chains far apart relative to their spread
    assert oracle_mod.rminus1(stuck) > 100.0
