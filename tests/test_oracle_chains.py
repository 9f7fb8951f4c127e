"""Long-run / ensemble pins for the oracle: Gaussian closed-form moments, AIES affine invariance and
the z^(d-1) factor, covariance vs numpy/LAPACK, split invariance, adaptation windows."""
import math

import numpy as np
import pytest

from paper_2606_04895_b200 import workloads as WL


def _moment_check(trace, mu, Sigma, nsig=4.0):
    """trace [T,B,d]; SE from the across-chain variance of per-chain time averages."""
    T, B, d = trace.shape
    m_c = trace.mean(axis=0)                               # [B,d]
    se = m_c.std(axis=0, ddof=1) / math.sqrt(B)
    assert np.all(np.abs(m_c.mean(axis=0) - mu) < nsig * se + 1e-12)
    xc = trace - mu[None, None, :]
    for i in range(d):
        for j in range(i, d):
            p_c = (xc[:, :, i] * xc[:, :, j]).mean(axis=0)
            se_ij = p_c.std(ddof=1) / math.sqrt(B)
            assert abs(p_c.mean() - Sigma[i, j]) < nsig * se_ij + 1e-12, (i, j)


@pytest.mark.parametrize("method", ["mh", "mala", "hmc"])
def test_gaussian_closed_form_moments(oracle_mod, method):
    """s=0, box ±10σ ⇒ posterior N(μ,Σ) (north_star); mean/cov within 4 MC standard errors."""
    w = WL.gaussian(6, 256, seed=41, cond=100.0)
    o = oracle_mod.Oracle(w)
    st = o.new_state(w.theta0)
    if method == "mh":
        st.step_mh(300, 5, 0.9)
        tr = st.step_mh(1500, 5, 0.9, thin=1)
        acc_band = (0.15, 0.5)
    elif method == "mala":
        st.step_mala(100, 5, 0.5)
        tr = st.step_mala(800, 5, 0.5, thin=1)
        acc_band = (0.6, 0.95)
    else:
        st.step_hmc(30, 5, 0.4, 4)
        tr = st.step_hmc(300, 5, 0.4, 4, thin=1)
        acc_band = (0.8, 1.0)
    _moment_check(tr, w.mu, w.Sigma)
    rate = st.n_accept.mean() / st.step
    assert acc_band[0] < rate < acc_band[1]


def test_mh_acceptance_asymptotic(oracle_mod):
    """Exactly whitened Gaussian, d=27: acceptance → 2Φ(−ε√d/2) = 0.435 at ε=0.3 (sanity)."""
    from scipy import stats
    w = WL.gaussian(27, 512, seed=43, cond=1e4)
    o = oracle_mod.Oracle(w)
    st = o.new_state(w.theta0)
    st.step_mh(200, 9, 0.3)
    rate = st.n_accept.mean() / 200
    assert rate == pytest.approx(2 * stats.norm.cdf(-0.3 * math.sqrt(27) / 2), abs=0.02)


def test_split_invariance_and_trace(oracle_mod):
    w = WL.tiny(n_chains=16)
    o = oracle_mod.Oracle(w)
    a, b = o.new_state(w.theta0), o.new_state(w.theta0)
    tr = a.step_mala(60, 3, 0.3, thin=20)
    for _ in range(6):
        b.step_mala(10, 3, 0.3)
    assert np.array_equal(a.theta, b.theta) and np.array_equal(a.logp, b.logp)
    assert np.array_equal(a.n_accept, b.n_accept) and a.step == b.step == 60
    assert np.array_equal(tr[-1], a.theta) and tr.shape == (3, 16, w.d)
    a2, b2 = o.new_state(w.theta0), o.new_state(w.theta0)
    a2.step_hmc(12, 3, 0.2, 5)
    b2.step_hmc(5, 3, 0.2, 5)
    b2.step_hmc(7, 3, 0.2, 5)
    assert np.array_equal(a2.theta, b2.theta)
    a3, b3 = o.new_state(w.theta0), o.new_state(w.theta0)
    a3.step_aies(20, 3)
    b3.step_aies(8, 3)
    b3.step_aies(12, 3)
    assert np.array_equal(a3.theta, b3.theta)
    # cached logp / grad stay consistent with θ
    lp, g = o.logp_grad(a.theta)
    np.testing.assert_allclose(a.logp, lp, rtol=0, atol=0)
    np.testing.assert_allclose(a.grad, g, rtol=0, atol=0)


def test_aies_affine_invariance(oracle_mod):
    """Same seed on π(Ax+b) from A⁻¹(x₀−b): affinely mapped walkers, identical accept bits."""
    w = WL.gaussian(4, 64, seed=51)
    w.lo = w.hi = None
    o1 = oracle_mod.Oracle(w)
    rng = np.random.default_rng(6)
    A = rng.standard_normal((4, 4)) + 2 * np.eye(4)
    bvec = rng.standard_normal(4)
    # y = A⁻¹(x − b): y ~ N(A⁻¹(μ − b), A⁻¹ Σ A⁻ᵀ)
    Ainv = np.linalg.inv(A)
    w2 = WL.gaussian(4, 64, seed=51)
    w2.lo = w2.hi = None
    w2.mu = Ainv @ (w.mu - bvec)
    w2.Sigma = Ainv @ w.Sigma @ Ainv.T
    w2.Sigma_inv = A.T @ w.Sigma_inv @ A
    o2 = oracle_mod.Oracle(w2)
    x0 = w.theta0.astype(np.float64)
    y0 = (x0 - bvec) @ Ainv.T
    s1, s2 = o1.new_state(x0), o2.new_state(y0)
    s1.step_aies(25, 17)
    s2.step_aies(25, 17)
    assert np.array_equal(s1.n_accept, s2.n_accept)
    np.testing.assert_allclose(s2.theta @ A.T + bvec, s1.theta, rtol=1e-9, atol=1e-9)


def test_aies_factor_pins_variance_d2(oracle_mod):
    """d=2 Gaussian with variances (1, 1e4): covariance within 4 SE (omitting z^(d−1) gives ≈0.69)."""
    w = WL.gaussian(2, 512, seed=61)
    w.mu = np.array([0.3, -20.0])
    w.Sigma = np.diag([1.0, 1e4])
    w.Sigma_inv = np.diag([1.0, 1e-4])
    w.lo = w.hi = None
    rng = np.random.default_rng(0)
    x0 = w.mu + rng.standard_normal((512, 2)) * np.array([1.0, 100.0])
    o = oracle_mod.Oracle(w)
    st = o.new_state(x0)
    st.step_aies(300, 23)
    tr = st.step_aies(3000, 23, thin=1)
    # batch means over time (walkers are coupled): 30 batches of 100 steps
    xc = (tr - w.mu) / np.array([1.0, 100.0])
    v = (xc ** 2).mean(axis=1).reshape(30, 100, 2).mean(axis=1)       # [30,2]
    se = v.std(axis=0, ddof=1) / math.sqrt(30)
    assert np.all(np.abs(v.mean(axis=0) - 1.0) < 4 * se + 0.01)
    assert np.all(np.abs(v.mean(axis=0) - 1.0) < 0.05)                # far from the 0.69 failure mode
    # map-level: log α = (d−1) ln z + Δ log π, and d=1 removes the factor
    thp, lpp, la = o.aies_map(x0[0], st.o.logp_grad(x0[:1])[0][0], x0[1], 1.7)
    np.testing.assert_allclose(thp, x0[1] + 1.7 * (x0[0] - x0[1]), rtol=1e-15)
    assert la == pytest.approx(math.log(1.7) + lpp - o.logp_grad(x0[:1])[0][0], abs=1e-12)
    w1 = WL.gaussian(1, 4, seed=62)
    w1.lo = w1.hi = None
    o1 = oracle_mod.Oracle(w1)
    xi, xj = np.array([0.2]), np.array([-0.4])
    lpi = o1.logp_grad(xi[None])[0][0]
    _, lpp1, la1 = o1.aies_map(xi, lpi, xj, 1.9)
    assert la1 == pytest.approx(lpp1 - lpi, abs=1e-14)


def test_aies_half_split_partner_R11(oracle_mod):
    """Partner of walker i in half h is other-half offset + hi32(raw·B/2); S1 sees updated S0."""
    w = WL.gaussian(3, 32, seed=71)
    o = oracle_mod.Oracle(w)
    st = o.new_state(w.theta0)
    x0, lp0 = st.theta.copy(), st.logp.copy()
    seed, B, half = 99, 32, 16
    st.step_aies(1, seed)
    cur, lp = x0.copy(), lp0.copy()
    for hh in range(2):
        own0, oth0 = (0, half) if hh == 0 else (half, 0)
        new = cur.copy()
        for r in range(half):
            i = own0 + r
            u, uz, raw = oracle_mod.control(seed, i, 0)
            j = oth0 + ((raw * half) >> 32)
            z = oracle_mod.stretch_z(uz, 2.0)
            thp, lpp, la = o.aies_map(cur[i], lp[i], cur[j], z)
            if oracle_mod.accept(u, la):
                new[i] = thp
                lp[i] = lpp
        cur = new
    assert np.array_equal(cur, st.theta)
    with pytest.raises(ValueError):
        o.new_state(w.theta0[:31]).step_aies(1, 1)


def test_covariance_and_cholesky_vs_numpy(oracle_mod):
    w = WL.lcdm(n_chains=2, hidden=8, n_hidden=1)
    o = oracle_mod.Oracle(w)
    rng = np.random.default_rng(12)
    X = w.mu + rng.standard_normal((4000, w.d)) @ np.linalg.cholesky(w.Sigma).T
    rc, Cm, L = o.cov_chol(X, jitter=1e-6)
    assert rc == 0
    Cnp = np.cov(X.T)
    np.testing.assert_allclose(Cm, Cnp, rtol=1e-10, atol=1e-12)
    Cj = Cnp + 1e-6 * np.diag(np.diag(Cnp))
    np.testing.assert_allclose(L, np.linalg.cholesky(Cj), rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(L @ L.T, Cj, rtol=1e-10, atol=1e-12)
    # rank-deficient sample set: jitter-retry still has to fail ⇒ L kept (zeros here), rc = -1
    Xdef = np.repeat(X[:1], 10, axis=0)
    rc2, _, _ = o.cov_chol(Xdef, jitter=1e-6)
    assert rc2 == -1


def test_adaptation_windows(oracle_mod):
    """After each window of `adapt_every` steps L = chol(cov(all post-accept states)·(1+jitter on diag))."""
    w = WL.gaussian(5, 64, seed=81)
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))        # start from a diagonal whitening
    o = oracle_mod.Oracle(w)
    o.set_adaptation(50, 1e-6)
    st = o.new_state(w.theta0)
    tr = st.step_mh(50, 4, 0.5, thin=1)
    X = tr.reshape(-1, w.d)
    C = np.cov(X.T)
    C = C + 1e-6 * np.diag(np.diag(C))
    np.testing.assert_allclose(o.get_whitening(), np.linalg.cholesky(C), rtol=1e-9, atol=1e-12)
    assert o.adapt_stats() == (1, 0)
    tr2 = st.step_mh(70, 4, 0.5, thin=1)            # window 2 ends after 50 of these 70 steps
    C2 = np.cov(tr2[:50].reshape(-1, w.d).T)
    C2 = C2 + 1e-6 * np.diag(np.diag(C2))
    np.testing.assert_allclose(o.get_whitening(), np.linalg.cholesky(C2), rtol=1e-9, atol=1e-12)
    assert o.adapt_stats() == (2, 0)
    # LLᵀ → Σ within Monte-Carlo error on the closed form
    Lw = o.get_whitening()
    rel = np.abs(Lw @ Lw.T - w.Sigma) / np.sqrt(np.outer(np.diag(w.Sigma), np.diag(w.Sigma)))
    assert rel.max() < 0.35


def test_chain_offset_streams(oracle_mod):
    """with chain offset c0 the oracle's local chain c draws the Philox stream of global chain
    c0 + c.  Pins: (i) the MH proposal of an accepted chain is θ + ε L ξ with ξ = the KAT-pinned normals of
    chain c0 + c (so the offset lands in counter word 0, nowhere else); (ii) the accept uniform is the control
    word of chain c0 + c; (iii) a shard with offset c0 reproduces chains [c0, c0 + n) of one big ensemble for
    the independent-chain samplers; (iv) offset 0 is the unsharded stream."""
    O = oracle_mod
    w = WL.gaussian(5, 96, seed=7, cond=30.0)
    c0, n, seed, eps = 40, 32, 11, 0.4
    big = O.Oracle(w).new_state(w.theta0)
    sh_o = O.Oracle(w)
    sh_o.set_chain_offset(c0)
    sh = sh_o.new_state(w.theta0[c0:c0 + n])
    th0 = sh.theta.copy()
    sh.step_mh(1, seed, eps)
    acc = sh.n_accept == 1
    assert acc.any() and (~acc).any()
    for c in np.flatnonzero(acc):
        xi = O.normals(seed, c0 + int(c), 0, w.d)
        assert np.allclose(sh.theta[c], th0[c] + eps * (w.L @ xi), rtol=0, atol=1e-13)
        assert math.log(O.control(seed, c0 + int(c), 0)[0]) < sh.last_log_alpha[c]
    for c in np.flatnonzero(~acc):
        assert not math.log(O.control(seed, c0 + int(c), 0)[0]) < sh.last_log_alpha[c]
    big.step_mh(1, seed, eps)
    for st in (big, sh):
        st.step_mala(3, seed, 0.3)
        st.step_hmc(2, seed, 0.2, 3)
    assert np.array_equal(big.theta[c0:c0 + n], sh.theta) and np.array_equal(big.n_accept[c0:c0 + n], sh.n_accept)
    z_o = O.Oracle(w)
    z_o.set_chain_offset(0)
    z = z_o.new_state(w.theta0[:n])
    z.step_mh(1, seed, eps); z.step_mala(3, seed, 0.3); z.step_hmc(2, seed, 0.2, 3)
    assert np.array_equal(big.theta[:n], z.theta)
    assert not np.array_equal(z.theta, sh.theta)
