"""GPU parity tests of the exact path (BEST_PREC_FP32) against the oracle, through the C-ABI.
T1 logp/grad, T2 single-step maps, T3 HMC trajectories, T4 split invariance, T5 moments,
T6 adaptation, T7 non-finite handling."""
import math

import numpy as np
import pytest

from paper_2606_04895_b200 import workloads as WL
from parity_util import TOL, accept_margins, check_logp_grad

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_04895_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    oracle.lib()
    return oracle


def _targets(name):
    if name == "tiny":
        return WL.tiny(), 4096
    if name == "tiny_silu":
        return WL.tiny(activation=WL.ACT_SILU, hidden=(50, 37)), 1111   # ragged widths and count
    if name == "lcdm":
        return WL.lcdm(n_chains=8), 4096
    if name == "lcdm_s3":
        return WL.lcdm(n_chains=8, mlp_scale=3.0), 1024
    if name == "sterile":
        return WL.sterile(n_chains=8), 1024
    raise KeyError(name)


@pytest.mark.parametrize("name", ["tiny", "tiny_silu", "lcdm", "lcdm_s3", "sterile"])
@pytest.mark.parametrize("variant", ["full", "mlp_only", "gauss_only"])
def test_T1_logp_grad(B, O, name, variant):
    w, n = _targets(name)
    pts = WL.probe_points(w, n, seed=17)
    if variant == "mlp_only":
        w = WL.mlp_only(w)
    elif variant == "gauss_only":
        w = WL.gaussian_only(w)
    ctx = B.Context(w, B.PREC_FP32)
    lp = np.zeros(n, np.float32)
    g = np.zeros((n, w.d), np.float32)
    ctx.logp_grad(pts, n, lp, g)
    lp_ref, g_ref = O.Oracle(w).logp_grad(pts)
    check_logp_grad(lp, g, lp_ref, g_ref, TOL[0], f"{name}/{variant}")
    # forward-only call and device-pointer call agree with the host-pointer call
    import torch
    lp2 = np.zeros(n, np.float32)
    ctx.logp_grad(pts, n, lp2, None)
    assert np.array_equal(lp, lp2)
    t_pts = torch.from_numpy(pts).cuda()
    t_lp = torch.empty(n, device="cuda")
    t_g = torch.empty(n, w.d, device="cuda")
    ctx.logp_grad(t_pts, n, t_lp, t_g, stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(t_lp.cpu().numpy(), lp) and np.array_equal(t_g.cpu().numpy(), g)
    ctx.close()


def f32(x):
    """The C-ABI takes ε and a as float: hand the oracle the very same value."""
    return float(np.float32(x))


def _single_step(B, O, w, method, seed, setup=None, prec=None, window=1e-6, **kw):
    kw = {k: (f32(v) if isinstance(v, float) else v) for k, v in kw.items()}
    ctx = B.Context(w, B.PREC_FP32 if prec is None else prec)
    orc = O.Oracle(w)
    if setup is not None:
        setup(ctx, orc)
    st = ctx.new_state(w.theta0)
    ost = orc.new_state(w.theta0)
    th0 = ost.theta.copy()
    getattr(st, "step_" + method)(1, seed, **kw)
    getattr(ost, "step_" + method)(1, seed, **kw)
    la = st.last_log_alpha()
    th, lp, gr = st.get_f64(want_grad=(method in ("mala", "hmc")))
    acc = st.get(want_grad=False)["n_accept"].astype(np.int64)
    acc_ref = ost.n_accept.astype(np.int64)
    m = accept_margins(O, seed, 0, w.n_chains, ost.last_log_alpha)
    mism = acc != acc_ref
    with np.errstate(invalid="ignore"):      # hard box: (-inf) - (-inf), masked by the where
        dla = np.abs(np.where(la == ost.last_log_alpha, 0.0, la - ost.last_log_alpha))
    info = dict(n=w.n_chains, mismatches=int(mism.sum()),
                max_margin_of_mismatch=float(m[mism].max()) if mism.any() else 0.0,
                max_dla=float(np.nanmax(dla)),
                accept_rate=float(acc_ref.mean()))
    print(f"[T2] {w.name}/{method}: {info}")
    # accept bits identical outside the logged margin set |log u − log α| < 1e-6 (north_star; 1e-5 for FP32_TC)
    assert not (mism & (m >= window)).any(), info
    same = ~mism
    # post-state: accepted chains carry the proposal (rel 1e-6 of the step scale), others unchanged
    scale = np.abs(ost.theta).max(axis=0)
    assert (np.abs(th[same] - ost.theta[same]) <= 1e-6 * scale + 1e-9).all()
    rej = same & (acc_ref == 0)
    assert np.array_equal(th[rej], th0[rej])
    assert np.abs(lp[same] - ost.logp[same]).max() <= TOL[0] * np.abs(ost.logp).max()
    if gr is not None:
        num = np.linalg.norm(gr[same] - ost.grad[same], axis=1)
        assert (num <= TOL[0] * np.linalg.norm(ost.grad[same], axis=1)).all()
    st.close()
    ctx.close()
    return info


@pytest.mark.parametrize("method,kw", [("mh", dict(eps=0.3)), ("mala", dict(eps=0.3)), ("aies", dict(a=2.0))])
def test_T2_single_step_tiny_64k(B, O, method, kw):
    w = WL.tiny().with_chains(65536, seed=5)
    _single_step(B, O, w, method, seed=1234, **kw)


@pytest.mark.parametrize("method,kw", [("mh", dict(eps=0.3)), ("mala", dict(eps=0.3))])
def test_T2_single_step_lcdm(B, O, method, kw):
    w = WL.lcdm(n_chains=2048)
    _single_step(B, O, w, method, seed=77, **kw)


def test_T2_single_step_sterile_aies_and_mala(B, O):
    w = WL.sterile(n_chains=1024)
    _single_step(B, O, w, "aies", seed=9, a=2.0)
    _single_step(B, O, w, "mala", seed=9, eps=0.01)


@pytest.mark.parametrize("nl", [1, 8, 16])
def test_T3_hmc_trajectory(B, O, nl):
    w = WL.tiny().with_chains(4096, seed=6)
    _single_step(B, O, w, "hmc", seed=31, eps=0.2, n_leapfrog=nl)
    if nl == 16:
        w = WL.lcdm(n_chains=512, mlp_scale=3.0)
        _single_step(B, O, w, "hmc", seed=32, eps=0.1, n_leapfrog=16)


def test_T4_split_invariance(B):
    import torch
    w = WL.tiny().with_chains(300, seed=8)
    ctx = B.Context(w, B.PREC_FP32)
    a, b = ctx.new_state(w.theta0), ctx.new_state(w.theta0)
    tr = torch.zeros(3, 300, w.d, device="cuda")
    a.step_mala(60, 3, 0.3, trace=tr, thin=20)
    for _ in range(6):
        b.step_mala(10, 3, 0.3)
    ga, gb = a.get(), b.get()
    for k in ("theta", "logp", "grad", "n_accept"):
        assert np.array_equal(ga[k], gb[k]), k
    assert ga["step"] == gb["step"] == 60 and ga["n_evals"] == gb["n_evals"] == 300 * 61
    torch.cuda.synchronize()
    assert np.array_equal(tr[-1].cpu().numpy(), ga["theta"])
    for meth, kw in (("mh", dict(eps=0.3)), ("hmc", dict(eps=0.2, n_leapfrog=5)), ("aies", dict(a=2.0))):
        a, b = ctx.new_state(w.theta0), ctx.new_state(w.theta0)
        getattr(a, "step_" + meth)(12, 3, **kw)
        getattr(b, "step_" + meth)(5, 3, **kw)
        getattr(b, "step_" + meth)(7, 3, **kw)
        assert np.array_equal(a.get()["theta"], b.get()["theta"]), meth
    ctx.close()


def _moments_vs_exact(trace, mu, Sigma, nsig=4.0):
    T, Bn, d = trace.shape
    m_c = trace.mean(axis=0)
    se = m_c.std(axis=0, ddof=1) / math.sqrt(Bn)
    assert np.all(np.abs(m_c.mean(axis=0) - mu) < nsig * se)
    xc = trace - mu
    for i in range(d):
        for j in range(i, d):
            p = (xc[:, :, i] * xc[:, :, j]).mean(axis=0)
            assert abs(p.mean() - Sigma[i, j]) < nsig * p.std(ddof=1) / math.sqrt(Bn), (i, j)


@pytest.mark.parametrize("method", ["mh", "mala", "hmc", "aies", "aies_de"])
@pytest.mark.parametrize("d", [6, 27])
def test_T5_gaussian_closed_form_moments(B, method, d):
    import torch
    if method.startswith("aies") and d == 27:
        pytest.skip("AIES moment parity is tested at small d (slow mixing at d=27, SURVEY §8(c))")
    w = WL.gaussian(d, 512, seed=40 + d, cond=100.0 if d == 6 else 1e4)
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    plan = {"mh": (dict(eps=2.4 / math.sqrt(d)), 400, 2400, 4), "mala": (dict(eps=0.5 if d == 6 else 0.3), 100, 800, 2),
            "hmc": (dict(eps=0.4 if d == 6 else 0.25, n_leapfrog=4), 30, 300, 1), "aies": (dict(a=2.0), 400, 3000, 5),
            "aies_de": (dict(sigma_gamma=0.1), 400, 3000, 5)}
    kw, burn, n, thin = plan[method]
    getattr(st, "step_" + method)(burn, 11, **kw)
    tr = torch.zeros(n // thin, 512, d, device="cuda")
    getattr(st, "step_" + method)(n, 11, trace=tr, thin=thin, **kw)
    torch.cuda.synchronize()
    trace = tr.cpu().numpy().astype(np.float64)
    if method.startswith("aies"):       # walkers are coupled: batch means over time
        xc = (trace - w.mu) / np.sqrt(np.diag(w.Sigma))
        v = (xc ** 2).mean(axis=1).reshape(30, -1, d).mean(axis=1)
        se = v.std(axis=0, ddof=1) / math.sqrt(30)
        assert np.all(np.abs(v.mean(axis=0) - 1.0) < 4 * se + 0.01)
    else:
        _moments_vs_exact(trace, w.mu, w.Sigma)
    rate = st.get(want_grad=False)["n_accept"].mean() / (burn + n)
    print(f"[T5] {method} d={d}: acceptance {rate:.3f}")
    assert 0.1 < rate <= 1.0
    ctx.close()


def test_T5_tiny_moments_gpu_vs_oracle(B, O):
    """tiny config, MALA: GPU long-run moments vs the oracle's (4 MC standard errors of the difference)."""
    import torch
    w = WL.tiny().with_chains(256, seed=12)
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    ost = O.Oracle(w).new_state(w.theta0)
    st.step_mala(100, 5, 0.3)
    ost.step_mala(100, 6, f32(0.3))     # different seed: independent runs
    tr = torch.zeros(500, 256, w.d, device="cuda")
    st.step_mala(500, 5, 0.3, trace=tr, thin=1)
    otr = ost.step_mala(500, 6, f32(0.3), thin=1)
    torch.cuda.synchronize()
    a, b = tr.cpu().numpy().astype(np.float64).mean(axis=0), otr.mean(axis=0)
    se = np.sqrt(a.var(axis=0, ddof=1) / 256 + b.var(axis=0, ddof=1) / 256)
    assert np.all(np.abs(a.mean(axis=0) - b.mean(axis=0)) < 4 * se)
    ra = st.get(want_grad=False)["n_accept"].mean() / 600
    assert abs(ra - ost.n_accept.mean() / 600) < 0.02
    ctx.close()


def test_T6_adaptation(B, O):
    """L after each window vs the oracle's covariance/Cholesky of the GPU's own trace (rel 1e-6)."""
    import torch
    w = WL.sterile(n_chains=1024, hidden=64, n_hidden=2)
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    st.set_adaptation(100, 1e-6)
    o = O.Oracle(w)
    for win in range(3):
        tr = torch.zeros(100, 1024, w.d, device="cuda")
        st.step_mh(100, 21, 0.3, trace=tr, thin=1)
        torch.cuda.synchronize()
        Lg = ctx.get_whitening()
        # the trace is fp32-rounded θ; the GPU accumulates fp64 θ ⇒ compare at fp32-trace accuracy
        rc, _, Lo = o.cov_chol(tr.cpu().numpy().astype(np.float64).reshape(-1, w.d), 1e-6)
        assert rc == 0
        scale = np.sqrt(np.outer(np.diag(Lo @ Lo.T), np.ones(w.d)))
        assert np.abs(Lg - Lo).max() / scale.max() < 1e-6, win
        assert np.allclose(np.triu(Lg, 1), 0.0)
    assert ctx.adapt_stats() == (3, 0)
    st.set_adaptation(0)
    ctx.close()


def test_T6_adaptation_matches_oracle_driver(B, O):
    """Same seeds, same windows: GPU whitening after 2 windows tracks the oracle's own adaptive run."""
    w = WL.gaussian(5, 256, seed=81)
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    st.set_adaptation(50, 1e-6)
    o = O.Oracle(w)
    o.set_adaptation(50, 1e-6)
    ost = o.new_state(w.theta0)
    st.step_mala(100, 4, 0.4)
    ost.step_mala(100, 4, f32(0.4))
    np.testing.assert_allclose(ctx.get_whitening(), o.get_whitening(), rtol=1e-9, atol=1e-11)
    th, _, _ = st.get_f64(want_grad=False)
    np.testing.assert_allclose(th, ost.theta, rtol=1e-9, atol=1e-9)
    ctx.close()


# ---- per-dimension step factors (R20) and hard box (R21) --------------------------
def _step_factors(d, seed):
    s = np.exp(np.random.default_rng(seed).uniform(np.log(0.3), np.log(3.0), d))
    s[-2:] = 10.0                                   # the paper's "10 times larger for the extension parameters"
    return s


@pytest.mark.parametrize("method,kw", [("mh", dict(eps=0.1)), ("mala", dict(eps=0.02)),
                                       ("hmc", dict(eps=0.03, n_leapfrog=4))])
def test_N1_step_scale_single_step(B, O, method, kw):
    w = WL.lcdm(n_chains=1024, mlp_scale=3.0 if method == "hmc" else 1.0)
    s = _step_factors(w.d, 3)
    info = _single_step(B, O, w, method, seed=91, setup=lambda c, o: (c.set_step_scale(s), o.set_step_scale(s)), **kw)
    assert 0.02 < info["accept_rate"] < 0.999, info     # both branches of the accept rule are exercised


def test_N1_step_scale_api(B, O):
    """Factors persist across set_whitening and adaptation; get_whitening returns the unscaled factor;
    NULL resets; bad factors are refused."""
    w = WL.gaussian(5, 256, seed=81)
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
    s = np.array([0.5, 2.0, 1.0, 3.0, 0.7])
    ctx = B.Context(w, B.PREC_FP32)
    ctx.set_step_scale(s)
    np.testing.assert_array_equal(ctx.get_whitening(), w.L)
    L2 = np.linalg.cholesky(w.Sigma)
    ctx.set_whitening(L2)
    np.testing.assert_array_equal(ctx.get_whitening(), np.tril(L2))
    st = ctx.new_state(w.theta0)
    st.set_adaptation(50, 1e-6)
    o = O.Oracle(w)
    o.set_whitening(L2)
    o.set_step_scale(s)
    o.set_adaptation(50, 1e-6)
    ost = o.new_state(w.theta0)
    st.step_mala(100, 4, 0.2)
    ost.step_mala(100, 4, f32(0.2))
    np.testing.assert_allclose(ctx.get_whitening(), o.get_whitening(), rtol=1e-9, atol=1e-11)
    th, _, _ = st.get_f64(want_grad=False)
    np.testing.assert_allclose(th, ost.theta, rtol=1e-9, atol=1e-9)
    for bad in (np.array([1.0, 0.0, 1, 1, 1]), np.array([1.0, -2.0, 1, 1, 1]), np.array([1.0, np.inf, 1, 1, 1]),
                np.array([1.0, np.nan, 1, 1, 1])):
        with pytest.raises(B.BestError) as e:
            ctx.set_step_scale(bad)
        assert e.value.code == B.BEST_ERR_ARG
    st.set_adaptation(0)
    ctx.set_step_scale(None)
    ost2 = O.Oracle(w)
    ost2.set_whitening(ctx.get_whitening())
    a, b2 = ctx.new_state(w.theta0), ost2.new_state(w.theta0)
    a.step_mh(3, 8, 0.3)
    b2.step_mh(3, 8, f32(0.3))
    np.testing.assert_allclose(a.get_f64(want_grad=False)[0], b2.theta, rtol=1e-9, atol=1e-9)
    ctx.close()


def _narrow_box(w, nsig):
    """box = μ ± nsig·σ per coordinate, starting points clipped into it"""
    sig = np.sqrt(np.diag(w.Sigma))
    w.lo, w.hi = w.mu - nsig * sig, w.mu + nsig * sig
    w.theta0 = np.clip(w.theta0, (w.lo + 1e-3 * sig).astype(np.float32), (w.hi - 1e-3 * sig).astype(np.float32))
    return w


@pytest.mark.parametrize("method,kw", [("mh", dict(eps=0.5)), ("mala", dict(eps=0.3)), ("hmc", dict(eps=0.3, n_leapfrog=4)),
                                       ("aies", dict(a=2.0))])
def test_N1_hard_box_single_step(B, O, method, kw):
    w = _narrow_box(WL.tiny().with_chains(8192, seed=12), 1.2)
    info = _single_step(B, O, w, method, seed=17, setup=lambda c, o: (c.set_hard_box(True), o.set_hard_box(True)), **kw)
    assert info["accept_rate"] < 0.9, info              # a visible share of the proposals leaves the box


def test_N1_hard_box_values_and_invariant(B, O):
    w = _narrow_box(WL.tiny().with_chains(4096, seed=13), 1.0)
    ctx = B.Context(w, B.PREC_FP32)
    o = O.Oracle(w)
    ctx.set_hard_box(True)
    o.set_hard_box(True)
    pts = WL.probe_points(w, 600, seed=3)
    lp = np.zeros(600, np.float32)
    g = np.zeros((600, w.d), np.float32)
    ctx.logp_grad(pts, 600, lp, g)
    lp_ref, g_ref = o.logp_grad(pts)
    outside = np.isneginf(lp_ref)
    assert 50 < outside.sum() < 550
    assert np.array_equal(np.isneginf(lp), outside)
    ins = ~outside
    assert np.abs(lp[ins] - lp_ref[ins]).max() <= TOL[0] * np.abs(lp_ref[ins]).max()
    num = np.linalg.norm(g - g_ref, axis=1)
    assert (num <= TOL[0] * np.linalg.norm(g_ref, axis=1)).all()     # gradient of the remaining terms everywhere
    st = ctx.new_state(w.theta0)
    for step in (lambda: st.step_mh(20, 5, 0.6), lambda: st.step_mala(20, 6, 0.3), lambda: st.step_hmc(5, 7, 0.3, 4),
                 lambda: st.step_aies(10, 8, 2.0)):
        step()
        th = st.get_f64(want_grad=False)[0]
        assert (th >= w.lo).all() and (th <= w.hi).all()
    acc = st.get(want_grad=False)["n_accept"]
    assert acc.min() >= 1
    wf = WL.tiny().with_chains(16, seed=13)
    wf.lo = wf.hi = None
    c2 = B.Context(wf, B.PREC_FP32)
    with pytest.raises(B.BestError) as e:
        c2.set_hard_box(True)
    assert e.value.code == B.BEST_ERR_ARG
    c2.close()
    ctx.close()


# ---- differential-evolution move, eq (2.16) (R23) ----------------------------------
@pytest.mark.parametrize("sg", [0.0, 0.3])
def test_N3_de_single_step(B, O, sg):
    _single_step(B, O, WL.tiny().with_chains(65536, seed=5), "aies_de", seed=1234, sigma_gamma=sg)
    _single_step(B, O, WL.sterile(n_chains=1024), "aies_de", seed=9, sigma_gamma=sg)


def test_N3_de_split_invariance_and_errors(B):
    w = WL.tiny().with_chains(300, seed=2)
    ctx = B.Context(w, B.PREC_FP32)
    a, b2 = ctx.new_state(w.theta0), ctx.new_state(w.theta0)
    a.step_aies_de(6, 11, f32(0.2))
    for _ in range(3):
        b2.step_aies_de(2, 11, f32(0.2))
    ga, gb = a.get(want_grad=False), b2.get(want_grad=False)
    assert np.array_equal(ga["theta"], gb["theta"]) and np.array_equal(ga["n_accept"], gb["n_accept"])
    assert ga["step"] == 6 and ga["n_accept"].sum() > 0
    for bad in (lambda: a.step_aies_de(1, 1, -0.1), lambda: ctx.new_state(w.theta0[:2]).step_aies_de(1, 1, 0.1),
                lambda: ctx.new_state(w.theta0[:7]).step_aies_de(1, 1, 0.1)):
        with pytest.raises(B.BestError) as e:
            bad()
        assert e.value.code == B.BEST_ERR_ARG
    ctx.new_state(w.theta0[:4]).step_aies_de(2, 1, 0.1)          # the smallest ensemble: two walkers per half
    ctx.close()


# ---- R - 1 of eq (4.1)-(4.2) on the device ------------------------------------------
def test_N4_rminus1_matches_oracle(B, O):
    import torch
    # (i) a real trace: tiny config, MALA, 256 chains x 200 samples
    w = WL.tiny().with_chains(256, seed=4)
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    tr = torch.zeros(200, 256, w.d, device="cuda")
    st.step_mala(200, 3, 0.3, trace=tr, thin=1)
    torch.cuda.synchronize()
    r_gpu = B.rminus1(tr)
    r_ref = O.rminus1(tr.cpu().numpy())
    assert r_gpu == pytest.approx(r_ref, rel=1e-9) and 0.0 < r_gpu < 1.0
    assert B.rminus1(tr) == r_gpu                                            # fixed summation order
    ctx.close()
    # (ii) sizes of the paper's runs: d = 29, ragged tails in every kernel (4099 chains x 67 samples), chains
    # displaced by ~ their own spread, correlated dimensions
    rng = np.random.default_rng(8)
    d, nb, n = 29, 4099, 67
    A = rng.standard_normal((d, d)) / math.sqrt(d) + np.eye(d)
    x = (rng.standard_normal((n, nb, d)) + 0.7 * rng.standard_normal((1, nb, d))) @ A.T + 5.0
    x32 = x.astype(np.float32)
    r_gpu = B.rminus1(torch.from_numpy(x32).cuda())
    assert r_gpu == pytest.approx(O.rminus1(x32), rel=1e-8)
    # (iii) tiny shapes and d = 1, 32
    for (n, nb, d) in ((2, 2, 1), (5, 3, 2), (40, 9, 32)):
        x32 = (rng.standard_normal((n, nb, d)) + rng.standard_normal((1, nb, d))).astype(np.float32)
        assert B.rminus1(torch.from_numpy(x32).cuda()) == pytest.approx(O.rminus1(x32), rel=1e-8), (n, nb, d)
    # (iv) stuck ensemble: large value, still accurate
    x32 = (0.01 * rng.standard_normal((50, 64, 6)) + rng.standard_normal((1, 64, 6))).astype(np.float32)
    r = B.rminus1(torch.from_numpy(x32).cuda())
    assert r > 1e3 and r == pytest.approx(O.rminus1(x32), rel=1e-6)


def test_N4_rminus1_errors(B):
    import ctypes as C
    import torch
    x = torch.randn(10, 8, 3, device="cuda")
    for call in (lambda: B.lib().best_rminus1(x.data_ptr(), 1, 8, 3, C.byref(C.c_double()), None),
                 lambda: B.lib().best_rminus1(x.data_ptr(), 10, 1, 3, C.byref(C.c_double()), None),
                 lambda: B.lib().best_rminus1(x.data_ptr(), 10, 8, 33, C.byref(C.c_double()), None),
                 lambda: B.lib().best_rminus1(x.cpu().numpy().ctypes.data, 10, 8, 3, C.byref(C.c_double()), None)):
        assert call() == B.BEST_ERR_ARG
    frozen = x.clone()
    frozen[:, :, 1] = frozen[0:1, :, 1]                 # dimension 1 never moves inside a chain: W_11 = 0
    with pytest.raises(B.BestError) as e:
        B.rminus1(frozen)
    assert e.value.code == B.BEST_ERR_NOT_SPD


# ---- burn-in loop (R22) ------------------------------------------------------------
@pytest.mark.parametrize("method,eps0,delta,nl", [("mh", 0.1, 0.234, 1), ("mala", 0.05, 0.574, 1), ("hmc", 0.05, 0.7, 3)])
def test_N2_burn_in_matches_oracle(B, O, method, eps0, delta, nl):
    """Same seeds and schedule: every block's step, the adapted step, the whitening factor after each
    iteration's covariance window, the final ensemble and the best-fit point track the oracle's loop."""
    w = WL.tiny().with_chains(256, seed=19)
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    o = O.Oracle(w)
    ost = o.new_state(w.theta0)
    eps, th_best, lp_best, hist = st.burn_in(method, 2, 110, 60, 8, 23, eps0, delta, n_leapfrog=nl)
    eps_o, th_o, lp_o, hist_o = ost.burn_in(method, 2, 110, 60, 8, 23, eps0, f32(delta), n_leapfrog=nl)
    assert len(hist) == len(hist_o) == 2 * 8
    np.testing.assert_allclose(hist, hist_o, rtol=1e-6)
    assert eps == pytest.approx(eps_o, rel=1e-6)
    # the emulator runs in fp32 (rel 1e-5 bar): positions agree to that, not to fp64 rounding
    np.testing.assert_allclose(ctx.get_whitening(), o.get_whitening(), rtol=1e-5, atol=1e-7)
    th, lp, _ = st.get_f64(want_grad=False)
    np.testing.assert_allclose(th, ost.theta, rtol=0, atol=1e-5 * np.abs(ost.theta).max())
    np.testing.assert_allclose(th_best, th_o, rtol=0, atol=1e-5 * np.abs(ost.theta).max())
    assert lp_best == pytest.approx(lp_o, rel=1e-5, abs=1e-5)
    assert ctx.adapt_stats() == (2, 0) and st.get(want_grad=False)["step"] == 220
    # adaptation is left switched off: more steps do not move the whitening factor
    L0 = ctx.get_whitening()
    st.step_mh(5, 1, 0.1)
    assert np.array_equal(ctx.get_whitening(), L0)
    ctx.close()


def test_N2_burn_in_arguments(B):
    w = WL.tiny().with_chains(16, seed=1)
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    for args in ((3, 1, 10, 5, 5, 1, 0.1, 0.5), ("mh", 1, 10, 5, 5, 1, 0.1, 0.0), ("mh", 1, 10, 5, 5, 1, 0.1, 1.0),
                 ("mh", 1, 10, 11, 5, 1, 0.1, 0.5), ("mh", 1, 10, 5, 0, 1, 0.1, 0.5), ("mh", 1, 10, 5, 5, 1, 0.0, 0.5)):
        with pytest.raises(B.BestError) as e:
            st.burn_in(*args)
        assert e.value.code == B.BEST_ERR_ARG
    eps, th, lp, hist = st.burn_in("mh", 0, 10, 5, 5, 1, 0.1, 0.5)          # no iterations: nothing happens
    assert eps == f32(0.1) and len(hist) == 0 and st.get(want_grad=False)["step"] == 0
    eps, th, lp, hist = st.burn_in("mh", 1, 10, 0, 1, 1, 0.1, 0.5)          # no adaptation: covariance window only
    assert eps == f32(0.1) and ctx.adapt_stats() == (1, 0)
    ctx.close()


def test_T7_nonfinite_and_far_outside(B):
    w = WL.lcdm(n_chains=256, hidden=64, n_hidden=2, mlp_scale=3.0)
    th0 = w.theta0.copy()
    th0[:128] += 1e6 * (w.hi - w.lo).astype(np.float32)        # far outside the box: huge penalty slope
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(th0)
    before = st.get()
    st.step_hmc(2, 5, 50.0, 8)                                  # absurd ε ⇒ divergent trajectories
    after = st.get()
    assert np.isfinite(after["theta"]).all() and np.isfinite(after["logp"]).all()
    rejected = after["n_accept"] == 0
    assert rejected.sum() >= 200
    assert np.array_equal(after["theta"][rejected], before["theta"][rejected])
    ctx.close()


def test_argument_errors(B):
    w = WL.tiny().with_chains(7, seed=1)
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    for call in (lambda: st.step_aies(1, 1, 2.0), lambda: st.step_mh(1, 1, 0.0), lambda: st.step_mala(1, 1, -1.0),
                 lambda: st.step_hmc(1, 1, 0.1, 0)):
        with pytest.raises(B.BestError) as e:
            call()
        assert e.value.code == B.BEST_ERR_ARG
    st2 = ctx.new_state(w.theta0[:6])
    with pytest.raises(B.BestError):
        st2.step_aies(1, 1, 1.0)
    st2.step_aies(2, 1, 2.0)
    st.step_mh(0, 1, 0.3)                                        # empty call is a no-op
    assert st.get()["step"] == 0
    lp = np.zeros(0, np.float32)
    ctx.logp_grad(np.zeros((0, w.d), np.float32), 0, lp, None)   # empty batch
    ctx.close()


def test_probe_l2_read(B):
    """best_probe_l2_read: an L2-resident buffer is read faster than HBM can deliver (6.5 TB/s measured copy)
    and slower than any plausible L2 (50 TB/s); argument errors are reported, not clamped."""
    gbs = B.probe_l2_read(16 << 20, 10)
    assert 3.0e3 < gbs < 5.0e4, gbs
    for bad in ((1 << 19, 10), (200 << 20, 10), ((16 << 20) + 16, 10), (16 << 20, 0)):
        with pytest.raises(B.BestError) as e:
            B.probe_l2_read(*bad)
        assert e.value.code == B.BEST_ERR_ARG


# ---- BEST_PREC_FP32_TC: the exact path with every GEMM on the tensor cores (fp16-pair split operands) -----------
@pytest.mark.parametrize("name", ["lcdm", "lcdm_s3", "sterile"])
@pytest.mark.parametrize("variant", ["full", "mlp_only"])
def test_T1_fp32tc_logp_grad(B, O, name, variant):
    """Same bar as the FFMA path: rel 1e-5 on log π and, norm-wise per point, on the gradient (R17), on the full and
    the MLP-only target; 2048 + 77 probe points (box faces, ±20σ outliers, on/off the banana ridge)."""
    base = _targets(name)[0]
    w = WL.mlp_only(base) if variant == "mlp_only" else base
    n = 2048 + 77
    pts = WL.probe_points(base, n, seed=17)
    ctx = B.Context(w, B.PREC_FP32_TC)
    lp = np.zeros(n, np.float32)
    g = np.zeros((n, w.d), np.float32)
    ctx.logp_grad(pts, n, lp, g)
    lp_ref, g_ref = O.Oracle(w).logp_grad(pts)
    e = check_logp_grad(lp, g, lp_ref, g_ref, TOL[0], f"fp32tc/{name}/{variant}")
    print(f"[T1-fp32tc] {name} {variant}: logp err/S {e[0]:.2e}, grad ratio {e[1]:.2e}")
    ctx.close()


@pytest.mark.parametrize("net,method,kw", [("lcdm", "mh", dict(eps=0.3)), ("lcdm", "mala", dict(eps=0.3)),
                                           ("lcdm_s3", "hmc", dict(eps=0.1, n_leapfrog=8)),
                                           ("sterile", "mala", dict(eps=0.01)), ("sterile", "aies", dict(a=2.0))])
def test_T2_fp32tc_single_step(B, O, net, method, kw):
    """Single-step maps from identical state and streams: accept decisions identical to the oracle's outside
    |log u − log α| < 1e-5 (best.h: the split-operand GEMMs carry ~1.5e-6 relative error on the MLP output, the
    FFMA path 3e-7), post-state and caches at the fp32 tolerance."""
    w = _targets(net)[0].with_chains(2048 + 40, seed=5)
    _single_step(B, O, w, method, seed=77, prec=B.PREC_FP32_TC, window=1e-5, **kw)


def test_fp32tc_unsupported_and_split_invariance(B):
    with pytest.raises(B.BestError) as e:
        B.Context(WL.tiny(hidden=(32, 32)), B.PREC_FP32_TC)
    assert e.value.code == B.BEST_ERR_UNSUPPORTED
    w = WL.lcdm(n_chains=300)
    ctx = B.Context(w, B.PREC_FP32_TC)
    a, b = ctx.new_state(w.theta0), ctx.new_state(w.theta0)
    a.step_mala(6, 3, f32(0.3)); b.step_mala(2, 3, f32(0.3)); b.step_mala(4, 3, f32(0.3))
    ga, gb = a.get(), b.get()
    for k in ("theta", "logp", "grad", "n_accept"):
        assert np.array_equal(ga[k], gb[k]), k
    ctx.close()
