"""Pins for the oracle's target: MLP vs torch fp64, finite differences, Gaussian vs scipy, penalty."""
import math

import numpy as np
import pytest
import torch
from scipy import stats

from paper_2606_04895_b200 import workloads as WL


def _torch_mlp(w):
    layers = []
    for k, (W, b) in enumerate(zip(w.W, w.b)):
        lin = torch.nn.Linear(W.shape[1], W.shape[0]).double()
        with torch.no_grad():
            lin.weight.copy_(torch.from_numpy(W.astype(np.float64)))
            lin.bias.copy_(torch.from_numpy(b.astype(np.float64)))
        layers.append(lin)
        if k < len(w.W) - 1:
            layers.append(torch.nn.Tanh() if w.activation == WL.ACT_TANH else torch.nn.SiLU())
    return torch.nn.Sequential(*layers)


@pytest.mark.parametrize("act", [WL.ACT_TANH, WL.ACT_SILU])
def test_mlp_matches_torch_fp64(oracle_mod, act):
    w = WL.tiny(activation=act, hidden=(48, 40, 24))
    o = oracle_mod.Oracle(w)
    th = WL.probe_points(w, 64, seed=5).astype(np.float64)
    th[:8] *= 6.0                                     # saturating region of tanh / SiLU tails
    out, grad = o.mlp(th)
    net = _torch_mlp(w)
    x = torch.from_numpy(th).requires_grad_(True)
    y = net(x).squeeze(-1)
    (g,) = torch.autograd.grad(y.sum(), x)
    np.testing.assert_allclose(out, y.detach().numpy(), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(grad, g.numpy(), rtol=1e-11, atol=1e-13)


def test_silu_overflow_safe(oracle_mod):
    w = WL.tiny(activation=WL.ACT_SILU)
    o = oracle_mod.Oracle(WL.mlp_only(w))
    th = np.full((2, w.d), 1e4)
    th[1] *= -1
    out, grad = o.mlp(th)
    assert np.all(np.isfinite(out)) and np.all(np.isfinite(grad))


def _fd_grad(f, th, h_rel=1e-5):
    g = np.zeros_like(th)
    for i in range(th.size):
        h = h_rel * max(1.0, abs(th[i]))
        tp, tm = th.copy(), th.copy()
        tp[i] += h
        tm[i] -= h
        g[i] = (f(tp) - f(tm)) / (2 * h)
    return g


@pytest.mark.parametrize("maker", ["tiny", "sterile_small", "lcdm_small"])
def test_full_target_gradient_finite_differences(oracle_mod, maker):
    if maker == "tiny":
        w = WL.tiny()
    elif maker == "sterile_small":
        w = WL.sterile(n_chains=8, hidden=32, n_hidden=2)
    else:
        w = WL.lcdm(n_chains=8, hidden=32, n_hidden=3, mlp_scale=3.0)
    o = oracle_mod.Oracle(w)
    pts = WL.probe_points(w, 32, seed=9).astype(np.float64)
    f = lambda t: o.logp_grad(t[None, :], want_grad=False)[0][0]
    _, grad = o.logp_grad(pts)
    worst = 0.0
    for r in range(pts.shape[0]):
        # skip points sitting exactly on a penalty kink (box face): FD straddles the C1 joint
        g_fd = _fd_grad(f, pts[r])
        err = np.linalg.norm(g_fd - grad[r]) / max(np.linalg.norm(grad[r]), 1e-12)
        worst = max(worst, err)
    assert worst < 1e-6


def test_gaussian_term_vs_scipy(oracle_mod):
    w = WL.gaussian_only(WL.lcdm(n_chains=4, hidden=8, n_hidden=1))
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    pts = WL.probe_points(WL.lcdm(n_chains=4, hidden=8, n_hidden=1), 64, seed=3).astype(np.float64)
    logp, grad = o.logp_grad(pts)
    ref = stats.multivariate_normal(mean=w.mu, cov=w.Sigma).logpdf(pts)
    # unnormalised: differences agree
    np.testing.assert_allclose(logp - logp[0], ref - ref[0], rtol=1e-9, atol=1e-8)
    g_ref = -np.linalg.solve(w.Sigma, (pts - w.mu).T).T
    np.testing.assert_allclose(grad, g_ref, rtol=1e-8, atol=1e-8)


def test_banana_term(oracle_mod):
    w = WL.sterile(n_chains=4, hidden=8, n_hidden=1)
    w = WL.gaussian_only(w)
    w.mu = w.Sigma_inv = None
    w.lo = w.hi = None
    o = oracle_mod.Oracle(w)
    th = np.zeros((3, 29))
    th[0, 27], th[0, 28] = 1.5, 2.25            # on the ridge θ28 = θ27²  ⇒ 0, zero gradient
    th[1, 27], th[1, 28] = 1.0, 1.3             # t = 0.3 ⇒ −0.09/(2·0.01) = −4.5
    th[2, 27], th[2, 28] = -2.0, 3.5            # t = −0.5 ⇒ −12.5
    logp, grad = o.logp_grad(th)
    np.testing.assert_allclose(logp, [0.0, -4.5, -12.5], atol=1e-12)
    assert np.abs(grad[0]).max() < 1e-12
    np.testing.assert_allclose(grad[1, [27, 28]], [2 * 1.0 * 0.3 / 0.01, -0.3 / 0.01], rtol=1e-12)
    assert np.count_nonzero(grad[1]) == 2


def test_box_penalty_R6(oracle_mod):
    # zero value / gradient inside and on the faces
    f0, df0 = oracle_mod.pen_f(0.0)
    assert f0 == 0.0 and df0 == 0.0
    assert oracle_mod.pen_f(-3.0) == (0.0, 0.0)
    # C1 at t = 40 and linear beyond
    fm, dfm = oracle_mod.pen_f(40.0)
    fp, dfp = oracle_mod.pen_f(40.0 + 1e-9)
    assert fp == pytest.approx(fm, rel=1e-8)           # value continuous (Δt·slope/f ≈ 1e-9)
    assert dfp == pytest.approx(dfm, rel=1e-15)         # slope continuous: C1 joint
    f60, df60 = oracle_mod.pen_f(60.0)
    assert df60 == dfp and f60 == pytest.approx(fm + dfm * 20.0, rel=1e-14)
    # e^t − 1 − t
    f1, df1 = oracle_mod.pen_f(1.0)
    assert f1 == pytest.approx(math.e - 2.0, rel=1e-14) and df1 == pytest.approx(math.e - 1, rel=1e-14)
    # on the target: 1% of the width outside ⇒ pen = e − 2 ≈ 0.72 (κ=1, γ=100); 5% ⇒ ≈ 142
    w = WL.gaussian(3, 1, seed=4)
    wb = WL.gaussian(3, 1, seed=4)
    wb.mu = wb.Sigma_inv = None
    o = oracle_mod.Oracle(wb)
    width = wb.hi - wb.lo
    th = (0.5 * (wb.lo + wb.hi))[None, :].repeat(5, 0)
    th[1, 0] = wb.hi[0]                          # on the face
    th[2, 0] = wb.hi[0] + 0.01 * width[0]
    th[3, 1] = wb.lo[1] - 0.05 * width[1]
    th[4, 2] = wb.lo[2] - 10.0 * width[2]        # t = 1000 ⇒ linear branch, finite
    logp, grad = o.logp_grad(th)
    assert logp[0] == 0.0 and logp[1] == 0.0 and np.all(grad[:2] == 0.0)
    assert -logp[2] == pytest.approx(math.e - 2.0, rel=1e-9)
    assert -logp[3] == pytest.approx(math.exp(5.0) - 6.0, rel=1e-9)
    assert grad[2, 0] == pytest.approx(-(math.e - 1.0) * 100.0 / width[0], rel=1e-9)   # pushes back in
    assert grad[3, 1] == pytest.approx(+(math.exp(5.0) - 1.0) * 100.0 / width[1], rel=1e-9)
    assert np.isfinite(logp[4]) and np.isfinite(grad[4]).all() and grad[4, 2] > 0
    _ = w


def test_whitening_constant_eq_2_12(oracle_mod):
    w = WL.lcdm(n_chains=2, hidden=8, n_hidden=1)
    o = oracle_mod.Oracle(w)
    sign, logdet = np.linalg.slogdet(w.L)
    assert sign == 1.0
    assert o.log_det_L() == pytest.approx(logdet, rel=1e-12)
    np.testing.assert_array_equal(o.get_whitening(), np.tril(w.L))
