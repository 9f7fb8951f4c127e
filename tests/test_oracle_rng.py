"""Pins for the oracle's RNG layer (Philox KATs, transforms' closed forms)."""
import math
import os

import numpy as np
import pytest
from scipy import stats

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden_constants():
    out = {}
    with open(os.path.join(GOLD, "paper_constants.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            out[k] = float(v)
    return out


def test_philox_known_answers(oracle_mod):
    n = 0
    with open(os.path.join(GOLD, "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = [int(x, 16) for x in line.split()]
            assert oracle_mod.philox(w[0:4], w[4:6]) == w[6:10]
            n += 1
    assert n == 3


def test_u01_endpoints_and_fp32_exact(oracle_mod):
    assert oracle_mod.u01(0) == 0.5 * 2.0 ** -23
    assert oracle_mod.u01(0xFFFFFFFF) == 1.0 - 0.5 * 2.0 ** -23
    assert oracle_mod.u01(0x1FF) == 0.5 * 2.0 ** -23         # low 9 bits are dropped
    assert oracle_mod.u01(0x200) == 1.5 * 2.0 ** -23
    for x in (0, 1 << 9, 0x80000000, 0xDEADBEEF, 0xFFFFFE00, 0xFFFFFFFF):
        u = oracle_mod.u01(x)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u                      # exactly representable in fp32


def test_stream_layout_R1(oracle_mod):
    """counter = (chain, step lo, step hi, slot), key = (seed lo, seed hi); slot 0 = control,
    slot 1+j = normals of dims 4j..4j+3 via Box–Muller pairs (reading R1/R3)."""
    seed, chain, step, d = 0x123456789ABCDEF0, 77, (5 << 32) | 9, 7
    key = [seed & 0xFFFFFFFF, seed >> 32]
    w = oracle_mod.philox([chain, step & 0xFFFFFFFF, step >> 32, 0], key)
    u, uz, raw = oracle_mod.control(seed, chain, step)
    assert (u, uz, raw) == (oracle_mod.u01(w[0]), oracle_mod.u01(w[1]), w[2])
    xi = oracle_mod.normals(seed, chain, step, d)
    for j in range(2):
        w = oracle_mod.philox([chain, step & 0xFFFFFFFF, step >> 32, 1 + j], key)
        for p in range(2):
            u1, u2 = oracle_mod.u01(w[2 * p]), oracle_mod.u01(w[2 * p + 1])
            r, phi = math.sqrt(-2 * math.log(u1)), 2 * math.pi * u2
            for t, val in enumerate((r * math.cos(phi), r * math.sin(phi))):
                k = 4 * j + 2 * p + t
                if k < d:
                    assert xi[k] == pytest.approx(val, rel=1e-14, abs=1e-15)
    # different chains / steps / seeds give different streams
    assert not np.allclose(xi, oracle_mod.normals(seed, chain + 1, step, d))
    assert not np.allclose(xi, oracle_mod.normals(seed, chain, step + 1, d))
    assert not np.allclose(xi, oracle_mod.normals(seed + 1, chain, step, d))


def test_normals_distribution(oracle_mod):
    d, n = 28, 36000                       # ~1e6 normals
    x = np.concatenate([oracle_mod.normals(11, c, 3, d) for c in range(n)])
    assert abs(x.mean()) < 4.0 / math.sqrt(x.size)
    assert abs(x.var() - 1.0) < 4.0 * math.sqrt(2.0 / x.size)
    assert abs(stats.kurtosis(x)) < 4.0 * math.sqrt(24.0 / x.size)
    assert stats.kstest(x, "norm").pvalue > 1e-3
    # components are uncorrelated across the Box–Muller pair and across dims
    X = x.reshape(n, d)
    Cm = np.corrcoef(X.T)
    assert np.abs(Cm - np.eye(d)).max() < 5.0 / math.sqrt(n)


def test_stretch_z_closed_forms(oracle_mod):
    g = _golden_constants()
    a = g["stretch_a"]
    assert oracle_mod.stretch_z(0.0, a) == g["stretch_z_at_u0"]
    assert oracle_mod.stretch_z(1.0, a) == g["stretch_z_at_u1"]
    # eq (2.15) is the inverse CDF of g(z) ∝ 1/sqrt(z) on [1/a, a] (eq 2.14):
    # G(z) = (sqrt z - 1/sqrt a) / (sqrt a - 1/sqrt a)
    for a_ in (2.0, 1.5, 3.0):
        for u in np.linspace(0, 1, 17):
            z = oracle_mod.stretch_z(float(u), a_)
            G = (math.sqrt(z) - 1 / math.sqrt(a_)) / (math.sqrt(a_) - 1 / math.sqrt(a_))
            assert G == pytest.approx(u, abs=1e-14)
            assert 1 / a_ - 1e-15 <= z <= a_ + 1e-15
    # E[z] = (a + 1 + 1/a)/3 by midpoint quadrature over u
    m = 4000
    us = (np.arange(m) + 0.5) / m
    zs = np.array([oracle_mod.stretch_z(float(u), a) for u in us])
    assert zs.mean() == pytest.approx(g["stretch_mean_z"], rel=1e-6)


def test_accept_rule_R7(oracle_mod):
    assert oracle_mod.accept(0.5, 0.0)                 # log 0.5 < 0
    assert not oracle_mod.accept(0.5, math.log(0.5))   # strict
    assert oracle_mod.accept(0.5, float("inf"))
    assert not oracle_mod.accept(0.5, float("-inf"))
    assert not oracle_mod.accept(0.5, float("nan"))    # NaN ⇒ reject
