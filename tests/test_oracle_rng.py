"""Pins for the oracle's random-number layer (CPU only).

Each test checks the oracle against something OTHER than itself: published known answers, scipy's
Poisson pmf, closed-form moments of the uniform ball.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest
from scipy import stats

import oracle
import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(key):
    with open(os.path.join(GOLD, "paper_values.txt")) as f:
        for line in f:
            if line.startswith(key + " "):
                return float(line.split()[1])
    raise KeyError(key)


def test_philox_known_answers(olib):
    """Philox4x32-10 with the standard constants reproduces the published vectors."""
    n = 0
    with open(os.path.join(GOLD, "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = [int(x, 16) for x in line.split()]
            ctr, key, want = np.array(w[:4], np.uint32), np.array(w[4:6], np.uint32), w[6:]
            out = np.zeros(4, np.uint32)
            olib.oracle_philox4x32_10(ctr.ctypes.data, key.ctypes.data, out.ctypes.data)
            assert [int(x) for x in out] == want
            n += 1
    assert n == 3


def test_philox_counter_sensitivity(olib):
    """Every counter/key word matters: flipping any one bit changes the block (no dropped field)."""
    base_c, base_k = np.array([1, 2, 3, 4], np.uint32), np.array([5, 6], np.uint32)
    ref = np.zeros(4, np.uint32)
    olib.oracle_philox4x32_10(base_c.ctypes.data, base_k.ctypes.data, ref.ctypes.data)
    for w in range(6):
        c, k = base_c.copy(), base_k.copy()
        if w < 4:
            c[w] ^= np.uint32(1 << 7)
        else:
            k[w - 4] ^= np.uint32(1 << 7)
        out = np.zeros(4, np.uint32)
        olib.oracle_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
        assert not np.array_equal(out, ref)
        # avalanche: about half of the 128 bits flip
        flips = sum(bin(int(a) ^ int(b)).count("1") for a, b in zip(out, ref))
        assert 30 < flips < 98


def test_u32_to_float_exact(olib):
    """S4: u = ((x>>9)+0.5) 2^-23 in (0,1), exactly representable; s = 2u-1 is antisymmetric."""
    for x in (0, 1, 511, 512, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF, 0x12345678):
        u = olib.oracle_unit01(x)
        assert u == ((x >> 9) + 0.5) / 2 ** 23          # exact in binary32 and binary64
        assert 0.0 < u < 1.0
        s = olib.oracle_sym_unit(x)
        assert s == 2.0 * ((x >> 9) + 0.5) / 2 ** 23 - 1.0
        assert olib.oracle_sym_unit(x ^ 0xFFFFFFFF) == -s
    assert olib.oracle_unit01(0) == 2.0 ** -24
    assert olib.oracle_unit01(0xFFFFFFFF) == 1.0 - 2.0 ** -24


@pytest.mark.parametrize("lam", [0.3, 5.0, 43.2, 157.72, 532.4, 2778.3])
def test_poisson_table_matches_pmf(olib, lam):
    """S2: table differences reproduce the Poisson pmf (scipy, independent implementation)."""
    T = np.zeros(4096, np.uint64)
    klo = C.c_int64()
    n = olib.oracle_poisson_table(lam, C.byref(klo), T.ctypes.data, len(T))
    assert n > 0
    Ti = [int(x) for x in T[:n]]
    assert all(b >= a for a, b in zip(Ti, Ti[1:]))
    # exact reference: 60-digit decimal arithmetic (scipy's own pmf is only good to ~1e-13 relative here)
    import decimal
    decimal.getcontext().prec = 60
    D = decimal.Decimal
    lamD = D(repr(lam))
    p = (-lamD).exp()
    cdf, ref = D(0), {}
    for kk in range(0, klo.value + n):
        cdf += p
        ref[kk] = cdf
        p = p * lamD / D(kk + 1)
    two64 = D(2) ** 64
    worst = max(abs(D(Ti[j]) / two64 - ref[klo.value + j]) for j in range(n - 1))
    # fp64 recurrence + cumulative sum: a few hundred ulp of 1.0 at most
    assert worst < D("2e-14"), worst
    assert Ti[-1] == 2 ** 64 - 1 or 1 - Ti[-1] / 2 ** 64 < 1e-15
    # and against scipy as a second, independent implementation (looser: its pmf carries ~1e-13 rel. error)
    k = np.arange(klo.value, klo.value + n)
    Tf = np.array(Ti, np.float64) / 2.0 ** 64
    assert np.max(np.abs(Tf - stats.poisson.cdf(k, lam))) < 1e-12


@pytest.mark.parametrize("lam", [43.2, 2778.3])
def test_poisson_draw_moments(olib, lam):
    """L67: N_p ~ Poisson with 'mean and variance lambda'."""
    rng = np.random.default_rng(7)
    n = 400000
    U = rng.integers(0, 2 ** 64, size=n, dtype=np.uint64)
    out = np.zeros(n, np.int64)
    olib.oracle_poisson_draws(lam, U.ctypes.data, n, out.ctypes.data)
    se_mean = math.sqrt(lam / n)
    assert abs(out.mean() - lam) < 4.5 * se_mean
    se_var = lam * math.sqrt(2.0 / n + 1.0 / (lam * n))
    assert abs(out.var() - lam) < 4.5 * se_var
    # inversion is monotone in U
    order = np.argsort(U)
    assert np.all(np.diff(out[order]) >= 0)
    # and exact: draw = number of k with CDF(k) <= U/2^64, checked against scipy at the sampled points
    cdf_below = stats.poisson.cdf(out - 1, lam)       # P(N <= draw-1) must be <= u
    u = U.astype(np.float64) / 2.0 ** 64
    assert np.all(cdf_below <= u + 1e-12)
    assert np.all(stats.poisson.cdf(out, lam) >= u - 1e-12)


def test_poisson_zero():
    o = oracle.lib()
    out = np.zeros(3, np.int64)
    U = np.array([0, 2 ** 63, 2 ** 64 - 1], np.uint64)
    o.oracle_poisson_draws(0.0, U.ctypes.data, 3, out.ctypes.data)
    assert list(out) == [0, 0, 0]


def test_lambda_matches_config_text():
    """configs[2] prints '~2.8k depletant insertions per move'; lambda = n_R 4 pi R^3/3 (L67, L156)."""
    cfg = workloads.config("C3")
    p = oracle.binding.make_params(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max)
    lam = oracle.lib().oracle_lambda(C.byref(p), cfg.n_R())
    assert abs(lam - _gold("C3_lambda")) < 0.05
    assert 2700 < lam < 2900
    for name in ("C1", "C2", "C4", "C5"):
        cfg = workloads.config(name)
        p = oracle.binding.make_params(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, cfg.disk_a,
                                       cfg.disk_s)
        lam = oracle.lib().oracle_lambda(C.byref(p), cfg.n_R())
        assert abs(lam / cfg.lam - 1.0) < 1e-6


def test_ball_samples_uniform(olib):
    """S3 / L67 'uniformly': moments and radial law of the cube-rejection ball sampler."""
    n, R = 600000, 0.6
    out = np.zeros((n, 3), np.float32)
    olib.oracle_ball_samples(1, 0, 3, 12345, n, R, out.ctypes.data)
    d = out.astype(np.float64)
    r = np.linalg.norm(d, axis=1)
    assert r.max() <= R * (1 + 1e-6)
    # mean 0, per-axis variance R^2/5, no cross-correlation
    se = R / math.sqrt(5 * n)
    assert np.all(np.abs(d.mean(0)) < 4.5 * se)
    assert np.all(np.abs((d * d).mean(0) - R * R / 5) < 4.5 * (R * R) * math.sqrt(12.0 / 175.0 / n))
    cov = np.cov(d.T)
    assert abs(cov[0, 1]) < 5 * (R * R / 5) / math.sqrt(n)
    assert abs(cov[0, 2]) < 5 * (R * R / 5) / math.sqrt(n)
    # fraction inside radius rho is (rho/R)^3
    for rho in (0.1, 0.3, 0.45, 0.55):
        p = (rho / R) ** 3
        assert abs((r < rho).mean() - p) < 4.5 * math.sqrt(p * (1 - p) / n)
    # distinct streams (different colloid id / step) give different points
    out2 = np.zeros((16, 3), np.float32)
    olib.oracle_ball_samples(1, 0, 3, 12346, 16, R, out2.ctypes.data)
    assert not np.array_equal(out2, out[:16])
    out3 = np.zeros((16, 3), np.float32)
    olib.oracle_ball_samples(1, 1, 3, 12345, 16, R, out3.ctypes.data)
    assert not np.array_equal(out3, out[:16])
