"""Pins for the oracle's two options (CPU only): SURVEY 8(f) NEXT-1, the shell-restricted insertion volume of PAPER.md
L158 (reading R-N1), and NEXT-4, the exact Rosenbluth form of the configurational-bias weight (refs 27, 28,
33; reading R-N4).

No expected value comes from the oracle: the shell's radial law and volume are closed forms, the acceptance targets
are the same Eq. 8 / Eq. 15 closed forms the default path is pinned to (the options change the sampling volume and the
weight, never the transition rate), and the cube root is compared with numpy's.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest

import oracle
import workloads
from oracle import binding
from oracle.binding import FLAG_ROSENBLUTH, FLAG_SHELL

from test_oracle_physics import iso_accept, lens, sphere_oracle

SQRT3_F32 = float(np.float32(1.7320508))


def _vp(a):
    return a.ctypes.data_as(C.c_void_p)


# ------------------------------------------------------------------ the libm-free cube root
def test_cbrt_fixed_matches_numpy_to_two_ulp():
    L = oracle.lib()
    t = np.concatenate([np.logspace(-12, 0.5, 40000), np.linspace(0.05, 0.25, 20000)]).astype(np.float32)
    got = np.array([L.oracle_cbrt_fixed(float(x)) for x in t[::7]], np.float64)
    want = np.cbrt(t[::7].astype(np.float64))
    assert np.max(np.abs(got / want - 1.0)) < 2.5e-7


# ------------------------------------------------------------------ the shell sampler
@pytest.mark.parametrize("shape,sigma_d,d_max,disk", [("sphere", 0.05, 0.05, (0.0, 0.0)), ("sphere", 0.2, 0.01, (0.0, 0.0)),
                                                     ("halfball", 0.2, 0.1, (0.0, 0.0)), ("spherodisk", 0.15, 0.02, (0.4, 0.1))])
def test_shell_radius_law_isotropy_and_lambda(shape, sigma_d, d_max, disk):
    """R-N1: R_in = max(0, r_in - sqrt(3) d_max) with r_in = R (sphere), r_d (half-ball), s + r_d (spherodisk);
    samples uniform in R_in < |d| <= R: (|d|^3 - R_in^3) / (R^3 - R_in^3) is uniform on (0,1), directions isotropic;
    lambda = n_R (4 pi / 3)(R^3 - R_in^3)."""
    L = oracle.lib()
    par = binding.make_params(shape, 1.0, sigma_d, 20.0, 0.1, *disk)
    R, rd = 0.5 * (1.0 + sigma_d), 0.5 * sigma_d
    r_in = {"sphere": R, "halfball": rd, "spherodisk": disk[1] + rd}[shape]
    want_rin = max(0.0, r_in - SQRT3_F32 * d_max)
    rin = C.c_float()
    n_R = 1234.5
    lam = L.oracle_shell(C.byref(par), n_R, d_max, 0, C.byref(rin))
    assert abs(rin.value - want_rin) < 1e-6
    assert abs(lam / (n_R * 4.0 * math.pi / 3.0 * (R ** 3 - want_rin ** 3)) - 1.0) < 2e-6
    n = 300000
    d = np.zeros((n, 3), np.float32)
    L.oracle_shell_samples(C.byref(par), d_max, 11, 3, 5, 77, n, _vp(d))
    d = d.astype(np.float64)
    r = np.linalg.norm(d, axis=1)
    assert r.min() >= want_rin * (1 - 1e-6) and r.max() <= R * (1 + 1e-6)
    u = np.sort((r ** 3 - want_rin ** 3) / (R ** 3 - want_rin ** 3))
    ks = np.max(np.abs(u - (np.arange(n) + 0.5) / n))
    assert ks < 1.95 / math.sqrt(n), ks                      # Kolmogorov-Smirnov, alpha = 0.001
    e = d / r[:, None]
    assert np.all(np.abs(e.mean(axis=0)) < 4.0 / math.sqrt(3 * n))
    m2 = e.T @ e / n
    assert np.all(np.abs(m2 - np.eye(3) / 3.0) < 4.0 * math.sqrt(4.0 / 45.0 / n) + 1e-9), m2


# ------------------------------------------------------------------ the transition rate is unchanged (Eq. 15)
def _iso_rate(sigma_d, n_R, d, ndraw, flags, eval_dmax, L_=None):
    """Acceptance rate of one fixed translation of length d of an isolated sphere (L_: a mutant build instead of the
    oracle library)."""
    L_ = L_ or oracle.lib()
    L_.oracle_set_threads(os.cpu_count() or 1)
    p4 = np.zeros((1, 4), np.float32)
    p4[0, :3] = 4.0
    par = binding.make_params("sphere", 1.0, sigma_d, 8.0, 0.1)
    h = L_.oracle_create(C.byref(par), 1, _vp(p4), None)
    assert h
    L_.oracle_set_flags(h, flags, eval_dmax)
    assert L_.oracle_build_cells(h, 1, 0) == 0
    u = np.random.default_rng(5).standard_normal(3)
    u /= np.linalg.norm(u)
    new = np.float32(4.0) + (d * u).astype(np.float32)
    d_eff = float(np.linalg.norm(new.astype(np.float64) - 4.0))
    out = np.empty(ndraw, np.uint8)
    assert L_.oracle_eval_moves(h, 1, 0, ndraw, 0, _vp(new), None, float(n_R), 0, _vp(out)) == 0
    L_.oracle_destroy(h)
    assert set(np.unique(out)) <= {1, 4}
    return float((out == 1).mean()), d_eff


@pytest.mark.parametrize("sigma_d,n_R,d,eval_dmax,ndraw", [(0.2, 47.746, 0.1, 0.1, 400000), (0.2, 47.746, 0.03, 0.02, 200000),
                                                            (0.05, 4583.66, 0.001, 0.001, 200000), (0.1, 50.0, 0.09, 0.06, 400000)])
def test_shell_isolated_colloid_keeps_the_closed_form(sigma_d, n_R, d, eval_dmax, ndraw):
    """north_star check 2 with the shell on: P(accept) = exp(-n_R (V_s - lens(d))) within 3 sigma.  The rejecting region
    (new exclusion sphere minus the old one) lies inside the shell for every |move| <= sqrt(3) d_max (Eq. 12)."""
    assert d <= SQRT3_F32 * eval_dmax
    acc, d_eff = _iso_rate(sigma_d, n_R, d, ndraw, FLAG_SHELL, eval_dmax)
    p = iso_accept(n_R, 0.5 * (1.0 + sigma_d), d_eff)
    assert abs(acc - p) < 3.0 * math.sqrt(p * (1 - p) / ndraw) + 1e-9, (acc, p)


def test_shell_minus_the_hard_core_violates_the_closed_form(tmp_path):
    """Why R-N1 does not take L158's "V_excl,i minus V'_core,i" with the colloid's hard core as the core: for a move
    longer than the depletant radius part of the new-minus-old region lies inside the new hard core, the literal shell
    misses it and accepts too often (Eq. 12's V_0 >= V'_excl minus V_excl fails).  Same measurement as above, mutated shell."""
    sigma_d, n_R, d, ndraw = 0.1, 50.0, 0.09, 400000
    from conftest import build_mutant_oracle
    literal = build_mutant_oracle(tmp_path, "literal_core", "  sh.Rin = rin - 1.7320508f * d_max;", "  sh.Rin = 0.5f * g.dcirc;")
    acc, d_eff = _iso_rate(sigma_d, n_R, d, ndraw, FLAG_SHELL, 0.06, literal)
    p = iso_accept(n_R, 0.55, d_eff)
    assert acc - p > 6.0 * math.sqrt(p * (1 - p) / ndraw), (acc, p)


def _pair_counts(ra, rb, nd, n_trial, n_R, sigma_d, flags, seed=7):
    """Accepted counts of the fixed move r_a -> r_b of sphere 0 next to the fixed sphere 1, and of its reverse."""
    L_ = oracle.lib()
    acc = []
    L_.oracle_set_threads(os.cpu_count() or 1)
    for r0, r1 in ((ra, rb), (rb, ra)):
        p4 = np.zeros((2, 4), np.float32)
        p4[0, :3] = [3.0 + (2.0 - r0), 4.0, 4.0]
        p4[1, :3] = [5.0, 4.0, 4.0]
        par = binding.make_params("sphere", 1.0, sigma_d, 8.0, 0.1)
        h = L_.oracle_create(C.byref(par), 2, _vp(p4), None)
        assert h
        L_.oracle_set_flags(h, flags, -1.0)
        assert L_.oracle_build_cells(h, 1, 0) == 0
        new = np.array([3.0 + (2.0 - r1), 4.0, 4.0], np.float32)
        out = np.empty(nd, np.uint8)
        assert L_.oracle_eval_moves(h, seed, 0, nd, 0, _vp(new), None, float(n_R), n_trial, _vp(out)) == 0
        assert set(np.unique(out)) <= ({1, 4} if n_trial == 0 else {1, 5})
        acc.append(int((out == 1).sum()))
        L_.oracle_destroy(h)
    L_.oracle_set_threads(1)
    return acc


def _ratio_error(ra, rb, nd, n_trial, n_R, sigma_d, flags):
    R = 0.5 * (1.0 + sigma_d)
    fwd, rev = _pair_counts(ra, rb, nd, n_trial, n_R, sigma_d, flags)
    want = math.exp(n_R * (lens(R, rb) - lens(R, ra)))
    return (fwd / max(rev, 1)) / want - 1.0, math.sqrt(1.0 / max(fwd, 1) + 1.0 / max(rev, 1)), fwd, rev


def test_shell_two_sphere_ratio_plain_rule():
    """Detailed balance w.r.t. the Asakura-Oosawa weight with a neighbour present and the shell on (check 3, per move)."""
    n_R = workloads.config("C1").n_R()
    err, sig, fwd, rev = _ratio_error(1.05, 1.12, 2000000, 0, n_R, 0.2, FLAG_SHELL)
    assert abs(err) < 3.0 * sig, (err, sig, fwd, rev)


# ------------------------------------------------------------------ the exact Rosenbluth weight (R-N4)
@pytest.mark.parametrize("n_trial,flags", [(2, FLAG_ROSENBLUTH), (4, FLAG_ROSENBLUTH), (10, FLAG_ROSENBLUTH),
                                           (4, FLAG_ROSENBLUTH | FLAG_SHELL)])
def test_rosenbluth_weight_obeys_detailed_balance_without_allowance(n_trial, flags):
    """acc(r->r')/acc(r'->r) = exp(n_R [V_ov(r') - V_ov(r)]) at 4e6 draws per direction within 3.3 sigma and NO systematic
    allowance (Eq. 16 as adopted, R-G1, needs 1 %: tests/test_oracle_physics.py).  Same geometry as the Eq. 16 pins:
    forward and reverse success fractions differ."""
    n_R = workloads.config("C1").n_R()
    err, sig, fwd, rev = _ratio_error(1.02, 1.10, 4000000, n_trial, n_R, 0.2, flags)
    assert abs(err) < 3.3 * sig, (n_trial, err, sig, fwd, rev)


# ------------------------------------------------------------------ bookkeeping
def test_flags_zero_is_the_default_path_and_options_keep_the_invariants():
    cfg = workloads.config("C2", 2048)
    pos, _ = workloads.generate(cfg)
    a = oracle.Oracle("sphere", 1.0, cfg.sigma_d, cfg.box_L, cfg.d_max, pos)
    b = oracle.Oracle("sphere", 1.0, cfg.sigma_d, cfg.box_L, cfg.d_max, pos)
    b.set_flags(0)
    a.run(1, 0, 5, cfg.n_R(), cfg.d_max)
    b.run(1, 0, 5, cfg.n_R(), cfg.d_max)
    assert np.array_equal(a.pos.view(np.uint32), b.pos.view(np.uint32)) and a.counters() == b.counters()
    s = oracle.Oracle("sphere", 1.0, cfg.sigma_d, cfg.box_L, cfg.d_max, pos)
    s.set_flags(FLAG_SHELL)
    s.run(1, 0, 20, cfg.n_R(), cfg.d_max)
    cs, ca = s.counters(), a.counters()
    assert s.count_overlaps() == 0
    assert cs["dep_needed"] <= cs["dep_drawn"] and cs["dep_evaluated"] == cs["dep_needed"]
    # the shell holds the fraction 1 - (R_in / R)^3 of the ball: that many fewer depletants are drawn per move
    R = 0.5 * (1.0 + cfg.sigma_d)
    frac = 1.0 - ((R - SQRT3_F32 * cfg.d_max) / R) ** 3
    per_move_s = cs["dep_drawn"] / (cs["trials_trans"] - cs["rej_boundary"] - cs["rej_hard"])
    per_move_a = ca["dep_drawn"] / (ca["trials_trans"] - ca["rej_boundary"] - ca["rej_hard"])
    assert abs(per_move_s / per_move_a / frac - 1.0) < 0.02


# ------------------------------------------------------------------ free-volume measurement (Fig. 4)
def _free_fraction(shape, pos, quat, L, sigma_d, n, disk=(0.0, 0.0)):
    p4 = np.zeros((len(pos), 4), np.float32)
    p4[:, :3] = pos
    o = oracle.Oracle(shape, 1.0, sigma_d, L, 0.1, p4, quat, *disk, threads=os.cpu_count() or 1)
    o.build_cells(3, 9)
    return o.free_volume(3, 9, n) / n


def test_free_volume_closed_forms():
    """Fraction of uniform test depletants that overlap no colloid = 1 - (excluded volume) / V: one sphere (4 pi R^3/3),
    two spheres with overlapping exclusion spheres (minus the lens, ref. 17), one half-ball and one spherodisk
    (Steiner volumes 0.557698 and 0.319281), 3 sigma at 2e6 points."""
    n, L = 2000000, 6.0
    V = L ** 3
    Vs = 4.0 * math.pi * 0.6 ** 3 / 3.0
    q = np.array([[0.3, -0.5, 0.2, 0.78]], np.float32)
    q /= np.linalg.norm(q)
    cases = [("sphere", [[1.0, 2.0, 3.0]], None, 0.2, (0.0, 0.0), Vs),
             ("sphere", [[1.0, 2.0, 3.0], [2.05, 2.0, 3.0]], None, 0.2, (0.0, 0.0), 2.0 * Vs - lens(0.6, 1.05)),
             ("sphere", [[5.9, 0.1, 3.0]], None, 0.2, (0.0, 0.0), Vs),                      # across the periodic boundary
             ("halfball", [[1.0, 2.0, 3.0]], q, 0.2, (0.0, 0.0), 0.557698),
             ("spherodisk", [[1.0, 2.0, 3.0]], q, 0.15, (0.4, 0.1), 0.319281)]
    for shape, pos, quat, sd, disk, vexcl in cases:
        got = _free_fraction(shape, pos, quat, L, sd, n, disk)
        want = 1.0 - vexcl / V
        assert abs(got - want) < 3.0 * math.sqrt(want * (1 - want) / n) + 1e-6, (shape, got, want)


def test_free_volume_equals_brute_force_on_the_same_points():
    """C1 (256 spheres): the same Philox points (rebuilt here from the separately pinned block function and u32->float map)
    against all 256 centres in numpy fp64 with the minimum image; equal counts up to points within 1e-6 of a surface."""
    cfg = workloads.config("C1")
    pos, _ = workloads.generate(cfg)
    o = oracle.Oracle("sphere", 1.0, cfg.sigma_d, cfg.box_L, cfg.d_max, pos, threads=os.cpu_count() or 1)
    o.build_cells(7, 2)
    n = 40000
    got = o.free_volume(7, 2, n)
    L_ = oracle.lib()
    pts = np.zeros((n, 3))
    ctr, key, out = np.zeros(4, np.uint32), np.array([7, 2], np.uint32), np.zeros(4, np.uint32)
    for s in range(n):
        ctr[:] = (s, 0, 0, 7)                    # purpose FREEVOL = 7, colour 0, attempt 0
        L_.oracle_philox4x32_10(_vp(ctr), _vp(key), _vp(out))
        pts[s] = [np.float32(L_.oracle_unit01(int(out[a]))) * np.float32(cfg.box_L) for a in range(3)]
    Lb = float(np.float32(cfg.box_L))
    d = pts[:, None, :] - pos[None, :, :3].astype(np.float64)
    d -= Lb * np.round(d / Lb)
    r = np.sqrt((d ** 2).sum(axis=2)).min(axis=1)
    R = 0.5 * (1.0 + cfg.sigma_d)
    free, border = int((r >= R).sum()), int((np.abs(r - R) < 1e-6).sum())
    assert abs(got - free) <= border, (got, free, border)
    assert 0.6 * n < got < 0.95 * n
