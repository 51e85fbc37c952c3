"""Physics pins for the oracle's move rule (CPU only).  SURVEY 8(c) checks 1-5 / BASELINE.json north_star.

None of the expected values below comes from the oracle: they are closed forms (Eq. 8/15 acceptance
exp(-n_R dV), the Asakura-Oosawa overlap volume), brute-force explicit-depletant sampling written here in
numpy fp64, or structural invariants of the checkerboard.
"""
import math
import os

import numpy as np
import pytest

import oracle
import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(key):
    with open(os.path.join(GOLD, "paper_values.txt")) as f:
        for line in f:
            if line.startswith(key + " "):
                return float(line.split()[1])
    raise KeyError(key)


def lens(R, r):
    """Overlap volume of two spheres of radius R at centre distance r (Asakura-Oosawa, ref. 17)."""
    return math.pi * (4 * R + r) * (2 * R - r) ** 2 / 12.0 if r < 2 * R else 0.0


def iso_accept(n_R, R, d):
    """north_star check 2: exp(-n_R (V_s - pi(4R+d)(2R-d)^2/12)); from Eq. 8 (L105) / Eq. 15 (L150)."""
    return math.exp(-n_R * (4 * math.pi * R ** 3 / 3 - lens(R, d)))


def make_oracle(cfg, pos, quat=None, threads=1, d_max_cap=None):
    return oracle.Oracle(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max if d_max_cap is None else d_max_cap,
                         pos, quat, cfg.disk_a, cfg.disk_s, threads=threads)


def sphere_oracle(pos, L, sigma_d, d_max_cap, threads=1):
    p4 = np.zeros((len(pos), 4), np.float32)
    p4[:, :3] = pos
    return oracle.Oracle("sphere", 1.0, sigma_d, L, d_max_cap, p4, threads=threads)


# ------------------------------------------------------------------ check 2: isolated colloid
def test_golden_closed_form_values():
    """The closed form itself reproduces the numbers SURVEY 8(c) prints (guards the test's own formula)."""
    c1 = workloads.config("C1")
    assert abs(iso_accept(c1.n_R(), 0.6, 0.1) / _gold("iso_accept_C1_d0.1") - 1) < 5e-3
    c3 = workloads.config("C3")
    assert abs(iso_accept(c3.n_R(), 0.525, 0.001) / _gold("iso_accept_C3_d0.001") - 1) < 5e-3


@pytest.mark.parametrize("cfgname,d,ndraw", [("C1", 0.1, 400000), ("C1", 0.03, 60000), ("C3", 0.001, 60000)])
def test_isolated_colloid_fixed_displacement(cfgname, d, ndraw):
    cfg = workloads.config(cfgname)
    L = 8.0
    o = sphere_oracle([[4.0, 4.0, 4.0]], L, cfg.sigma_d, 0.1)
    o.build_cells(1, 0)
    rng = np.random.default_rng(5)
    u = rng.standard_normal(3)
    u /= np.linalg.norm(u)
    new = np.float32(4.0) + (d * u).astype(np.float32)
    d_eff = float(np.linalg.norm(new.astype(np.float64) - 4.0))
    acc = 0
    for k in range(ndraw):
        out = o.eval_move(1, k, 0, new, None, cfg.n_R())
        assert out in (1, 4)
        acc += out == 1
    R = 0.5 * (1.0 + cfg.sigma_d)
    p = iso_accept(cfg.n_R(), R, d_eff)
    assert abs(acc / ndraw - p) < 3.0 * math.sqrt(p * (1 - p) / ndraw) + 1e-9, (acc / ndraw, p)


def test_isolated_colloid_sweeps_binned_by_step_length():
    """north_star check 2 through the whole sweep path (selection, trial move, confinement, depletants):
    acceptance of translations of length d, boundary rejections excluded, vs the closed form, 3 sigma per bin.
    10^6 trials."""
    cfg = workloads.config("C1")
    L, n = 8.0, 1000000
    o = sphere_oracle([[1.0, 2.0, 3.0]], L, cfg.sigma_d, cfg.d_max)
    R = 0.5 * (1.0 + cfg.sigma_d)
    traj, outc = o.run(1, 0, n, cfg.n_R(), cfg.d_max, traj=True, outcomes=True)
    outc = outc[:, 0]
    assert set(np.unique(outc)) <= {1, 2, 4}
    # accepted steps: displacement from the trajectory (fp64 minimum image)
    prev = np.concatenate([[[1.0, 2.0, 3.0]], traj[:-1, 0, :3].astype(np.float64)])
    disp = traj[:, 0, :3].astype(np.float64) - prev
    disp -= L * np.round(disp / L)
    dlen = np.linalg.norm(disp, axis=1)
    assert np.all(dlen[outc != 1] == 0.0)                    # rejected moves leave the pose untouched
    assert np.all(np.abs(disp) <= cfg.d_max + 1e-6)
    # expected number of accepted steps per length bin: N_nb * E[1{d in bin} * P_acc(d) | not boundary].
    # Delta uniform in the cube; P(not boundary | Delta) = prod_a (1 - |Delta_a|/w) since the grid shift is
    # uniform (L180).  Quadrature by fp64 Monte Carlo over Delta (2e7 points, error << statistical error).
    rng = np.random.default_rng(0)
    m = 20000000
    D = (rng.random((m, 3)) * 2 - 1) * cfg.d_max
    wgt = np.prod(1 - np.abs(D) / o.w, axis=1)
    dl = np.linalg.norm(D, axis=1)
    pacc = np.exp(-cfg.n_R() * (4 * math.pi * R ** 3 / 3 - math.pi * (4 * R + dl) * (2 * R - dl) ** 2 / 12))
    n_nb = int((outc != 2).sum())
    p_nb = wgt.mean()
    assert abs(n_nb / n - p_nb) < 4 * math.sqrt(p_nb * (1 - p_nb) / n)      # confinement statistics
    edges = np.array([0.0, 0.01, 0.02, 0.03, 0.04, 0.05, 0.065, 0.08, 0.1, 0.18])
    for lo, hi in zip(edges[:-1], edges[1:]):
        sel = (dl >= lo) & (dl < hi)
        p_bin = (wgt * pacc * sel).mean() / p_nb                # P(accepted and d in bin | not boundary)
        got = int(((outc == 1) & (dlen >= lo) & (dlen < hi)).sum())
        exp = n_nb * p_bin
        assert abs(got - exp) < 3.0 * math.sqrt(exp) + 3, (lo, hi, got, exp)
    # total acceptance
    p_tot = (wgt * pacc).mean() / p_nb
    assert abs((outc == 1).sum() / n_nb - p_tot) < 3.0 * math.sqrt(p_tot / n_nb)


# ------------------------------------------------------------------ check 3: two spheres, AO potential
def _pair_ratio(n_R, sigma_d, r_a, r_b, ndraw, n_trial=0):
    """Acceptance of the fixed move r_a -> r_b and of its reverse, sphere 0 moved along x, sphere 1 fixed."""
    L = 8.0
    acc = []
    for (r0, r1) in ((r_a, r_b), (r_b, r_a)):
        o = sphere_oracle([[3.0 + (2.0 - r0), 4.0, 4.0], [5.0, 4.0, 4.0]], L, sigma_d, 0.1)
        o.build_cells(1, 0)
        new = np.array([3.0 + (2.0 - r1), 4.0, 4.0], np.float32)
        a = 0
        for k in range(ndraw):
            out = o.eval_move(7, k, 0, new, None, n_R, n_trial)
            assert out in (1, 4, 5)
            a += out == 1
        # effective separations after fp32 rounding
        acc.append(a)
    return acc


def test_two_sphere_fixed_move_ratio_plain():
    """acc(r->r')/acc(r'->r) = exp(n_R [V_ov(r') - V_ov(r)])  (detailed balance w.r.t. exp(-beta U_AO))."""
    cfg = workloads.config("C1")
    n_R, R, nd = cfg.n_R(), 0.6, 400000
    ra, rb = 1.05, 1.12
    fwd, rev = _pair_ratio(n_R, cfg.sigma_d, ra, rb, nd)
    want = math.exp(n_R * (lens(R, rb) - lens(R, ra)))
    got = fwd / rev
    rel = math.sqrt(1 / fwd + 1 / rev)
    assert abs(got / want - 1) < 3.0 * rel, (got, want, fwd, rev)
    # absolute level too: acceptance of r->r' is exp(-n_R [V_s - lens(d) - (V_ov(r) - tripleoverlap...)])
    # (not closed-form in general) -> only the isolated limit is checked in check 2.


def test_two_sphere_separation_histogram():
    """north_star check 3: P(r) ~ r^2 exp(-beta U_AO(r)) for r < L/2 in a periodic box; well vs outside."""
    sigma_d, d_max, n_R = 0.4, 0.2, 9.0
    L = 4 * (1.0 + sigma_d + 2 * d_max) + 0.01
    R = 0.5 * (1 + sigma_d)
    o = sphere_oracle([[1.0, 1.0, 1.0], [3.5, 3.0, 2.0]], L, sigma_d, d_max)
    n = 1500000
    traj, _ = o.run(3, 0, n, n_R, d_max, traj=True)
    d = traj[:, 0, :3].astype(np.float64) - traj[:, 1, :3].astype(np.float64)
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=1)
    assert r.min() >= 1.0 - 1e-6                                  # check 1
    r_hi = 2.4
    assert r_hi < L / 2
    in_well = (r < 1 + sigma_d)
    in_ref = (r >= 1 + sigma_d) & (r < r_hi)
    rr = np.linspace(1.0, 1 + sigma_d, 20001)
    boltz = rr ** 2 * np.exp(n_R * np.array([lens(R, x) for x in rr]))
    w_well = float(((boltz[1:] + boltz[:-1]) * 0.5 * np.diff(rr)).sum())
    w_ref = (r_hi ** 3 - (1 + sigma_d) ** 3) / 3.0
    want = w_well / w_ref
    # blocked estimate of the ratio
    nb = 30
    ratios = [in_well[k * (n // nb):(k + 1) * (n // nb)].sum() / max(1, in_ref[k * (n // nb):(k + 1) * (n // nb)].sum())
              for k in range(nb)]
    got = in_well.sum() / in_ref.sum()
    err = np.std(ratios, ddof=1) / math.sqrt(nb)
    assert abs(got - want) < 4 * err + 0.01 * want, (got, want, err)
    assert err < 0.2 * want      # modest resolving power (slow diffusion); the sharp AO pin is the ratio test above
    # the well is really populated above the ideal r^2 law (attraction present)
    ideal = ((1 + sigma_d) ** 3 - 1) / 3.0 / w_ref
    assert got > ideal + 3 * err


# ------------------------------------------------------------------ check 4: explicit depletants, many-body
def _explicit_acceptance(centres, quats, gauge_dist, i, new_c, new_q, n_R, rd, R_circ, nbath, rng):
    """Sec. III.B literally (L64-68): a grand-canonical ideal-gas bath of depletants in the free volume of
    the OLD configuration (Poisson number, uniform positions, those overlapping a colloid removed); the move
    is accepted iff no bath particle overlaps the NEW pose.  Only bath particles inside a cube around the
    new pose can matter.  gauge_dist(x, c, q) = distance from x to the colloid (fp64)."""
    half = R_circ + rd + 1e-9
    V = (2 * half) ** 3
    acc = 0
    for _ in range(nbath):
        m = rng.poisson(n_R * V)
        x = new_c + (rng.random((m, 3)) * 2 - 1) * half
        free = np.ones(m, bool)
        for j in range(len(centres)):
            free &= gauge_dist(x, centres[j], quats[j]) >= rd
        hit = free & (gauge_dist(x, new_c, new_q) < rd)
        acc += not hit.any()
    return acc


def _sphere_dist(x, c, q):
    return np.linalg.norm(x - c, axis=1) - 0.5


def test_explicit_bath_agrees_with_implicit_many_body_spheres():
    """4 colloids in a tight cluster: acceptance of a fixed move of colloid 0, implicit oracle vs explicit
    depletant bath.  The three neighbours' exclusion zones overlap each other and the moved one (non-pairwise
    free volume), which exercises 'depletants that overlap ... surrounding colloids are not considered' (L72)."""
    sigma_d, n_R = 0.4, 12.0
    L = 8.0
    c = np.array([[4.0, 4.0, 4.0], [5.15, 4.1, 4.0], [4.2, 5.18, 4.1], [4.1, 4.3, 5.2]])
    o = sphere_oracle(c, L, sigma_d, 0.2)
    assert o.count_overlaps() == 0
    o.build_cells(1, 0)
    new = np.array([4.06, 4.05, 4.04], np.float32)
    nd = 150000
    outs = np.array([o.eval_move(11, k, 0, new, None, n_R) for k in range(nd)])
    assert set(np.unique(outs)) <= {1, 4}
    acc_i = int((outs == 1).sum())
    rng = np.random.default_rng(42)
    nb = 150000
    acc_e = _explicit_acceptance(c, [None] * 4, _sphere_dist, 0, new.astype(np.float64), None, n_R, 0.5 * sigma_d, 0.5,
                                 nb, rng)
    pi, pe = acc_i / nd, acc_e / nb
    assert 0.02 < pe < 0.98
    assert abs(pi - pe) < 3.5 * math.sqrt(pi * (1 - pi) / nd + pe * (1 - pe) / nb), (pi, pe)
    # and it differs measurably from the isolated-colloid value: the neighbours matter
    p_iso = iso_accept(n_R, 0.7, float(np.linalg.norm(new.astype(np.float64) - 4.0)))
    assert abs(pe - p_iso) > 10 * math.sqrt(pe * (1 - pe) / nb)


def _spherodisk_dist(a, s):
    from scipy.spatial.transform import Rotation

    def f(x, c, q):
        M = Rotation.from_quat(np.r_[q[1:], q[0]]).as_matrix().T
        b = (x - c) @ M.T
        rho = np.hypot(b[:, 0], b[:, 1])
        return np.hypot(np.maximum(rho - a, 0.0), b[:, 2]) - s
    return f


def test_explicit_bath_agrees_with_implicit_spherodisk_rotation():
    """Same comparison for an anisotropic shape and a combined translation + rotation of colloid 0."""
    cfg = workloads.config("C5")
    n_R = 40.0
    L = 8.0
    rng = np.random.default_rng(9)
    c = np.array([[4.0, 4.0, 4.0], [4.0, 4.1, 4.32], [4.75, 4.0, 3.9]])
    q = np.array([[1, 0, 0, 0], [1, 0, 0, 0], [0.70710678, 0, 0.70710678, 0]], np.float64)
    p4 = np.zeros((3, 4), np.float32)
    p4[:, :3] = c
    o = oracle.Oracle("spherodisk", 1.0, cfg.sigma_d, L, 0.1, p4, q.astype(np.float32), cfg.disk_a, cfg.disk_s, threads=1)
    assert o.count_overlaps() == 0
    o.build_cells(1, 0)
    new_c = np.array([4.03, 3.98, 4.0], np.float32)
    ang = 0.25
    new_q = np.array([math.cos(ang / 2), math.sin(ang / 2), 0, 0], np.float32)      # tilt about x
    nd = 100000
    outs = np.array([o.eval_move(13, k, 0, new_c, new_q, n_R) for k in range(nd)])
    assert set(np.unique(outs)) <= {1, 4}
    pi = (outs == 1).mean()
    dist = _spherodisk_dist(cfg.disk_a, cfg.disk_s)
    nb = 100000
    acc_e = _explicit_acceptance(c, q, dist, 0, new_c.astype(np.float64), new_q.astype(np.float64), n_R,
                                 0.5 * cfg.sigma_d, 0.5, nb, rng)
    pe = acc_e / nb
    assert 0.02 < pe < 0.98
    assert abs(pi - pe) < 3.5 * math.sqrt(pi * (1 - pi) / nd + pe * (1 - pe) / nb), (pi, pe)


# ------------------------------------------------------------------ configurational bias (Eq. 16, G1-G3)
def test_cb_isolated_colloid_always_accepts_with_many_trials():
    """G1 special case: no other colloids => every Eq.-16 factor is exactly 1, so the move is accepted
    whenever each rejecting depletant found at least one valid reinsertion (n_trial large makes that sure).
    The printed form of Eq. 16 (without the prime) would give random factors (N_i+1)/(N'_i+1) instead."""
    cfg = workloads.config("C1")
    o = sphere_oracle([[1.0, 2.0, 3.0]], 8.0, cfg.sigma_d, cfg.d_max)
    n = 1500
    _, outc = o.run(5, 0, n, cfg.n_R(), cfg.d_max, n_trial=3000, outcomes=True)
    outc = outc[:, 0]
    nb = (outc != 2).sum()
    assert (outc == 1).sum() >= 0.993 * nb
    # the plain rule on the same moves rejects nearly all of them
    o2 = sphere_oracle([[1.0, 2.0, 3.0]], 8.0, cfg.sigma_d, cfg.d_max)
    _, outp = o2.run(5, 0, n, cfg.n_R(), cfg.d_max, n_trial=0, outcomes=True)
    assert (outp[:, 0] == 1).sum() < 0.2 * nb


def _pair_counts(L_, ra, rb, nd, n_trial, n_R, sigma_d, seed=7):
    """Accepted counts of the fixed move r_a -> r_b and of its reverse (sphere 0 moved along x towards / away from the
    fixed sphere 1), nd independent evaluations each, through the batched export oracle_eval_moves of library L_."""
    import ctypes as C
    from oracle import binding
    acc = []
    L_.oracle_set_threads(os.cpu_count() or 1)     # draws are independent streams: the thread count changes no bit
    for r0, r1 in ((ra, rb), (rb, ra)):
        p4 = np.zeros((2, 4), np.float32)
        p4[0, :3] = [3.0 + (2.0 - r0), 4.0, 4.0]
        p4[1, :3] = [5.0, 4.0, 4.0]
        par = binding.make_params("sphere", 1.0, sigma_d, 8.0, 0.1)
        h = L_.oracle_create(C.byref(par), 2, p4.ctypes.data_as(C.c_void_p), None)
        assert h
        assert L_.oracle_build_cells(h, 1, 0) == 0
        new = np.array([3.0 + (2.0 - r1), 4.0, 4.0], np.float32)
        out = np.empty(nd, np.uint8)
        rc = L_.oracle_eval_moves(h, seed, 0, nd, 0, new.ctypes.data_as(C.c_void_p), None, float(n_R), n_trial,
                                  out.ctypes.data_as(C.c_void_p))
        assert rc == 0
        assert set(np.unique(out)) <= ({1, 4} if n_trial == 0 else {1, 5})
        acc.append(int((out == 1).sum()))
        L_.oracle_destroy(h)
    L_.oracle_set_threads(1)
    return acc


def _ratio_error(L_, ra, rb, nd, n_trial, n_R, sigma_d):
    """(measured fwd/rev acceptance ratio) / exp(n_R [V_ov(r_b) - V_ov(r_a)]) - 1, and its 1-sigma statistical error.
    The target is detailed balance w.r.t. the Asakura-Oosawa weight (ref. 17 L276; Eq. 8 L105 / Eq. 15)."""
    R = 0.5 * (1.0 + sigma_d)
    fwd, rev = _pair_counts(L_, ra, rb, nd, n_trial, n_R, sigma_d)
    want = math.exp(n_R * (lens(R, rb) - lens(R, ra)))
    return (fwd / max(rev, 1)) / want - 1.0, math.sqrt(1.0 / max(fwd, 1) + 1.0 / max(rev, 1)), fwd, rev


# Geometry of the Eq. 16 pins: C1's depletants (sigma_d = 0.2, n_R = 47.7), sphere 0 moved from separation 1.02 to 1.10
# from a fixed neighbour.  The old-only crescent faces the neighbour and is partly covered by its exclusion sphere,
# the new-only crescent faces away and is free: the forward and reverse success fractions of Eq. 16 differ (s != s').
_CB_GEOM = dict(ra=1.02, rb=1.10, sigma_d=0.2)
_CB_DRAWS = 4000000


@pytest.mark.parametrize("n_trial", [1, 4, 10])
def test_cb_two_sphere_fixed_move_ratio(n_trial):
    """R-G1 / R-G2 / R-G3 pin.  CB samples the same AO weight as the plain rule: acc(r->r')/acc(r'->r) =
    exp(n_R [V_ov(r') - V_ov(r)]), 4e6 draws per direction, tolerance 3 sigma + 1 % (the adopted form
    leaves < 1 %, the printed prime-less Eq. 16 is 2-14 % off).  test_cb_ratio_pin_rejects_wrong_readings shows that
    this very measurement fails for the printed form, for swapped forward/reverse roles and for a skipped 0/0 rule."""
    n_R = workloads.config("C1").n_R()
    err, sig, fwd, rev = _ratio_error(oracle.lib(), nd=_CB_DRAWS, n_trial=n_trial, n_R=n_R, **_CB_GEOM)
    assert abs(err) < 3.0 * sig + 0.01, (n_trial, err, sig, fwd, rev)


def _mutant_library(tmp_path, name, old, new):
    from conftest import build_mutant_oracle
    return build_mutant_oracle(tmp_path, name, old, new)


_EQ16 = "const float wk = (float)(Npins * (Npi + 1u)) / (float)((Nins + 1u) * Ni);"
_MUTANTS = {
    # the formula as PAPER.md L172 prints it: (N_i + 1) where the adopted reading R-G1 has (N'_i + 1)
    "printed_eq16": (_EQ16, "const float wk = (float)(Npins * (Ni + 1u)) / (float)((Nins + 1u) * Ni);", (4, 10)),
    # R-G2 with the roles of the forward (old centre) and reverse (new centre) counts exchanged
    "roles_swapped": (_EQ16, "const float wk = (float)(Nins * (Ni + 1u)) / (float)((Npins + 1u) * Npi);", (4, 10)),
    # R-G3 dropped: a rejecting depletant without a valid forward reinsertion is skipped instead of rejecting
    "zero_rule_skipped": ("if (Npins == 0) return OUT_CB;", "if (Npins == 0) continue;", (1, 4)),
}


@pytest.mark.parametrize("name", sorted(_MUTANTS))
def test_cb_ratio_pin_rejects_wrong_readings(tmp_path, name):
    """The pin's resolving power, shown on throw-away builds of the oracle with ONE reading changed: each must FAIL
    the tolerance of test_cb_two_sphere_fixed_move_ratio by at least half again (measured: printed form +3 % at n_trial = 4,
    +16 % at 10; swapped roles +11 % / +56 %; skipped 0/0 rule > +100 %), while the adopted form sits at |err| < 0.3 %."""
    old, new, trials = _MUTANTS[name]
    L_ = _mutant_library(tmp_path, name, old, new)
    n_R = workloads.config("C1").n_R()
    for n_trial in trials:
        err, sig, fwd, rev = _ratio_error(L_, nd=_CB_DRAWS, n_trial=n_trial, n_R=n_R, **_CB_GEOM)
        assert abs(err) > 1.5 * (3.0 * sig + 0.01), (name, n_trial, err, sig, fwd, rev)


def test_cb_zero_forward_weight_rule_thin_crescent():
    """R-G3 on its own: a short step (d = 0.01, crescents 1.2 % of the insertion sphere) with n_trial = 1 makes
    N'_ins = 0 the common case, so nearly every move with a rejecting depletant ends in outcome 5 through the 0/0
    rule alone -- CB accepts only slightly more often than the plain rule -- and the forward/reverse ratio still
    obeys detailed balance (it would not if the rule were anything but 'reject': see the mutant above)."""
    n_R = workloads.config("C1").n_R()
    g = dict(ra=1.05, rb=1.06, sigma_d=0.2)
    nd = 2000000
    L_ = oracle.lib()
    err, sig, fwd, rev = _ratio_error(L_, nd=nd, n_trial=1, n_R=n_R, **g)
    assert abs(err) < 3.0 * sig + 0.005, (err, sig)
    pf, pr = _pair_counts(L_, g["ra"], g["rb"], nd, 0, n_R, g["sigma_d"])
    # plain acceptance = P(no rejecting depletant); CB adds the moves whose (few) rejecting depletants all found a
    # valid free reinsertion in ONE try: at most a few per cent of the rejected ones
    for cb, plain in ((fwd, pf), (rev, pr)):
        assert plain < cb < plain + 0.06 * (nd - plain), (cb, plain)
    R = 0.6
    assert abs((pf / pr) / math.exp(n_R * (lens(R, g["rb"]) - lens(R, g["ra"]))) - 1) < 3.0 * math.sqrt(1 / pf + 1 / pr)


def test_cb_zero_trials_equals_plain_and_zero_density_is_hard_mc():
    cfg = workloads.config("C1")
    pos, _ = workloads.generate(cfg)
    a, b = make_oracle(cfg, pos), make_oracle(cfg, pos)
    a.run(1, 0, 20, 0.0, cfg.d_max, n_trial=0)
    b.run(1, 0, 20, 0.0, cfg.d_max, n_trial=4)
    assert np.array_equal(a.pos, b.pos)               # S23: no depletants => accept unless hard overlap
    ca = a.counters()
    assert ca["rej_depletant"] == 0 and ca["dep_drawn"] == 0 and ca["accept_trans"] > 0


# ------------------------------------------------------------------ check 1 + structural invariants
@pytest.mark.parametrize("name,N,sweeps", [("C1", None, 100), ("C2", 2048, 30), ("C3", 4096, 10), ("C4", 512, 40),
                                            ("C5", 512, 40), ("C6", 512, 40), ("C7", 4096, 15)])
def test_zero_overlaps_and_bookkeeping(name, N, sweeps):
    cfg = workloads.config(name, N)
    pos, quat = workloads.generate(cfg)
    o = make_oracle(cfg, pos, quat)
    assert o.count_overlaps(both_ways=False) == 0
    tried_total = 0
    for s in range(sweeps):
        before_p = o.pos.copy()
        before_q = None if o.quat is None else o.quat.copy()
        o.build_cells(cfg.seed, s)
        cs, cp, shift = o.cells()
        assert cs[-1] == cfg.N and np.array_equal(np.sort(cp), np.arange(cfg.N))
        nonempty = int((np.diff(cs.astype(np.int64)) > 0).sum())
        o.sweep(cfg.seed, s, cfg.n_R(), cfg.d_max, cfg.a_max, cfg.n_trial)
        out = o.outcomes()
        tp, tq = o.trial_poses()
        tried = out != 0
        assert tried.sum() == nonempty                        # S12: one trial per non-empty active cell
        tried_total += int(tried.sum())
        acc = out == 1
        assert np.array_equal(o.pos[~acc], before_p[~acc])    # rejected / untried: untouched
        assert np.array_equal(o.pos[acc, :3], tp[acc, :3])    # accepted: the trial pose, bit for bit
        if before_q is not None:
            assert np.array_equal(o.quat[~acc], before_q[~acc])
            assert np.array_equal(o.quat[acc], tq[acc])
            assert np.allclose(np.linalg.norm(o.quat.astype(np.float64), axis=1), 1.0, atol=1e-6)
        assert o.pos[:, :3].min() >= 0.0 and o.pos[:, :3].max() < np.float32(cfg.box_L)
        # confinement (L180): every particle is still in the cell it was binned into
        t = o.pos[:, :3] - shift[None, :]
        t = np.where(t < 0, t + np.float32(cfg.box_L), t).astype(np.float32)
        ci = np.minimum((t / np.float32(o.w)).astype(np.int64), o.n_c - 1)
        lin = (ci[:, 2] * o.n_c + ci[:, 1]) * o.n_c + ci[:, 0]
        owner = np.repeat(np.arange(o.n_c ** 3), np.diff(cs.astype(np.int64)))
        assert np.array_equal(lin[cp], owner)
    assert o.count_overlaps(both_ways=True) == 0              # check 1 (Eq. 5)
    c = o.counters()
    assert c["trials_trans"] + c["trials_rot"] == tried_total
    rej = c["rej_boundary"] + c["rej_hard"] + c["rej_depletant"] + c["rej_cb"]
    assert c["accept_trans"] + c["accept_rot"] + rej == tried_total
    assert c["dep_needed"] <= c["dep_drawn"]
    if cfg.a_max > 0:
        assert abs(c["trials_rot"] / tried_total - 0.5) < 5 / math.sqrt(tried_total)      # S7: 50/50
    else:
        assert c["trials_rot"] == 0
    if cfg.n_trial == 0:
        assert c["rej_cb"] == 0 and c["cb_reinsertions"] == 0
    else:
        assert c["rej_depletant"] == 0


def test_parallel_order_equals_sequential_order():
    """Independence of same-colour cells (L180): the OpenMP loop over active cells gives the same bits."""
    cfg = workloads.config("C3", 8192)
    pos, _ = workloads.generate(cfg)
    a, b = make_oracle(cfg, pos, threads=1), make_oracle(cfg, pos, threads=4)
    oracle.lib().oracle_set_threads(1)
    a.run(1, 0, 6, cfg.n_R(), cfg.d_max)
    oracle.lib().oracle_set_threads(4)
    b.run(1, 0, 6, cfg.n_R(), cfg.d_max)
    oracle.lib().oracle_set_threads(1)
    assert np.array_equal(a.pos, b.pos)
    assert a.counters() == b.counters()


def test_grid_shift_varies():
    """L180: 'grid lines are randomly shifted' (once per sweep, S11): uniform in [0, w) on every axis, axes uncorrelated."""
    cfg = workloads.config("C1")
    pos, _ = workloads.generate(cfg)
    o = make_oracle(cfg, pos)
    shifts = []
    for s in range(200):
        o.build_cells(1, s)
        shifts.append(o.cells()[2].copy())
        o.sweep(1, s, 0.0, 0.0)
    sh = np.array(shifts, np.float64) / o.w
    assert sh.min() > 0 and sh.max() < 1
    assert np.all(np.abs(sh.mean(0) - 0.5) < 4 * math.sqrt(1 / 12 / 200))
    assert np.all(np.abs(np.corrcoef(sh.T)[np.triu_indices(3, 1)]) < 0.3)


# ------------------------------------------------------------------ colour order of a sweep (R-2, L180)
_N_ORDERS = 100000


def _colour_order_chi2(L_, n=_N_ORDERS):
    """chi^2 of (position, colour) counts against n/8 (49 degrees of freedom: rows and columns of a permutation sum to
    n) and, for each of the 7 neighbouring position pairs, of the ordered colour pairs against n/56 (55 d.o.f.)."""
    out = np.empty(8, np.uint32)
    orders = np.empty((n, 8), np.int64)
    for k in range(n):
        L_.oracle_colour_order(11 + k // 1000, k % 1000, out.ctypes.data)
        orders[k] = out
    assert np.array_equal(np.sort(orders, axis=1), np.tile(np.arange(8), (n, 1))), "not a permutation of 0..7"
    pos_counts = np.zeros((8, 8))
    for p in range(8):
        pos_counts[p] = np.bincount(orders[:, p], minlength=8)
    chi_pos = float(((pos_counts - n / 8.0) ** 2 / (n / 8.0)).sum())
    chi_pairs = []
    for p in range(7):
        c = np.bincount(orders[:, p] * 8 + orders[:, p + 1], minlength=64).reshape(8, 8).astype(np.float64)
        assert np.all(np.diag(c) == 0)
        off = c[~np.eye(8, dtype=bool)]
        chi_pairs.append(float(((off - n / 56.0) ** 2 / (n / 56.0)).sum()))
    return chi_pos, chi_pairs


def _colour_order_is_uniform(chi_pos, chi_pairs):
    from scipy.stats import chi2
    return chi_pos < chi2.ppf(1 - 1e-3, 49) and max(chi_pairs) < chi2.ppf(1 - 1e-3 / 7, 55)


def test_colour_order_is_a_uniform_random_permutation():
    """R-2 pin ("the checkerboard coloring is permuted randomly"): over 10^5 sweeps every colour takes every
    one of the 8 places with frequency 1/8 and every ordered pair of colours is equally likely in neighbouring places
    (chi^2, alpha = 10^-3 overall each) -- what a uniform random permutation means, independent of how it is drawn."""
    chi_pos, chi_pairs = _colour_order_chi2(oracle.lib())
    assert _colour_order_is_uniform(chi_pos, chi_pairs), (chi_pos, chi_pairs)
    assert len({tuple(oracle.binding.colour_order(3, s)) for s in range(50)}) > 40


_SWAP = "    const uint32_t t = perm[i]; perm[i] = perm[r]; perm[r] = t;"


@pytest.mark.parametrize("name,old,new", [
    ("constant_order", _SWAP, "    (void)r;"),                                                # never permuted
    ("range_off_by_one", "mulhi32(wds[j], (uint32_t)i + 1u)", "mulhi32(wds[j], (uint32_t)i)"),  # r in 0..i-1: cyclic permutations only
])
def test_colour_order_pin_rejects_wrong_shuffles(tmp_path, name, old, new):
    L_ = _mutant_library(tmp_path, name, old, new)
    chi_pos, chi_pairs = _colour_order_chi2(L_, 20000)
    assert not _colour_order_is_uniform(chi_pos, chi_pairs), (name, chi_pos, chi_pairs)


# ------------------------------------------------------------------ which occupant of an active cell is tried (a3, S12)
def _occupant_pick_histogram(L_, sweeps=1500):
    """Cells two depletant-widened diameters wide hold several spheres (q = 1: w ~ 2 sigma_c).  n_R = 0 and a tiny step,
    so a sweep only records WHO was tried (outcome code != 0).  hist[k][s] = how often the s-th occupant (ascending
    particle id) of a k-occupied cell was the one tried; also checks that every non-empty cell tries exactly one."""
    import ctypes as C
    import dataclasses
    from oracle import binding
    cfg = dataclasses.replace(workloads.config("C1"), N=520, phi_c=0.15, q=1.0, d_max=0.01)
    pos, _ = workloads.generate(cfg)
    pos = np.ascontiguousarray(pos, np.float32).copy()
    par = binding.make_params("sphere", cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max)
    h = L_.oracle_create(C.byref(par), cfg.N, pos.ctypes.data, None)
    assert h
    nc, w = C.c_int32(), C.c_float()
    L_.oracle_grid(h, C.byref(nc), C.byref(w))
    ncell = nc.value ** 3
    cs, cp, sh = np.empty(ncell + 1, np.uint32), np.empty(cfg.N, np.uint32), np.empty(3, np.float32)
    out = np.empty(cfg.N, np.uint8)
    hist = np.zeros((8, 8), np.int64)
    for s in range(sweeps):
        assert L_.oracle_build_cells(h, 5, s) == 0
        L_.oracle_cells(h, cs.ctypes.data, cp.ctypes.data, sh.ctypes.data)
        assert L_.oracle_sweep(h, 5, s, 0.0, cfg.d_max, 0.0, 0) == 0
        L_.oracle_outcomes(h, out.ctypes.data)
        counts = np.diff(cs.astype(np.int64))
        cell_of_entry = np.repeat(np.arange(ncell), counts)
        slot = np.arange(cfg.N) - cs[cell_of_entry].astype(np.int64)
        tried = out[cp] != 0
        per_cell = np.bincount(cell_of_entry, weights=tried, minlength=ncell)
        assert np.array_equal(per_cell, (counts > 0).astype(np.float64)), "a non-empty cell tries exactly one occupant"
        k = np.minimum(counts[cell_of_entry], 7)
        np.add.at(hist, (k[tried], np.minimum(slot[tried], 7)), 1)
    L_.oracle_destroy(h)
    return hist


def _pick_is_uniform(hist):
    ok, seen = True, 0
    for k in (2, 3, 4):
        n = int(hist[k].sum())
        if n < 5000:
            continue
        seen += 1
        f = hist[k, :k] / n
        ok = ok and bool(np.all(np.abs(f - 1.0 / k) < 4.0 * math.sqrt((1.0 / k) * (1 - 1.0 / k) / n)))
    assert seen == 3, hist
    return ok


def test_occupant_of_an_active_cell_is_picked_uniformly():
    """a3 / S12 pin (north_star "in each active cell one colloid gets a trial"): in cells with k = 2, 3, 4
    occupants each occupant is the one tried with frequency 1/k within 4 sigma, over ~3 x 10^5 cell visits."""
    hist = _occupant_pick_histogram(oracle.lib())
    assert hist[1, 0] == hist[1].sum() and hist[2:5].sum() > 10 ** 5
    assert _pick_is_uniform(hist), hist[:5, :5]


def test_occupant_pick_pin_rejects_always_the_first(tmp_path):
    L_ = _mutant_library(tmp_path, "first_occupant", "c.cell_pid[b + mulhi32(rs.v[0], nocc)]", "c.cell_pid[b]")
    assert not _pick_is_uniform(_occupant_pick_histogram(L_, 300) * 5)


def test_self_axis_rotation_always_accepted():
    """S6 pin: rotating an isolated half-ball / spherodisk about its own symmetry axis changes no volume."""
    for shape, extra in (("halfball", {}), ("spherodisk", dict(disk_a=0.4, disk_s=0.1))):
        p4 = np.array([[4.0, 4.0, 4.0, 0.0]], np.float32)
        q0 = np.array([[math.cos(0.3), 0.0, math.sin(0.3), 0.0]], np.float32)   # tilt about y
        o = oracle.Oracle(shape, 1.0, 0.2, 8.0, 0.1, p4, q0, threads=1, **extra)
        o.build_cells(1, 0)
        # spin about the body axis: q' = q0 * (cos a, 0, 0, sin a)  (body-frame rotation about z)
        a = 0.4
        w0, x0, y0, z0 = [float(t) for t in q0[0]]
        w1, x1, y1, z1 = math.cos(a), 0.0, 0.0, math.sin(a)
        qn = np.array([w0 * w1 - x0 * x1 - y0 * y1 - z0 * z1, w0 * x1 + x0 * w1 + y0 * z1 - z0 * y1,
                       w0 * y1 - x0 * z1 + y0 * w1 + z0 * x1, w0 * z1 + x0 * y1 - y0 * x1 + z0 * w1], np.float32)
        outs = [o.eval_move(1, k, 0, p4[0, :3], qn, 60.0) for k in range(3000)]
        assert sum(x == 1 for x in outs) >= 2990              # fp32 axis noise may flip a boundary sample
        # a tilt by the same angle about a perpendicular axis is mostly rejected
        qt = np.array([math.cos(0.3 + a), 0.0, math.sin(0.3 + a), 0.0], np.float32)
        outs = [o.eval_move(1, k, 0, p4[0, :3], qt, 60.0) for k in range(3000)]
        assert sum(x == 1 for x in outs) < 1500
