"""GPU parity: the CUDA path (through the C-ABI, include/hpmc.h) against the CPU oracle, element by element,
on the same seeded inputs.  Bar (BASELINE.json north_star): per-move outcome codes and fp32 poses BIT-EXACT
after every sweep; integer counters that both sides define (everything except dep_evaluated / philox_blocks,
which describe each implementation's own work) equal.

The default runs the configs' full lengths (min(1000, sweeps) per north_star: C1 100, C2 4 x 1000, C3 200 at
1,048,576 spheres, C4 500, C5 500 sweeps; about 80 s on a B200 box with 16 host cores for the oracle).
HPMC_PARITY_SHORT=1 shortens them for local iterations.
"""
import os

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

FULL = os.environ.get("HPMC_PARITY_SHORT", "0") != "1"
SHARED_COUNTERS = ("trials_trans", "accept_trans", "trials_rot", "accept_rot", "rej_boundary", "rej_hard",
                   "rej_depletant", "rej_cb", "dep_drawn", "dep_needed", "cb_reinsertions")


def _mk(cfg, pos, quat, threads=None):
    import torch
    import oracle
    import paper_1508_07077_b200 as hp
    o = oracle.Oracle(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, pos, quat, cfg.disk_a, cfg.disk_s,
                      threads=threads or os.cpu_count())
    dpos = torch.from_numpy(pos.copy()).cuda()
    dquat = None if quat is None else torch.from_numpy(quat.copy()).cuda()
    h = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, dpos, dquat, cfg.disk_a, cfg.disk_s)
    return o, h, dpos, dquat


def _bits(a):
    return np.ascontiguousarray(a).view(np.uint32)


def run_parity(cfg, pos, quat, sweeps, n_R, step0=0, check_cells_every=10, options=0):
    o, h, dpos, dquat = _mk(cfg, pos, quat)
    assert (o.n_c, np.float32(o.w)) == (h.n_c, np.float32(h.w))
    if options:
        o.set_flags(options)          # same bit values on both sides: 1 shell (R-N1), 2 Rosenbluth weight (R-N4)
        h.set_options(options)
    for s in range(step0, step0 + sweeps):
        o.build_cells(cfg.seed, s)
        h.build_cells(cfg.seed, s)
        if (s - step0) % check_cells_every == 0:
            cs, cp, sh = h.cells()
            ocs, ocp, osh = o.cells()
            assert np.array_equal(np.float32(sh), osh)
            assert np.array_equal(cs.cpu().numpy().view(np.uint32), ocs), "cell_start differs at sweep %d" % s
            assert np.array_equal(cp.cpu().numpy().view(np.uint32), ocp), "cell_pid differs at sweep %d" % s
        o.sweep(cfg.seed, s, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)
        h.sweep(cfg.seed, s, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)
        out = h.outcomes().cpu().numpy()
        oo = o.outcomes()
        if not np.array_equal(out, oo):
            bad = np.nonzero(out != oo)[0]
            raise AssertionError("outcome mask differs at sweep %d: %d particles, first %d gpu=%d oracle=%d"
                                 % (s, len(bad), bad[0], out[bad[0]], oo[bad[0]]))
        assert np.array_equal(_bits(dpos.cpu().numpy()), _bits(o.pos)), "positions differ at sweep %d" % s
        if quat is not None:
            assert np.array_equal(_bits(dquat.cpu().numpy()), _bits(o.quat)), "orientations differ at sweep %d" % s
    gc, oc = h.counters(), o.counters()
    for k in SHARED_COUNTERS:
        assert gc[k] == oc[k], (k, gc[k], oc[k])
    assert gc["dep_evaluated"] >= gc["dep_needed"]
    tried = gc["trials_trans"] + gc["trials_rot"]
    assert tried > 0
    h.close()
    return gc


def test_c1_spheres_256():
    cfg = workloads.config("C1")
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, 100, cfg.n_R(), check_cells_every=1)
    assert c["accept_trans"] > 0 and c["rej_depletant"] > 0 and c["rej_hard"] > 0 and c["rej_boundary"] > 0


def test_c2_spheres_65536_melted_density_sweep():
    """configs[1]: fcc lattice melted 1000 sweeps (by the ORACLE, n_R = 0), then the four reservoir densities."""
    import oracle
    cfg = workloads.config("C2")
    pos, _ = workloads.generate(cfg)
    melt = oracle.Oracle(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, pos, threads=os.cpu_count())
    melt.run(cfg.seed, 100000, 1000, 0.0, cfg.d_max)
    assert melt.counters()["rej_hard"] > 0
    pos = melt.pos.copy()
    n = 1000 if FULL else 25
    for phi in cfg.phi_d_r:
        run_parity(cfg, pos, None, n, cfg.n_R(phi))


def test_c3_spheres_reduced_many_sweeps():
    cfg = workloads.config("C3", 32768)
    pos, _ = workloads.generate(cfg)
    run_parity(cfg, pos, None, 200 if FULL else 40, cfg.n_R())


def test_c3_spheres_full_size():
    """configs[2] at full size (1,048,576 spheres, 1,404,928 cells), the launch configuration bench.py times."""
    cfg = workloads.config("C3")
    pos, _ = workloads.generate(cfg)
    c = run_parity(cfg, pos, None, 200 if FULL else 3, cfg.n_R(), check_cells_every=1)
    assert c["dep_drawn"] > 2000 * (c["trials_trans"] - c["rej_boundary"] - c["rej_hard"])


def test_spheres_beyond_one_wave_4m():
    """Four times configs[2]: 4,194,304 spheres at C3's densities (178^3 cells) need more CTAs than the device holds at
    once, so the sweep falls back to one launch per pass (3874 CTAs); two sweeps, bit for bit."""
    if not FULL:
        pytest.skip("long: 25 s of input placement")
    cfg = workloads.config("C3", 4194304)
    pos, _ = workloads.generate(cfg)
    c = run_parity(cfg, pos, None, 2, cfg.n_R(), check_cells_every=1)
    assert c["trials_trans"] > 3000000


def test_c3_small_steps_accepting_moves_use_all_depletants():
    """Accepted moves at C3's density must test all ~2.8k depletants: tiny steps make acceptance common."""
    import dataclasses
    cfg = dataclasses.replace(workloads.config("C3", 8192), d_max=0.0005)
    pos, _ = workloads.generate(cfg)
    # cell width is fixed by d_max_cap = cfg.d_max here
    c = run_parity(cfg, pos, None, 10, cfg.n_R())
    assert c["accept_trans"] > 0.1 * c["trials_trans"]


def test_c4_halfballs():
    cfg = workloads.config("C4")
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, 500 if FULL else 30, cfg.n_R())
    assert c["accept_rot"] > 0 and c["accept_trans"] > 0 and c["rej_hard"] > 0


def test_c5_spherodisks_configurational_bias():
    cfg = workloads.config("C5")
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, 500 if FULL else 30, cfg.n_R())
    assert c["cb_reinsertions"] > 0 and c["rej_cb"] > 0 and c["accept_rot"] > 0


@pytest.mark.parametrize("name,N,n_trial,sweeps", [("C5", None, 4, 120), ("C5", 4096, 40, 40), ("C1", None, 10, 100),
                                                   ("C4", 4096, 3, 40)])
def test_configurational_bias_through_the_item_queue_kernel(monkeypatch, name, N, n_trial, sweeps):
    """The CB stage of the item-queue kernel (HPMC_CB_KERNEL=queue: windows of depletant indices, reinsertion items,
    product folded in ascending k): C5 itself, a large n_trial (PAPER.md L228 recommends n_trial >~ 10), and CB on
    spheres and half-balls."""
    import dataclasses
    monkeypatch.setenv("HPMC_CB_KERNEL", "queue")
    cfg = dataclasses.replace(workloads.config(name, N), n_trial=n_trial)
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, sweeps if FULL else 15, cfg.n_R())
    assert c["cb_reinsertions"] > 0 and c["rej_cb"] > 0


@pytest.mark.parametrize("name,N,sweeps,d_max", [("C1", None, 100, None), ("C2", 16384, 60, None), ("C3", 65536, 30, None),
                                                 ("C3", 16384, 30, 0.0005), ("C4", 4096, 40, None)])
def test_shell_restricted_insertion_volume(name, N, sweeps, d_max):
    """HPMC_OPT_SHELL (reading R-N1): depletants drawn in the shell
    R_in < |d| <= R, N_d ~ Poisson(n_R V_shell).  Bit parity of outcomes, poses and counters as for the default path;
    the small-step case has a thin shell (R_in / R = 0.998), the half-balls R_in = 0 (the whole ball through the shell
    sampler)."""
    import dataclasses
    cfg = workloads.config(name, N)
    if d_max is not None:
        cfg = dataclasses.replace(cfg, d_max=d_max)
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, sweeps if FULL else 10, cfg.n_R(), options=1)
    assert c["dep_drawn"] > 0 and c["rej_depletant"] > 0
    if d_max is not None:
        assert c["accept_trans"] > 0.1 * c["trials_trans"]


@pytest.mark.parametrize("kernel", ["warp", "queue"])
@pytest.mark.parametrize("name,N,n_trial,options,sweeps", [("C5", None, 4, 2, 100), ("C5", 4096, 10, 2, 40),
                                                           ("C1", None, 4, 3, 100), ("C4", 4096, 1, 2, 40)])
def test_rosenbluth_weight_option(monkeypatch, kernel, name, N, n_trial, options, sweeps):
    """HPMC_OPT_ROSENBLUTH (NEXT-4, reading R-N4): weight N'_ins / (N_ins + 1), n_trial forward and n_trial - 1 reverse
    reinsertions; through both CB kernels, alone and together with the shell option, down to n_trial = 1 (no reverse
    reinsertion at all)."""
    import dataclasses
    monkeypatch.setenv("HPMC_CB_KERNEL", kernel)
    cfg = dataclasses.replace(workloads.config(name, N), n_trial=n_trial)
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, sweeps if FULL else 10, cfg.n_R(), options=options)
    assert c["cb_reinsertions"] > 0 and c["rej_cb"] > 0


@pytest.mark.parametrize("name,N", [("C1", None), ("C3", 65536), ("C4", None), ("C5", None)])
def test_free_volume_measurement(name, N):
    """hpmc_free_volume: the number of free test depletants is an integer and
    must EQUAL the oracle's on the same Philox points, before and after a few sweeps; also the empty sample."""
    cfg = workloads.config(name, N)
    pos, quat = workloads.generate(cfg)
    o, h, dpos, dquat = _mk(cfg, pos, quat)
    n = 1000000 if FULL else 100000
    for s in range(3):
        o.build_cells(cfg.seed, s); h.build_cells(cfg.seed, s)
        fo, fg = o.free_volume(cfg.seed, s, n), h.free_volume(cfg.seed, s, n)
        assert fg == fo, (s, fg, fo)
        assert 0.05 * n < fg < 0.95 * n
        o.sweep(cfg.seed, s, cfg.n_R(), cfg.d_max, cfg.a_max, cfg.n_trial)
        h.sweep(cfg.seed, s, cfg.n_R(), cfg.d_max, cfg.a_max, cfg.n_trial)
    h.build_cells(cfg.seed, 9)
    assert h.free_volume(cfg.seed, 9, 0) == 0
    import paper_1508_07077_b200 as hp
    with pytest.raises(hp.HPMCError) as e:
        h.free_volume(cfg.seed, 8, 10)                   # no cell list for (seed, 8)
    assert e.value.code == -3
    h.close()


@pytest.mark.parametrize("n_trial,kernel,options,N,sweeps", [(0, None, 0, None, 200), (10, "warp", 0, None, 100), (10, "queue", 0, None, 100),
                                                             (40, None, 2, 4096, 40), (0, None, 1, 4096, 60)])
def test_c6_oblate_ellipsoids(monkeypatch, n_trial, kernel, options, N, sweeps):
    """the paper's discoids (oblate ellipsoids a = b = 0.5, c = 0.25, depletant radius 0.25, L228)
    through both move kernels: plain rule, configurational bias with n_trial = 10 (PAPER.md: n_trial >~ 10) on either CB
    kernel, n_trial = 40 with the Rosenbluth weight, the shell option; plus the free-volume count."""
    import dataclasses
    if kernel:
        monkeypatch.setenv("HPMC_CB_KERNEL", kernel)
    cfg = dataclasses.replace(workloads.config("C6", N), n_trial=n_trial)
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, sweeps if FULL else 10, cfg.n_R(), options=options)
    assert c["accept_rot"] > 0 and c["accept_trans"] > 0 and c["rej_hard"] > 0
    assert (c["rej_cb"] if n_trial else c["rej_depletant"]) > 0
    if n_trial == 0 and not options:
        o, h, dpos, dquat = _mk(cfg, pos, quat)
        o.build_cells(cfg.seed, 0); h.build_cells(cfg.seed, 0)
        assert h.free_volume(cfg.seed, 0, 200000) == o.free_volume(cfg.seed, 0, 200000)
        h.close()


@pytest.mark.parametrize("n_trial,kernel,options,N,sweeps", [(0, None, 0, None, 200), (4, "warp", 0, 4096, 60), (20, None, 2, 4096, 40),
                                                             (0, None, 1, 4096, 60)])
def test_c7_tetrahedra(monkeypatch, n_trial, kernel, options, N, sweeps):
    """regular tetrahedra (Fig. 1), the one shape that is not a body of revolution (the
    kernels stage the whole quaternion per neighbour): plain rule at 32,768 particles on the dense aligned lattice
    (phi_c = 0.20: many support-function pair tests), CB on both kernels, Rosenbluth weight, shell; free-volume count."""
    import dataclasses
    if kernel:
        monkeypatch.setenv("HPMC_CB_KERNEL", kernel)
    cfg = dataclasses.replace(workloads.config("C7", N), n_trial=n_trial)
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, sweeps if FULL else 10, cfg.n_R(), options=options)
    assert c["accept_rot"] > 0 and c["accept_trans"] > 0 and c["rej_hard"] > 0
    assert (c["rej_cb"] if n_trial else c["rej_depletant"]) > 0
    if n_trial == 0 and not options:
        o, h, dpos, dquat = _mk(cfg, pos, quat)
        o.build_cells(cfg.seed, 0); h.build_cells(cfg.seed, 0)
        assert h.free_volume(cfg.seed, 0, 200000) == o.free_volume(cfg.seed, 0, 200000)
        h.close()


@pytest.mark.parametrize("name,N,options", [("C1", None, 0), ("C3", 16384, 1), ("C4", 4096, 0), ("C5", 512, 0), ("C6", 4096, 0),
                                            ("C7", 4096, 1)])
def test_warp_per_cell_kernel_plain_rule(monkeypatch, name, N, options):
    """HPMC_MOVE_KERNEL=warp: the first kernel design (one warp per active cell, 32 depletants per step, ballot exit;
    north_star's sketch) on every shape, plain rule, with and without the shell option: same bits as the oracle."""
    import dataclasses
    monkeypatch.setenv("HPMC_MOVE_KERNEL", "warp")
    cfg = dataclasses.replace(workloads.config(name, N), n_trial=0)
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, 40 if FULL else 10, cfg.n_R(), options=options)
    assert c["rej_depletant"] > 0


def test_one_launch_per_pass_mode(monkeypatch):
    """HPMC_SWEEP_LAUNCHES=8: the item-queue kernel launched once per checkerboard pass (no neighbour waits) instead of
    once per sweep; same bits."""
    monkeypatch.setenv("HPMC_SWEEP_LAUNCHES", "8")
    for name, N, sweeps in (("C3", 65536, 10), ("C4", 4096, 10)):
        cfg = workloads.config(name, N)
        pos, quat = workloads.generate(cfg)
        run_parity(cfg, pos, quat, sweeps, cfg.n_R())


def test_c5_dense_after_compression_hard_overlaps():
    """More hard-overlap (MPR) decisions: the same discoids in a box 8 % smaller per axis than a loose lattice."""
    import dataclasses
    cfg = dataclasses.replace(workloads.config("C5", 4096), phi_c=0.17, n_trial=2)
    pos, quat = workloads.generate(cfg)
    c = run_parity(cfg, pos, quat, 60, cfg.n_R())
    assert c["rej_hard"] > 100


@pytest.mark.parametrize("shape", ["sphere", "halfball"])
def test_edge_cases(shape):
    import dataclasses
    base = workloads.config("C1" if shape == "sphere" else "C4", 216 if shape == "halfball" else 48)
    pos, quat = workloads.generate(base)
    # (a) no depletants: plain hard-particle MC
    run_parity(base, pos, quat, 10, 0.0)
    # (b) zero step: every trial is the identity and is accepted
    cfg0 = dataclasses.replace(base, d_max=0.0, a_max=0.0)
    o, h, dpos, dquat = _mk(dataclasses.replace(cfg0, d_max=0.1), pos, quat)
    o.build_cells(1, 0); h.build_cells(1, 0)
    o.sweep(1, 0, base.n_R(), 0.0, 0.0, 0); h.sweep(1, 0, base.n_R(), 0.0, 0.0, 0)
    out = h.outcomes().cpu().numpy()
    assert np.array_equal(out, o.outcomes()) and set(np.unique(out)) <= {0, 1}
    h.close()
    # (c) a single particle (all but one cell empty), CB with the largest trial count the key layout allows
    one = dataclasses.replace(base, N=1, n_trial=300, phi_c=base.phi_c / base.N)      # same box, one particle
    p1 = pos[:1].copy()
    q1 = None if quat is None else quat[:1].copy()
    o, h, dpos, dquat = _mk(one, p1, q1)
    for s in range(20):
        o.build_cells(1, s); h.build_cells(1, s)
        o.sweep(1, s, base.n_R(), one.d_max, one.a_max, 300); h.sweep(1, s, base.n_R(), one.d_max, one.a_max, 300)
        assert np.array_equal(h.outcomes().cpu().numpy(), o.outcomes())
        assert np.array_equal(_bits(dpos.cpu().numpy()), _bits(o.pos))
    h.close()


def test_error_codes():
    import torch
    import paper_1508_07077_b200 as hp
    pos = torch.zeros((8, 4), device="cuda")
    with pytest.raises(hp.HPMCError) as e:
        hp.HPMC("sphere", 1.0, 0.2, 3.0, 0.1, pos)             # box too small: n_c < 4
    assert e.value.code == -2
    with pytest.raises(hp.HPMCError) as e:
        hp.HPMC("halfball", 1.0, 0.2, 30.0, 0.1, pos, None)    # anisotropic without orientations
    assert e.value.code == -1
    h = hp.HPMC("sphere", 1.0, 0.2, 8.0, 0.1, pos)
    with pytest.raises(hp.HPMCError) as e:
        h.sweep(1, 0, 1.0, 0.1)                                 # no build_cells
    assert e.value.code == -3
    h.build_cells(1, 0)
    with pytest.raises(hp.HPMCError) as e:
        h.sweep(1, 1, 1.0, 0.1)                                 # build for another step
    assert e.value.code == -3
    with pytest.raises(hp.HPMCError) as e:
        h.sweep(1, 0, 1.0, 0.2)                                 # d_max > cap
    assert e.value.code == -4
    with pytest.raises(hp.HPMCError) as e:
        h.sweep(1, 0, -1.0, 0.1)
    assert e.value.code == -1
    h.close()


@pytest.mark.parametrize("name,N,n_R_scale", [("C1", None, 1.0), ("C4", 4096, 1.0), ("C4", 4096, 0.0), ("C5", 512, 1.0), ("C7", 4096, 1.0)])
def test_host_buffer_step_matches_device_path(name, N, n_R_scale):
    """hpmc_step_host (library-owned buffers, host<->device copies inside) gives the same bits in the host arrays,
    through the sparse download (few accepted particles: only their poses come back and are patched in) and the full
    one (C4 without depletants: more than N/4 particles accepted per sweep)."""
    import torch
    import paper_1508_07077_b200 as hp
    cfg = workloads.config(name, N)
    pos, quat = workloads.generate(cfg)
    o, h, dpos, _ = _mk(cfg, pos, quat)
    hh = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, None, None, cfg.disk_a, cfg.disk_s, N=cfg.N)
    hpos = torch.from_numpy(pos.copy()).pin_memory()
    hquat = None if quat is None else torch.from_numpy(quat.copy()).pin_memory()
    hout = torch.zeros(cfg.N, dtype=torch.uint8).pin_memory()
    n_R = cfg.n_R() * n_R_scale
    full = 16 * cfg.N * (1 if quat is None else 2)
    sparse_seen = full_seen = False
    for s in range(8):
        o.build_cells(1, s); o.sweep(1, s, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)
        hh.step_host(hpos, hquat, hout, 1, s, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)
        assert np.array_equal(hout.numpy(), o.outcomes())
        assert np.array_equal(_bits(hpos.numpy()), _bits(o.pos))
        if quat is not None:
            assert np.array_equal(_bits(hquat.numpy()), _bits(o.quat))
        h2d, d2h = hh.step_host_bytes()
        assert h2d == full
        nacc = int((o.outcomes() == 1).sum())
        if nacc <= cfg.N // 4:
            assert d2h == cfg.N + 4 + nacc * (4 + full // cfg.N); sparse_seen = True
        else:
            assert d2h == cfg.N + 4 + full; full_seen = True
    assert full_seen if n_R_scale == 0.0 else sparse_seen
    hh.close(); h.close()


@pytest.mark.parametrize("n_c_target", [4, 6, 8])
def test_small_grids_wrap_rows_and_minimum_image(n_c_target):
    """Boxes of 4, 6 and 8 cells per axis: every row of the neighbourhood walk wraps for a large share of the cells,
    the kernel's "no minimum image needed" shortcut is off (n_c = 4), barely on (6) or on for the inner cells (8)."""
    import dataclasses
    base = workloads.config("C1")
    w_min = base.sigma_c + base.sigma_d + 2 * base.d_max
    L = w_min * (n_c_target + 0.6)
    N = max(8, int(0.25 * L ** 3 / (np.pi / 6)))
    cfg = dataclasses.replace(base, N=N, phi_c=N * (np.pi / 6) / L ** 3)
    pos, _ = workloads.generate(cfg)
    o, h, dpos, _ = _mk(cfg, pos, None)
    assert h.n_c == n_c_target == o.n_c
    h.close()
    c = run_parity(cfg, pos, None, 60, cfg.n_R(), check_cells_every=5)
    assert c["rej_depletant"] > 0 and c["rej_hard"] > 0


@pytest.mark.parametrize("phi_d", [0.00003, 0.002, 0.6])
def test_poisson_table_extremes(phi_d):
    """Tiny and large lambda: a threshold table of a few entries (every guide bucket holds several thresholds or none)
    and one of ~1300 entries; N_d parity shows up in dep_drawn."""
    import dataclasses
    cfg = dataclasses.replace(workloads.config("C3", 4096), phi_d_r=(phi_d,))
    pos, _ = workloads.generate(cfg)
    c = run_parity(cfg, pos, None, 12, cfg.n_R())
    assert c["dep_drawn"] > 0


def test_dense_fcc_crystal_neighbour_pool():
    """A dense fcc crystal (phi = 0.66: 12 neighbours inside the list radius of every move) at a size where the tiles
    are large: the per-tile neighbour pool must hold (the library reports HPMC_E_NEIGHBOR_OVERFLOW otherwise)."""
    import dataclasses
    cfg = dataclasses.replace(workloads.config("C2", 4 * 64 ** 3), phi_c=0.66, q=0.08, d_max=0.03, phi_d_r=(0.1,))
    pos, _ = workloads.generate(cfg)
    c = run_parity(cfg, pos, None, 3, cfg.n_R(), check_cells_every=1)
    assert c["rej_hard"] > 0



def _clustered_slab(cfg, frac=1.0 / 3.0):
    """The paper's use case is depletion-driven aggregation (Fig. 7): a dense fcc slab (phi = 0.66
    locally) filling a third of the box along z, the rest empty.  Positions only; no arithmetic of the method."""
    L = cfg.box_L
    nn = (4.0 * (np.pi / 6.0) / 0.66) ** (1.0 / 3.0) / np.sqrt(2.0)      # nearest-neighbour distance of fcc at phi = 0.66
    a = nn * np.sqrt(2.0)
    ncx = int(L / a)
    ncz = int(frac * L / a)
    ax, az = L / ncx, a                                                   # stretched to fit the box in x, y (periodic)
    base = np.array([(0, 0, 0), (0.5, 0.5, 0), (0.5, 0, 0.5), (0, 0.5, 0.5)], np.float64)
    ii, kk = np.arange(ncx), np.arange(ncz)
    g = np.stack(np.meshgrid(ii, ii, kk, indexing="ij"), -1).reshape(-1, 1, 3) + base[None]
    pos = g.reshape(-1, 3) * np.array([ax, ax, az]) + 0.25 * a
    assert ax / np.sqrt(2.0) > 1.0005 * cfg.sigma_c
    p4 = np.zeros((len(pos), 4), np.float32)
    p4[:, :3] = pos
    assert p4[:, :3].max() < np.float32(L)
    return p4


def test_clustered_slab_neighbour_pool_recovers():
    """A clustered system at low MEAN density (the paper's aggregation use case, L218): a close-packed slab in a
    C3-sized box, ~8e5 spheres with 12 listed neighbours each where the box average suggests ~5.  The move kernel
    must split tiles whose neighbour pool overflows and stay bit-exact (no HPMC_E_NEIGHBOR_OVERFLOW)."""
    import dataclasses
    cfg = dataclasses.replace(workloads.config("C3"), q=0.08, d_max=0.03, phi_d_r=(0.1,))
    pos = _clustered_slab(cfg)
    cfg = dataclasses.replace(cfg, N=len(pos), phi_c=len(pos) * (np.pi / 6) / cfg.box_L ** 3)
    assert cfg.N >= 500000 and abs(cfg.box_L - workloads.config("C3").box_L) < 1e-3
    c = run_parity(cfg, pos, None, 3, cfg.n_R(), check_cells_every=1)
    assert c["rej_hard"] > 0 and c["rej_depletant"] > 0


def test_clustered_slab_large_tiles_forced(monkeypatch):
    """The same slab with the tile size forced far above what the pool holds: every tile of the slab overflows and
    is split (several times) inside the CTA."""
    import dataclasses
    monkeypatch.setenv("HPMC_CELLS_PER_CTA", "400")
    monkeypatch.setenv("HPMC_POOL_CAP_OFF", "1")
    cfg = dataclasses.replace(workloads.config("C3"), q=0.08, d_max=0.03, phi_d_r=(0.1,))
    pos = _clustered_slab(cfg, frac=0.12)
    cfg = dataclasses.replace(cfg, N=len(pos), phi_c=len(pos) * (np.pi / 6) / cfg.box_L ** 3)
    run_parity(cfg, pos, None, 2, cfg.n_R(), check_cells_every=1)


@pytest.mark.parametrize("cells_per_cta,tile", [(600, 64), (None, 64)])
def test_several_tiles_per_cta(monkeypatch, cells_per_cta, tile):
    """The multi-tile loop of the move kernel is only reached by systems larger than one wave (> ~2.4 M spheres);
    force it at C3's size with tiles of 64 cells: fewer, larger CTA shares without the work ramp (the request for 600
    cells is cut to the neighbour-pool bound, ~180), and the default shares with the ramp (up to ~180 cells)."""
    if cells_per_cta:
        monkeypatch.setenv("HPMC_CELLS_PER_CTA", str(cells_per_cta))
    monkeypatch.setenv("HPMC_TILE_BIG", str(tile))
    cfg = workloads.config("C3")
    pos, _ = workloads.generate(cfg)
    run_parity(cfg, pos, None, 2, cfg.n_R(), check_cells_every=1)
