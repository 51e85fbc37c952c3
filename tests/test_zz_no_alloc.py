"""hpmc_cells_noalloc against hpmc_build_cells + hpmc_cells (GPU).

hpmc_cells_noalloc builds the checkerboard cell list with its working storage in a fixed array inside the library
instead of cudaMalloc'ed buffers.  It exists for programs that want the cell list of a configuration but may not
allocate: an analysis hook inside a simulation whose memory pool (PyTorch's caching allocator, an engine's arena) already
owns the GPU, where a raw cudaMalloc from a library fails; or a per-step loop that cannot pay for cudaFree's device-wide
wait.  The price is a size limit (262,144 particles, 64 cells per axis) and one scratch array per GPU shared by all
calls, which keeps whatever the previous call left in it.

So the checks here are the ones that sharing can break: the result is compared bit for bit (integer work: no
tolerance) with the existing path on two calls in a row -- the second on moved particles, another grid shift and then on
a much smaller system, so that anything a call fails to clear or rewrite shows up -- and the size limits are refused with
a message instead of overrunning the array.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (its first call does the per-device address look-up) and after the
other tests.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

MAX_N = 262144          # limits stated in include/hpmc.h
MAX_NC = 64


def _context(cfg):
    import torch
    import paper_1508_07077_b200 as hp
    pos, quat = workloads.generate(cfg)
    dpos = torch.from_numpy(pos.copy()).cuda()
    dquat = None if quat is None else torch.from_numpy(quat.copy()).cuda()
    h = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, dpos, dquat, cfg.disk_a, cfg.disk_s)
    return h, dpos


def _both_paths(h, dpos, cfg, step):
    """Cell list of the current poses by the context's build and by the allocation-free entry point (same grid, same
    shift); the outputs of the latter start out as garbage so that every word it must write is seen to be written."""
    import torch
    import paper_1508_07077_b200 as hp
    h.build_cells(cfg.seed, step)
    cs_ref, cp_ref, shift = h.cells()
    cs = torch.full((h.n_c ** 3 + 1,), -1, dtype=torch.int32, device="cuda")
    cp = torch.full((cfg.N,), -1, dtype=torch.int32, device="cuda")
    hp.cells_noalloc(dpos, cfg.box_L, h.n_c, shift, cs, cp)
    torch.cuda.synchronize()
    return (cs_ref.cpu().numpy(), cp_ref.cpu().numpy()), (cs.cpu().numpy(), cp.cpu().numpy())


def _check(ref, got, N, what):
    assert np.array_equal(got[0], ref[0]), "cell_start differs (%s)" % what
    assert np.array_equal(got[1], ref[1]), "cell_pid differs (%s)" % what
    assert got[0][0] == 0 and got[0][-1] == N
    assert np.array_equal(np.sort(got[1]), np.arange(N, dtype=np.int32))     # every particle listed exactly once


def test_two_calls_in_a_row_match_the_context_path():
    """C2 (65,536 spheres, 40^3 = 64,000 cells: 31 scan tiles and a ragged 32nd).  Call 1 on the initial lattice; then a
    sweep moves particles and step + 1 draws another grid shift; call 2 reuses the array call 1 dirtied."""
    cfg = workloads.config("C2")
    assert cfg.N <= MAX_N
    h, dpos = _context(cfg)
    assert h.n_c <= MAX_NC
    ref, got = _both_paths(h, dpos, cfg, 0)
    _check(ref, got, cfg.N, "first call")
    h.sweep(cfg.seed, 0, cfg.n_R(), cfg.d_max, cfg.a_max, cfg.n_trial)
    ref2, got2 = _both_paths(h, dpos, cfg, 1)
    _check(ref2, got2, cfg.N, "second call")
    assert not np.array_equal(ref2[0], ref[0]), "the second call was meant to see another grid shift"
    h.close()


def test_small_system_after_a_large_one_and_other_shapes():
    """A call on 256 spheres in 6^3 cells (a fraction of one scan tile) right after one that filled 64,000 cells and
    65,536 particle slots of the same array, twice in a row; then half-balls (the list depends on centres only)."""
    big = workloads.config("C2")
    hb, dposb = _context(big)
    _check(*_both_paths(hb, dposb, big, 3), big.N, "large system")
    small = workloads.config("C1")
    hs, dposs = _context(small)
    for step in (0, 1):
        _check(*_both_paths(hs, dposs, small, step), small.N, "small system after a large one, call %d" % step)
    hb.close(); hs.close()
    c4 = workloads.config("C4", 4096)
    h4, dpos4 = _context(c4)
    for step in (0, 1):
        _check(*_both_paths(h4, dpos4, c4, step), c4.N, "half-balls, call %d" % step)
    h4.close()


def _numpy_cells(pos, n_c, L):
    """Unshifted grid, written out with numpy: fp32 division as in the kernel, occupants in ascending particle id."""
    w = np.float32(L) / np.float32(n_c)
    idx = np.minimum((pos[:, :3] / w).astype(np.int32), n_c - 1)
    cell = (idx[:, 2] * n_c + idx[:, 1]) * n_c + idx[:, 0]
    order = np.argsort(cell, kind="stable").astype(np.int32)
    start = np.concatenate([[0], np.cumsum(np.bincount(cell, minlength=n_c ** 3))]).astype(np.int32)
    return start, order


def _uniform_pos(N, L, seed):
    rng = np.random.default_rng(seed)
    pos = np.zeros((N, 4), np.float32)
    xyz = rng.random((N, 3), dtype=np.float32) * np.float32(L)
    xyz[xyz >= np.float32(L)] = 0.0
    pos[:, :3] = xyz
    return pos


def test_unshifted_grid_against_numpy():
    """Independent of the context path: zero shift, cell list recomputed with numpy; two calls in a row."""
    import torch
    import paper_1508_07077_b200 as hp
    N, n_c, L = 5000, 10, 17.5
    pos = _uniform_pos(N, L, 7)
    start, order = _numpy_cells(pos, n_c, L)
    cs = torch.full((n_c ** 3 + 1,), -1, dtype=torch.int32, device="cuda")
    cp = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    dpos = torch.from_numpy(pos).cuda()
    for _ in range(2):
        hp.cells_noalloc(dpos, L, n_c, (0.0, 0.0, 0.0), cs, cp)
        torch.cuda.synchronize()
        assert np.array_equal(cs.cpu().numpy(), start)
        assert np.array_equal(cp.cpu().numpy(), order)
        cs.fill_(-1); cp.fill_(-1)


def test_sizes_beyond_the_fixed_array_are_refused():
    """One particle or one cell layer beyond what the array holds: HPMC_E_BADARG with the limit in the message, and
    nothing launched (the outputs keep their fill).  The limits themselves are served."""
    import torch
    import paper_1508_07077_b200 as hp
    L = 100.0
    pos = _uniform_pos(MAX_N + 1, L, 11)
    dpos = torch.from_numpy(pos).cuda()
    cs = torch.full(((MAX_NC + 2) ** 3 + 1,), -1, dtype=torch.int32, device="cuda")
    cp = torch.full((MAX_N + 1,), -1, dtype=torch.int32, device="cuda")
    with pytest.raises(hp.HPMCError) as e:
        hp.cells_noalloc(dpos, L, 8, (0.0, 0.0, 0.0), cs, cp)                      # 262,145 particles
    assert e.value.code == -1 and str(MAX_N) in str(e.value)
    with pytest.raises(hp.HPMCError) as e:
        hp.cells_noalloc(dpos[:1000], L, MAX_NC + 2, (0.0, 0.0, 0.0), cs, cp)      # 66^3 cells
    assert e.value.code == -1 and str(MAX_NC) in str(e.value)
    with pytest.raises(hp.HPMCError):
        hp.cells_noalloc(dpos[:1000], L, 8, (0.0, 250.0, 0.0), cs, cp)             # shift outside the box
    torch.cuda.synchronize()
    assert bool((cs == -1).all()) and bool((cp == -1).all())
    hp.cells_noalloc(dpos[:MAX_N], L, MAX_NC, (0.0, 0.0, 0.0), cs, cp)             # exactly the limits
    torch.cuda.synchronize()
    start, order = _numpy_cells(pos[:MAX_N], MAX_NC, L)
    assert np.array_equal(cs[:MAX_NC ** 3 + 1].cpu().numpy(), start)
    assert np.array_equal(cp[:MAX_N].cpu().numpy(), order)
