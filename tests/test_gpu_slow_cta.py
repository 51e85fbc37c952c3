"""The one-launch sweep and slow CTAs (GPU).

In the cooperative move kernel a CTA waits, between checkerboard passes, for the CTAs that own neighbouring cells.  How
long such a wait lasts is set by the slowest neighbour, and that has no small bound: n_trial up to 65535 is accepted, and
in an aggregated system (Fig. 7) the CTAs of the empty region have nothing to do while those of the
cluster reinsert for hundreds of milliseconds per pass.  A wait bounded in polls turned exactly that case into
HPMC_E_CUDA with invalid poses (round-2 advisor finding); now the wait is bounded only by a wall-clock guard of 60 s
against a lost CTA, and a CTA that hits the guard abandons the sweep instead of walking cells its neighbour still writes.

No oracle here (2 x 65535 reinsertions per rejecting depletant are out of its reach): the reference is the library's
warp-per-cell kernel, which runs one launch per pass and has no waits; both kernels are bit-exact against the oracle in
tests/test_gpu_parity.py.
"""
import dataclasses
import os
import subprocess
import sys

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SHARED_COUNTERS = ("trials_trans", "accept_trans", "rej_boundary", "rej_hard", "rej_depletant", "rej_cb", "dep_drawn",
                   "dep_needed", "cb_reinsertions")


def _slab():
    """A close-packed slab filling a third of a C2-sized box (47,916 spheres, 42^3 cells), the rest empty."""
    from test_gpu_parity import _clustered_slab
    cfg = dataclasses.replace(workloads.config("C2"), q=0.08, d_max=0.03, phi_d_r=(0.4,))
    pos = _clustered_slab(cfg)
    return dataclasses.replace(cfg, N=len(pos), phi_c=len(pos) * (np.pi / 6) / cfg.box_L ** 3), pos


def _one_sweep(cfg, pos, n_trial):
    import torch
    import paper_1508_07077_b200 as hp
    dpos = torch.from_numpy(pos.copy()).cuda()
    h = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, dpos)
    h.build_cells(cfg.seed, 0)
    h.sweep(cfg.seed, 0, cfg.n_R(), cfg.d_max, 0.0, n_trial)
    c = h.counters()                       # synchronises; raises HPMCError if the kernel flagged anything
    out = h.outcomes().cpu().numpy()
    h.close()
    return dpos.cpu().numpy(), out, c


def test_slow_neighbour_pass_is_waited_for(monkeypatch):
    """n_trial = 65535 on the slab: ~0.8 s per pass in the cluster's CTAs while their neighbours idle (the poll-bounded
    wait of round 2 gave up after ~0.3 s here).  The sweep must finish without an error and agree bit for bit with the
    kernel that has no waits."""
    cfg, pos = _slab()
    p_q, o_q, c_q = _one_sweep(cfg, pos, 65535)
    monkeypatch.setenv("HPMC_CB_KERNEL", "warp")          # read by hpmc_init: the next context uses one launch per pass
    p_w, o_w, c_w = _one_sweep(cfg, pos, 65535)
    assert np.array_equal(o_q, o_w)
    assert np.array_equal(p_q.view(np.uint32), p_w.view(np.uint32))
    for k in SHARED_COUNTERS:
        assert c_q[k] == c_w[k], (k, c_q[k], c_w[k])
    assert c_q["cb_reinsertions"] > 10 ** 10 and c_q["accept_trans"] > 0


_CHILD = r"""
import sys
sys.path.insert(0, %(root)r); sys.path.insert(0, %(tests)r)
import torch
import paper_1508_07077_b200 as hp
from test_gpu_slow_cta import _slab
cfg, pos = _slab()
dpos = torch.from_numpy(pos.copy()).cuda()
h = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, dpos)
h.build_cells(cfg.seed, 0)
h.sweep(cfg.seed, 0, cfg.n_R(), cfg.d_max, 0.0, 20000)          # ~0.25 s per pass in the cluster's CTAs
try:
    h.counters()
    print("NO-ERROR")
except hp.HPMCError as e:
    print("ERROR %%d %%s" %% (e.code, e))
# the flag is cleared and the pass counters are where the next sweep expects them: a quick sweep of the same kernel
# (configurational bias, but no depletants) runs and reports nothing
h.build_cells(cfg.seed, 1)
h.sweep(cfg.seed, 1, 0.0, cfg.d_max, 0.0, 20000)
c = h.counters()
print("NEXT-SWEEP-OK %%d" %% c["trials_trans"])
"""


def test_wait_limit_abandons_the_sweep_without_hanging():
    """The guard itself, with a build whose limit is 1 us instead of 60 s (the clock is looked at every 4096 polls, so it
    strikes after a millisecond or two): the slow sweep must end with HPMC_E_CUDA -- not hang, not go on silently -- and
    leave the context usable."""
    from paper_1508_07077_b200 import build as cuda_build
    so = os.path.join(ROOT, "paper_1508_07077_b200", "libhpmc_b200_waitlimit.so")
    cuda_build.build(defines=("HPMC_WAIT_LIMIT_NS=1000ull",), out=so)
    env = dict(os.environ, HPMC_LIBRARY_PATH=so)
    env.pop("HPMC_CB_KERNEL", None)
    r = subprocess.run([sys.executable, "-c", _CHILD % {"root": ROOT, "tests": os.path.join(ROOT, "tests")}], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "ERROR -5" in r.stdout and "abandoned the sweep" in r.stdout, r.stdout
    assert "NEXT-SWEEP-OK" in r.stdout, r.stdout
