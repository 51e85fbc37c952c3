"""ctypes loader for the CPU oracle (TEST INFRASTRUCTURE; see hpmc_oracle.cpp).

The shared object is compiled in-tree from ``hpmc_oracle.cpp`` on first use (g++ is part of
the image, on the GPU box too) with ``-O2 -ffp-contract=off``; an ``-mfma`` twin is built and
picked when the running CPU has FMA so that the explicitly written ``fmaf`` is one instruction.
Both give the same bits: ``fmaf`` is exactly rounded either way.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hpmc_oracle.cpp")
_LOCK = threading.Lock()
_LIB = None

COUNTER_NAMES = (
    "trials_trans", "accept_trans", "trials_rot", "accept_rot", "rej_boundary", "rej_hard",
    "rej_depletant", "rej_cb", "dep_drawn", "dep_needed", "dep_evaluated", "cb_reinsertions",
    "philox_blocks",
)

SHAPES = {"sphere": 0, "halfball": 1, "spherodisk": 2, "ellipsoid": 3, "tetrahedron": 4}
FLAG_SHELL, FLAG_ROSENBLUTH = 1, 2


class OracleParams(C.Structure):
    _fields_ = [("shape", C.c_int32), ("sigma_c", C.c_float), ("disk_a", C.c_float), ("disk_s", C.c_float),
                ("sigma_d", C.c_float), ("box_L", C.c_float), ("d_max_cap", C.c_float)]


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return " fma " in line + " "
    except OSError:
        pass
    return False


def _so_path(fma: bool) -> str:
    return os.path.join(_HERE, "liboracle_fma.so" if fma else "liboracle_generic.so")


def build(force: bool = False) -> str:
    """Compile both variants if missing or older than the source; return the one to load."""
    for fma in (False, True):
        so = _so_path(fma)
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fno-math-errno",
                   "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", so + ".tmp%d" % os.getpid(), _SRC]
            if fma:
                cmd.insert(1, "-mfma")
            subprocess.run(cmd, check=True)
            os.replace(so + ".tmp%d" % os.getpid(), so)
    return _so_path(_cpu_has_fma())


def apply_signatures(L: C.CDLL) -> C.CDLL:
    """ctypes signatures of every oracle_* export, on the oracle library or on a throw-away mutant build of it
    (tests compile hpmc_oracle.cpp with one line changed to show that a pin catches the change)."""
    vp, u32, i32, i64, f32, f64 = C.c_void_p, C.c_uint32, C.c_int32, C.c_int64, C.c_float, C.c_double
    P = C.POINTER
    sig = {
        "oracle_create": (vp, [P(OracleParams), i64, vp, vp]),
        "oracle_destroy": (None, [vp]),
        "oracle_set_flags": (i32, [vp, u32, f32]),
        "oracle_cbrt_fixed": (f32, [f32]),
        "oracle_shell": (f64, [P(OracleParams), f64, f32, u32, P(f32)]),
        "oracle_shell_samples": (None, [P(OracleParams), f32, u32, u32, u32, u32, i64, vp]),
        "oracle_grid": (i32, [vp, P(i32), P(f32)]),
        "oracle_set_threads": (None, [i32]),
        "oracle_get_threads": (i32, []),
        "oracle_build_cells": (i32, [vp, u32, u32]),
        "oracle_sweep": (i32, [vp, u32, u32, f64, f32, f32, i32]),
        "oracle_colour_order": (i32, [u32, u32, vp]),
        "oracle_counters": (i32, [vp, vp]),
        "oracle_reset_counters": (i32, [vp]),
        "oracle_outcomes": (i32, [vp, vp]),
        "oracle_trial_poses": (i32, [vp, vp, vp]),
        "oracle_cells": (i32, [vp, vp, vp, vp]),
        "oracle_run": (i32, [vp, u32, u32, i64, f64, f32, f32, i32, vp, vp]),
        "oracle_eval_move": (i32, [vp, u32, u32, i64, vp, vp, f64, i32]),
        "oracle_eval_moves": (i32, [vp, u32, u32, i64, i64, vp, vp, f64, i32, vp]),
        "oracle_count_overlaps": (i64, [vp, i32]),
        "oracle_free_volume": (i32, [vp, u32, u32, i64, vp]),
        "oracle_philox4x32_10": (None, [vp, vp, vp]),
        "oracle_unit01": (f32, [u32]),
        "oracle_sym_unit": (f32, [u32]),
        "oracle_poisson_table": (i64, [f64, P(i64), vp, i64]),
        "oracle_poisson_draws": (None, [f64, vp, i64, vp]),
        "oracle_lambda": (f64, [P(OracleParams), f64]),
        "oracle_ball_samples": (None, [u32, u32, u32, u32, i64, f32, vp]),
        "oracle_dep_overlap": (None, [P(OracleParams), vp, vp, i64, vp]),
        "oracle_pair_overlap": (None, [P(OracleParams), vp, vp, vp, i64, vp]),
        "oracle_support": (None, [P(OracleParams), vp, vp, vp]),
        "oracle_quat_axis": (None, [vp, vp]),
        "oracle_rotate_cayley": (None, [vp, vp, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    return L


def lib() -> C.CDLL:
    global _LIB
    with _LOCK:
        if _LIB is None:
            _LIB = apply_signatures(C.CDLL(build()))
    return _LIB


def colour_order(seed: int, step: int) -> np.ndarray:
    """The order in which sweep (seed, step) visits the 8 checkerboard colours (R-2)."""
    out = np.empty(8, np.uint32)
    lib().oracle_colour_order(seed, step, _ptr(out))
    return out


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def make_params(shape, sigma_c, sigma_d, box_L, d_max_cap, disk_a=0.0, disk_s=0.0) -> OracleParams:
    return OracleParams(SHAPES[shape] if isinstance(shape, str) else int(shape), sigma_c, disk_a, disk_s,
                        sigma_d, box_L, d_max_cap)


class Oracle:
    """Host-memory twin of the C-ABI context: same calls, numpy buffers, updated in place."""

    def __init__(self, shape, sigma_c, sigma_d, box_L, d_max_cap, pos4, quat4=None, disk_a=0.0, disk_s=0.0,
                 threads=None):
        self.L = lib()
        self.params = make_params(shape, sigma_c, sigma_d, box_L, d_max_cap, disk_a, disk_s)
        self.pos = np.ascontiguousarray(pos4, dtype=np.float32).copy()
        assert self.pos.ndim == 2 and self.pos.shape[1] == 4
        self.N = self.pos.shape[0]
        self.quat = None if quat4 is None else np.ascontiguousarray(quat4, dtype=np.float32).copy()
        if threads is not None:
            self.L.oracle_set_threads(int(threads))
        self.h = self.L.oracle_create(C.byref(self.params), self.N, _ptr(self.pos), _ptr(self.quat))
        if not self.h:
            raise ValueError("oracle_create failed (bad arguments or n_c < 4)")
        nc, w = C.c_int32(), C.c_float()
        self.L.oracle_grid(self.h, C.byref(nc), C.byref(w))
        self.n_c, self.w = nc.value, w.value

    def __del__(self):
        h, self.h = getattr(self, "h", None), None
        if h:
            self.L.oracle_destroy(h)

    def set_flags(self, flags, eval_dmax=-1.0):
        """Options of the following sweeps: FLAG_SHELL (R-N1), FLAG_ROSENBLUTH (R-N4); eval_dmax: step size assumed by
        eval_move(s) for the shell."""
        self.L.oracle_set_flags(self.h, int(flags), float(eval_dmax))

    def build_cells(self, seed, step):
        rc = self.L.oracle_build_cells(self.h, seed, step)
        assert rc == 0, rc

    def sweep(self, seed, step, n_R, d_max, a_max=0.0, n_trial=0):
        rc = self.L.oracle_sweep(self.h, seed, step, float(n_R), d_max, a_max, n_trial)
        if rc:
            raise RuntimeError("oracle_sweep rc=%d" % rc)

    def run(self, seed, step0, n, n_R, d_max, a_max=0.0, n_trial=0, traj=False, outcomes=False):
        tr = np.empty((n, self.N, 4), np.float32) if traj else None
        oc = np.empty((n, self.N), np.uint8) if outcomes else None
        rc = self.L.oracle_run(self.h, seed, step0, n, float(n_R), d_max, a_max, n_trial, _ptr(tr), _ptr(oc))
        if rc:
            raise RuntimeError("oracle_run rc=%d" % rc)
        return tr, oc

    def counters(self):
        out = np.zeros(len(COUNTER_NAMES), np.uint64)
        self.L.oracle_counters(self.h, _ptr(out))
        return {k: int(v) for k, v in zip(COUNTER_NAMES, out)}

    def reset_counters(self):
        self.L.oracle_reset_counters(self.h)

    def outcomes(self):
        out = np.zeros(self.N, np.uint8)
        self.L.oracle_outcomes(self.h, _ptr(out))
        return out

    def trial_poses(self):
        p = np.zeros((self.N, 4), np.float32)
        q = np.zeros((self.N, 4), np.float32)
        self.L.oracle_trial_poses(self.h, _ptr(p), _ptr(q))
        return p, q

    def cells(self):
        cs = np.zeros(self.n_c ** 3 + 1, np.uint32)
        cp = np.zeros(self.N, np.uint32)
        sh = np.zeros(3, np.float32)
        self.L.oracle_cells(self.h, _ptr(cs), _ptr(cp), _ptr(sh))
        return cs, cp, sh

    def eval_move(self, seed, draw, i, pos3, quat4, n_R, n_trial=0):
        p = np.ascontiguousarray(pos3, np.float32)
        q = None if quat4 is None else np.ascontiguousarray(quat4, np.float32)
        return self.L.oracle_eval_move(self.h, seed, draw, i, _ptr(p), _ptr(q), float(n_R), n_trial)

    def eval_moves(self, seed, draw0, n, i, pos3, quat4, n_R, n_trial=0):
        """Outcome codes of n independent evaluations (draw0 .. draw0+n-1) of the same prescribed move."""
        p = np.ascontiguousarray(pos3, np.float32)
        q = None if quat4 is None else np.ascontiguousarray(quat4, np.float32)
        out = np.empty(n, np.uint8)
        rc = self.L.oracle_eval_moves(self.h, seed, draw0, n, i, _ptr(p), _ptr(q), float(n_R), n_trial, _ptr(out))
        if rc:
            raise RuntimeError("oracle_eval_moves rc=%d" % rc)
        return out

    def free_volume(self, seed, step, n):
        """Number of n uniform test depletants that overlap no colloid (needs build_cells(seed, step))."""
        out = np.zeros(1, np.uint64)
        rc = self.L.oracle_free_volume(self.h, seed, step, int(n), _ptr(out))
        if rc:
            raise RuntimeError("oracle_free_volume rc=%d" % rc)
        return int(out[0])

    def count_overlaps(self, both_ways=True):
        return int(self.L.oracle_count_overlaps(self.h, 1 if both_ways else 0))
