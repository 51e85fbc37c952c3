"""ctypes binding of include/hpmc.h: same names, argument marshalling only.

PyTorch supplies device buffers (torch.Tensor.data_ptr()) and the stream; nothing is computed here.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

COUNTER_NAMES = (
    "trials_trans", "accept_trans", "trials_rot", "accept_rot", "rej_boundary", "rej_hard",
    "rej_depletant", "rej_cb", "dep_drawn", "dep_needed", "dep_evaluated", "cb_reinsertions",
    "philox_blocks",
)
SHAPES = {"sphere": 0, "halfball": 1, "spherodisk": 2, "ellipsoid": 3, "tetrahedron": 4}
OPT_SHELL, OPT_ROSENBLUTH = 1, 2          # hpmc_set_options

EXPORTS = (
    "hpmc_init", "hpmc_destroy", "hpmc_build_cells", "hpmc_sweep", "hpmc_run", "hpmc_counters",
    "hpmc_reset_counters", "hpmc_outcomes", "hpmc_grid", "hpmc_cells", "hpmc_upload", "hpmc_download",
    "hpmc_step_host", "hpmc_launch_count", "hpmc_time_move_kernel", "hpmc_move_kernel_ms", "hpmc_last_error",
    "hpmc_alu_peaks", "hpmc_set_options", "hpmc_free_volume", "hpmc_step_host_bytes", "hpmc_cells_noalloc",
)


class HPMCError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("hpmc error %d: %s" % (code, msg))
        self.code = code


class Params(C.Structure):
    """hpmc_params"""
    _fields_ = [("shape", C.c_int32), ("sigma_c", C.c_float), ("disk_a", C.c_float), ("disk_s", C.c_float),
                ("sigma_d", C.c_float), ("box_L", C.c_float), ("d_max_cap", C.c_float)]


class Counters(C.Structure):
    """hpmc_counters_t"""
    _fields_ = [(n, C.c_uint64) for n in COUNTER_NAMES]


ALU_KINDS = ("fadd", "fmul", "ffma", "imad", "imadwide_lop3_pair", "lop3", "fadd_lop3_mix", "philox_blocks_ilp1", "philox_blocks_ilp2",
             "philox_blocks_ilp4")


class AluPeaks(C.Structure):
    """hpmc_alu_peaks_t"""
    _fields_ = [("num_sms", C.c_int32), ("sm_clock_khz", C.c_int32), ("sm_mhz_during", C.c_double),
                ("rate", C.c_double * 10)]


def library_path() -> str:
    """In-tree library; HPMC_LIBRARY_PATH selects another build of the same sources (tuning builds)."""
    return os.environ.get("HPMC_LIBRARY_PATH") or os.path.join(_HERE, "libhpmc_b200.so")


def load_library() -> C.CDLL:
    """Load libhpmc_b200.so (built in-tree by paper_1508_07077_b200/build.py).  Raises if it is missing:
    the product path never falls back to a CPU implementation."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        raise HPMCError(-5, "CUDA library %s not built; run `python -c 'import __graft_entry__ as g; g.build()'`" % path)
    L = C.CDLL(path)
    vp, u32, i32, i64, f32, f64 = C.c_void_p, C.c_uint32, C.c_int32, C.c_int64, C.c_float, C.c_double
    P = C.POINTER
    sig = {
        "hpmc_init": (i32, [P(vp), P(Params), i64, vp, vp, vp]),
        "hpmc_destroy": (None, [vp]),
        "hpmc_build_cells": (i32, [vp, u32, u32]),
        "hpmc_sweep": (i32, [vp, u32, u32, f64, f32, f32, i32]),
        "hpmc_run": (i32, [vp, u32, u32, i64, f64, f32, f32, i32]),
        "hpmc_set_options": (i32, [vp, u32]),
        "hpmc_step_host_bytes": (i32, [vp, P(i64), P(i64)]),
        "hpmc_free_volume": (i32, [vp, u32, u32, i64, P(C.c_uint64)]),
        "hpmc_counters": (i32, [vp, P(Counters)]),
        "hpmc_reset_counters": (i32, [vp]),
        "hpmc_outcomes": (i32, [vp, vp]),
        "hpmc_grid": (i32, [vp, P(i32), P(f32)]),
        "hpmc_cells": (i32, [vp, vp, vp, P(f32 * 3)]),
        "hpmc_upload": (i32, [vp, vp, vp]),
        "hpmc_download": (i32, [vp, vp, vp, vp]),
        "hpmc_step_host": (i32, [vp, vp, vp, vp, u32, u32, f64, f32, f32, i32]),
        "hpmc_launch_count": (i64, [vp]),
        "hpmc_time_move_kernel": (i32, [vp, i32]),
        "hpmc_move_kernel_ms": (i32, [vp, P(f64), P(i64)]),
        "hpmc_last_error": (C.c_char_p, [vp]),
        "hpmc_alu_peaks": (i32, [P(AluPeaks), vp]),
        "hpmc_cells_noalloc": (i32, [vp, i64, f32, i32, P(f32 * 3), vp, vp, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _LIB = L
    return L


def alu_peaks(stream=None):
    """hpmc_alu_peaks: measured per-SM-per-clock rates of the plain ALU pipes on the current device."""
    import torch
    L = load_library()
    s = torch.cuda.current_stream() if stream is None else stream
    out = AluPeaks()
    rc = L.hpmc_alu_peaks(C.byref(out), C.c_void_p(s.cuda_stream))
    if rc:
        raise HPMCError(rc, (L.hpmc_last_error(None) or b"").decode())
    d = {"num_sms": out.num_sms, "sm_clock_khz": out.sm_clock_khz, "sm_mhz_during": out.sm_mhz_during}
    d.update({k: out.rate[i] for i, k in enumerate(ALU_KINDS)})
    return d


def _dptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def cells_noalloc(pos4, box_L, n_c, shift3, cell_start, cell_pid, stream=None):
    """hpmc_cells_noalloc: the checkerboard cell list of `pos4` written into the caller's `cell_start` (n_c^3 + 1 int32)
    and `cell_pid` (N int32) CUDA tensors, with no device allocation inside the library -- for callers whose memory pool
    owns the GPU or who cannot pay for cudaMalloc / cudaFree in their loop (include/hpmc.h has the whole contract: at most
    262,144 particles and n_c <= 64, one shared scratch array per GPU, so calls that overlap on the GPU race).
    Asynchronous on `stream` (default: torch's current stream); the three tensors must stay alive until it has run."""
    import torch
    L = load_library()
    s = torch.cuda.current_stream() if stream is None else stream
    for t in (pos4, cell_start, cell_pid):
        assert t.is_cuda and t.is_contiguous()
    assert pos4.dtype == torch.float32 and pos4.shape[1] == 4
    assert cell_start.dtype == torch.int32 and cell_pid.dtype == torch.int32
    assert cell_pid.numel() >= pos4.shape[0] and cell_start.numel() >= int(n_c) ** 3 + 1
    sh = (C.c_float * 3)(*[float(x) for x in shift3])
    rc = L.hpmc_cells_noalloc(_dptr(pos4), int(pos4.shape[0]), float(box_L), int(n_c), C.byref(sh), _dptr(cell_start),
                              _dptr(cell_pid), C.c_void_p(s.cuda_stream))
    if rc:
        raise HPMCError(rc, (L.hpmc_last_error(None) or b"").decode())


class HPMC:
    """One simulation context (hpmc_ctx).  `pos4` / `quat4` are CUDA float32 tensors of shape (N,4), borrowed and
    updated in place; pass pos4=None, N=... for library-owned pose buffers (host-buffer path)."""

    def __init__(self, shape, sigma_c, sigma_d, box_L, d_max_cap, pos4=None, quat4=None, disk_a=0.0, disk_s=0.0,
                 N=None, stream=None):
        import torch
        self.L = load_library()
        self.torch = torch
        self.params = Params(SHAPES[shape] if isinstance(shape, str) else int(shape), sigma_c, disk_a, disk_s,
                             sigma_d, box_L, d_max_cap)
        if pos4 is not None:
            assert pos4.is_cuda and pos4.dtype == torch.float32 and pos4.is_contiguous() and pos4.shape[1] == 4
            N = pos4.shape[0]
            if quat4 is not None:
                assert quat4.is_cuda and quat4.dtype == torch.float32 and quat4.is_contiguous() and quat4.shape == pos4.shape
        self.N = int(N)
        self.pos4, self.quat4 = pos4, quat4           # keep the borrowed tensors alive
        if stream is None and not torch.cuda.is_available():
            raise HPMCError(-5, "no CUDA device: this library has no CPU path")
        s = torch.cuda.current_stream() if stream is None else stream
        self.stream = s
        h = C.c_void_p()
        rc = self.L.hpmc_init(C.byref(h), C.byref(self.params), self.N, _dptr(pos4), _dptr(quat4),
                              C.c_void_p(s.cuda_stream))
        if rc:
            raise HPMCError(rc, (self.L.hpmc_last_error(None) or b"").decode())
        self.h = h
        nc, w = C.c_int32(), C.c_float()
        self._ck(self.L.hpmc_grid(self.h, C.byref(nc), C.byref(w)))
        self.n_c, self.w = nc.value, w.value

    def _ck(self, rc):
        if rc:
            raise HPMCError(rc, (self.L.hpmc_last_error(self.h) or b"").decode())

    def close(self):
        h, self.h = getattr(self, "h", None), None
        if h:
            self.L.hpmc_destroy(h)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the calls of include/hpmc.h, same names
    def build_cells(self, seed, step):
        self._ck(self.L.hpmc_build_cells(self.h, seed, step))

    def sweep(self, seed, step, n_R, d_max, a_max=0.0, n_trial=0):
        self._ck(self.L.hpmc_sweep(self.h, seed, step, float(n_R), d_max, a_max, n_trial))

    def free_volume(self, seed, step, n_samples):
        out = C.c_uint64(0)
        self._ck(self.L.hpmc_free_volume(self.h, seed, step, int(n_samples), C.byref(out)))
        return int(out.value)

    def step_host_bytes(self):
        a, b = C.c_int64(0), C.c_int64(0)
        self._ck(self.L.hpmc_step_host_bytes(self.h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def set_options(self, options):
        self._ck(self.L.hpmc_set_options(self.h, int(options)))

    def run(self, seed, step0, n_sweeps, n_R, d_max, a_max=0.0, n_trial=0):
        self._ck(self.L.hpmc_run(self.h, seed, step0, n_sweeps, float(n_R), d_max, a_max, n_trial))

    def counters(self):
        c = Counters()
        self._ck(self.L.hpmc_counters(self.h, C.byref(c)))
        return {n: int(getattr(c, n)) for n in COUNTER_NAMES}

    def reset_counters(self):
        self._ck(self.L.hpmc_reset_counters(self.h))

    def outcomes(self):
        out = self.torch.empty(self.N, dtype=self.torch.uint8, device="cuda")
        self._ck(self.L.hpmc_outcomes(self.h, _dptr(out)))
        return out

    def cells(self):
        cs = self.torch.empty(self.n_c ** 3 + 1, dtype=self.torch.int32, device="cuda")
        cp = self.torch.empty(self.N, dtype=self.torch.int32, device="cuda")
        sh = (C.c_float * 3)()
        self._ck(self.L.hpmc_cells(self.h, _dptr(cs), _dptr(cp), C.byref(sh)))
        return cs, cp, [sh[0], sh[1], sh[2]]

    def upload(self, host_pos4, host_quat4=None):
        self._ck(self.L.hpmc_upload(self.h, _dptr(host_pos4), _dptr(host_quat4)))

    def download(self, host_pos4=None, host_quat4=None, host_outcome=None):
        self._ck(self.L.hpmc_download(self.h, _dptr(host_pos4), _dptr(host_quat4), _dptr(host_outcome)))

    def step_host(self, host_pos4, host_quat4, host_outcome, seed, step, n_R, d_max, a_max=0.0, n_trial=0):
        self._ck(self.L.hpmc_step_host(self.h, _dptr(host_pos4), _dptr(host_quat4), _dptr(host_outcome), seed, step,
                                       float(n_R), d_max, a_max, n_trial))

    def launch_count(self):
        return int(self.L.hpmc_launch_count(self.h))

    def time_move_kernel(self, enable=True):
        self._ck(self.L.hpmc_time_move_kernel(self.h, 1 if enable else 0))

    def move_kernel_ms(self):
        ms, n = C.c_double(), C.c_int64()
        self._ck(self.L.hpmc_move_kernel_ms(self.h, C.byref(ms), C.byref(n)))
        return ms.value, n.value
