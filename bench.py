#!/usr/bin/env python
"""bench.py -- throughput of the implicit-depletant checkerboard trial move on B200 (BASELINE.json metric).

A "step" is one sweep of the whole hot path over the workload: hpmc_build_cells (cell-list build) followed by
hpmc_sweep (the 8 checkerboard passes of the move kernel).  Workload at N=1: BASELINE.json configs[2] (C3), the
configuration north_star's target is quoted on: 1,048,576 hard spheres, phi_c = 0.25, q = 0.05, phi_d^r = 0.30
(~2.8k depletants drawn per move), d_max = 0.05, seeded synthetic input (workloads/).  N > 1: one independent
replica per GPU ("replicas only"), weak scaling, no collective on the data path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C3] [--n N]

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/, as it stands) instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

# Algorithmic work per unit, in lane-operations (one thread executing one plain ALU instruction).  The table is
# frozen in BASELINE.md section 3 (derivation: DESIGN.md section 6); it multiplies the COUNTERS of the timed run
# (dep_needed, trials, cb_reinsertions), never what the kernel happened to execute.
#   per Philox block 40 (10 rounds x (2 wide multiplies + 2 three-input XORs)); per cube-rejection attempt 62 (block +
#   3 x bits->float/scale + |d|^2 + compare); attempts per depletant 6/pi = 1.91
OPS_PER_NEEDED_DEPLETANT = {"sphere": 131.0,      # 1.91 x 62 + old/new pose tests 11 + ~2 neighbour tests
                            "halfball": 167.0,    # + 15 + 15 closed-form new/old tests + 0.07 n_nbr x 25
                            "spherodisk": 167.0,
                            "ellipsoid": 420.0,
                            "tetrahedron": 500.0}  # frame + point-to-tetrahedron distance (one or two faces) for the new and the old pose    # + two point-to-ellipse distances of ~125 ops (6 Newton steps) instead of closed forms
OPS_PER_MOVE = {"sphere": 500.0,                  # 3 Philox blocks, 27-cell walk (~20 candidates x 12 + 9 rows x 8), table search, commit
                "halfball": 1500.0,               # + axis staging, ~2 support-function pair tests of ~400 ops (a6)
                "spherodisk": 1500.0, "ellipsoid": 1500.0, "tetrahedron": 2000.0}
OPS_PER_CB_REINSERTION = {"sphere": 150.0, "halfball": 190.0, "spherodisk": 190.0, "ellipsoid": 440.0, "tetrahedron": 520.0}   # 1.91 x 62 + both pose tests + neighbour tests
# INT / FP32 split of the same totals (lower bound = max(FP / FP rate, INT / INT rate, all / issue rate,
# bytes / HBM)).  Integer work does not depend on the shape: per cube-rejection attempt one Philox block (20 wide
# multiplies + 20 three-input XORs) + 3 bit operations of the bits->float conversion = 43, x 6/pi attempts = 82 per needed
# depletant or reinsertion; per move 3 Philox blocks (120) + ~80 of row addressing and table search = 200.  The rest of
# each total is non-FMA FP32 (differences, products, compares of the overlap tests).  The totals above stay as frozen.
INT_OPS_PER_NEEDED_DEPLETANT = 82.0
INT_OPS_PER_CB_REINSERTION = 82.0
INT_OPS_PER_MOVE = 200.0
PHILOX_BLOCKS_PER_DEPLETANT = 6.0 / 3.141592653589793
BYTES_PER_PARTICLE_PER_PASS = 16.0 # every pass reads the cell-ordered float4 array once (re-reads by neighbouring cells are L2 hits)
BYTES_PER_CELL_PER_PASS = 4.0      # ... and each cell_start word once
BYTES_PER_MOVE = 1.0               # outcome code
BYTES_PER_ACCEPT = 48.0
LANES_PER_SM_PER_CLK = 128.0       # 4 SMSPs x 32 lanes x 1 warp-instruction per clock: the issue bound (kept as peak_issue_bound)
KERNEL_SOURCES = ("moveq.cuh", "move.cuh", "geometry.cuh", "philox.cuh", "cells.cuh", "hpmc_lib.cu")


def kernel_sources_sha():
    """sha256 over the CUDA sources: a stored ncu traffic figure is only quoted while the kernels are unchanged."""
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_1508_07077_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the move kernel from the tracked capture
    profiles/ncu_traffic.json (written from an `ncu --set full` run; names the source hash it was taken at).  None if
    there is no capture of THIS source state for this workload."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(path):
        return None, None
    with open(path) as f:
        d = json.load(f)
    e = d.get(workload)
    if not e or e.get("kernel_sources_sha") != kernel_sources_sha():
        return None, None
    return float(e["dram_bytes_per_launch"]), e.get("source")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--n", type=int, default=None, help="override particle count (debug; invalidates the headline)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the short runs of C1, C2, C4, C5 (per_config)")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f:
            t = [x.strip() for x in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0])); mx.append(float(t[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), t[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}
        return out


def reduce_over_ranks(total_ms, work, device, world):
    """Replicas only: the job's time is the MAX over ranks of the timed duration, its work the SUM over
    ranks.  The one place bench.py talks to torch.distributed besides the barrier; covered by a gloo test on CPU."""
    import torch
    t = torch.tensor([total_ms], dtype=torch.float64, device=device)
    w = torch.tensor(list(work), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(x) for x in w.tolist()]


def oracle_sample(cfg, pos, quat, sweeps, step0, min_seconds=0.0, max_sweeps=None, threads=None):
    """Time the CPU oracle, as it stands, on `sweeps` sweeps of the same workload with all host cores (or `threads`);
    with min_seconds > 0 keep adding sweeps until that much CPU wall time has been spent (bounded by max_sweeps)."""
    import oracle
    threads = threads or os.cpu_count() or 1
    o = oracle.Oracle(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, pos, quat, cfg.disk_a, cfg.disk_s,
                      threads=threads)
    times = []
    s = 0
    while s < sweeps or (sum(times) < min_seconds and (max_sweeps is None or s < max_sweeps)):
        t0 = time.perf_counter()
        o.build_cells(cfg.seed, step0 + s)
        o.sweep(cfg.seed, step0 + s, cfg.n_R(), cfg.d_max, cfg.a_max, cfg.n_trial)
        times.append(time.perf_counter() - t0)
        s += 1
    c = o.counters()
    return o, c, times, oracle.lib().oracle_get_threads()


def workload_desc(cfg, phi=None):
    phi = cfg.phi_d_r[0] if phi is None else phi
    return ("%s: %d hard %ss, phi_c=%.2f, q=%.2f, phi_d^r=%.2f (lambda=%.0f depletants drawn/move), d_max=%.3g, "
            "a_max=%.3g, n_trial=%d" % (cfg.name, cfg.N, cfg.shape, cfg.phi_c, cfg.q, phi, cfg.lam * phi / cfg.phi_d_r[0],
                                        cfg.d_max, cfg.a_max, cfg.n_trial))


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pos, quat = workloads.generate(cfg)
    # warm-up sweeps advance the same trajectory, then K timed sweeps (each step = one full oracle sweep)
    o, c0, tw, threads = oracle_sample(cfg, pos, quat, args.warmup, 0)
    o.reset_counters()
    times = []
    for s in range(args.steps):
        t0 = time.perf_counter()
        o.build_cells(cfg.seed, args.warmup + s)
        o.sweep(cfg.seed, args.warmup + s, cfg.n_R(), cfg.d_max, cfg.a_max, cfg.n_trial)
        times.append(time.perf_counter() - t0)
    c = o.counters()
    total = sum(times)
    moves = c["trials_trans"] + c["trials_rot"]
    val = moves / total
    line = {
        "impl": "reference", "metric": "colloid_trial_moves_per_s", "value": val, "unit": "moves/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_desc(cfg), "step": "one sweep = cell build + 8 checkerboard passes"},
        "depletant_insertions_per_s": {"needed": c["dep_needed"] / total, "drawn": c["dep_drawn"] / total,
                                       "evaluated": c["dep_evaluated"] / total},
        "cpu_baseline": {"value": val, "unit": "moves/s", "cores": threads, "kind": "oracle",
                         "sample": "%d full sweeps of the same workload, OpenMP over active cells" % args.steps},
        "e2e": {"value": val, "unit": "moves/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def roofline_block(cfg, c, n_c, passes, launches, kernel_ms, step_ms_total, alu, pk, clocks, workload_key):
    """Roofline of the move kernel (K-B) from the counters `c` of the timed run and its event-timed duration.
    The lower bound on its time is the larger of (a) the Philox blocks the algorithm needs divided by the MEASURED
    block rate of the SMs (the wide-multiply pipe binds a Philox stream: hpmc_alu_peaks) and (b) all algorithmic
    lane-operations divided by the measured two-pipe issue rate; `peak` is the lane-op rate that bound corresponds to."""
    moves = c["trials_trans"] + c["trials_rot"]
    alg_ops = (c["dep_needed"] * OPS_PER_NEEDED_DEPLETANT[cfg.shape] + moves * OPS_PER_MOVE[cfg.shape]
               + c["cb_reinsertions"] * OPS_PER_CB_REINSERTION[cfg.shape])
    blocks = ((c["dep_needed"] + c["cb_reinsertions"]) * PHILOX_BLOCKS_PER_DEPLETANT + 3.0 * moves)
    alg_bytes = (passes * (BYTES_PER_PARTICLE_PER_PASS * cfg.N * (1 if cfg.shape == "sphere" else 2)
                           + BYTES_PER_CELL_PER_PASS * (n_c ** 3 + 1))
                 + moves * BYTES_PER_MOVE + (c["accept_trans"] + c["accept_rot"]) * BYTES_PER_ACCEPT)
    kernel_s = kernel_ms * 1e-3
    sms, hz = alu["num_sms"], pk["sm_max_mhz"] * 1e6
    int_ops = (c["dep_needed"] * INT_OPS_PER_NEEDED_DEPLETANT + moves * INT_OPS_PER_MOVE
               + c["cb_reinsertions"] * INT_OPS_PER_CB_REINSERTION)
    fp_ops = alg_ops - int_ops
    t_philox = blocks / (alu["philox_blocks_ilp4"] * sms * hz)
    t_issue = alg_ops / (alu["fadd_lop3_mix"] * sms * hz)
    t_fp = fp_ops / (min(alu["fadd"], alu["fmul"]) * sms * hz)                 # non-FMA FP32 stream
    t_int = int_ops / (alu["imadwide_lop3_pair"] * sms * hz)                   # IMAD.WIDE + LOP3 stream (the Philox mix)
    t_hbm = alg_bytes / (pk["hbm_gbs"] * 1e9)
    terms = {"fp32": t_fp, "int": t_int, "issue": t_issue, "philox_blocks": t_philox, "hbm": t_hbm}
    binding = max(("fp32", "int", "issue", "philox_blocks"), key=lambda k: terms[k])
    t_alu = terms[binding]
    peak = alg_ops / t_alu
    ach = alg_ops / kernel_s if kernel_s > 0 else 0.0
    hbm_ach = alg_bytes / kernel_s / 1e9 if kernel_s > 0 else 0.0
    issue_peak = sms * LANES_PER_SM_PER_CLK * hz
    seen_mhz = clocks.get("sm_mhz") or pk["sm_max_mhz"]
    traffic, traffic_src = ncu_traffic(workload_key)
    cbk = os.environ.get("HPMC_CB_KERNEL")        # the library's rule (hpmc_lib.cu): item queue iff n_trial >= 16 or N >= 200000
    cb_warp = cfg.n_trial > 0 and (cbk == "warp" or (cbk != "queue" and cfg.n_trial < 16 and cfg.N < 200000))
    kern = ("k_move<%s,cb> (warp per cell, 8 launches per sweep)" % cfg.shape if cb_warp else
            "k_moveq<%s,%s> (item queue, %d launch%s per sweep)" % (cfg.shape, "cb" if cfg.n_trial > 0 else "plain",
                                                                     round(launches / max(1, passes / 8)),
                                                                     "" if launches * 8 == passes else "es"))
    return {
        "bound": "alu" if t_alu >= t_hbm else "hbm",
        "achieved": ach / 1e12, "peak": peak / 1e12, "unit": "Tlaneop/s", "frac": t_alu / kernel_s if kernel_s > 0 else None,
        "frac_cycles": (t_alu * hz) / (kernel_s * seen_mhz * 1e6) if kernel_s > 0 else None,
        "traffic": traffic, "traffic_source": traffic_src,
        "peak_source": "measured live: hpmc_alu_peaks on this device (per SM per clock: %.1f FP32 non-FMA, %.1f IMAD.WIDE+LOP3, "
                       "%.1f two-pipe issue lane-ops, %.3f Philox blocks) x %d SMs x %.0f MHz; binding term: %s; HBM %s" % (
                           min(alu["fadd"], alu["fmul"]), alu["imadwide_lop3_pair"], alu["fadd_lop3_mix"],
                           alu["philox_blocks_ilp4"], sms, pk["sm_max_mhz"], binding, pk["source"]),
        # time lower bound = max over the pipes; every term in microseconds per launch, and the fraction the
        # combined-issue term alone gives (the only ALU term of the round-1 and round-2 lines, kept for comparison)
        "binding_term": binding,
        "terms_us_per_launch": {k: 1e6 * v / max(1, launches) for k, v in terms.items()},
        "frac_issue_term_only": t_issue / kernel_s if kernel_s > 0 else None,
        "alg_int_laneops_per_launch": int_ops / max(1, launches), "alg_fp32_laneops_per_launch": fp_ops / max(1, launches),
        "peak_issue_bound": issue_peak / 1e12, "frac_of_issue_bound": ach / issue_peak,
        "alg_laneops_per_launch": alg_ops / max(1, launches), "alg_philox_blocks_per_launch": blocks / max(1, launches),
        "alg_bytes_per_launch": alg_bytes / max(1, launches),
        "kernel": kern, "launches": launches, "passes": passes, "avg_launch_ms": kernel_ms / max(1, launches),
        "us_per_pass": 1e3 * kernel_ms / max(1, passes),
        "share_of_step": kernel_ms / step_ms_total if step_ms_total else None,
        "hbm": {"achieved": hbm_ach, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": hbm_ach / pk["hbm_gbs"]},
        "alg_ops_per_needed_depletant": OPS_PER_NEEDED_DEPLETANT[cfg.shape], "alg_ops_per_move": OPS_PER_MOVE[cfg.shape],
        "alg_ops_per_cb_reinsertion": OPS_PER_CB_REINSERTION[cfg.shape],
    }


def timed_run(hp, torch, cfg, seed, pos, quat, n_R, steps, warmup, flush, step0=0, options=0, free_volume_samples=0):
    """`warmup` untimed + `steps` timed sweeps of one configuration from the given poses; returns the counters of the
    timed sweeps, per-step event times, the move kernel's event time and launch count, the grid size, the poses before
    and after the timed sweeps and (free_volume_samples > 0) the free-volume fraction of the final configuration."""
    dpos = torch.from_numpy(pos.copy()).cuda()
    dquat = None if quat is None else torch.from_numpy(quat.copy()).cuda()
    h = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, dpos, dquat, cfg.disk_a, cfg.disk_s)
    if options:
        h.set_options(options)

    def step(s):
        h.build_cells(seed, s)
        h.sweep(seed, s, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)

    for s in range(warmup):
        step(step0 + s)
    torch.cuda.synchronize()
    start_pos = dpos.cpu().numpy()
    h.reset_counters()
    l0 = h.launch_count()
    h.time_move_kernel(True)
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    torch.cuda.synchronize()
    for k in range(steps):
        if flush is not None:
            flush.zero_()                  # evict the working set from L2 between timed steps (not timed)
        starts[k].record()
        step(step0 + warmup + k)
        ends[k].record()
    torch.cuda.synchronize()
    step_ms = [a.elapsed_time(b) for a, b in zip(starts, ends)]
    kms, kl = h.move_kernel_ms()
    h.time_move_kernel(False)
    c = h.counters()
    out = dict(c=c, step_ms=step_ms, kernel_ms=kms, kernel_launches=kl, launches=h.launch_count() - l0, n_c=h.n_c,
               start_pos=start_pos, final_pos=dpos.cpu().numpy(), final_quat=None if dquat is None else dquat.cpu().numpy())
    if free_volume_samples:
        s_fv = step0 + warmup + steps
        h.build_cells(seed, s_fv)
        out["free_volume_fraction"] = h.free_volume(seed, s_fv, free_volume_samples) / free_volume_samples
    h.close()
    return out


def per_config_lines(hp, torch, alu, pk, flush, clocks):
    """moves/s, depletant insertions/s, us per pass and roofline fraction of the other BASELINE.json configurations
    (C1, C2 at its four reservoir densities after melting 1000 sweeps at n_R = 0 through the library, C4, C5), of the two
    NEXT-2 shapes (C6 ellipsoids with n_trial = 10, C7 tetrahedra) and of C3 with the shell option, each a short
    device-timed run from its seeded initial state.  Context for the C3 headline, same kernels, same clocks."""
    import numpy as np
    out = {}
    plan = [("C1", 200, 0), ("C2", 50, 0), ("C4", 50, 0), ("C5", 50, 0), ("C6", 50, 0), ("C7", 50, 0), ("C3", 10, hp.OPT_SHELL)]
    for name, steps, options in plan:
        cfg = workloads.config(name)
        pos, quat = workloads.generate(cfg)
        dens = [(None, cfg.n_R())]
        if name == "C2":
            m = timed_run(hp, torch, cfg, cfg.seed, pos, quat, 0.0, 1000, 0, None, step0=100000)   # melt (configs[1])
            pos = m["final_pos"]
            dens = [(phi, cfg.n_R(phi)) for phi in cfg.phi_d_r]
        for phi, n_R in dens:
            r = timed_run(hp, torch, cfg, cfg.seed, pos, quat, n_R, steps, 5, flush, options=options,
                          free_volume_samples=1000000)
            c = r["c"]
            tot_s = sum(r["step_ms"]) * 1e-3
            moves = c["trials_trans"] + c["trials_rot"]
            rf = roofline_block(cfg, c, r["n_c"], 8 * steps, r["kernel_launches"], r["kernel_ms"], sum(r["step_ms"]), alu, pk,
                                clocks, name if not options else None)
            # mean-square displacement over the timed sweeps per wall-clock second (Fig. 8's figure of merit, L240)
            dr = (r["final_pos"][:, :3].astype(np.float64) - r["start_pos"][:, :3].astype(np.float64))
            dr -= cfg.box_L * np.round(dr / cfg.box_L)
            msd = float((dr ** 2).sum(axis=1).mean())
            key = name if phi is None else "%s phi_d^r=%.1f" % (name, phi)
            if options:
                key += " HPMC_OPT_SHELL"
            out[key] = {
                "workload": workload_desc(cfg, phi) + (" + HPMC_OPT_SHELL (R-N1)" if options else ""),
                "moves_per_s": moves / tot_s, "dep_needed_per_s": c["dep_needed"] / tot_s,
                "dep_evaluated_per_s": c["dep_evaluated"] / tot_s, "dep_drawn_per_s": c["dep_drawn"] / tot_s,
                "ms_per_step": 1e3 * tot_s / steps, "us_per_pass": rf["us_per_pass"], "acceptance":
                (c["accept_trans"] + c["accept_rot"]) / max(1, moves), "roofline_frac": rf["frac"],
                "frac_of_issue_bound": rf["frac_of_issue_bound"], "kernel": rf["kernel"], "steps": steps,
                "dep_needed_per_move": c["dep_needed"] / max(1, moves), "dep_drawn_per_move": c["dep_drawn"] / max(1, moves),
                "free_volume_fraction": r.get("free_volume_fraction"), "msd_per_s": msd / tot_s, "msd_per_sweep": msd / steps,
            }
    return out


def main():
    args = parse_args()
    cfg = workloads.config(args.workload, args.n)
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    import paper_1508_07077_b200 as hp

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pk = peaks()
    hp.alu_peaks()                         # warm-up of the micro-benchmark (clocks, instruction cache)
    alu = hp.alu_peaks()                   # measured ALU pipe rates of THIS device (per SM per clock)

    # replicas only: every rank runs the same configuration from its own seeded input
    import dataclasses
    rcfg = dataclasses.replace(cfg, seed=cfg.seed + rank)
    pos, quat = workloads.generate(rcfg)
    dpos = torch.from_numpy(pos.copy()).cuda()
    dquat = None if quat is None else torch.from_numpy(quat.copy()).cuda()
    h = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, dpos, dquat, cfg.disk_a, cfg.disk_s)
    n_R = cfg.n_R()
    flush = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step(s):
        h.build_cells(rcfg.seed, s)
        h.sweep(rcfg.seed, s, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for s in range(args.warmup):
        step(s)
    torch.cuda.synchronize()
    h.reset_counters()
    launches0 = h.launch_count()
    h.time_move_kernel(True)
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    barrier()
    sampler = ClockSampler(local)
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                      # evict the working set from L2 between timed steps (not timed)
        starts[k].record()
        step(args.warmup + k)
        ends[k].record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in zip(starts, ends)]
    total_ms = sum(step_ms)
    move_ms, move_launches = h.move_kernel_ms()
    h.time_move_kernel(False)
    c = h.counters()
    launches = h.launch_count() - launches0
    moves = c["trials_trans"] + c["trials_rot"]

    # max over ranks of the timed duration, sum over ranks of the work
    job_ms, (g_moves, g_eval, g_needed, g_drawn) = reduce_over_ranks(
        total_ms, [moves, c["dep_evaluated"], c["dep_needed"], c["dep_drawn"]], "cuda", world)
    tot_s = job_ms * 1e-3

    # ---- SURVEY 8(d) / BASELINE.md 3: the same sweep repeated from IDENTICAL initial poses (identical work every time),
    # median of the event times; `value` above stays the base contract's K consecutive sweeps of one trajectory
    reps = None
    if world == 1:
        n_rep, n_skip = 7, 2
        pos_ref = torch.from_numpy(pos.copy()).cuda()
        quat_ref = None if quat is None else torch.from_numpy(quat.copy()).cuda()
        h.reset_counters()
        ra = [torch.cuda.Event(enable_timing=True) for _ in range(n_rep + n_skip)]
        rb = [torch.cuda.Event(enable_timing=True) for _ in range(n_rep + n_skip)]
        for r in range(n_rep + n_skip):
            dpos.copy_(pos_ref)
            if dquat is not None:
                dquat.copy_(quat_ref)
            flush.zero_()
            ra[r].record()
            step(0)
            rb[r].record()
        torch.cuda.synchronize()
        cr = h.counters()
        rep_ms = sorted(a.elapsed_time(b) for a, b in zip(ra[n_skip:], rb[n_skip:]))
        rep_moves = (cr["trials_trans"] + cr["trials_rot"]) / (n_rep + n_skip)
        med = statistics.median(rep_ms)
        reps = {"n": n_rep, "untimed_first": n_skip, "sweep": "step 0 from the seeded initial poses, poses restored before every repetition",
                "ms_median": med, "ms_min": rep_ms[0], "ms_max": rep_ms[-1], "moves_per_repetition": rep_moves,
                "moves_per_s_median": rep_moves / (med * 1e-3)}

    # ---- e2e: the same step through the host-buffer C-ABI call, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hh = hp.HPMC(cfg.shape, cfg.sigma_c, cfg.sigma_d, cfg.box_L, cfg.d_max, None, None, cfg.disk_a, cfg.disk_s, N=cfg.N)
        hpos = torch.from_numpy(pos.copy()).pin_memory()
        hquat = None if quat is None else torch.from_numpy(quat.copy()).pin_memory()
        hout = torch.zeros(cfg.N, dtype=torch.uint8).pin_memory()
        for s in range(args.warmup):
            hh.step_host(hpos, hquat, hout, rcfg.seed, s, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)
        hh.reset_counters()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(args.steps):
            hh.step_host(hpos, hquat, hout, rcfg.seed, args.warmup + k, n_R, cfg.d_max, cfg.a_max, cfg.n_trial)
        e1.record()
        barrier()
        ce = hh.counters()
        te, (we,) = reduce_over_ranks(e0.elapsed_time(e1), [ce["trials_trans"] + ce["trials_rot"]], "cuda", world)
        # bytes the library really moved in the last step: whole pose arrays up; outcome codes and, when few particles
        # moved, only the accepted particles' poses down (hpmc_step_host's sparse download), else the whole arrays
        h2d, d2h = hh.step_host_bytes()
        e2e = {"value": we / (te * 1e-3), "unit": "moves/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "ms_per_step": te / args.steps,
               "note": "d2h = outcome codes (N bytes) + list and poses of the accepted particles (sparse download)"}
        hh.close()

    if rank == 0:
        wkey = cfg.name if args.n is None else None
        roofline = roofline_block(cfg, c, h.n_c, 8 * args.steps, move_launches, move_ms, total_ms, alu, pk, clocks, wkey)
        per_config = None
        if not args.no_per_config and world == 1 and cfg.name == "C3" and args.n is None:
            per_config = per_config_lines(hp, torch, alu, pk, flush, clocks)
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            # bounded sample: about 12 s of oracle time on this box's cores (3 sweeps at least, 2000 at most)
            _, oc, times, threads = oracle_sample(cfg, pos, quat, 3, args.warmup, min_seconds=12.0, max_sweeps=2000)
            ns = len(times)
            om = oc["trials_trans"] + oc["trials_rot"]
            cpu = {"value": om / sum(times), "unit": "moves/s", "cores": threads, "kind": "oracle",
                   "sample": "%d sweeps of the same workload from the same initial poses (%.1f s)" % (ns, sum(times)),
                   "dep_needed_per_s": oc["dep_needed"] / sum(times)}
            # the same oracle on ONE core (SURVEY 8(d) "Oracle timing" (i)): two sweeps from the same initial poses
            _, oc1, t1, th1 = oracle_sample(cfg, pos, quat, 2, args.warmup, threads=1)
            cpu["single_thread"] = {"value": (oc1["trials_trans"] + oc1["trials_rot"]) / sum(t1), "unit": "moves/s",
                                    "cores": th1, "dep_needed_per_s": oc1["dep_needed"] / sum(t1),
                                    "sample": "%d sweeps (%.1f s)" % (len(t1), sum(t1))}
        line = {
            "metric": "colloid_trial_moves_per_s", "value": g_moves / tot_s, "unit": "moves/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": job_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_desc(cfg), "step": "one sweep = cell build + 8 checkerboard passes",
                       "l2": "flushed between timed steps (512 MiB write)", "parallelism": "replicas x%d" % world,
                       "moves_per_step": g_moves / args.steps / world},
            "depletant_insertions_per_s": {"evaluated": g_eval / tot_s, "needed": g_needed / tot_s, "drawn": g_drawn / tot_s},
            "acceptance": (c["accept_trans"] + c["accept_rot"]) / max(1, moves),
            "roofline": roofline, "alu_peaks_per_sm_per_clk": alu, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches, "clocks": clocks, "per_config": per_config, "wall_s_timed_region": t_wall,
            "repetitions": reps,
        }
        print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
