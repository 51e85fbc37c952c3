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

# Algorithmic work per unit: lane-operations (one thread executing one plain ALU instruction).
OPS_PER_NEEDED_DEPLETANT = 131.0   # 1.91 attempts x (40 INT Philox + 22 convert/scale/|d|^2/compare) + 11 pose tests + ~2 nbr
OPS_PER_MOVE = 500.0               # 3 Philox blocks, 27-cell staging, hard overlap, table search, commit
BYTES_PER_PARTICLE_PER_PASS = 16.0 # every pass reads the cell-ordered float4 array once (re-reads by neighbouring cells are L2 hits)
BYTES_PER_CELL_PER_PASS = 4.0      # ... and each cell_start word once
BYTES_PER_MOVE = 1.0               # outcome code
BYTES_PER_ACCEPT = 48.0
# dram__bytes_read.sum + dram__bytes_write.sum of one move-kernel launch at C3, ncu --set full (profiles/r1f_summary.md:
# 22.50 MB read + 0 written; capture d saw 2.8..4.9 MB of write-backs of the preceding build on top)
NCU_TRAFFIC_BYTES_PER_LAUNCH_C3 = 22.5e6
LANES_PER_SM_PER_CLK = 128.0       # 4 SMSPs x 32 lanes: issue-rate peak of the plain ALU pipes
NUM_SMS = 148


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


def oracle_sample(cfg, pos, quat, sweeps, step0, min_seconds=0.0, max_sweeps=None):
    """Time the CPU oracle, as it stands, on `sweeps` sweeps of the same workload with all host cores; with
    min_seconds > 0 keep adding sweeps until that much CPU wall time has been spent (bounded by max_sweeps)."""
    import oracle
    threads = os.cpu_count() or 1
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


def workload_desc(cfg):
    return ("%s: %d hard %ss, phi_c=%.2f, q=%.2f, phi_d^r=%.2f (lambda=%.0f depletants drawn/move), d_max=%.3g, "
            "a_max=%.3g, n_trial=%d" % (cfg.name, cfg.N, cfg.shape, cfg.phi_c, cfg.q, cfg.phi_d_r[0], cfg.lam, cfg.d_max,
                                        cfg.a_max, cfg.n_trial))


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
        nq = 2 if quat is not None else 1
        e2e = {"value": we / (te * 1e-3), "unit": "moves/s",
               "h2d_bytes_per_step": 16 * cfg.N * nq, "d2h_bytes_per_step": 16 * cfg.N * nq + cfg.N,
               "ms_per_step": te / args.steps}
        hh.close()

    if rank == 0:
        alg_ops = c["dep_needed"] * OPS_PER_NEEDED_DEPLETANT + moves * OPS_PER_MOVE
        alg_bytes = (move_launches * (BYTES_PER_PARTICLE_PER_PASS * cfg.N + BYTES_PER_CELL_PER_PASS * (h.n_c ** 3 + 1))
                     + moves * BYTES_PER_MOVE + (c["accept_trans"] + c["accept_rot"]) * BYTES_PER_ACCEPT)
        move_s = move_ms * 1e-3
        alu_peak = NUM_SMS * LANES_PER_SM_PER_CLK * pk["sm_max_mhz"] * 1e6          # lane-ops/s at max boost clock
        alu_ach = alg_ops / move_s if move_s > 0 else 0.0
        hbm_ach = alg_bytes / move_s / 1e9 if move_s > 0 else 0.0
        t_alu, t_hbm = alg_ops / alu_peak, alg_bytes / (pk["hbm_gbs"] * 1e9)
        roofline = {
            "bound": "alu" if t_alu >= t_hbm else "hbm",
            "achieved": alu_ach / 1e12, "peak": alu_peak / 1e12, "unit": "Tlaneop/s", "frac": alu_ach / alu_peak,
            "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH_C3 if (cfg.name == "C3" and args.n is None) else None,
            "alg_bytes_per_launch": alg_bytes / max(1, move_launches), "alg_laneops_per_launch": alg_ops / max(1, move_launches),
            "kernel": "k_moveq (8 launches per step)", "launches": move_launches,
            "avg_launch_ms": move_ms / max(1, move_launches), "share_of_step": move_ms / total_ms if total_ms else None,
            "peak_source": "derived: 148 SM x 128 lanes/clk x %.0f MHz (DESIGN.md); HBM %s" % (pk["sm_max_mhz"], pk["source"]),
            "hbm": {"achieved": hbm_ach, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": hbm_ach / pk["hbm_gbs"]},
            "alg_ops_per_needed_depletant": OPS_PER_NEEDED_DEPLETANT, "alg_ops_per_move": OPS_PER_MOVE,
        }
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            # bounded sample: about 12 s of oracle time on this box's cores (3 sweeps at least, 2000 at most)
            _, oc, times, threads = oracle_sample(cfg, pos, quat, 3, args.warmup, min_seconds=12.0, max_sweeps=2000)
            ns = len(times)
            om = oc["trials_trans"] + oc["trials_rot"]
            cpu = {"value": om / sum(times), "unit": "moves/s", "cores": threads, "kind": "oracle",
                   "sample": "%d sweeps of the same workload from the same initial poses (%.1f s)" % (ns, sum(times)),
                   "dep_needed_per_s": oc["dep_needed"] / sum(times)}
        line = {
            "metric": "colloid_trial_moves_per_s", "value": g_moves / tot_s, "unit": "moves/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": job_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_desc(cfg), "step": "one sweep = cell build + 8 checkerboard passes",
                       "l2": "flushed between timed steps (512 MiB write)", "parallelism": "replicas x%d" % world,
                       "moves_per_step": g_moves / args.steps / world},
            "depletant_insertions_per_s": {"evaluated": g_eval / tot_s, "needed": g_needed / tot_s, "drawn": g_drawn / tot_s},
            "acceptance": (c["accept_trans"] + c["accept_rot"]) / max(1, moves),
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "wall_s_timed_region": t_wall,
        }
        print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
