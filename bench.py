#!/usr/bin/env python
"""bench.py -- throughput of the g(3) hot path (libg3, include/g3.h) on BASELINE.json's headline
workload: config 4, N = 32768 water-like sites, 500 frames, r_max = 0.7 nm, 64^3 bins.

A "step" is one pass of the WHOLE hot path (quantise, cell list, neighbour lists, triplet
histogram, merge, normalise: SURVEY.md 8(a) rows a1..a6) over one seeded synthetic trajectory
of `--frames` frames (default: the workload's 500).  The metric is distinct triplets binned per
second (frames/s is reported beside it).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--frames F]

Prints ONE JSON line (rank 0).  `value` is device-timed with positions resident in HBM; `e2e` is
the same step through the C ABI's host entry points (pinned host positions in, host results out,
copies inside the timed region).  `roofline` and `cpu_baseline` are described in DESIGN.md 6.
With --gpus N > 1 every rank processes its own trajectory of the same shape (frames are
independent; "split the trajectory, merge the results"): weak
scaling, no data-path collective; --shard-one-trajectory instead splits the ONE seeded trajectory
over the ranks with sharding.frame_shard (strong scaling).  Run as `python bench.py --gpus N`
(no torchrun) it launches the N ranks itself through torch.distributed.run on 127.0.0.1.
"""
from __future__ import annotations

import argparse
import json
import os
import re
import socket
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import WORKLOADS, frame_iter, grid_to_pos  # noqa: E402

METRIC = "g3_distinct_triplets_binned_per_s"
UNIT = "triplets/s"
WORKLOAD_INDEX = 4
ALGO_INSTR_PER_TRIPLET = 12          # fixed algorithmic instruction count
SM_LANES = 128                       # 4 schedulers x 32 lanes, one warp instruction per cycle each
def ncu_lsu_busy(kernel: str):
    """`l1tex__data_pipe_lsu_wavefronts` (% of peak) of `kernel` from its ncu summary under profiles/:
    the shared-memory data pipe is what binds both hot kernels; None if absent."""
    path = os.path.join(ROOT, "profiles", TRAFFIC_PROFILES.get(kernel, ""))
    try:
        m = re.search(r"l1tex__data_pipe_lsu_wavefronts\.avg\.pct_of_peak_sustained_elapsed`\) \| ([0-9.]+) %", open(path).read())
    except OSError:
        return None
    return float(m.group(1)) / 100.0 if m else None


ALGO_INSTR_PER_DISPLACEMENT = 9       # MSD: 3 subtractions, 3 multiply-adds, one 128-bit accumulate
ALGO_INSTR_PER_QTET_ATOM = 210        # q_tet: exact keys + top-4 insertion of ~6 list-head entries (150) + Eq. 1 in fp64 (60)
# wide g2: per candidate pair the second pair search tests (3 coordinate differences, 3 multiply-adds,
# 1 comparison with the cut-off) and, per pair that lands in [r_max, 2 r_max), 2 for the shell and 1 add
ALGO_INSTR_PER_G2W_CANDIDATE = 7
ALGO_INSTR_PER_G2W_HIT = 3


def g2w_candidate_pairs(pos_frame: np.ndarray, box: float, ncell: int) -> int:
    """Unordered candidate pairs the wide-g2 search of one frame has to test on an ncell^3 grid: a
    particle against the later members of its own cell and against the 62 cells of the forward half
    of the 5x5x5 stencil (every pair within 2 r_max once).  Counted from the cell
    occupancies of the frame, on the host, outside every timed region."""
    m = np.rint(pos_frame * (1048576.0 / box)).astype(np.int64) % 1048576
    cid = (m * ncell) >> 20
    occ = np.zeros((ncell, ncell, ncell), dtype=np.int64)
    np.add.at(occ, (cid[:, 0], cid[:, 1], cid[:, 2]), 1)
    total = int((occ * (occ - 1) // 2).sum())
    for dx in range(-2, 3):
        for dy in range(-2, 3):
            for dz in range(-2, 3):
                if (dx, dy, dz) > (0, 0, 0):
                    total += int((occ * np.roll(occ, (-dx, -dy, -dz), axis=(0, 1, 2))).sum())
    return total


TRAFFIC_PROFILES = {"tiled_triplet_kernel": "r3_triplet_kernel.md", "neighbour_cell_kernel": "r3_neighbour_kernel.md"}


def ncu_traffic(kernel: str, frames_per_launch: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, read from the ncu
    summary committed under profiles/ (a line `traffic: dram_bytes_per_launch=<B> frames_per_launch=<F>`).
    None when the file is missing or was captured at another batch size."""
    path = os.path.join(ROOT, "profiles", TRAFFIC_PROFILES.get(kernel, ""))
    try:
        m = re.search(r"dram_bytes_per_launch=([0-9.eE+]+)\s+frames_per_launch=(\d+)", open(path).read())
    except OSError:
        return None, None
    if not m or int(m.group(2)) != frames_per_launch:
        return None, os.path.relpath(path, ROOT)
    return float(m.group(1)), os.path.relpath(path, ROOT)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return d, "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.1 and len(r) >= 7] or \
               [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower() == "active" for r in rows)]

        def num(s):
            try:
                return float(s)
            except ValueError:
                return float("nan")
        return {"sm_mhz": statistics.median(num(r[0]) for r in rows), "sm_max_mhz": num(rows[0][1]),
                "power_w_max": max(num(r[2]) for r in rows), "samples": len(rows), "reasons": reasons}


def make_positions(w, n_frames: int, rank: int) -> np.ndarray:
    """fp64 [F, n, 3] seeded synthetic frames (workloads/frames.py); rank r > 0 gets its own seed."""
    ms = list(frame_iter(w, n_frames, seed=w.seed + 1000 * rank))
    return grid_to_pos(np.stack(ms, axis=0), w.box)


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline_leg(w, budget_s: float = 15.0):
    """The oracle as it stands (oracle/g3_oracle.c, cell-grid routine, OpenMP over centres) on a
    bounded sample of the same workload: whole frames (generated BEFORE the clock starts) until
    ~budget_s of wall time on all host cores, then one frame on ONE thread (the analogue of the
    paper's serial code)."""
    import oracle
    oracle.build()
    T_r, T_t = oracle.thresholds(w.box, w.r_max, w.n_r, w.n_t)
    cores = oracle.num_threads()
    # how many frames fit the budget: time one, then generate the sample up front
    ms = list(frame_iter(w, 2))
    H = np.zeros((w.n_r, w.n_r, w.n_t), dtype=np.uint64)
    stats = np.zeros(3, dtype=np.uint64)
    t0 = time.perf_counter()
    oracle.frame_cells(ms[0], T_r, T_t, H, stats)
    per_frame = max(time.perf_counter() - t0, 1e-3)
    n_sample = int(min(w.n_frames, max(2, budget_s / per_frame)))
    ms = list(frame_iter(w, n_sample))
    H[:] = 0
    stats[:] = 0
    t0 = time.perf_counter()
    for m in ms:
        oracle.frame_cells(m, T_r, T_t, H, stats)
    dt = time.perf_counter() - t0
    triplets = int(stats[1]) // 2
    # single thread, one frame
    oracle.set_num_threads(1)
    H1 = np.zeros_like(H)
    s1 = np.zeros(3, dtype=np.uint64)
    t0 = time.perf_counter()
    oracle.frame_cells(ms[0], T_r, T_t, H1, s1)
    dt1 = time.perf_counter() - t0
    oracle.set_num_threads(cores)
    return {"value": triplets / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n_sample} frame(s) of {w.name} ({triplets} distinct triplets), frames generated "
                      f"before the timed region, {dt:.1f} s wall",
            "frames_per_s": n_sample / dt, "cpu_model": cpu_model(), "nproc": os.cpu_count(),
            "single_thread": {"value": (int(s1[1]) // 2) / dt1, "unit": UNIT, "cores": 1,
                              "sample": f"frame 0 of {w.name} ({int(s1[1]) // 2} distinct triplets), {dt1:.1f} s wall"}}


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores, same metric and config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = WORKLOADS[WORKLOAD_INDEX]
    import oracle
    oracle.build()
    T_r, T_t = oracle.thresholds(w.box, w.r_max, w.n_r, w.n_t)
    frames_per_step = max(1, args.ref_frames)
    need = frames_per_step * (args.steps + args.warmup)
    ms = list(frame_iter(w, min(need, w.n_frames)))
    H = np.zeros((w.n_r, w.n_r, w.n_t), dtype=np.uint64)
    stats = np.zeros(3, dtype=np.uint64)
    V = oracle.volumes(w.r_max, w.n_r, w.n_t)
    k = 0

    def step():
        nonlocal k
        for _ in range(frames_per_step):
            oracle.frame_cells(ms[k % len(ms)], T_r, T_t, H, stats)
            k += 1
        oracle.normalise(H, V, int(stats[0]), w.n, w.box)

    for _ in range(args.warmup):
        step()
    before = int(stats[1])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    triplets = (int(stats[1]) - before) // 2
    value = triplets / dt
    sample = f"{frames_per_step} frame(s) of {w.name} per step ({triplets // args.steps} distinct triplets)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
        "data": "synthetic", "frames_per_s": frames_per_step * args.steps / dt,
        "config": {"workload": f"config4 {w.name}: N={w.n}, L={w.box}, r_max={w.r_max}, "
                               f"{w.n_r}x{w.n_r}x{w.n_t} bins; bounded sample: {sample}"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(),
                         "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def other_configs_leg(g3, torch, stream, peak_tinstr, steps: int):
    """"also reported for the other four configs".  Whole path (a1..a6), device
    resident, full BASELINE.json sizes, CUDA events; one warm-up step, then `steps` timed ones."""
    out = {}
    for widx in (1, 2, 3, 5):
        w = WORKLOADS[widx]
        try:
            d_pos = torch.from_numpy(make_positions(w, w.n_frames, 0)).cuda()
            with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t) as plan:
                def step():
                    plan.reset()
                    plan.accumulate_frames(d_pos)
                    return plan.finalize()
                step()
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                for _ in range(steps):
                    _, _, stats = step()
                e1.record(stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / steps
                triplets = (stats[1] + stats[2]) // 2
                out[f"config{widx}"] = {
                    "workload": f"{w.name}: N={w.n}, L={w.box}, r_max={w.r_max}, {w.n_r}x{w.n_r}x{w.n_t} bins, "
                                f"{w.n_frames} frames",
                    "value": triplets / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": steps,
                    "frames_per_s": w.n_frames / (ms * 1e-3), "triplets_per_step": triplets,
                    "whole_step_frac": triplets / (ms * 1e-3) * ALGO_INSTR_PER_TRIPLET / 1e12 / peak_tinstr,
                    "batch_frames": plan.info(g3.G3_INFO_BATCH_FRAMES), "slabs": plan.info(g3.G3_INFO_SLABS),
                    "kernel": plan.info(g3.G3_INFO_KERNEL), "cells_per_edge": plan.info(g3.G3_INFO_CELLS_PER_EDGE),
                    "max_neighbours": plan.info(g3.G3_INFO_MAX_NEIGHBOURS)}
            del d_pos
            torch.cuda.empty_cache()
        except Exception as e:  # the headline numbers stay valid
            out[f"config{widx}"] = {"error": str(e)}
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libg3 has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_1708_08619_b200 import build
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    import paper_1708_08619_b200 as g3
    from paper_1708_08619_b200.sharding import merge_counts

    w = WORKLOADS[WORKLOAD_INDEX]
    F_total = args.frames or w.n_frames
    if args.shard_one_trajectory:                                     # strong scaling: one trajectory, frames split
        from paper_1708_08619_b200.sharding import frame_shard
        f0, f1 = frame_shard(F_total, rank, world)
        pos = make_positions(w, F_total, 0)[f0:f1]
    else:                                                             # weak scaling: one trajectory per rank
        pos = make_positions(w, F_total, rank)                        # fp64 [F, n, 3]
    F = pos.shape[0]
    h_pos = torch.from_numpy(np.ascontiguousarray(pos)).pin_memory()
    d_pos = h_pos.cuda(non_blocking=True)
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()

    free_before = torch.cuda.mem_get_info()[0]
    plan = g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, timing=True,
                   batch_frames=args.batch_frames or None, triplet_warps=args.triplet_warps or None)

    def step_device():
        plan.reset()
        plan.accumulate_frames(d_pos)
        counts, _, stats = plan.finalize(want_g3=False)
        if world > 1:
            counts = merge_counts(counts)            # one sum of the 2 MiB histogram per run
        frames_all = stats[0]
        if world > 1:
            from paper_1708_08619_b200.sharding import merge_frames
            frames_all = merge_frames(stats[0], device="cuda")
        g = plan.normalize(counts, frames_all)
        return counts, g, stats

    def step_host():
        plan.reset()
        plan.accumulate_frames_host(h_pos)
        return plan.finalize_host()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        """(ms per step as the max over ranks, last result); CUDA events on the launching stream."""
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.time()
        e0.record(stream)
        out = None
        for _ in range(steps):
            out = fn()
        e1.record(stream)
        barrier()
        t1 = time.time()
        ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item()) / steps, out, t0, t1

    # the first step configures the plan (buffers sized for one batch, tables, memsets): its wall
    # time and the device memory the plan then holds are reported, outside the timed region
    t_first = time.time()
    step_device()
    torch.cuda.synchronize()
    plan_info = {"first_step_ms": (time.time() - t_first) * 1e3,
                 "device_bytes": int(free_before - torch.cuda.mem_get_info()[0]),
                 "note": "free device memory before g3_plan_create minus after the first step "
                         "(neighbour lists of one batch dominate; include/g3.h G3_OPT_BATCH_FRAMES)"}
    for _ in range(max(args.warmup, 3) - 1):
        step_device()
    plan.clear_timing()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    ms_dev, (counts, g, stats), t0, t1 = timed(step_device, args.steps)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    launches = plan.info(g3.G3_INFO_KERNEL_LAUNCHES) // args.steps
    tri_ns = plan.info(g3.G3_INFO_TRIPLET_NS)
    nb_ns = plan.info(g3.G3_INFO_NEIGHBOUR_NS)
    tri_launches = plan.info(g3.G3_INFO_TIMED_LAUNCHES)
    triplets_rank = (stats[1] + stats[2]) // 2                         # distinct triplets per step
    tot = torch.tensor([triplets_rank], dtype=torch.int64, device="cuda")
    if world > 1:
        dist.all_reduce(tot)
    triplets_all = int(tot.item())
    frames_all_ranks = F_total if args.shard_one_trajectory else F * world

    for _ in range(2):
        step_host()
    ms_e2e, (h_counts, h_g3, h_stats), _, _ = timed(step_host, args.steps)
    assert h_stats[1] == stats[1], "host and device entry points disagree"

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    pk, pk_kind = peaks()
    sm_count = plan.info(g3.G3_INFO_SM_COUNT)
    sm_hz = float(pk.get("sm_max_mhz", 1965.0)) * 1e6
    peak_tinstr = sm_count * SM_LANES * sm_hz / 1e12
    tri_s = tri_ns * 1e-9 / max(tri_launches, 1)                       # avg triplet-kernel launch
    trip_per_launch = triplets_rank * args.steps / max(tri_launches, 1)
    achieved = trip_per_launch * ALGO_INSTR_PER_TRIPLET / tri_s / 1e12 if tri_s > 0 else 0.0
    batch = plan.info(g3.G3_INFO_BATCH_FRAMES)
    tri_traffic, tri_traffic_src = ncu_traffic("tiled_triplet_kernel", batch)
    nb_traffic, _ = ncu_traffic("neighbour_cell_kernel", batch)
    alg_bytes_per_launch = min(batch, F) * w.n * 24              # N x 24 B of positions per frame
    roofline = {
        "bound": "alu", "kernel": "tiled_triplet_kernel", "achieved": achieved, "peak": peak_tinstr,
        "unit": "Tinstr/s", "frac": achieved / peak_tinstr,
        "traffic": tri_traffic,
        "traffic_unit": f"bytes of DRAM traffic per launch (ncu --set full, {tri_traffic_src})",
        "traffic_algorithmic_bytes": alg_bytes_per_launch,
        "neighbour_kernel_traffic": nb_traffic,
        "lsu_data_pipe_busy_ncu": {"tiled_triplet_kernel": ncu_lsu_busy("tiled_triplet_kernel"),
                                   "neighbour_cell_kernel": ncu_lsu_busy("neighbour_cell_kernel"),
                                   "note": "both hot kernels are bound by the shared-memory data pipe "
                                           "(atomics + operand loads), not by issue slots: DESIGN.md 6"},
        "peak_kind": f"{sm_count} SMs x {SM_LANES} lanes x sm_max_mhz ({pk_kind}); DESIGN.md 6",
        "algorithmic_instr_per_triplet": ALGO_INSTR_PER_TRIPLET,
        "triplets_per_launch": trip_per_launch, "kernel_ms_per_launch": tri_s * 1e3,
        "kernel_launches_per_step": tri_launches / args.steps,
        "kernel_share_of_step": tri_ns * 1e-6 / args.steps / ms_dev,
        "neighbour_kernel_share_of_step": nb_ns * 1e-6 / args.steps / ms_dev,
        "kernel_triplets_per_s": trip_per_launch / tri_s if tri_s > 0 else 0.0,
        "whole_step_frac": triplets_rank / (ms_dev * 1e-3) * ALGO_INSTR_PER_TRIPLET / 1e12 / peak_tinstr,
        "neighbour_kernel_ms_per_launch": nb_ns * 1e-6 / max(tri_launches, 1),
        "hbm_gbs_achieved_step": F * w.n * 24 / (ms_dev * 1e-3) / 1e9,
        "hbm_gbs_peak": pk.get("hbm_gbs"),
    }
    # the two candidate ceilings measured live on this GPU (g3_microbench): the
    # shared-atomic rate for random slots of a tile as large as the kernel's, and the issue rate
    atomic_rate = g3.microbench(0, min(plan.info(g3.G3_INFO_TILE_BINS), 56000), 1 << 15)
    issue_rate = g3.microbench(1, 0, 1 << 18)
    roofline.update({
        "shared_atomic_per_s_measured": atomic_rate,
        "frac_of_shared_atomic_ceiling": roofline["kernel_triplets_per_s"] / atomic_rate,
        "issue_tinstr_per_s_measured": issue_rate / 1e12,
        "binding_ceiling_triplets_per_s": min(atomic_rate, issue_rate / ALGO_INSTR_PER_TRIPLET),
        "frac_of_binding_ceiling": roofline["kernel_triplets_per_s"]
                                   / min(atomic_rate, issue_rate / ALGO_INSTR_PER_TRIPLET),
    })
    # q_tet on the same cell list, timed as the EXTRA cost over the g3 path
    # (same trajectory, a second plan with G3_OPT_QTET_BINS on; the difference of two device times)
    qtet = None
    try:
        if world > 1:
            raise RuntimeError("measured at --gpus 1 only")
        with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, qtet_bins=200) as qplan:
            def step_q():
                qplan.reset()
                qplan.accumulate_frames(d_pos)
                qplan.finalize(want_g3=False)
                return qplan.finalize_qtet()
            step_q()
            ms_q, (qh, qs), _, _ = timed(step_q, 2)
            extra = max(ms_q - ms_dev, 1e-6)
            rate = qs[0] / (extra * 1e-3)
            qtet = {"atoms_binned_per_step": qs[0], "extra_ms_per_step": extra,
                    "atoms_per_s_extra": rate, "bins": 200,
                    "roofline": {"bound": "alu", "unit": "Tinstr/s", "peak": peak_tinstr,
                                 "algorithmic_instr_per_atom": ALGO_INSTR_PER_QTET_ATOM,
                                 "achieved": rate * ALGO_INSTR_PER_QTET_ATOM / 1e12,
                                 "frac": rate * ALGO_INSTR_PER_QTET_ATOM / 1e12 / peak_tinstr}}
    except Exception as e:  # the g3 numbers above stay valid
        qtet = {"error": str(e)}
    # g2 over the whole r_jk range [0, 2 r_max) (G3_OPT_G2_WIDE), timed as the
    # EXTRA cost of its second pair search over the g3 path
    g2w = None
    try:
        if world > 1:
            raise RuntimeError("measured at --gpus 1 only")
        with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, g2_wide=True) as gplan:
            def step_g():
                gplan.reset()
                gplan.accumulate_frames(d_pos)
                gplan.finalize(want_g3=False)
                return gplan.finalize_g2()
            step_g()
            ms_g, (c2w, _), _, _ = timed(step_g, 2)
            extra = max(ms_g - ms_dev, 1e-6)
            pairs = int(c2w.cpu().numpy().view(np.uint64)[w.n_r:].sum())
            g2w = {"shells": 2 * w.n_r, "extra_ms_per_step": extra, "outer_ordered_pairs_per_step": pairs,
                   "outer_pairs_per_s_extra": pairs / (extra * 1e-3)}
            ncell = gplan.info(g3.G3_INFO_CELLS_PER_EDGE)
            if ncell >= 5:                       # the half-stencil kernel serves this grid
                cand = g2w_candidate_pairs(pos[0], w.box, ncell) * F          # frames of one trajectory are alike
                instr = cand * ALGO_INSTR_PER_G2W_CANDIDATE + (pairs // 2) * ALGO_INSTR_PER_G2W_HIT
                g2w["roofline"] = {"bound": "alu", "unit": "Tinstr/s", "peak": peak_tinstr,
                                   "kernel": "g2_wide_cell_kernel",
                                   "candidate_pairs_per_step": cand,
                                   "algorithmic_instr_per_candidate": ALGO_INSTR_PER_G2W_CANDIDATE,
                                   "algorithmic_instr_per_hit": ALGO_INSTR_PER_G2W_HIT,
                                   "achieved": instr / (extra * 1e-3) / 1e12,
                                   "frac": instr / (extra * 1e-3) / 1e12 / peak_tinstr,
                                   "note": "candidates counted from the cell occupancies of frame 0 x frames; "
                                           "time = the extra device time of a step with G3_OPT_G2_WIDE"}
    except Exception as e:  # the g3 numbers above stay valid
        g2w = {"error": str(e)}
    # MSD over all time origins at the same shape (unwrapped random walk,
    # N = 32768, F frames, every lag), device-resident; CUDA events around the g3_msd calls
    msd = None
    try:
        from workloads import unwrapped_walk
        d_walk = torch.from_numpy(grid_to_pos(unwrapped_walk(w.n, F, seed=w.seed), w.box)).cuda()
        g3.msd(d_walk, w.box)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(3):
            g3.msd(d_walk, w.box)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_msd = e0.elapsed_time(e1) / 3
        # g3_msd_static: the same kernels with the scratch in libg3's built-in array (no allocation)
        ms_msd_static = None
        try:
            s_out = torch.empty((F, 2), dtype=torch.int64, device="cuda")
            m_out = torch.empty(F, dtype=torch.float64, device="cuda")
            g3.msd_static(d_walk, w.box, sums=s_out, out=m_out)
            e0.record(stream)
            for _ in range(3):
                g3.msd_static(d_walk, w.box, sums=s_out, out=m_out)
            e1.record(stream)
            torch.cuda.synchronize()
            ms_msd_static = e0.elapsed_time(e1) / 3
        except g3.G3Error:                       # G3_ELIMIT: --frames beyond the built-in scratch
            pass
        disp = w.n * F * (F + 1) // 2
        rate = disp / (ms_msd * 1e-3)
        msd = {"ms": ms_msd, "ms_no_alloc_entry": ms_msd_static,
               "displacements_per_s": rate, "frames": F, "lags": F,
               "hbm_gbs_achieved": F * w.n * 24 / (ms_msd * 1e-3) / 1e9,
               "roofline": {"bound": "alu", "unit": "Tinstr/s", "peak": peak_tinstr,
                            "algorithmic_instr_per_displacement": ALGO_INSTR_PER_DISPLACEMENT,
                            "achieved": rate * ALGO_INSTR_PER_DISPLACEMENT / 1e12,
                            "frac": rate * ALGO_INSTR_PER_DISPLACEMENT / 1e12 / peak_tinstr,
                            "note": "with every lag the kernel is bound by integer issue and shared-memory "
                                    "loads, not by HBM (algorithmic bytes F x N x 24 are read once)"}}
        del d_walk
    except Exception as e:  # the g3 numbers above stay valid
        msd = {"error": str(e)}
    others = None
    if world == 1 and not args.no_other_configs and not args.frames:
        others = other_configs_leg(g3, torch, stream, peak_tinstr, args.other_steps)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_leg(w, args.cpu_budget)
    nbytes = w.n_r * w.n_r * w.n_t * 8
    line = {
        "metric": METRIC, "value": triplets_all / (ms_dev * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_dev,
        "higher_is_better": True, "scaling": "strong" if args.shard_one_trajectory else "weak",
        "vs_baseline": None, "dtype": "f32+int64",
        "data": "synthetic", "frames_per_s": frames_all_ranks / (ms_dev * 1e-3),
        "config": {"workload": f"config4 {w.name}: N={w.n}, L={w.box}, r_max={w.r_max}, "
                               f"{w.n_r}x{w.n_r}x{w.n_t} bins, {frames_all_ranks} frames per step over {world} GPU(s)",
                   "frames_per_step": frames_all_ranks, "triplets_per_step": triplets_all,
                   "batch_frames": plan.info(g3.G3_INFO_BATCH_FRAMES),
                   "kernel": plan.info(g3.G3_INFO_KERNEL),
                   "l2": f"inputs larger than L2 ({F * w.n * 24 / 2**20:.0f} MiB of positions per step)",
                   "parallelism": (f"one trajectory, frames sharded over {world} GPU(s)" if args.shard_one_trajectory
                                   else f"one trajectory per GPU ({world} GPU(s))") + ", one histogram sum per run"},
        "clocks": clocks,
        "e2e": {"value": triplets_all / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e,
                "frames_per_s": frames_all_ranks / (ms_e2e * 1e-3),
                "h2d_bytes_per_step": F * w.n * 24, "d2h_bytes_per_step": 2 * nbytes + 24},
        "gpu_launches": launches * args.steps,
        "gpu_launches_per_step": launches,
        "roofline": roofline,
        "plan": plan_info,
        "qtet": qtet,
        "g2_wide": g2w,
        "msd": msd,
        "configs": others,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def launch_ranks(args) -> int:
    """`python bench.py --gpus N` without torchrun: start the N ranks here, one per GPU, through
    torch.distributed.run on 127.0.0.1 (split the trajectory, merge the
    results).  NCCL's communicator log is left on so that the ranks can be counted from stderr."""
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    env.setdefault("MASTER_ADDR", "127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd, env=env).returncode


def run_launch_check(args) -> int:
    """What the launcher starts, without a GPU: every rank joins a gloo group, reports its rank
    and the block of frames --shard-one-trajectory would give it; rank 0 prints one JSON line."""
    import torch
    import torch.distributed as dist
    from paper_1708_08619_b200.sharding import frame_shard
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    F = args.frames or WORKLOADS[WORKLOAD_INDEX].n_frames
    b, e = frame_shard(F, rank, world)
    mine = torch.tensor([rank, b, e, os.getpid()], dtype=torch.int64)
    rows = [mine]
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("gloo")
        rows = [torch.zeros(4, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(rows, mine)
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"launched": world, "ranks": [int(r[0]) for r in rows],
                          "shards": [[int(r[1]), int(r[2])] for r in rows],
                          "pids": [int(r[3]) for r in rows], "frames": F}), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--frames", type=int, default=0, help="frames per step (default: the workload's)")
    ap.add_argument("--batch-frames", type=int, default=0)
    ap.add_argument("--triplet-warps", type=int, default=0)
    ap.add_argument("--ref-frames", type=int, default=4, help="frames per step of --impl reference")
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the configs 1, 2, 3, 5 block")
    ap.add_argument("--other-steps", type=int, default=2)
    ap.add_argument("--shard-one-trajectory", action="store_true",
                    help="strong scaling: split the one seeded trajectory over the ranks (sharding.frame_shard)")
    ap.add_argument("--launch-check", action="store_true",
                    help="CPU only: start the ranks (gloo), report rank count and frame shards, no GPU work")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return launch_ranks(args)
    if args.launch_check:
        return run_launch_check(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
