#!/usr/bin/env python
"""bench.py — periodic FoF throughput on B200 (BASELINE.json metric: linked particles/s, pair
tests/s, achieved HBM GB/s vs peak).

A "step" is one pass of the whole hot path (fof_link + fof_groups: H0-H8 of DESIGN.md §1) over
one synthetic particle set.  Default workload: BASELINE.json configs[2] (256^3 clustered
particles, the configuration north_star's 40 %-of-roofline target is quoted on).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl ours|reference]

N > 1 (under torchrun): replicas by default (north_star fixes one GPU): every rank runs an
independent particle set (seed + rank); value = all ranks' particles / max time, "scaling": "weak".
`--mode slab` times the SHARDED path instead (section 2.3): the one particle set of the
workload cut into z slabs, ghost exchange + local fof_link + label merge + cross-rank groups; "scaling": "strong".
`--impl reference` times the CPU oracle (oracle/, as it stands) on rank 0 only.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2510_26851_b200 import inputs  # noqa: E402

METRIC = "fof_linked_particles_per_s"
UNIT = "particles/s"

# Algorithmic bytes per particle of each profiled stage (the compulsory streams of
# SURVEY.md section 8d split per kernel).  Cell arrays, neighbour re-reads and scan state are
# implementation cost and are deliberately NOT counted.
# NOTE on per-stage fractions: the byte model charges streams to the stage that SURVEY.md's reference pipeline
# would run them in.  Where the design removed or merged a pass the per-stage figure is not a statement about
# that kernel: link.labels is charged 24 B (flatten 8 + canonicalise 12 + write 4) although the union-find is
# rooted at the minimum original index and needs neither a flatten nor a min pass (its "achieved" can exceed
# the HBM peak); groups.count is charged 8 B but runs inside link.labels (its stage time is 0 when fof_groups
# follows fof_link on the same labels); groups.clear, link.clear and link.offsets move no algorithmic bytes.
# Only the sum (124 B per particle, `roofline.path`) is the figure north_star's 40 % target refers to.
ALG_BYTES_PER_PARTICLE = {
    "link.clear": 0,
    "link.hist": 12,               # read pos (histogram)
    "link.offsets": 0,
    "link.partition": 12,          # read pos (reorder); the bin-contiguous intermediate is not counted
    "link.cell_sort": 16,          # write sorted (x, y, z, idx)
    "link.pairs": 16 + 4,          # read sorted once, write parent
    "link.labels": 16 + 4 + 4,     # the model's flatten (8) + canonicalise (8) streams, then gather the root's
                                   # label and write labels (original order)
    "groups.clear": 0,
    "groups.count": 4 + 4,         # read labels, size RMW
    "groups.compact": 4 + 4,       # read sizes, write id map
    "groups.reduce": 12 + 4 + 4 + 4,  # read pos, mass, labels, id
    "groups.finish": 0,
    # block path (FOF_PATH_BLOCKS): the same 84 B of the link phase, charged to its four kernels
    "block.partition": 12 + 12 + 16,   # one pass reads pos and writes the records (no histogram pass)
    "block.link": 16 + 4,              # read the records once, write the local forests
    "block.cross": 0,
    "block.flatten": 8 + 12 + 4,       # flatten + canonicalise + labels
}
ALG_BYTES_TOTAL = 124  # link 84 + groups 40


def peaks():
    """(hbm GB/s, source)"""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (measured copy, burst)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"


class ClockSampler:
    """SM clock and throttle reasons sampled through NVML every ~2 ms while the timed region runs (falls back to
    `nvidia-smi -lms 5` if the NVML binding is missing)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.p, self.index, self.stop, self.nv = [], None, index, False, None

    def _physical_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            try:
                return int(vis.split(",")[self.index])
            except Exception:
                pass
        return self.index

    def __enter__(self):
        try:
            import pynvml as nv

            nv.nvmlInit()
            self.nv = nv
            self.h = nv.nvmlDeviceGetHandleByIndex(self._physical_index())
            self.mx = float(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
            self.t = threading.Thread(target=self._poll, daemon=True)
            self.t.start()
            return self
        except Exception:
            self.nv = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "5"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.p = None
        return self

    def _poll(self):
        nv = self.nv
        bits = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
        while not self.stop:
            try:
                sm = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    rs = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    rs = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.rows.append([str(sm), str(self.mx), "0"] +
                                 ["Active" if rs & bits[n] else "Not Active"
                                  for n in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")])
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        for line in self.p.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.nv is not None:
            self.stop = True
            self.t.join(timeout=2)
            return
        if self.p is not None:
            time.sleep(0.15)
            self.p.terminate()
            try:
                self.p.wait(timeout=2)
            except Exception:
                self.p.kill()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "how": "NVML, ~2 ms period" if self.nv else "nvidia-smi -lms 5"}


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def workload_for_rank(name: str, rank: int) -> inputs.Workload:
    import dataclasses

    w = inputs.CONFIGS[name]
    return dataclasses.replace(w, seed=w.seed + 1000 * rank) if rank else w


def max_over_ranks_ms(ms: float, world: int, device) -> float:
    """Device time of the slowest rank (the contract's "max over ranks"); identity at world 1."""
    if world == 1:
        return float(ms)
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, n_per_rank: int, ms_step: float) -> float:
    """Replicas only: every rank links its own n_per_rank particles per step."""
    return world * n_per_rank / (ms_step * 1e-3)


def time_oracle(pos, w, mass=None):
    """One pass of the oracle (cell list + union-find + groups), wall clock, single thread."""
    import oracle

    t0 = time.perf_counter()
    lab, E = oracle.labels_cells(pos, w.L, w.b)
    og = oracle.groups(pos, lab, w.L, w.N_min, mass=mass)
    return time.perf_counter() - t0, lab, E, og


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, rank 0 only."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    w = inputs.CONFIGS[args.workload]
    budget_s = 150.0
    # bounded sample: the full workload if K+W passes fit the budget, else the same recipe at a
    # smaller particle count (same density, same b, same halo population per particle)
    probe = inputs.scaled(w, min(w.n_side, 64))
    t_probe, *_ = time_oracle(inputs.make_positions(probe), probe)
    per_particle = t_probe / probe.N
    n_side = w.n_side
    while n_side > 32 and per_particle * n_side ** 3 * (args.steps + args.warmup) > budget_s:
        n_side //= 2
    ws = w if n_side == w.n_side else inputs.scaled(w, n_side)
    pos = inputs.make_positions(ws)
    for _ in range(args.warmup):
        time_oracle(pos, ws)
    t = 0.0
    for _ in range(args.steps):
        t += time_oracle(pos, ws)[0]
    value = ws.N * args.steps / t
    sample = (f"{ws.name}: N={ws.N} of the workload's {w.N} particles per step"
              + ("" if ws is w else " (same recipe, density, b and halo population per particle; smaller box)"))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "N": w.N, "L": w.L, "b": w.b, "N_min": w.N_min, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def run_slab(args):
    """--mode slab (N >= 2 ranks): the sharded path of PAPER.md section 2.3 on ONE particle set (strong scaling).
    Every rank generates the seeded set, keeps its z slab, and a step is slab_fof_groups: ghost layer to the rank
    below (ring send/recv), fof_link on own + ghost particles, equivalence pairs all-gathered, sparse merge, then
    the cross-rank group construction (four small all-gathers).  Timed on the device, max over ranks."""
    import torch
    import torch.distributed as dist

    from paper_2510_26851_b200 import binding as B, slab

    rank, local_rank, world = dist_env()
    one_gpu = os.environ.get("FOF_BENCH_ONE_GPU") == "1"   # functional check only: all ranks on cuda:0 over gloo
    if world < 2:
        raise SystemExit("--mode slab needs at least two ranks (torchrun); one rank is the monolithic path")
    B.lib()
    dev = torch.device("cuda", 0 if one_gpu else local_rank)
    torch.cuda.set_device(dev)
    if not one_gpu:
        os.environ.setdefault("NCCL_DEBUG", "INFO")  # the driver counts the ranks in the NCCL log
        dist.init_process_group("nccl", device_id=dev)
    else:
        dist.init_process_group("gloo")
    w = inputs.CONFIGS[args.workload]
    pos_np = inputs.make_positions(w)
    N = w.N
    own = slab.split_into_slabs(pos_np, w.L, world)[rank]
    dpos = torch.from_numpy(pos_np[own]).to(dev)
    dids = torch.from_numpy(own.astype(np.int32)).to(dev)
    del pos_np

    def step():
        return slab.slab_fof_groups(dpos, dids, w.L, w.b, N, N_min=w.N_min)

    for _ in range(max(args.warmup, 3)):
        labels, cat = step()
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier()
    torch.cuda.synchronize()
    with ClockSampler(dev.index) as clk:
        e0.record(stream)
        for _ in range(args.steps):
            labels, cat = step()
        e1.record(stream)
        torch.cuda.synchronize()
    dist.barrier()
    ms_step = max_over_ranks_ms(e0.elapsed_time(e1), world, dev if not one_gpu else "cpu") / args.steps
    k = torch.tensor([cat["K"], int(dpos.shape[0])], dtype=torch.int64, device=dev if not one_gpu else "cpu")
    dist.all_reduce(k)
    if rank == 0:
        line = {"metric": METRIC, "value": N / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": w.name, "N": N, "L": w.L, "b": w.b, "N_min": w.N_min, "mode": "slab",
                           "parallelism": f"{world} z slabs, ghost layer 1.001 b, ring exchange + 5 all-gathers",
                           "groups_kept": int(k[0].item()), "particles_owned_total": int(k[1].item()),
                           "l2": "per-rank inputs + workspace exceed the 126 MB L2" if N * 32 / world > 126e6 else "fits L2"},
                "roofline": None, "cpu_baseline": None,
                "e2e": None, "gpu_launches": None, "clocks": clk.summary(),
                "note": "step = slab_fof_groups (exchange included); host-side index building (torch sort / unique) is "
                        "inside the timed region"}
        print(json.dumps(line), flush=True)
    dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2510_26851_b200 import binding as B

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    B.lib()  # fail loudly if libfof_b200.so is missing
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    w = workload_for_rank(args.workload, rank)
    pos_np = inputs.make_positions(w)
    N = w.N
    hpos = torch.from_numpy(pos_np).pin_memory()
    dpos = hpos.to(dev, non_blocking=True)
    f = B.FoF(N, w.L, w.b, w.N_min, device=dev, grid=args.grid, path=args.path)
    out = f.alloc_groups()
    labels = torch.empty(N, dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        f.link(dpos, labels)
        return f.groups(dpos, labels, out=out)["K"]

    for _ in range(max(args.warmup, 3)):
        K_groups = step()
    torch.cuda.synchronize()

    # ---- stage breakdown: a pass of its own with events around every stage (they cost ~0.06 ms per step,
    # so they stay out of the timed region); it also tells which stage dominates
    n_break = max(3, min(args.steps, 10))
    B.fof_profile_only(f.h, None)
    B.fof_profile_enable(f.h, n_break)
    for _ in range(n_break):
        step()
    torch.cuda.synchronize()
    stages = B.fof_profile_read(f.h)
    B.fof_profile_enable(f.h, 0)
    top = max(stages, key=lambda k: stages[k])

    # ---- timed region: device-resident inputs; K steps bracketed by barrier + synchronize; only the
    # dominant stage carries events (two per step), its live time feeds the roofline
    B.fof_profile_only(f.h, top)
    B.fof_profile_enable(f.h, args.steps)
    launches0 = B.fof_launch_count(f.h)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    with ClockSampler(local_rank) as clk:
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        torch.cuda.synchronize()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = B.fof_launch_count(f.h) - launches0
    top_ms_live = B.fof_profile_read(f.h)[top]
    B.fof_profile_enable(f.h, 0)
    B.fof_profile_only(f.h, None)
    E, pair_tests, grid_pairs = f.link_stats()
    ms_step = max_over_ranks_ms(ms_total, world, dev) / args.steps
    value = whole_job_value(world, N, ms_step)

    # ---- NEXT-1: halo decoration sigma + frozen-assignment backward, timed on their own
    # (not part of the step: the BASELINE metric is fof_link + fof_groups)
    next1 = None
    if not args.no_next1:
        og = f.groups(dpos, labels, particle_group=True)
        Kk = og["K"]
        gcom = torch.randn((max(Kk, 1), 3), device=dev)[:Kk]
        gsig = torch.randn(max(Kk, 1), device=dev)[:Kk]
        for _ in range(2):
            sig = f.group_sigma(dpos, og)
            gp = f.groups_backward(dpos, og, grad_com=gcom, group_sigma=sig, grad_sigma=gsig)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        reps = 10
        torch.cuda.synchronize()
        ev[0].record(stream)
        for _ in range(reps):
            sig = f.group_sigma(dpos, og)
        ev[1].record(stream)
        for _ in range(reps):
            gp = f.groups_backward(dpos, og, grad_com=gcom, group_sigma=sig, grad_sigma=gsig)
        ev[2].record(stream)
        torch.cuda.synchronize()
        t_sig, t_bwd = ev[0].elapsed_time(ev[1]) / reps, ev[1].elapsed_time(ev[2]) / reps
        pk = peaks()[0]
        next1 = {"sigma_ms": t_sig, "backward_ms": t_bwd,
                 "sigma_alg_GBps": 16 * N / (t_sig * 1e-3) / 1e9, "backward_alg_GBps": 28 * N / (t_bwd * 1e-3) / 1e9,
                 "sigma_frac_of_hbm_peak": 16 * N / (t_sig * 1e-3) / 1e9 / pk,
                 "backward_frac_of_hbm_peak": 28 * N / (t_bwd * 1e-3) / 1e9 / pk,
                 "alg_bytes": "sigma: pos 12 + group id 4 per particle; backward: pos 12 + group id 4 + grad 12"}
        del gp, sig, og

    # ---- NEXT-3: S = 16 stochastic-edge samples on one binning (PAPER.md 3.2: S = 16;
    # candidate radius 1.5 b, alpha = 5), timed on their own
    next3 = None
    if not args.no_next3:
        S = 16
        f3 = B.FoF(N, w.L, float(np.float32(1.5 * w.b)), w.N_min, device=dev)
        lab3 = torch.empty(N, dtype=torch.int32, device=dev)
        f3.link(dpos, lab3)
        lp3 = torch.zeros(1, dtype=torch.float64, device=dev)
        g3 = torch.empty((N, 3), dtype=torch.float32, device=dev)
        for smp in range(2):
            B.fof_link_stochastic(f3.h, w.b, 5.0, 2024, smp, lab3, lp3, g3, f3.ws)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        ev[0].record(stream)
        f3.link(dpos, lab3)
        ev[1].record(stream)
        for smp in range(S):
            B.fof_link_stochastic(f3.h, w.b, 5.0, 2024, smp, lab3, lp3, g3, f3.ws)
        ev[2].record(stream)
        torch.cuda.synchronize()
        e3, cand3, _ = f3.link_stats()
        t_bin, t_smp = ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2]) / S
        # the same S samples in one batched call (candidate filter, tests and p_ij shared by four samples at a time)
        labS = torch.empty((S, N), dtype=torch.int32, device=dev)
        lpS = torch.zeros(S, dtype=torch.float64, device=dev)
        gS = torch.empty((S, N, 3), dtype=torch.float32, device=dev)
        scr = torch.empty(max(B.fof_stochastic_scratch_bytes(f3.h, S), 4), dtype=torch.uint8, device=dev)
        B.fof_link_stochastic_batch(f3.h, w.b, 5.0, 2024, 0, S, labS, lpS, gS, scr, f3.ws)
        torch.cuda.synchronize()
        ev[0].record(stream)
        B.fof_link_stochastic_batch(f3.h, w.b, 5.0, 2024, 0, S, labS, lpS, gS, scr, f3.ws)
        ev[1].record(stream)
        torch.cuda.synchronize()
        t_batch = ev[0].elapsed_time(ev[1]) / S
        same = bool(torch.equal(labS[S - 1], lab3))   # the last single sample was sample S - 1
        # the same S samples from the potential-edge list: built once per link (two calls: the first sizes the
        # buffer), then every sample is a stream over it
        f3.stochastic_list(w.b, 5.0)
        torch.cuda.synchronize()
        ev[0].record(stream)
        slist, records = f3.stochastic_list(w.b, 5.0)
        ev[1].record(stream)
        labL = torch.empty((S, N), dtype=torch.int32, device=dev)
        gL = torch.empty((S, N, 3), dtype=torch.float32, device=dev)
        B.fof_link_stochastic_list(f3.h, slist, 2024, 0, S, labL, lpS, gL, scr, f3.ws)
        torch.cuda.synchronize()
        t_build = ev[0].elapsed_time(ev[1])
        ev[0].record(stream)
        B.fof_link_stochastic_list(f3.h, slist, 2024, 0, S, labL, lpS, gL, scr, f3.ws)
        ev[1].record(stream)
        torch.cuda.synchronize()
        t_list = ev[0].elapsed_time(ev[1]) / S
        same_list = bool(torch.equal(labL, labS))
        gmax = float(gS.abs().max().item())
        grad_diff = float((gL - gS).abs().max().item()) / gmax if gmax > 0 else 0.0
        del labS, gS, labL, gL, slist, scr
        next3 = {"samples": S, "binning_ms": t_bin, "ms_per_sample": t_smp, "batched_ms_per_sample": t_batch,
                 "batched_labels_equal_single": same,
                 "list": {"build_ms": t_build, "records": records, "bytes": int(B.fof_stochastic_list_bytes(f3.h, records)),
                          "ms_per_sample": t_list, "ms_per_sample_with_build": t_list + t_build / S,
                          "labels_equal_batched": same_list, "score_max_rel_diff_vs_batched": grad_diff,
                          "what": "fof_stochastic_list_build once per link (count + fill, both calls timed), then "
                                  "fof_link_stochastic_list: every sample streams the 32-byte records"},
                 "potential_edges": cand3, "sampled_edges_last": e3,
                 "potential_edges_per_s": cand3 / (t_smp * 1e-3), "particles_per_s_per_sample": N / (t_smp * 1e-3),
                 "config": "b_cand = 1.5 b, alpha = 5, log p(y) and score function on"}
        f3.close()
        del f3, lab3, g3

    # ---- NEXT-4: six-dimensional sub-halo pass inside every kept halo, timed on its own
    next4 = None
    if not args.no_next4:
        og = f.groups(dpos, labels, particle_group=True)
        gen = torch.Generator(device=dev).manual_seed(4)
        dvel = torch.randn((N, 3), device=dev, generator=gen) * 50.0      # synthetic velocities, 50 per axis
        sub = torch.empty(N, dtype=torch.int32, device=dev)
        args6 = (f.h, dpos, dvel, og["particle_group"], og["group_size"], og["K"], 1.0, 100.0 ** 2, float(w.b), sub, f.ws)
        for _ in range(2):
            B.fof_subgroups(*args6)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record(stream)
        for _ in range(5):
            B.fof_subgroups(*args6)
        ev[1].record(stream)
        torch.cuda.synchronize()
        sizes = og["group_size"].to(torch.float64)
        pairs = float((sizes * (sizes - 1) / 2).sum().item())
        t6 = ev[0].elapsed_time(ev[1]) / 5
        members = int(sizes.sum().item())
        nsub = int(torch.unique(sub[og["particle_group"] >= 0]).numel())
        next4 = {"ms": t6, "halos": og["K"], "members": members, "pairs_in_halos": pairs,
                 "pair_tests_per_s": pairs / (t6 * 1e-3), "sub_halos": nsub,
                 "config": "sigma_x = 1, sigma_v = 100^2 (velocities ~ N(0, 50)), ell = b"}
        f.link(dpos, labels)  # restore the link state that fof_subgroups overwrote
        del dvel, sub, og

    # ---- end to end: host buffers through the C ABI (fof_run_host), copies inside the timed region
    cap = out["cap"]
    h2 = B.fof_create(N, w.L, w.b, w.N_min)
    if args.grid:
        B.fof_set_grid(h2, args.grid)
    dev_buf = torch.empty(B.fof_host_device_bytes(h2, cap) + 256, dtype=torch.uint8, device=dev)
    pin = lambda *s, dt=torch.int32: torch.empty(*s, dtype=dt).pin_memory()  # noqa: E731
    hl, gl, gs = pin(N), pin(cap), pin(cap)
    gm, gc = pin(cap, dt=torch.float32), pin((cap, 3), dt=torch.float32)
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        Kh = B.fof_run_host(h2, hpos, None, hl, gl, gs, gm, gc, None, cap, dev_buf)
    barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(e2e_steps):
        Kh = B.fof_run_host(h2, hpos, None, hl, gl, gs, gm, gc, None, cap, dev_buf)
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    e2e_ms = max_over_ranks_ms(e0.elapsed_time(e1), world, dev) / e2e_steps
    assert Kh == K_groups, (Kh, K_groups)
    assert torch.equal(hl.to(dev), labels), "host-path labels differ from device-path labels"

    # ---- the same call split in two (fof_host_submit / fof_host_wait): two inputs in flight, so the copy of input
    # k+1 and of result k-1 overlap the linking of input k.  The library's streams are its own: host clock around
    # the loop, device idle on both sides.
    dev_buf2 = torch.empty_like(dev_buf)
    bufs = (dev_buf, dev_buf2)
    outs = ((hl, gl, gs, gm, gc), (pin(N), pin(cap), pin(cap), pin(cap, dt=torch.float32), pin((cap, 3), dt=torch.float32)))
    pipe_steps = 2 * e2e_steps

    def pipe(n):
        Ks = []
        B.fof_host_submit(h2, 0, hpos, None, *outs[0], None, cap, bufs[0])
        for k in range(1, n):
            B.fof_host_submit(h2, k % 2, hpos, None, *outs[k % 2], None, cap, bufs[k % 2])
            Ks.append(B.fof_host_wait(h2, (k - 1) % 2))
        Ks.append(B.fof_host_wait(h2, (n - 1) % 2))
        return Ks

    pipe(3)
    for o in outs:
        o[0].fill_(-1)
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    Ks = pipe(pipe_steps)
    torch.cuda.synchronize()
    pipe_ms = max_over_ranks_ms((time.perf_counter() - t0) * 1e3, world, dev) / pipe_steps
    barrier()
    assert all(k == K_groups for k in Ks), Ks
    for o in outs:
        assert torch.equal(o[0].to(dev), labels), "pipelined host-path labels differ from device-path labels"
    # what the two big copies cost on their own (one after the other, nothing else running)
    e0.record(stream)
    for _ in range(3):
        dev_buf[: hpos.numel() * 4].view(torch.float32).copy_(hpos.view(-1), non_blocking=True)
        hl.copy_(labels, non_blocking=True)
    e1.record(stream)
    torch.cuda.synchronize()
    copies_ms = e0.elapsed_time(e1) / 3
    B.fof_destroy(h2)
    del dev_buf2

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (live CUDA-event times from inside the timed region)
    peak, peak_src = peaks()
    alg = ALG_BYTES_PER_PARTICLE.get(top, 0) * N
    hbm_achieved = alg / (top_ms_live * 1e-3) / 1e9 if top_ms_live > 0 else 0.0
    # traffic: dram bytes per launch of that kernel from the committed ncu --set full capture (profiles/traffic.json,
    # written by `python -m paper_2510_26851_b200.traffic_from_ncu`); null if the CUDA sources changed since
    traffic, traffic_source = None, "no profiles/traffic.json"
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        try:
            from paper_2510_26851_b200.traffic_from_ncu import source_hash

            with open(tpath) as fh:
                doc = json.load(fh)
            if doc.get("source_hash") == source_hash():
                traffic = doc.get(args.workload, {}).get(top)
                traffic_source = f"profiles/traffic.json ({doc.get('report')}, sources {doc.get('source_hash')})"
            else:
                traffic_source = (f"profiles/traffic.json is stale: captured from sources {doc.get('source_hash')}, "
                                  f"this tree is {source_hash()}")
        except Exception as exc:  # noqa: BLE001
            traffic_source = f"profiles/traffic.json unreadable: {exc}"
    total_alg = ALG_BYTES_TOTAL * N
    path = {"alg_bytes_per_step": total_alg, "achieved": total_alg / (ms_step * 1e-3) / 1e9,
            "frac": total_alg / (ms_step * 1e-3) / 1e9 / peak,
            "frac_of_8000_nominal": total_alg / (ms_step * 1e-3) / 1e9 / 8000.0, "unit": "GB/s", "peak": peak}
    if top in ("link.pairs", "block.link"):
        # link_kernel is bound by FP32/ALU issue, not by HBM: 9 FP32 operations per
        # distance test (3 sub, 3 mul, 2 add, 1 compare; no FMA by definition of the predicate) against
        # the non-FMA FP32 issue rate measured on this device in this run.
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        alu_peak = B.fof_measure_fp32_issue() / 1e9  # G lane-operations / s, measured in this run (fof.h)
        alu_achieved = 9.0 * pair_tests / (top_ms_live * 1e-3) / 1e9
        roofline = {"bound": "alu", "kernel": top, "achieved": alu_achieved, "peak": alu_peak, "unit": "GOP/s",
                    "frac": alu_achieved / alu_peak, "traffic": traffic, "traffic_source": traffic_source,
                    "peak_source": "measured in this run: fof_measure_fp32_issue (non-FMA FADD + FMUL stream on all "
                                   f"{sms} SMs, best of 4 launches)",
                    "alg_ops_per_launch": 9 * pair_tests, "kernel_ms": top_ms_live,
                    "hbm": {"alg_bytes_per_launch": alg, "achieved": hbm_achieved, "peak": peak, "unit": "GB/s",
                            "frac": hbm_achieved / peak, "peak_source": peak_src},
                    "path": path}
    else:
        roofline = {"bound": "hbm", "kernel": top, "achieved": hbm_achieved, "peak": peak, "unit": "GB/s",
                    "frac": hbm_achieved / peak, "traffic": traffic, "traffic_source": traffic_source,
                    "peak_source": peak_src,
                    "alg_bytes_per_launch": alg, "kernel_ms": top_ms_live, "path": path}

    # ---- the oracle timed beside it on the host cores (a reported baseline, not the target)
    cpu = None
    parity = None
    if world == 1 and not args.no_cpu:
        t_cpu, lab, E_ref, og = time_oracle(pos_np, w)
        cpu = {"value": N / t_cpu, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"full workload {w.name} (N={N}), 1 pass, {t_cpu:.2f} s, host has {os.cpu_count()} cores"}
        parity = bool(np.array_equal(labels.cpu().numpy(), lab) and E == E_ref and K_groups == og["K"]
                      and np.array_equal(out["group_size"][:K_groups].cpu().numpy(), og["group_size"]))
        # second CPU figure: the same oracle with its pair search on all host cores (per-slab edge
        # buffers, serial union); labels must equal the single-thread pass
        import oracle

        cores = os.cpu_count() or 1
        t0 = time.perf_counter()
        lab_mt, E_mt = oracle.labels_cells_threads(pos_np, w.L, w.b, cores)
        oracle.groups(pos_np, lab_mt, w.L, w.N_min)
        t_mt = time.perf_counter() - t0
        cpu["all_cores"] = {"value": N / t_mt, "unit": UNIT, "cores": cores, "kind": "oracle, pair search on all cores + serial union",
                            "seconds": round(t_mt, 3), "labels_equal_single_thread": bool(np.array_equal(lab_mt, lab) and E_mt == E_ref)}

    t_pairs = stages.get("link.pairs") or stages.get("block.link")
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "L": w.L, "b": w.b, "N_min": w.N_min, "grid_n": f.grid[0],
                   "cells": f.grid[1], "groups_kept": K_groups, "true_edges": E, "pair_tests": pair_tests, "grid_pairs": grid_pairs,
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "l2": "inputs + workspace per step exceed the 126 MB L2 (pos 12N + sorted 16N + labels 4N ...)"
                         if N * 32 > 126e6 else "working set fits L2 (small workload)"},
        "pair_tests_per_s": pair_tests / (t_pairs * 1e-3) if t_pairs else None,
        "grid_pairs_per_s": grid_pairs / (t_pairs * 1e-3) if t_pairs and grid_pairs else None,
        "path": f.link_path()[0],
        "stage_ms": {k: round(v, 5) for k, v in stages.items()},
        "stage_ms_note": f"separate pass of {n_break} steps with events around every stage; the timed region carries "
                         f"events around {top} only (roofline.kernel_ms)",
        "roofline": roofline, "cpu_baseline": cpu, "parity_vs_oracle_in_this_run": parity,
        "e2e": {"value": whole_job_value(world, N, pipe_ms), "unit": UNIT, "ms_per_step": pipe_ms, "steps": pipe_steps,
                "h2d_bytes_per_step": int(hpos.numel() * 4),
                "d2h_bytes_per_step": int(N * 4 + Kh * (4 + 4 + 4 + 12) + 8),
                "call": "fof_host_submit / fof_host_wait, two inputs in flight (every step: pinned pos host -> device, "
                        "fof_link + fof_groups, labels + group records device -> host); host clock around the loop",
                "single_call": {"call": "fof_run_host (one blocking call per step, CUDA events)",
                                "value": whole_job_value(world, N, e2e_ms), "ms_per_step": e2e_ms,
                                "steps": e2e_steps},
                "copies_only_ms": copies_ms,
                "copies_only_note": "pos host -> device then labels device -> host, back to back with nothing else "
                                    "running: the floor of the single call without its kernels"},
        "gpu_launches": int(launches), "clocks": clk.summary(), "next1": next1, "next3": next3, "next4": next4,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--grid", type=int, default=None, help="force n cells per axis (tuning knob)")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default, weak scaling) or the z-slab sharded path (strong scaling)")
    ap.add_argument("--path", default="auto", choices=["auto", "cells", "blocks"],
                    help="implementation of H1-H5 (fof_set_path); results are identical")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-next1", action="store_true", help="skip the sigma / backward timing")
    ap.add_argument("--no-next3", action="store_true", help="skip the stochastic-edge sample timing")
    ap.add_argument("--no-next4", action="store_true", help="skip the sub-halo pass timing")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.mode == "slab":
        run_slab(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
