#!/usr/bin/env python
"""bench.py -- the measurement contract of this repo.

A *step* is one pass of the whole hot path over one batch of synthetic particles:
hot_build (keys, sort, gather, tree, groups) + hot_forces (moments, walk, P-P / P-C kernels, scatter).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 0..4] [--scale S] [--theta T] [--order P] [--nleaf L] [--ncrit C]

Default workload: BASELINE.json configs[2] (the N = 2^24 clustered mix the metric is quoted on),
theta = 0.6, quadrupole order.  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# flops per interaction counted from the library's own inner loops:
# FMA = 2, add / multiply = 1, rsqrt = 1; a packed f32x2 instruction counts once per lane-operation.
#   P-P:          4 add + 3 mul + 6 fma + rsqrt            = 20
#   P-C order 0:  3 add + 3 mul + 7 fma + rsqrt            = 21
#   P-C order 2:  4 add + 11 mul + 21 fma + rsqrt          = 58    (constant factors folded into the staged moments)
#   P-C order 4: 10 add + 68 mul + 96 fma + rsqrt          = 271   (as compiled: FADD2 / FMUL2 / FFMA2 per sink pair in SASS)
FLOPS_PP = 20
FLOPS_PC = {0: 21, 2: 58, 4: 271, 6: 271 + 563, 8: 271 + 1589}  # 6, 8: + the generated terms of degree 5 .. p (fmaf = 2, multiply = 1)
# roofline.traffic: DRAM bytes of one forces_kernel launch (ncu --set full: dram__bytes_read.sum + dram__bytes_write.sum),
# looked up in profiles/forces_traffic.csv by workload; null where no capture was taken
def ncu_traffic(config, n, theta, order, nleaf, ncrit):
    import csv

    try:
        with open(os.path.join(ROOT, "profiles", "forces_traffic.csv")) as f:
            for r in csv.DictReader(l for l in f if not l.startswith("#")):
                if (int(r["config"]), int(r["n"]), float(r["theta"]), int(r["order"]), int(r["nleaf"]), int(r["ncrit"])) == \
                        (config, n, theta, order, nleaf, ncrit):
                    return float(r["dram_bytes"])
    except (OSError, KeyError, ValueError):
        pass
    return None


# FP32 peak derived from unit counts and clocks (B200_PROFILING.md: 148 SMs, clocks.max.sm 1965 MHz;
# 128 FP32 lanes per SM, FMA = 2 flops): 148 * 128 * 2 * 1.965e9
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
SORT_BYTES_PER_BODY = 8 * 24 - 4      # 8 passes x (12 B read + 12 B write); pass 0 reads no index (it is the position)
SORT_BYTES_SURVEY = 8 + 8 * 24        # SURVEY 8(d) count for d = 8 (with a histogram pre-pass over the keys; here keygen counts)
KEYGEN_BYTES_PER_BODY = 40          # 12 B pos + 4 B mass read; 8 B key + 16 B float4 body written (+ digit histograms)
GATHER_BYTES_PER_BODY = 36          # 4 B permutation + 16 B float4 gathered, 16 B written
# tree + hash + groups: the sorted keys twice (levels, emit) and the per-body level word written and read,
# per cell the SoA record (key 8, first, count, mask, child, parent 4 each), the 16-byte walk record, the leaf list
# entry or hash slot (4): 24 B per body + 48 B per cell
TREE_BYTES = (24, 48)
# upward pass: 16 B per body read once; per cell the three 32-byte records written (centre/mass/b_max, raw and staged
# quadrupole) and, for the internal eighth, its children's 64 B read: 16 B per body + 104 B per cell (order 2)
MOMENTS_BYTES = (16, 104)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--scale", type=int, default=None)
    ap.add_argument("--theta", type=float, default=None)
    ap.add_argument("--order", type=int, default=None)
    ap.add_argument("--tol", type=float, default=None, help="error-bound criterion (hot_forces_tol): absolute acceleration tolerance per interaction; not the BASELINE workload")
    ap.add_argument("--nleaf", type=int, default=16)
    ap.add_argument("--ncrit", type=int, default=256)
    ap.add_argument("--background", action="store_true", help="periodic configs: per-cell background subtraction (hot_set_background)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def workload(args, rank=0):
    from paper_1310_4502_b200 import workloads as W

    w = W.config(args.config, args.scale)
    if rank:  # independent replicas on the other ranks: same recipe, another seed
        gen = {0: W.uniform_cube, 1: W.plummer_sphere, 2: W.clustered_mix}.get(args.config)
        if gen is not None:
            w2 = gen(w.n, W.SEED0 + args.config + 1000 * rank)
            w2.eps, w2.theta, w2.order = w.eps, w.theta, w.order
            w = w2
    if args.theta is not None:
        w.theta = args.theta
    elif args.config == 2:
        w.theta = 0.6
    if args.order is not None:
        w.order = args.order
    return w


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "samples": len(sm),
                "reasons": sorted(reasons)}


_ORACLE_TREES = {}


def _oracle_tree(args, w_full):
    """The oracle's tree of the bench workload itself where its build takes well under a minute (n <= 2^24: keys, stable
    sort, tree, groups and the moments of every cell); a replica made by the same generator for the 2^27-body config,
    whose build alone takes many minutes.  Returns (tree, workload it was built on, build seconds)."""
    from oracle import oracle as O
    from paper_1310_4502_b200 import workloads as W

    key = (args.config, args.scale, args.nleaf, args.ncrit)
    if key not in _ORACLE_TREES:
        w = w_full
        if w_full.n > (1 << 24):
            w = W.config(args.config, 64)  # a 64^3 lattice made by the same recipe
        t0 = time.perf_counter()
        T = O.Tree(w.pos, w.mass, w.lo, w.size, periodic=w.periodic, nleaf=args.nleaf, ncrit=args.ncrit)
        _ORACLE_TREES[key] = (T, w, time.perf_counter() - t0)
    return _ORACLE_TREES[key]


def cpu_oracle_sample(args, w_full, budget_s=12.0, threads=None):
    """The oracle as it stands on a bounded sample: its whole path on the bench workload, the walk + evaluation on
    random sink groups until the budget is spent, the build charged pro rata."""
    import numpy as np

    from oracle import oracle as O

    T, w, t_build = _oracle_tree(args, w_full)
    O.set_num_threads(threads or os.cpu_count() or 1)
    nthreads = O.num_threads()
    counts = T.cells()["count"][T.groups()]
    order = np.random.default_rng(0).permutation(T.ngroups)
    done, inter, t_eval, chunk = 0, 0, 0.0, max(8, nthreads * 2)
    while done < T.ngroups and t_eval < budget_s:
        sel = order[done:done + chunk]
        t1 = time.perf_counter()
        if args.tol is not None:
            _, _, l0, l2, l4, lpp = T.forces_tol(args.tol, w.eps, groups=sel)
            lpc = l0 + l2 + l4
        else:
            _, _, lpc, lpp = T.forces(w_full.theta, w.eps, w_full.order, groups=sel)
        t_eval += time.perf_counter() - t1
        inter += int((counts[sel] * (lpc + lpp)).sum())
        done += len(sel)
    frac = done / T.ngroups
    t = t_eval + t_build * frac
    nbodies = int(counts[order[:done]].sum())
    return {"value": inter / t / 1e9, "unit": "Ginteractions/s", "cores": nthreads, "kind": "oracle",
            "n": w.n, "same_workload_as_gpu": w.n == w_full.n, "interactions_per_particle": inter / max(nbodies, 1),
            "sample": (f"{w.name}, n={w.n}: oracle keys+sort+tree+groups+moments in full ({t_build:.1f} s, charged pro rata), "
                       f"walk + evaluation of {done}/{T.ngroups} random sink groups "
                       f"({nbodies} bodies, {t_eval:.1f} s on {nthreads} threads), theta={w_full.theta}, order={w_full.order}, double precision"),
            "seconds": t, "interactions": inter}


def run_reference(args):
    """--impl reference: the oracle, timed on the host cores, same metric and config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload(args)
    vals = []
    for _ in range(max(1, args.warmup > 0)):
        cpu_oracle_sample(args, w, budget_s=2.0)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        vals.append(cpu_oracle_sample(args, w, budget_s=8.0))
    wall = time.perf_counter() - t0
    inter = sum(v["interactions"] for v in vals)
    secs = sum(v["seconds"] for v in vals)
    value = inter / secs / 1e9
    base = vals[-1]
    one = cpu_oracle_sample(args, w, budget_s=4.0, threads=1)
    cfg = config_dict(args, w)
    cfg["cpu_sample_n"] = base["n"]
    out = {"impl": "reference", "metric": "interactions_per_second", "value": value, "unit": "Ginteractions/s",
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": cfg, "gpu_launches": 0,
           "cpu_baseline": {"value": value, "unit": "Ginteractions/s", "cores": base["cores"], "kind": "oracle",
                            "sample": base["sample"], "n": base["n"], "same_workload_as_gpu": base["same_workload_as_gpu"],
                            "interactions_per_particle": base["interactions_per_particle"],
                            "value_1_thread": one["value"]},
           "e2e": {"value": value, "unit": "Ginteractions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def reduce_over_ranks(dist, ms, inter, device):
    """Whole-job figures of N independent replicas: the slowest rank's time, the interactions of all."""
    import torch

    tms = torch.tensor([ms], dtype=torch.float64, device=device)
    tint = torch.tensor([float(inter)], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(tms, op=dist.ReduceOp.MAX)
        dist.all_reduce(tint, op=dist.ReduceOp.SUM)
    return float(tms.item()), float(tint.item())


def config_dict(args, w):
    return {"workload": f"BASELINE.json configs[{args.config}]: {w.name}, n={w.n}, "
                        f"{'periodic' if w.periodic else 'open'}, eps={w.eps:g}, theta={w.theta:g}, order={w.order}",
            "n": w.n, "theta": w.theta, "eps": w.eps, "order": w.order, "nleaf": args.nleaf, "ncrit": args.ncrit,
            "l2": "inputs (pos+mass 16 B/body) and every per-step array exceed the 126 MB L2 at n >= 2^23; "
                  "each step rebuilds keys, tree and moments from the caller's arrays",
            "parallelism": "replicas only (one independent problem per GPU, no collective)"}


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    import numpy as np
    import torch

    import paper_1310_4502_b200 as hot

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    w = workload(args, rank)
    hot.hot_set_params(args.nleaf, args.ncrit)
    hot.hot_set_background(bool(args.background))
    pos = torch.from_numpy(w.pos).cuda()
    mass = torch.from_numpy(w.mass).cuda()
    acc = torch.empty((w.n, 3), dtype=torch.float32, device="cuda")
    pot = torch.empty(w.n, dtype=torch.float32, device="cuda")

    def step():
        hot.hot_build(pos, mass, w.lo, w.size, w.periodic)
        if args.tol is not None:
            hot.hot_forces_tol(args.tol, w.eps, acc=acc, pot=pot)
        else:
            hot.hot_forces(w.theta, w.eps, w.order, acc=acc, pot=pot)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage = {}
    e0.record()
    for _ in range(args.steps):
        step()
        st = hot.hot_stats()
        for k in ("ms_keygen", "ms_sort", "ms_gather", "ms_tree", "ms_moments", "ms_farfield", "ms_walk", "ms_coarse", "ms_eval",
                  "ms_build_total", "ms_forces_total"):
            stage[k] = stage.get(k, 0.0) + st[k] / args.steps
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1) / args.steps
    clocks = sampler.stop() if rank == 0 else None
    st = hot.hot_stats()
    inter = st["pp_interactions"] + st["pc_interactions"]
    ms_max, inter_all = reduce_over_ranks(dist, ms, inter, "cuda")

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hp = torch.from_numpy(w.pos).pin_memory(); hm = torch.from_numpy(w.mass).pin_memory()
        ha = torch.empty((w.n, 3), dtype=torch.float32).pin_memory(); hq = torch.empty(w.n, dtype=torch.float32).pin_memory()
        hot.hot_step_host(hp.numpy(), hm.numpy(), w.lo, w.size, w.periodic, w.theta, w.eps, w.order, ha.numpy(), hq.numpy())
        barrier()
        t0 = time.perf_counter()
        nrep = max(1, min(args.steps, 3))
        for _ in range(nrep):
            hot.hot_step_host(hp.numpy(), hm.numpy(), w.lo, w.size, w.periodic, w.theta, w.eps, w.order, ha.numpy(), hq.numpy())
        torch.cuda.synchronize()
        te = torch.tensor([(time.perf_counter() - t0) / nrep], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": inter_all / float(te.item()) / 1e9, "unit": "Ginteractions/s",
               "ms_per_step": 1e3 * float(te.item()), "h2d_bytes_per_step": 16 * w.n, "d2h_bytes_per_step": 16 * w.n}
        assert np.isfinite(ha.numpy()).all()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    # particle-cell interactions by the order they were evaluated at (hot_stats; a mix under --tol), + the generated terms of orders 6, 8
    flops = (st["pp_interactions"] * FLOPS_PP + st["pc_monopole"] * FLOPS_PC[0] + st["pc_quadrupole"] * FLOPS_PC[2]
             + st["pc_hexadecapole"] * FLOPS_PC[4] + (st["pc_interactions"] * (FLOPS_PC[w.order] - FLOPS_PC[4]) if w.order > 4 and args.tol is None else 0))
    # with --background the far cells are evaluated in the background stage (hot_stats ms_coarse): count both launches
    kern_s = (stage["ms_eval"] + (stage["ms_coarse"] if args.background and w.periodic else 0.0)) * 1e-3
    achieved = flops / kern_s / 1e12
    tf_scalar, tf_packed = hot.hot_measure_fp32()  # register-only FMA chains on this device, after the timed region
    tf_2reg, tf_3reg, tf_s3reg = hot.hot_measure_fp32_operands()  # the same pipe fed from the register file
    traffic = None if args.tol is not None else ncu_traffic(args.config, w.n, w.theta, w.order, args.nleaf, args.ncrit)
    out = {
        "metric": "interactions_per_second", "value": inter_all / (ms_max * 1e-3) / 1e9, "unit": "Ginteractions/s",
        "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms_max,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(args, w),
        "force_eval_s_per_step": ms_max * 1e-3,
        "interactions_per_step": {"pp": st["pp_interactions"], "pc": st["pc_interactions"],
                                  "per_particle": inter / w.n},
        "kernel_only_Ginteractions_per_s": inter / kern_s / 1e9,
        "stages_ms": {k: round(v, 4) for k, v in stage.items()},
        "tree": {"n_cells": st["n_cells"], "n_groups": st["n_groups"], "max_level": st["max_level"],
                 "cells_visited": st["cells_visited"], "walk_spills": st["walk_spills"],
                 "list_entries": st["list_entries"], "list_rounds": st["list_chunks"]},
        "hbm_stages": {
            "keygen_GBps": KEYGEN_BYTES_PER_BODY * w.n / (stage["ms_keygen"] * 1e-3) / 1e9,
            "sort_GBps": SORT_BYTES_PER_BODY * w.n / (stage["ms_sort"] * 1e-3) / 1e9,
            "sort_GBps_survey_count": SORT_BYTES_SURVEY * w.n / (stage["ms_sort"] * 1e-3) / 1e9,
            "gather_GBps": GATHER_BYTES_PER_BODY * w.n / (stage["ms_gather"] * 1e-3) / 1e9,
            "tree_GBps": (TREE_BYTES[0] * w.n + TREE_BYTES[1] * st["n_cells"]) / (stage["ms_tree"] * 1e-3) / 1e9,
            "moments_GBps": (MOMENTS_BYTES[0] * w.n + MOMENTS_BYTES[1] * st["n_cells"]) / (max(stage["ms_moments"], 1e-6) * 1e-3) / 1e9,
            "walk_list_GBps": 2 * 4 * st["list_entries"] / (stage["ms_walk"] * 1e-3) / 1e9,
            "walk_Gcells_per_s": st["cells_visited"] / (stage["ms_walk"] * 1e-3) / 1e9},
        "gpu_launches": int((st["launches_build"] + st["launches_forces"]) * args.steps),
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "forces_kernel (P-P + P-C interaction lists of all sink groups, packed f32x2)",
                     "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
                     "traffic": traffic,
                     "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md Roofline); "
                                    "MEASURED_PEAKS.json holds no FP32 figure",
                     "peak_measured_ffma_TFLOPs": {"scalar": tf_scalar, "packed_f32x2": tf_packed,
                                                   "packed_2_register_sources": tf_2reg, "packed_3_register_sources": tf_3reg,
                                                   "scalar_3_register_sources": tf_s3reg},
                     "frac_of_measured_ffma": achieved / max(tf_scalar, tf_packed),
                     "flops_per_interaction": {"pp": FLOPS_PP, "pc": FLOPS_PC[w.order] if args.tol is None else {"0": FLOPS_PC[0], "2": FLOPS_PC[2], "4": FLOPS_PC[4]}},
                     "kernel_ms": kern_s * 1e3, "kernel_share_of_step": kern_s * 1e3 / ms_max},
    }
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        out["hbm_stages"]["peak_GBps"] = peaks.get("hbm_gbs")
    except (OSError, ValueError):
        out["hbm_stages"]["peak_GBps"] = 6650.0
    pk = out["hbm_stages"]["peak_GBps"]
    out["hbm_stages"]["frac_of_peak"] = {k[:-5]: out["hbm_stages"][k] / pk for k in ("keygen_GBps", "sort_GBps", "gather_GBps", "tree_GBps", "moments_GBps")}
    build_bytes = (KEYGEN_BYTES_PER_BODY + SORT_BYTES_PER_BODY + GATHER_BYTES_PER_BODY + TREE_BYTES[0]) * w.n + TREE_BYTES[1] * st["n_cells"]
    out["hbm_stages"]["build_GBps"] = build_bytes / (stage["ms_build_total"] * 1e-3) / 1e9
    out["hbm_stages"]["frac_of_peak"]["build"] = out["hbm_stages"]["build_GBps"] / pk
    if e2e:
        out["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        cb = cpu_oracle_sample(args, w)
        out["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "n", "same_workload_as_gpu",
                                                  "interactions_per_particle")}
        out["cpu_baseline"]["value_1_thread"] = cpu_oracle_sample(args, w, budget_s=4.0, threads=1)["value"]
        out["config"]["cpu_sample_n"] = cb["n"]
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
