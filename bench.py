#!/usr/bin/env python
"""bench.py -- throughput of the WP-CCC hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1]

One "step" = one pass of the whole hot path over one batch: wpccc_propagate of every
trajectory of the workload (geometry, direct GEMM + assembly, transfer tables + contraction + rotation, factorisation,
RK4 sweep) followed by wpccc_probabilities.  The workload is BASELINE.json configs[1] (two-centre p + H with electron
transfer: 172 states, quadrature 64 x 16 x 128, 16 impact parameters, 1600 RK4 steps), the smallest configuration that
exercises every row; inputs are seeded and synthetic (wpccc_inputs).  metric = trajectory * RK4-steps / s.

`value`: basis tables already resident in HBM (a0 staged once, outside the timed region).
`e2e`:   the same job from HOST buffers: wpccc_setup_basis (H2D of the radial tables) + propagate + probabilities
         + D2H of the probabilities and cross sections, all inside the timed region.
N > 1 (torchrun): the 16 N impact parameters are sharded round-robin, 16 per rank (weak scaling); the only exchange
is the all-gather of the final amplitudes before the cross-section integral (paper_2403_04252_b200/shard.py).
--impl reference: the CPU oracle (oracle/), as it stands, on the host cores, on a bounded sample of the same workload.
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
sys.path.insert(0, ROOT)

METRIC = "trajectory*RK4-steps/s"
NOMINAL_FP64_TENSOR_OVER_BF16 = 45.0 / 2250.0      # blackwell_cuda_programming.md table: B200 FP64 tensor 45 TF, bf16 2.25 PF


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]), src="measured")
    return dict(hbm_gbs=6650.0, bf16=1590.0, bf16_sustained=1400.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 7:
                self.rows.append(f)

    def mark(self):
        return len(self.rows)

    def summary(self, lo=0, hi=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        rows = self.rows[lo:hi] or self.rows[-3:]
        try:
            sm = sorted(float(r[0]) for r in rows)
            reasons = [n for k, n in ((3, "hw_slowdown"), (4, "hw_thermal_slowdown"), (5, "sw_thermal_slowdown"), (6, "sw_power_cap"))
                       if any(r[k].lower().startswith("active") for r in rows)]
            return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "power_w_max": max(float(r[2]) for r in rows),
                    "samples": len(rows), "reasons": reasons}
        except Exception as e:      # pragma: no cover
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["parse error: %s" % e]}

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()


def workload(cfg_idx, world, rank):
    """(problem, run, local trajectory indices): BASELINE.json configs[cfg_idx]; for world > 1 the impact-parameter set is
    refined to world x as many log-spaced values over the same range and sharded round-robin (16 per rank for cfg 1)."""
    from wpccc_inputs import CONFIGS, build_config, log_spaced
    from paper_2403_04252_b200.shard import shard_indices
    prob, run = build_config(cfg_idx)
    if world > 1:
        c = CONFIGS[cfg_idx]
        bs = np.asarray(c["b"], float)
        bs = log_spaced(bs.min(), bs.max(), len(bs) * world)
        vs = np.asarray(c["v"], float)
        run = dict(run, b=np.tile(bs, len(vs)), v=np.repeat(vs, len(bs)), vgroup=np.repeat(np.arange(len(vs), dtype=np.int32), len(bs)))
    return prob, run, shard_indices(len(run["b"]), rank, world)


def family_work(prob, b_local, n_steps, units=None):
    """Algorithmic work of each kernel family for ONE step of the bench.
    Returns {family: (bound, work, unit)} with work in flops (tensor / alu) or bytes (hbm).
    units: positions per step each family actually processed (wpccc_last_units): on a symmetric z-grid the node
    tables and the contraction run once per mirror pair (b, -z), (b, +z), and only that work is counted."""
    two = len(prob.centres) == 2
    n_traj_local = len(b_local)
    groups = len(set(np.asarray(b_local).tolist()))       # one-centre: trajectories with equal b share every matrix
    n_pos = (n_traj_local if two else groups) * (2 * n_steps + 1)
    Nc = [c.n_states for c in prob.centres]
    N = sum(Nc)
    E = 0
    for c in prob.centres:
        l = np.asarray(c.l)
        for lam in range(prob.lambda_max + 1):
            for a1 in range(len(l)):
                ok = (np.abs(l[a1] - l[a1:]) <= lam) & (lam <= l[a1] + l[a1:]) & (((l[a1] + l[a1:] + lam) % 2) == 0)
                E += int(ok.sum())
    out = {"direct_gemm": ("tensor", 2.0 * prob.Nr * E * n_pos, "flop")}
    if two:
        q = prob.quad
        nodes = q["n_rho"] * q["n_z"]
        nqc = [int(sum(int(x) + 1 for x in c.l)) for c in prob.centres]
        nrad = [len(c.l) for c in prob.centres]
        n_con = (units or {}).get("transfer_contraction") or n_pos
        n_tab = (units or {}).get("transfer_tables") or n_pos
        out["transfer_contraction"] = ("tensor", 3 * 4.0 * nqc[0] * nqc[1] * nodes * n_con, "flop")
        # node tables: bound by the HBM write of X and Xh for every (column, node) of both sides
        out["transfer_tables"] = ("hbm", 8.0 * 2 * (nqc[0] + nqc[1]) * nodes * n_tab, "byte")
        out["rotation"] = ("hbm", 16.0 * (3 * Nc[0] * Nc[1] + 6 * nqc[0] * nqc[1]) * n_pos, "byte")
        out["direct_assemble"] = ("hbm", 16.0 * (Nc[0] ** 2 + Nc[1] ** 2) * n_pos, "byte")
        out["factor"] = ("alu", (8.0 * Nc[1] ** 2 * Nc[0] + 8.0 / 3.0 * Nc[1] ** 3) * n_pos, "flop")
        out["sweep"] = ("hbm", 16.0 * (N * N + 2 * Nc[0] * Nc[1] + Nc[1] ** 2) * 4 * n_steps * n_traj_local, "byte")
    else:
        out["direct_assemble"] = ("hbm", 8.0 * N * N * n_pos, "byte")
        out["sweep"] = ("hbm", 8.0 * N * N * 4 * n_steps * groups, "byte")
    return out


def run_ours(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the WP-CCC hot path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import paper_2403_04252_b200 as wp
    from paper_2403_04252_b200.shard import gather_amplitudes

    prob, run, mine = workload(args.config, world, rank)
    b_all, v_all, vg_all = run["b"], run["v"], run["vgroup"]
    b, v = b_all[mine], v_all[mine]
    n_steps, z0, z1 = run["n_steps"], run["z_min"], run["z_max"]
    if args.window_steps:                                                  # not the headline: a window of the configured step size around z = 0
        hz = (z1 - z0) / n_steps
        n_steps = int(args.window_steps)
        z0, z1 = -0.5 * n_steps * hz, 0.5 * n_steps * hz
    n_vg = int(vg_all.max()) + 1
    basis = wp.setup_basis(prob)
    if args.direct_tables:
        basis.enable_direct_tables(True)
    N = basis.n_tot
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def step():
        C = wp.propagate(basis, b, v, z0, z1, n_steps)
        Call = gather_amplitudes(C, len(b_all), rank, world)
        return wp.probabilities(basis, Call, b=b_all, vgroup=vg_all, n_vgroups=n_vg)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    sampler = ClockSampler(local_rank) if rank == 0 else None
    for _ in range(args.warmup):
        step()
    barrier()
    m0 = sampler.mark() if sampler else 0
    evs, launches, fam_ms, units_step = [], 0, {}, {}
    for _ in range(args.steps):
        flush.fill_(1)                                                     # L2 flush between timed iterations
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        out = step()
        e1.record()
        evs.append((e0, e1))
        tm = wp.last_timing(basis)                                         # synchronises; per-family event times of this step
        launches += sum(n for _, n in tm.values()) + 4                     # + init amplitudes, probabilities, 2 x cross sections
        units_step = wp.last_units(basis)                                  # positions per family of this step (same every step)
        for k, (ms, n) in tm.items():
            a = fam_ms.setdefault(k, [0.0, 0])
            a[0] += ms; a[1] += n
    barrier()
    m1 = sampler.mark() if sampler else 0
    ms_step = sum(e0.elapsed_time(e1) for e0, e1 in evs) / args.steps
    t = torch.tensor([ms_step], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item())
    units = len(b_all) * n_steps                                           # trajectory * RK4-steps per step, all ranks
    value = units / (ms_step * 1e-3)

    # ---- e2e: the same job from host buffers through the public API, H2D and D2H inside the timed region
    h2d = sum(np.asarray(getattr(c, k)).nbytes for c in prob.centres for k in ("u", "g", "eps", "l", "kind", "nq")) + np.asarray(prob.w).nbytes + b.nbytes + v.nbytes
    keys = ("P_state", "P_nl", "P_class", "sigma_nl", "sigma_class")
    d2h, e2e_ms = 0, []
    for it in range(1 + min(args.steps, 3)):
        barrier()
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        bs2 = wp.setup_basis(prob)                                         # H2D of every table
        C = wp.propagate(bs2, b, v, z0, z1, n_steps)
        Call = gather_amplitudes(C, len(b_all), rank, world)
        o = wp.probabilities(bs2, Call, b=b_all, vgroup=vg_all, n_vgroups=n_vg)
        host = {k: o[k].cpu() for k in keys}                               # D2H (synchronises)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) * 1e3
        bs2.close()
        d2h = sum(x.numel() * x.element_size() for x in host.values())
        if it > 0:
            e2e_ms.append(dt)
    t = torch.tensor([sum(e2e_ms) / len(e2e_ms)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_val = units / (float(t.item()) * 1e-3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    clocks = sampler.summary(m0, m1)
    sampler.stop()

    # ---- roofline of the dominant kernel family (device time measured with CUDA events inside the library, on the
    # stream each kernel was launched on, during the timed steps above)
    pk = measured_peaks()
    dmma, dfma = wp.fp64_peak(1), wp.fp64_peak(0)
    work = family_work(prob, b, n_steps, units_step)
    if args.direct_tables:                                                 # NEXT-1: 16 B read + 8 B written per entry and position
        work["direct_gemm"] = ("hbm", work["direct_gemm"][1] / (2.0 * prob.Nr) * 24.0, "byte")
    fams = {}
    for k, (ms, n) in fam_ms.items():
        if n == 0 or k not in work:
            continue
        bound, w, unit = work[k]
        per_step_ms = ms / args.steps
        if bound == "hbm":
            ach, peak, u = w / (per_step_ms * 1e-3) / 1e9, pk["hbm_gbs"], "GB/s"
        else:
            ach, peak, u = w / (per_step_ms * 1e-3) / 1e12, (dmma if bound == "tensor" else dfma), "TFLOP/s"
        fams[k] = {"bound": bound, "achieved": round(ach, 3), "peak": round(peak, 3), "unit": u, "frac": round(ach / peak, 4),
                   "ms_per_step": round(per_step_ms, 3), "launches_per_step": n // args.steps}
    dom = max(fams, key=lambda k: fams[k]["ms_per_step"])
    roof = dict(fams[dom])
    roof.update({"kernel": dom, "traffic": None,
                 "peak_source": ("in-run FP64 micro-benchmark through wpccc_fp64_peak (DMMA m8n8k4 %.2f, DFMA %.2f TFLOP/s); "
                                 "MEASURED_PEAKS.json (%s) has no fp64 figure: bf16 burst %.1f x nominal fp64-tensor/bf16 ratio %.3f = %.2f TFLOP/s; hbm %.1f GB/s"
                                 % (dmma, dfma, pk["src"], pk["bf16"], NOMINAL_FP64_TENSOR_OVER_BF16, pk["bf16"] * NOMINAL_FP64_TENSOR_OVER_BF16, pk["hbm_gbs"]))})
    tr = os.path.join(ROOT, "profiles", "traffic.json")                    # dram bytes per launch from the committed ncu --set full capture
    if os.path.exists(tr):
        roof["traffic"] = json.load(open(tr)).get(dom)

    Nc = [c.n_states for c in prob.centres]
    elems_per_pos = (Nc[0] ** 2 + Nc[1] ** 2 + 3 * Nc[0] * Nc[1]) if len(Nc) == 2 else Nc[0] ** 2
    line = {
        "metric": METRIC, "value": round(value, 3), "unit": "trajectory*steps/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": round(ms_step, 3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[%d]: %s, N_tot=%d states, %d trajectories x %d RK4 steps per step%s" % (
                       args.config, "two-centre p+H with electron transfer, quadrature %dx%dx%d" % (prob.quad["n_rho"], prob.quad["n_phi"], prob.quad["n_z"]) if prob.quad else "one-centre",
                       N, len(b_all), n_steps, (" (%d per rank)" % len(b) if world > 1 else "") + (" [window of the configured step size around z = 0, not the full z-range]" if args.window_steps else "")),
                   "l2": "512 MiB buffer written between timed iterations (L2 flush); window buffers of one step are several GB >> L2",
                   "parallelism": "dp%d over impact parameters" % world,
                   "direct": "prefix/suffix tables (NEXT-1)" if args.direct_tables else "DMMA GEMM",
                   "mirror_pairs": "body-frame integrals of (b,-z),(b,+z) evaluated together: %d of %d positions per step run the node tables and the contraction; roofline work counts those only" % (
                       units_step.get("transfer_contraction", 0), units_step.get("rotation", 0)) if prob.quad else "n/a"},
        "matrix_elements_per_s": round(elems_per_pos * len(b_all) * (2 * n_steps + 1) / (ms_step * 1e-3), 1),
        "clocks": clocks,
        "e2e": {"value": round(e2e_val, 3), "unit": "trajectory*steps/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)},
        "gpu_launches": int(launches),
        "roofline": roof,
        "kernel_families": fams,
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.config, budget_steps=args.cpu_steps)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def cpu_sample(cfg_idx, n_rk4_steps):
    """The oracle, as it stands, on a bounded sample of the workload: ONE trajectory (the middle impact parameter) for
    n_rk4_steps RK4 steps around closest approach (same step size).  Returns (seconds, description, threads)."""
    from oracle import propagate as oprop
    from wpccc_inputs import build_config
    prob, run = build_config(cfg_idx)
    h = (run["z_max"] - run["z_min"]) / run["n_steps"]
    i = len(run["b"]) // 2
    t0 = time.perf_counter()
    oprop.propagate(prob, float(run["b"][i]), float(run["v"][i]), -0.5 * n_rk4_steps * h, 0.5 * n_rk4_steps * h, n_rk4_steps)
    dt = time.perf_counter() - t0
    try:
        from threadpoolctl import threadpool_info
        thr = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        thr = os.cpu_count() or 1
    sample = "configs[%d], 1 trajectory (b=%.4g, v=%.3g), %d RK4 steps of the configured size around z=0 (%d evaluations of S,H + %d solves)" % (
        cfg_idx, run["b"][i], run["v"][i], n_rk4_steps, 2 * n_rk4_steps + 1, 4 * n_rk4_steps)
    return dt, sample, thr


def cpu_baseline(cfg_idx, budget_steps=5):
    dt, sample, thr = cpu_sample(cfg_idx, budget_steps)
    return {"value": round(budget_steps / dt, 5), "unit": "trajectory*steps/s", "cores": int(thr), "kind": "oracle", "sample": sample,
            "seconds": round(dt, 2), "host_cores": os.cpu_count()}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = 2                                               # RK4 steps of one trajectory per bench "step" (bounded sample)
    for _ in range(min(args.warmup, 1)):
        cpu_sample(args.config, 1)
    tot, sample, thr = 0.0, "", 1
    for _ in range(args.steps):
        dt, sample, thr = cpu_sample(args.config, n)
        tot += dt
    val = n * args.steps / tot
    line = {"impl": "reference", "metric": METRIC, "value": round(val, 5), "unit": "trajectory*steps/s", "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(tot / args.steps * 1e3, 1), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[%d], bounded sample per step: %s" % (args.config, sample), "parallelism": "host cores"},
            "cpu_baseline": {"value": round(val, 5), "unit": "trajectory*steps/s", "cores": int(thr), "kind": "oracle", "sample": sample},
            "e2e": {"value": round(val, 5), "unit": "trajectory*steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--cpu-steps", type=int, default=16, help="RK4 steps of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--direct-tables", action="store_true", help="SURVEY.md 8(f) NEXT-1: radial sums from prefix/suffix tables instead of the DMMA GEMM (family direct_gemm then counts HBM bytes)")
    ap.add_argument("--window-steps", type=int, default=0, help="propagate only this many RK4 steps (configured step size) around z = 0; for configs whose full run takes many minutes")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        print("bench.py: warmup raised to 3 (timing rules)", file=sys.stderr)
        args.warmup = 3
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world:
        if args.gpus > 1:
            raise SystemExit("bench.py --gpus %d must be launched with torchrun (WORLD_SIZE=%d)" % (args.gpus, world))
    run_ours(args)


if __name__ == "__main__":
    main()
