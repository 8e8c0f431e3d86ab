#!/usr/bin/env python
"""bench.py -- throughput of the WP-CCC hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--no-per-config]

One "step" = one pass of the whole hot path over one batch: wpccc_propagate of every
trajectory of the workload (geometry, direct GEMM + assembly, transfer tables + contraction + rotation, factorisation,
RK4 sweep) followed by wpccc_probabilities.  The headline workload is BASELINE.json configs[3], the largest
single-GPU configuration (BASELINE.json quotes its metric on no particular one): He2+ + H two-centre, 572 states,
quadrature 96 x 24 x 192, 128 impact parameters.  Its whole job (3000 RK4 steps) takes minutes, so a step is one window
of 64 RK4 steps of the configured size of all 128 trajectories, successive steps walking through the configured z-range
from z_min with the amplitudes carried over (wpccc_propagate, WPCCC_INIT_FROM_DC); metric = trajectory * RK4-steps / s
is intensive.  The same run then measures the other four configurations for a few steps each (key `per_config`; whole
jobs).  Inputs are seeded and synthetic (wpccc_inputs).

`value`: basis tables already resident in HBM (a0 staged once, outside the timed region).
`e2e`:   the same step from HOST buffers: wpccc_setup_basis (H2D of the radial tables) + H2D of the amplitudes a window
         continues from + propagate + probabilities + D2H of the probabilities and cross sections, all timed.
N > 1 (torchrun): the impact parameters are refined N-fold over the same range and sharded round-robin (weak scaling);
the only exchange is the all-gather of the final amplitudes before the cross-section integral (shard.py).
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
    # a z-grid symmetric about 0: F(R) is contracted once per mirror pair (b, -z), (b, +z) (wpccc_last_units)
    n_gemm = (units or {}).get("direct_gemm") or n_pos
    out = {"direct_gemm": ("tensor", 2.0 * prob.Nr * E * n_gemm, "flop")}
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
        # a7, solve_route 0: Hermitian rank-N_T update A = I - K K^H on the lower triangle (4 N_P^2 N_T flops) + complex Cholesky
        # (4/3 N_P^3); counted against the DFMA peak (the DMMA peak of mma.m8n8k4 is the same number on this chip)
        out["factor"] = ("alu", (4.0 * Nc[1] ** 2 * Nc[0] + 4.0 / 3.0 * Nc[1] ** 3) * n_pos, "flop")
        out["sweep"] = ("hbm", 16.0 * (N * N + 2 * Nc[0] * Nc[1] + Nc[1] ** 2) * 4 * n_steps * n_traj_local, "byte")
    else:
        out["direct_assemble"] = ("hbm", 8.0 * N * N * n_pos, "byte")
        out["sweep"] = ("hbm", 8.0 * N * N * 4 * n_steps * groups, "byte")
    return out


# What one bench "step" is for each configuration: the whole job (every RK4 step of the configured z-range) of
# STEP_BATCH[cfg] trajectories.  configs[3] (128 impact parameters x 3000 steps, minutes of GPU time) runs as 16 batches of 8
# impact parameters (every 16th of the log-spaced set, so each batch spans the whole b-range): with 8 trajectories per call
# the mirror stash (the body-frame integrals of all 3000 half-step positions beyond z = 0, 78 GB)
# fits the 180 GB of HBM and every pair (b, -z), (b, +z) is evaluated once -- this is how the library runs that job
# fastest; successive bench steps walk through the 16 batches.  --window-steps instead takes windows of RK4 steps of the
# configured size walking through z from z_min (amplitudes carried over, WPCCC_INIT_FROM_DC), all trajectories at once.
STEP_BATCH = {0: None, 1: None, 2: None, 3: 8, 4: None}


class Job:
    """One configuration staged on the GPU and its bench step."""

    def __init__(self, wp, cfg, world, rank, window=None, direct_tables=False, batch=None):
        self.wp, self.cfg = wp, cfg
        self.prob, run, self.mine = workload(cfg, world, rank)
        self.b_all, self.v_all, self.vg_all = run["b"], run["v"], run["vgroup"]
        self.b_job, self.v_job = self.b_all[self.mine], self.v_all[self.mine]          # this rank's trajectories of the whole job
        self.b_run, self.world = self.b_all, world                                      # the whole job's global list (rank r owns r, r + world, ..)
        self.n_batches = (len(self.b_job) // batch) if (batch and not window and len(self.b_job) > batch and len(self.b_job) % batch == 0) else 1
        self.b, self.v = self.b_job, self.v_job
        self.select_batch(0)
        self.n_steps_job, self.z0, self.z1 = run["n_steps"], run["z_min"], run["z_max"]
        self.hz = (self.z1 - self.z0) / self.n_steps_job
        self.window = min(window, self.n_steps_job) if window else None
        self.n_steps = self.window or self.n_steps_job            # RK4 steps per bench step
        self.n_vg = int(self.vg_all.max()) + 1
        self.basis = wp.setup_basis(self.prob)
        if direct_tables:
            self.basis.enable_direct_tables(True)
        self.k, self.C, self.n_singular = 0, None, 0
        self.world, self.rank = world, rank

    def select_batch(self, k):
        """Trajectories of bench step k: every n_batches-th of the job's list, starting at k mod n_batches."""
        if self.n_batches > 1:
            sl = slice(k % self.n_batches, None, self.n_batches)
            self.b, self.v = self.b_job[sl], self.v_job[sl]
            # the same batch on every rank; all ranks' trajectories of this step in the order gather_amplitudes returns them
            self.b_all = self.b_run.reshape(-1, self.world)[sl].reshape(-1)
            self.vg_all = np.zeros(len(self.b_all), np.int32)
            self.v_all = np.full(len(self.b_all), self.v[0])

    def span(self):
        """z-range of the next step."""
        if not self.window:
            return self.z0, self.z1, None
        per_job = self.n_steps_job // self.window
        k = self.k % per_job
        if k == 0:
            self.C = None                                           # (re)start at z_min with c = 1s
        za = self.z0 + k * self.window * self.hz
        return za, za + self.window * self.hz, self.C

    def step(self, basis=None, C0="walk"):
        from paper_2403_04252_b200.shard import gather_amplitudes
        wp, basis = self.wp, basis or self.basis
        za, zb, Cw = self.span()
        C = wp.propagate(basis, self.b, self.v, za, zb, self.n_steps, C0=Cw if C0 == "walk" else C0, allow_singular=True)
        if C0 == "walk":
            self.C, self.k = C, self.k + 1
            if self.n_batches > 1:
                self.select_batch(self.k)
        Call = gather_amplitudes(C, len(self.b_all), self.rank, self.world)
        return wp.probabilities(basis, Call, b=self.b_all, vgroup=self.vg_all, n_vgroups=self.n_vg)

    def describe(self):
        prob = self.prob
        kind = ("two-centre, Z_P=%g, quadrature %dx%dx%d" % (prob.Z_proj, prob.quad["n_rho"], prob.quad["n_phi"], prob.quad["n_z"])) if prob.quad else "one-centre"
        what = ("one window of %d RK4 steps of the configured size (h=%.4g) of all trajectories per step, successive steps walking through z from z_min=%g "
                "(amplitudes carried over); the full job is %d such steps" % (self.window, self.hz, self.z0, self.n_steps_job)) if self.window else \
               ("the whole job per step: z in [%g, %g], %d RK4 steps" % (self.z0, self.z1, self.n_steps_job))
        if self.n_batches > 1:
            what += ("; the %d impact parameters run as %d batches of %d (every %dth of the log-spaced set), one batch per bench step, successive steps "
                     "walking through the batches: with %d trajectories per call the mirror stash holds every position beyond z = 0" % (
                         len(self.b_job), self.n_batches, len(self.b), self.n_batches, len(self.b)))
        return "BASELINE.json configs[%d]: %s, N_tot=%d states, %d trajectories; %s" % (self.cfg, kind, self.basis.n_tot, len(self.b_job), what)

    def close(self):
        self.basis.close()
        self.basis = None
        self.C = None


def measure(job, torch, dist, world, n_warm, n_timed, flush, sampler=None):
    """Times n_timed steps of the job (CUDA events on the current stream, L2 flushed between steps, max over ranks);
    returns (ms_per_step, family times, launches, units per family, clock marks)."""
    wp = job.wp

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(n_warm):
        job.step()
    barrier()
    m0 = sampler.mark() if sampler else 0
    evs, launches, fam_ms, units_step = [], 0, {}, {}
    for _ in range(n_timed):
        flush.fill_(1)                                                     # L2 flush between timed iterations
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        job.step()
        e1.record()
        evs.append((e0, e1))
        tm = wp.last_timing(job.basis)                                     # synchronises; per-family event times of this step
        launches += sum(n for _, n in tm.values()) + 4                     # + init amplitudes, probabilities, 2 x cross sections
        units_step = wp.last_units(job.basis)                              # positions per family of this step
        st = wp.last_status(job.basis, len(job.b))
        job.n_singular = max(job.n_singular, sum(1 for x in st if x is not None))
        for k, (ms, n) in tm.items():
            a = fam_ms.setdefault(k, [0.0, 0])
            a[0] += ms; a[1] += n
    barrier()
    m1 = sampler.mark() if sampler else 0
    ms_step = sum(e0.elapsed_time(e1) for e0, e1 in evs) / n_timed
    t = torch.tensor([ms_step], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item()), fam_ms, launches, units_step, (m0, m1)


def families(job, fam_ms, n_timed, units_step, pk, dmma, dfma, direct_tables=False):
    work = family_work(job.prob, job.b, job.n_steps, units_step)
    if direct_tables:                                                      # NEXT-1: 16 B read + 8 B written per entry and position
        work["direct_gemm"] = ("hbm", work["direct_gemm"][1] / (2.0 * job.prob.Nr) * 24.0, "byte")
    fams = {}
    for k, (ms, n) in fam_ms.items():
        if n == 0 or k not in work:
            continue
        bound, w, unit = work[k]
        per_step_ms = ms / n_timed
        if bound == "hbm":
            ach, peak, u = w / (per_step_ms * 1e-3) / 1e9, pk["hbm_gbs"], "GB/s"
        else:
            ach, peak, u = w / (per_step_ms * 1e-3) / 1e12, (dmma if bound == "tensor" else dfma), "TFLOP/s"
        fams[k] = {"bound": bound, "achieved": round(ach, 3), "peak": round(peak, 3), "unit": u, "frac": round(ach / peak, 4),
                   "ms_per_step": round(per_step_ms, 3), "launches_per_step": n // n_timed}
    return fams


def elements_per_position(prob):
    Nc = [c.n_states for c in prob.centres]
    return (Nc[0] ** 2 + Nc[1] ** 2 + 3 * Nc[0] * Nc[1]) if len(Nc) == 2 else Nc[0] ** 2


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

    window = args.window_steps or None
    job = Job(wp, args.config, world, rank, window=window, direct_tables=args.direct_tables, batch=STEP_BATCH[args.config])
    prob, b, v, b_all = job.prob, job.b, job.v, job.b_all
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ms_step, fam_ms, launches, units_step, (m0, m1) = measure(job, torch, dist, world, args.warmup, args.steps, flush, sampler)
    units = len(b_all) * job.n_steps                                       # trajectory * RK4-steps per step, all ranks
    value = units / (ms_step * 1e-3)

    # ---- e2e: the same step from host buffers through the public API, H2D and D2H inside the timed region
    h2d = sum(np.asarray(getattr(c, k)).nbytes for c in prob.centres for k in ("u", "g", "eps", "l", "kind", "nq")) + np.asarray(prob.w).nbytes + b.nbytes + v.nbytes
    keys = ("P_state", "P_nl", "P_class", "sigma_nl", "sigma_class")
    C_host = None
    if job.window:                                                         # a window continues from amplitudes: they come from the host too
        _, _, Cw = job.span()
        C_host = (Cw if Cw is not None else torch.zeros((len(b), job.basis.n_tot), dtype=torch.complex128, device="cuda")).cpu().pin_memory()
        h2d += C_host.numel() * 16
    d2h, e2e_ms = 0, []
    for it in range(1 + min(args.steps, 3)):
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        bs2 = wp.setup_basis(prob)                                         # H2D of every table
        if args.direct_tables:
            bs2.enable_direct_tables(True)
        o = job.step(basis=bs2, C0=C_host.cuda(non_blocking=True) if C_host is not None else None)
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

    # ---- roofline of the dominant kernel family (device time measured with CUDA events inside the library, on the
    # stream each kernel was launched on, during the timed steps above)
    pk = measured_peaks()
    dmma, dfma = wp.fp64_peak(1), wp.fp64_peak(0)
    fams = families(job, fam_ms, args.steps, units_step, pk, dmma, dfma, args.direct_tables)
    dom = max(fams, key=lambda k: fams[k]["ms_per_step"])
    roof = dict(fams[dom])
    roof.update({"kernel": dom, "traffic": None,
                 "timing": "CUDA events on the stream the kernels run on; families launched once per chunk of positions (node tables, contraction) "
                           "are sampled on every 8th launch group and scaled by the number of groups",
                 "peak_source": ("in-run FP64 micro-benchmark through wpccc_fp64_peak (DMMA m8n8k4 %.2f, DFMA %.2f TFLOP/s); "
                                 "MEASURED_PEAKS.json (%s) has no fp64 figure: bf16 burst %.1f x nominal fp64-tensor/bf16 ratio %.3f = %.2f TFLOP/s; hbm %.1f GB/s"
                                 % (dmma, dfma, pk["src"], pk["bf16"], NOMINAL_FP64_TENSOR_OVER_BF16, pk["bf16"] * NOMINAL_FP64_TENSOR_OVER_BF16, pk["hbm_gbs"]))})
    tr = os.path.join(ROOT, "profiles", "traffic.json")                    # dram bytes per launch from the committed ncu --set full captures
    if os.path.exists(tr):
        tj = json.load(open(tr))
        roof["traffic"] = tj.get("configs[%d]" % args.config, {}).get(dom)
        roof["traffic_source"] = "not measured in this run: ncu --set full capture recorded in profiles/traffic.json (%s)" % tj.get("_source", "")

    per_config = {str(args.config): {"value": round(value, 3), "ms_per_step": round(ms_step, 3), "steps": args.steps, "warmup": args.warmup,
                                     "workload": job.describe(), "dominant": dom, "frac": fams[dom]["frac"], "kernel_families": fams}}
    line = {
        "metric": METRIC, "value": round(value, 3), "unit": "trajectory*steps/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": round(ms_step, 3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": job.describe() + ((" (%d trajectories per rank)" % len(b)) if world > 1 else ""),
                   "l2": "512 MiB buffer written between timed iterations (L2 flush); window buffers of one step are several GB >> L2",
                   "parallelism": "dp%d over impact parameters" % world,
                   "direct": "prefix/suffix tables (NEXT-1)" if args.direct_tables else "DMMA GEMM",
                   "overlap_solve": "solve_route 0: blocked Cholesky factor of I - K K^H + triangular solves per RK4 stage" if prob.quad else "n/a (S = I)",
                   "not_positive_definite": ("%d of %d trajectories met a position where the overlap matrix of the configured basis and quadrature is not positive "
                                             "definite (DESIGN.md A23); they are flagged (WPCCC_ESINGULAR, amplitudes NaN), every kernel still ran for them" % (job.n_singular, len(b))) if prob.quad else "n/a",
                   "mirror_pairs": ("body-frame integrals of (b,-z),(b,+z) evaluated together where the z-range of a step is symmetric about 0: %d of %d positions per step ran the node tables and the contraction; roofline work counts those only" % (
                       units_step.get("transfer_contraction", 0), units_step.get("rotation", 0))) if prob.quad else "n/a"},
        "matrix_elements_per_s": round(elements_per_position(prob) * len(b_all) * (2 * job.n_steps + 1) / (ms_step * 1e-3), 1),
        "clocks": clocks,
        "e2e": {"value": round(e2e_val, 3), "unit": "trajectory*steps/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)},
        "gpu_launches": int(launches),
        "roofline": roof,
        "kernel_families": fams,
    }
    job.close()
    del job
    wp.release_workspace()
    torch.cuda.empty_cache()

    # ---- the other configurations, a few steps each in the same run (BASELINE.json north_star: steps/s "reported for each")
    if world == 1 and args.per_config:
        for cfg in (0, 1, 2, 4, 3):
            if str(cfg) in per_config:
                continue
            n_warm, n_timed = (3, 5) if cfg in (0, 1) else (1, 2)
            j2 = Job(wp, cfg, 1, 0, batch=STEP_BATCH[cfg])
            if cfg in (2, 4):                                               # whole jobs of several seconds: warm up on short windows first
                jw = Job(wp, cfg, 1, 0, window=16)
                jw.basis.close(); jw.basis = j2.basis
                for _ in range(3):
                    jw.step()
                jw.basis = None
            ms2, fam2, ln2, un2, _ = measure(j2, torch, dist, 1, n_warm, n_timed, flush)
            f2 = families(j2, fam2, n_timed, un2, pk, dmma, dfma)
            d2 = max(f2, key=lambda k: f2[k]["ms_per_step"])
            per_config[str(cfg)] = {"value": round(len(j2.b_all) * j2.n_steps / (ms2 * 1e-3), 3), "ms_per_step": round(ms2, 3), "steps": n_timed, "warmup": n_warm,
                                    "workload": j2.describe(), "dominant": d2, "frac": f2[d2]["frac"], "kernel_families": f2,
                                    "matrix_elements_per_s": round(elements_per_position(j2.prob) * len(j2.b_all) * (2 * j2.n_steps + 1) / (ms2 * 1e-3), 1)}
            line["gpu_launches"] += int(ln2)
            if cfg in (2, 4):
                # the same job with the radial sums of eq. (7) read from prefix/suffix tables instead of the
                # DMMA GEMM (wpccc_enable_direct_tables; exact, parity-tested): the step is then bound by the RK4 sweep
                j2.basis.enable_direct_tables(True)
                ms3, fam3, ln3, un3, _ = measure(j2, torch, dist, 1, 1, 2, flush)
                f3 = families(j2, fam3, 2, un3, pk, dmma, dfma, direct_tables=True)
                d3 = max(f3, key=lambda k: f3[k]["ms_per_step"])
                per_config[str(cfg)]["table_route"] = {"value": round(len(j2.b_all) * j2.n_steps / (ms3 * 1e-3), 3), "ms_per_step": round(ms3, 3), "steps": 2, "warmup": 1,
                                                       "direct": "prefix/suffix tables (NEXT-1)", "dominant": d3, "frac": f3[d3]["frac"], "kernel_families": f3}
                line["gpu_launches"] += int(ln3)
                j2.basis.enable_direct_tables(False)
            j2.close()
            del j2
            wp.release_workspace()
            torch.cuda.empty_cache()
    line["per_config"] = {k: per_config[k] for k in sorted(per_config)}
    if world == 1 and args.paper_shape:
        line["paper_shape"] = paper_shape_sweep(wp, torch, flush)
    sampler.stop()
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.config, budget_steps=args.cpu_steps or CPU_STEPS[args.config])
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def paper_shape_sweep(wp, torch, flush, lmax_1c=(0, 2, 4, 6, 8, 10), lmax_2c=(0, 1, 2, 3, 4, 5)):
    """the paper's own workload shape: p + H at 100 keV, the 6001-point geometric
    z-grid from -300 to 300, eight impact parameters, basis grown through l_max (1C N = 42 .. 4257, 2C N = 60 .. 1910).
    Timed on the 128 central steps of that grid (all eight trajectories; the cost per step does not depend on z), reported
    per RK4 step and extrapolated to the 6000 steps of a whole path."""
    from wpccc_inputs.paper_shape import paper_problem
    out = []
    for two, lms in ((False, lmax_1c), (True, lmax_2c)):
        for lm in lms:
            rec = {"mode": "2C" if two else "1C", "l_max": lm}
            try:
                prob, run = paper_problem(two, lm)
                rec["N"] = prob.n_tot
                g = run["zgrid"]
                mid = len(g) // 2
                win = g[mid - 64: mid + 65]
                basis = wp.setup_basis(prob)
                for _ in range(2):
                    wp.propagate_grid(basis, run["b"], run["v"], win, allow_singular=True)
                ms = []
                for _ in range(3):
                    flush.fill_(1)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    wp.propagate_grid(basis, run["b"], run["v"], win, allow_singular=True)
                    e1.record()
                    torch.cuda.synchronize()
                    ms.append(e0.elapsed_time(e1))
                per_step = sum(ms) / len(ms) / 128.0
                rec.update({"ms_per_rk4_step_8_paths": round(per_step, 4), "trajectory_steps_per_s": round(8 * 1e3 / per_step, 1),
                            "whole_path_6000_steps_s_extrapolated": round(per_step * 6000 / 1e3, 2),
                            "flagged_not_positive_definite": sum(1 for x in wp.last_status(basis, 8) if x is not None)})
                basis.close()
            except Exception as e:                                    # a size beyond a kernel's design limit is reported, not hidden
                rec["error"] = str(e)[:300]
            wp.release_workspace()
            torch.cuda.empty_cache()
            out.append(rec)
    return out


CPU_STEPS = {0: 400, 1: 16, 2: 40, 3: 1, 4: 40}     # RK4 steps of one trajectory the oracle does in roughly 10-30 s


def cpu_sample(cfg_idx, n_rk4_steps):
    """The oracle, as it stands, on a bounded sample of the workload: ONE trajectory (the middle impact parameter) for
    n_rk4_steps RK4 steps around closest approach (same step size).  Returns (seconds, description, threads)."""
    from oracle import propagate as oprop
    from wpccc_inputs import build_config
    prob, run = build_config(cfg_idx)
    h = (run["z_max"] - run["z_min"]) / run["n_steps"]
    i = len(run["b"]) // 2
    t0, c0 = time.perf_counter(), time.process_time()
    oprop.propagate(prob, float(run["b"][i]), float(run["v"][i]), -0.5 * n_rk4_steps * h, 0.5 * n_rk4_steps * h, n_rk4_steps)
    dt, cpu = time.perf_counter() - t0, time.process_time() - c0
    # threads the oracle actually used: CPU time of the process (all threads) / wall time.  The oracle is numpy as it
    # stands: its matrix products run on the BLAS thread pool, everything else is single-threaded Python
    thr = max(1, int(round(cpu / dt)))
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
    n = {0: 50, 1: 2, 2: 5, 3: 1, 4: 5}[args.config]    # RK4 steps of one trajectory per bench "step" (bounded sample)
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
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs[i] of the headline line (default: the largest single-GPU configuration)")
    ap.add_argument("--per-config", dest="per_config", action="store_true", default=True, help="also measure the other four configurations (a few steps each) into per_config")
    ap.add_argument("--no-per-config", dest="per_config", action="store_false")
    ap.add_argument("--paper-shape", action="store_true", help="SURVEY.md 8(f) NEXT-3: also time the paper's own workload shape (l_max sweep on the geometric z-grid) into paper_shape")
    ap.add_argument("--cpu-steps", type=int, default=0, help="RK4 steps of the cpu_baseline sample (0: per-config default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--direct-tables", action="store_true", help="SURVEY.md 8(f) NEXT-1: radial sums from prefix/suffix tables instead of the DMMA GEMM (family direct_gemm then counts HBM bytes)")
    ap.add_argument("--window-steps", type=int, default=0, help="RK4 steps per bench step (windows walking through z from z_min) instead of the per-config default")
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
