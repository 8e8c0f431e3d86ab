#!/usr/bin/env python
"""Writes the full-trajectory goldens of SURVEY.md 8(d) "T2 propagation": final amplitudes X(z_max) (PAPER.md L106:
"X(z_max) ... yields the transition probabilities") and the drift max |c^H S c - 1| of whole trajectories of the five
BASELINE.json configs, computed by the CPU oracle ONLY (this script imports `oracle/` and `wpccc_inputs/`, nothing of
the CUDA path; the -m gpu tests load the files and compare the CUDA result with them to 1e-9).

    python tests/golden/make_trajectory_goldens.py --config 1 --pick 0        # one trajectory -> traj_cfg1_pick0.npz
    python tests/golden/make_trajectory_goldens.py --list                      # the picks

Picks: cfg 0 all four b x 1000 steps; cfg 1 b indices {0, 8, 15} x 1600 steps; cfg 2 and cfg 4 the
first / middle / last (v, b) of the trajectory list x 4000 steps; cfg 3 two b on the window z in [-6, 6], 300 steps of
the configured size 0.04 (a full cfg 3 trajectory is days of oracle time), chosen where the configured quadrature
leaves the overlap matrix positive definite (A23).  Hours of CPU time in total; run once, files committed.
Each file records the git commit and the SHA-256 of every oracle / input-generator source it was computed with.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import subprocess
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import propagate as oprop          # noqa: E402
from wpccc_inputs import build_config          # noqa: E402

# config -> list of (v index, b index); window: None = the configured z-range, else (z_min, z_max, n_steps)
PICKS = {
    0: dict(traj=[(0, 0), (0, 1), (0, 2), (0, 3)], window=None),
    1: dict(traj=[(0, 0), (0, 8), (0, 15)], window=None),
    2: dict(traj=[(0, 0), (1, 32), (2, 63)], window=None),
    3: dict(traj=[(0, 100), (0, 127)], window=(-6.0, 6.0, 300)),
    4: dict(traj=[(0, 0), (6, 48), (11, 95)], window=None),
}


def source_hashes():
    out = {}
    for pkg in ("oracle", "wpccc_inputs"):
        d = os.path.join(ROOT, pkg)
        for f in sorted(os.listdir(d)):
            if f.endswith(".py"):
                out["%s/%s" % (pkg, f)] = hashlib.sha256(open(os.path.join(d, f), "rb").read()).hexdigest()
    return out


def git_head():
    try:
        return subprocess.run(["git", "-C", ROOT, "rev-parse", "HEAD"], capture_output=True, text=True, check=True).stdout.strip()
    except Exception:
        return "unknown"


def trajectory(cfg, pick):
    from wpccc_inputs.configs import CONFIGS
    c = CONFIGS[cfg]
    iv, ib = PICKS[cfg]["traj"][pick]
    b, v = float(np.asarray(c["b"], float)[ib]), float(np.asarray(c["v"], float)[iv])
    win = PICKS[cfg]["window"]
    z0, z1, n = (c["z_min"], c["z_max"], c["n_steps"]) if win is None else win
    return b, v, float(z0), float(z1), int(n), iv, ib


def path_of(cfg, pick):
    return os.path.join(HERE, "traj_cfg%d_pick%d.npz" % (cfg, pick))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int)
    ap.add_argument("--pick", type=int)
    ap.add_argument("--list", action="store_true")
    a = ap.parse_args()
    if a.list:
        for cfg in PICKS:
            for k in range(len(PICKS[cfg]["traj"])):
                print(cfg, k, trajectory(cfg, k), os.path.exists(path_of(cfg, k)))
        return
    cfg, pick = a.config, a.pick
    b, v, z0, z1, n, iv, ib = trajectory(cfg, pick)
    prob, _ = build_config(2 if cfg == 4 else cfg)          # configs[4] shares the basis of configs[2]
    t0 = time.perf_counter()
    C, drift = oprop.propagate(prob, b, v, z0, z1, n, track_norm=True)
    dt = time.perf_counter() - t0
    hs = source_hashes()
    np.savez(path_of(cfg, pick), C=C, drift=np.float64(drift), b=np.float64(b), v=np.float64(v), z_min=np.float64(z0), z_max=np.float64(z1),
             n_steps=np.int64(n), iv=np.int64(iv), ib=np.int64(ib), config=np.int64(cfg), git=np.array(git_head()),
             sources=np.array(sorted(hs.items())), oracle_seconds=np.float64(dt))
    print("configs[%d] pick %d: b=%.6g v=%.6g %d steps, %.0f s, drift %.3e, sum|c|^2 %.12f -> %s" % (
        cfg, pick, b, v, n, dt, drift, float((np.abs(C) ** 2).sum()), path_of(cfg, pick)))


if __name__ == "__main__":
    main()
