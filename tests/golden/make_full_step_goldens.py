#!/usr/bin/env python
"""Writes tests/golden/full_step_cfg<N>.txt: ONE outer iteration of the CPU oracle over the FULL velocity grid of a
BASELINE.json config ("one full-weight cfg4 step is run once and archived"), from the seeded
perturbed state the GPU test reproduces.  Calls only oracle/ and the input generators; never the CUDA path.

    python tests/golden/make_full_step_goldens.py --configs 2 3 4 [--out DIR] [--threads N]

Cost: config 2 ~4 min and config 3 ~23 min on 7 threads of an 8-core container; config 4 (5.5e11 phase points) 51 min on the 16 host
threads of the GPU box (1.8e8 points/s).
The file holds, as repr(float) text: residual triple, mass-rescale factor, per field (14) the maximum absolute value,
the sum and the sum of squares over fluid cells, the 14 fields at SAMPLE_CELLS seeded fluid cells, and the wall density at
SAMPLE_FACES seeded wall faces.  tests/test_parity_gpu.py::test_full_weight_step_against_archived_oracle compares the GPU
step with it (fields 1e-11, residual 1e-9).
"""
import argparse
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

from oracle import dvm_oracle            # noqa: E402
from paper_1810_00348_b200 import workloads as W   # noqa: E402

SAMPLE_CELLS, SAMPLE_FACES = 384, 192
STATE_SEED = {2: 1002, 3: 1003, 4: 1004}


def seeded_state(cfg):
    """(workload, prim8 state, sample cell indices) - shared with the GPU test through this module"""
    wl = W.config(cfg)
    prim = W.perturbed_state(wl, seed=STATE_SEED[cfg], amp_q=0.005)
    rng = np.random.default_rng(STATE_SEED[cfg] + 7)
    fluid = np.arange(wl.n_cells) if wl.solid is None else np.flatnonzero(wl.solid.reshape(-1) == 0)
    cells = np.sort(rng.choice(fluid, size=min(SAMPLE_CELLS, len(fluid)), replace=False))
    return wl, prim, cells


def sample_faces(nface, rho_w, cfg):
    rng = np.random.default_rng(STATE_SEED[cfg] + 11)
    walls = np.flatnonzero(rho_w != 0.0)
    if len(walls) == 0:
        return walls
    return np.sort(rng.choice(walls, size=min(SAMPLE_FACES, len(walls)), replace=False))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[2, 3, 4])
    ap.add_argument("--out", default=str(Path(__file__).resolve().parent))
    ap.add_argument("--threads", type=int, default=0)
    args = ap.parse_args()
    out = Path(args.out)
    out.mkdir(parents=True, exist_ok=True)
    for cfg in args.configs:
        wl, prim, cells = seeded_state(cfg)
        o = dvm_oracle.Oracle(wl)
        o.set_state(prim, None)          # wall densities: those of the uniform initial state (odvm_init_state)
        t0 = time.time()
        p14 = o.step(nthreads=args.threads)
        dt = time.time() - t0
        fluid = np.ones(wl.n_cells, bool) if wl.solid is None else wl.solid.reshape(-1) == 0
        faces = sample_faces(o.nface, o.rho_w, cfg)
        lines = [f"# full-weight oracle step of {wl.name}: {wl.n_fluid} fluid cells x {wl.n_vel} velocities = {wl.phase_points:.4e} points",
                 f"# written by tests/golden/make_full_step_goldens.py (oracle only), {o.threads} threads, {dt:.0f} s",
                 f"# state: workloads.perturbed_state(seed={STATE_SEED[cfg]}, amp_q=0.005), wall densities of the initial state",
                 "resid " + " ".join(repr(float(x)) for x in o.resid),
                 "scale " + repr(float(o.scale))]
        for m in range(14):
            f = p14[m][fluid]
            lines.append(f"field {m} " + " ".join(repr(float(x)) for x in (np.abs(f).max(), f.sum(), (f * f).sum())))
        for c in cells:
            lines.append(f"cell {int(c)} " + " ".join(repr(float(x)) for x in p14[:, c]))
        for fidx in faces:
            lines.append(f"face {int(fidx)} " + repr(float(o.rho_w[fidx])))
        (out / f"full_step_cfg{cfg}.txt").write_text("\n".join(lines) + "\n")
        print(f"cfg{cfg}: {dt:.0f} s, {wl.phase_points / dt:.3e} points/s, wrote {out / f'full_step_cfg{cfg}.txt'}", flush=True)


if __name__ == "__main__":
    main()
