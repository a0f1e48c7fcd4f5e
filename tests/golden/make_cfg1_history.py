#!/usr/bin/env python
"""Writes tests/golden/history_cfg1.txt: the CPU oracle's 200 outer iterations of BASELINE.json configs[1] (32^3 cells x 24^3
velocities, Kn = 0.1) from the uniform initial state - the residual triple (reading G9) and the
mass-rescale factor of EVERY iteration, and the 14 macroscopic fields at SAMPLE_CELLS seeded cells plus the
wall density at SAMPLE_FACES seeded faces every FIELD_EVERY iterations.  Calls only oracle/ and the input generators; never
the CUDA path.

    python tests/golden/make_cfg1_history.py [--iterations 200] [--threads N] [--out DIR]

Cost: about 25 minutes on 7 threads of an 8-core container (4.4e8 phase points per iteration).
tests/test_parity_gpu.py::test_config1_200_iterations_against_archived_oracle_history runs the GPU solver freely for the same
200 iterations and compares the whole history with this file.
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

SAMPLE_CELLS, SAMPLE_FACES, FIELD_EVERY, SEED = 192, 96, 25, 1001


def samples(wl, nface):
    """(cell indices, face indices) - shared with the GPU test through this module"""
    rng = np.random.default_rng(SEED)
    cells = np.sort(rng.choice(wl.n_cells, size=SAMPLE_CELLS, replace=False))
    faces = np.sort(rng.choice(nface, size=SAMPLE_FACES, replace=False))
    return cells, faces


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--iterations", type=int, default=200)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--out", default=str(Path(__file__).resolve().parent))
    args = ap.parse_args()
    wl = W.config(1)
    o = dvm_oracle.Oracle(wl)
    cells, faces = samples(wl, o.nface)
    lines = []
    t0 = time.time()
    for it in range(1, args.iterations + 1):
        p14 = o.step(nthreads=args.threads)
        lines.append(f"iter {it} " + " ".join(repr(float(x)) for x in (*o.resid, o.scale)))
        if it % FIELD_EVERY == 0 or it == args.iterations:
            for m in range(14):
                lines.append(f"fmax {it} {m} " + repr(float(np.abs(p14[m]).max())))
            for c in cells:
                lines.append(f"cell {it} {int(c)} " + " ".join(repr(float(x)) for x in p14[:, c]))
            for f in faces:
                lines.append(f"face {it} {int(f)} " + repr(float(o.rho_w[f])))
        if it % 10 == 0:
            print(f"iteration {it}: resid {o.resid}, {time.time() - t0:.0f} s", flush=True)
    dt = time.time() - t0
    head = [f"# oracle history of {wl.name}: {args.iterations} iterations from the uniform initial state, {wl.phase_points:.4e} points each",
            f"# written by tests/golden/make_cfg1_history.py (oracle only), {o.threads} threads, {dt:.0f} s",
            "# iter n r_rho r_mom r_E scale | fmax n field max|field| | cell n index 14 fields | face n index rho_w"]
    out = Path(args.out)
    out.mkdir(parents=True, exist_ok=True)
    (out / "history_cfg1.txt").write_text("\n".join(head + lines) + "\n")
    print(f"wrote {out / 'history_cfg1.txt'} in {dt:.0f} s")


if __name__ == "__main__":
    main()
