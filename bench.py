#!/usr/bin/env python
"""bench.py - phase-space point-updates/s of the DVM outer iteration (arXiv 1810.00348) on B200, fp64.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config IDX] [--kernel auto|slice|tile]
    python bench.py --impl reference ...      # the CPU oracle on the host cores, bounded sample

A "step" is one outer iteration (all of DESIGN.md's hot-path rows a1-a7) of the workload.  Default workload:
BASELINE.json configs[4] (128^3 x 64^3 cavity, Kn = 0.01, memory-reduction path, f never materialised), the
largest single-GPU configuration and the one the target is stated on; --config picks another (0-4: BASELINE.json;
5: the paper's own cube run, 191 x 181 x 181 stretched cells x 48^3 velocities; 6: a 16-level slab of config 4 for ncu).
Default multi-GPU mode (replicas only): with --gpus N every rank runs an independent replica,
timing is max over ranks, value = total units / that time ("scaling": "weak").  --shard instead splits the velocity blocks
of ONE problem over the ranks (one fp64 all-reduce of the velocity sums per iteration; "scaling": "strong").
Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "phase-space point-updates/s (fp64, 1 B200)"
UNIT = "point-updates/s"


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            try:
                pw.append(float(f[2]))
            except ValueError:
                pass
            for nme, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        sm.sort(); pw.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm),
                "power_w": pw[len(pw) // 2] if pw else None}


def max_over_ranks(values, dist, device):
    """Device-timed figures are taken as the max over ranks (every rank ends up with the same list)."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_value(world, units_per_rank_step, ms_per_step):
    """Replicas only: every rank processes the same number of units per step."""
    return world * units_per_rank_step / (ms_per_step * 1e-3)


def workload_for(args):
    from paper_1810_00348_b200 import workloads
    return workloads.config(args.config)


# DESIGN.md section 6 (roofline).  Unit = one phase-space point-update.
#  * HBM: the tile kernel writes one fp64 face value per point and reads it back (4 x 4 tile columns): 8 B / point
#    algorithmic (16 B for the slice kernel's in-place slice), against the measured copy bandwidth of MEASURED_PEAKS.json.
#  * fp64 pipe: what the kernel EXECUTES, counted from its SASS and confirmed by ncu (profiles/): FP64_SLOTS_PER_POINT
#    warp-level fp64 instructions (DFMA / DADD / DMUL) per 32 points, each holding the 16-lane fp64 pipe of an SM
#    sub-partition for 2 clocks; peak = 148 SM x 64 lanes x 1.965 GHz FMA-lane-slots per second.  The 13 velocity sums run
#    on the fp64 tensor-core (DMMA) pipe and are reported separately.
#  * the figure SURVEY.md section 8(d) calls "algorithmic" (45 fp64 issue slots per point with one FMA per moment) is kept as
#    `algorithmic_equivalent`: the kernel does not execute those slots (factorised exp, tensor-core sums), so it is context,
#    not the roofline fraction.
# The binding roofline is the unit with the highest utilisation; bench.py computes both fractions live and names it.
ALGO_FP64_SLOTS_PER_POINT = 45.0
FP64_LANE_SLOTS_PEAK = 148 * 64 * 1.965e9          # fp64 FMA-lane issue slots per second
FP64_PEAK_TFLOPS = 2 * FP64_LANE_SLOTS_PEAK / 1e12
# ncu evidence per workload (profiles/r02_*.md), taken at the commit named there; None = not captured.
#   traffic: dram__bytes_read.sum + dram__bytes_write.sum per sweep launch; inst / fp64 / dmma: thread-level instructions per
#   point-update (smsp__inst_executed.sum x 32 / points, SASS opcode shares of the level loop); pipe / issue: ncu percentages
NCU = {
    "cfg4_cavity_128^3x64^3_Kn0.01": {"traffic": 4.3476e12, "inst_per_point": 29.1, "fp64_inst_per_point": 14.5, "dmma_per_point": 1.25,
                                      "pipe_fp64_active_pct": 36.6, "pipe_tensor_active_pct": 25.2, "pipe_shared_active_pct": 62.5,
                                      "issue_active_pct": 36.8, "commit": "42e5d51", "source": "profiles/r02_cfg4_counters.md"},
    "cfg3_cube_96x64x64_v48^3_Ma2": {"traffic": 3.3836e11, "inst_per_point": 31.2, "fp64_inst_per_point": 15.2, "dmma_per_point": 1.25,
                                     "pipe_fp64_active_pct": 34.2, "pipe_tensor_active_pct": 24.2, "pipe_shared_active_pct": 58.8,
                                     "issue_active_pct": 35.1, "commit": "42e5d51", "source": "profiles/r02_cfg4_counters.md"},
}
FP32_SLOTS_PER_POINT = 11.25                        # --precision mixed: fp32 instructions per point of the tile kernel (ncu, profiles/r02_mixed_precision.md)
FP32_LANE_SLOTS_PEAK = 148 * 128 * 1.965e9          # fp32 FMA-lane issue slots per second
FP64_SLOTS_PER_POINT = {"tile": 14.5, "slice": 70.0}   # executed fp64 instructions per point (SASS count)


def algorithmic_bytes_per_point(kernel_name, order=1):
    # one face value written and read back per point (tile), one in-place slice value (slice); two of each at order 2
    return {"slice": 16.0, "tile": 8.0}[kernel_name] * (2 if order == 2 else 1)


# --------------------------------------------------------------------------------------------------
def cpu_oracle_sample(wl, budget_s=15.0):
    """Time the oracle as it stands on a bounded sample: one outer iteration over a zero-weight velocity subset
    sized for ~budget_s seconds of CPU work (the oracle skips zero-weight velocities)."""
    from paper_1810_00348_b200 import workloads
    from oracle import dvm_oracle
    cores = os.cpu_count() or 1
    est_rate = 4.5e6 * cores   # measured on the GPU box's host: ~4e6 point-updates/s per thread
    n_vel_target = max(8, int(est_rate * budget_s / wl.n_fluid))
    keep = max(2, min(min(wl.mx, wl.my, wl.mz), int(round(n_vel_target ** (1.0 / 3.0)))))
    sub = workloads.sparse_weight_subset(wl, keep=keep) if keep < max(wl.mx, wl.my, wl.mz) else wl
    nv = int((sub.w_x > 0).sum() * (sub.w_y > 0).sum() * (sub.w_z > 0).sum())
    # cap host memory: every thread holds 13 long-double accumulators + one f per cell
    per_thread = wl.n_cells * (13 * 16 + 8)
    nthreads = max(1, min(cores, nv, int(24e9 // per_thread)))
    o = dvm_oracle.Oracle(sub)
    t0 = time.perf_counter()
    o.step(nthreads=nthreads)
    dt = time.perf_counter() - t0
    pts = wl.n_fluid * nv
    return {"value": pts / dt, "unit": UNIT, "cores": int(o.threads), "kind": "oracle",
            "sample": f"1 outer iteration over {nv} of {wl.n_vel} velocities (zero-weight subset, {keep} nodes/axis) "
                      f"x {wl.n_fluid} cells = {pts:.3e} points in {dt:.2f} s"}, dt, pts


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = workload_for(args)
    vals = []
    for i in range(args.warmup + args.steps):
        cb, dt, pts = cpu_oracle_sample(wl, budget_s=args.ref_budget)
        if i >= args.warmup:
            vals.append((dt, pts, cb))
    tot_t = sum(v[0] for v in vals)
    tot_p = sum(v[1] for v in vals)
    cb = dict(vals[-1][2]); cb["value"] = tot_p / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": tot_p / tot_t, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / len(vals), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "physical_cells": [wl.nx, wl.ny, wl.nz], "velocity_nodes": [wl.mx, wl.my, wl.mz],
                       "phase_points_per_iteration": wl.phase_points, "kernel": "oracle (CPU)", "parallelism": "host cores",
                       "note": "each step = one oracle iteration over a bounded velocity subset"},
            "cpu_baseline": cb,
            "e2e": {"value": tot_p / tot_t, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    from paper_1810_00348_b200 import dvm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if torch.cuda.device_count() <= local:
        sys.exit(f"bench.py: rank {rank} needs cuda:{local} but this node shows {torch.cuda.device_count()} GPU(s); there is no CPU fallback")
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")

    wl = workload_for(args)
    kernel = {"auto": dvm.KERNEL_AUTO, "slice": dvm.KERNEL_SLICE, "tile": dvm.KERNEL_TILE}[args.kernel]
    s = dvm.Solver(wl, kernel=kernel, device=f"cuda:{local}", max_f_mbytes=args.max_f_mbytes, tile_rv=args.tile_rv,
                   order=args.order, tile_axis=args.tile_axis,
                   precision=dvm.PREC_MIXED if args.precision == "mixed" else dvm.PREC_F64,
                   shard=(rank, world) if args.shard else None)
    # --shard: ONE problem, its velocity blocks spread over the ranks, one NCCL all-reduce of the velocity sums per iteration
    # (strong scaling).  Default: independent replicas (north_star: no sharding).
    iterate = (lambda n: s.iterate_sharded(n)) if args.shard else s.iterate
    mixed = args.precision == "mixed"
    stream = torch.cuda.current_stream(dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident timing: W warm-up steps, then exactly K steps ----
    iterate(args.warmup)
    barrier()
    l0 = s.launch_count()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    for k in range(args.steps):
        iterate(1)
        ev[k + 1].record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches = s.launch_count() - l0
    step_ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[args.steps])
    res = s.residual()

    # ---- end-to-end through the C ABI with host buffers (pinned), copies inside the timed region ----
    n8, n14 = 8 * wl.n_cells, 14 * wl.n_cells
    h_in = torch.empty(n8, dtype=torch.float64).pin_memory()
    h_rw = torch.empty(max(s.nface, 1), dtype=torch.float64).pin_memory()
    h_out = torch.empty(n14, dtype=torch.float64).pin_memory()
    h_rw_out = torch.empty(max(s.nface, 1), dtype=torch.float64).pin_memory()
    p14, rw = s.get_state()
    h_in.copy_(p14[:8].reshape(-1).cpu()); h_rw[: s.nface].copy_(rw.cpu())
    e2e_steps = max(1, min(args.steps, args.e2e_steps))

    def step_host():
        if not (args.shard and world > 1):
            return s.step_host(h_in, h_rw, 1, h_out, h_rw_out)
        # sharded: the same host -> device -> host round trip around the sweep / all-reduce / update of one iteration
        s.set_state(h_in.view(8, -1).to(dev, non_blocking=True), h_rw[: s.nface].to(dev, non_blocking=True))
        s.iterate_sharded(1)
        p14_, rw_ = s.get_state()
        h_out.copy_(p14_.reshape(-1), non_blocking=True); h_rw_out[: s.nface].copy_(rw_, non_blocking=True)
        torch.cuda.synchronize(dev)

    step_host()  # warm
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        step_host()
        h_in.copy_(h_out[:n8]); h_rw.copy_(h_rw_out)
    torch.cuda.synchronize(dev)
    e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_steps

    total_ms, e2e_ms = max_over_ranks([total_ms, e2e_ms], dist, dev)

    # ---- fp64 peak of this board, measured: register-resident DFMA chains on every SM, ~0.3 s, after the timed
    # region and under its own clock sampler, ~1.5 s (a pure fp64 stream is power-limited: the clock it holds is part of the result)
    fp64_probe = None
    if rank == 0 and not args.no_fp64_probe:
        torch.cuda.synchronize(dev)
        psampler = ClockSampler(local)
        psampler.start()
        dvm.fp64_peak_probe(f"cuda:{local}", rounds=1_000_000)                 # nvidia-smi comes up, clocks settle under the load
        rate, pms = dvm.fp64_peak_probe(f"cuda:{local}", rounds=8_000_000)     # ~1.3 s: several clock samples
        fp64_probe = {"lane_ops_per_s": rate, "tflops": 2e-12 * rate, "ms": pms, "clocks": psampler.stop(),
                      "kernel": "dfma_probe_kernel (csrc/fp64_probe.cu): 8 DFMA chains per thread, 2048 threads per SM",
                      "nominal_lane_ops_per_s": FP64_LANE_SLOTS_PEAK}
    total_bytes, f_bytes = s.workspace_bytes()

    if rank == 0:
        pts = wl.phase_points
        ms_per_step = total_ms / args.steps
        value = whole_job_value(1 if args.shard else world, pts, ms_per_step)
        kname = "slice" if s.kernel_used() == dvm.KERNEL_SLICE else "tile"
        peak, peak_src, _ = measured_peaks()
        # dominant kernel = the sweep (one launch per step); its duration is the step minus the small table / update launches,
        # measured here as the step itself (upper bound on the sweep time -> lower bound on achieved)
        bpp = algorithmic_bytes_per_point(kname, args.order) * (0.5 if mixed else 1.0)   # single-precision faces
        secs = ms_per_step * 1e-3
        hbm_gbs = bpp * pts / secs / 1e9
        # executed-instruction counts come from ncu captures of ONE variant per precision (order 1, the library's choice of the
        # tile variant, no workspace cap - or the slice kernel); for any other variant they are not evidence and are left out
        counted_variant = kname == "slice" or (args.order == 1 and args.tile_rv == 0 and args.tile_axis == 0 and args.max_f_mbytes == 0)
        alu = "fp32" if mixed else "fp64"
        if mixed:
            # single-precision sweep: 11.25 fp32 instructions per point (4 FADD + 3.25 FMUL + 4 FFMA, ncu) on the 128-lane
            # fp32 pipe; the fp64 side is one F2F (widening for the tensor-core sums) + 1.25 DMMA per point
            inst_per_point, lane_peak = FP32_SLOTS_PER_POINT, FP32_LANE_SLOTS_PEAK
        else:
            inst_per_point, lane_peak = FP64_SLOTS_PER_POINT[kname], FP64_LANE_SLOTS_PEAK      # executed fp64 lane slots
        alu_slots = inst_per_point * pts / secs if counted_variant else None
        frac_hbm = hbm_gbs / peak
        alu_peak_src = "derived: 148 SM x %d lanes x 2 flop x 1.965 GHz (DESIGN.md section 6)" % (128 if mixed else 64)
        if fp64_probe is not None and not mixed:
            lane_peak = fp64_probe["lane_ops_per_s"]          # the fp64 denominator is the measured one
            alu_peak_src = "measured in this run: dvm_fp64_peak_probe (roofline.fp64_peak_measured)"
        frac_alu = alu_slots / lane_peak if counted_variant else None
        # the ncu evidence belongs to the default variant (order 1, library's choice of the tile variant, no workspace cap)
        default_variant = not mixed and counted_variant and kname == "tile"
        ncu = NCU.get(wl.name, {}) if default_variant else {}
        if frac_alu is None or frac_hbm >= frac_alu:
            roof = {"bound": "hbm", "achieved": hbm_gbs, "peak": peak, "unit": "GB/s", "frac": frac_hbm,
                    "traffic": ncu.get("traffic"), "peak_source": peak_src}
        else:
            roof = {"bound": "alu", "achieved": 2.0 * alu_slots / 1e12, "peak": 2e-12 * lane_peak,
                    "unit": "TFLOP/s", "frac": frac_alu, "traffic": ncu.get("traffic"),
                    "peak_source": alu_peak_src}
        roof.update({"kernel": f"sweep_{kname}_kernel", "launch_ms": ms_per_step,
                     "algorithmic_bytes_per_point": bpp,
                     "algorithmic_bytes_source": "constant: the design's face traffic per point (DESIGN.md section 6); ncu dram bytes "
                                                 "of the default variant are in 'traffic' (profiles/r02_cfg4_counters.md)",
                     "hbm_achieved_gbs": hbm_gbs, "hbm_peak_gbs": peak, "hbm_frac": frac_hbm,
                     alu + "_executed_inst_per_point": inst_per_point if counted_variant else None,
                     alu + "_executed_tflops": 2.0 * alu_slots / 1e12 if counted_variant else None,
                     alu + "_peak_tflops": 2e-12 * lane_peak,
                     alu + "_pipe_frac": frac_alu,
                     alu + "_peak_source": alu_peak_src,
                     "fp64_peak_measured": fp64_probe,
                     alu + "_counts_note": None if counted_variant else "no instruction count was taken for this variant "
                                           "(order / velocities per thread / axis / workspace cap): pipe fraction not reported",
                     "algorithmic_equivalent": {"fp64_slots_per_point": ALGO_FP64_SLOTS_PER_POINT,
                                                "tflops": 2.0 * ALGO_FP64_SLOTS_PER_POINT * pts / secs / 1e12,
                                                "note": "SURVEY.md 8(d) count with one FMA per moment and a divide; not executed"},
                     "ncu": ncu,
                     "note": "no unit is saturated: the kernel is latency / issue bound at 8 warps per SM; the unit with the "
                             "highest utilisation is named as the bound"})
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None,
            "dtype": "f32 sweep, f64 moments" if mixed else "f64", "data": "synthetic",
            "config": {"workload": wl.name, "physical_cells": [wl.nx, wl.ny, wl.nz], "velocity_nodes": [wl.mx, wl.my, wl.mz],
                       "phase_points_per_iteration": pts, "kernel": kname, "precision": args.precision,
                       "tile_rv": s.tile_rv() if kname == "tile" else None,
                       "tile_axis": s.tile_axis() if kname == "tile" else None,
                       "order": args.order, "max_f_mbytes": args.max_f_mbytes,
                       "parallelism": ("velocity shards x%d, 1 all-reduce / iteration" % world) if args.shard and world > 1
                       else "replicas only" if world > 1 else "1 GPU",
                       "l2": "inputs larger than L2 (f workspace %.1f GB, fields %.2f GB)" % (f_bytes / 1e9, (total_bytes - f_bytes) / 1e9)
                       if total_bytes > 126e6 else "working set smaller than L2 (config is a parity case)",
                       "workspace_bytes": total_bytes, "f_workspace_bytes": f_bytes,
                       "full_6d_f_bytes_never_allocated": 8 * wl.n_cells * wl.n_vel,
                       "residual_after_run": [float(x) for x in res], "step_ms": [round(x, 3) for x in step_ms]},
            "roofline": roof,
            "e2e": {"value": whole_job_value(1 if args.shard else world, pts, e2e_ms), "unit": UNIT,
                    "h2d_bytes_per_step": 8 * (n8 + s.nface), "d2h_bytes_per_step": 8 * (n14 + s.nface)},
            "gpu_launches": int(launches),
            "clocks": clocks,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"], _, _ = cpu_oracle_sample(wl, budget_s=args.ref_budget)
        print(json.dumps(line))
    s.close()
    if dist is not None:
        dist.destroy_process_group()


def self_launch_command(gpus, argv, env):
    """The command that starts `gpus` ranks of this script (the driver's own launch line: torch.distributed.run, one node, one
    process per GPU, rendezvous on 127.0.0.1), or None when there is nothing to start: one GPU, or a launcher has already set
    WORLD_SIZE.  Host logic only - tests/test_bench_ranks.py checks it without a GPU."""
    if gpus <= 1 or "WORLD_SIZE" in env:
        return None
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), str(Path(__file__).resolve()), *argv]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--kernel", default="auto", choices=["auto", "slice", "tile"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--ref-budget", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fp64-probe", action="store_true", help="skip the 0.3 s fp64 peak measurement after the timed region")
    ap.add_argument("--max-f-mbytes", type=int, default=0, help="cap (MiB) on the f workspace of the tile kernel (0 = none)")
    ap.add_argument("--tile-rv", type=int, default=0, choices=[0, 2, 3, 4], help="velocities per thread of the tile kernel (0 = library's choice)")
    ap.add_argument("--tile-axis", type=int, default=0, choices=[0, 1, 2, 3], help="velocity axis in the wide role of the tile kernel (1 + axis; 0 = library's choice)")
    ap.add_argument("--order", type=int, default=1, choices=[1, 2], help="order of the upwind sweep")
    ap.add_argument("--shard", action="store_true",
                    help="with --gpus N: shard the velocity blocks of ONE problem over the N ranks (NCCL all-reduce of the velocity "
                         "sums per iteration, strong scaling) instead of N independent replicas")
    ap.add_argument("--precision", default="f64", choices=["f64", "mixed"],
                    help="f64 (BASELINE.json's metric) or mixed = the paper's timing precision: single-precision sweep, double moments")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    cmd = self_launch_command(args.gpus, sys.argv[1:], os.environ)
    if cmd is not None:
        # --gpus N without a launcher: start the N ranks here (one process per GPU, NCCL) and pass their output through;
        # rank 0 prints the one JSON line with n_gpus = N
        sys.exit(subprocess.run(cmd, env=dict(os.environ, NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "WARN"))).returncode)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE = {world} ranks")
    run_gpu(args)


if __name__ == "__main__":
    main()
