"""Velocity-space sharding, host side, on CPU:
the partition of the velocity blocks over the ranks, and the sweep -> all-reduce -> update loop of the binding over two gloo
ranks with the oracle's partial velocity sums standing in for the GPU sweep (the sweep itself needs a GPU: the emulated-rank
parity test is tests/test_parity_gpu.py::test_velocity_shards_emulated_on_one_gpu)."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

from paper_1810_00348_b200 import workloads as W

ROOT = Path(__file__).resolve().parents[1]


def _boxes(b):
    return sorted(tuple(int(x) for x in row[:6]) for row in b)


@pytest.mark.parametrize("cfg", [0, 3, 4])
@pytest.mark.parametrize("count", [2, 3, 8])
def test_shards_partition_the_velocity_blocks(cfg, count):
    """Every velocity block of the unsharded plan belongs to exactly one rank; rank sizes differ by at most one."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(cfg)
    full = _boxes(dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z))
    parts = [_boxes(dvm.plan_shard_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, r, count)) for r in range(count)]
    assert sorted(sum(parts, [])) == full
    assert len(set(sum(parts, []))) == len(full)
    sizes = [len(p) for p in parts]
    assert max(sizes) - min(sizes) <= 1
    # and every velocity node triple is covered exactly once
    cover = np.zeros((wl.mx, wl.my, wl.mz), dtype=int)
    for p in parts:
        for (x0, nx, y0, ny, z0, nz) in p:
            cover[x0:x0 + nx, y0:y0 + ny, z0:z0 + nz] += 1
    assert (cover == 1).all()


def test_more_shards_than_blocks_is_an_error():
    from paper_1810_00348_b200 import dvm
    wl = W.config(0)          # 8 velocity blocks (one per octant)
    assert len(dvm.plan_shard_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, 7, 8)) == 1
    with pytest.raises(dvm.DvmError):
        dvm.plan_shard_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, 8, 9)
    with pytest.raises(dvm.DvmError):
        dvm.plan_shard_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    from oracle import dvm_oracle
    from paper_1810_00348_b200 import dvm
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.config(0)
    full = dvm_oracle.Oracle(wl)
    prim, rho_w = full.prim8.copy(), full.rho_w.copy()
    full.step(nthreads=1)
    # this rank's share of the velocity sums: the oracle restricted to each of its velocity blocks (weights zeroed outside the
    # block's box; same state and wall densities), summed
    part = np.zeros((13, wl.n_cells))
    for row in dvm.plan_shard_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, rank, world):
        x0, nx, y0, ny, z0, nz = (int(v) for v in row[:6])
        def keep(w, a, n):
            m = np.zeros_like(w); m[a:a + n] = w[a:a + n]; return m
        o = dvm_oracle.Oracle(wl.with_(w_x=keep(wl.w_x, x0, nx), w_y=keep(wl.w_y, y0, ny), w_z=keep(wl.w_z, z0, nz)))
        o.set_state(prim, rho_w)
        o.step(nthreads=1)
        part += o.raw13

    class HostShard(dvm.Solver):
        """The binding's sharded loop with the GPU calls replaced by the oracle's partial sums."""
        def __init__(self):
            self.shard = (rank, world)
            self.buf = torch.zeros(13 * wl.n_cells, dtype=torch.float64)
            self.calls, self.results = [], []
        def sweep(self):
            self.buf.copy_(torch.from_numpy(part.reshape(-1))); self.calls.append("sweep")
        def update(self):
            self.results.append(self.buf.clone().numpy()); self.calls.append("update")
        def reduce_buffer(self):
            return self.buf
        def plan_signature(self):
            return sig
        def close(self):
            pass
        def __del__(self):
            pass

    sig = (2, 4, 1, 0)
    s = HostShard()
    s.iterate_sharded(2)
    # ranks whose libraries planned different block shapes must be stopped before the first all-reduce
    sig = (2, 4 - rank, 1, 0)
    bad = HostShard()
    try:
        bad.iterate_sharded(1)
        mismatch = "not detected"
    except dvm.DvmError as e:
        mismatch = "detected" if "different sweeps" in str(e) and bad.calls == ["sweep"] else f"wrong state {e} {bad.calls}"
    dist.barrier()
    dist.destroy_process_group()
    err = max(float(np.abs(r.reshape(13, -1) - full.raw13).max()) for r in s.results)
    out.put((rank, s.calls, err, float(part[0].max()), float(full.raw13[0].max()), float(np.abs(full.raw13).max()), mismatch))


def test_sweep_allreduce_update_loop_over_two_gloo_ranks():
    """Two ranks: each holds half of the velocity blocks' sums (from the oracle); after the binding's all-reduce both hold
    the full sums of the unsharded oracle step, in the order sweep, update, sweep, update."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, calls, err, rho_part, rho_full, fmax, mismatch in res:
        assert calls == ["sweep", "update", "sweep", "update"]
        assert mismatch == "detected"
        assert err <= 1e-13 * fmax
        assert rho_part < 0.75 * rho_full          # a rank alone holds only a part of the density sum
