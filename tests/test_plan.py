"""Host logic of the tile sweep (no GPU): the work decomposition returned by dvm_plan_query must hand items out in an
order in which every dependency comes earlier - the property that rules out deadlock of the persistent kernel."""
import numpy as np
import pytest

from paper_1810_00348_b200 import dvm, workloads as W


def plan(wl, target=296, max_blocks=0, rv=0, order=1):
    return dvm.plan_query(wl.nx, wl.ny, wl.nz, wl.xi_x, wl.xi_y, wl.xi_z, target_ctas=target, max_blocks=max_blocks, rv=rv,
                          order=order)


@pytest.mark.parametrize("wl,target,max_blocks", [
    (W.config(0), 296, 0), (W.config(1), 296, 0), (W.config(2), 296, 0), (W.config(3), 296, 0),
    (W.cavity(0, 0, 0.1, nxyz=(13, 9, 11), mxyz=(10, 7, 9)), 296, 0),
    (W.cavity(0, 0, 0.1, nxyz=(13, 9, 11), mxyz=(10, 7, 9)), 4, 0),
    (W.cube_flow(4, 12, box=(6, 4, 4), vrange=8.0), 37, 0),
    (W.config(1), 296, 5), (W.config(2), 296, 24), (W.config(0), 296, 1),
    (W.cavity(0, 0, 0.1, nxyz=(13, 9, 11), mxyz=(10, 7, 9)), 16, 3),
])
@pytest.mark.parametrize("rv,order", [(4, 1), (3, 1), (2, 1), (2, 2)])
def test_items_cover_everything_once_in_dependency_order(wl, target, max_blocks, rv, order):
    counts, items = plan(wl, target, max_blocks, rv, order)
    n = counts["n_items"]
    assert len(items) == n == counts["n_vblocks"] * counts["ntx"] * counts["nty"]
    assert counts["ntx"] == -(-wl.nx // 4) and counts["nty"] in (-(-wl.ny // 4), -(-wl.ny // 2))   # tiles are 4 x 4 or 4 x 2
    vb, ti, tj, px, py, ps, xslot, octant, fslot = items.T
    B = counts["batch"]
    assert B == (min(max_blocks, counts["n_vblocks"]) if max_blocks else counts["n_vblocks"])
    assert np.array_equal(fslot, vb % B)
    later = vb >= B   # items of a later batch share their face slots with the block B places earlier
    # every (velocity block, tile) exactly once
    key = (vb.astype(np.int64) * counts["nty"] + tj) * counts["ntx"] + ti
    assert len(np.unique(key)) == n
    idx = np.arange(n)
    # predecessors are earlier items (or absent) ...
    for p in (px, py, ps):
        assert np.all((p == -1) | ((p >= 0) & (p < idx)))
    # ... and are the right ones: upwind tile in x / y of the same velocity block
    has = px >= 0
    assert np.array_equal(ti > 0, has)
    assert np.all(vb[px[has]] == vb[has]) and np.all(ti[px[has]] == ti[has] - 1) and np.all(tj[px[has]] == tj[has])
    has = (py >= 0) & (tj > 0)
    assert np.array_equal(tj > 0, has)
    assert np.all(vb[py[has]] == vb[has]) and np.all(tj[py[has]] == tj[has] - 1) and np.all(ti[py[has]] == ti[has])
    # first tile row of a later batch: waits for the last reader of its y-face slot in the previous batch
    first = (tj == 0)
    assert np.array_equal(py[first] >= 0, later[first])
    sel = first & later
    assert np.all(vb[py[sel]] == vb[sel] - B) and np.all(ti[py[sel]] == ti[sel]) and np.all(tj[py[sel]] == counts["nty"] - 1)
    # x-face slot reuse: the item that overwrites slot tj % P waits for the last reader of the previous user
    P = counts["P"]
    assert np.array_equal(xslot, tj % P)
    has = (ps >= 0) & (tj >= P)
    assert np.array_equal(has, (ti == 0) & (tj >= P))
    assert np.all(vb[ps[has]] == vb[has]) and np.all(ti[ps[has]] == counts["ntx"] - 1) and np.all(tj[ps[has]] == tj[has] - P)
    sel = (ti == 0) & (tj < P)
    assert np.array_equal(ps[sel] >= 0, later[sel])
    sel = sel & later
    assert np.all(vb[ps[sel]] == vb[sel] - B) and np.all(ti[ps[sel]] == counts["ntx"] - 1)
    assert np.all(tj[ps[sel]] % P == tj[sel] % P) and np.all(tj[ps[sel]] + P >= counts["nty"])
    # batches are handed out one after the other
    assert np.all(np.diff(vb // B) >= 0)


def test_velocity_blocks_partition_the_velocity_grid():
    """Octants come from node signs (the cube case has a shifted xi_x grid: unequal halves)."""
    wl = W.config(3)
    counts, items = plan(wl)
    assert (wl.xi_x < 0).sum() != (wl.xi_x >= 0).sum()
    # blocks of 16 x (8 x 4 | 4 x 8) nodes: at least ceil(n/512) per octant, all octants present
    assert set(np.unique(items[:, 7])) == set(range(8))
    assert counts["n_vblocks"] >= -(-wl.n_vel // 512)


def test_plan_rejects_bad_input():
    wl = W.config(0)
    with pytest.raises(dvm.DvmError):
        dvm.plan_query(0, 8, 8, wl.xi_x, wl.xi_y, wl.xi_z)


@pytest.mark.parametrize("cfg", [2, 3, 4])
@pytest.mark.parametrize("rv", [4, 3, 2])
def test_stratified_subset_puts_one_velocity_in_every_block(cfg, rv):
    """The full-size one-step parity cases keep one velocity per velocity block of the tile kernel (a zero-weight
    velocity is identically zero inside that kernel): exactly one kept velocity in each block of dvm_plan_vblocks, both
    signs present on every axis, and the in-block positions of the two seeds differ."""
    wl = W.config(cfg)
    boxes = dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, rv)
    counts, items = dvm.plan_query(wl.nx, wl.ny, wl.nz, wl.xi_x, wl.xi_y, wl.xi_z, rv=rv, max_items=1)
    assert len(boxes) == counts["n_vblocks"]
    kept = []
    for seed in (0, 1):
        sub = W.stratified_weight_subset(wl, boxes, seed)
        kx, ky, kz = (np.flatnonzero(w) for w in (sub.w_x, sub.w_y, sub.w_z))
        for b in boxes:
            n = (((kx >= b[0]) & (kx < b[0] + b[1])).sum() * ((ky >= b[2]) & (ky < b[2] + b[3])).sum()
                 * ((kz >= b[4]) & (kz < b[4] + b[5])).sum())
            assert n == 1
        assert len(kx) * len(ky) * len(kz) == len(boxes)
        for xi, k in ((wl.xi_x, kx), (wl.xi_y, ky), (wl.xi_z, kz)):
            assert (xi[k] < 0).any() and (xi[k] >= 0).any()
        kept.append((kx, ky, kz))
    assert not np.array_equal(kept[0][0], kept[1][0])


@pytest.mark.parametrize("rv,order,nvb,na", [(4, 1, 512, 16), (3, 1, 384, 12), (2, 1, 512, 8), (2, 2, 256, 8)])
def test_velocity_block_boxes(rv, order, nvb, na):
    """dvm_plan_vblocks: the boxes tile the velocity grid exactly once, stay inside one sign octant, and fit the lanes of
    the kernel variant (NA x nbb x ncb = velocities per block)."""
    wl = W.config(3)
    boxes = dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, rv, order)
    cover = np.zeros((wl.mx, wl.my, wl.mz), dtype=np.int32)
    for a0, n_a, b0, n_b, c0, n_c, code, shape in boxes:
        nbb, ncb = shape // 256, shape % 256
        NA, wide = code % 65536, code // 65536 - 1
        assert NA == na and NA * nbb * ncb == nvb
        lim = [0, 0, 0]
        lim[wide] = NA
        lim[[a for a in range(3) if a != wide][0]] = nbb
        lim[[a for a in range(3) if a != wide][1]] = ncb
        assert 0 < n_a <= lim[0] and 0 < n_b <= lim[1] and 0 < n_c <= lim[2]
        cover[a0:a0 + n_a, b0:b0 + n_b, c0:c0 + n_c] += 1
        for xi, lo, cnt in ((wl.xi_x, a0, n_a), (wl.xi_y, b0, n_b), (wl.xi_z, c0, n_c)):
            s = xi[lo:lo + cnt] >= 0
            assert s.all() or not s.any()
    assert (cover == 1).all()
    with pytest.raises(dvm.DvmError):
        dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, 4, 2)      # the second-order kernel carries 2 velocities per thread


def test_library_picks_the_variant_that_fills_its_lanes():
    """Config 3 (48 nodes per axis, xi_x shifted: 20 / 28 per sign, xi_y and xi_z 24 / 24): blocks 12 wide along xi_y or xi_z
    with 4 x 8 (xi_x x the other) pairs have no padded lane at all; config 4 (32 per sign half) keeps 16-wide blocks
    along xi_x; the paper's cube run (24 / 24 / 24) takes 12-wide blocks."""
    for cfg, na, fill in ((3, 12, 1.0), (4, 16, 1.0), (5, 12, 1.0), (2, 16, 1.0)):
        wl = W.config(cfg)
        boxes = dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z)
        NA, wide = boxes[0][6] % 65536, boxes[0][6] // 65536 - 1
        nvb = NA * (boxes[0][7] // 256) * (boxes[0][7] % 256)
        assert NA == na
        assert wl.n_vel / (len(boxes) * nvb) == pytest.approx(fill)
        if cfg == 3:
            assert wide in (1, 2)


@pytest.mark.parametrize("wide", [1, 2, 3])
def test_plans_with_every_wide_axis(wide):
    wl = W.cavity(0, 0, 0.1, nxyz=(13, 9, 11), mxyz=(10, 7, 9))
    for rv, order in ((4, 1), (3, 1), (2, 2)):
        boxes = dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, rv, order, wide)
        assert all(b[6] // 65536 == wide for b in boxes)
        cover = np.zeros((wl.mx, wl.my, wl.mz), dtype=np.int32)
        for a0, n_a, b0, n_b, c0, n_c, code, shape in boxes:
            cover[a0:a0 + n_a, b0:b0 + n_b, c0:c0 + n_c] += 1
        assert (cover == 1).all()
        counts, items = dvm.plan_query(wl.nx, wl.ny, wl.nz, wl.xi_x, wl.xi_y, wl.xi_z, rv=rv, order=order, wide_axis=wide)
        assert counts["n_vblocks"] == len(boxes)
