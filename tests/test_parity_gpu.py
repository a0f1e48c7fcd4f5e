"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances: macroscopic fields 1e-11 relative (max-norm per field, G17) after
EVERY iteration, residual history 1e-9 (BASELINE.json north_star)."""
import numpy as np
import pytest

from paper_1810_00348_b200 import workloads as W
from tests.parity import assert_fields, assert_residual

pytestmark = pytest.mark.gpu

KERNELS = [1, 2]  # DVM_KERNEL_SLICE, DVM_KERNEL_TILE


def fluid_mask(wl):
    return None if wl.solid is None else wl.solid.reshape(-1) == 0


def make(wl, kernel, **kw):
    """Every kernel variant exists on a B200: a failure to create or configure one is a test failure, never a skip."""
    from paper_1810_00348_b200 import dvm
    return dvm.Solver(wl, kernel=kernel, **kw)


def compare_step(s, o, what, check_raw=True):
    """GPU solver `s` and oracle `o` have just taken one iteration from the same state: compare everything."""
    fm = fluid_mask(o.wl)
    g14 = s.moments().cpu().numpy()
    errs = assert_fields(g14, o.prim14, fm, what=what)
    assert_residual(s.residual(), o.resid, what=what)
    g_rw = s.get_state()[1].cpu().numpy()
    assert np.abs(g_rw - o.rho_w).max() <= 1e-11 * np.abs(o.rho_w).max(), what
    assert abs(s.mass_scale() - o.scale) <= 1e-12 * abs(o.scale), what
    if check_raw:
        graw = s.raw_moments().cpu().numpy()
        for m in range(13):
            sc = np.abs(o.raw13[m]).max()
            assert np.abs(graw[m] - o.raw13[m]).max() <= 1e-11 * max(sc, 1e-3), (what, m)
        gfl = s.wall_flux().cpu().numpy()
        assert np.abs(gfl - o.flux_out).max() <= 1e-11 * np.abs(o.flux_out).max(), what
    return errs


def lockstep(wl, kernel, iters, oracle_mod, state=None, rho_w=None, check_raw=True, **kw):
    o = oracle_mod.Oracle(wl)
    s = make(wl, kernel, **kw)
    if state is not None:
        o.set_state(state, rho_w)
        s.set_state(state, rho_w)
    assert s.nface == o.nface
    g_rw0 = s.get_state()[1].cpu().numpy()
    if state is None:
        assert np.allclose(g_rw0, o.rho_w, rtol=1e-13, atol=0)
    worst = {}
    for it in range(iters):
        s.iterate(1)
        o.step()
        errs = compare_step(s, o, f"{wl.name} kernel {kernel} {kw} iteration {it + 1}", check_raw)
        for k_, v in errs.items():
            worst[k_] = max(worst.get(k_, 0), v)
    hist = s.residual_history()
    assert hist.shape == (iters, 3)
    for it in range(iters):
        assert_residual(hist[it], o.history[it], what=f"history {it}")
    s.close()
    return worst


@pytest.mark.parametrize("kernel", KERNELS)
def test_config0_every_iteration(oracle_mod, kernel):
    """BASELINE.json configs[0]: 8^3 x 8^3, Kn = 1, 20 iterations, parity after every iteration."""
    lockstep(W.config(0), kernel, 20, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_config1_perturbed_one_step(oracle_mod, kernel):
    """BASELINE.json configs[1] kernel-level test: 32^3 x 24^3, fields perturbed by seeded noise (seed 1810)."""
    wl = W.config(1)
    st = W.perturbed_state(wl, seed=1810)
    lockstep(wl, kernel, 1, oracle_mod, state=st, rho_w=np.ones(6 * 32 * 32))


@pytest.mark.parametrize("kernel", KERNELS)
def test_config1_perturbed_with_heat_flux(oracle_mod, kernel):
    """seed-348 variant with q += U(-0.01, 0.01)^3 to exercise the Shakhov term; two steps."""
    wl = W.config(1)
    st = W.perturbed_state(wl, seed=348, amp_q=0.01)
    lockstep(wl, kernel, 2, oracle_mod, state=st, rho_w=np.ones(6 * 32 * 32))


@pytest.mark.parametrize("kernel", KERNELS)
def test_config1_lockstep_first_iterations(oracle_mod, kernel):
    """Config 1 in lock-step with the oracle, every field and the residual after every iteration (the full 200
    iterations would take the oracle ~25 minutes; the bench kernel gets 10, the baseline kernel 4)."""
    lockstep(W.config(1), kernel, 10 if kernel == 2 else 4, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_ragged_nonuniform_cavity(oracle_mod, kernel):
    """Sizes that are not multiples of any tile or block: 13 x 9 x 11 tanh-stretched cells, 10 x 7 x 9 velocities
    (odd counts put a node at xi = 0: octants of unequal size)."""
    wl = W.cavity(0, 0, 0.075, stretch=1.5, nxyz=(13, 9, 11), mxyz=(10, 7, 9))
    lockstep(wl, kernel, 3, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_cube_flow_small(oracle_mod, kernel):
    """Config-3 structure at reduced size: free stream + zero-gradient outflow + solid mask, shifted velocity grid."""
    wl = W.cube_flow(4, 12, box=(6, 4, 4), vrange=8.0)
    lockstep(wl, kernel, 3, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_degenerate_shapes(oracle_mod, kernel):
    """One cell thick in y and z with zero-gradient side faces (the 1-D special case), and a single velocity per octant."""
    wl = W.cavity(1, 6, 0.5, nxyz=(12, 1, 1))
    zg = W.FaceBC(W.ZERO_GRADIENT)
    wl = wl.with_(faces=[W.FaceBC(W.WALL_DIFFUSE, 1.2, 1.0, (0, 0, 0)), W.FaceBC(W.FREESTREAM, 0.9, 1.1, (0.1, 0, 0)),
                         zg, zg, zg, zg], rescale_mass=0)
    lockstep(wl, kernel, 2, oracle_mod)
    lockstep(W.cavity(3, 2, 1.0), kernel, 2, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_closed_box_fixed_point(oracle_mod, kernel):
    """P7 on the GPU: equilibrium gas in a closed box with stationary isothermal walls stays put; asserts on field
    deviations (the momentum residual is rounding noise there)."""
    wl = W.cavity(8, 24, 0.1, U_w=0.0)
    s = make(wl, kernel)
    for it in range(2):
        s.iterate(1)
        g = s.moments().cpu().numpy()
        assert np.abs(g[0] - 1).max() < 1e-12 and np.abs(g[4] - 1).max() < 1e-12
        assert np.abs(g[1:4]).max() < 1e-12 and np.abs(g[5:]).max() < 1e-12
    s.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_closed_box_with_solid_block(oracle_mod, kernel):
    """P12 on the GPU: equilibrium gas around a masked block in a closed box stays put; then the same geometry with the lid
    moving, in lock-step with the oracle (solid ghosts on the slow path of the tile kernel, mass rescale with a mask)."""
    wl = W.cavity(6, 24, 0.1, U_w=0.0)
    solid = np.zeros((6, 6, 6), dtype=np.uint8)
    solid[2:4, 1:3, 3:5] = 1
    wl = wl.with_(solid=solid)
    s = make(wl, kernel)
    s.iterate(2)
    g = s.moments().cpu().numpy()
    fluid = solid.reshape(-1) == 0
    assert np.abs(g[0][fluid] - 1).max() < 1e-12 and np.abs(g[4][fluid] - 1).max() < 1e-12 and np.abs(g[1:4]).max() < 1e-12
    assert np.abs(g[:, ~fluid]).max() == 0.0
    s.close()
    lockstep(W.cavity(6, 12, 0.3).with_(solid=solid), kernel, 3, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_uniform_free_stream_is_preserved(oracle_mod, kernel):
    """P11 on the GPU: an empty box with free-stream faces at the state of the gas keeps that state, and agrees with the
    oracle; non-uniform ragged grid."""
    fs = W.FaceBC(W.FREESTREAM, 1.1, 0.9, (0.3, -0.2, 0.1))
    wl = W.cavity(0, 24, 0.2, stretch=1.5, nxyz=(6, 5, 7)).with_(
        faces=[fs] * 6, rescale_mass=0, rho0=0.9, u0=(0.3, -0.2, 0.1), T0=1.1)
    s = make(wl, kernel)
    o = oracle_mod.Oracle(wl)
    for it in range(2):
        s.iterate(1)
        c = o.step()
        g = s.moments().cpu().numpy()
        assert np.abs(g[0] - 0.9).max() < 1e-11 and np.abs(g[4] - 1.1).max() < 1e-11 and np.abs(g[1] - 0.3).max() < 1e-11
        assert np.abs(g - c).max() < 1e-13   # q and sigma are ~1e-12 here: absolute comparison with the oracle
    s.close()


def stratified(wl, seed, rv=0):
    """One velocity in every velocity block of the tile kernel: the tile kernel carries
    g = w f, so a velocity of weight 0 is identically 0 inside it and only the kept ones test anything - hence one per
    block, at rotating in-block positions, instead of a handful of random nodes."""
    from paper_1810_00348_b200 import dvm
    return W.stratified_weight_subset(wl, dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, rv), seed)


@pytest.mark.parametrize("seed", [0, 1])
@pytest.mark.parametrize("kernel", KERNELS)
def test_config2_full_size_stratified_step(oracle_mod, kernel, seed):
    """Config 2 at full physical size (64^3 tanh grid, 32^3 velocities), one velocity per velocity block (64): one step
    from a perturbed state; raw moments, wall fluxes, wall densities, fields and residual must agree."""
    wl = stratified(W.config(2), seed)
    st = W.perturbed_state(wl, seed=2 + seed, amp_q=0.01 * seed)
    lockstep(wl, kernel, 1, oracle_mod, state=st, rho_w=None)


@pytest.mark.parametrize("seed", [0, 1])
def test_config3_full_size_stratified_step(oracle_mod, seed):
    """Config 3 at full size (96 x 64 x 64 cells with the 16^3 solid cube, 48^3 shifted velocity grid) in the launch
    configuration bench.py times (tile kernel), one velocity in each of its 288 velocity blocks: one step from the
    free-stream state (seed 0) or from a perturbed state (seed 1)."""
    wl = stratified(W.config(3), seed)
    if seed == 0:
        lockstep(wl, 2, 1, oracle_mod)
    else:
        lockstep(wl, 2, 1, oracle_mod, state=W.perturbed_state(wl, seed=3, amp_q=0.01), rho_w=None)


@pytest.mark.parametrize("seed", [0, 1])
def test_config4_full_size_stratified_step(oracle_mod, seed):
    """Config 4 at full size (128^3 cells x 64^3 velocities: 5.5e11 phase points swept by the GPU), one velocity in each
    of the 512 velocity blocks (the oracle sweeps those 512): one step from a perturbed state; raw moments, wall
    fluxes, wall densities, fields and residual must agree."""
    wl = stratified(W.config(4), seed)
    st = W.perturbed_state(wl, seed=4 + seed, amp_q=0.01 * seed)
    lockstep(wl, 2, 1, oracle_mod, state=st, rho_w=None)


def test_initial_wall_density_closed_form_gpu(oracle_mod):
    """rho_w^0 straight after dvm_create on configs[3] (Mach-2 free stream hitting the cube: u_0 . n != 0) against the closed
    half-range flux of the drifting Maxwellian, rho_0 [sqrt(T_0/4 pi) e^{-S^2} + (U_n/2)(1 + erf S)] / sqrt(T_w/4 pi) with
    S = U_n / sqrt T_0 (Eq.(9); oracle step 1; CPU pin test_initial_wall_density_with_gas_moving_into_the_wall):
    the library computes rho_w^0 in its own host code, and lock-step tests only show that it equals the oracle's.  The cube's
    upstream faces start at 6.48, its lee faces at 0.004, the side faces at 1; tolerance = the second-order error of the
    half-range trapezoid sums, 0.02 h^2."""
    from math import erf, exp, pi, sqrt
    wl = W.config(3)
    s = make(wl, 2)
    o = oracle_mod.Oracle(wl)
    cell, dirn, _ = o.face_table()
    rw = s.get_state()[1].cpu().numpy()
    s.close()
    assert rw.shape == cell.shape
    h = wl.xi_x[1] - wl.xi_x[0]
    walls = np.flatnonzero((cell >= 0) & (rw > 0))
    assert len(walls) == 6 * 16 * 16            # the faces of the 16^3 cube; the domain faces are not walls
    for d in range(6):
        un = wl.u0[d // 2] * (1.0 if d & 1 else -1.0)
        S = un / sqrt(wl.T0)
        closed = wl.rho0 * (sqrt(wl.T0 / (4 * pi)) * exp(-S * S) + 0.5 * un * (1.0 + erf(S))) / sqrt(wl.solid_bc.T / (4 * pi))
        sel = walls[dirn[walls] == d]
        assert len(sel) == 256
        assert np.abs(rw[sel] - closed).max() <= 0.02 * h * h, (d, rw[sel][0], closed)
    front, rear = rw[walls[dirn[walls] == 1]][0], rw[walls[dirn[walls] == 0]][0]
    assert front > 1000 * rear


def test_paper_cube_full_size_stratified_step(oracle_mod):
    """The paper's own cube workload (bench --config 5: 191 x 181 x 181 stretched cells with the 31^3 solid cube, 48^3
    velocities: 6.9e11 phase points swept by the GPU) at full size in the launch configuration bench.py times (RV = 3), one
    velocity in each of the 288 velocity blocks (the oracle sweeps those: 1.8e9 points), one step from a perturbed state with
    heat flux."""
    wl = stratified(W.config(5), 1)
    lockstep(wl, 2, 1, oracle_mod, state=W.perturbed_state(wl, seed=55, amp_q=0.01), rho_w=None, check_raw=False)


@pytest.mark.parametrize("rv", [2, 3])
def test_config3_stratified_step_other_variants(oracle_mod, rv):
    """The RV = 2 (8 x 8 x 8 velocity blocks) and RV = 3 (12 x 8 x 4) variants of the tile kernel on config 3 at full size, one
    velocity per block."""
    wl = stratified(W.config(3), 1, rv=rv)
    lockstep(wl, 2, 1, oracle_mod, state=W.perturbed_state(wl, seed=33), rho_w=None, tile_rv=rv)


def test_paper_cube_grid_runs_on_the_variant_chosen_for_it(oracle_mod):
    """The paper's cube run has 24 nodes per sign half on every axis: the library picks the 12-wide RV = 3 variant for it
    (no padded lanes); reduced-size grid with that velocity grid, in lock-step."""
    wl = W.cube_flow_paper(5, 6, 6, 7, 48)
    s = make(wl, 2)
    s.iterate(1)
    assert s.tile_rv() == 3
    s.close()
    lockstep(stratified(wl, 0), 2, 2, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_paper_cube_grid_small(oracle_mod, kernel):
    """The paper's own cube workload shape at reduced size: geometric
    cell expansion 1.02 / 1.03 away from the solid cube, unshifted velocity grid on [-4, 4]^3, free stream on all six
    outer faces, Kn = 1; sizes that are not multiples of the tile (18 x 17 x 17 cells)."""
    wl = W.cube_flow_paper(5, 6, 6, 7, 12)
    lockstep(wl, kernel, 3, oracle_mod)


def test_workspace_cap_batches(oracle_mod):
    """DVM_OPT_MAX_F_MBYTES (smaller velocity batches cap the memory of the stored f): config 1 with the f
    workspace capped well below the uncapped size sweeps its 27 velocity blocks in batches; same results."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(1)
    s0 = dvm.Solver(wl, kernel=2)
    s0.iterate(1)
    _, f_full = s0.workspace_bytes()
    s0.close()
    cap_mb = max(1, int(f_full / 4 / 2**20))
    o = oracle_mod.Oracle(wl)
    s = dvm.Solver(wl, kernel=2, max_f_mbytes=cap_mb)
    for it in range(3):
        s.iterate(1)
        c14 = o.step()
        assert_fields(s.moments().cpu().numpy(), c14, what=f"capped workspace, iteration {it + 1}")
        assert_residual(s.residual(), o.resid)
    _, f_cap = s.workspace_bytes()
    assert f_cap <= cap_mb * 2**20 and f_cap < f_full / 3
    s.close()


def test_P10_paper_iteration_count_soft_pin():
    """Soft pin P10: the paper's cavity run (Kn = 1, 64^3 x 64^3, U_w = 0.1 v_m, velocity range
    [-4, 4]^3, trapezoid rule) reaches its 1e-9 criterion in 36 iterations on a K40.  The criterion's exact form is our
    reading G9 (max of three norm ratios), so the count is only required to land near the paper's; GPU only (one oracle
    iteration of this size is ~20 core-minutes)."""
    from paper_1810_00348_b200 import dvm
    wl = W.cavity(64, 64, 1.0, vrange=4.0, U_w=0.1)
    s = dvm.Solver(wl)
    n = 0
    while n < 80:
        s.iterate(4)
        n += 4
        if s.residual().max() < 1e-9:
            break
    hist = s.residual_history().max(axis=1)
    first = int(np.argmax(hist < 1e-9)) + 1
    assert hist[-1] < 1e-9, hist[-5:]
    assert 25 <= first <= 50, first
    assert np.all(np.diff(np.log(hist[2:first])) < 0)   # monotone convergence
    print("P10: residual < 1e-9 after", first, "iterations (paper: 36)")
    s.close()


def test_P10b_paper_cube_iteration_count_soft_pin():
    """Soft pin for the paper's second case (supersonic flow past a cube, Ma = 2, Kn = 1, 191 x 181 x 181 cells x
    48^3 velocities, converged "after 41 iterations"), like P10 for the cavity.  The paper gives neither its grid cell by cell
    (the streamwise split 75 + 31 + 85 of the 191 cells is ours, workloads.cube_flow_paper) nor the exact form of its criterion
    (reading G9), so the count only has to land near 41: 35 <= n <= 60 to 1e-9, falling monotonically.  GPU only: 6.9e11 phase
    points per iteration, about 1.8 s each here (one oracle iteration of this size: hours)."""
    from paper_1810_00348_b200 import dvm
    wl = W.cube_flow_paper()
    s = dvm.Solver(wl)
    n = 0
    while n < 72:
        s.iterate(4)
        n += 4
        if s.residual().max() < 1e-9:
            break
    hist = s.residual_history().max(axis=1)
    first = int(np.argmax(hist < 1e-9)) + 1
    assert hist[-1] < 1e-9, hist[-5:]
    assert 35 <= first <= 60, first
    assert np.all(np.diff(np.log(hist[2:first])) < 0)   # monotone convergence
    print("P10b: residual < 1e-9 after", first, "iterations (paper: 41)")
    s.close()


def test_config1_long_run_history_is_sane():
    """Config 1 for its full 200 iterations on the GPU: finite fields, residual decreasing to its rounding floor,
    mass conserved by the rescale (G18) - properties that hold without the oracle (200 oracle iterations take ~25 min)."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(1)
    s = dvm.Solver(wl)
    s.iterate(200)
    hist = s.residual_history()
    assert hist.shape == (200, 3) and np.isfinite(hist).all()
    assert hist[199].max() < 1e-3 * hist[1].max()
    g = s.moments().cpu().numpy()
    assert np.isfinite(g).all()
    vol = np.outer(np.outer(np.diff(wl.zf), np.diff(wl.yf)).reshape(-1), np.diff(wl.xf)).reshape(-1)
    assert abs((g[0] * vol).sum() - 1.0) < 1e-12
    # mirror symmetry in y (G11) survives 200 iterations on the GPU up to reduction-order noise
    r = g.reshape(14, wl.nz, wl.ny, wl.nx)
    assert np.abs(r[0] - r[0][:, ::-1, :]).max() < 1e-10 and np.abs(r[2] + r[2][:, ::-1, :]).max() < 1e-10
    s.close()


def test_errors_and_state_roundtrip():
    from paper_1810_00348_b200 import dvm
    wl = W.config(0)
    s = dvm.Solver(wl)
    with pytest.raises(dvm.DvmError):
        s.residual()  # before the first iteration
    s.iterate(3)
    p, r = s.get_state()
    s2 = dvm.Solver(wl)
    s2.set_state(p[:8].contiguous(), r)
    s.iterate(1)
    s2.iterate(1)
    assert (s.moments() - s2.moments()).abs().max().item() < 1e-13  # checkpoint / resume
    total, fbytes = s.workspace_bytes()
    assert fbytes < total
    bad = wl.with_(xf=wl.xf[::-1].copy())
    with pytest.raises(dvm.DvmError):
        dvm.Solver(bad)
    s.close(); s2.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_f_never_materialised(kernel):
    """Memory-reduction path: the f workspace holds faces / one slice per velocity, never the
    6-D array; config 1 (32^3 x 24^3: the 6-D f would be 3.6 GB)."""
    wl = W.config(1)
    s = make(wl, kernel)
    s.iterate(1)
    total, fbytes = s.workspace_bytes()
    assert fbytes < 8 * wl.n_cells * wl.n_vel / 6
    s.close()


# ---------------------------------------------------------------------------------------------------------------------
# Round 2: dense cases with several x-blocks per sign half, GPU counterparts of pins P13-P16, the one-step map along the
# real trajectories, run-to-run reproducibility, the dependency protocol under stress.
VARIANTS = [(1, {}), (2, {"tile_rv": 4, "tile_axis": 1}), (2, {"tile_rv": 3, "tile_axis": 1}), (2, {"tile_rv": 2, "tile_axis": 1}),
            (2, {"tile_rv": 4, "tile_axis": 2}), (2, {"tile_rv": 3, "tile_axis": 3}), (2, {"tile_rv": 2, "tile_axis": 3})]


@pytest.mark.parametrize("kernel,kw", VARIANTS)
def test_dense_wide_velocity_grid(oracle_mod, kernel, kw):
    """Every lane compared: 40 xi_x nodes (20 per sign half = 16 + 4 for RV = 4, 8 + 8 + 4 for RV = 2: several x-blocks per
    half, the last partly filled) x 10 x 9, on 6 x 5 x 7 cells; then the same grid shifted so that the halves are 17 / 23."""
    wl = W.cavity(0, 0, 0.3, nxyz=(6, 5, 7), mxyz=(40, 10, 9))
    lockstep(wl, kernel, 2, oracle_mod, state=W.perturbed_state(wl, seed=40, amp_q=0.01), rho_w=None, **kw)
    sh = wl.with_(xi_x=wl.xi_x + 0.9, name=wl.name + "_shifted")
    assert (sh.xi_x < 0).sum() == 17
    lockstep(sh, kernel, 2, oracle_mod, **kw)


@pytest.mark.parametrize("kernel,kw", VARIANTS)
def test_moving_hot_walls(oracle_mod, kernel, kw):
    """GPU counterparts of pins P13 / P14 / P3b: walls with T_w != 1 moving with three non-zero velocity components
    (lock-step), and the gas drifting with its walls stays put (Eq.(8), reading G3)."""
    faces = [W.FaceBC(W.WALL_DIFFUSE, 0.7, 1.0, (0.0, 0.12, -0.07)), W.FaceBC(W.WALL_DIFFUSE, 1.3, 1.0, (0.0, -0.05, 0.1)),
             W.FaceBC(W.WALL_DIFFUSE, 1.1, 1.0, (0.2, 0.0, 0.05)), W.FaceBC(W.WALL_DIFFUSE, 0.9, 1.0, (-0.1, 0.0, 0.0)),
             W.FaceBC(W.WALL_DIFFUSE, 1.2, 1.0, (0.16, -0.08, 0.0)), W.FaceBC(W.WALL_DIFFUSE, 0.8, 1.0, (-0.16, 0.04, 0.0))]
    wl = W.cavity(0, 12, 0.4, nxyz=(6, 5, 7)).with_(faces=faces)
    lockstep(wl, kernel, 3, oracle_mod, **kw)
    fs = W.FaceBC(W.FREESTREAM, 1.2, 0.9, (0.3, 0.0, 0.0))
    wall = W.FaceBC(W.WALL_DIFFUSE, 1.2, 1.0, (0.3, 0.0, 0.0))
    ch = W.cavity(0, 32, 0.2, vrange=7.0, stretch=1.5, nxyz=(5, 4, 6)).with_(
        faces=[fs, fs, wall, wall, wall, wall], rescale_mass=0, rho0=0.9, u0=(0.3, 0.0, 0.0), T0=1.2)
    s = make(ch, kernel, **kw)
    s.iterate(2)
    g = s.moments().cpu().numpy()
    assert np.abs(g[0] - 0.9).max() < 1e-11 and np.abs(g[4] - 1.2).max() < 1e-11 and np.abs(g[1] - 0.3).max() < 1e-11
    assert np.abs(g[2:4]).max() < 1e-11 and np.abs(g[5:]).max() < 1e-11
    s.close()


def test_config1_200_iterations_against_archived_oracle_history():
    """BASELINE.json configs[1] for its full 200 iterations, GPU running freely from the initial state, against the oracle's own
    200 iterations archived in tests/golden/history_cfg1.txt (written by tests/golden/make_cfg1_history.py, which calls only
    oracle/; ~45 min of host cores, hence archived): the residual triple of EVERY iteration at 1e-9 r + 1e-13 (north_star
    "residual histories must agree to 1e-9") - the absolute term takes over where the residual reaches its
    rounding floor, which the test locates and reports - the mass-rescale factor of the last iteration at 1e-12, and every 25
    iterations the 14 fields at 192 seeded cells (1e-11 of the field's max norm) and the wall density at 96 seeded faces."""
    from pathlib import Path
    import importlib.util
    from paper_1810_00348_b200 import dvm
    gdir = Path(__file__).parent / "golden"
    spec = importlib.util.spec_from_file_location("make_cfg1_history", gdir / "make_cfg1_history.py")
    mh = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mh)                      # for the seeded sample indices; the oracle is not run here
    wl = W.config(1)
    hist, fmax, cellv, facev = {}, {}, {}, {}
    for line in (gdir / "history_cfg1.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, n, *v = line.split()
        n = int(n)
        if k == "iter":
            hist[n] = np.array([float(x) for x in v])
        elif k == "fmax":
            fmax.setdefault(n, {})[int(v[0])] = float(v[1])
        elif k == "cell":
            cellv.setdefault(n, {})[int(v[0])] = np.array([float(x) for x in v[1:]])
        elif k == "face":
            facev.setdefault(n, {})[int(v[0])] = float(v[1])
    assert sorted(hist) == list(range(1, 201)) and sorted(cellv) == list(range(25, 201, 25))
    s = dvm.Solver(wl, kernel=dvm.KERNEL_TILE)
    cells, faces = mh.samples(wl, s.nface)
    groups = {"rho": [0], "u": [1, 2, 3], "T": [4], "q": [5, 6, 7], "sigma": [8, 9, 10, 11, 12, 13]}
    done = 0
    for n in sorted(cellv):
        s.iterate(n - done)
        done = n
        g14, rw = s.get_state()
        g14, rw = g14.cpu().numpy(), rw.cpu().numpy()
        assert sorted(cellv[n]) == [int(c) for c in cells] and sorted(facev[n]) == [int(f) for f in faces]
        gold = np.stack([cellv[n][int(c)] for c in cells], axis=1)           # [14][cells]
        for name, idx in groups.items():
            scale = max(fmax[n][m] for m in idx)
            err = np.abs(g14[idx][:, cells] - gold[idx]).max()
            assert err <= 1e-11 * scale, (n, name, err / scale)
        gw = np.array([facev[n][int(f)] for f in faces])
        assert np.abs(rw[faces] - gw).max() <= 1e-11 * np.abs(gw).max(), n
    gh = s.residual_history()
    assert gh.shape == (200, 3)
    for n in range(1, 201):
        assert_residual(gh[n - 1], hist[n][:3], what=f"config 1, iteration {n} of 200")
    scal = np.array([hist[n][3] for n in range(1, 201)])
    assert abs(s.mass_scale() - scal[-1]) <= 1e-12 * scal[-1]
    # where the oracle's residual stops falling (its rounding floor): from there on the comparison is the absolute 1e-13
    r = np.array([hist[n][:3].max() for n in range(1, 201)])
    floor_at = next((n for n in range(1, 200) if r[n:].min() > 0.5 * r[n - 1] and r[n - 1] < 1e-10), None)
    print(f"cfg1: residual {r[0]:.2e} -> {r[-1]:.2e}; oracle rounding floor reached at iteration {floor_at}")
    assert r[-1] < 1e-9 * r[1]
    s.close()


def test_config1_one_step_map_along_the_200_iterations(oracle_mod):
    """the GPU runs config 1 for its 200 iterations; at n = 50, 100, 199 the state is handed to
    the oracle, which takes ONE iteration from it; fields, wall densities, raw sums, wall fluxes and residual of the
    GPU's own next iteration must agree with it (the full lock-step of 200 oracle iterations would take ~25 minutes)."""
    wl = W.config(1)
    s = make(wl, 2)
    o = oracle_mod.Oracle(wl)
    done = 0
    for n in (50, 100, 199):
        s.iterate(n - done)
        p14, rw = s.get_state()
        o.set_state(p14[:8].cpu().numpy(), rw.cpu().numpy())
        s.iterate(1)
        o.step()
        compare_step(s, o, f"config 1, iteration {n} -> {n + 1}")
        done = n + 1
    assert s.iterations_done() == 200
    hist = s.residual_history()
    assert hist.shape == (200, 3) and hist[199].max() < 1e-3 * hist[1].max()
    s.close()


def test_config2_runs_to_residual_1e6_with_one_step_checks(oracle_mod):
    """BASELINE.json configs[2]: run to residual 1e-6 (cap 5000) on the GPU with the full velocity grid; at the initial
    state, half way and at the converged state, the one-step map is checked against the oracle on the stratified velocity
    subset (one velocity per block; an oracle iteration over all 32^3 velocities is ~2 core-hours)."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(2)
    s = make(wl, 2)
    states = [tuple(x.cpu().numpy() for x in s.get_state())]
    n = 0
    while n < 5000:
        s.iterate(20)
        n += 20
        if s.residual().max() < 1e-6:
            break
    hist = s.residual_history().max(axis=1)
    first = int(np.argmax(hist < 1e-6)) + 1
    assert hist[-1] < 1e-6, (n, hist[-3:])
    print("config 2: residual < 1e-6 after", first, "iterations")
    assert hist[first - 1] < hist[first // 2] < hist[5]
    states.append(tuple(x.cpu().numpy() for x in s.get_state()))
    s.close()
    # a state half way: rerun to first // 2 (cheap: ~20 ms per iteration)
    s = make(wl, 2)
    s.iterate(first // 2)
    states.insert(1, tuple(x.cpu().numpy() for x in s.get_state()))
    s.close()
    sub = stratified(wl, 0)
    for idx, (p14, rw) in enumerate(states):
        o = oracle_mod.Oracle(sub)
        g = make(sub, 2)
        o.set_state(p14[:8], rw)
        g.set_state(p14[:8], rw)
        g.iterate(1)
        o.step()
        compare_step(g, o, f"config 2 one-step map at sampled state {idx}")
        g.close()


def test_run_to_run_reproducibility():
    """The REDs of the tile kernel land in an order that varies from run to run (north_star: 'reduction order only'):
    two runs of 5 iterations of a ragged case agree to 1e-12, far inside the 1e-11 parity tolerance."""
    wl = W.cavity(0, 0, 0.075, stretch=1.5, nxyz=(13, 9, 11), mxyz=(20, 14, 18))
    out = []
    for rep in range(2):
        s = make(wl, 2)
        s.iterate(5)
        out.append(s.moments().cpu().numpy())
        s.close()
    scale = np.abs(out[0]).max(axis=1, keepdims=True) + 1e-300
    assert (np.abs(out[0] - out[1]) / scale).max() < 1e-12


@pytest.mark.parametrize("ctas", [1, 4])
@pytest.mark.parametrize("rv", [4, 3, 2])
def test_dependency_protocol_under_stress(oracle_mod, ctas, rv):
    """compute-sanitizer is closed on this pool, so the done-flag / face-slot protocol of the tile kernel is stressed
    instead: many velocity blocks (5 x 3 x 5 per axis and octant pattern), tiny tiles (9 x 10 x 3 cells), a workspace cap
    that forces several batches sharing face slots, and a persistent grid of 1 or 4 CTAs so that items are picked up long
    after their predecessors finished or right behind them.  Lock-step with the oracle."""
    wl = W.cavity(0, 0, 0.2, nxyz=(9, 10, 3), mxyz=(36, 20, 18))
    full = make(wl, 2, tile_rv=rv)
    full.iterate(1)
    _, fbytes = full.workspace_bytes()
    full.close()
    lockstep(wl, 2, 2, oracle_mod, state=W.perturbed_state(wl, seed=77), rho_w=None, tile_rv=rv, max_ctas=ctas,
             max_f_mbytes=max(1, int(fbytes / 3 / 2**20)))


# ---------------------------------------------------------------------------------------------------------------------
# Second-order upwind sweep (DVM_OPT_ORDER = 2; oracle pins in tests/test_oracle_order2.py), both kernels:
# the slice kernel with a second stored slice, the tile kernel with two z-planes in registers and two-deep faces.
@pytest.mark.parametrize("kernel", KERNELS)
def test_order2_config0_every_iteration(oracle_mod, kernel):
    lockstep(W.config(0).with_(order=2), kernel, 20, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_order2_ragged_stretched_cavity(oracle_mod, kernel):
    wl = W.cavity(0, 0, 0.075, stretch=1.5, nxyz=(13, 9, 11), mxyz=(10, 7, 9)).with_(order=2)
    lockstep(wl, kernel, 3, oracle_mod)
    wide = W.cavity(0, 0, 0.3, nxyz=(6, 5, 7), mxyz=(40, 10, 9)).with_(order=2)
    lockstep(wide, kernel, 2, oracle_mod, state=W.perturbed_state(wide, seed=41, amp_q=0.01), rho_w=None)


@pytest.mark.parametrize("kernel", KERNELS)
def test_order2_cube_flows(oracle_mod, kernel):
    """free stream + zero-gradient outflow + solid mask; then the paper's stretched cube grid at reduced size"""
    lockstep(W.cube_flow(4, 12, box=(6, 4, 4), vrange=8.0).with_(order=2), kernel, 3, oracle_mod)
    lockstep(W.cube_flow_paper(5, 6, 6, 7, 12).with_(order=2), kernel, 3, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_order2_degenerate_and_solid_block(oracle_mod, kernel):
    wl = W.cavity(1, 6, 0.5, nxyz=(12, 1, 1))
    zg = W.FaceBC(W.ZERO_GRADIENT)
    wl = wl.with_(faces=[W.FaceBC(W.WALL_DIFFUSE, 1.2, 1.0, (0, 0, 0)), W.FaceBC(W.FREESTREAM, 0.9, 1.1, (0.1, 0, 0)),
                         zg, zg, zg, zg], rescale_mass=0, order=2)
    lockstep(wl, kernel, 2, oracle_mod)
    solid = np.zeros((6, 6, 6), dtype=np.uint8)
    solid[2:4, 1:3, 3:5] = 1
    lockstep(W.cavity(6, 12, 0.3).with_(solid=solid, order=2), kernel, 3, oracle_mod)
    lockstep(W.cavity(3, 2, 1.0).with_(order=2), kernel, 2, oracle_mod)


@pytest.mark.parametrize("kernel", KERNELS)
def test_order2_config1_first_iterations(oracle_mod, kernel):
    wl = W.config(1).with_(order=2)
    lockstep(wl, kernel, 3, oracle_mod, state=W.perturbed_state(wl, seed=1810, amp_q=0.01), rho_w=np.ones(6 * 32 * 32))


def test_order2_config3_full_size_stratified_step(oracle_mod):
    """second-order tile kernel on config 3 at full size, one velocity in each of its (256-velocity) blocks"""
    from paper_1810_00348_b200 import dvm
    wl = W.config(3).with_(order=2)
    sub = W.stratified_weight_subset(wl, dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, 2, 2), 1)
    lockstep(sub, 2, 1, oracle_mod, state=W.perturbed_state(sub, seed=35, amp_q=0.01), rho_w=None)


def test_order2_fixed_points_on_the_tile_kernel():
    wl = W.cavity(8, 24, 0.1, U_w=0.0).with_(order=2)
    s = make(wl, 2)
    s.iterate(2)
    g = s.moments().cpu().numpy()
    assert np.abs(g[0] - 1).max() < 1e-12 and np.abs(g[4] - 1).max() < 1e-12 and np.abs(g[1:4]).max() < 1e-12
    assert s.tile_rv() == 2
    s.close()


# ---------------------------------------------------------------------------------------------------------------------
# Full-weight steps against the archived oracle: tests/golden/full_step_cfg<N>.txt is written by
# tests/golden/make_full_step_goldens.py (oracle only; config 4 took ~1.9 h of 16 host cores) - every velocity of the
# configuration contributes, not a subset.
def _golden_full_steps():
    from pathlib import Path
    return sorted(int(p.stem.split("cfg")[1]) for p in (Path(__file__).parent / "golden").glob("full_step_cfg*.txt"))


@pytest.mark.parametrize("cfg", _golden_full_steps())
def test_full_weight_step_against_archived_oracle(cfg):
    from pathlib import Path
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_goldens", Path(__file__).parent / "golden" / "make_full_step_goldens.py")
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)                      # imports oracle/ (test infrastructure) for the writer; not used here
    wl, prim, cells = mg.seeded_state(cfg)
    gold = {"cell": {}, "face": {}, "field": {}}
    for line in (Path(__file__).parent / "golden" / f"full_step_cfg{cfg}.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        if k == "resid":
            gold["resid"] = np.array([float(x) for x in v])
        elif k == "scale":
            gold["scale"] = float(v[0])
        else:
            gold[k][int(v[0])] = np.array([float(x) for x in v[1:]])
    s = make(wl, 2)
    s.set_state(prim, None)
    s.iterate(1)
    g14 = s.moments().cpu().numpy()
    rw = s.get_state()[1].cpu().numpy()
    assert sorted(gold["cell"]) == [int(c) for c in cells]
    fmax = np.array([gold["field"][m][0] for m in range(14)])
    groups = {"rho": [0], "u": [1, 2, 3], "T": [4], "q": [5, 6, 7], "sigma": [8, 9, 10, 11, 12, 13]}
    for name, idx in groups.items():
        scale = fmax[idx].max()
        err = max(np.abs(g14[idx, c] - gold["cell"][c][idx]).max() for c in gold["cell"])
        assert err <= 1e-11 * scale, (name, err / scale)
    fluid = np.ones(wl.n_cells, bool) if wl.solid is None else wl.solid.reshape(-1) == 0
    for m in range(14):
        f = g14[m][fluid]
        amax, ssum, ssq = gold["field"][m]
        assert abs(np.abs(f).max() - amax) <= 1e-11 * fmax[[i for i in groups.values() if m in i][0]].max()
        assert abs((f * f).sum() - ssq) <= 1e-10 * max(ssq, 1e-300)
        assert abs(f.sum() - ssum) <= 1e-10 * np.abs(f).sum()
    for fidx, val in gold["face"].items():
        assert abs(rw[fidx] - val[0]) <= 1e-11 * abs(val[0])
    assert_residual(s.residual(), gold["resid"], what=f"archived full-weight step of config {cfg}")
    assert abs(s.mass_scale() - gold["scale"]) <= 1e-12 * abs(gold["scale"])
    s.close()


@pytest.mark.parametrize("axis", [1, 2, 3])
@pytest.mark.parametrize("rv,order", [(4, 1), (3, 1), (2, 2)])
def test_every_wide_axis_of_the_tile_kernel(oracle_mod, axis, rv, order):
    """DVM_OPT_TILE_AXIS: the velocity axis that plays the wide role (RV nodes per thread x 4 lane groups) is a free choice;
    every choice on a ragged stretched cavity with unequal node counts per axis (10 x 7 x 9), on the cube flow (shifted
    xi_x, solid block: slow path) and on a wide grid with several blocks along each axis."""
    kw = {"tile_rv": rv, "tile_axis": axis}
    wl = W.cavity(0, 0, 0.075, stretch=1.5, nxyz=(13, 9, 11), mxyz=(10, 7, 9)).with_(order=order)
    lockstep(wl, 2, 2, oracle_mod, **kw)
    lockstep(W.cube_flow(4, 12, box=(6, 4, 4), vrange=8.0).with_(order=order), 2, 2, oracle_mod, **kw)
    wide = W.cavity(0, 0, 0.3, nxyz=(6, 5, 7), mxyz=(18, 26, 34)).with_(order=order)
    lockstep(wide, 2, 1, oracle_mod, state=W.perturbed_state(wide, seed=60 + axis, amp_q=0.01), rho_w=None, **kw)


# ---------------------------------------------------------------------------------------------------------------------
# Velocity-space sharding (DVM_OPT_SHARD_COUNT): one GPU stands in for n ranks.  The n
# solvers run one after the other (no kernel waits on another); the sum of their accumulators stands in for the all-reduce.
@pytest.mark.parametrize("nranks,case", [(2, "cfg0"), (3, "ragged"), (2, "cube"), (4, "cfg1"), (2, "mixed"), (3, "order2")])
def test_velocity_shards_emulated_on_one_gpu(oracle_mod, nranks, case):
    from paper_1810_00348_b200 import dvm
    kw = {}
    if case == "cfg0":
        wl, iters = W.config(0), 5
    elif case == "ragged":
        wl, iters = W.cavity(0, 0, 0.075, stretch=1.5, nxyz=(13, 9, 11), mxyz=(10, 7, 9)), 3
    elif case == "cube":
        wl, iters = W.cube_flow(4, 12, box=(6, 4, 4), vrange=8.0), 3
    elif case == "cfg1":
        wl, iters = W.config(1), 2
    elif case == "order2":
        wl, iters, kw = W.cavity(0, 0, 0.3, stretch=1.5, nxyz=(9, 6, 7), mxyz=(12, 8, 10)).with_(order=2), 3, dict(order=2)
    else:
        wl, iters, kw = W.config(0), 3, dict(precision=dvm.PREC_MIXED)
    o = oracle_mod.Oracle(wl)
    ranks = [dvm.Solver(wl, kernel=2, shard=(r, nranks), **kw) for r in range(nranks)]
    fm = fluid_mask(wl)
    for it in range(iters):
        for s in ranks:
            s.sweep()
        total = sum(s.reduce_buffer() for s in ranks)          # stands in for the all-reduce
        part_rho = [float(s.reduce_buffer().view(-1, 16)[:, 0].sum()) for s in ranks]
        for s in ranks:
            s.reduce_buffer().copy_(total)
            s.update()
        o.step()
        what = f"{case} {nranks} ranks iteration {it + 1}"
        assert all(0 < p < (1 - 1e-9) * sum(part_rho) for p in part_rho), what       # every rank holds a part, none all of it
        g14 = ranks[0].moments().cpu().numpy()
        if case == "mixed":
            from tests.parity import tol32
            assert np.abs(g14 - o.prim14).max() <= 3 * tol32(wl), what
        else:
            assert_fields(g14, o.prim14, fm, what=what)
            assert_residual(ranks[0].residual(), o.resid, what=what)
            assert np.abs(ranks[0].get_state()[1].cpu().numpy() - o.rho_w).max() <= 1e-11 * np.abs(o.rho_w).max(), what
        # the replicated state is bit-identical on every rank (same sums, same update)
        for s in ranks[1:]:
            assert np.array_equal(s.moments().cpu().numpy(), g14), what
    # a sharded solver refuses the unsharded calls
    with pytest.raises(dvm.DvmError):
        ranks[0].iterate(1)
    with pytest.raises(dvm.DvmError):
        ranks[0].update()
    for s in ranks:
        s.close()


def test_sweep_update_is_iterate_with_one_rank(oracle_mod):
    """dvm_sweep; dvm_update on an unsharded solver is dvm_iterate(1) (same launches): lock-step with the oracle; the slice
    kernel refuses the split."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(0)
    o = oracle_mod.Oracle(wl)
    s = make(wl, 2)
    for it in range(3):
        s.sweep()
        with pytest.raises(dvm.DvmError):
            s.sweep()
        s.update()
        o.step()
        compare_step(s, o, f"sweep/update iteration {it + 1}")
    s.iterate_sharded(1)
    o.step()
    compare_step(s, o, "iterate_sharded with one rank")
    s.close()
    s = make(wl, 1)
    with pytest.raises(dvm.DvmError):
        s.sweep()
    s.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_free_molecular_plates_converged_solution(oracle_mod, kernel):
    """GPU counterpart of pins P17 / P18: Couette flow and heat transfer between parallel plates at Kn = 1e9, 40 iterations on a
    6 x 1 x 1 channel with 24^3 velocities: the converged GPU fields equal the oracle's (1e-11) and carry the textbook
    free-molecular shear stress -rho U / (2 sqrt pi) and heat flux F (T1 - T2) / (2 sqrt pi) up to the 4 % quadrature error of
    the half-range sums at this node spacing (P17 / P18 show that error is second order)."""
    import math
    zg = W.FaceBC(W.ZERO_GRADIENT)
    U, T1, T2 = 0.4, 1.3, 0.8
    cases = {"couette": (W.FaceBC(W.WALL_DIFFUSE, 1.0, 1.0, (0.0, -U / 2, 0.0)), W.FaceBC(W.WALL_DIFFUSE, 1.0, 1.0, (0.0, U / 2, 0.0))),
             "fourier": (W.FaceBC(W.WALL_DIFFUSE, T1, 1.0, (0.0, 0.0, 0.0)), W.FaceBC(W.WALL_DIFFUSE, T2, 1.0, (0.0, 0.0, 0.0)))}
    for name, (lo, hi) in cases.items():
        wl = W.cavity(1, 24, 1e9, nxyz=(6, 1, 1), vrange=7.0).with_(faces=[lo, hi, zg, zg, zg, zg], rescale_mass=1)
        o = oracle_mod.Oracle(wl)
        s = make(wl, kernel)
        s.iterate(40)
        for _ in range(40):
            o.step()
        g = s.moments().cpu().numpy()
        assert np.abs(g - o.prim14).max() <= 1e-11 * np.abs(o.prim14).max(), name
        if name == "couette":
            exact = -U / (2 * math.sqrt(math.pi))
            assert abs(g[11, 0] - exact) < 0.04 * abs(exact) and g[11, 0] < 0
        else:
            exact = 2 * math.sqrt(T1 * T2) / (math.sqrt(T1) + math.sqrt(T2)) * (T1 - T2) / (2 * math.sqrt(math.pi))
            assert abs(g[5, 0] - exact) < 0.04 * abs(exact) and g[5, 0] > 0
        s.close()


_NCCL_ONE_RANK = r'''
import os, sys, numpy as np, torch, torch.distributed as dist
sys.path.insert(0, os.environ["DVM_ROOT"])
from paper_1810_00348_b200 import dvm, workloads as W
from oracle import dvm_oracle
try:
    dist.init_process_group("nccl", init_method="tcp://127.0.0.1:" + os.environ["DVM_PORT"], rank=0, world_size=1,
                            device_id=torch.device("cuda:0"))
except Exception as e:                       # no usable NCCL on this box: an environment matter, reported as such
    print("NCCL-UNAVAILABLE", repr(e)); sys.exit(0)
wl = W.config(0)
o = dvm_oracle.Oracle(wl)
s = dvm.Solver(wl, kernel=dvm.KERNEL_TILE)
buf = s.reduce_buffer()
assert buf.is_cuda and buf.dtype == torch.float64 and buf.is_contiguous() and buf.numel() == 16 * wl.n_cells
for it in range(3):
    s.sweep()
    dist.all_reduce(buf, op=dist.ReduceOp.SUM)      # the collective of iterate_sharded, on the solver's own accumulator and stream
    s.update()
    o.step()
    g = s.moments().cpu().numpy()
    assert np.abs(g - o.prim14).max() <= 1e-11 * np.abs(o.prim14).max(), it
s.close()
dist.destroy_process_group()
print("NCCL-OK")
'''


def test_allreduce_of_the_accumulator_through_nccl():
    """The all-reduce step of the sharded iteration, on the real accumulator through NCCL (one rank: the sum is the identity, the
    plumbing - a torch view of the solver's own allocation as the NCCL operand, ordered on the solver's stream - is the same)."""
    import os
    import socket
    import subprocess
    import sys
    from pathlib import Path
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, DVM_ROOT=str(Path(__file__).resolve().parents[1]), DVM_PORT=str(port))
    r = subprocess.run([sys.executable, "-c", _NCCL_ONE_RANK], env=env, capture_output=True, text=True, timeout=300)
    if "NCCL-UNAVAILABLE" in r.stdout:
        pytest.skip("NCCL could not be initialised on this box: " + r.stdout.strip()[-200:])
    assert r.returncode == 0 and "NCCL-OK" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]


def test_failed_plan_can_be_repeated_with_other_options(oracle_mod):
    """A plan that cannot be met (a 1 MiB cap on the f workspace of a 64^3 grid: one velocity block's faces alone need more)
    fails with DVM_EINVAL after the library has already chosen its variant.  The solver must come out of it as the caller
    configured it - kernel, velocities per thread and wide axis read back as "the library chooses", no workspace held - so that
    the next attempt, here with the cap lifted and the single-precision sweep selected (which a left-over choice of 2
    velocities per thread would make invalid), plans afresh and runs within the single-precision bound of the double oracle."""
    from paper_1810_00348_b200 import dvm
    from tests.parity import tol32
    wl = W.cavity(64, 8, 1.0, nxyz=(64, 64, 16))
    s = dvm.Solver(wl, max_f_mbytes=1)
    held = s.workspace_bytes()[0]
    with pytest.raises(dvm.DvmError) as e:
        s.iterate(1)
    assert e.value.code == dvm.EINVAL and "cannot be met" in str(e.value)
    assert (s.kernel_used(), s.tile_rv(), s.tile_axis()) == (dvm.KERNEL_AUTO, 0, 0)     # as requested, not as planned
    assert s.workspace_bytes() == (held, 0) and s.iterations_done() == 0
    s.set_option(dvm.OPT_MAX_F_MBYTES, 0)
    s.set_option(dvm.OPT_PRECISION, dvm.PREC_MIXED)
    s.iterate(1)
    assert s.kernel_used() == dvm.KERNEL_TILE and s.tile_rv() in (3, 4) and s.precision() == dvm.PREC_MIXED
    o = oracle_mod.Oracle(wl)
    c14 = o.step()
    err = float(np.abs(s.moments().cpu().numpy() - c14).max())
    assert 1e-10 < err <= tol32(wl), err
    s.close()


def test_state_cannot_change_under_a_pending_sweep_or_on_one_shard(oracle_mod):
    """dvm_step_host on a velocity-sharded solver and dvm_set_state / dvm_step_host between dvm_sweep and dvm_update are refused
    BEFORE anything is written: the state afterwards is bit-for-bit the state before (a rank whose replicated state changed alone
    would silently diverge from the others)."""
    import torch
    from paper_1810_00348_b200 import dvm
    wl = W.config(0)
    other = torch.as_tensor(W.perturbed_state(wl, seed=5), device="cuda:0")
    h_in = torch.as_tensor(W.perturbed_state(wl, seed=6)).contiguous()
    h_out = torch.empty(14 * wl.n_cells, dtype=torch.float64)
    # one shard of two
    s = dvm.Solver(wl, kernel=2, shard=(0, 2))
    before = s.get_state()[0].clone()
    with pytest.raises(dvm.DvmError) as e:
        s.step_host(h_in, None, 1, h_out, None)
    assert e.value.code == dvm.EINVAL
    assert torch.equal(s.get_state()[0], before)
    s.close()
    # sweep pending
    s = dvm.Solver(wl, kernel=2)
    s.iterate(1)
    s.sweep()
    before = s.get_state()[0].clone()
    for call in (lambda: s.set_state(other), lambda: s.step_host(h_in, None, 1, h_out, None), lambda: s.step_host(h_in, None, 0, h_out, None)):
        with pytest.raises(dvm.DvmError) as e:
            call()
        assert e.value.code == dvm.EINVAL
        assert torch.equal(s.get_state()[0], before)
    s.update()
    # the pair sweep; update is one iteration: residual and history are addressed by the device-side counter
    o = oracle_mod.Oracle(wl)
    o.step(); o.step()
    assert_residual(s.residual(), o.resid, what="sweep; update after refused calls")
    hist = s.residual_history()
    assert hist.shape == (2, 3)
    assert_residual(hist[0], o.history[0]); assert_residual(hist[1], o.history[1])
    s.close()


def test_graph_replay_is_reported(monkeypatch):
    """dvm_graph_active tells how dvm_iterate issues its iterations: the tile kernel replays a captured CUDA graph (1), the
    slice kernel and DVM_GRAPH=0 use plain launches (0); a failed capture would read 2.  Before the first iteration: 0."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(0)
    s = dvm.Solver(wl, kernel=dvm.KERNEL_TILE)
    assert s.graph_active() == 0
    s.iterate(2)
    assert s.graph_active() == 1, dvm.lib().dvm_last_error()
    s.close()
    s = dvm.Solver(wl, kernel=dvm.KERNEL_SLICE)
    s.iterate(1)
    assert s.graph_active() == 0
    s.close()
    monkeypatch.setenv("DVM_GRAPH", "0")
    s = dvm.Solver(wl, kernel=dvm.KERNEL_TILE)
    s.iterate(1)
    assert s.graph_active() == 0
    s.close()


def test_fp64_peak_probe_is_plausible():
    """dvm_fp64_peak_probe (bench.py's measured fp64 denominator): a register-resident DFMA stream cannot beat the nominal
    148 SM x 64 lanes x 1.965 GHz and, on a healthy board, reaches at least half of it; bad arguments are refused."""
    from paper_1810_00348_b200 import dvm
    rate, ms = dvm.fp64_peak_probe("cuda:0", rounds=500_000)
    nominal = 148 * 64 * 1.965e9
    assert 0.5 * nominal < rate <= 1.02 * nominal, rate
    assert ms > 0
    with pytest.raises(dvm.DvmError):
        dvm.fp64_peak_probe("cuda:0", rounds=0)
