"""GPU parity of the single-precision sweep (DVM_OPT_PRECISION = DVM_PREC_MIXED; PAPER.md:313:
the paper's timings are single precision).  f is carried in IEEE single by the tile kernel (factor tables, faces, plane,
arithmetic of Eq.(7)); the velocity sums, wall fluxes, moment update and residual stay double.

What parity means here (reading G22, derivation in tests/test_oracle_f32.py): against the DOUBLE oracle every field,
wall density and raw sum agrees to tol32 = 16 x 2^-24 x (nx + ny + nz) ABSOLUTE in the units of DESIGN.md section 2 (the
rigorous bound of the rounding along the longest upwind path), and the GPU's error is of the same class as that of the
oracle's own single-precision sweep (f32 = 1): its root-mean-square is at most 4 times the oracle's.  The single-precision
oracle and the GPU round at different points (direct exp against tabulated factors), so they are not compared bit for bit."""
import numpy as np
import pytest

from paper_1810_00348_b200 import workloads as W
from tests.parity import tol32

pytestmark = pytest.mark.gpu
TILE = 2


def fluid_mask(wl):
    return slice(None) if wl.solid is None else wl.solid.reshape(-1) == 0


def make(wl, **kw):
    from paper_1810_00348_b200 import dvm
    return dvm.Solver(wl, kernel=TILE, precision=dvm.PREC_MIXED, **kw)


def rms(a):
    return float(np.sqrt(np.mean(np.square(a))))


def mixed_lockstep(wl, iters, oracle_mod, state=None, rho_w=None, with_f32_oracle=True, **kw):
    """One-step map of the single-precision GPU sweep against the double oracle from the SAME state n, every iteration
    (the state fed to both sides is the double oracle's)."""
    from paper_1810_00348_b200 import dvm
    o64 = oracle_mod.Oracle(wl)
    o32 = oracle_mod.Oracle(wl.with_(f32=True)) if with_f32_oracle else None
    s = make(wl, **kw)
    assert s.precision() == dvm.PREC_MIXED
    if state is not None:
        o64.set_state(state, rho_w)
    fm = fluid_mask(wl)
    tol = tol32(wl)
    seen = 0.0
    for it in range(iters):
        what = f"{wl.name} {kw} iteration {it + 1}"
        s.set_state(o64.prim8, o64.rho_w)
        if o32 is not None:
            o32.set_state(o64.prim8, o64.rho_w)
            o32.step()
        s.iterate(1)
        o64.step()
        g14 = s.moments().cpu().numpy()
        d = (g14 - o64.prim14)[:, fm]
        assert np.isfinite(g14).all(), what
        assert np.abs(d).max() <= tol * max(1.0, np.abs(o64.prim14).max()), (what, np.abs(d).max(axis=1), tol)
        seen = max(seen, np.abs(d).max())
        g_rw = s.get_state()[1].cpu().numpy()
        # (a stratified weight subset leaves wall densities far from O(1): Phi_unit is built from the zeroed weights)
        assert np.abs(g_rw - o64.rho_w).max() <= tol * max(1.0, np.abs(o64.rho_w).max()), what
        graw = s.raw_moments().cpu().numpy()
        assert np.abs(graw - o64.raw13).max() <= tol * max(1.0, np.abs(o64.raw13).max()), what
        gfl = s.wall_flux().cpu().numpy()
        assert np.abs(gfl - o64.flux_out).max() <= tol * max(1.0, np.abs(o64.flux_out).max()), what
        assert abs(s.mass_scale() - o64.scale) <= tol * abs(o64.scale), what
        assert np.all(np.abs(np.asarray(s.residual()) - o64.resid) <= 2 * tol * np.maximum(1.0, o64.resid)), (what, s.residual(), o64.resid)
        if o32 is not None:
            d32 = (o32.prim14 - o64.prim14)[:, fm]
            assert rms(d) <= 4 * rms(d32) + 1e-10, (what, rms(d), rms(d32))
    # the mode is really single precision: far from the 1e-11 of the double kernel
    assert seen > 1e-10, seen
    s.close()
    return seen


def test_mixed_config0_every_iteration(oracle_mod):
    """BASELINE.json configs[0], 20 iterations, one-step map every iteration."""
    mixed_lockstep(W.config(0), 20, oracle_mod)


def test_mixed_config0_free_run(oracle_mod):
    """The single-precision GPU iteration run on its own for 20 iterations stays within 3 tol32 of the double oracle's run."""
    wl = W.config(0)
    o = oracle_mod.Oracle(wl)
    s = make(wl)
    s.iterate(20)
    for _ in range(20):
        o.step()
    g14 = s.moments().cpu().numpy()
    assert np.abs(g14 - o.prim14).max() <= 3 * tol32(wl)
    hist = s.residual_history()
    assert np.all(np.abs(hist - np.asarray(o.history)) <= 6 * tol32(wl))
    s.close()


@pytest.mark.parametrize("seed,amp_q", [(1810, 0.0), (348, 0.01)])
def test_mixed_config1_perturbed(oracle_mod, seed, amp_q):
    """BASELINE.json configs[1] kernel-level test (32^3 x 24^3, seeded noise), with and without heat flux; the library picks
    the 12-wide RV = 3 variant for 12-node sign halves."""
    wl = W.config(1)
    st = W.perturbed_state(wl, seed=seed, amp_q=amp_q)
    mixed_lockstep(wl, 2, oracle_mod, state=st, rho_w=np.ones(6 * 32 * 32))


@pytest.mark.parametrize("rv", [3, 4])
@pytest.mark.parametrize("axis", [1, 2, 3])
def test_mixed_ragged_nonuniform_cavity_all_variants(oracle_mod, rv, axis):
    """13 x 9 x 11 tanh-stretched cells, 10 x 7 x 9 velocities (ragged tiles, a node at xi = 0): both single-precision
    variants, each velocity axis in the wide role."""
    wl = W.cavity(0, 0, 0.075, stretch=1.5, nxyz=(13, 9, 11), mxyz=(10, 7, 9))
    mixed_lockstep(wl, 2, oracle_mod, tile_rv=rv, tile_axis=axis)


@pytest.mark.parametrize("rv", [3, 4])
def test_mixed_dense_wide_velocity_grid(oracle_mod, rv):
    """40 x 10 x 9 velocities with a shifted 17 / 23 split: several x-blocks per sign half with a partly filled last block,
    every lane compared."""
    wl = W.cavity(0, 0, 0.3, nxyz=(6, 5, 7), mxyz=(40, 10, 9))
    xi = wl.xi_x + 0.13 * 3
    wl = wl.with_(xi_x=xi)
    mixed_lockstep(wl, 2, oracle_mod, tile_rv=rv)


def test_mixed_cube_flow_small(oracle_mod):
    """Free stream + zero-gradient outflow + solid block (the slow path of levels with a solid ghost) in single precision."""
    wl = W.cube_flow(4, 12, box=(6, 4, 4), vrange=8.0)
    mixed_lockstep(wl, 3, oracle_mod)


def test_mixed_degenerate_shapes(oracle_mod):
    """One cell thick in y and z, zero-gradient side faces, walls with T_w != 1."""
    wl = W.cavity(1, 6, 0.5, nxyz=(12, 1, 1))
    zg = W.FaceBC(W.ZERO_GRADIENT)
    wl = wl.with_(faces=[W.FaceBC(W.WALL_DIFFUSE, 1.2, 1.0, (0, 0, 0)), W.FaceBC(W.FREESTREAM, 0.9, 1.1, (0.1, 0, 0)),
                         zg, zg, zg, zg], rescale_mass=0)
    mixed_lockstep(wl, 2, oracle_mod)


def test_mixed_closed_box_fixed_point(oracle_mod):
    """GPU counterpart of the single-precision P7: the uniform equilibrium between stationary walls stays put to tol32."""
    wl = W.cavity(6, 24, 1.0, U_w=0.0)
    s = make(wl)
    s.iterate(3)
    g14 = s.moments().cpu().numpy()
    tol = tol32(wl)
    assert np.abs(g14[0] - 1).max() <= tol and np.abs(g14[4] - 1).max() <= tol
    assert np.abs(g14[1:4]).max() <= tol and np.abs(g14[5:]).max() <= tol
    s.close()


def test_mixed_workspace_cap_and_stress(oracle_mod):
    """Capped workspace (batches of velocity blocks) and a persistent grid of 4 CTAs: the dependency protocol with
    single-precision faces."""
    wl = W.cavity(0, 0, 0.2, nxyz=(9, 10, 3), mxyz=(36, 20, 18))
    mixed_lockstep(wl, 2, oracle_mod, with_f32_oracle=False, max_f_mbytes=1, max_ctas=4)


def test_mixed_config4_full_size_stratified_step(oracle_mod):
    """Config 4 at full size in the launch configuration `bench.py --precision mixed` times, one velocity in each of the 512
    velocity blocks, one step from a perturbed state with heat flux."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(4)
    wl = W.stratified_weight_subset(wl, dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, 0), 1)
    st = W.perturbed_state(wl, seed=5, amp_q=0.01)
    mixed_lockstep(wl, 1, oracle_mod, state=st, rho_w=None, with_f32_oracle=False)


def test_mixed_config3_full_size_stratified_step(oracle_mod):
    """Config 3 at full size (solid cube, free stream, shifted 48^3 grid: the RV = 3 variant), one velocity per block."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(3)
    wl = W.stratified_weight_subset(wl, dvm.plan_vblocks(wl.xi_x, wl.xi_y, wl.xi_z, 0), 0)
    mixed_lockstep(wl, 1, oracle_mod, state=W.perturbed_state(wl, seed=3, amp_q=0.01), rho_w=None, with_f32_oracle=False)


def test_mixed_refuses_what_it_does_not_cover():
    """DVM_PREC_MIXED is a mode of the first-order tile kernel with 3 or 4 velocities per thread: everything else is EINVAL."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(0)
    for kw in (dict(kernel=1), dict(kernel=TILE, order=2), dict(kernel=TILE, tile_rv=2)):
        s = dvm.Solver(wl, precision=dvm.PREC_MIXED, **kw)
        with pytest.raises(dvm.DvmError) as e:
            s.iterate(1)
        assert e.value.code == dvm.EINVAL
        s.close()
    s = dvm.Solver(wl)
    with pytest.raises(dvm.DvmError):
        s.set_option(dvm.OPT_PRECISION, 5)
    s.close()


def test_mixed_f_workspace_is_half(oracle_mod):
    """Faces and factor tables are single: the f workspace is half of the double kernel's."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(1)
    a, b = dvm.Solver(wl, kernel=TILE, tile_rv=4), make(wl, tile_rv=4)
    a.iterate(1); b.iterate(1)
    assert b.workspace_bytes()[1] * 2 == a.workspace_bytes()[1]
    a.close(); b.close()


def test_mixed_config2_runs_to_residual_1e6_like_the_double_run():
    """BASELINE.json configs[2] "run to residual 1e-6" in single precision: the residual history follows the double run's to
    the stated tolerance down to 1e-6 (reached at the same iteration +- 1), then stops at its rounding floor of ~1e-7
    (G22) where the double run goes on falling; the converged fields of the two runs agree to 3 tol32."""
    from paper_1810_00348_b200 import dvm
    wl = W.config(2)
    runs = {}
    for prec in (dvm.PREC_F64, dvm.PREC_MIXED):
        s = dvm.Solver(wl, kernel=TILE, precision=prec)
        s.iterate(160)
        runs[prec] = (s.residual_history().max(axis=1), s.moments().cpu().numpy())
        s.close()
    h64, h32 = runs[dvm.PREC_F64][0], runs[dvm.PREC_MIXED][0]
    first64, first32 = int(np.argmax(h64 < 1e-6)) + 1, int(np.argmax(h32 < 1e-6)) + 1
    assert h64[first64 - 1] < 1e-6 and h32[first32 - 1] < 1e-6 and abs(first64 - first32) <= 1, (first64, first32)
    above = h64 > 2e-6
    assert np.all(np.abs(h32[above] - h64[above]) <= 0.05 * h64[above])
    assert h64[-1] < 1e-8 and 1e-8 < h32[-1] < 1e-6          # the double run keeps falling, the single one sits on its floor
    assert np.abs(runs[dvm.PREC_MIXED][1] - runs[dvm.PREC_F64][1]).max() <= 3 * tol32(wl)


def _golden_full_steps():
    from pathlib import Path
    return sorted(int(p.stem.split("cfg")[1]) for p in (Path(__file__).parent / "golden").glob("full_step_cfg*.txt"))


@pytest.mark.parametrize("cfg", _golden_full_steps())
def test_mixed_full_weight_step_against_archived_double_oracle(cfg):
    """The single-precision sweep over EVERY velocity of configs 2 - 4 (all lanes of all velocity blocks carry weight) against
    the archived full-weight step of the DOUBLE oracle (tests/golden/full_step_cfg<N>.txt): sampled cells, wall densities,
    field maxima, residual and rescale factor at tol32."""
    from pathlib import Path
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_goldens", Path(__file__).parent / "golden" / "make_full_step_goldens.py")
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
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
    s = make(wl)
    s.set_state(prim, None)
    s.iterate(1)
    g14 = s.moments().cpu().numpy()
    rw = s.get_state()[1].cpu().numpy()
    tol = tol32(wl)
    worst = 0.0
    for c, ref in gold["cell"].items():
        err = np.abs(g14[:, c] - ref).max()
        worst = max(worst, err)
        assert err <= tol, (cfg, c, err, tol)
    assert worst > 1e-10                               # single precision did take part
    fluid = np.ones(wl.n_cells, bool) if wl.solid is None else wl.solid.reshape(-1) == 0
    for m in range(14):
        assert abs(np.abs(g14[m][fluid]).max() - gold["field"][m][0]) <= tol
    for fidx, val in gold["face"].items():
        assert abs(rw[fidx] - val[0]) <= tol * max(1.0, abs(val[0]))
    assert np.all(np.abs(np.asarray(s.residual()) - gold["resid"]) <= 2 * tol * np.maximum(1.0, gold["resid"]))
    assert abs(s.mass_scale() - gold["scale"]) <= tol * abs(gold["scale"])
    s.close()
