"""Pins of the oracle's single-precision sweep (`f32 = 1`; reading G22; "All of the testings are
based on ... single precision computations").  CPU only.

What "parity at fp32" means (G22): the sweep of Eq.(7) runs in IEEE single (every stored or combined value of f is a
single), the velocity sums of Eq.(5) are accumulated in double or better.  One update is a combination of positive terms
made with at most ~8 roundings (u = 2^-24 each) in the oracle's operation order, ~16 in the GPU's (tabulated factors,
reciprocal), and an error of an upwind value is passed on with weights a_d / den that sum to less than 1, so after the
longest upwind path of L = nx + ny + nz cells

    |f32 - f64| <= K u L max f,   K = 8 (oracle), 16 (GPU),

and a velocity sum of positive weights inherits the bound relative to sum w |phi| f, which is O(1) in the units of DESIGN.md
section 2.  `tol32(wl)` = 16 u L is therefore the ABSOLUTE tolerance, in those units, of every field of the fp32 mode; the
errors measured here are 10-100 times smaller (they add like a random walk and are damped by collisions).
"""
import numpy as np
import pytest

from paper_1810_00348_b200 import workloads as W
from tests.parity import tol32

U32 = 2.0 ** -24


@pytest.fixture(scope="module")
def oracle_mod():
    from oracle import dvm_oracle
    dvm_oracle.build()
    return dvm_oracle


def test_f32_values_are_singles_and_order1_double_is_untouched(oracle_mod):
    """Every f the single-precision sweep returns is exactly a single; with f32 = 0 the field is not (so the switch
    does something) and equals what the struct without the flag gave (default path)."""
    wl = W.cavity(6, 8, 0.5)
    o64, o32 = oracle_mod.Oracle(wl), oracle_mod.Oracle(wl.with_(f32=True))
    prim = W.perturbed_state(wl, seed=5, amp_q=0.01)
    rho_w = np.random.default_rng(6).uniform(0.9, 1.1, o64.nface)
    for (ia, ib, ic) in [(0, 0, 0), (5, 2, 7), (3, 4, 1)]:
        f64 = o64.sweep_velocity(ia, ib, ic, prim, rho_w)
        f32 = o32.sweep_velocity(ia, ib, ic, prim, rho_w)
        assert np.array_equal(f32, f32.astype(np.float32).astype(np.float64))
        assert not np.array_equal(f64, f64.astype(np.float32).astype(np.float64))
        L = wl.nx + wl.ny + wl.nz
        if f64.max() < 1e-37:
            # the corner of the velocity grid, f ~ exp(-108): below the range of a single, the sweep carries denormals / zeros;
            # the error is absolute and immaterial (the smallest normal single is 1.2e-38)
            assert np.abs(f32 - f64).max() < 1.2e-38
        else:
            err = np.abs(f32 - f64).max() / f64.max()
            assert 1e-9 < err <= 8 * U32 * L


def test_f32_one_dimensional_recurrence_in_numpy_float32(oracle_mod):
    """NY = NZ = 1, zero-gradient y, z faces (the P5 setting), on a stretched grid with a different state in every cell:
    Eq.(7) is the two-term recurrence f_i = (S_i/tau_i + a_i f_{i-1}) / (1/tau_i + a_i).  Written out with numpy float32
    scalars, one rounding per operation, it must reproduce the oracle's single-precision sweep BIT FOR BIT for every
    velocity of the grid: the rounding points are the ones G22 states.  Mutation-checked on a scratch copy of the oracle:
    leaving out the rounding of tau, f^S, a_d, g_w, 1/tau, a_d f_up, either running sum or the quotient fails this test; only
    the rounding of the product rho_w g_w can be left out unnoticed (it changes 4 of 108 ghost terms by half an ulp, which the
    next rounding absorbs)."""
    wl = W.cavity(1, 6, 0.5, nxyz=(12, 1, 1), stretch=1.5)
    zg = W.FaceBC(W.ZERO_GRADIENT)
    faces = [W.FaceBC(W.WALL_DIFFUSE, 1.2, 1.0, (0, 0, 0)), W.FaceBC(W.FREESTREAM, 0.9, 1.1, (0.1, 0, 0)), zg, zg, zg, zg]
    wl = wl.with_(faces=faces, rescale_mass=0, f32=True)
    o = oracle_mod.Oracle(wl)
    prim = W.perturbed_state(wl, seed=77, amp_q=0.01)
    rho_w = np.full(o.nface, 0.7)
    f4 = np.float32
    widths = np.diff(wl.xf)
    taus = [f4(o.tau(prim[0, i], prim[4, i])) for i in range(12)]
    for (ia, ib, ic) in [(a_, b_, c_) for a_ in range(6) for b_ in range(6) for c_ in range(6)]:   # every velocity of the grid
        xi = (wl.xi_x[ia], wl.xi_y[ib], wl.xi_z[ic])
        f = o.sweep_velocity(ia, ib, ic, prim, rho_w)[0, 0, :]
        if xi[0] > 0:
            up = f4(0.7 * float(f4(o.gwall(0, xi))))        # rho_w enters as a double; g_w and the product are rounded
            cells = range(12)
        else:
            up = f4(o.feq([1.1, 0.1, 0, 0, 0.9, 0, 0, 0], xi))
            cells = range(11, -1, -1)
        out = np.zeros(12)
        for i in cells:
            S = f4(o.feq(prim[:, i], xi))
            a = f4(abs(xi[0]) / widths[i])
            num = f4(S / taus[i])
            den = f4(f4(1.0) / taus[i])
            num = f4(num + f4(a * up))
            den = f4(den + a)
            up = f4(num / den)
            out[i] = float(up)
        assert np.array_equal(f, out), (ia, ib, ic)


def test_f32_step_stays_within_the_stated_bound_of_the_double_step(oracle_mod):
    """cfg0, 20 iterations in lock step from the same states: every field of the single-precision step is within
    tol32 (absolute, DESIGN.md units) of the double step - and visibly different from it."""
    wl = W.config(0)
    o64, o32 = oracle_mod.Oracle(wl), oracle_mod.Oracle(wl.with_(f32=True))
    worst = 0.0
    for it in range(20):
        o32.set_state(o64.prim8, o64.rho_w)        # same state n on both sides: the one-step map is compared
        p64, p32 = o64.step(), o32.step()
        err = np.abs(p32 - p64).max()
        worst = max(worst, err)
        assert err <= tol32(wl)
        assert np.abs(o32.rho_w - o64.rho_w).max() <= tol32(wl)
    assert worst > 1e-9


def test_f32_free_run_does_not_drift(oracle_mod):
    """The single-precision iteration run on its own for 20 iterations stays within a few tol32 of the double run: the
    outer iteration does not amplify the rounding of the sweep (it is a contraction towards the same fixed point)."""
    wl = W.config(0)
    o64, o32 = oracle_mod.Oracle(wl), oracle_mod.Oracle(wl.with_(f32=True))
    for it in range(20):
        p64, p32 = o64.step(), o32.step()
    assert np.abs(p32 - p64).max() <= 3 * tol32(wl)
    # mass is restored by the rescale in either precision
    vol = np.multiply.outer(np.multiply.outer(np.diff(wl.zf), np.diff(wl.yf)), np.diff(wl.xf)).reshape(-1)
    assert abs((p32[0] * vol).sum() - o32.mass0) < 1e-12


def test_f32_closed_box_is_a_fixed_point_to_single_rounding(oracle_mod):
    """P7 in single precision: the uniform equilibrium between stationary isothermal walls stays put to tol32 (to 1e-13
    in double): the discrete wall normalisation survives the rounding of f."""
    wl = W.cavity(6, 24, 1.0, U_w=0.0).with_(f32=True)
    o = oracle_mod.Oracle(wl)
    p14 = o.step()
    assert np.abs(p14[0] - 1).max() <= tol32(wl) and np.abs(p14[4] - 1).max() <= tol32(wl)
    assert np.abs(p14[1:4]).max() <= tol32(wl) and np.abs(p14[5:]).max() <= tol32(wl)
    assert np.abs(o.rho_w[o.rho_w != 0] - 1).max() <= tol32(wl)


def test_f32_with_order2_is_refused(oracle_mod):
    wl = W.config(0).with_(f32=True, order=2)
    o = oracle_mod.Oracle(wl)
    with pytest.raises(RuntimeError):
        o.step()
