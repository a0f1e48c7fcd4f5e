"""Pins of the oracle's second-order upwind sweep (order = 2; "extend the first order upwind scheme to second
order by storing three consecutive slices"; reading G21 of DESIGN.md: finite-volume second-order upwind, face values
extrapolated linearly from the two upwind cell centres, first order where the second upwind cell is missing).

None of these compares the oracle with itself: the expected values are the textbook (3, -4, 1) / 2h stencil, the closed
form of a two-term linear recurrence (numpy.roots), linear extrapolation done by numpy.polyfit, the conservation identity
of a flux-difference scheme, the decay rate of the continuous equation, and exact fixed points.  CPU only.
"""
import math

import numpy as np
import pytest

from paper_1810_00348_b200 import workloads as W


def one_d(n, m=6, Kn=0.5, stretch=0.0, order=2):
    """NY = NZ = 1 with zero-gradient side faces: Eq.(7) reduced to one dimension; wall at x-, free stream at x+."""
    wl = W.cavity(1, m, Kn, nxyz=(n, 1, 1), stretch=stretch)
    zg = W.FaceBC(W.ZERO_GRADIENT)
    faces = [W.FaceBC(W.WALL_DIFFUSE, 1.2, 1.0, (0, 0, 0)), W.FaceBC(W.FREESTREAM, 0.9, 1.1, (0.1, 0, 0)), zg, zg, zg, zg]
    return wl.with_(faces=faces, rescale_mass=0, order=order)


UNIFORM_STATE = np.array([1.1, 0.05, 0.02, -0.01, 0.9, 0.01, 0.0, 0.02])


def test_uniform_grid_interior_stencil_is_3_m4_1(oracle_mod):
    """On a uniform grid the second-order upwind difference is (3 f_i - 4 f_{i-1} + f_{i-2}) / 2h (textbook): the stored
    field of one velocity must satisfy xi (3 f_i - 4 f_{i-1} + f_{i-2}) / 2h + (f_i - S) / tau = 0 at every cell that has two
    upwind fluid cells, and the first-order Eq.(7) with the ghost value at the first cell."""
    n = 14
    wl = one_d(n)
    o = oracle_mod.Oracle(wl)
    prim = np.repeat(UNIFORM_STATE[:, None], wl.n_cells, axis=1)
    rho_w = np.full(o.nface, 0.7)
    tau = o.tau(UNIFORM_STATE[0], UNIFORM_STATE[4])
    h = 1.0 / n
    for ia in (4, 5, 1, 0):
        xi = (wl.xi_x[ia], wl.xi_y[1], wl.xi_z[2])
        f = o.sweep_velocity(ia, 1, 2, prim, rho_w)[0, 0, :]
        S = o.feq(UNIFORM_STATE, xi)
        if xi[0] < 0:
            f = f[::-1]
            ghost = o.feq([1.1, 0.1, 0, 0, 0.9, 0, 0, 0], xi)
        else:
            ghost = 0.7 * o.gwall(0, xi)
        a = abs(xi[0])
        scale = (np.abs(f).max() + abs(S) + abs(ghost)) * (a / h + 1 / tau)
        res = a * (3 * f[2:] - 4 * f[1:-1] + f[:-2]) / (2 * h) + (f[2:] - S) / tau
        assert np.abs(res).max() < 1e-13 * scale
        assert abs(a * (f[0] - ghost) / h + (f[0] - S) / tau) < 1e-13 * scale
        # second cell: one upwind fluid cell only -> its upwind face value is f_0, its own downwind face (3 f_1 - f_0) / 2
        assert abs(a * ((3 * f[1] - f[0]) / 2 - f[0]) / h + (f[1] - S) / tau) < 1e-13 * scale


def test_one_dimensional_closed_form(oracle_mod):
    """Uniform state, uniform grid: e_i = f_i - S obeys (1/tau + 3a/2) e_i = 2a e_{i-1} - (a/2) e_{i-2} for i >= 2, whose
    solution is A r1^i + B r2^i with r1, r2 the roots of the characteristic polynomial (numpy.roots) and A, B fixed by the
    two starting cells."""
    n = 16
    wl = one_d(n, Kn=0.8)
    o = oracle_mod.Oracle(wl)
    prim = np.repeat(UNIFORM_STATE[:, None], wl.n_cells, axis=1)
    rho_w = np.full(o.nface, 0.7)
    tau = o.tau(UNIFORM_STATE[0], UNIFORM_STATE[4])
    for ia in (3, 5):
        xi = (wl.xi_x[ia], wl.xi_y[4], wl.xi_z[0])
        a = abs(xi[0]) * n
        f = o.sweep_velocity(ia, 4, 0, prim, rho_w)[0, 0, :]
        e = f - o.feq(UNIFORM_STATE, xi)
        r = np.roots([1 / tau + 1.5 * a, -2 * a, 0.5 * a])
        AB = np.linalg.solve(np.array([[1.0, 1.0], [r[0], r[1]]]), e[:2].astype(complex))
        expect = (AB[0] * r[0] ** np.arange(n) + AB[1] * r[1] ** np.arange(n)).real
        assert np.allclose(e, expect, rtol=1e-11, atol=1e-15 * abs(e[0]))


@pytest.mark.parametrize("order,rate", [(1, 2.0), (2, 4.0)])
def test_observed_order_of_the_decay_rate(oracle_mod, order, rate):
    """xi f' = (S - f) / tau decays like exp(-x / (xi tau)).  Far from the boundary the discrete field decays by a fixed
    ratio per cell; its rate -log(ratio) / h converges to 1 / (xi tau) at first order for Eq.(7) and at second order for
    order = 2: halving h divides the error by 2 and by 4."""
    errs = []
    for n in (48, 96):
        wl = one_d(n, Kn=3.0, order=order)
        o = oracle_mod.Oracle(wl)
        prim = np.repeat(UNIFORM_STATE[:, None], wl.n_cells, axis=1)
        rho_w = np.full(o.nface, 0.7)
        tau = o.tau(UNIFORM_STATE[0], UNIFORM_STATE[4])
        ia = 4
        xi = (wl.xi_x[ia], wl.xi_y[2], wl.xi_z[3])
        f = o.sweep_velocity(ia, 2, 3, prim, rho_w)[0, 0, :]
        e = f - o.feq(UNIFORM_STATE, xi)
        ratio = e[n // 2 + 1] / e[n // 2]
        lam = -math.log(ratio) * n
        errs.append(abs(lam - 1.0 / (xi[0] * tau)))
    assert errs[0] / errs[1] == pytest.approx(rate, rel=0.12)


def _sides(o, wl):
    prim_n = o.prev_prim8
    rhoS = o.rho_equilibrium(prim_n)
    dx, dy, dz = np.diff(wl.xf), np.diff(wl.yf), np.diff(wl.zf)
    V = (dz[:, None, None] * dy[None, :, None] * dx[None, None, :]).reshape(-1)
    fluid = np.ones(wl.n_cells, bool) if wl.solid is None else wl.solid.reshape(-1) == 0
    tau = np.array([o.tau(r, t) if ok else 1.0 for r, t, ok in zip(prim_n[0], prim_n[4], fluid)])
    lhs = (V * (rhoS - o.raw13[0]) / tau)[fluid].sum()
    cell, dirn, area = o.face_table()
    rhs = (area * (o.flux_out - o.flux_in))[cell >= 0].sum()
    return lhs, rhs


@pytest.mark.parametrize("kind", ["cavity", "cube"])
def test_conservation_identity(oracle_mod, kind):
    """A flux-difference scheme telescopes whatever the face values are: sum_c V_c (rhoS_c - rho_c) / tau_c equals the net
    flux through the boundary faces, now with the extrapolated values at the outflow faces.  Stretched grid; free stream,
    zero gradient and a solid block.  The result differs from the first-order one (the pin is not vacuous)."""
    if kind == "cavity":
        wl = W.cavity(7, 8, 1.0, stretch=1.5).with_(order=2)
        tol = 5e-14
    else:
        wl = W.cube_flow(2, 10, box=(5, 3, 3), vrange=7.0).with_(order=2)
        tol = 3e-13
    o = oracle_mod.Oracle(wl)
    o1 = oracle_mod.Oracle(wl.with_(order=1))
    for it in range(3):
        o.step()
        o1.step()
        lhs, rhs = _sides(o, wl)
        assert abs(lhs) > 1e-6
        assert lhs == pytest.approx(rhs, abs=tol)
    assert np.abs(o.prim14[0] - o1.prim14[0]).max() > 1e-3


def _line_to_face(xc, fc, x1, f1, xface):
    """value at xface of the straight line through (x1, f1), (xc, fc): numpy.polyfit, not a formula of ours"""
    return np.polyval(np.polyfit([x1, xc], [f1, fc], 1), xface)


def test_face_values_are_linear_extrapolations(oracle_mod):
    """On a stretched 3-D grid, take the stored field of single velocities and rebuild Eq.(7) in flux-difference form with
    face values extrapolated by numpy.polyfit from the two upwind cell CENTRES (cell value where there is no upwind fluid
    cell, ghost value at a boundary face): the residual must vanish at every cell; and the wall-incident flux of the
    oracle must be the sum of the extrapolated values at the outflow faces."""
    wl = W.cavity(0, 6, 0.7, stretch=1.4, nxyz=(6, 5, 4)).with_(order=2, rescale_mass=0)
    o = oracle_mod.Oracle(wl)
    prim = W.perturbed_state(wl, seed=21, amp_q=0.01)
    rng = np.random.default_rng(21)
    rho_w = rng.uniform(0.9, 1.1, o.nface)
    nx, ny, nz = wl.nx, wl.ny, wl.nz
    faces = [wl.xf, wl.yf, wl.zf]
    cen = [0.5 * (a[1:] + a[:-1]) for a in faces]
    n = (nx, ny, nz)
    off = [0, ny * nz, 2 * ny * nz, 2 * ny * nz + nx * nz, 2 * ny * nz + 2 * nx * nz, 2 * ny * nz + 2 * nx * nz + nx * ny]

    def face_slot(d, i, j, k):
        return off[d] + (k * ny + j if d < 2 else k * nx + i if d < 4 else j * nx + i)

    flux = np.zeros(o.nface)
    for (ia, ib, ic) in [(5, 4, 3), (0, 1, 5), (4, 0, 2), (1, 5, 0)]:
        xi = np.array([wl.xi_x[ia], wl.xi_y[ib], wl.xi_z[ic]])
        wgt = wl.w_x[ia] * wl.w_y[ib] * wl.w_z[ic]
        f = o.sweep_velocity(ia, ib, ic, prim, rho_w)      # [k][j][i]
        s = np.where(xi >= 0, 1, -1)

        def val(idx):
            return f[idx[2], idx[1], idx[0]]

        def down_face_value(idx, d):
            """value at the downwind face (along d) of cell idx"""
            up = list(idx); up[d] -= s[d]
            if up[d] < 0 or up[d] >= n[d]:
                return val(idx)
            xface = faces[d][idx[d] + 1] if s[d] > 0 else faces[d][idx[d]]
            return _line_to_face(cen[d][idx[d]], val(idx), cen[d][up[d]], val(up), xface)

        worst = 0.0
        for k in range(nz):
            for j in range(ny):
                for i in range(nx):
                    idx = [i, j, k]
                    c = (k * ny + j) * nx + i
                    Wc = prim[:, c]
                    tau = o.tau(Wc[0], Wc[4])
                    res = (val(idx) - o.feq(Wc, xi)) / tau
                    for d in range(3):
                        width = faces[d][idx[d] + 1] - faces[d][idx[d]]
                        up = list(idx); up[d] -= s[d]
                        if up[d] < 0 or up[d] >= n[d]:
                            dirn = 2 * d + (0 if s[d] > 0 else 1)
                            fin = rho_w[face_slot(dirn, i, j, k)] * o.gwall(dirn, xi)
                        else:
                            fin = down_face_value(up, d)
                        fout = down_face_value(idx, d)
                        res += abs(xi[d]) * (fout - fin) / width
                        dn = list(idx); dn[d] += s[d]
                        if dn[d] < 0 or dn[d] >= n[d]:
                            dirn = 2 * d + (1 if s[d] > 0 else 0)
                            flux[face_slot(dirn, i, j, k)] += wgt * abs(xi[d]) * fout
                    worst = max(worst, abs(res) * tau / abs(val(idx)))
        assert worst < 1e-12
    # the same four velocities alone (all other weights zero) through odvm_step: wall-incident fluxes
    wx, wy, wz = np.zeros(6), np.zeros(6), np.zeros(6)
    tot = np.zeros(o.nface)
    for (ia, ib, ic) in [(5, 4, 3), (0, 1, 5), (4, 0, 2), (1, 5, 0)]:
        wx[:] = 0; wy[:] = 0; wz[:] = 0
        wx[ia], wy[ib], wz[ic] = wl.w_x[ia], wl.w_y[ib], wl.w_z[ic]
        o1 = oracle_mod.Oracle(wl.with_(w_x=wx.copy(), w_y=wy.copy(), w_z=wz.copy()))
        o1.set_state(prim, rho_w)
        o1.step()
        tot += o1.flux_out
    assert np.allclose(tot, flux, rtol=1e-12, atol=1e-18)
    assert np.abs(flux).max() > 0


def test_fixed_points_survive(oracle_mod):
    """Uniform Maxwellians have zero slope, so every fixed point of the first-order scheme is one of the second-order
    scheme: closed box at rest (P7), box with a solid block (P12), free stream (P11), gas moving with its walls (P14)."""
    wl = W.cavity(5, 24, 0.1, U_w=0.0).with_(order=2)
    solid = np.zeros((5, 5, 5), dtype=np.uint8)
    solid[1:3, 2:4, 1:3] = 1
    for w_ in (wl, wl.with_(solid=solid)):
        o = oracle_mod.Oracle(w_)
        fluid = np.ones(w_.n_cells, bool) if w_.solid is None else w_.solid.reshape(-1) == 0
        for it in range(2):
            p = o.step()
            assert np.abs(p[0][fluid] - 1).max() < 1e-13 and np.abs(p[4][fluid] - 1).max() < 2e-13
            assert np.abs(p[1:4][:, fluid]).max() < 1e-13 and np.abs(p[5:][:, fluid]).max() < 1e-13
    fs = W.FaceBC(W.FREESTREAM, 1.1, 0.9, (0.3, -0.2, 0.1))
    wf = W.cavity(0, 24, 0.2, stretch=1.5, nxyz=(6, 5, 4)).with_(
        faces=[fs] * 6, rescale_mass=0, rho0=0.9, u0=(0.3, -0.2, 0.1), T0=1.1, order=2)
    o = oracle_mod.Oracle(wf)
    for it in range(2):
        p = o.step()
        assert np.abs(p[0] - 0.9).max() < 1e-11 and np.abs(p[4] - 1.1).max() < 1e-11 and np.abs(p[1] - 0.3).max() < 1e-11


def test_second_order_changes_the_cavity_solution_but_keeps_its_symmetry(oracle_mod):
    """Cavity, a few iterations with order = 2: stable, mass conserved by the rescale, y-mirror symmetry intact (G11), and
    the fields differ from the first-order ones at O(h) (so the option is live)."""
    wl = W.cavity(6, 8, 1.0).with_(order=2)
    o = oracle_mod.Oracle(wl)
    o1 = oracle_mod.Oracle(wl.with_(order=1))
    hist = []
    for it in range(6):
        p = o.step()
        p1 = o1.step()
        hist.append(o.resid.max())
        assert o.total_mass(p[0]) == pytest.approx(o.mass0, rel=1e-14)
    F = p.reshape(14, wl.nz, wl.ny, wl.nx)
    for m in (0, 1, 3, 4, 5, 7, 8, 9, 10, 12):
        assert np.abs(F[m] - F[m][:, ::-1, :]).max() < 1e-13
    for m in (2, 6, 11, 13):
        assert np.abs(F[m] + F[m][:, ::-1, :]).max() < 1e-13
    assert hist[-1] < hist[1]
    assert 1e-4 < np.abs(p[1] - p1[1]).max() < 0.1
