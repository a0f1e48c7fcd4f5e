"""Seeded synthetic input generators, shared by the CPU oracle's tests and the CUDA path's tests / bench.

This module holds NONE of the method's arithmetic: it only builds the arrays and parameter
records that are handed, unchanged, to both sides (physical face coordinates, the solid mask,
velocity nodes and 1-D quadrature weights, gas / boundary-condition records, seeded
perturbations of a macroscopic state).  It imports neither `oracle/` nor the CUDA binding.

The five workloads restate BASELINE.json `configs[0..4]` (recipe in DESIGN.md "Input recipe");
they stand in for the paper's cavity (Sec. 4.1) and cube (PAPER.md:275, 293,
Sec. 4.2) runs and for the Table 2 grid sizes.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional

import numpy as np

# boundary-condition type codes (same numeric values as include/dvm.h and oracle/dvm_oracle.h;
# the three files state the numbers independently - they are an interface, not arithmetic)
WALL_DIFFUSE = 0
FREESTREAM = 1
ZERO_GRADIENT = 2

# order of the six domain faces everywhere in this repository
FACE_NAMES = ("x-", "x+", "y-", "y+", "z-", "z+")


@dataclass
class FaceBC:
    type: int = WALL_DIFFUSE
    T: float = 1.0
    rho: float = 1.0
    u: tuple = (0.0, 0.0, 0.0)


@dataclass
class Workload:
    name: str
    # physical grid: face coordinates (n+1 each), optional solid mask [nz][ny][nx] uint8
    xf: np.ndarray
    yf: np.ndarray
    zf: np.ndarray
    solid: Optional[np.ndarray]
    # velocity grid: nodes and 1-D weights per axis (tensor grid, w_alpha = product)
    xi_x: np.ndarray
    xi_y: np.ndarray
    xi_z: np.ndarray
    w_x: np.ndarray
    w_y: np.ndarray
    w_z: np.ndarray
    # gas
    Kn: float
    omega: float
    Pr: float
    rho0: float
    u0: tuple
    T0: float
    # boundary conditions
    faces: List[FaceBC] = field(default_factory=list)
    solid_bc: FaceBC = field(default_factory=FaceBC)
    rescale_mass: int = 1
    wall_norm: int = 0
    iterations: int = 1
    order: int = 1          # 1 = first-order upwind Eq.(7); 2 = second-order upwind (G21)
    f32: bool = False       # True = the sweep in IEEE single, velocity sums in double (G22)

    @property
    def nx(self):
        return len(self.xf) - 1

    @property
    def ny(self):
        return len(self.yf) - 1

    @property
    def nz(self):
        return len(self.zf) - 1

    @property
    def mx(self):
        return len(self.xi_x)

    @property
    def my(self):
        return len(self.xi_y)

    @property
    def mz(self):
        return len(self.xi_z)

    @property
    def n_cells(self):
        return self.nx * self.ny * self.nz

    @property
    def n_fluid(self):
        return self.n_cells - (0 if self.solid is None else int(self.solid.sum()))

    @property
    def n_vel(self):
        return self.mx * self.my * self.mz

    @property
    def phase_points(self):
        return self.n_fluid * self.n_vel

    def with_(self, **kw):
        return replace(self, **kw)


# ---------------------------------------------------------------------------------------------
# grids
# ---------------------------------------------------------------------------------------------
def uniform_faces(n: int, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
    return lo + (hi - lo) * np.arange(n + 1, dtype=np.float64) / n


def tanh_faces(n: int, beta: float = 1.5) -> np.ndarray:
    """Wall-clustered faces on [0,1]: x_i = 1/2 [1 + tanh(beta (2i/n - 1)) / tanh(beta)] (G12)."""
    s = 2.0 * np.arange(n + 1, dtype=np.float64) / n - 1.0
    x = 0.5 * (1.0 + np.tanh(beta * s) / math.tanh(beta))
    x[0], x[-1] = 0.0, 1.0
    return x


def trapezoid_nodes(m: int, lo: float, hi: float):
    """Nodes include both range ends; weights h, h/2 at the two ends (PAPER.md:269 'trapezoidal rule')."""
    xi = np.linspace(lo, hi, m, dtype=np.float64)
    h = (hi - lo) / (m - 1)
    w = np.full(m, h, dtype=np.float64)
    w[0] = w[-1] = 0.5 * h
    return xi, w


# ---------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------
def cavity(n: int, m: int, Kn: float, *, vrange: float = 6.0, U_w: float = 0.16, stretch: float = 0.0,
           Pr: float = 2.0 / 3.0, omega: float = 0.81, iterations: int = 1, name: str = "",
           nxyz=None, mxyz=None) -> Workload:
    """Lid-driven cubic cavity: six diffuse walls at T_w = 1, the z+ wall moves in +x at U_w (G11)."""
    nx, ny, nz = (n, n, n) if nxyz is None else nxyz
    mx, my, mz = (m, m, m) if mxyz is None else mxyz
    mk = (lambda q: tanh_faces(q, stretch)) if stretch > 0 else uniform_faces
    xi_x, w_x = trapezoid_nodes(mx, -vrange, vrange)
    xi_y, w_y = trapezoid_nodes(my, -vrange, vrange)
    xi_z, w_z = trapezoid_nodes(mz, -vrange, vrange)
    faces = [FaceBC(WALL_DIFFUSE, 1.0, 1.0, (0.0, 0.0, 0.0)) for _ in range(6)]
    faces[5] = FaceBC(WALL_DIFFUSE, 1.0, 1.0, (U_w, 0.0, 0.0))
    return Workload(name or f"cavity_{nx}x{ny}x{nz}_v{mx}x{my}x{mz}_Kn{Kn:g}", mk(nx), mk(ny), mk(nz), None,
                    xi_x, xi_y, xi_z, w_x, w_y, w_z, Kn, omega, Pr, 1.0, (0.0, 0.0, 0.0), 1.0,
                    faces, FaceBC(), 1, 0, iterations)


def cube_flow(cells_per_side: int = 16, m: int = 48, *, box=(6, 4, 4), Kn: float = 0.1, Ma: float = 2.0,
              vrange: float = 10.0, iterations: int = 50, name: str = "") -> Workload:
    """Supersonic flow past a cube (G13/G14): lengths in cube sides, cube centred in the box."""
    cps = cells_per_side
    nx, ny, nz = box[0] * cps, box[1] * cps, box[2] * cps
    xf = uniform_faces(nx, 0.0, float(box[0]))
    yf = uniform_faces(ny, 0.0, float(box[1]))
    zf = uniform_faces(nz, 0.0, float(box[2]))
    solid = np.zeros((nz, ny, nx), dtype=np.uint8)
    i0, j0, k0 = (nx - cps) // 2, (ny - cps) // 2, (nz - cps) // 2
    solid[k0:k0 + cps, j0:j0 + cps, i0:i0 + cps] = 1
    U_inf = Ma * math.sqrt(5.0 / 6.0)  # Ma * sqrt(gamma/2), gamma = 5/3, speeds in sqrt(2 R T0)
    xi_x, w_x = trapezoid_nodes(m, -vrange, vrange)
    xi_x = xi_x + U_inf
    xi_y, w_y = trapezoid_nodes(m, -vrange, vrange)
    xi_z, w_z = trapezoid_nodes(m, -vrange, vrange)
    fs = FaceBC(FREESTREAM, 1.0, 1.0, (U_inf, 0.0, 0.0))
    faces = [fs, FaceBC(ZERO_GRADIENT), fs, fs, fs, fs]
    return Workload(name or f"cube_{nx}x{ny}x{nz}_v{m}", xf, yf, zf, solid,
                    xi_x, xi_y, xi_z, w_x, w_y, w_z, Kn, 0.81, 2.0 / 3.0, 1.0, (U_inf, 0.0, 0.0), 1.0,
                    faces, FaceBC(WALL_DIFFUSE, 1.0, 1.0, (0.0, 0.0, 0.0)), 0, 0, iterations)


def geometric_faces(n_lo: int, n_mid: int, n_hi: int, r_lo: float, r_hi: float, side: float = 1.0) -> np.ndarray:
    """Faces of an axis with n_mid uniform cells across a body of length `side` centred at 0, and cells growing by the
    cell-by-cell ratios r_lo / r_hi away from it (1.02 in front and at the sides, 1.03 behind the cube)."""
    h = side / n_mid
    lo = -0.5 * side - np.cumsum(h * r_lo ** np.arange(1, n_lo + 1))
    hi = 0.5 * side + np.cumsum(h * r_hi ** np.arange(1, n_hi + 1))
    mid = -0.5 * side + h * np.arange(n_mid + 1)
    return np.concatenate([lo[::-1], mid, hi]).astype(np.float64)


def cube_flow_paper(n_cube: int = 31, n_front: int = 75, n_side: int = 75, n_rear: int = 85, m: int = 48, *,
                    Kn: float = 1.0, Ma: float = 2.0, vrange: float = 4.0, iterations: int = 41, name: str = "") -> Workload:
    """The paper's own cube workload shape: 191 x 181 x 181 cells with
    geometric expansion 1.02 (front, sides) / 1.03 (rear) away from a unit cube of n_cube^3 solid cells, Ma = 2, Kn = 1,
    48^3 velocities on [-4, 4]^3 (not shifted), free-stream Maxwellian for every entering particle.
    The paper does not give its grid cell by cell: with 31 cells across the cube the lateral count (2 x 75 + 31 = 181) and
    half-width (6.0) match its 181 cells / 12 units; the streamwise split 75 + 31 + 85 = 191 is ours."""
    xf = geometric_faces(n_front, n_cube, n_rear, 1.02, 1.03)
    yf = geometric_faces(n_side, n_cube, n_side, 1.02, 1.02)
    zf = yf.copy()
    nx, ny, nz = len(xf) - 1, len(yf) - 1, len(zf) - 1
    solid = np.zeros((nz, ny, nx), dtype=np.uint8)
    solid[n_side:n_side + n_cube, n_side:n_side + n_cube, n_front:n_front + n_cube] = 1
    U_inf = Ma * math.sqrt(5.0 / 6.0)
    xi_x, w_x = trapezoid_nodes(m, -vrange, vrange)
    xi_y, w_y = trapezoid_nodes(m, -vrange, vrange)
    xi_z, w_z = trapezoid_nodes(m, -vrange, vrange)
    fs = FaceBC(FREESTREAM, 1.0, 1.0, (U_inf, 0.0, 0.0))
    return Workload(name or f"cube_paper_{nx}x{ny}x{nz}_v{m}", xf, yf, zf, solid,
                    xi_x, xi_y, xi_z, w_x, w_y, w_z, Kn, 0.81, 2.0 / 3.0, 1.0, (U_inf, 0.0, 0.0), 1.0,
                    [fs] * 6, FaceBC(WALL_DIFFUSE, 1.0, 1.0, (0.0, 0.0, 0.0)), 0, 0, iterations)


def config(idx: int) -> Workload:
    """BASELINE.json configs[idx] as concrete arrays."""
    if idx == 0:
        return cavity(8, 8, 1.0, iterations=20, name="cfg0_cavity_8^3x8^3_Kn1")
    if idx == 1:
        return cavity(32, 24, 0.1, iterations=200, name="cfg1_cavity_32^3x24^3_Kn0.1")
    if idx == 2:
        return cavity(64, 32, 0.075, stretch=1.5, iterations=5000, name="cfg2_cavity_tanh_64^3x32^3_Kn0.075")
    if idx == 3:
        return cube_flow(16, 48, iterations=50, name="cfg3_cube_96x64x64_v48^3_Ma2")
    if idx == 4:
        return cavity(128, 64, 0.01, iterations=50, name="cfg4_cavity_128^3x64^3_Kn0.01")
    if idx == 5:   # not in BASELINE.json: the paper's own cube run
        return cube_flow_paper(name="cfg5_cube_paper_191x181x181_v48^3_Ma2_Kn1")
    if idx == 6:   # not in BASELINE.json: a 16-level slab of config 4 (same x-y plane, velocity grid and gas), the stand-in
        # for config 4 under `ncu --set full`, whose replay passes save and restore the whole 52 GB workspace of config 4
        return cavity(0, 64, 0.01, iterations=50, nxyz=(128, 128, 16), name="cfg6_slab_of_cfg4_128x128x16_v64^3_Kn0.01")
    raise ValueError(f"no config {idx}")


# ---------------------------------------------------------------------------------------------
# seeded states
# ---------------------------------------------------------------------------------------------
def uniform_state(wl: Workload) -> np.ndarray:
    """prim8 [8][nz*ny*nx]: rho, ux, uy, uz, T, qx, qy, qz of the uniform initial state."""
    n = wl.n_cells
    p = np.zeros((8, n), dtype=np.float64)
    p[0] = wl.rho0
    p[1], p[2], p[3] = wl.u0
    p[4] = wl.T0
    return p


def perturbed_state(wl: Workload, seed: int = 1810, *, amp_rho: float = 0.05, amp_T: float = 0.05,
                    amp_u: float = 0.05, amp_q: float = 0.0) -> np.ndarray:
    """BASELINE.json configs[1] kernel-level state: rho,T *(1+U(-a,a)), u += U(-a,a)^3, q += U(-aq,aq)^3."""
    rng = np.random.default_rng(seed)
    p = uniform_state(wl)
    n = wl.n_cells
    p[0] *= 1.0 + rng.uniform(-amp_rho, amp_rho, n)
    p[4] *= 1.0 + rng.uniform(-amp_T, amp_T, n)
    for d in range(3):
        p[1 + d] += rng.uniform(-amp_u, amp_u, n)
    if amp_q > 0:
        for d in range(3):
            p[5 + d] += rng.uniform(-amp_q, amp_q, n)
    if wl.solid is not None:
        p[:, wl.solid.reshape(-1) != 0] = 0.0
    return p


def sparse_weight_subset(wl: Workload, keep: int = 8, seed: int = 100348) -> Workload:
    """Zero all but `keep` seeded nodes per axis in the 1-D weights (at least one node of each sign per axis).

    Used for the full-size one-step parity of configs 3-4: the oracle skips zero-weight velocities,
    the CUDA path sweeps everything; raw moments and wall fluxes must still agree.
    """
    rng = np.random.default_rng(seed)

    def thin(xi, w):
        m = len(xi)
        if keep >= m:
            return w.copy()
        neg = np.flatnonzero(xi < 0)
        pos = np.flatnonzero(xi >= 0)
        sel = {int(rng.choice(neg)), int(rng.choice(pos))}
        while len(sel) < keep:
            sel.add(int(rng.integers(0, m)))
        out = np.zeros_like(w)
        idx = np.array(sorted(sel))
        out[idx] = w[idx]
        return out

    return wl.with_(w_x=thin(wl.xi_x, wl.w_x), w_y=thin(wl.xi_y, wl.w_y), w_z=thin(wl.xi_z, wl.w_z),
                    name=wl.name + f"_wsub{keep}")


def stratified_weight_subset(wl: Workload, boxes, seed: int = 0) -> Workload:
    """Zero all but ONE node per 1-D velocity block and axis in the 1-D weights, so that the kept velocities (their tensor
    product) put exactly one velocity into every velocity block of the CUDA tile kernel.

    `boxes` is the block table of `dvm.plan_vblocks` (rows a0, na, b0, nb, c0, nc, ...): only its node ranges are used
    here.  The position of the kept node inside its 1-D block rotates with the block and with `seed`, so that the kept
    velocities visit different register slots, lane-quad roles and lane positions of the kernel.  The oracle skips the
    zero-weight velocities; the CUDA path sweeps everything (full-size one-step parity).
    """
    boxes = np.asarray(boxes)

    def thin(w, starts_counts, stride):
        out = np.zeros_like(w)
        for n, (lo, cnt) in enumerate(sorted(set(starts_counts))):
            pos = (stride * n + 1 + seed) % cnt
            out[lo + pos] = w[lo + pos]
        return out

    bx = [(int(r[0]), int(r[1])) for r in boxes]
    by = [(int(r[2]), int(r[3])) for r in boxes]
    bz = [(int(r[4]), int(r[5])) for r in boxes]
    return wl.with_(w_x=thin(wl.w_x, bx, 5), w_y=thin(wl.w_y, by, 3), w_z=thin(wl.w_z, bz, 1),
                    name=wl.name + f"_strat{seed}")
