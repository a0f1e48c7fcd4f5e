"""ctypes front end of the CPU ORACLE (oracle/dvm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import
this module.  It never imports the CUDA binding (paper_1810_00348_b200.dvm) and shares no code with it;
a workload record (paper_1810_00348_b200.workloads.Workload, plain arrays + parameters) is the only
thing both sides see.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libdvm_oracle.so"
_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


class _Problem(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("xf", _dp), ("yf", _dp), ("zf", _dp),
        ("solid", C.POINTER(C.c_ubyte)),
        ("mx", C.c_int), ("my", C.c_int), ("mz", C.c_int),
        ("xi_x", _dp), ("xi_y", _dp), ("xi_z", _dp),
        ("w_x", _dp), ("w_y", _dp), ("w_z", _dp),
        ("Kn", C.c_double), ("omega", C.c_double), ("Pr", C.c_double),
        ("bc_type", C.c_int * 7),
        ("bc_T", C.c_double * 7), ("bc_rho", C.c_double * 7), ("bc_u", (C.c_double * 3) * 7),
        ("rescale_mass", C.c_int), ("wall_norm", C.c_int), ("order", C.c_int),
        ("f32", C.c_int),
    ]


def build(force: bool = False) -> Path:
    """Compile oracle/dvm_oracle.c with gcc (plain -O2, OpenMP, no fast-math)."""
    src = _HERE / "dvm_oracle.c"
    hdr = _HERE / "dvm_oracle.h"
    if not force and _SO.exists() and _SO.stat().st_mtime >= max(src.stat().st_mtime, hdr.stat().st_mtime):
        return _SO
    tmp = _SO.with_suffix(f".{os.getpid()}.tmp")
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", str(tmp), str(src), "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_SO))
        PP = C.POINTER(_Problem)
        L.odvm_num_faces.argtypes = [PP]
        L.odvm_face_table.argtypes = [PP, _ip, _ip, _dp]
        L.odvm_c_omega.argtypes = [C.c_double]
        L.odvm_c_omega.restype = C.c_double
        L.odvm_tau.argtypes = [PP, C.c_double, C.c_double]
        L.odvm_tau.restype = C.c_double
        L.odvm_feq.argtypes = [PP, _dp, _dp]
        L.odvm_feq.restype = C.c_double
        L.odvm_gwall.argtypes = [PP, C.c_int, _dp]
        L.odvm_gwall.restype = C.c_double
        L.odvm_phi_unit.argtypes = [PP, _dp]
        L.odvm_rho_equilibrium.argtypes = [PP, _dp, _dp]
        L.odvm_init_state.argtypes = [PP, C.c_double, _dp, C.c_double, _dp, _dp, _dp]
        L.odvm_total_mass.argtypes = [PP, _dp]
        L.odvm_total_mass.restype = C.c_double
        L.odvm_step.argtypes = [PP, _dp, _dp, C.c_double, _dp, _dp, _dp, _dp, _dp, _dp, _dp, C.c_int]
        L.odvm_sweep_velocity.argtypes = [PP, _dp, _dp, C.c_int, C.c_int, C.c_int, _dp]
        _lib = L
    return _lib


def _arr(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_dp)


class Oracle:
    """One problem instance; holds the state (W^n, rho_w^n) between `step()` calls."""

    def __init__(self, wl):
        self.wl = wl
        self._keep = [_arr(x) for x in (wl.xf, wl.yf, wl.zf, wl.xi_x, wl.xi_y, wl.xi_z, wl.w_x, wl.w_y, wl.w_z)]
        p = _Problem()
        p.nx, p.ny, p.nz = wl.nx, wl.ny, wl.nz
        p.xf, p.yf, p.zf = (_p(a) for a in self._keep[0:3])
        if wl.solid is not None:
            self._solid = np.ascontiguousarray(wl.solid, dtype=np.uint8).reshape(-1)
            p.solid = self._solid.ctypes.data_as(C.POINTER(C.c_ubyte))
        else:
            self._solid = None
            p.solid = None
        p.mx, p.my, p.mz = wl.mx, wl.my, wl.mz
        p.xi_x, p.xi_y, p.xi_z = (_p(a) for a in self._keep[3:6])
        p.w_x, p.w_y, p.w_z = (_p(a) for a in self._keep[6:9])
        p.Kn, p.omega, p.Pr = wl.Kn, wl.omega, wl.Pr
        for b, bc in enumerate(list(wl.faces) + [wl.solid_bc]):
            p.bc_type[b] = bc.type
            p.bc_T[b] = bc.T
            p.bc_rho[b] = bc.rho
            for d in range(3):
                p.bc_u[b][d] = bc.u[d]
        p.rescale_mass, p.wall_norm = wl.rescale_mass, wl.wall_norm
        p.order = getattr(wl, "order", 1)
        p.f32 = 1 if getattr(wl, "f32", False) else 0   # the sweep in IEEE single (reading G22), sums in extended precision
        self.p = p
        self.n = wl.n_cells
        self.nface = lib().odvm_num_faces(C.byref(p))
        if self.nface < 0:
            raise MemoryError("oracle face table")
        # state
        self.prim8 = np.zeros((8, self.n))
        self.rho_w = np.zeros(self.nface)
        m0 = C.c_double()
        u0 = _arr(wl.u0)
        rc = lib().odvm_init_state(C.byref(p), wl.rho0, _p(u0), wl.T0, _p(self.prim8), _p(self.rho_w), C.byref(m0))
        if rc:
            raise RuntimeError("odvm_init_state failed")
        self.mass0 = m0.value
        self.prim14 = None
        self.raw13 = None
        self.flux_out = None
        self.flux_in = None
        self.resid = None
        self.scale = None
        self.threads = None
        self.history = []

    # -- helpers used by the pins ---------------------------------------------------------------
    def face_table(self):
        cell = np.zeros(self.nface, dtype=np.int32)
        dirn = np.zeros(self.nface, dtype=np.int32)
        area = np.zeros(self.nface)
        lib().odvm_face_table(C.byref(self.p), cell.ctypes.data_as(_ip), dirn.ctypes.data_as(_ip), _p(area))
        return cell, dirn, area

    def c_omega(self):
        return lib().odvm_c_omega(self.wl.omega)

    def tau(self, rho, T):
        return lib().odvm_tau(C.byref(self.p), rho, T)

    def feq(self, W8, xi3):
        W8, xi3 = _arr(W8), _arr(xi3)
        return lib().odvm_feq(C.byref(self.p), _p(W8), _p(xi3))

    def gwall(self, b, xi3):
        xi3 = _arr(xi3)
        return lib().odvm_gwall(C.byref(self.p), b, _p(xi3))

    def phi_unit(self):
        out = np.zeros(self.nface)
        lib().odvm_phi_unit(C.byref(self.p), _p(out))
        return out

    def rho_equilibrium(self, prim8=None):
        prim8 = _arr(self.prim8 if prim8 is None else prim8)
        out = np.zeros(self.n)
        lib().odvm_rho_equilibrium(C.byref(self.p), _p(prim8), _p(out))
        return out

    def total_mass(self, rho):
        rho = _arr(rho)
        return lib().odvm_total_mass(C.byref(self.p), _p(rho))

    def sweep_velocity(self, ia, ib, ic, prim8=None, rho_w=None):
        prim8 = _arr(self.prim8 if prim8 is None else prim8)
        rho_w = _arr(self.rho_w if rho_w is None else rho_w)
        f = np.zeros(self.n)
        lib().odvm_sweep_velocity(C.byref(self.p), _p(prim8), _p(rho_w), ia, ib, ic, _p(f))
        return f.reshape(self.wl.nz, self.wl.ny, self.wl.nx)

    # -- the iteration --------------------------------------------------------------------------
    def set_state(self, prim8, rho_w=None):
        self.prim8 = _arr(prim8).reshape(8, self.n).copy()
        if rho_w is not None:
            self.rho_w = _arr(rho_w).reshape(self.nface).copy()

    def step(self, nthreads: int = 0):
        """One outer iteration; updates the held state and returns prim14 [14][ncell]."""
        raw = np.zeros((13, self.n))
        prim14 = np.zeros((14, self.n))
        rho_w = np.zeros(self.nface)
        fo = np.zeros(self.nface)
        fi = np.zeros(self.nface)
        res = np.zeros(3)
        sc = C.c_double()
        rc = lib().odvm_step(C.byref(self.p), _p(self.prim8), _p(self.rho_w), self.mass0, _p(raw), _p(prim14),
                             _p(rho_w), _p(fo), _p(fi), _p(res), C.byref(sc), nthreads)
        if rc < 0:
            raise RuntimeError(f"odvm_step failed ({rc})")
        self.threads = rc
        self.prev_prim8, self.prev_rho_w = self.prim8, self.rho_w
        self.raw13, self.prim14, self.flux_out, self.flux_in = raw, prim14, fo, fi
        self.resid, self.scale = res, sc.value
        self.prim8 = prim14[:8].copy()
        self.rho_w = rho_w
        self.history.append(res.copy())
        return prim14
