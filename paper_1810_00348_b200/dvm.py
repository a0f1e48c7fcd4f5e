"""Thin Python binding of the C ABI in include/dvm.h (same names; argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libdvm_b200.so.  PyTorch is used for device
memory (the solver's workspace is obtained through the torch caching allocator), streams and nothing
else.  There is no CPU fallback: if the library is missing or no CUDA device is present this fails loudly.
This module never imports anything under oracle/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_CSRC = _PKG / "csrc"
# DVM_B200_LIB names another build of the same library (kernel experiments); default: the in-tree build
_SO = Path(os.environ.get("DVM_B200_LIB", str(_PKG / "libdvm_b200.so")))
_INCLUDE = _PKG.parent / "include"

OK, EINVAL, ENOMEM, ECUDA, ENONFINITE = 0, -1, -2, -3, -4
WALL_DIFFUSE, FREESTREAM, ZERO_GRADIENT = 0, 1, 2
KERNEL_AUTO, KERNEL_SLICE, KERNEL_TILE = 0, 1, 2
OPT_KERNEL = 1
OPT_MAX_F_MBYTES = 2
OPT_TILE_RV = 3
OPT_MAX_CTAS = 4
OPT_ORDER = 5
OPT_TILE_AXIS = 6
OPT_PRECISION = 7
OPT_SHARD_COUNT = 8
OPT_SHARD_RANK = 9
PREC_F64, PREC_MIXED = 0, 1

# every symbol include/dvm.h declares (checked by tests/test_abi.py)
SYMBOLS = (
    "dvm_create", "dvm_iterate", "dvm_moments", "dvm_residual", "dvm_num_faces", "dvm_iterations_done",
    "dvm_get_state", "dvm_set_state", "dvm_raw_moments", "dvm_wall_flux", "dvm_residual_history",
    "dvm_mass_scale", "dvm_step_host", "dvm_set_option", "dvm_workspace_bytes", "dvm_launch_count",
    "dvm_kernel_used", "dvm_tile_rv", "dvm_tile_axis", "dvm_precision", "dvm_plan_query", "dvm_plan_vblocks",
    "dvm_plan_shard_vblocks", "dvm_sweep", "dvm_update", "dvm_reduce_buffer", "dvm_destroy", "dvm_last_error",
    "dvm_residual_noalloc", "dvm_graph_active", "dvm_fp64_peak_probe",
)

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


class DvmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"dvm error {code}: {msg}")
        self.code = code


def build(force: bool = False, verbose: bool = False) -> Path:
    """Compile csrc/*.cu for sm_100a into libdvm_b200.so (in-tree)."""
    srcs = sorted(_CSRC.glob("*.cu"))
    deps = srcs + sorted(_CSRC.glob("*.cuh")) + [_INCLUDE / "dvm.h"]
    if not force and _SO.exists() and _SO.stat().st_mtime >= max(p.stat().st_mtime for p in deps):
        return _SO
    tmp = _SO.with_suffix(f".{os.getpid()}.tmp")
    cmd = ["nvcc", *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), *map(str, srcs)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _SO)
    return _SO


_dp = C.POINTER(C.c_double)


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("xf", _dp), ("yf", _dp), ("zf", _dp),
                ("solid", C.POINTER(C.c_ubyte))]


class _VGrid(C.Structure):
    _fields_ = [("mx", C.c_int), ("my", C.c_int), ("mz", C.c_int), ("xi_x", _dp), ("xi_y", _dp), ("xi_z", _dp),
                ("w_x", _dp), ("w_y", _dp), ("w_z", _dp)]


class _Gas(C.Structure):
    _fields_ = [("Kn", C.c_double), ("omega", C.c_double), ("Pr", C.c_double), ("rho0", C.c_double),
                ("u0", C.c_double * 3), ("T0", C.c_double)]


class _FaceBC(C.Structure):
    _fields_ = [("type", C.c_int), ("T", C.c_double), ("rho", C.c_double), ("u", C.c_double * 3)]


class _BC(C.Structure):
    _fields_ = [("face", _FaceBC * 6), ("solid", _FaceBC), ("rescale_mass", C.c_int), ("wall_norm", C.c_int)]


_ALLOC = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class _Device(C.Structure):
    _fields_ = [("stream", C.c_void_p), ("alloc", _ALLOC), ("free_", _FREE), ("ctx", C.c_void_p)]


_lib = None


def lib():
    """Load libdvm_b200.so (building it if the sources are newer).  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        if "DVM_B200_LIB" not in os.environ:
            build()   # no-op when the library is newer than every source
        L = C.CDLL(str(_SO))
        vp = C.c_void_p
        L.dvm_create.argtypes = [C.POINTER(_Grid), C.POINTER(_VGrid), C.POINTER(_Gas), C.POINTER(_BC),
                                 C.POINTER(_Device), C.POINTER(vp)]
        L.dvm_iterate.argtypes = [vp, C.c_int]
        L.dvm_moments.argtypes = [vp, vp]
        L.dvm_residual.argtypes = [vp, _dp]
        L.dvm_num_faces.argtypes = [vp]
        L.dvm_iterations_done.argtypes = [vp]
        L.dvm_get_state.argtypes = [vp, vp, vp]
        L.dvm_set_state.argtypes = [vp, vp, vp]
        L.dvm_raw_moments.argtypes = [vp, vp]
        L.dvm_wall_flux.argtypes = [vp, vp]
        L.dvm_residual_history.argtypes = [vp, _dp, C.c_int]
        L.dvm_mass_scale.argtypes = [vp, _dp]
        L.dvm_step_host.argtypes = [vp, vp, vp, C.c_int, vp, vp]
        L.dvm_set_option.argtypes = [vp, C.c_int, C.c_int]
        L.dvm_workspace_bytes.argtypes = [vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        L.dvm_kernel_used.argtypes = [vp]
        L.dvm_tile_rv.argtypes = [vp]
        L.dvm_precision.argtypes = [vp]
        L.dvm_sweep.argtypes = [vp]
        L.dvm_update.argtypes = [vp]
        L.dvm_reduce_buffer.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_size_t)]
        L.dvm_plan_shard_vblocks.argtypes = [C.POINTER(_VGrid), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.c_int]
        L.dvm_tile_axis.argtypes = [vp]
        L.dvm_plan_query.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(_VGrid), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                     C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_int]
        L.dvm_plan_vblocks.argtypes = [C.POINTER(_VGrid), C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.c_int]
        L.dvm_launch_count.argtypes = [vp]
        L.dvm_graph_active.argtypes = [vp]
        L.dvm_launch_count.restype = C.c_longlong
        L.dvm_destroy.argtypes = [vp]
        L.dvm_last_error.restype = C.c_char_p
        L.dvm_residual_noalloc.argtypes = [vp, vp, C.c_longlong, vp, vp]
        L.dvm_fp64_peak_probe.argtypes = [vp, C.c_longlong, _dp, _dp]
        _lib = L
    return _lib


def _check(rc):
    if rc < 0:
        raise DvmError(rc, lib().dvm_last_error().decode())
    return rc


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def plan_query(nx, ny, nz, xi_x, xi_y, xi_z, target_ctas=296, max_blocks=0, max_items=1 << 22, rv=0, order=1, wide_axis=0):
    """dvm_plan_query: (counts dict, items int32 [n][9]) of the tile kernel's work decomposition (host only)."""
    keep = [_f64(a) for a in (xi_x, xi_y, xi_z)]
    v = _VGrid(len(keep[0]), len(keep[1]), len(keep[2]), *(a.ctypes.data_as(_dp) for a in keep), None, None, None)
    counts = (C.c_int * 5)()
    n = _check(lib().dvm_plan_query(nx, ny, nz, C.byref(v), target_ctas, max_blocks, rv, order, wide_axis, counts, None, 0))
    items = np.zeros((min(n, max_items), 9), dtype=np.int32)
    _check(lib().dvm_plan_query(nx, ny, nz, C.byref(v), target_ctas, max_blocks, rv, order, wide_axis, counts,
                                items.ctypes.data_as(C.POINTER(C.c_int)), len(items)))
    return {"n_vblocks": counts[0], "ntx": counts[1], "nty": counts[2], "P": counts[3], "batch": counts[4],
            "n_items": n}, items


def plan_vblocks(xi_x, xi_y, xi_z, rv=0, order=1, wide_axis=0):
    """dvm_plan_vblocks: int32 [n][8] = x0, nx, y0, ny, z0, nz, NA + 65536 (1 + wide axis), 256 nbb + ncb per velocity block
    (host only); wide_axis: 0 = the library's choice, 1 + axis otherwise."""
    keep = [_f64(a) for a in (xi_x, xi_y, xi_z)]
    v = _VGrid(len(keep[0]), len(keep[1]), len(keep[2]), *(a.ctypes.data_as(_dp) for a in keep), None, None, None)
    n = _check(lib().dvm_plan_vblocks(C.byref(v), rv, order, wide_axis, None, 0))
    out = np.zeros((n, 8), dtype=np.int32)
    _check(lib().dvm_plan_vblocks(C.byref(v), rv, order, wide_axis, out.ctypes.data_as(C.POINTER(C.c_int)), n))
    return out


def plan_shard_vblocks(xi_x, xi_y, xi_z, rank, count, rv=0, order=1, wide_axis=0):
    """dvm_plan_shard_vblocks: the velocity blocks (as plan_vblocks) of rank `rank` of `count` (host only)."""
    keep = [_f64(a) for a in (xi_x, xi_y, xi_z)]
    v = _VGrid(len(keep[0]), len(keep[1]), len(keep[2]), *(a.ctypes.data_as(_dp) for a in keep), None, None, None)
    n = _check(lib().dvm_plan_shard_vblocks(C.byref(v), rv, order, wide_axis, rank, count, None, 0))
    out = np.zeros((n, 8), dtype=np.int32)
    _check(lib().dvm_plan_shard_vblocks(C.byref(v), rv, order, wide_axis, rank, count, out.ctypes.data_as(C.POINTER(C.c_int)), n))
    return out


def fp64_peak_probe(device="cuda:0", rounds: int = 2_000_000):
    """dvm_fp64_peak_probe on `device`: (fp64 lane-operations per second the board sustains on register-resident DFMA chains,
    milliseconds of the timed launch).  Measurement aid for bench.py's roofline."""
    import torch
    with torch.cuda.device(torch.device(device)):
        sink = torch.zeros(1, dtype=torch.float64, device=device)
        rate, ms = C.c_double(), C.c_double()
        _check(lib().dvm_fp64_peak_probe(sink.data_ptr(), int(rounds), C.byref(rate), C.byref(ms)))
    return rate.value, ms.value


RESIDUAL_NOALLOC_MAX_CELLS = 1 << 24


def residual_noalloc(prim_old, prim_new, out3, stream=None):
    """dvm_residual_noalloc: the residual triple (r_rho, r_mom, r_E) between two macroscopic states on the GPU,
    written to `out3`, for hosts that cannot allocate device memory (all of HBM already in their own pool, a latency-critical
    loop, a context where the CUDA allocator may not be entered): the call makes no allocation, its partial sums sit in a fixed
    3 MiB array of the library image.  Limits that follow (include/dvm.h has the full text): at most RESIDUAL_NOALLOC_MAX_CELLS
    cells (DvmError EINVAL beyond); every call shares that array, so calls that could overlap on the GPU must be serialised by the
    caller; the first call on a GPU does a one-time set-up and belongs in start-up code, before any stream capture.

    prim_old, prim_new: CUDA float64 tensors [>= 5][ncell] (rho, ux, uy, uz, T first; the outputs of Solver.moments() or
    get_state() fit as they are), contiguous, same shape; out3: CUDA float64 tensor of 3 elements on the same GPU, supplied by the
    caller - this function allocates nothing either.  stream: a torch.cuda.Stream (default: torch's current stream of that GPU).
    Asynchronous; returns out3."""
    import torch
    if not (prim_old.is_cuda and prim_new.is_cuda and out3.is_cuda):
        raise DvmError(EINVAL, "residual_noalloc: CUDA tensors required (there is no CPU fallback)")
    if prim_old.dtype != torch.float64 or prim_new.dtype != torch.float64 or out3.dtype != torch.float64:
        raise DvmError(EINVAL, "residual_noalloc: float64 tensors required")
    if prim_old.shape != prim_new.shape or prim_old.dim() != 2 or prim_old.shape[0] < 5 or out3.numel() < 3:
        raise DvmError(EINVAL, "residual_noalloc: prim_old / prim_new must be [>= 5][ncell] and alike, out3 must hold 3 values")
    if not (prim_old.is_contiguous() and prim_new.is_contiguous() and out3.is_contiguous()):
        raise DvmError(EINVAL, "residual_noalloc: contiguous tensors required")
    st = torch.cuda.current_stream(out3.device) if stream is None else stream
    _check(lib().dvm_residual_noalloc(prim_old.data_ptr(), prim_new.data_ptr(), int(prim_old.shape[1]), out3.data_ptr(),
                                      st.cuda_stream))
    return out3


class Solver:
    """dvm_create / dvm_iterate / dvm_moments / dvm_residual (+ support calls) for one workload record."""

    def __init__(self, wl, kernel: int = KERNEL_AUTO, device: str = "cuda:0", max_f_mbytes: int = 0, tile_rv: int = 0,
                 max_ctas: int = 0, order: int = 0, tile_axis: int = 0, precision: int = -1, shard=None):
        import torch
        if not torch.cuda.is_available():
            raise DvmError(ECUDA, "no CUDA device: the DVM solver has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.wl = wl
        self.ncell = wl.n_cells
        L = lib()
        keep = [_f64(x) for x in (wl.xf, wl.yf, wl.zf, wl.xi_x, wl.xi_y, wl.xi_z, wl.w_x, wl.w_y, wl.w_z)]
        g = _Grid(wl.nx, wl.ny, wl.nz, *(a.ctypes.data_as(_dp) for a in keep[0:3]), None)
        if wl.solid is not None:
            solid = np.ascontiguousarray(wl.solid, dtype=np.uint8).reshape(-1)
            g.solid = solid.ctypes.data_as(C.POINTER(C.c_ubyte))
        v = _VGrid(wl.mx, wl.my, wl.mz, *(a.ctypes.data_as(_dp) for a in keep[3:9]))
        gas = _Gas(wl.Kn, wl.omega, wl.Pr, wl.rho0, (C.c_double * 3)(*wl.u0), wl.T0)
        bc = _BC()
        for b, f in enumerate(list(wl.faces) + [wl.solid_bc]):
            dst = bc.face[b] if b < 6 else bc.solid
            dst.type, dst.T, dst.rho = f.type, f.T, f.rho
            for d in range(3):
                dst.u[d] = f.u[d]
        bc.rescale_mass, bc.wall_norm = wl.rescale_mass, wl.wall_norm

        # device memory comes from the torch caching allocator; tensors are kept alive in this dict
        self._blocks = {}

        def _alloc(nbytes, ctx):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
            except Exception:
                return None
            self._blocks[t.data_ptr()] = t
            return t.data_ptr()

        def _free(ptr, ctx):
            self._blocks.pop(ptr, None)

        self._alloc_cb, self._free_cb = _ALLOC(_alloc), _FREE(_free)
        self.stream = torch.cuda.current_stream(self.device)
        dev = _Device(self.stream.cuda_stream, self._alloc_cb, self._free_cb, None)
        h = C.c_void_p()
        _check(L.dvm_create(C.byref(g), C.byref(v), C.byref(gas), C.byref(bc), C.byref(dev), C.byref(h)))
        self._h = h
        self.nface = _check(L.dvm_num_faces(h))
        order = order or getattr(wl, "order", 1)
        if order != 1:
            self.set_option(OPT_ORDER, int(order))
        if kernel != KERNEL_AUTO:
            self.set_option(OPT_KERNEL, kernel)
        if max_f_mbytes:
            self.set_option(OPT_MAX_F_MBYTES, int(max_f_mbytes))
        if tile_rv:
            self.set_option(OPT_TILE_RV, int(tile_rv))
        if max_ctas:
            self.set_option(OPT_MAX_CTAS, int(max_ctas))
        if tile_axis:
            self.set_option(OPT_TILE_AXIS, int(tile_axis))
        if precision < 0:
            precision = PREC_MIXED if getattr(wl, "f32", False) else PREC_F64
        if precision != PREC_F64:
            self.set_option(OPT_PRECISION, int(precision))
        # velocity-space sharding: shard = (rank, count); this solver sweeps 1 of `count` parts of the velocity blocks
        self.shard = (0, 1) if shard is None else (int(shard[0]), int(shard[1]))
        if self.shard[1] > 1:
            self.set_option(OPT_SHARD_COUNT, self.shard[1])
            self.set_option(OPT_SHARD_RANK, self.shard[0])

    # -- the four calls of the north star ---------------------------------------------------------
    def iterate(self, n: int = 1):
        _check(lib().dvm_iterate(self._h, n))

    # -- velocity-space sharding (DVM_OPT_SHARD_COUNT): sweep -> all-reduce over the ranks -> update ---------------
    def sweep(self):
        _check(lib().dvm_sweep(self._h))

    def update(self):
        _check(lib().dvm_update(self._h))

    def reduce_buffer(self):
        """The [ncell][16] fp64 accumulator the ranks must sum between sweep() and update(), as a torch view of the solver's
        own allocation (no copy)."""
        ptr, n = C.c_void_p(), C.c_size_t()
        _check(lib().dvm_reduce_buffer(self._h, C.byref(ptr), C.byref(n)))
        block = self._blocks[ptr.value]
        return block[: 8 * n.value].view(self.torch.float64)

    def plan_signature(self):
        """What every rank of a sharded run must agree on for the ranks' velocity blocks to partition the velocity grid: kernel
        variant, velocities per thread, wide axis, precision (valid once the first sweep has planned the workspace)."""
        return (self.kernel_used(), self.tile_rv(), self.tile_axis(), self.precision())

    def iterate_sharded(self, n: int = 1, group=None):
        """n outer iterations of a velocity-sharded solver: every rank sweeps its velocity blocks, one all-reduce (sum, fp64;
        NCCL through torch.distributed) of the velocity sums per iteration, then every rank updates the replicated macroscopic
        state.  With one rank this is iterate(n).

        Stream order: the kernels of dvm_sweep / dvm_update run on the stream the solver was created with, torch's collective
        orders itself against torch's CURRENT stream; the loop therefore runs with the solver's stream made current, whatever
        stream the caller is on.  After the first sweep (which plans the workspace) the ranks compare their plan_signature():
        ranks that chose different block shapes would count velocities twice or not at all."""
        if self.shard[1] == 1:
            return self.iterate(n)
        import contextlib
        import torch
        import torch.distributed as dist
        buf = self.reduce_buffer()
        on_stream = torch.cuda.stream(self.stream) if buf.is_cuda else contextlib.nullcontext()
        with on_stream:
            for _ in range(n):
                self.sweep()
                if not getattr(self, "_shard_plan_checked", False):
                    sigs = [None] * dist.get_world_size(group)
                    dist.all_gather_object(sigs, tuple(self.plan_signature()), group=group)
                    if any(sg != sigs[0] for sg in sigs):
                        raise DvmError(EINVAL, f"sharded ranks planned different sweeps (kernel, rv, axis, precision): {sigs}")
                    self._shard_plan_checked = True
                dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
                self.update()

    def moments(self, out=None):
        out = self._dev_empty(14 * self.ncell) if out is None else out
        _check(lib().dvm_moments(self._h, out.data_ptr()))
        return out.view(14, self.ncell)

    def residual(self):
        r = np.zeros(3)
        _check(lib().dvm_residual(self._h, r.ctypes.data_as(_dp)))
        return r

    # -- support calls ------------------------------------------------------------------------------
    def _dev_empty(self, n):
        return self.torch.empty(n, dtype=self.torch.float64, device=self.device)

    def set_option(self, option, value):
        _check(lib().dvm_set_option(self._h, option, value))

    def iterations_done(self):
        return _check(lib().dvm_iterations_done(self._h))

    def get_state(self):
        p, r = self._dev_empty(14 * self.ncell), self._dev_empty(max(self.nface, 1))
        _check(lib().dvm_get_state(self._h, p.data_ptr(), r.data_ptr()))
        return p.view(14, self.ncell), r[: self.nface]

    def set_state(self, prim8, rho_w=None):
        t = self.torch
        p = t.as_tensor(np.ascontiguousarray(prim8, dtype=np.float64) if isinstance(prim8, np.ndarray) else prim8,
                        device=self.device).contiguous()
        assert p.numel() == 8 * self.ncell
        r = None
        if rho_w is not None:
            r = t.as_tensor(np.ascontiguousarray(rho_w, dtype=np.float64) if isinstance(rho_w, np.ndarray) else rho_w,
                            device=self.device).contiguous()
            assert r.numel() == self.nface
        _check(lib().dvm_set_state(self._h, p.data_ptr(), None if r is None else r.data_ptr()))
        t.cuda.current_stream(self.device).synchronize()

    def raw_moments(self):
        out = self._dev_empty(13 * self.ncell)
        _check(lib().dvm_raw_moments(self._h, out.data_ptr()))
        return out.view(13, self.ncell)

    def wall_flux(self):
        out = self._dev_empty(max(self.nface, 1))
        _check(lib().dvm_wall_flux(self._h, out.data_ptr()))
        return out[: self.nface]

    def residual_history(self, max_n=1 << 14):
        buf = np.zeros(3 * max(max_n, 1))
        n = _check(lib().dvm_residual_history(self._h, buf.ctypes.data_as(_dp), max_n))
        return buf[: 3 * n].reshape(n, 3)

    def mass_scale(self):
        v = C.c_double()
        _check(lib().dvm_mass_scale(self._h, C.byref(v)))
        return v.value

    def step_host(self, host_prim8, host_rho_w, n, host_prim14_out, host_rho_w_out):
        """End-to-end call with HOST (pinned torch or numpy) buffers; copies run inside the call."""
        def ptr(x):
            if x is None:
                return None
            return x.data_ptr() if hasattr(x, "data_ptr") else x.ctypes.data
        _check(lib().dvm_step_host(self._h, ptr(host_prim8), ptr(host_rho_w), n, ptr(host_prim14_out), ptr(host_rho_w_out)))

    def workspace_bytes(self):
        a, b = C.c_size_t(), C.c_size_t()
        _check(lib().dvm_workspace_bytes(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def kernel_used(self):
        return _check(lib().dvm_kernel_used(self._h))

    def tile_rv(self):
        return _check(lib().dvm_tile_rv(self._h))

    def tile_axis(self):
        return _check(lib().dvm_tile_axis(self._h))

    def precision(self):
        return _check(lib().dvm_precision(self._h))

    def launch_count(self):
        return int(lib().dvm_launch_count(self._h))

    def graph_active(self):
        """1: iterations replay the captured CUDA graph; 0: plain launches, no graph in use; 2: plain launches because the
        capture failed (dvm_graph_active)."""
        return _check(lib().dvm_graph_active(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib().dvm_destroy(self._h)
            self._h = None
            self._blocks.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
