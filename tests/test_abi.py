"""CPU checks of the C-ABI boundary: the library builds for sm_100a, loads, and exports every symbol that
include/dvm.h declares; without a GPU the product path fails loudly (no CPU fallback)."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


def declared_symbols():
    text = (ROOT / "include" / "dvm.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dvm_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_exported():
    from paper_1810_00348_b200 import dvm
    so = dvm.build()
    L = ctypes.CDLL(str(so))
    names = declared_symbols()
    assert len(names) >= 19
    for n in names:
        assert hasattr(L, n), n
    assert sorted(dvm.SYMBOLS) == names


def test_binding_does_not_import_oracle():
    src = (ROOT / "paper_1810_00348_b200" / "dvm.py").read_text()
    assert "import oracle" not in src and "from oracle" not in src
    for f in (ROOT / "paper_1810_00348_b200" / "csrc").iterdir():
        assert "oracle/" not in f.read_text().replace("nothing shared with oracle/", "").replace("shares nothing with oracle/", "")


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1810_00348_b200 import dvm, workloads
    with pytest.raises(dvm.DvmError):
        dvm.Solver(workloads.config(0))


def test_create_rejects_bad_input_without_gpu():
    """Argument validation happens before any CUDA call."""
    from paper_1810_00348_b200 import dvm
    L = dvm.lib()
    h = ctypes.c_void_p()
    assert L.dvm_create(None, None, None, None, None, ctypes.byref(h)) == dvm.EINVAL
    assert b"NULL" in L.dvm_last_error()
    assert L.dvm_iterate(None, 1) == dvm.EINVAL
    assert L.dvm_sweep(None) == dvm.EINVAL and L.dvm_update(None) == dvm.EINVAL
    assert L.dvm_reduce_buffer(None, None, None) == dvm.EINVAL
    assert L.dvm_set_option(None, dvm.OPT_SHARD_COUNT, 2) == dvm.EINVAL
    assert L.dvm_precision(None) == dvm.EINVAL
    assert L.dvm_destroy(None) == 0


def _create(nx=4, ny=4, nz=4, m=4, **kw):
    """dvm_create on hand-made arrays; returns the error code (validation happens before any CUDA call)."""
    import numpy as np
    from paper_1810_00348_b200 import dvm
    L = dvm.lib()
    dp = ctypes.POINTER(ctypes.c_double)
    xf = kw.get("xf", np.linspace(0.0, 1.0, nx + 1)); yf = np.linspace(0.0, 1.0, ny + 1); zf = np.linspace(0.0, 1.0, nz + 1)
    xi = kw.get("xi", np.linspace(-3.0, 3.0, m)); w = kw.get("w", np.full(m, 6.0 / (m - 1)))
    keep = [np.ascontiguousarray(a, dtype=np.float64) for a in (xf, yf, zf, xi, w)]
    g = dvm._Grid(nx, ny, nz, keep[0].ctypes.data_as(dp), keep[1].ctypes.data_as(dp), keep[2].ctypes.data_as(dp), None)
    v = dvm._VGrid(m, m, m, *([keep[3].ctypes.data_as(dp)] * 3), *([keep[4].ctypes.data_as(dp)] * 3))
    gas = dvm._Gas(kw.get("Kn", 1.0), 0.81, 2.0 / 3.0, 1.0, (ctypes.c_double * 3)(0, 0, 0), 1.0)
    bc = dvm._BC()
    for b in range(6):
        bc.face[b].type, bc.face[b].T, bc.face[b].rho = kw.get("bctype", 0), 1.0, 1.0
    bc.solid.type, bc.solid.T = 0, 1.0
    h = ctypes.c_void_p()
    rc = L.dvm_create(ctypes.byref(g), ctypes.byref(v), ctypes.byref(gas), ctypes.byref(bc), None, ctypes.byref(h))
    if rc == 0:
        L.dvm_destroy(h)
    return rc, L.dvm_last_error().decode()


def test_create_validation_edge_cases():
    """Degenerate and maximum sizes, bad arrays: every case is refused with DVM_EINVAL and a message (on a GPU box a valid
    case would succeed; without a device it stops at DVM_ECUDA, after validation)."""
    import numpy as np
    from paper_1810_00348_b200 import dvm
    assert _create(nx=0)[0] == dvm.EINVAL                                         # empty grid
    rc, msg = _create(nx=2000, ny=2000, nz=2000)                                  # 8e9 cells: beyond the 32-bit cell index
    assert rc == dvm.EINVAL and "too many cells" in msg
    assert _create(xf=np.array([0.0, 0.5, 0.5, 0.75, 1.0]))[0] == dvm.EINVAL      # faces not strictly increasing
    assert _create(xi=np.array([-3.0, 1.0, -1.0, 3.0]))[0] == dvm.EINVAL          # nodes not increasing
    assert _create(w=np.array([2.0, -2.0, 2.0, 2.0]))[0] == dvm.EINVAL            # negative weight
    assert _create(Kn=0.0)[0] == dvm.EINVAL
    assert _create(bctype=7)[0] == dvm.EINVAL
    rc, msg = _create()                                                            # valid input
    assert rc in (0, dvm.ECUDA), msg
