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
    assert L.dvm_destroy(None) == 0
