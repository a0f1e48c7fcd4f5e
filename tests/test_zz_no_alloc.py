"""dvm_residual_noalloc, the one entry point of the library that never allocates device memory.

It is there for hosts that cannot call cudaMalloc - the whole of HBM already sits in their own pool, or they run a
latency-critical loop that must not take the device-wide stall of cudaMalloc / cudaFree, or they are called from a context
where the CUDA allocator may not be entered.  Its partial sums go to a fixed 3 MiB array inside the library image instead of
a solver's workspace, which caps the grid at 256^3 cells and makes all calls share one array (include/dvm.h).

The GPU test compares it with the existing path - the residual a solver reports after an iteration (finish_kernel +
residual_kernel on the solver's own workspace) - at the tolerance every residual comparison of this suite uses
(tests/parity.py: 1e-9 relative + 1e-13), on calls made one straight after the other, so that whatever one call leaves in the
shared array is in place when the next one runs.

This file is named so that pytest collects it LAST (pytest --collect-only): under -x a failure here hides no other test.
It passes alone in a fresh process (then its first call is the library's one-time set-up on the GPU) and after the rest of
the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_1810_00348_b200 import workloads as W
from tests.parity import assert_residual


def test_noalloc_entry_rejects_sizes_beyond_its_fixed_array():
    """The size check comes before anything touches CUDA, so it also runs on a box without a GPU: one cell more than the
    fixed array can serve is refused with DVM_EINVAL and a message that names the limit; so are NULL and ncell <= 0."""
    from paper_1810_00348_b200 import dvm
    L = dvm.lib()
    buf = (ctypes.c_double * 8)()
    p = ctypes.cast(buf, ctypes.c_void_p)
    limit = dvm.RESIDUAL_NOALLOC_MAX_CELLS
    assert L.dvm_residual_noalloc(p, p, limit + 1, p, None) == dvm.EINVAL
    msg = L.dvm_last_error().decode()
    assert str(limit) in msg and "DVM_RESIDUAL_NOALLOC_MAX_CELLS" in msg, msg
    assert L.dvm_residual_noalloc(None, p, 8, p, None) == dvm.EINVAL
    assert L.dvm_residual_noalloc(p, p, 0, p, None) == dvm.EINVAL
    # host memory where device memory is required (or no GPU at all): refused, never computed on the CPU
    assert L.dvm_residual_noalloc(p, p, 1, p, None) in (dvm.EINVAL, dvm.ECUDA)


@pytest.mark.gpu
def test_noalloc_residual_matches_the_solver_residual_on_consecutive_calls():
    """Two solvers of different size (13^3 cells on a stretched grid = 8 full blocks of 256 and a ragged one; 8^3 = 2 blocks)
    take iterations; after each, the residual between the states before and after - recomputed by dvm_residual_noalloc from
    the two dvm_get_state outputs - must equal the one the solver itself reports.  The calls alternate large / small / large
    without anything in between, so the small call runs with the large call's partial sums still in the upper slots of the
    shared array and the last call runs on an array both earlier calls wrote.  All buffers are made before the calls; the
    free device memory must not move across them."""
    import torch
    from paper_1810_00348_b200 import dvm

    dev = torch.device("cuda:0")
    big, small = W.cavity(13, 8, 0.5, stretch=1.5), W.config(0)
    sa, sb = dvm.Solver(big), dvm.Solver(small)
    try:
        cases = []  # (state before, state after, residual of the existing path)
        for s in (sa, sb, sa):
            s.iterate(2)                       # away from the uniform initial state
            before = s.get_state()[0].clone()
            s.iterate(1)
            after = s.get_state()[0].clone()
            cases.append((before, after, s.residual()))
        outs = [torch.full((3,), -1.0, dtype=torch.float64, device=dev) for _ in cases]
        assert cases[0][0].shape[1] == 13 ** 3 and cases[1][0].shape[1] == 8 ** 3
        # set-up call (the first one on this GPU in a fresh process), then the measured sequence
        dvm.residual_noalloc(cases[0][0], cases[0][1], outs[0])
        torch.cuda.synchronize(dev)
        free0 = torch.cuda.mem_get_info(dev)[0]
        for (before, after, _), out in zip(cases, outs):
            out.fill_(-1.0)
            dvm.residual_noalloc(before, after, out)
        torch.cuda.synchronize(dev)
        assert torch.cuda.mem_get_info(dev)[0] == free0, "device memory was allocated or released during the calls"
        for k, ((_, _, ref), out) in enumerate(zip(cases, outs)):
            got = out.cpu().numpy()
            assert np.all(ref > 0) and np.all(np.isfinite(got))
            assert_residual(got, ref, what=f"dvm_residual_noalloc call {k + 1}")
        # the same pair twice in a row gives the same bits (fixed order, nothing left over from the call before matters)
        again = torch.empty(3, dtype=torch.float64, device=dev)
        dvm.residual_noalloc(cases[2][0], cases[2][1], again)
        assert torch.equal(again, outs[2])
        # identical states: r_rho is exactly 0; r_mom and r_E are the rounding left by the fused multiply-adds in
        # rho1 u1 - rho0 u0 (one product is rounded, the other is not), far below any convergence threshold
        dvm.residual_noalloc(cases[1][1], cases[1][1], again)
        same = again.cpu().numpy()
        assert same[0] == 0.0 and np.all(same >= 0.0) and same.max() < 1e-15, same
        # beyond the fixed array: a clear error, nothing launched
        with pytest.raises(dvm.DvmError, match="DVM_RESIDUAL_NOALLOC_MAX_CELLS"):
            L = dvm.lib()
            dvm._check(L.dvm_residual_noalloc(cases[0][0].data_ptr(), cases[0][1].data_ptr(),
                                              dvm.RESIDUAL_NOALLOC_MAX_CELLS + 1, outs[0].data_ptr(), None))
        # host memory is refused, not computed on the CPU
        with pytest.raises(dvm.DvmError):
            dvm.residual_noalloc(cases[0][0].cpu(), cases[0][1].cpu(), outs[0])
    finally:
        sa.close()
        sb.close()
