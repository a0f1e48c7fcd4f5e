"""Parity metric of DESIGN.md reading G17 (shared by the GPU parity tests and smoke())."""
import numpy as np

FIELD_GROUPS = {"rho": [0], "u": [1, 2, 3], "T": [4], "q": [5, 6, 7], "sigma": [8, 9, 10, 11, 12, 13]}
TOL_FIELDS = 1e-11      # north_star: macroscopic fields, relative, per iteration
TOL_ZERO = 1e-13        # absolute, for a field that is identically zero in the oracle


def field_errors(gpu14, cpu14, fluid=None):
    """max|gpu - cpu| / max|cpu| per field group (vector / tensor fields normalised over all components)."""
    out = {}
    g = np.asarray(gpu14)
    c = np.asarray(cpu14)
    if fluid is not None:
        g, c = g[:, fluid], c[:, fluid]
    for name, idx in FIELD_GROUPS.items():
        scale = np.abs(c[idx]).max()
        err = np.abs(g[idx] - c[idx]).max()
        out[name] = err / scale if scale > 1e-12 else err * (TOL_FIELDS / TOL_ZERO)
    return out


def assert_fields(gpu14, cpu14, fluid=None, tol=TOL_FIELDS, what=""):
    errs = field_errors(gpu14, cpu14, fluid)
    bad = {k: v for k, v in errs.items() if not v <= tol}
    assert not bad, f"{what}: field parity {bad} (all: {errs})"
    return errs


def assert_residual(r_gpu, r_cpu, what=""):
    """north_star 'residual histories agree to 1e-9': |r_gpu - r_cpu| <= 1e-9 r_cpu + 1e-13 (step 7)."""
    r_gpu, r_cpu = np.asarray(r_gpu), np.asarray(r_cpu)
    assert np.all(np.abs(r_gpu - r_cpu) <= 1e-9 * np.abs(r_cpu) + 1e-13), f"{what}: residual {r_gpu} vs {r_cpu}"


def tol32(wl, K=16.0):
    """Absolute tolerance (units of DESIGN.md section 2) of every field of the single-precision sweep against the double
    oracle: K u L with u = 2^-24 and L = nx + ny + nz the longest upwind path (reading G22; derivation in
    tests/test_oracle_f32.py)."""
    return K * 2.0 ** -24 * (wl.nx + wl.ny + wl.nz)
