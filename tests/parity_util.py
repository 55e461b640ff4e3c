"""Shared comparison rules for the GPU parity tests (reading C6)."""
import numpy as np

from oracle import sp2_oracle as O

TOL_D = 1e-3          # BASELINE north_star: max |D_gpu - D_ref| <= 1e-3
TOL_TRACE_REL = 1e-3  # |trace - N_occ| <= 1e-3 N_occ
TOL_IDEM = 1e-3       # ||D^2 - D||_F / sqrt(N) <= 1e-3


def branch_prefix_check(gpu, ref, N_occ):
    """Reading C6: on the common prefix the signs must be identical on every layer up to the first layer n*
    where the oracle's margin |d_n| is within the trace noise delta = 5e-4 max(1, N_occ).
    Returns (n_star, first_mismatch) with first_mismatch None or >= n_star."""
    delta = 5e-4 * max(1.0, N_occ)
    n_common = min(len(gpu["sigma"]), len(ref["sigma"]))
    n_star = n_common
    for n in range(n_common):
        if abs(ref["margin"][n]) <= delta:
            n_star = n
            break
    mism = None
    for n in range(n_common):
        if gpu["sigma"][n] != ref["sigma"][n]:
            mism = n
            break
    assert mism is None or mism >= n_star, (
        f"branch differs at layer {mism + 1} where the oracle margin {ref['margin'][mism]:.3e} > delta {delta:.3e}")
    return n_star, mism


def replay_check(gpu, H32, N_occ, bounds, eigs=None):
    """Reading C6 (ii): the GPU's per-layer traces must match the FP64 recursion replayed under the GPU's own
    branch sequence (scalar recursion on the eigenvalues when known, else the matrix oracle)."""
    sig = gpu["sigma"]
    if eigs is not None:
        rep = O.scalar_recursion(eigs, N_occ, bounds[0], bounds[1], forced_sigma=sig)
    else:
        _, rep = O.sp2_ref(H32, N_occ, bounds, forced_sigma=sig)
    tol = 1e-3 * max(1.0, N_occ)
    n = len(sig)
    for key in ("trace_S", "trace_X"):
        a, b = np.array(gpu[key][:n]), np.array(rep[key][:n])
        assert np.abs(a - b).max() <= tol, f"{key}: {np.abs(a - b).max()} > {tol}"
    a, b = np.array(gpu["iderr"][:n]), np.array(rep["iderr"][:n])
    assert np.abs(a - b).max() <= tol
    return rep


def acceptance(D64, Dref, N_occ):
    err = float(np.abs(D64 - Dref).max())
    tr = float(abs(np.trace(D64) - N_occ))
    idem = O.idempotency_error(D64)
    return err, tr, idem


def assert_acceptance(D64, Dref, N_occ, what=""):
    err, tr, idem = acceptance(D64, Dref, N_occ)
    assert err <= TOL_D, f"{what} max|D-Dref|={err}"
    assert tr <= TOL_TRACE_REL * max(N_occ, 1.0), f"{what} |trace-N_occ|={tr}"
    assert idem <= TOL_IDEM, f"{what} idempotency={idem}"
    assert np.array_equal(D64, D64.T), f"{what} D not exactly symmetric"
    return err, tr, idem
