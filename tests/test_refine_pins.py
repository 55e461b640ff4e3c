"""Pins of the NEXT-1 oracle functions (refine_ref, energy_ref, iderr_ref): Eq. 16.

What fixes them independently of the oracle's own code:
  * on the eigenvalues, f_final is the scalar polynomial 2x^2 - x^4 or (2x - x^2)^2 (H = Q diag Q^T, so
    f(S) = Q diag(f(s)) Q^T): checked through the eigenbasis, not by re-typing the matrix formula;
  * both polynomials have f(0) = 0, f(1) = 1, f'(0) = f'(1) = 0 (second-order convergence), so the
    idempotency error must at least square: IdErr(f(S)) <= C IdErr(S)^2 with Theorem 1's C;
  * the energy of the exact density matrix of H = Q diag(eps) Q^T is the sum of the occupied eigenvalues
    (Eqs. 3-6), and Tr[D H] is variational: any idempotent D of the right trace gives E >= E*.
"""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W

C_THM1 = (71.0 + 17.0 * np.sqrt(17.0)) / 32.0


def _partially_converged(w, layers_short=2):
    """S_n of the FP64 oracle stopped a few layers before convergence, and the sign of its last layer."""
    _, full = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
    n = full["n_layers"] - layers_short
    S, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=0.0, max_layers=n)
    return S, int(st["sigma"][-1])


@pytest.mark.parametrize("last_sigma", [1, -1])
def test_refine_is_the_scalar_polynomial_on_the_eigenvalues(last_sigma):
    rng = np.random.default_rng(5)
    Q = W.haar_orthogonal(rng, 48)
    s = rng.uniform(0.0, 1.0, 48)
    S = (Q * s) @ Q.T
    got = O.refine_ref(S, last_sigma)
    f = 2 * s**2 - s**4 if last_sigma < 0 else (2 * s - s**2) ** 2
    assert np.abs(got - (Q * f) @ Q.T).max() < 1e-13
    # the two forms are mirror images under x -> 1 - x (particle-hole symmetry of the SP2 pair)
    other = O.refine_ref(np.eye(48) - S, -last_sigma)
    assert np.abs((np.eye(48) - other) - got).max() < 1e-13


def test_refine_polynomials_fix_0_and_1_to_second_order():
    x = np.array([0.0, 1.0])
    h = 1e-4
    for last_sigma in (1, -1):
        f = lambda t: O.refine_ref(np.diag(np.atleast_1d(t)), last_sigma).diagonal()
        assert np.allclose(f(x), x, atol=0)
        # derivative vanishes at both fixed points: |f(x +- h) - f(x)| = O(h^2)
        assert np.abs(f(np.array([h]))[0]) < 5 * h * h
        assert np.abs(f(np.array([1 - h]))[0] - 1.0) < 5 * h * h


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_refinement_squares_the_idempotency_error(seed):
    w = W.config1(seed)
    S, last_sigma = _partially_converged(w)
    e0 = O.iderr_ref(S)
    D = O.refine_ref(S, last_sigma)
    e1 = O.iderr_ref(D)
    assert e0 > 1e-9                                  # genuinely unconverged input
    assert 0.0 <= e1 <= C_THM1 * e0 * e0 + 1e-13      # Theorem 1 with the continued alternation
    assert abs(np.trace(D) - w.N_occ) < abs(np.trace(S) - w.N_occ) + 1e-12
    # the wrong continuation (same sign twice) is still a contraction but must not beat the alternating one by
    # orders of magnitude; what matters: the reading C15 choice meets the theorem's bound
    Dstar = (w.Q[:, : int(w.N_occ)]) @ (w.Q[:, : int(w.N_occ)]).T
    assert np.abs(D - Dstar).max() < np.abs(S - Dstar).max()


def test_iderr_and_energy_definitions():
    rng = np.random.default_rng(9)
    A = rng.standard_normal((20, 20)); X = (A + A.T) / 2
    B = rng.standard_normal((20, 20)); H = (B + B.T) / 2
    # brute force double loops
    tr_xh = sum(X[i, k] * H[k, i] for i in range(20) for k in range(20))
    tr_x_x2 = sum(X[i, i] for i in range(20)) - sum(X[i, k] * X[k, i] for i in range(20) for k in range(20))
    assert abs(O.energy_ref(X, H) - tr_xh) < 1e-12
    assert abs(O.iderr_ref(X) - tr_x_x2) < 1e-12
    # only H's lower triangle is read (reading C22)
    H2 = H.copy(); H2[np.triu_indices(20, 1)] = 7.0
    assert abs(O.energy_ref(X, H2) - tr_xh) < 1e-12


@pytest.mark.parametrize("seed", [0, 1])
def test_energy_of_converged_density_is_sum_of_occupied_eigenvalues(seed):
    w = W.config1(seed)
    D, _ = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
    E_star = float(np.sort(w.eps)[: int(w.N_occ)].sum())
    # H32 is the FP32 rounding of Q diag(eps) Q^T: eigenvalues move by ~1e-8 each
    assert abs(O.energy_ref(D, w.H32) - E_star) < 1e-5
    S, last_sigma = _partially_converged(w, 3)
    E0 = O.energy_ref(S, w.H32)
    E1 = O.energy_ref(O.refine_ref(S, last_sigma), w.H32)
    assert abs(E1 - E_star) < abs(E0 - E_star)        # "rapid improvement ... in the last layer"
