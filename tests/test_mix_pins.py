"""Pins of the NEXT-2 oracle (generalized_mix_ref, fermi_function): Eqs. 17-20.

Independent of the oracle's own matrix code:
  * on H = Q diag(eps) Q^T the network acts on each eigenvalue: F~(H) = Q diag(1 - sum_i c_i e_i) Q^T with the SCALAR
    recursion e_0 = eps, e_n = th1 e^2 + th2 e + th3 (Eq. 17 as printed), evaluated in a plain Python loop;
  * special weight vectors reduce it to known things: c = (1, 0, ...) gives I - E_0, whose eigenvalues are the
    rescaled energies reversed; c = (0, ..., 0, 1) with the SP2 polynomials gives I - (the reversed projector), i.e.
    the zero-temperature density matrix of Eq. 3 -- the "folding" of P:246;
  * a truncated SP2 network is a smooth, monotonically decreasing approximation of a step at eps = 1/2, as the
    Fermi function of Eq. 20 is: F(0) ~ 1, F(1/2) = 1/2 exactly, F(1) ~ 0, F(eps) + F(1 - eps) = 1.
"""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W


def _scalar_net(eps, theta, c):
    out = []
    for e in eps:
        acc = c[0] * e
        for k in range(len(theta)):
            e = theta[k][0] * e * e + theta[k][1] * e + theta[k][2]
            acc += c[k + 1] * e
        out.append(1.0 - acc)
    return np.array(out)


@pytest.mark.parametrize("seed", [0, 1])
def test_mix_equals_scalar_network_on_eigenvalues(seed):
    rng = np.random.default_rng(seed)
    n, L = 40, 7
    Q = W.haar_orthogonal(rng, n)
    lam = rng.uniform(-1, 1, n)
    H32 = ((Q * lam) @ Q.T).astype(np.float32)
    theta = np.column_stack([rng.normal(0.8, 0.3, L), rng.normal(0.3, 0.3, L), rng.normal(0, 0.05, L)])
    c = rng.normal(0, 0.4, L + 1)
    F = O.generalized_mix_ref(H32, theta, c, bounds=(-1.5, 2.0))
    lam32 = np.linalg.eigvalsh(O.symmetrize_lower(H32))          # eigenvalues of the FP32-rounded input
    want = np.sort(_scalar_net((lam32 + 1.5) / 3.5, theta, c))
    assert np.abs(np.sort(np.linalg.eigvalsh((F + F.T) / 2)) - want).max() < 1e-10
    # and in the known eigenbasis (rounding of H to FP32 moves it by ~1e-7)
    Fq = (Q * _scalar_net((lam + 1.5) / 3.5, theta, c)) @ Q.T
    assert np.abs(F - Fq).max() < 2e-5


def test_special_weight_vectors_and_folding():
    w = W.config1(0)
    e0, e1 = w.bounds
    L = 24
    # the SP2 polynomials in the natural variable: x^2 sends eps -> 0, 2x - x^2 sends eps -> 1.  Use the oracle's own
    # sigma sequence of the reversed problem: a layer S -> S^2 (sigma = +1) is E -> 2E - E^2 on E = 1 - S, and vice versa.
    _, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=L)
    L = st["n_layers"]
    theta = np.array([(-1.0, 2.0, 0.0) if s > 0 else (1.0, 0.0, 0.0) for s in st["sigma"]])
    c = np.zeros(L + 1); c[0] = 1.0
    F0 = O.generalized_mix_ref(w.H32, theta, c, w.bounds)
    H = O.symmetrize_lower(w.H32)
    assert np.abs(F0 - (np.eye(w.N) - (H - e0 * np.eye(w.N)) / (e1 - e0))).max() < 1e-14
    c = np.zeros(L + 1); c[-1] = 1.0
    FL = O.generalized_mix_ref(w.H32, theta, c, w.bounds)
    Dstar = w.Q[:, : int(w.N_occ)] @ w.Q[:, : int(w.N_occ)].T
    assert np.abs(FL - Dstar).max() < 1e-6                        # zero-temperature limit = Eq. 3's D
    D, _ = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=L)
    assert np.abs(FL - D).max() < 1e-10                           # same recursion written on E = I - S


def test_fermi_function_eq20():
    b = 40.0
    assert O.fermi_function(0.5, b) == 0.5
    x = np.linspace(0, 1, 101)
    f = O.fermi_function(x, b)
    assert np.all(np.diff(f) < 0) and abs(f[0] - 1) < 1e-8 and f[-1] < 1e-8
    assert np.abs(f + O.fermi_function(1 - x, b) - 1).max() < 1e-15
    # slope at the chemical potential: dF/deps = -beta/4
    h = 1e-6
    assert abs((O.fermi_function(0.5 + h, b) - O.fermi_function(0.5 - h, b)) / (2 * h) + b / 4) < 1e-6


def test_truncated_sp2_is_a_smooth_step_like_the_fermi_function():
    # an SP2 expansion stopped early "generates a smooth approximation to the Heaviside step function"
    L = 6
    theta = np.array([(1.0, 0.0, 0.0) if k % 2 else (-1.0, 2.0, 0.0) for k in range(L)])
    c = np.zeros(L + 1); c[-1] = 1.0
    x = np.linspace(0, 1, 201)
    f = _scalar_net(x, theta, c)
    assert np.all(np.diff(f) <= 1e-15) and f[0] == 1.0 and f[-1] == 0.0
    mid = x[np.argmin(np.abs(f - 0.5))]
    # it is closer to a Fermi function of some finite beta than to the sharp step
    best = min(np.abs(f - O.fermi_function(x - mid + 0.5, b)).max() for b in np.linspace(5, 200, 80))
    assert best < 0.5 * np.abs(f - (x < mid)).max()


def test_stored_fermi_fit_reproduces_eq20():
    """tests/golden/fermi_fit_beta40_L11.json (written by tests/golden/make_fermi_fit.py: LM fit of Eqs. 17-18 to Eq. 20,
    beta = 40, 11 layers -- the workload of Fig. 6): the stored coefficients, run through this file's own scalar
    loop and through the oracle's matrix network, give the Fermi function within the stored residual.  The paper shows
    the error curve only as an image; its text claims the accuracy of rational Pade schemes, i.e. small against
    the width 1/beta of the step -- asserted here as < 1e-3."""
    import json
    import os

    fit = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "fermi_fit_beta40_L11.json")))
    theta, c = np.array(fit["theta"]), np.array(fit["c"])
    assert theta.shape == (11, 3) and c.shape == (12,) and fit["beta"] == 40.0
    x = np.linspace(0.0, 1.0, 401)
    F = 1.0 / (np.exp(40.0 * (x - 0.5)) + 1.0)                       # Eq. 20 retyped
    got = _scalar_net(x, theta, c)
    err = np.abs(got - F).max()
    assert err <= fit["max_error_fine_grid"] * (1 + 1e-9) < 1e-3
    assert np.abs(O.fermi_function(x, 40.0) - F).max() < 1e-15
    # a monotonically decreasing step: ~1 at 0, 1/2 at 1/2, ~0 at 1
    assert abs(got[0] - 1.0) < 1e-4 and abs(got[200] - 0.5) < 1e-4 and abs(got[-1]) < 1e-4
    # the oracle's matrix network on a rotated H with spectrum x and bounds (0, 1)
    rng = np.random.default_rng(5)
    Q = W.haar_orthogonal(rng, 48)
    lam = rng.uniform(0.0, 1.0, 48)
    H32 = ((Q * lam) @ Q.T).astype(np.float32)
    Fm = O.generalized_mix_ref(H32, theta, c, bounds=(0.0, 1.0))
    lam32, V = np.linalg.eigh(O.symmetrize_lower(H32))
    ref = (V * (1.0 / (np.exp(40.0 * (lam32 - 0.5)) + 1.0))) @ V.T
    assert np.abs(Fm - ref).max() <= fit["max_error_fine_grid"] + 1e-9
