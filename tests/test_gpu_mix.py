"""GPU parity of the NEXT-2 row: sp2_generalized_mix (Eqs. 17-18) against the FP64 oracle
generalized_mix_ref and against the scalar network on the known eigenvalues."""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W

pytestmark = pytest.mark.gpu

# north_star's elementwise bar for the mixed-precision path
TOL = 1e-3


@pytest.fixture(scope="module")
def env(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    torch.cuda.set_device(0)
    h = api.Handle(4096, 0, 64)
    yield api, h, torch
    h.close()


def _fermi_like_network(L, rng, jitter=0.02):
    """Alternating SP2 polynomials in the natural variable with seeded perturbations (config 4's recipe shape:
    w = 1 + N(0, 0.02), b = N(0, 0.005)) and a full weight vector c."""
    theta = []
    for k in range(L):
        base = (1.0, 0.0) if k % 2 else (-1.0, 2.0)
        wk = 1.0 + rng.normal(0, jitter)
        theta.append((wk * base[0], wk * base[1], rng.normal(0, 0.005)))
    c = rng.normal(0, 0.05, L + 1)
    c[-1] += 1.0
    return np.array(theta), c


@pytest.mark.parametrize("n,tile,auto", [(128, 1, False), (300, 1, True), (1100, 1, False), (1024, 3, False),
                                         (2000, 3, True)])
def test_mix_matches_oracle_and_scalar_network(env, n, tile, auto):
    api, h, torch = env
    rng = np.random.default_rng(n)
    Q = W.haar_orthogonal(rng, n)
    lam = rng.uniform(-1, 1, n)
    H32 = np.ascontiguousarray(((Q * lam) @ Q.T).astype(np.float32))
    H32 = np.ascontiguousarray((H32 + H32.T) / 2)
    L = 10
    theta, c = _fermi_like_network(L, rng)
    bounds = None if auto else (-1.0, 1.0)
    opts = api.make_opts(tile_config=tile)
    Hd = torch.from_numpy(H32).cuda()
    F, info = h.generalized_mix(Hd, theta, c, bounds=bounds, opts=opts)
    F = F.cpu().numpy().astype(np.float64)
    if auto:
        bounds = h.gershgorin(Hd)
    ref = O.generalized_mix_ref(H32, theta, c, bounds)
    err = np.abs(F - ref).max()
    # scalar network (Eq. 17 as printed) on the eigenvalues, through the known eigenbasis
    e = (lam - bounds[0]) / (bounds[1] - bounds[0])
    acc = c[0] * e
    for k in range(L):
        e = theta[k, 0] * e * e + theta[k, 1] * e + theta[k, 2]
        acc = acc + c[k + 1] * e
    closed = (Q * (1.0 - acc)) @ Q.T
    print(f"mix n={n} tile={tile} auto={auto}: max|F-ref|={err:.2e} max|F-closed|={np.abs(F - closed).max():.2e}")
    assert err <= TOL and np.abs(F - closed).max() <= TOL
    assert np.array_equal(F, F.T)
    assert info["n_layers"] == L


def test_mix_special_weights_reduce_to_known_calls(env):
    api, h, torch = env
    w = W.config1(1, n=384)
    Hd = torch.from_numpy(w.H32).cuda()
    L = 6
    theta = np.array([(1.0, 0.0, 0.0) if k % 2 else (-1.0, 2.0, 0.0) for k in range(L)])
    # c = (1, 0, ..., 0): F = I - E_0 = S_0 of Alg. 1: one affine map of H, no product involved
    c = np.zeros(L + 1); c[0] = 1.0
    F, _ = h.generalized_mix(Hd, theta, c, bounds=w.bounds)
    e0, e1 = w.bounds
    S0 = (e1 * np.eye(w.N) - O.symmetrize_lower(w.H32)) / (e1 - e0)
    assert np.abs(F.cpu().numpy() - S0).max() <= 3e-7
    # c = (0, ..., 0, 1): F = I - E_L; the same network through sp2_generalized in the reversed variable gives S_L
    # with the branches swapped (x^2 <-> 2x - x^2) and F = S_L
    c = np.zeros(L + 1); c[-1] = 1.0
    F, _ = h.generalized_mix(Hd, theta, c, bounds=w.bounds)
    theta_rev = np.array([(-1.0, 2.0, 0.0) if k % 2 else (1.0, 0.0, 0.0) for k in range(L)])
    X, _ = h.generalized(Hd, theta_rev, bounds=w.bounds)
    assert np.abs(F.cpu().numpy() - X.cpu().numpy()).max() <= 5e-6
    with pytest.raises(ValueError):
        h.generalized_mix(Hd, theta, np.zeros(L), bounds=w.bounds)
    with pytest.raises(api.SP2Error):
        h.generalized_mix(Hd, theta, np.zeros(L + 1), bounds=w.bounds, opts=api.make_opts(tile_config=2))
    with pytest.raises(api.SP2Error):
        h.generalized_mix(Hd, theta, np.full(L + 1, np.nan), bounds=w.bounds)


def test_fermi_function_from_the_fitted_network(env):
    """The thing the output mix was built for (Eqs. 17-20; Fig. 6): with the LM-fitted coefficients of
    tests/golden/fermi_fit_beta40_L11.json (11 layers, beta = 40; written by tests/golden/make_fermi_fit.py from the
    oracle's definitions), sp2_generalized_mix turns H into the finite-temperature density matrix F(H).  Compared
    elementwise with the oracle's matrix network, and with the exact Q diag(F(eps)) Q^T within the fit's own residual."""
    import json
    import os

    api, h, torch = env
    fit = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "fermi_fit_beta40_L11.json")))
    theta, c = np.array(fit["theta"]), np.array(fit["c"])
    n = 1024
    rng = np.random.default_rng(2024)
    Q = W.haar_orthogonal(rng, n)
    lam = rng.uniform(0.0, 1.0, n)                       # the rescaled energies of Eq. 20: bounds (0, 1)
    lam[:64] = rng.uniform(0.45, 0.55, 64)               # ... with extra weight inside the thermal window 1/beta
    H32 = ((Q * lam) @ Q.T).astype(np.float32)
    H32 = np.ascontiguousarray((H32 + H32.T) / 2)
    for tile in (1, 3):
        F, info = h.generalized_mix(torch.from_numpy(H32).cuda(), theta, c, bounds=(0.0, 1.0),
                                    opts=api.make_opts(tile_config=tile))
        F = F.cpu().numpy().astype(np.float64)
        ref = O.generalized_mix_ref(H32, theta, c, (0.0, 1.0))
        exact = (Q * O.fermi_function(lam, fit["beta"])) @ Q.T
        e_ref, e_exact = np.abs(F - ref).max(), np.abs(F - exact).max()
        occ = float(np.trace(F))
        print(f"Fermi fit (11 layers, beta = 40) N={n} tile={tile}: max|F - oracle network| = {e_ref:.2e}, "
              f"max|F - exact Fermi matrix| = {e_exact:.2e} (fit residual {fit['max_error_fine_grid']:.2e}), "
              f"Tr F = {occ:.4f} against sum F(eps) = {O.fermi_function(lam, fit['beta']).sum():.4f}")
        assert e_ref <= 2e-5                              # measured 1.0e-6 / 1.6e-6
        assert e_exact <= fit["max_error_fine_grid"] + 2e-5   # measured 2.4e-6 / 2.8e-6 (the matrix error averages the fit's)
        assert np.array_equal(F, F.T) and info["n_layers"] == 11
        assert abs(occ - O.fermi_function(lam, fit["beta"]).sum()) <= 1e-3 * n
