"""Pins of the NEXT-3 oracle (accelerated_layer, sp2_accelerated_ref): section V.A, reading C27.

The paper's explicit W_n, B_n are only in its supplementary material (not available): "parity unpinned" against the
paper's own formulas.  What the text does fix, and what is checked here:
  * each layer is a generalized projection X -> f(W X + B) with real weights: the two maps are exactly the SP2
    polynomials composed with an affine map, so on the eigenvalues they are scalar quadratics (checked in a plain loop);
  * "highest slope ... around the HOMO or LUMO eigenvalues, but without risking switching places": the chosen a
    is the LARGEST for which no unoccupied value overtakes an occupied one -- a slightly larger a must break the order;
  * "shift and re-scale the eigenvalue spectrum to [0, 1]": every eigenvalue stays in [0, 1];
  * a = 1 gives back x^2 / 2x - x^2, i.e. plain Alg. 1;
  * the result is the same D (closed form Q_occ Q_occ^T), reached in clearly fewer layers -- Fig. 5's example went from
    28 to 17 layers for N = 100, N_occ = 10; its matrix is unspecified, so this is checked as a ratio on an
    input of that shape.
"""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W


def test_layer_polynomials_fixed_points_range_and_standard_limit():
    x = np.linspace(0, 1, 1001)
    for h, l in [(0.6, 0.4), (0.9, 0.05), (0.51, 0.49), (1.0, 0.0)]:
        for sigma_force, tr in ((1, 0.0), (-1, 1e9)):
            # force the branch through N_occ: a huge N_occ makes the occupation-raising branch B win
            sigma, th, h2, l2, _ = O.accelerated_layer(N_S=50.0, N_X=40.0, n_dim=100, N_occ=tr, h=h, l=l)
            assert sigma == sigma_force
            p = th[0] * x * x + th[1] * x + th[2]
            assert p.min() >= -1e-15 and p.max() <= 1 + 1e-15          # spectrum stays in [0, 1]
            occ, un = p[x >= h], p[x <= l]
            assert un.max() <= occ.min() + 1e-12                        # no switching of places
            assert abs(h2 - occ.min()) < 1e-5 and abs(l2 - un.max()) < 1e-5   # the tracked bounds are the images
            if sigma > 0:
                assert abs(p[-1] - 1) < 1e-15
            else:
                assert abs(p[0]) < 1e-15
            if (h, l) == (1.0, 0.0):
                want = x * x if sigma > 0 else 2 * x - x * x
                assert np.abs(p - want).max() < 1e-15                   # plain SP2


def test_a_is_the_largest_admissible():
    h, l = 0.7, 0.3
    x = np.linspace(0, 1, 2001)
    aA, aB = 2 / (2 - l), 2 / (1 + h)
    for eps in (1e-3, 1e-2):
        a = aA + eps
        p = (a * x + 1 - a) ** 2
        # a larger a leaves the hole side worse than the optimum: max over [0, l] grows
        assert p[x <= l].max() > ((aA * x + 1 - aA) ** 2)[x <= l].max()
        a = aB + eps
        q = 2 * a * x - (a * x) ** 2
        assert q[x >= h].min() < (2 * aB * x - (aB * x) ** 2)[x >= h].min()
    # and the slope at the eigenvalue being separated is larger than plain SP2's
    assert 2 * aA * (aA * h + 1 - aA) > 2 * h
    assert 2 * aB - 2 * aB * aB * l > 2 - 2 * l


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_accelerated_reaches_the_same_density_in_fewer_layers(seed):
    w = W.config1(seed)
    nocc = int(w.N_occ)
    homo, lumo = np.sort(w.eps)[nocc - 1], np.sort(w.eps)[nocc]
    D0, s0 = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
    # estimates 1 % inside the gap on each side (valid bounds: homo_est >= homo, lumo_est <= lumo)
    g = lumo - homo
    D1, s1 = O.sp2_accelerated_ref(w.H32, w.N_occ, w.bounds, homo + 0.01 * g, lumo - 0.01 * g, tol=w.tol,
                                   max_layers=w.max_layers, keep_history=True)
    Dstar = w.Q[:, :nocc] @ w.Q[:, :nocc].T
    assert np.abs(D1 - Dstar).max() < 1e-6 and abs(np.trace(D1) - nocc) < 1e-6
    assert O.idempotency_error(D1) < 1e-7
    assert s1["n_layers"] <= 0.8 * s0["n_layers"]
    # matrix recursion = scalar recursion on the eigenvalues, every layer; order and range preserved throughout
    e0, e1 = w.bounds
    ev = (e1 - np.linalg.eigvalsh(O.symmetrize_lower(w.H32))) / (e1 - e0)       # eigenvalues of S_0 (descending in energy)
    occ = ev >= np.sort(ev)[::-1][nocc - 1]
    for k, th in enumerate(s1["theta"]):
        ev = th[0] * ev * ev + th[1] * ev + th[2]
        assert ev.min() >= -1e-12 and ev.max() <= 1 + 1e-12
        assert ev[occ].min() > ev[~occ].max()
        assert ev[occ].min() >= s1["h"][k] - 1e-9 and ev[~occ].max() <= s1["l"][k] + 1e-9
        assert abs(ev.sum() - s1["trace_S"][k]) < 1e-9
        assert np.abs(np.sort(ev) - np.linalg.eigvalsh(s1["S_hist"][k])).max() < 1e-9


def test_fig5_shaped_example_layer_ratio():
    # Fig. 5: H in R^{100x100}, N_occ = 10: 28 layers without, 17 with acceleration (ratio 0.61).  The matrix is
    # unspecified; on a uniformly random symmetric H of that shape the ratio must be of that order.
    H = W.uniform_symmetric(4, 100)
    ev = np.linalg.eigvalsh(O.symmetrize_lower(H))
    homo, lumo = ev[9], ev[10]
    b = O.gershgorin_bounds(O.symmetrize_lower(H))
    _, s0 = O.sp2_ref(H, 10, b, tol=1e-9, max_layers=200)
    _, s1 = O.sp2_accelerated_ref(H, 10, b, homo, lumo, tol=1e-9, max_layers=200)
    ratio = s1["n_layers"] / s0["n_layers"]
    print(f"Fig.5-shaped: {s0['n_layers']} -> {s1['n_layers']} layers (ratio {ratio:.2f}; paper: 28 -> 17, 0.61)")
    assert 0.4 <= ratio <= 0.8


def test_invalid_estimates_are_rejected():
    w = W.config1(0)
    with pytest.raises(ValueError):
        O.sp2_accelerated_ref(w.H32, w.N_occ, w.bounds, 0.1, -0.1)
