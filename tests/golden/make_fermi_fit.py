"""Writes tests/golden/fermi_fit_beta40_L11.json: coefficients (theta, c) of the generalized SP2 network of Eqs. 17-18
 fitted to the Fermi function of Eq. 20 at beta = 40 with 11 layers -- the workload of the paper's
Fig. 6 -- by Levenberg-Marquardt on a uniform grid with unit weights (Eq. 19).

Harness only: the trainer is not part of the library.  This script calls scipy's least_squares and
`oracle/` (fermi_function for the target, generalized_mix_ref to confirm that the scalar network below is the oracle's
network); it never touches the CUDA path.  The paper prints no coefficients (Fig. 6 is an image), so the stored values
are this fit's, not the paper's; what the paper fixes is the model (Eqs. 17-18), the target (Eq. 20), the loss (Eq. 19),
the optimiser (LM), beta = 40 and 11 layers.

    python tests/golden/make_fermi_fit.py          # ~1 minute on the host cores
"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import sp2_oracle as O  # noqa: E402

BETA, L, GRID = 40.0, 11, 2001
OUT = os.path.join(HERE, "fermi_fit_beta40_L11.json")


def network(theta, c, eps):
    """Eqs. 17-18 as printed: eps_0 = eps, eps_n = th1 eps^2 + th2 eps + th3, F~ = 1 - sum_i c_i eps_i."""
    e = np.asarray(eps, dtype=np.float64)
    acc = c[0] * e
    for k in range(len(theta)):
        e = theta[k][0] * e * e + theta[k][1] * e + theta[k][2]
        acc = acc + c[k + 1] * e
    return 1.0 - acc


def fit():
    from scipy.optimize import least_squares

    x = np.linspace(0.0, 1.0, GRID)
    target = O.fermi_function(x, BETA)

    def residual(p):
        return network(p[: 3 * L].reshape(L, 3), p[3 * L:], x) - target

    best = None
    for seed in range(4):
        # start: the truncated SP2 expansion itself (alternating 2x - x^2, x^2; output = last layer), jittered
        rng = np.random.default_rng(seed)
        theta0 = np.array([(1.0, 0.0, 0.0) if k % 2 else (-1.0, 2.0, 0.0) for k in range(L)])
        theta0 = theta0 + (rng.normal(0.0, 0.02, (L, 3)) if seed else 0.0)
        c0 = np.zeros(L + 1)
        c0[-1] = 1.0
        with np.errstate(over="ignore", invalid="ignore"):
            r = least_squares(residual, np.concatenate([theta0.ravel(), c0]), method="lm", xtol=1e-15, ftol=1e-15,
                              gtol=1e-15, max_nfev=20000)
        err = float(np.abs(r.fun).max())
        print(f"seed {seed}: max error {err:.3e}, rms {np.sqrt(np.mean(r.fun ** 2)):.3e}, {r.nfev} evaluations")
        if best is None or err < best[0]:
            best = (err, r.x.copy(), seed)
    return best


def main():
    import scipy

    err, p, seed = fit()
    theta, c = p[: 3 * L].reshape(L, 3), p[3 * L:]
    x = np.linspace(0.0, 1.0, GRID)
    fine = np.linspace(0.0, 1.0, 20 * (GRID - 1) + 1)
    err_fine = float(np.abs(network(theta, c, fine) - O.fermi_function(fine, BETA)).max())
    # the scalar network above is the oracle's matrix network on a diagonal H with bounds (0, 1)
    pts = np.linspace(0.0, 1.0, 64)
    Fm = O.generalized_mix_ref(np.diag(pts).astype(np.float32), theta, c, bounds=(0.0, 1.0))
    assert np.abs(np.diag(Fm) - network(theta, c, pts.astype(np.float32).astype(np.float64))).max() < 1e-12
    e, lo, hi = x, 0.0, 1.0
    for k in range(L):
        e = theta[k, 0] * e * e + theta[k, 1] * e + theta[k, 2]
        lo, hi = min(lo, float(e.min())), max(hi, float(e.max()))
    out = {"what": "generalized SP2 network (Eqs. 17-18, P:240-252) fitted to Eq. 20 (P:267) by LM on Eq. 19's loss; "
                   "the paper prints no coefficients (Fig. 6, P:254, is an image): these are this fit's",
           "written_by": "tests/golden/make_fermi_fit.py", "scipy": scipy.__version__, "beta": BETA, "layers": L,
           "grid_points": GRID, "start_seed": seed, "max_error_on_grid": err, "max_error_fine_grid": err_fine,
           "rms_error_on_grid": float(np.sqrt(np.mean((network(theta, c, x) - O.fermi_function(x, BETA)) ** 2))),
           "range_of_intermediate_values": [lo, hi],
           "theta": [[float(v) for v in row] for row in theta], "c": [float(v) for v in c]}
    with open(OUT, "w") as f:
        json.dump(out, f, indent=1)
    print(f"wrote {OUT}: max error {err:.3e} on the grid, {err_fine:.3e} on a 20x finer grid, intermediate values in "
          f"[{lo:.3f}, {hi:.3f}]")


if __name__ == "__main__":
    main()
