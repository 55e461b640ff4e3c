"""Writes tests/golden/oracle_small_cases.json from the FP64 oracle ONLY (never the CUDA path).

    python tests/golden/make_golden.py

The inputs are the seeded generators of paper_2101_06385_b200/workloads.py (which hold none of the method's
arithmetic).  The file freezes the oracle's per-layer decisions on tiny inputs so that an accidental change of the
oracle's arithmetic is caught by tests/test_oracle_pins.py::test_golden_small_cases."""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from oracle import sp2_oracle as O  # noqa: E402
from paper_2101_06385_b200 import workloads as W  # noqa: E402

CASES = [
    ("cfg1_seed0_N16_explicit", lambda: W.config1(0, n=16), "explicit"),
    ("cfg1_seed1_N24_auto", lambda: W.config1(1, n=24), "auto"),
    ("uniform10_nocc5_auto", None, "auto"),          # shape of the paper's Fig. 2 input
    ("uniform100_nocc10_auto", None, "auto"),        # shape of the paper's Fig. 5 input
]


def build():
    out = {}
    for name, mk, mode in CASES:
        if name.startswith("uniform10_"):
            H32, nocc = W.uniform_symmetric(2, 10), 5.0
        elif name.startswith("uniform100_"):
            H32, nocc = W.uniform_symmetric(5, 100), 10.0
        else:
            w = mk()
            H32, nocc = w.H32, w.N_occ
        bounds = (-1.0, 1.0) if mode == "explicit" else None
        D, st = O.sp2_ref(H32, nocc, bounds, tol=1e-9, max_layers=100)
        out[name] = {"n": int(H32.shape[0]), "n_occ": nocc, "bounds_mode": mode,
                     "bounds": [float(b) for b in st["bounds"]], "sigma": [int(s) for s in st["sigma"]],
                     "n_layers": int(st["n_layers"]), "stop_reason": int(st["stop_reason"]),
                     "trace_S": [float(f"{x:.12e}") for x in st["trace_S"]],
                     "trace_D": float(f"{np.trace(D):.12e}"), "D00": float(f"{D[0, 0]:.12e}")}
    return out


def build_next_rows():
    """Frozen values of the next-row oracles (refine_ref / energy_ref / iderr_ref, generalized_mix_ref,
    sp2_accelerated_ref) on tiny seeded inputs."""
    r = lambda x: float(f"{x:.12e}")
    out = {}
    w = W.config1(0, n=16)
    S, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=0.0, max_layers=8)
    for sg in (1, -1):
        D = O.refine_ref(S, sg)
        out[f"refine_cfg1_N16_8layers_sigma{sg:+d}"] = {
            "iderr_in": r(O.iderr_ref(S)), "iderr_out": r(O.iderr_ref(D)), "D00": r(D[0, 0]), "D10": r(D[1, 0]),
            "energy_in": r(O.energy_ref(S, w.H32)), "energy_out": r(O.energy_ref(D, w.H32))}
    rng = np.random.default_rng(3)
    theta = np.column_stack([rng.normal(0.8, 0.3, 5), rng.normal(0.3, 0.3, 5), rng.normal(0, 0.05, 5)])
    c = rng.normal(0, 0.4, 6)
    F = O.generalized_mix_ref(w.H32, theta, c, w.bounds)
    out["mix_cfg1_N16_L5"] = {"F00": r(F[0, 0]), "F10": r(F[1, 0]), "trace_F": r(np.trace(F)),
                              "fermi_beta40_at_0p4": r(float(O.fermi_function(0.4, 40.0)))}
    w = W.config1(1, n=24)
    e = np.sort(w.eps)
    no = int(w.N_occ)
    D, st = O.sp2_accelerated_ref(w.H32, w.N_occ, w.bounds, e[no - 1], e[no], tol=1e-9, max_layers=100)
    out["accelerated_cfg1_seed1_N24"] = {"sigma": [int(s) for s in st["sigma"]], "n_layers": [int(st["n_layers"])],
                                         "theta_layer1": [r(x) for x in st["theta"][0]],
                                         "theta_layer2": [r(x) for x in st["theta"][1]],
                                         "trace_S": [r(x) for x in st["trace_S"]], "D00": r(D[0, 0])}
    return out


if __name__ == "__main__":
    for name, fn in (("oracle_small_cases.json", build), ("oracle_next_rows.json", build_next_rows)):
        path = os.path.join(HERE, name)
        with open(path, "w") as f:
            json.dump(fn(), f, indent=1, sort_keys=True)
        print("wrote", path)
