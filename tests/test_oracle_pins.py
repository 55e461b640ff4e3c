"""Pins for oracle/sp2_oracle.py against what the paper and the mathematics fix (CPU only).

Each test names the passage it pins (P:n = PAPER.md line n).  None of them retypes the oracle's
own formula: they use closed forms, LAPACK, brute-force loops, invariants and analytic cases."""
import math

import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W


def _checks(H32, D, N_occ, Dstar):
    return (np.abs(D - Dstar).max(), abs(np.trace(D) - N_occ), O.idempotency_error(D),
            O.commutator_norm(H32, D) / np.linalg.norm(H32.astype(np.float64)))


@pytest.mark.parametrize("seed", [0, 1, 2])
@pytest.mark.parametrize("auto", [False, True])
def test_config1_closed_form_density(seed, auto):
    """Eq. 6: H = Q diag(eps) Q^T by construction, so D* = Q_occ Q_occ^T with no eigensolver.
    BASELINE north_star's four checks: D vs D*, trace, idempotency, commutator."""
    w = W.config1(seed)
    D, st = O.sp2_ref(w.H32, w.N_occ, None if auto else w.bounds, tol=w.tol, max_layers=w.max_layers)
    err, tr, idem, comm = _checks(w.H32, D, w.N_occ, O.closed_form_density(w.Q, w.N_occ))
    assert err < 1e-6 and tr < 1e-6 and idem < 1e-8 and comm < 1e-8
    assert st["stop_reason"] in (O.STOP_TOL, O.STOP_IDERR_NONPOS, O.STOP_PARAM_FREE)
    assert st["n_layers"] < (45 if auto else 30)


def test_eig_density_agrees_with_closed_form_and_lapack():
    """Eqs. 3-6: the LAPACK route and the constructed projector coincide."""
    w = W.config1(3)
    De, E = O.eig_density(w.H32, w.N_occ)
    assert np.abs(De - O.closed_form_density(w.Q, w.N_occ)).max() < 1e-6
    assert np.abs(np.sort(w.eps) - E).max() < 1e-6
    r = np.array([0, 5, 77]); c = np.array([3, 5, 120])
    assert np.allclose(O.closed_form_density_entries(w.Q, w.N_occ, r, c), De[r, c], atol=1e-6)


def test_small_tight_binding_vs_eigh():
    """Config-2 recipe at 64 sites (N=256): D from SP2 equals the eigenprojector (gap permitting)."""
    w = W.config2(0, n_sites=64)
    De, E = O.eig_density(w.H32, w.N_occ)
    k = int(w.N_occ)
    gap = E[k] - E[k - 1]
    D, st = O.sp2_ref(w.H32, w.N_occ, None, tol=1e-9, max_layers=200)
    assert gap > 0
    assert np.abs(D - De).max() < 1e-9
    assert abs(np.trace(D) - w.N_occ) < 1e-6


@pytest.mark.parametrize("seed", [0, 1])
def test_matrix_oracle_equals_scalar_recursion(seed):
    """Proof of Thm 1: eigenvalues of S_n follow the scalar map, so every per-layer
    N_S, N_X, IdErr_n, sigma_n, the stop layer and reason come from an O(N L) loop on eps."""
    w = W.config1(seed)
    for bounds in [w.bounds, (-7.0, 6.5)]:
        D, st = O.sp2_ref(w.H32, w.N_occ, bounds, tol=w.tol, max_layers=w.max_layers)
        sc = O.scalar_recursion(np.linalg.eigvalsh(O.symmetrize_lower(w.H32)), w.N_occ, *bounds, tol=w.tol,
                                max_layers=w.max_layers)
        assert st["sigma"] == sc["sigma"] and st["n_layers"] == sc["n_layers"]
        assert st["stop_reason"] == sc["stop_reason"]
        for key in ("trace_S", "trace_X", "iderr"):
            assert np.allclose(st[key], sc[key], rtol=0, atol=1e-9)
        assert np.allclose(np.sort(np.linalg.eigvalsh(D)), np.sort(sc["lam"]), atol=1e-9)


def test_forced_sigma_replay():
    """Reading C6: replaying a branch sequence reproduces the same run; flipping one sign changes it."""
    w = W.config1(0)
    D, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol)
    D2, st2 = O.sp2_ref(w.H32, w.N_occ, w.bounds, forced_sigma=st["sigma"])
    assert np.array_equal(D, D2) and st2["n_layers"] == st["n_layers"]
    sc = O.scalar_recursion(w.eps, w.N_occ, *w.bounds, forced_sigma=[1] * 6)
    assert np.allclose(sc["lam"], O.scalar_initial(w.eps, *w.bounds) ** 64)   # six squarings: x^(2^6)


def test_polynomial_order_doubles():
    """the expansion order doubles per recursion (30 steps -> order 2^30)."""
    lam = O.scalar_recursion(np.array([0.3]), 0.0, 0.0, 1.0, forced_sigma=[1] * 30)["lam"]
    assert math.isclose(lam[0], (1 - 0.3) ** (2 ** 30), rel_tol=1e-6, abs_tol=1e-300)
    # 2x - x^2 branch: 1 - (1-x)^2 per step
    lam = O.scalar_recursion(np.array([0.3]), 1.0, 0.0, 1.0, forced_sigma=[-1] * 5)["lam"]
    assert math.isclose(lam[0], 1 - (1 - 0.7) ** 32, rel_tol=1e-12)


def test_theorem1_constant():
    """P:292, Eqs. 22-23: both maxima equal C = (71 + 17 sqrt 17)/32 ~ 4.41."""
    lam = np.linspace(1e-6, 1 - 1e-6, 2_000_001)
    g = lam - lam * lam
    a = 2 * lam - lam * lam
    b = 2 * lam * lam - lam ** 4
    m22 = ((a * a - a ** 4) / (g * g)).max()
    m23 = ((b - b * b) / (g * g)).max()
    assert abs(m22 - O.THEOREM1_C) < 1e-8 and abs(m23 - O.THEOREM1_C) < 1e-8
    assert abs(O.THEOREM1_C - 4.41) < 5e-3


@pytest.mark.parametrize("seed", range(4))
def test_theorem1_inequality_on_oracle_sequence(seed):
    """Thm 1 with Alg. 1's indices: whenever sigma_{n-1} != sigma_{n-2},
    IdErr_n <= C IdErr_{n-2}^2 in (near-)exact arithmetic.  A wrong index convention fails this."""
    w = W.config1(seed)
    _, st = O.sp2_ref(w.H32, w.N_occ, (-3.0, 2.5), tol=1e-7, max_layers=80)
    ide, sg = [None] + st["iderr"], [0] + st["sigma"]
    checked = 0
    for n in range(3, st["n_layers"] + 1):
        if sg[n - 1] != sg[n - 2] and ide[n - 2] > 1e-6:
            assert ide[n] <= O.THEOREM1_C * ide[n - 2] ** 2 * (1 + 1e-9) + 1e-12
            checked += 1
    assert checked >= 3


def test_norm_sandwich():
    """||X - X^2||_2 <= Tr[X - X^2] <= N ||X - X^2||_2 for eigenvalues in [0,1]."""
    w = W.config1(0)
    _, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=0.0, max_layers=12, keep_history=True)
    for S in st["S_hist"]:
        R = S - S @ S
        n2 = np.linalg.norm(R, 2)
        tr = np.trace(R)
        assert n2 <= tr * (1 + 1e-10) + 1e-13 and tr <= S.shape[0] * n2 * (1 + 1e-10) + 1e-13


def test_iderr_is_trace_of_S_minus_S2():
    """IdErr_n = Tr[S_{n-1} - S_{n-1}^2]; brute-force triple-loop square on a tiny matrix."""
    H = W.uniform_symmetric(0, 10)                       # Fig. 2's shape
    _, st = O.sp2_ref(H, 5, None, max_layers=6, keep_history=True)
    e0, e1 = st["bounds"]
    S = [(e1 * np.eye(10) - O.symmetrize_lower(H)) / (e1 - e0)] + st["S_hist"]
    for n in range(1, 7):
        P = S[n - 1]
        X = np.zeros((10, 10))
        for i in range(10):
            for j in range(10):
                for k in range(10):
                    X[i, j] += P[i, k] * P[k, j]
        assert abs(st["iderr"][n - 1] - (np.trace(P) - np.trace(X))) < 1e-12
        assert abs(st["trace_X"][n - 1] - np.trace(X)) < 1e-12
        expect = X if st["sigma"][n - 1] == 1 else 2 * P - X          # Eq. 10
        assert np.abs(S[n] - expect).max() < 1e-13


def test_sign_minimises_occupation_error():
    """sigma_n is the sign alternative with the smaller |Tr[S_n] - N_occ|."""
    w = W.config1(1)
    _, st = O.sp2_ref(w.H32, w.N_occ, (-2.0, 3.0), max_layers=15)
    sc_eigs = np.linalg.eigvalsh(O.symmetrize_lower(w.H32))
    lam = O.scalar_initial(sc_eigs, -2.0, 3.0)
    for n in range(st["n_layers"]):
        plus, minus = (lam ** 2).sum(), (2 * lam - lam ** 2).sum()
        best = 1 if abs(plus - w.N_occ) < abs(minus - w.N_occ) else -1
        if abs(abs(plus - w.N_occ) - abs(minus - w.N_occ)) > 1e-9:
            assert st["sigma"][n] == best
        lam = lam ** 2 if st["sigma"][n] == 1 else 2 * lam - lam ** 2


def test_initial_layer_reverses_and_rescales():
    """S_0 has H's eigenvalues in reverse order inside [0,1]."""
    H = np.diag([-2.0, 0.0, 6.0]).astype(np.float32)
    S0 = O.initial_layer(O.symmetrize_lower(H), -2.0, 6.0)
    assert np.allclose(np.diag(S0), [1.0, 0.75, 0.0])


def test_gershgorin():
    """Textbook Gershgorin: encloses eigvalsh; exact on diagonal matrices; hand example."""
    assert O.gershgorin_bounds(np.diag([3.0, -1.0, 2.0])) == (-1.0, 3.0)
    A = np.array([[2.0, -1.0, 0.5], [-1.0, 0.0, 0.25], [0.5, 0.25, -3.0]])
    assert O.gershgorin_bounds(A) == (-3.75, 3.5)
    for seed in range(3):
        H = O.symmetrize_lower(W.uniform_symmetric(seed, 40))
        lo, hi = O.gershgorin_bounds(H)
        E = np.linalg.eigvalsh(H)
        assert lo <= E[0] and E[-1] <= hi


def test_diagonal_hamiltonian_and_extreme_occupations():
    """Diagonal H: the matrix recursion is the scalar recursion and D is a 0/1 diagonal;
    N_occ = 0 and N_occ = N give D = 0 and D = I (reading C18)."""
    eps = np.array([-1.0, -0.6, -0.2, 0.3, 0.5, 0.9])
    H = np.diag(eps).astype(np.float32)
    D, st = O.sp2_ref(H, 3, (-1.5, 1.5), tol=1e-12)
    assert np.allclose(D, np.diag([1, 1, 1, 0, 0, 0]), atol=1e-9)
    D0, _ = O.sp2_ref(H, 0, (-1.5, 1.5), tol=1e-12)
    D6, _ = O.sp2_ref(H, 6, (-1.5, 1.5), tol=1e-12)
    assert np.allclose(D0, 0, atol=1e-9) and np.allclose(D6, np.eye(6), atol=1e-9)


def test_two_by_two_analytic_and_tie_rule():
    """N=2 analytic: H = [[0,t],[t,0]] has eigenvalues -t,+t; with N_occ=1 the projector on (1,-1)/sqrt2.
    Spectrum symmetric about the band centre with N_occ = N/2 makes the Sign argument exactly 0 at
    layer 1 (reading C4): tie -> +1 at n=1, then alternate."""
    t = 0.5
    H = np.array([[0.0, t], [t, 0.0]], dtype=np.float32)
    D, st = O.sp2_ref(H, 1, (-1.0, 1.0), tol=1e-13, max_layers=100)
    assert st["margin"][0] == 0.0 and st["sigma"][0] == 1
    assert np.allclose(D, 0.5 * np.array([[1, -1], [-1, 1]]), atol=1e-9)
    # a tie at a later layer alternates: sigma_prev = +1 and d = 0 -> -1
    assert O._sign_rule(1.0, 1.0, 1.0, 1, 0.0) == (-1, 0.0)
    assert O._sign_rule(1.0, 1.0, 1.0, -1, 0.0) == (1, 0.0)
    # eps_alt > 0 biases toward alternation
    assert O._sign_rule(1.0, 1.0, 1.0, 1, 1e-3)[0] == -1 and O._sign_rule(1.0, 1.0, 1.0, -1, 1e-3)[0] == 1


def test_one_by_one():
    H = np.array([[0.3]], dtype=np.float32)
    D, _ = O.sp2_ref(H, 1, (-1.0, 1.0), tol=1e-14, max_layers=100)
    assert abs(D[0, 0] - 1.0) < 1e-9
    with pytest.raises(ValueError):
        O.sp2_ref(H, 1, None)                            # Gershgorin of a 1x1 is degenerate


def test_stop_reasons():
    w = W.config1(0)
    _, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=1e-5, max_layers=60)
    assert st["stop_reason"] == O.STOP_TOL and st["iderr"][-1] <= 1e-5 < st["iderr"][-2]
    _, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=1e-5, max_layers=5)
    assert st["stop_reason"] == O.STOP_MAX_LAYERS and st["n_layers"] == 5
    _, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=0.0, max_layers=200)     # paper's rule alone
    assert st["stop_reason"] in (O.STOP_IDERR_NONPOS, O.STOP_PARAM_FREE) and st["n_layers"] < 40


def test_generalized_equals_scalar_polynomial():
    """Eq. 17 / P:218: X_L = Q diag(p(eps)) Q^T with p from the scalar recursion."""
    w = W.config4(0, n=96, layers=30)
    eigs = np.linalg.eigvalsh(O.symmetrize_lower(w.H32))
    sig = O.scalar_recursion(eigs, w.N_occ, *w.bounds, max_layers=30)["sigma"]
    sig = (sig + [1, -1] * 30)[:30]
    theta = O.theta_from_wb(w.extra["weights"], w.extra["biases"], sig)
    X, st = O.sp2_generalized_ref(w.H32, theta, w.bounds)
    p = O.scalar_generalized(w.eps, theta, *w.bounds)
    assert np.abs(X - (w.Q * p) @ w.Q.T).max() < 1e-7
    assert abs(st["trace_S"][-1] - p.sum()) < 1e-7
    # theta = (sigma, 1 - sigma, 0) is plain SP2 (Eq. 10)
    th = O.theta_from_wb(np.ones(8), np.zeros(8), sig[:8])
    X8, _ = O.sp2_generalized_ref(w.H32, th, w.bounds)
    D8, _ = O.sp2_ref(w.H32, w.N_occ, w.bounds, forced_sigma=sig[:8])
    assert np.abs(X8 - D8).max() < 1e-13
    # hand-worked scalar: eps = 0 -> lambda_0 = 0.5 ; theta = (2, -1, 0.25) -> 2*0.25 - 0.5 + 0.25 = 0.25
    assert math.isclose(O.scalar_generalized(np.array([0.0]), [[2.0, -1.0, 0.25]], -1.0, 1.0)[0], 0.25)


def test_split_fp16_bits_and_identity():
    """Eqs. 12-13, reading C9: hand-worked bit patterns and |X - (hi+lo)| <= 2^-22 |X|."""
    x = np.array([1.0 + 2.0 ** -11 + 2.0 ** -20, 0.1, -0.333333, 2.0 ** -15, 3.0e-6], dtype=np.float32)
    hi, lo = O.split_fp16(x)
    # 1 + 2^-11 + 2^-20 : hi = RNE -> 1 + 2^-10 (above the tie), lo = FP16[2^-11 + 2^-20 - 2^-10] = -(2^-11 - 2^-20)
    assert hi[0] == np.float16(1.0 + 2.0 ** -10)
    assert float(lo[0]) == float(np.float16(-(2.0 ** -11) + 2.0 ** -20))
    assert hi.view(np.uint16)[0] == 0x3C01
    # exact tie rounds to even: 1 + 2^-11 -> 1.0 (mantissa even), lo = 2^-11
    h2, l2 = O.split_fp16(np.array([1.0 + 2.0 ** -11], dtype=np.float32))
    assert h2.view(np.uint16)[0] == 0x3C00 and float(l2[0]) == 2.0 ** -11
    normal = np.abs(x) >= 2.0 ** -3                      # lo stays a normal FP16 number there
    rec = hi.astype(np.float64) + lo.astype(np.float64)
    assert np.all(np.abs(x.astype(np.float64) - rec)[normal] <= 2.0 ** -22 * np.abs(x)[normal])
    # subnormal hi kept, not flushed (C9): 3e-6 < 2^-14
    assert hi[4] != 0 and abs(float(hi[4]) - 3.0e-6) <= 2.0 ** -25


def test_mixed_square_is_eq15_and_close_to_exact_square():
    """Eq. 15: hi hi + hi lo + (hi lo)^T; brute force on N=6, and the dropped lo*lo term plus the
    split error bound |C - S^2| <= ~2^-21 |S||S| in the FP16-normal range."""
    rng = np.random.default_rng(0)
    A = rng.uniform(0.25, 1.0, (6, 6))
    S = (0.5 * (A + A.T)).astype(np.float32)
    hi, lo = O.split_fp16(S)
    C = O.mixed_square_exact(hi, lo)
    h, l = hi.astype(np.float64), lo.astype(np.float64)
    for i in range(6):
        for j in range(6):
            ref = sum(h[i, k] * h[k, j] + h[i, k] * l[k, j] + h[j, k] * l[k, i] for k in range(6))
            assert abs(C[i, j] - ref) < 1e-14
    S64 = S.astype(np.float64)
    assert np.all(np.abs(C - S64 @ S64) <= 2.0 ** -20 * (np.abs(S64) @ np.abs(S64)))
    assert np.array_equal(C, C.T)


def test_mixed_emulation_meets_acceptance_bars():
    """Sizing aid: the emulated Alg. 2 arithmetic stays inside BASELINE north_star's tolerances."""
    w = W.config1(0)
    D, st = O.sp2_mixed_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
    Dref, _ = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
    assert np.abs(D - Dref).max() < 1e-4
    assert abs(np.trace(D) - w.N_occ) < 1e-3 * w.N_occ and O.idempotency_error(D) < 1e-3
