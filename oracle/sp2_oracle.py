"""FP64 CPU oracle for the SP2 hot path of arxiv 2101.06385 -- TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this file.  It shares no code with the CUDA path (`paper_2101_06385_b200/`)
and never imports it; the product path never imports this.

Everything here is plain NumPy in FP64, written in the paper's order and notation so that it
can be checked against PAPER.md by eye (P:n = /root/reference/PAPER.md line n):

  gershgorin_bounds        textbook Gershgorin discs ("Spectral bound estimates of H", Alg. 1 P:136;
                           Gershgorin is the reading C3 of DESIGN.md)
  sp2_ref                  Alg. 1 step by step, S_0 from W_0, B_0, activation
                           X_n = S_{n-1}^2 as a plain FP64 product, sigma_n / IdErr_n / stop rule
                           exactly as printed; `tol` and `max_layers` are the two extra stop tests
                           of reading C8.  No refinement (f_final, Eq. 16) -- out of the hot path.
  sp2_generalized_ref      X_{n+1} = f(W_n X_n + B_n) with scalar weights/biases, i.e. the
                           matrix form of Eq. 17: S_n = th1 X_n + th2 S_{n-1} + th3 I.
  theta_from_wb            reading C19: layer S_n = w_n (sigma_n X_n + (1-sigma_n) S_{n-1}) + b_n I.
  scalar_recursion         the same recursion applied to each eigenvalue (proof of Thm 1).
  eig_density              D = Q theta(mu I - E) Q^T (Eqs. 3-6) by LAPACK eigh.
  split_fp16               Eqs. 12-13 with IEEE round-to-nearest-even conversions (C9).
  mixed_square_exact       Eq. 15 evaluated in FP64 from given hi/lo (products of two
                           FP16 numbers are exact in FP64): the exact target of the tensor-core square.
  sp2_accelerated_ref      the accelerated Deep-NN SP2 of section V.A: real-valued sigma_n chosen for the
                           steepest projection at the HOMO / LUMO eigenvalues "without risking switching places", spectrum
                           kept in [0, 1].  The paper's explicit W_n, B_n are in its supplementary material, which is not
                           available: the formulas here are RE-DERIVED from that description (reading C27) and
                           are "parity unpinned" against the paper's own; they are pinned by mathematics instead.
  generalized_mix_ref      the optimised finite-temperature expansion of Eqs. 17-18 in matrix form:
                           E_0 = rescaled H in natural order, E_n = th1 E^2 + th2 E + th3 I, F~ = I - sum c_i E_i.
  fermi_function           Eq. 20.
  refine_ref               the final refinement f_final of Eq. 16 in FP64: two composed layers with
                           alternating signs; which of the two forms applies follows reading C15 of
                           DESIGN.md (continue the alternation from the last applied sign).
  energy_ref               alpha = Tr[D H] (the observable of Fig. 2), plain FP64.
  truncate_blocks,         the blocked-sparse variant the paper suggests for matrices with decay ("further performance
  sp2_blocked_ref          increases might also be gained by considering a sparse matrix implementation"): Alg. 1
                           in which, before every square, the off-diagonal b x b blocks of S whose Frobenius norm is
                           <= tau are set to zero (reading C28).  tau = 0 is sp2_ref exactly.
  sp2_mixed_ref            Alg. 1 with Alg. 2 as the activation, emulated: FP16 hi/lo split,
                           Eq. 15 products, FP32 rounding of X_n and S_n.  An EMULATION of the arithmetic
                           (FP64 accumulation instead of the tensor core's FP32), used only to size
                           tolerances; parity is always judged against sp2_ref.

Pins (tests/test_oracle_pins.py): closed-form D = Q_occ Q_occ^T, trace, idempotency, commutator,
scalar recursion for every per-layer trace/branch, Theorem 1's inequality and constant, the norm
sandwich of P:120, Gershgorin vs eigvalsh / diagonal matrices, brute-force triple loops on tiny N,
analytic N=1, N=2 cases, tie rule.  The paper prints no worked numeric example (Figs. 2, 5, 6 are
images; their matrices are unspecified), so no golden value comes from the paper: "parity unpinned
by paper examples", pinned by mathematics instead.
"""
from __future__ import annotations

import numpy as np

STOP_NONE, STOP_IDERR_NONPOS, STOP_PARAM_FREE, STOP_TOL, STOP_MAX_LAYERS = 0, 1, 2, 3, 4


def symmetrize_lower(H32):
    """O0: widen the FP32 input exactly and mirror its lower triangle (the library reads the
    lower triangle only, so both sides see the same symmetric matrix)."""
    H = np.asarray(H32, dtype=np.float64)
    return np.tril(H) + np.tril(H, -1).T


def gershgorin_bounds(H):
    """eps_min = min_i (H_ii - R_i), eps_max = max_i (H_ii + R_i), R_i = sum_{j != i} |H_ij|."""
    H = np.asarray(H, dtype=np.float64)
    d = np.diag(H)
    R = np.abs(H).sum(axis=1) - np.abs(d)
    return float((d - R).min()), float((d + R).max())


def initial_layer(H, eps_min, eps_max):
    """W_0 = -(eps_N - eps_1)^{-1} I, B_0 = eps_N (eps_N - eps_1)^{-1} I, S_0 = W_0 X_0 + B_0."""
    n = H.shape[0]
    W0 = -1.0 / (eps_max - eps_min)
    B0 = eps_max / (eps_max - eps_min)
    return W0 * H + B0 * np.eye(n)


def _sign_rule(N_S, N_X, N_occ, sigma_prev, eps_alt):
    """sigma_n = Sign(|2 N_S - N_X - N_occ| - |N_X - N_occ| - sigma_{n-1} eps); a zero
    argument alternates (reading C4: -sigma_{n-1}, and +1 when sigma_{n-1} = 0)."""
    d = abs(2.0 * N_S - N_X - N_occ) - abs(N_X - N_occ) - sigma_prev * eps_alt
    if d > 0:
        return 1, d
    if d < 0:
        return -1, d
    return (-sigma_prev if sigma_prev != 0 else 1), d


def sp2_ref(H32, N_occ, bounds=None, tol=0.0, max_layers=120, eps_alt=0.0, forced_sigma=None,
            square=None, keep_history=False):
    """Alg. 1.  Returns (D, stats) with stats = dict of per-layer lists
    trace_S (N_S after the layer), trace_X (N_X), iderr (IdErr_n), sigma, margin (the Sign argument),
    plus 'stop_reason', 'n_layers', 'bounds'.  `forced_sigma` replays a given branch sequence
    (reading C6); `square` replaces the activation (default: plain FP64 S @ S)."""
    H = symmetrize_lower(H32)
    n_dim = H.shape[0]
    eps_min, eps_max = gershgorin_bounds(H) if bounds is None else (float(bounds[0]), float(bounds[1]))
    if not (eps_max > eps_min):
        raise ValueError("degenerate spectral bounds")
    S = initial_layer(H, eps_min, eps_max)
    N_S = float(np.trace(S))
    sigma_hist = [0]                                   # sigma_0 = 0 (C4)
    iderr_hist = [None]                                # IdErr is indexed from 1
    st = {"trace_S": [], "trace_X": [], "iderr": [], "sigma": [], "margin": [], "S_hist": []}
    n = 0
    stop = STOP_NONE
    while stop == STOP_NONE:
        n += 1
        X = (S @ S) if square is None else square(S)   # X_n = f(S_{n-1})
        N_X = float(np.trace(X))
        iderr = N_S - N_X                              # IdErr_n
        sigma, d = _sign_rule(N_S, N_X, N_occ, sigma_hist[n - 1], eps_alt)
        if forced_sigma is not None:
            sigma = int(forced_sigma[n - 1])
        S = sigma * X + (1 - sigma) * S                # W_n = sigma_n I, B_n = (I - W_n) S_{n-1}
        N_S = sigma * N_X + (1 - sigma) * N_S          # updated occupation of S_n
        sigma_hist.append(sigma)
        iderr_hist.append(iderr)
        st["trace_S"].append(N_S); st["trace_X"].append(N_X); st["iderr"].append(iderr)
        st["sigma"].append(sigma); st["margin"].append(d)
        if keep_history:
            st["S_hist"].append(S.copy())
        if iderr <= 0.0:
            stop = STOP_IDERR_NONPOS
        elif n > 2 and sigma_hist[n - 1] != sigma_hist[n - 2] and iderr > 4.5 * iderr_hist[n - 2] ** 2:
            stop = STOP_PARAM_FREE
        elif tol > 0.0 and iderr <= tol:
            stop = STOP_TOL
        elif n >= max_layers or (forced_sigma is not None and n >= len(forced_sigma)):
            stop = STOP_MAX_LAYERS
    st["stop_reason"] = stop
    st["n_layers"] = n
    st["bounds"] = (eps_min, eps_max)
    return S, st


def theta_from_wb(weights, biases, sigma=None):
    """Reading C19: S_n = w_n (sigma_n X_n + (1 - sigma_n) S_{n-1}) + b_n I
    => theta_n = (w sigma, w (1 - sigma), b) in Eq. 17's order."""
    w = np.asarray(weights, dtype=np.float64)
    b = np.asarray(biases, dtype=np.float64)
    s = np.ones_like(w) if sigma is None else np.asarray(sigma, dtype=np.float64)
    return np.stack([w * s, w * (1.0 - s), b], axis=1)


def sp2_generalized_ref(H32, theta, bounds=None, square=None):
    """L fixed layers S_n = th1 S_{n-1}^2 + th2 S_{n-1} + th3 I (Eq. 17 in matrix form)."""
    H = symmetrize_lower(H32)
    n_dim = H.shape[0]
    eps_min, eps_max = gershgorin_bounds(H) if bounds is None else (float(bounds[0]), float(bounds[1]))
    if not (eps_max > eps_min):
        raise ValueError("degenerate spectral bounds")
    S = initial_layer(H, eps_min, eps_max)
    I = np.eye(n_dim)
    st = {"trace_S": [], "trace_X": []}
    for th1, th2, th3 in np.asarray(theta, dtype=np.float64):
        X = (S @ S) if square is None else square(S)
        st["trace_X"].append(float(np.trace(X)))
        S = th1 * X + th2 * S + th3 * I
        st["trace_S"].append(float(np.trace(S)))
    st["bounds"] = (eps_min, eps_max)
    return S, st


def scalar_initial(eigs, eps_min, eps_max):
    return (eps_max - np.asarray(eigs, dtype=np.float64)) / (eps_max - eps_min)


def scalar_recursion(eigs, N_occ, eps_min, eps_max, tol=0.0, max_layers=120, eps_alt=0.0, forced_sigma=None,
                     square=None):
    """Alg. 1 on the eigenvalues: lambda_j^(i) = lambda_j^(i-1) + sigma_i (lambda_j^(i-1) - (lambda_j^(i-1))^2)
    (P:294), with N_S = sum lambda, N_X = sum lambda^2.  Same outputs as sp2_ref minus the matrix.
    `square` replaces the elementwise activation like sp2_ref's hook (default: lam * lam); the stop-rule pins use
    it to put a chosen error on one layer's X."""
    lam = scalar_initial(eigs, eps_min, eps_max)
    N_S = float(lam.sum())
    sig = [0]
    ide = [None]
    st = {"trace_S": [], "trace_X": [], "iderr": [], "sigma": [], "margin": []}
    n, stop = 0, STOP_NONE
    while stop == STOP_NONE:
        n += 1
        x = (lam * lam) if square is None else square(lam)
        N_X = float(x.sum())
        iderr = N_S - N_X
        sigma, d = _sign_rule(N_S, N_X, N_occ, sig[n - 1], eps_alt)
        if forced_sigma is not None:
            sigma = int(forced_sigma[n - 1])
        lam = sigma * x + (1 - sigma) * lam
        N_S = sigma * N_X + (1 - sigma) * N_S
        sig.append(sigma); ide.append(iderr)
        st["trace_S"].append(N_S); st["trace_X"].append(N_X); st["iderr"].append(iderr)
        st["sigma"].append(sigma); st["margin"].append(d)
        if iderr <= 0.0:
            stop = STOP_IDERR_NONPOS
        elif n > 2 and sig[n - 1] != sig[n - 2] and iderr > 4.5 * ide[n - 2] ** 2:
            stop = STOP_PARAM_FREE
        elif tol > 0.0 and iderr <= tol:
            stop = STOP_TOL
        elif n >= max_layers or (forced_sigma is not None and n >= len(forced_sigma)):
            stop = STOP_MAX_LAYERS
    st["stop_reason"], st["n_layers"], st["lam"] = stop, n, lam
    return st


def scalar_generalized(eigs, theta, eps_min, eps_max):
    """Eq. 17 on each eigenvalue: eps_n = th1 eps_{n-1}^2 + th2 eps_{n-1} + th3."""
    lam = scalar_initial(eigs, eps_min, eps_max)
    for th1, th2, th3 in np.asarray(theta, dtype=np.float64):
        lam = th1 * lam * lam + th2 * lam + th3
    return lam


def eig_density(H32, N_occ):
    """D = Q theta(mu I - E) Q^T (Eq. 6): projector on the N_occ lowest eigenvectors."""
    E, V = np.linalg.eigh(symmetrize_lower(H32))
    k = int(round(N_occ))
    Vo = V[:, :k]
    return Vo @ Vo.T, E


def closed_form_density(Q, n_occ):
    """H was built as Q diag(eps) Q^T with the occupied eigenvalues first: D* = Q_occ Q_occ^T."""
    Qo = np.asarray(Q, dtype=np.float64)[:, : int(round(n_occ))]
    return Qo @ Qo.T


def closed_form_density_entries(Q, n_occ, rows, cols):
    """Sampled entries D*_ij = sum_{k < N_occ} Q_ik Q_jk, one by one (for full-size parity)."""
    Qo = np.asarray(Q, dtype=np.float64)[:, : int(round(n_occ))]
    return np.einsum("ik,ik->i", Qo[np.asarray(rows)], Qo[np.asarray(cols)])


def split_fp16(X32):
    """Eqs. 12-13: X0 = FP16[X], X1 = FP16[X - X0]; RNE conversions, subnormals kept (C9);
    the subtraction is done in FP32 (exact: X - X0 is representable)."""
    X32 = np.asarray(X32, dtype=np.float32)
    hi = X32.astype(np.float16)
    lo = (X32 - hi.astype(np.float32)).astype(np.float16)
    return hi, lo


def mixed_square_exact(hi, lo):
    """Eq. 15: X^2 ~ X0 X0 + X0 X1 + (X0 X1)^T with exact products and FP64 sums."""
    h = np.asarray(hi, dtype=np.float64)
    l = np.asarray(lo, dtype=np.float64)
    B = h @ l
    return h @ h + B + B.T


def mixed_square_emulated(S):
    """Alg. 2 on an FP64 copy of an FP32 matrix: split, Eq. 15, round the result to FP32."""
    hi, lo = split_fp16(np.asarray(S, dtype=np.float32))
    return mixed_square_exact(hi, lo).astype(np.float32).astype(np.float64)


def sp2_mixed_ref(H32, N_occ, bounds=None, tol=0.0, max_layers=120, eps_alt=0.0, forced_sigma=None):
    """Alg. 1 with the emulated Alg. 2 activation (the state is rounded to FP32 before each split).
    Tolerance-sizing aid only (see module docstring)."""
    def sq_round(S):
        return mixed_square_emulated(S.astype(np.float32))
    return sp2_ref(H32, N_occ, bounds, tol, max_layers, eps_alt, forced_sigma, square=sq_round)


def idempotency_error(D):
    """||D^2 - D||_F / sqrt(N) (acceptance measure of BASELINE.json north_star)."""
    D = np.asarray(D, dtype=np.float64)
    return float(np.linalg.norm(D @ D - D) / np.sqrt(D.shape[0]))


def commutator_norm(H32, D):
    H = symmetrize_lower(H32)
    D = np.asarray(D, dtype=np.float64)
    return float(np.linalg.norm(H @ D - D @ H))


THEOREM1_C = (71.0 + 17.0 * np.sqrt(17.0)) / 32.0


def refine_ref(S, last_sigma):
    """Eq. 16: f_final(S) = 2 S^2 - S^4 or (2 S - S^2)^2, "the result of composing two layers in a
    single step with sigma_n = 1 and sigma_{n-1} = -1 or sigma_n = -1 and sigma_{n-1} = 1".
    Reading C15: the alternation continues from the last APPLIED sign, so
      last_sigma = -1: next layer squares (X = S^2), the one after applies 2X - X^2  ->  2 S^2 - S^4
      last_sigma = +1: next layer applies T = 2S - S^2, the one after squares          ->  (2S - S^2)^2
    Plain FP64 products ("standard double precision")."""
    S = np.asarray(S, dtype=np.float64)
    if last_sigma not in (1, -1):
        raise ValueError("last_sigma must be +1 or -1")
    X = S @ S
    if last_sigma < 0:
        return 2.0 * X - X @ X
    T = 2.0 * S - X
    return T @ T


def energy_ref(D, H):
    """alpha = Tr[D H], with H symmetrised from its lower triangle like everywhere else."""
    D = np.asarray(D, dtype=np.float64)
    return float(np.sum(D * symmetrize_lower(H).T))


def iderr_ref(X):
    """IdErr = Tr[X - X^2]."""
    X = np.asarray(X, dtype=np.float64)
    return float(np.trace(X) - np.sum(X * X.T))


def generalized_mix_ref(H32, theta, c, bounds=None):
    """Eqs. 17-18 in matrix form.  eps_0 of Eq. 17 is "the eigenvalues eps_i in [0,1] of the re-scaled
    Hamiltonian" in natural order (reading C26): E_0 = (H - eps_min I)/(eps_max - eps_min);
    E_n = th_{n-1,1} E_{n-1}^2 + th_{n-1,2} E_{n-1} + th_{n-1,3} I (Eq. 17);  F~ = I - sum_{i=0}^{L} c_i E_i (Eq. 18)."""
    H = symmetrize_lower(H32)
    n = H.shape[0]
    e0, e1 = gershgorin_bounds(H) if bounds is None else (float(bounds[0]), float(bounds[1]))
    theta = np.asarray(theta, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    if c.shape != (theta.shape[0] + 1,):
        raise ValueError("c must have L + 1 entries")
    I = np.eye(n)
    E = (H - e0 * I) / (e1 - e0)
    acc = c[0] * E
    for k in range(theta.shape[0]):
        E = theta[k, 0] * (E @ E) + theta[k, 1] * E + theta[k, 2] * I
        acc = acc + c[k + 1] * E
    return I - acc


def fermi_function(eps, beta):
    """Eq. 20: F(eps) = (exp(beta (eps - 1/2)) + 1)^-1 on the rescaled energies eps in [0, 1]."""
    return 1.0 / (np.exp(beta * (np.asarray(eps, dtype=np.float64) - 0.5)) + 1.0)


def accelerated_layer(N_S, N_X, n_dim, N_occ, h, l, sigma_prev=0, eps_alt=0.0):
    """One layer's weights of the accelerated scheme (section V.A; reading C27).

    State: all eigenvalues of S in [0, 1]; unoccupied ones in [0, l], occupied ones in [h, 1], 0 <= l < h <= 1
    (l, h = rescaled LUMO / HOMO estimates, "prior knowledge of the re-scaled HOMO and LUMO eigenvalues").
    Two generalized projections, each the SP2 polynomial composed with an affine map (the "shift and re-scale"):
      A(x) = (a x + 1 - a)^2,  a = 2 / (2 - l):  A(1) = 1, and A(0) = A(l): the largest a for which no unoccupied
             eigenvalue is mapped above A(0) -- steepest at the HOMO side without switching places, range in [0, 1];
      B(x) = 2 a x - (a x)^2,  a = 2 / (1 + h):  B(0) = 0, and B(h) = B(1).
    a = 1 (l = 0 or h = 1) gives back x^2 and 2x - x^2.  The branch is chosen as in Alg. 1: the one whose
    occupation Tr[.] is closer to N_occ, both traces following from N_S = Tr S, N_X = Tr S^2 and N.
    Returns (sigma, theta (th1, th2, th3), h', l')."""
    aA = 2.0 / (2.0 - l)
    aB = 2.0 / (1.0 + h)
    trA = aA * aA * N_X + 2.0 * aA * (1.0 - aA) * N_S + (1.0 - aA) ** 2 * n_dim
    trB = 2.0 * aB * N_S - aB * aB * N_X
    d = abs(trB - N_occ) - abs(trA - N_occ) - sigma_prev * eps_alt
    if d > 0.0:
        sigma = 1
    elif d < 0.0:
        sigma = -1
    else:
        sigma = -sigma_prev if sigma_prev != 0 else 1
    if sigma > 0:
        theta = (aA * aA, 2.0 * aA * (1.0 - aA), (1.0 - aA) ** 2)
        h2 = (aA * h + 1.0 - aA) ** 2
        l2 = max((1.0 - aA) ** 2, (aA * l + 1.0 - aA) ** 2)
    else:
        theta = (-aB * aB, 2.0 * aB, 0.0)
        h2 = min(2.0 * aB * h - (aB * h) ** 2, 2.0 * aB - aB * aB)
        l2 = 2.0 * aB * l - (aB * l) ** 2
    return sigma, theta, h2, l2, d


def sp2_accelerated_ref(H32, N_occ, bounds, homo, lumo, tol=0.0, max_layers=120, eps_alt=0.0, keep_history=False):
    """Alg. 1 with the accelerated weights of section V.A.  homo / lumo: estimates of the highest occupied / lowest
    unoccupied eigenvalue of H (energy units; lumo > homo), bounds: spectral bounds as in sp2_ref.
    Stop tests: IdErr_n <= 0, IdErr_n <= tol, n = max_layers (the parameter-free test of Alg. 1 rests on Theorem 1,
    which is proved for the alternating x^2 / 2x - x^2 pair only, so it is not applied here)."""
    H = symmetrize_lower(H32)
    n_dim = H.shape[0]
    eps_min, eps_max = gershgorin_bounds(H) if bounds is None else (float(bounds[0]), float(bounds[1]))
    S = initial_layer(H, eps_min, eps_max)
    I = np.eye(n_dim)
    h = (eps_max - homo) / (eps_max - eps_min)         # S_0 reverses the order: the HOMO is the smallest occupied value
    l = (eps_max - lumo) / (eps_max - eps_min)
    if not (0.0 <= l < h <= 1.0):
        raise ValueError("need eps_min <= homo < lumo <= eps_max")
    N_S = float(np.trace(S))
    st = {"trace_S": [], "trace_X": [], "iderr": [], "sigma": [], "theta": [], "h": [], "l": [], "margin": [],
          "S_hist": []}
    n, stop, sigma_prev = 0, STOP_NONE, 0
    while stop == STOP_NONE:
        n += 1
        X = S @ S
        N_X = float(np.trace(X))
        iderr = N_S - N_X
        sigma, th, h, l, d = accelerated_layer(N_S, N_X, n_dim, N_occ, h, l, sigma_prev, eps_alt)
        S = th[0] * X + th[1] * S + th[2] * I
        N_S = float(np.trace(S))
        sigma_prev = sigma
        st["trace_S"].append(N_S); st["trace_X"].append(N_X); st["iderr"].append(iderr); st["sigma"].append(sigma)
        st["theta"].append(th); st["h"].append(h); st["l"].append(l); st["margin"].append(d)
        if keep_history:
            st["S_hist"].append(S.copy())
        if iderr <= 0.0:
            stop = STOP_IDERR_NONPOS
        elif tol > 0.0 and iderr <= tol:
            stop = STOP_TOL
        elif n >= max_layers:
            stop = STOP_MAX_LAYERS
    st["stop_reason"], st["n_layers"], st["bounds"] = stop, n, (eps_min, eps_max)
    return S, st


def truncate_blocks(S, tau, block=128):
    """Reading C28 (P:206 names no rule): cut S into block x block blocks on a fixed grid; an OFF-DIAGONAL block whose
    Frobenius norm is <= tau is set to zero (with its mirror image, so S stays symmetric); diagonal blocks are always
    kept (they carry the trace).  Returns (S_truncated, kept) with kept[I, J] = 1 for blocks that survive."""
    S = np.array(S, dtype=np.float64)
    n = S.shape[0]
    nb = (n + block - 1) // block
    kept = np.ones((nb, nb), dtype=np.int8)
    if tau <= 0.0:
        return S, kept
    for I in range(nb):
        for J in range(I):
            blk = S[I * block:(I + 1) * block, J * block:(J + 1) * block]
            if np.sqrt(np.sum(blk * blk)) <= tau:
                S[I * block:(I + 1) * block, J * block:(J + 1) * block] = 0.0
                S[J * block:(J + 1) * block, I * block:(I + 1) * block] = 0.0
                kept[I, J] = kept[J, I] = 0
    return S, kept


def sp2_blocked_ref(H32, N_occ, bounds=None, tau=0.0, block=128, tol=0.0, max_layers=120, eps_alt=0.0,
                    forced_sigma=None, square=None):
    """Alg. 1 on block-truncated iterates (reading C28).  Layer n:
         S' = truncate_blocks(S_{n-1}, tau);  X_n = S' S';  N_X = Tr X_n;  IdErr_n = N_S - N_X with N_S = Tr S'
         (= Tr S_{n-1}: diagonal blocks are never cut);  sigma_n by Alg. 1's rule;  S_n = sigma_n X_n + (1 - sigma_n) S'.
    Same stop tests and outputs as sp2_ref, plus st["kept_fraction"][n-1] = surviving fraction of the b x b blocks and
    st["work_fraction"][n-1] = fraction of the block products S'_IK S'_KJ (I >= J) whose two factors both survive --
    the tensor-core work a blocked implementation has left.
    square: test hook (default None = the plain NumPy product `Sp @ Sp`): a callable A -> A @ A in FP64 computed by another
    library routine, for the sizes (N > 8192) where NumPy needs minutes per layer.  Nothing else changes."""
    H = symmetrize_lower(H32)
    eps_min, eps_max = gershgorin_bounds(H) if bounds is None else (float(bounds[0]), float(bounds[1]))
    if not (eps_max > eps_min):
        raise ValueError("degenerate spectral bounds")
    S = initial_layer(H, eps_min, eps_max)
    N_S = float(np.trace(S))
    sigma_hist, iderr_hist = [0], [None]
    st = {"trace_S": [], "trace_X": [], "iderr": [], "sigma": [], "margin": [], "kept_fraction": [],
          "work_fraction": []}
    n, stop = 0, STOP_NONE
    while stop == STOP_NONE:
        n += 1
        Sp, kept = truncate_blocks(S, tau, block)
        X = Sp @ Sp if square is None else square(Sp)
        N_X = float(np.trace(X))
        iderr = N_S - N_X
        sigma, d = _sign_rule(N_S, N_X, N_occ, sigma_hist[n - 1], eps_alt)
        if forced_sigma is not None:
            sigma = int(forced_sigma[n - 1])
        S = sigma * X + (1 - sigma) * Sp
        N_S = sigma * N_X + (1 - sigma) * N_S
        sigma_hist.append(sigma); iderr_hist.append(iderr)
        st["trace_S"].append(N_S); st["trace_X"].append(N_X); st["iderr"].append(iderr)
        st["sigma"].append(sigma); st["margin"].append(d)
        k = kept.astype(np.float64)
        st["kept_fraction"].append(float(k.mean()))
        pairs = np.tril(k @ k)                       # pairs[I, J] = number of K with both factors kept
        st["work_fraction"].append(float(pairs.sum() / (kept.shape[0] * np.tril(np.ones_like(k)).sum())))
        if iderr <= 0.0:
            stop = STOP_IDERR_NONPOS
        elif n > 2 and sigma_hist[n - 1] != sigma_hist[n - 2] and iderr > 4.5 * iderr_hist[n - 2] ** 2:
            stop = STOP_PARAM_FREE
        elif tol > 0.0 and iderr <= tol:
            stop = STOP_TOL
        elif n >= max_layers or (forced_sigma is not None and n >= len(forced_sigma)):
            stop = STOP_MAX_LAYERS
    st["stop_reason"], st["n_layers"], st["bounds"] = stop, n, (eps_min, eps_max)
    return S, st
