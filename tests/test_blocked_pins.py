"""Pins for the blocked-sparse oracle (oracle.truncate_blocks / sp2_blocked_ref, reading C28), CPU only.
The paper states no truncation rule, so nothing here comes from the paper's text: the pins are the mathematics --
tau = 0 is Alg. 1 itself, the truncation is a symmetric projection with a known Frobenius error, the result converges to
the LAPACK projector at a rate set by tau, and the work that is left follows the decay of the density matrix."""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W


def test_tau_zero_is_alg1_exactly():
    """tau = 0 keeps every block: bit-identical to sp2_ref (same operations in the same order)."""
    for w in (W.config1(0), W.decaying_chain(0, n=300)):
        D0, s0 = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
        D1, s1 = O.sp2_blocked_ref(w.H32, w.N_occ, w.bounds, tau=0.0, block=64, tol=w.tol, max_layers=w.max_layers)
        assert np.array_equal(D0, D1) and s0["sigma"] == s1["sigma"] and s0["trace_S"] == s1["trace_S"]
        assert s0["n_layers"] == s1["n_layers"] and s0["stop_reason"] == s1["stop_reason"]
        assert all(k == 1.0 for k in s1["kept_fraction"]) and all(abs(k - 1.0) < 1e-15 for k in s1["work_fraction"])


def test_truncate_blocks_by_hand():
    """A 6 x 6 matrix in 2 x 2 blocks: block (1,0) has norm 0.5, block (2,0) norm 0.01, block (2,1) norm 0.2."""
    S = np.eye(6)
    S[2:4, 0:2] = [[0.3, 0.0], [0.0, 0.4]]
    S[4:6, 0:2] = [[0.006, 0.0], [0.0, 0.008]]
    S[4:6, 2:4] = [[0.2, 0.0], [0.0, 0.0]]
    S = np.tril(S) + np.tril(S, -1).T
    T, kept = O.truncate_blocks(S, 0.1, block=2)
    assert kept.tolist() == [[1, 1, 0], [1, 1, 1], [0, 1, 1]]
    assert np.all(T[4:6, 0:2] == 0) and np.all(T[0:2, 4:6] == 0) and np.array_equal(T[2:4, 0:2], S[2:4, 0:2])
    assert np.array_equal(T, T.T) and np.trace(T) == np.trace(S)
    # the Frobenius error is the norm of what was cut (both mirror images)
    assert abs(np.linalg.norm(S - T) - np.sqrt(2) * 0.01) < 1e-15
    # the threshold is inclusive (<= tau), and a tiny diagonal block survives
    T2, k2 = O.truncate_blocks(S, 0.2, block=2)
    assert k2[2, 1] == 0
    Z = np.diag([1e-9] * 4)
    assert np.array_equal(O.truncate_blocks(Z, 1.0, block=2)[0], Z)      # diagonal blocks are never cut


@pytest.mark.parametrize("tau", [1e-8, 1e-6, 1e-4])
def test_blocked_result_against_lapack_and_error_scales_with_tau(tau):
    """On a Hamiltonian with decay the truncated recursion still reaches the eigenprojector; its error is bounded by
    a modest multiple of tau per layer and grows with tau; trace and idempotency stay within the same bound."""
    w = W.decaying_chain(1, n=512)
    De, E = O.eig_density(w.H32, w.N_occ)
    k = int(w.N_occ)
    assert E[k] - E[k - 1] > 0.5                                          # the staggered onsite term keeps the gap
    D, st = O.sp2_blocked_ref(w.H32, w.N_occ, None, tau=tau, block=32, tol=1e-9, max_layers=100)
    err = np.abs(D - De).max()
    nb = 512 // 32
    assert err <= 4.0 * tau * st["n_layers"] + 1e-9, (err, st["n_layers"])
    assert abs(np.trace(D) - w.N_occ) <= 4.0 * tau * st["n_layers"] * nb + 1e-8
    assert O.idempotency_error(D) <= 4.0 * tau * st["n_layers"] + 1e-8
    assert st["work_fraction"][-1] < 0.5                                  # the far blocks of a decaying D are gone


def test_error_is_monotone_in_tau_and_work_follows_decay():
    w = W.decaying_chain(2, n=512)
    De, _ = O.eig_density(w.H32, w.N_occ)
    errs, work = [], []
    for tau in (0.0, 1e-8, 1e-6, 1e-4, 1e-1):
        D, st = O.sp2_blocked_ref(w.H32, w.N_occ, None, tau=tau, block=32, tol=1e-9, max_layers=100)
        errs.append(np.abs(D - De).max())
        work.append(np.mean(st["work_fraction"]))
    assert errs[0] < 1e-8 and all(errs[i] <= errs[i + 1] * 1.5 + 1e-12 for i in range(len(errs) - 1))
    assert errs[-1] > 1e-2                                                # a cut at 1e-1 removes real couplings
    assert work[0] == 1.0 and all(work[i] >= work[i + 1] for i in range(len(work) - 1)) and work[-2] < 0.6


def test_no_decay_no_savings():
    """A dense Haar-rotated H (config 1's shape) has no block structure: nothing is cut at a small tau and the result
    equals Alg. 1's."""
    w = W.config1(2, n=256)
    D0, s0 = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
    D1, s1 = O.sp2_blocked_ref(w.H32, w.N_occ, w.bounds, tau=1e-6, block=64, tol=w.tol, max_layers=w.max_layers)
    assert min(s1["kept_fraction"]) == 1.0 and np.array_equal(D0, D1)


def test_blocked_traces_follow_the_matrix():
    """N_S reported by the blocked oracle is Tr S_n of its own iterate, N_X = ||S'||_F^2 of the truncated one."""
    w = W.decaying_chain(3, n=256)
    b = O.gershgorin_bounds(O.symmetrize_lower(w.H32))
    S = O.initial_layer(O.symmetrize_lower(w.H32), *b)
    _, st = O.sp2_blocked_ref(w.H32, w.N_occ, b, tau=1e-5, block=32, tol=0.0, max_layers=6)
    for n in range(6):
        Sp, _ = O.truncate_blocks(S, 1e-5, 32)
        assert abs(st["trace_X"][n] - np.sum(Sp * Sp)) < 1e-10
        sg = st["sigma"][n]
        S = sg * (Sp @ Sp) + (1 - sg) * Sp
        assert abs(st["trace_S"][n] - np.trace(S)) < 1e-10
