"""GPU parity of the blocked-sparse variant (opts.trunc_tau > 0, reading C28): off-diagonal 128 x 128
blocks of S with Frobenius norm <= tau count as zero before every square -- their operand tiles are neither loaded nor
multiplied.  Oracle: sp2_blocked_ref (FP64, the same rule); references: the LAPACK eigenprojector."""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W
from tests import parity_util as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    torch.cuda.set_device(0)
    h = api.Handle(4096, 0, 120)
    yield api, h, torch
    h.close()


@pytest.fixture(scope="module")
def big_env(cuda_device):
    """Sizes with more than 32 K-blocks of 128 (the sparse K-masks are four 32-bit ballot words: N = 4224 reaches the
    second word, 8192 fills two, 16384 all four)."""
    import torch

    from paper_2101_06385_b200 import api

    torch.cuda.set_device(0)
    h = api.Handle(16384, 0, 120)
    yield api, h, torch
    h.close()


def _decaying_chain_case(api, h, torch, n, tau, with_eig, square=None):
    w = W.decaying_chain(n, n=n)
    opts = api.make_opts(tol=w.tol, max_layers=w.max_layers, trunc_tau=tau)
    Dg, info = h.density_matrix(torch.from_numpy(w.H32).cuda(), w.N_occ, opts)
    assert torch.equal(Dg, Dg.T)
    D = Dg.cpu().numpy().astype(np.float64)
    used = info["bounds"]
    Dref, st = O.sp2_blocked_ref(w.H32, w.N_occ, used, tau=tau, block=128, tol=w.tol, max_layers=w.max_layers,
                                 square=square)
    err_o = np.abs(D - Dref).max()
    wf_o = float(np.mean(st["work_fraction"][: info["n_layers"]]))
    msg = (f"blocked N={n} tau={tau:g}: layers gpu/oracle {info['n_layers']}/{st['n_layers']}, work fraction gpu "
           f"{info['work_fraction']:.4f} oracle {wf_o:.4f}, max|D-Dref|={err_o:.2e}")
    if n <= 4224:
        P.assert_acceptance(D, Dref, w.N_occ, f"N={n} tau={tau}")
    else:                                  # the same three bars, the FP64 product on the device in the harness
        Dd = Dg.double()
        idem = float(torch.linalg.norm(Dd @ Dd - Dd) / np.sqrt(n))
        assert err_o <= P.TOL_D and idem <= P.TOL_IDEM, msg
        assert abs(float(torch.trace(Dd)) - w.N_occ) <= P.TOL_TRACE_REL * w.N_occ
    if with_eig:
        De, E = O.eig_density(w.H32, w.N_occ)
        err_e = np.abs(D - De).max()
        msg += f" max|D-D_eig|={err_e:.2e}"
        assert err_e <= P.TOL_D
    print(msg)
    return w, info, st, wf_o


@pytest.mark.parametrize("n,tau", [(2048, 1e-7), (2048, 1e-5), (1000, 1e-6), (3000, 1e-6)])
def test_decaying_chain(env, n, tau):
    api, h, torch = env
    w, info, st, wf_o = _decaying_chain_case(api, h, torch, n, tau, with_eig=True)
    assert abs(info["n_layers"] - st["n_layers"]) <= 2
    P.branch_prefix_check(info, st, w.N_occ)
    k = min(info["n_layers"], st["n_layers"])
    assert np.abs(np.array(info["trace_X"][:k]) - np.array(st["trace_X"][:k])).max() <= 1e-3 * w.N_occ
    # the tensor-core work that is left follows the oracle's count of surviving block products
    assert abs(info["work_fraction"] - wf_o) <= 0.05
    if n >= 2048:
        assert info["work_fraction"] < 0.5


@pytest.mark.parametrize("n", [4224, 8192, 16384])
def test_decaying_chain_more_than_32_k_blocks(big_env, n):
    """nb = 33, 64, 128 K-blocks: every word of the K-masks and sparse_bit's word selection.  Oracle: sp2_blocked_ref
    itself; at N = 16384 its one matrix product per layer is computed in FP64 on the device (the `square` hook: NumPy
    needs ~11 s per layer there), everything else -- truncation rule, traces, branch rule, stop tests -- is the oracle's
    NumPy code.  The LAPACK projector is compared at N = 4224 only (minutes beyond)."""
    api, h, torch = big_env

    def square_fp64_on_device(A):
        Ad = torch.from_numpy(A).cuda()
        return (Ad @ Ad).cpu().numpy()

    w, info, st, wf_o = _decaying_chain_case(api, h, torch, n, 1e-6, with_eig=(n <= 4224),
                                            square=square_fp64_on_device if n > 8192 else None)
    assert abs(info["n_layers"] - st["n_layers"]) <= 2
    P.branch_prefix_check(info, st, w.N_occ)
    k = min(info["n_layers"], st["n_layers"])
    assert np.abs(np.array(info["trace_X"][:k]) - np.array(st["trace_X"][:k])).max() <= P.TRACE_NOISE_REL * w.N_occ
    assert abs(info["work_fraction"] - wf_o) <= 0.05
    assert info["work_fraction"] < 0.2


def test_nothing_cut_is_the_dense_layer_at_33_k_blocks(big_env):
    """The 'nothing cut' check with a second mask word in use (N = 4224: nb = 33, four rounds of 128 x 128 tiles): on a
    dense H every block product is executed (work fraction exactly 1), the branch sequence and the layer count are the
    dense kernel's, and D agrees to FP32 rounding.  Bit-identity is asserted at N = 2048 only (next test): there both
    launches are one round of whole tiles, while here the dense launch interleaves K over two rounds and cuts its last
    round into column strips (measured max difference 4.2e-6)."""
    api, h, torch = big_env
    w = W.gapped_dense(3, 4224, (-1.0, -0.2), (0.2, 1.0), 2112, "gapped_N4224", bounds=(-1.0, 1.0), device="cuda")
    Hd = torch.from_numpy(w.H32).cuda()
    o_d = api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=w.max_layers, tile_config=1, exact_diag=0)
    o_s = api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=w.max_layers, trunc_tau=1e-30)
    D0, i0 = h.density_matrix(Hd, w.N_occ, o_d)
    D1, i1 = h.density_matrix(Hd, w.N_occ, o_s)
    assert i1["work_fraction"] == 1.0
    assert i0["sigma"] == i1["sigma"] and i0["n_layers"] == i1["n_layers"]
    diff = float((D0 - D1).abs().max())
    print(f"N=4224 nothing cut: bits equal = {torch.equal(D0, D1)}, max diff {diff:.2e}")
    assert diff <= 2e-5
    ref = O.closed_form_density_entries(w.Q, w.N_occ, np.arange(0, 4224, 7), np.arange(0, 4224, 7)[::-1].copy())
    got = D1.double().cpu().numpy()[np.arange(0, 4224, 7), np.arange(0, 4224, 7)[::-1]]
    assert np.abs(got - ref).max() <= P.TOL_D


def test_nothing_cut_is_the_dense_layer_bit_for_bit(env):
    """With a threshold below every non-zero block norm the sparse instantiation multiplies the K-blocks in the dense
    order: at N = 2048 (one round, no strips) D equals the dense kernel's (exact_diag = 0, 128 x 128 tiles) bit for bit
    on a dense H, where every block product is executed; on a banded H the (numerically) zero blocks come for free."""
    api, h, torch = env
    for w, dense in ((W.config2(0), True), (W.decaying_chain(5, n=2048, decay=40.0, cutoff=400), False)):
        Hd = torch.from_numpy(w.H32).cuda()
        o_d = api.make_opts(tol=w.tol, max_layers=w.max_layers, tile_config=1, exact_diag=0)
        o_s = api.make_opts(tol=w.tol, max_layers=w.max_layers, trunc_tau=1e-30)
        D0, i0 = h.density_matrix(Hd, w.N_occ, o_d)
        D1, i1 = h.density_matrix(Hd, w.N_occ, o_s)
        print(f"{w.name}: work fraction {i1['work_fraction']:.3f}")
        if dense:
            assert i1["work_fraction"] == 1.0
            assert torch.equal(D0, D1) and i0["sigma"] == i1["sigma"] and i0["trace_S"] == i1["trace_S"]
        else:
            # block norms are kept in 2^48 fixed point: blocks with norm below 2^-24.5 = 4e-8 count as zero for any
            # tau > 0 (the dense kernel carries values of 1e-20 there), everything else is multiplied as before
            assert i1["work_fraction"] < 1.0 and i0["sigma"] == i1["sigma"]
            assert float((D0 - D1).abs().max()) <= 2e-6


def test_config2_with_truncation(env):
    """BASELINE configs[1] is the one config whose H has structure (a cutoff radius), but with randomly numbered sites and
    a gap of 1e-3 its density matrix has no block decay at N = 2048: a small tau cuts (almost) nothing and the result
    stays within the acceptance bars of the LAPACK projector."""
    api, h, torch = env
    w = W.config2(0)
    D, info = h.density_matrix(torch.from_numpy(w.H32).cuda(), w.N_occ,
                               api.make_opts(tol=w.tol, max_layers=w.max_layers, trunc_tau=1e-7))
    De, _ = O.eig_density(w.H32, w.N_occ)
    print(f"config2 tau=1e-7: layers {info['n_layers']} work fraction {info['work_fraction']:.3f} "
          f"err {np.abs(D.cpu().numpy() - De).max():.2e}")
    P.assert_acceptance(D.cpu().numpy().astype(np.float64), De, w.N_occ, "config2 blocked")
    assert info["work_fraction"] > 0.9


def test_blocked_generalized_and_argument_errors(env):
    api, h, torch = env
    w = W.decaying_chain(7, n=1536)
    theta = np.array([[1.0, 0.0, 0.0], [-1.0, 2.0, 0.0]] * 5)
    b = O.gershgorin_bounds(O.symmetrize_lower(w.H32))
    X, info = h.generalized(torch.from_numpy(w.H32).cuda(), theta, bounds=b, opts=api.make_opts(trunc_tau=1e-6))
    S = O.initial_layer(O.symmetrize_lower(w.H32), *b)
    for t1, t2, t3 in theta:                       # the same rule, written out: truncate, square, combine
        Sp, _ = O.truncate_blocks(S, 1e-6, 128)
        S = t1 * (Sp @ Sp) + t2 * Sp + t3 * np.eye(S.shape[0])
    assert np.abs(X.cpu().numpy() - S).max() <= 1e-4
    Hd = torch.from_numpy(w.H32).cuda()
    for bad in (dict(tile_config=3), dict(tile_config=2), dict(tile_config=4)):
        with pytest.raises(api.SP2Error) as e:
            h.density_matrix(Hd, w.N_occ, api.make_opts(trunc_tau=1e-6, **bad))
        assert e.value.status == -1


def test_small_n_keeps_the_blocked_variant_and_resident_solves_reset_the_diagnostics(env):
    """N <= 256 normally goes to the one-launch resident kernel, which has no blocked-sparse variant: with trunc_tau > 0
    the call must stay on the layer kernel (not drop the option silently), and a resident solve afterwards must report
    'dense' through sp2_last_sparse_work instead of the previous solve's counts."""
    import ctypes as C

    api, h, torch = env
    w = W.decaying_chain(3, n=200)
    Hd = torch.from_numpy(w.H32).cuda()
    D, info = h.density_matrix(Hd, w.N_occ, api.make_opts(tol=w.tol, max_layers=w.max_layers, trunc_tau=1e-6))
    assert info["launches"] > 1                      # one kernel per layer, not the resident launch
    assert 0.0 < info["work_fraction"] <= 1.0
    Dref, st = O.sp2_blocked_ref(w.H32, w.N_occ, info["bounds"], tau=1e-6, block=128, tol=w.tol, max_layers=w.max_layers)
    P.assert_acceptance(D.cpu().numpy().astype(np.float64), Dref, w.N_occ, "N=200 blocked")
    wk = (C.c_double * 2)()
    h.lib.sp2_last_sparse_work(h._h, wk)
    assert wk[1] > 0
    D2, info2 = h.density_matrix(Hd, w.N_occ, api.make_opts(tol=w.tol, max_layers=w.max_layers))
    assert info2["launches"] == 1                    # resident path
    h.lib.sp2_last_sparse_work(h._h, wk)
    assert wk[0] == 0.0 and wk[1] == 0.0
    assert h.lib.sp2_last_round_sync_broken(h._h) == 0
    assert float((D - D2).abs().max()) <= 2 * P.TOL_D
