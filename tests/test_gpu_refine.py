"""GPU parity of the NEXT-1 row: sp2_refine_energy (final refinement f_final, Eq. 16, in enhanced
precision; Tr[D H], Tr[D], IdErr) against the FP64 oracle (refine_ref / energy_ref / iderr_ref) and against closed
forms.  Sizes span several 128-tiles, several accumulation chunks (K > 512) and ragged tails."""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W

pytestmark = pytest.mark.gpu

# Enhanced precision: FP16 hi/lo operands as in Eq. 15 and chunked accumulation: the tensor core adds at most
# enh_kc K-blocks into one FP32 accumulator (its adds truncate: each shrinks the running sum by ~0.36 ulp on average;
# a plain layer at N = 16384 chains ~1500 such adds, 6e-5); chunk sums are then added error-free (two-sum pair).
# Library default since round 3: enh_kc = 4 = 48 MMA results per chunk: an entry dominated by one large product loses
# <= ~24 * 0.36 * 2^-23 ~ 1e-6 of its value in the worst case, half of that on average; with |D'_ij| <= 1 and the two
# layers partly compensating (the second squares a nearly idempotent matrix) the bar stays 1e-6 absolute: measured
# 6.8e-7 at most over every case below (3e-7 with enh_kc = 2, the round-2 default, still tested explicitly).
TOL_REFINE = 1e-6


@pytest.fixture(scope="module")
def env(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    torch.cuda.set_device(0)
    h = api.Handle(2304, 0, 120)
    yield api, h, torch
    h.close()


@pytest.mark.parametrize("n", [128, 1100, 1280, 2304])
@pytest.mark.parametrize("last_sigma", [1, -1])
def test_refine_against_closed_form_polynomial(env, n, last_sigma):
    """S = Q diag(s) Q^T with s near 0/1: f_final(S) = Q diag(f(s)) Q^T is known without any product."""
    api, h, torch = env
    rng = np.random.default_rng(100 + n)
    Q = W.haar_orthogonal(rng, n)
    nocc = n // 2
    s = np.concatenate([1.0 - rng.uniform(0, 2e-2, nocc), rng.uniform(0, 2e-2, n - nocc)])
    S64 = (Q * s) @ Q.T
    S32 = np.ascontiguousarray(((S64 + S64.T) / 2).astype(np.float32))
    H32 = np.ascontiguousarray(((Q * np.linspace(-1, 1, n)) @ Q.T).astype(np.float32))
    D, res = h.refine_energy(torch.from_numpy(S32).cuda(), last_sigma, torch.from_numpy(H32).cuda())
    D = D.cpu().numpy().astype(np.float64)
    ref = O.refine_ref(S32, last_sigma)                       # FP64 f_final of the same FP32 input
    f = 2 * s**2 - s**4 if last_sigma < 0 else (2 * s - s**2) ** 2
    closed = (Q * f) @ Q.T                                    # closed form of the unrounded input
    err = np.abs(D - ref).max()
    print(f"refine n={n} sigma={last_sigma}: max|D'-ref|={err:.2e} max|D'-closed|={np.abs(D - closed).max():.2e} "
          f"iderr {res['iderr_in']:.3e} -> {res['iderr_out']:.3e}")
    assert err <= TOL_REFINE
    assert np.abs(D - closed).max() <= 3e-6                   # includes the FP32 rounding of S itself, amplified <= 4x
    assert np.array_equal(D, D.T)                             # exact symmetry
    # observables, FP64 on both sides, of the arrays the library saw / produced
    assert abs(res["trace_in"] - np.trace(S32.astype(np.float64))) <= 1e-9 * n
    assert abs(res["iderr_in"] - O.iderr_ref(S32)) <= 1e-6
    assert abs(res["energy_in"] - O.energy_ref(S32, H32)) <= 1e-5
    assert abs(res["trace_out"] - np.trace(D)) <= 1e-9 * n
    assert abs(res["iderr_out"] - O.iderr_ref(D)) <= 1e-6
    if n == 1280:
        # the accuracy / speed knob: 2 K-blocks per tensor-core chunk (the round-2 default) is tighter, 8 is looser
        errs = {}
        for kc in (2, 8):
            o = api.make_opts()
            o.enh_kc = kc
            Dk, _ = h.refine_energy(torch.from_numpy(S32).cuda(), last_sigma, torch.from_numpy(H32).cuda(), opts=o)
            errs[kc] = np.abs(Dk.cpu().numpy().astype(np.float64) - ref).max()
        print(f"  enh_kc 2 / default 4 / 8: {errs[2]:.2e} / {err:.2e} / {errs[8]:.2e}")
        assert errs[2] <= 5e-7 and errs[2] <= err <= errs[8] + 1e-7
    assert abs(res["energy_out"] - O.energy_ref(D, H32)) <= 1e-5
    assert res["iderr_out"] < 0.05 * res["iderr_in"]          # quadratic: 2e-2 -> <= 4.5 * (2e-2)^2 per eigenvalue


@pytest.mark.parametrize("n,auto", [(1280, False), (1100, True)])
def test_refine_after_solve_improves_energy_and_idempotency(env, n, auto):
    api, h, torch = env
    w = W.config1(3, n=n)
    H = torch.from_numpy(w.H32).cuda()
    opts = api.make_opts(bounds=None if auto else w.bounds, tol=w.tol, max_layers=w.max_layers)
    D0, info = h.density_matrix(H, w.N_occ, opts)
    last_sigma = info["sigma"][-1]
    D1, res = h.refine_energy(D0, last_sigma, H)
    D0n, D1n = D0.cpu().numpy().astype(np.float64), D1.cpu().numpy().astype(np.float64)
    ref = O.refine_ref(D0n, last_sigma)
    Dstar = w.Q[:, : int(w.N_occ)] @ w.Q[:, : int(w.N_occ)].T
    E_star = float(np.sort(w.eps)[: int(w.N_occ)].sum())
    idem0, idem1 = O.idempotency_error(D0n), O.idempotency_error(D1n)
    print(f"solve+refine n={n}: max|D1-ref|={np.abs(D1n - ref).max():.2e} idem {idem0:.2e} -> {idem1:.2e} "
          f"E err {res['energy_in'] - E_star:.3e} -> {res['energy_out'] - E_star:.3e} "
          f"max|D-D*| {np.abs(D0n - Dstar).max():.2e} -> {np.abs(D1n - Dstar).max():.2e}")
    assert np.abs(D1n - ref).max() <= TOL_REFINE
    assert idem1 < idem0                                       # "multiple orders of magnitude in the last layer"
    assert idem1 <= 2e-6
    assert abs(res["energy_out"] - E_star) <= abs(res["energy_in"] - E_star) + 1e-6
    assert np.abs(D1n - Dstar).max() <= 1e-3 and abs(res["trace_out"] - w.N_occ) <= 1e-3 * w.N_occ


def test_refine_errors_and_tiny_sizes(env):
    api, h, torch = env
    S = torch.tensor([[0.999]], dtype=torch.float32, device="cuda")
    Hm = torch.tensor([[-0.5]], dtype=torch.float32, device="cuda")
    D, res = h.refine_energy(S, -1, Hm)
    x = 0.999
    x = float(np.float32(x))
    assert abs(float(D[0, 0]) - (2 * x**2 - x**4)) < 1e-7
    assert abs(res["energy_out"] - (-0.5) * float(D[0, 0])) < 1e-9
    with pytest.raises(api.SP2Error):
        h.refine_energy(S, 0, Hm)
    big = torch.zeros((4096, 4096), dtype=torch.float32, device="cuda")
    with pytest.raises(api.SP2Error):
        h.refine_energy(big, 1, big)                           # larger than the handle's N_max
    with pytest.raises(TypeError):
        h.refine_energy(S.cpu(), 1, Hm)                        # no CPU fallback


def test_enhanced_accumulation_in_every_layer_is_more_accurate(env):
    """tile_config = 4: the whole solve with the chunked tensor-core accumulation (accuracy option, NEXT-4)."""
    api, h, torch = env
    w = W.config1(5, n=2048)
    H = torch.from_numpy(w.H32).cuda()
    Dstar = w.Q[:, : int(w.N_occ)] @ w.Q[:, : int(w.N_occ)].T
    out = {}
    for tile in (1, 4):
        opts = api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=w.max_layers, tile_config=tile)
        D, info = h.density_matrix(H, w.N_occ, opts)
        Dn = D.cpu().numpy().astype(np.float64)
        out[tile] = (np.abs(Dn - Dstar).max(), O.idempotency_error(Dn), abs(np.trace(Dn) - w.N_occ), info["n_layers"])
        assert np.array_equal(Dn, Dn.T) and info["status"] == 0
    print(f"N=2048 plain (err, idem, trace err, layers) {out[1]}  enhanced {out[4]}")
    assert out[4][0] <= 1e-3 and out[4][1] <= 1e-3
    assert out[4][1] < 0.5 * out[1][1] and out[4][2] < 0.5 * out[1][2] + 1e-6
