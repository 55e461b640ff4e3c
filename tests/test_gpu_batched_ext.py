"""GPU parity of the batched path's generalisations: the accelerated weights of section V.A
 with per-matrix HOMO / LUMO estimates -- repeated small solves in molecular dynamics are that scheme's use
case -- and the generalized network (Eq. 17) applied to a batch, both through the one-launch resident
kernel.  Oracles: sp2_accelerated_ref, sp2_generalized_ref, and the closed forms Q_occ Q_occ^T / Q p(eps) Q^T."""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W
from tests import parity_util as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def benv(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    torch.cuda.set_device(0)
    h = api.Handle(256, 256, 80)
    yield api, h, torch
    h.close()


@pytest.mark.parametrize("n,b,auto", [(256, 150, False), (256, 40, True), (100, 37, False), (128, 64, True)])
def test_batched_accelerated(benv, n, b, auto):
    api, h, torch = benv
    rng = np.random.default_rng(n + b)
    Hs = np.empty((b, n, n), dtype=np.float32)
    hl = np.empty((b, 2))
    ws = []
    for m in range(b):
        k = int(rng.integers(n // 4, 3 * n // 4))
        w = W.gapped_dense(0, n, (-1.0, -0.06), (0.06, 1.0), k, "ba", bounds=(-1.0, 1.0), rng=rng)
        es = np.sort(w.eps)
        g = es[k] - es[k - 1]
        hl[m] = (es[k - 1] + 0.02 * g, es[k] - 0.02 * g)          # estimates 2 % inside the true gap
        Hs[m] = w.H32
        ws.append(w)
    noccs = np.array([w.N_occ for w in ws])
    Hd = torch.from_numpy(Hs).cuda()
    bounds = None if auto else (-1.0, 1.0)
    o_acc = api.make_opts(bounds=bounds, tol=1e-5, max_layers=80)
    D, info = h.density_matrix_batched(Hd, noccs, o_acc, homo_lumo=hl)
    Dp, info_p = h.density_matrix_batched(Hd, noccs, api.make_opts(bounds=bounds, tol=1e-5, max_layers=80))
    assert np.all(info["per_status"] == 0) and np.all(info_p["per_status"] == 0)
    D = D.cpu().numpy().astype(np.float64)
    ratio = info["n_layers"].sum() / info_p["n_layers"].sum()
    print(f"batched accelerated N={n} B={b} auto={auto}: layers {info['n_layers'].mean():.1f} vs plain "
          f"{info_p['n_layers'].mean():.1f} (ratio {ratio:.2f})")
    assert ratio <= 0.85
    for m in range(b):
        P.assert_acceptance(D[m], O.closed_form_density(ws[m].Q, ws[m].N_occ), ws[m].N_occ, f"matrix {m}")
    for m in (0, b // 2, b - 1):
        w = ws[m]
        bm = O.gershgorin_bounds(O.symmetrize_lower(w.H32)) if auto else (-1.0, 1.0)
        Dref, st = O.sp2_accelerated_ref(w.H32, w.N_occ, bm, hl[m, 0], hl[m, 1], tol=1e-5, max_layers=80)
        sg = api.batched_stats(info, m)
        P.assert_acceptance(D[m], Dref, w.N_occ, f"matrix {m} vs accelerated oracle")
        P.branch_prefix_check(sg, st, w.N_occ)
        assert abs(int(info["n_layers"][m]) - st["n_layers"]) <= 2
        k = min(len(sg["trace_S"]), len(st["trace_S"]))
        nstar, mism = P.branch_prefix_check(sg, st, w.N_occ)
        kk = k if mism is None else mism
        assert np.abs(np.array(sg["trace_S"][:kk]) - np.array(st["trace_S"][:kk])).max() <= 1e-3 * max(1.0, w.N_occ)


def test_batched_accelerated_argument_errors(benv):
    api, h, torch = benv
    w = W.config1(0, n=64)
    Hd = torch.from_numpy(np.stack([w.H32] * 3)).cuda()
    with pytest.raises(api.SP2Error) as e:       # accelerated without estimates
        h.density_matrix_batched(Hd, 32.0, api.make_opts(bounds=w.bounds, accelerated=1))
    assert e.value.status == -1
    with pytest.raises(api.SP2Error) as e:       # lumo <= homo
        h.density_matrix_batched(Hd, 32.0, api.make_opts(bounds=w.bounds), homo_lumo=np.array([[0.1, -0.1]] * 3))
    assert e.value.status == -1
    with pytest.raises(api.SP2Error) as e:       # estimates outside the caller's bounds
        h.density_matrix_batched(Hd, 32.0, api.make_opts(bounds=w.bounds), homo_lumo=np.array([[-2.0, 0.05]] * 3))
    assert e.value.status == -1


@pytest.mark.parametrize("n,b", [(200, 19), (256, 80), (64, 33)])
def test_batched_generalized_network(benv, n, b):
    """Config-4-shaped networks (gapless spectra, per-layer branch + weight + bias scalars, reading C19) on a batch:
    X_L against Q diag(p(eps)) Q^T for every matrix and against the FP64 matrix oracle for a few."""
    api, h, torch = benv
    L = 14
    rng = np.random.default_rng(7 * n + b)
    sig = np.array([1, -1] * (L // 2))
    theta = O.theta_from_wb(1.0 + rng.normal(0, 0.02, L), rng.normal(0, 0.005, L), sig)
    Hs = np.empty((b, n, n), dtype=np.float32)
    ws = []
    for m in range(b):
        w = W.config4(1000 * n + m, n=n, layers=L)
        Hs[m] = w.H32
        ws.append(w)
    X, info = h.generalized_batched(torch.from_numpy(Hs).cuda(), theta, bounds=(-1.0, 1.0))
    assert np.all(info["per_status"] == 0)
    X = X.cpu().numpy().astype(np.float64)
    for m in range(b):
        p = O.scalar_generalized(ws[m].eps, theta, -1.0, 1.0)
        assert np.abs(X[m] - (ws[m].Q * p) @ ws[m].Q.T).max() <= P.TOL_D, f"matrix {m}"
        assert np.array_equal(X[m], X[m].T)
        sg = api.batched_stats(info, m)
        assert abs(sg["trace_S"][-1] - p.sum()) <= 1e-3 * n
    for m in (0, b - 1):
        Xref, st = O.sp2_generalized_ref(Hs[m], theta, (-1.0, 1.0))
        assert np.abs(X[m] - Xref).max() <= 1e-4
        assert np.allclose(api.batched_stats(info, m)["trace_S"], st["trace_S"], atol=1e-3)
    # Gershgorin bounds per matrix (eps_min >= eps_max) against the oracle's own
    Xa, ia = h.generalized_batched(torch.from_numpy(Hs[:4].copy()).cuda(), theta)
    for m in range(4):
        Xref, _ = O.sp2_generalized_ref(Hs[m], theta, None)
        assert np.abs(Xa[m].cpu().numpy() - Xref).max() <= 1e-4
