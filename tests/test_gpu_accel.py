"""GPU parity of the NEXT-3 row: sp2_density_matrix with opts.accelerated (section V.A; reading C27)
against the FP64 oracle sp2_accelerated_ref and the closed-form density matrix."""
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
    h = api.Handle(4096, 8, 120)
    yield api, h, torch
    h.close()


def _estimates(w, inside=0.01):
    nocc = int(w.N_occ)
    e = np.sort(w.eps)
    g = e[nocc] - e[nocc - 1]
    return e[nocc - 1] + inside * g, e[nocc] - inside * g


@pytest.mark.parametrize("n,seed,auto,tile", [(128, 0, False, 0), (128, 1, True, 0), (640, 2, False, 1),
                                              (1100, 3, True, 1), (2048, 4, False, 3)])
def test_accelerated_matches_oracle_and_saves_layers(env, n, seed, auto, tile):
    api, h, torch = env
    w = W.config1(seed, n=n)
    Hd = torch.from_numpy(w.H32).cuda()
    hl = _estimates(w)
    bounds = None if auto else w.bounds
    std = api.make_opts(bounds=bounds, tol=w.tol, max_layers=w.max_layers, tile_config=tile)
    acc = api.make_opts(bounds=bounds, tol=w.tol, max_layers=w.max_layers, tile_config=tile, homo_lumo=hl)
    D0, i0 = h.density_matrix(Hd, w.N_occ, std)
    D1, i1 = h.density_matrix(Hd, w.N_occ, acc)
    used = i1["bounds"]
    Dref, st = O.sp2_accelerated_ref(w.H32, w.N_occ, used, hl[0], hl[1], tol=w.tol, max_layers=w.max_layers)
    D = D1.cpu().numpy().astype(np.float64)
    nocc = int(w.N_occ)
    Dstar = w.Q[:, :nocc] @ w.Q[:, :nocc].T
    err, idem, tr = np.abs(D - Dref).max(), O.idempotency_error(D), abs(np.trace(D) - w.N_occ)
    print(f"accel n={n} auto={auto}: layers std {i0['n_layers']} acc {i1['n_layers']} (oracle {st['n_layers']}) "
          f"max|D-Dref|={err:.2e} max|D-D*|={np.abs(D - Dstar).max():.2e} idem={idem:.2e} |tr-Nocc|={tr:.2e} "
          f"stop={i1['stop_reason']}")
    assert i1["status"] == 0
    assert err <= P.TOL_D and np.abs(D - Dstar).max() <= P.TOL_D
    assert tr <= P.TOL_TRACE_REL * w.N_occ and idem <= P.TOL_IDEM
    assert np.array_equal(D, D.T)
    assert i1["n_layers"] <= 0.85 * i0["n_layers"]                 # the point of the scheme (Fig. 5: 28 -> 17)
    assert abs(i1["n_layers"] - st["n_layers"]) <= 2               # noise-floor stop vs FP64 tol stop (C6 / C8 / C25)
    # branch sequence: identical to the oracle's wherever the oracle's decision margin is above the trace noise
    k = min(i1["n_layers"], st["n_layers"])
    for j in range(k):
        if abs(st["margin"][j]) <= 5e-4 * max(1.0, w.N_occ):
            break
        assert i1["sigma"][j] == st["sigma"][j], f"layer {j + 1}"
        assert abs(i1["trace_S"][j] - st["trace_S"][j]) <= 1e-3 * max(1.0, w.N_occ)


def test_accelerated_argument_checks(env):
    api, h, torch = env
    w = W.config1(0)
    Hd = torch.from_numpy(w.H32).cuda()
    for hl in [(0.1, -0.1), (0.0, 0.0), (-5.0, 0.05), (float("nan"), 0.1)]:
        with pytest.raises(api.SP2Error):
            h.density_matrix(Hd, w.N_occ, api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=60, homo_lumo=hl))
    # estimates outside Gershgorin bounds are detected on the device
    with pytest.raises(api.SP2Error):
        h.density_matrix(Hd, w.N_occ, api.make_opts(bounds=None, tol=w.tol, max_layers=60, homo_lumo=(-50.0, 60.0)))
    # batched call: not available
    Hb = torch.from_numpy(np.stack([w.H32] * 2)).cuda()
    with pytest.raises(api.SP2Error):
        h.density_matrix_batched(Hb, w.N_occ, api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=60,
                                                            homo_lumo=_estimates(w)))
    # a = 1 limit: estimates at the spectral bounds' ends give plain Alg. 1's branch polynomials
    o = api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=60, homo_lumo=(w.bounds[0], w.bounds[1]))
    D1, i1 = h.density_matrix(Hd, w.N_occ, o)
    D0, i0 = h.density_matrix(Hd, w.N_occ, api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=60))
    assert i1["sigma"][: min(i0["n_layers"], i1["n_layers"]) - 1] == i0["sigma"][: min(i0["n_layers"], i1["n_layers"]) - 1]
    assert np.abs(D1.cpu().numpy() - D0.cpu().numpy()).max() <= 1e-4
