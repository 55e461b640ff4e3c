"""One small solve per kernel instantiation of the library -- k_sp2_layer<128,1>, <256,1>, <256,2>, <128,1,ENH>,
<128,1,MIX>, <256,2,MIX>, k_sp2_resident<128,1>, <256,2> and every HBM kernel -- each checked against the FP64
oracle.  Sized to run under compute-sanitizer (racecheck / synccheck / memcheck on the hand-written mbarrier, TMEM and
cluster protocols; verdicts under profiles/): several tiles per launch, two rounds where the grid allows, small K."""
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
    h = api.Handle(640, 8, 40)
    yield api, h, torch
    h.close()


@pytest.mark.parametrize("tile", [1, 2, 3, 4])
def test_layer_kernel_instantiation(env, tile):
    api, h, torch = env
    w = W.config1(3, n=600)
    opts = api.make_opts(tol=w.tol, max_layers=40, tile_config=tile, control=2)     # Gershgorin + plain launches
    D, info = h.density_matrix(torch.from_numpy(w.H32).cuda(), w.N_occ, opts)
    Dref, st = O.sp2_ref(w.H32, w.N_occ, info["bounds"], tol=w.tol, max_layers=40)
    P.assert_acceptance(D.cpu().numpy().astype(np.float64), Dref, w.N_occ, f"tile {tile}")
    assert abs(info["n_layers"] - st["n_layers"]) <= 2


@pytest.mark.parametrize("tile", [1, 3])
def test_mix_instantiation(env, tile):
    api, h, torch = env
    w = W.config4(2, n=520, layers=6)
    rng = np.random.default_rng(1)
    theta = O.theta_from_wb(1.0 + rng.normal(0, 0.02, 6), rng.normal(0, 0.005, 6), [1, -1] * 3)
    c = rng.normal(0, 0.2, 7)
    F, _ = h.generalized_mix(torch.from_numpy(w.H32).cuda(), theta, c, bounds=w.bounds, opts=api.make_opts(tile_config=tile))
    assert np.abs(F.cpu().numpy() - O.generalized_mix_ref(w.H32, theta, c, w.bounds)).max() <= 1e-4


def test_refinement_instantiation(env):
    api, h, torch = env
    w = W.config1(4, n=600)
    Hd = torch.from_numpy(w.H32).cuda()
    D, info = h.density_matrix(Hd, w.N_occ, api.make_opts(bounds=w.bounds, tol=1e-3, max_layers=40, tile_config=1))
    D1, res = h.refine_energy(D, info["sigma"][-1], Hd)
    ref = O.refine_ref(D.cpu().numpy().astype(np.float64), info["sigma"][-1])
    assert np.abs(D1.cpu().numpy() - ref).max() <= 1e-6
    assert abs(res["energy_out"] - O.energy_ref(D1.cpu().numpy(), w.H32)) <= 1e-5


@pytest.mark.parametrize("n", [100, 256])
def test_resident_instantiation(env, n):
    api, h, torch = env
    w = W.config5(5, batch=5, n=n)
    D, info = h.density_matrix_batched(torch.from_numpy(w.H32).cuda(), w.N_occ, api.make_opts(tol=w.tol, max_layers=40))
    for m in range(5):
        b = O.gershgorin_bounds(O.symmetrize_lower(w.H32[m]))
        Dref, _ = O.sp2_ref(w.H32[m], w.N_occ, b, tol=w.tol, max_layers=40)
        P.assert_acceptance(D[m].cpu().numpy().astype(np.float64), Dref, w.N_occ, f"matrix {m}")
