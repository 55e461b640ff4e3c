"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle, element by element on the same
seeded inputs (BASELINE configs 1, 2, 4 in full; ragged and edge sizes).  Tolerances are BASELINE north_star's."""
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
    h = api.Handle(4096, 0, 200)
    yield api, h, torch
    h.close()


def _solve(env, w, bounds, **kw):
    api, h, torch = env
    opts = api.make_opts(bounds=bounds, tol=w.tol, max_layers=w.max_layers, **kw)
    D, info = h.density_matrix(torch.from_numpy(w.H32).cuda(), w.N_occ, opts)
    return D.cpu().numpy().astype(np.float64), info


@pytest.mark.parametrize("control", [0, 1, 2, 3])
@pytest.mark.parametrize("tile", [1, 2, 3, 4])
def test_config1_all_tiles_and_control_modes(env, tile, control):
    """BASELINE configs[0] (N=128, explicit bounds): every tile configuration and control mode gives the same
    result; D, trace, idempotency within tolerance; branch sequence per reading C6."""
    w = W.config1(0)
    D, info = _solve(env, w, w.bounds, tile_config=tile, control=control)
    Dref, st = O.sp2_ref(w.H32, w.N_occ, w.bounds, tol=w.tol, max_layers=w.max_layers)
    P.assert_acceptance(D, Dref, w.N_occ, f"tile{tile}/ctl{control}")
    P.branch_prefix_check(info, st, w.N_occ)
    P.replay_check(info, w.H32, w.N_occ, w.bounds, eigs=w.eps)
    assert abs(info["n_layers"] - st["n_layers"]) <= 2
    assert info["stop_reason"] in (1, 2, 3, 6)
    assert info["status"] == 0


@pytest.mark.parametrize("seed", [0, 1, 2])
@pytest.mark.parametrize("auto", [False, True])
def test_config1_seeds_auto_and_explicit_bounds(env, seed, auto):
    w = W.config1(seed)
    D, info = _solve(env, w, None if auto else w.bounds)
    used = info["bounds"]
    if auto:   # C3: device Gershgorin vs the oracle's, then iterate the oracle from the GPU's exact bounds
        g = O.gershgorin_bounds(O.symmetrize_lower(w.H32))
        assert abs(used[0] - g[0]) <= 1e-5 * abs(g[0]) and abs(used[1] - g[1]) <= 1e-5 * abs(g[1])
        assert used[0] <= w.eps.min() and w.eps.max() <= used[1]
    Dref, st = O.sp2_ref(w.H32, w.N_occ, used, tol=w.tol, max_layers=w.max_layers)
    P.assert_acceptance(D, Dref, w.N_occ)
    assert np.abs(D - O.closed_form_density(w.Q, w.N_occ)).max() <= P.TOL_D
    P.branch_prefix_check(info, st, w.N_occ)
    P.replay_check(info, w.H32, w.N_occ, used, eigs=w.eps)


@pytest.mark.parametrize("n,tile", [(3000, 3), (3500, 3), (3000, 1)])
def test_ragged_sizes_with_several_rounds_and_tail_strips(env, n, tile):
    """More work items than CTA slots, ragged N, and a last partial round that the host cuts into column strips
    (256-pair tiles: N = 3000 -> 78 tiles on 74 slots, 4 left over -> 16 strips of 64 columns; N = 3500 -> 105 tiles,
    31 left over -> 62 strips of 128; 128-tiles at N = 3000 -> 300 tiles on 148 slots, 4 left over -> 8 strips of 64).
    The closed form D* = Q_occ Q_occ^T is the reference; the FP64 oracle is compared through the scalar recursion."""
    api, h, torch = env
    k = n // 2
    w = W.gapped_dense(n, n, (-1.0, -0.15), (0.15, 1.0), k, "ragged-rounds", bounds=(-1.0, 1.0))
    opts = api.make_opts(bounds=w.bounds, tol=1e-5, max_layers=80, tile_config=tile)
    D, info = h.density_matrix(torch.from_numpy(w.H32).cuda(), float(k), opts)
    D = D.cpu().numpy().astype(np.float64)
    Dstar = O.closed_form_density(w.Q, w.N_occ)
    st = O.scalar_recursion(w.eps, w.N_occ, -1.0, 1.0, tol=1e-5, max_layers=80)
    print(f"N={n} tile={tile}: layers {info['n_layers']}/{st['n_layers']} max|D-D*|={np.abs(D - Dstar).max():.2e}")
    P.assert_acceptance(D, Dstar, float(k), f"N={n} tile={tile}")
    assert np.array_equal(D, D.T)
    assert abs(info["n_layers"] - st["n_layers"]) <= 2
    P.branch_prefix_check(info, st, w.N_occ)
    P.replay_check(info, None, w.N_occ, (-1.0, 1.0), eigs=w.eps)


@pytest.mark.parametrize("n", [1, 2, 10, 100, 127, 129, 300, 777])
def test_ragged_and_tiny_sizes(env, n):
    """Sizes that are not a multiple of the tile (padding of S_0 must be inert), several tiles + ragged tail."""
    api, h, torch = env
    rng = np.random.default_rng(n)
    k = n // 2
    if n == 1:
        H32 = np.array([[0.3]], dtype=np.float32)
        k = 1
    else:
        w = W.gapped_dense(n, n, (-1.0, -0.2), (0.2, 1.0), k, "ragged", bounds=(-1.0, 1.0))
        H32 = w.H32
    opts = api.make_opts(bounds=(-1.0, 1.0), tol=1e-5, max_layers=80)
    D, info = h.density_matrix(torch.from_numpy(H32).cuda(), float(k), opts)
    D = D.cpu().numpy().astype(np.float64)
    Dref, st = O.sp2_ref(H32, float(k), (-1.0, 1.0), tol=1e-5, max_layers=80)
    P.assert_acceptance(D, Dref, float(k), f"N={n}")
    assert abs(info["n_layers"] - st["n_layers"]) <= 2


def test_config2_tight_binding(env):
    """BASELINE configs[1] (N=2048, Gershgorin bounds, gap ~1e-3): hardest conditioning (C14)."""
    w = W.config2(0)
    D, info = _solve(env, w, None)
    used = info["bounds"]
    g = O.gershgorin_bounds(O.symmetrize_lower(w.H32))
    assert abs(used[0] - g[0]) <= 1e-5 * abs(g[0]) and abs(used[1] - g[1]) <= 1e-5 * abs(g[1])
    Dref, st = O.sp2_ref(w.H32, w.N_occ, used, tol=w.tol, max_layers=w.max_layers)
    De, E = O.eig_density(w.H32, w.N_occ)
    k = int(w.N_occ)
    print(f"config2: gap={E[k] - E[k - 1]:.3e} layers gpu/oracle={info['n_layers']}/{st['n_layers']} "
          f"stop={info['stop_reason']}/{st['stop_reason']} err_vs_oracle={np.abs(D - Dref).max():.2e} "
          f"err_vs_eig={np.abs(D - De).max():.2e}")
    P.assert_acceptance(D, Dref, w.N_occ, "config2")
    assert np.abs(D - De).max() <= P.TOL_D
    P.branch_prefix_check(info, st, w.N_occ)
    P.replay_check(info, w.H32, w.N_occ, used, eigs=E)


def test_config4_generalized_network(env):
    """BASELINE configs[3]: N=4096 gapless, 30 layers with branch + weight + bias per layer; X_L against the same
    scalar recursion on H's eigenvalues (X_L = Q diag(p(eps)) Q^T) and against the FP64 matrix oracle."""
    api, h, torch = env
    w = W.config4(0)
    L = w.extra["layers"]
    sig = O.scalar_recursion(w.eps, w.N_occ, *w.bounds, max_layers=L)["sigma"]
    sig = (sig + [1, -1] * L)[:L]                      # C19: branch from the trace rule on the scalar recursion
    X, info = h.generalized_wb(torch.from_numpy(w.H32).cuda(), sig, w.extra["weights"], w.extra["biases"],
                               bounds=w.bounds)
    X = X.cpu().numpy().astype(np.float64)
    theta = O.theta_from_wb(w.extra["weights"], w.extra["biases"], sig)
    p = O.scalar_generalized(w.eps, theta, *w.bounds)
    Xs = (w.Q * p) @ w.Q.T
    err = np.abs(X - Xs).max()
    print(f"config4: max|X_L - Q p(eps) Q^T| = {err:.2e}; trace {info['trace_S'][-1]:.4f} vs {p.sum():.4f}")
    assert err <= P.TOL_D
    assert abs(info["trace_S"][-1] - p.sum()) <= 1e-3 * w.N_occ
    assert np.array_equal(X, X.T)
    # per-layer traces against the scalar recursion
    lam = O.scalar_initial(w.eps, *w.bounds)
    for n in range(L):
        lam = theta[n, 0] * lam * lam + theta[n, 1] * lam + theta[n, 2]
        assert abs(info["trace_S"][n] - lam.sum()) <= 1e-3 * w.N_occ
    Xref, _ = O.sp2_generalized_ref(w.H32[:512, :512], theta, (-1.2, 1.2))   # matrix oracle on a 512 block
    X5, _ = h.generalized(torch.from_numpy(np.ascontiguousarray(w.H32[:512, :512])).cuda(), theta, bounds=(-1.2, 1.2))
    assert np.abs(X5.cpu().numpy() - Xref).max() <= P.TOL_D


def test_generalized_theta_and_bias_on_padded_size(env):
    """theta_3 I must touch only the first N diagonal entries when N is padded (N=200 -> 256)."""
    api, h, torch = env
    w = W.config4(1, n=200, layers=12)
    rng = np.random.default_rng(5)
    sig = np.array([1, -1] * 6)
    theta = O.theta_from_wb(1.0 + rng.normal(0, 0.03, 12), rng.normal(0, 0.01, 12), sig)
    X, info = h.generalized(torch.from_numpy(w.H32).cuda(), theta, bounds=w.bounds)
    Xref, st = O.sp2_generalized_ref(w.H32, theta, w.bounds)
    assert np.abs(X.cpu().numpy() - Xref).max() <= 1e-4
    assert np.allclose(info["trace_S"], st["trace_S"], atol=1e-3)


def test_single_layer_square_within_fp32_accumulation_bound(env):
    """Row a4: one layer with theta = (1,0,0) from S_0 = X (H = -X, bounds (-1,0)) is Eq. 15.  The exact target is
    hi hi + hi lo + (hi lo)^T evaluated in FP64 from the same hi/lo bits; the tensor-core result must be within
    an FP32 accumulation bound: 3K/16 MMA accumulations, each losing at most one ulp (2^-23) of the running sum
    (the tensor core truncates rather than rounds), i.e. (3K/16) 2^-23 (|hi||hi| + 2|hi||lo|); and exactly symmetric."""
    api, h, torch = env
    for n, k in [(384, 13), (1024, 13), (1024, 0)]:
        rng = np.random.default_rng(n)
        A = rng.uniform(-1, 1, (n, n)) / np.sqrt(n)
        X = (0.5 * (A + A.T)).astype(np.float32)
        opts = api.make_opts(fp16_scale_log2=k)
        Y, info = h.generalized(torch.from_numpy(-X).cuda(), np.array([[1.0, 0.0, 0.0]]), bounds=(-1.0, 0.0), opts=opts)
        Y = Y.cpu().numpy().astype(np.float64)
        hi, lo = O.split_fp16(X * np.float32(2.0 ** k))
        C = O.mixed_square_exact(hi, lo) * 2.0 ** (-2 * k)
        ah, al = np.abs(hi.astype(np.float64)), np.abs(lo.astype(np.float64))
        bound = 2.0 * (3 * n / 16) * 2.0 ** -24 * (ah @ ah + 2 * ah @ al) * 2.0 ** (-2 * k) + 1e-30
        assert np.all(np.abs(Y - C) <= bound), f"N={n} k={k}: {np.abs(Y - C).max()} vs bound {bound.max()}"
        assert np.array_equal(Y, Y.T)
        assert abs(info["trace_X_diag"][0] - np.trace(C)) <= np.trace(bound)     # the tensor core truncates: bias < 0
        X64 = X.astype(np.float64)
        assert abs(info["trace_X"][0] - np.sum(X64 * X64)) <= 1e-9 * n     # FP64 pre-trace ||S||_F^2


def test_split_bit_exact(env):
    """Row a3: hi/lo bit patterns identical to the IEEE RNE restatement (Eqs. 12-13, C9), scaled and unscaled,
    vector and scalar paths, subnormal range included."""
    api, h, torch = env
    rng = np.random.default_rng(0)
    for n in (64, 257, 1024):
        X = (rng.standard_normal((n, n)) * 10.0 ** rng.uniform(-7, 0, (n, n))).astype(np.float32)
        X[0, 0] = 1.0 + 2.0 ** -11          # exact tie
        for k in (0, 13):
            hi, lo = api.split_fp16(torch.from_numpy(X).cuda(), k)
            rh, rl = O.split_fp16(X * np.float32(2.0 ** k))
            assert np.array_equal(hi.cpu().numpy().view(np.uint16), rh.view(np.uint16))
            assert np.array_equal(lo.cpu().numpy().view(np.uint16), rl.view(np.uint16))


def test_gershgorin_matches_oracle(env):
    api, h, torch = env
    for n in (3, 64, 65, 1000, 2048):
        Hs = W.uniform_symmetric(n, n)
        Hs[np.triu_indices(n, 1)] += 0.25      # make the upper triangle disagree: only the lower one may be read
        g = h.gershgorin(torch.from_numpy(Hs).cuda())
        r = O.gershgorin_bounds(O.symmetrize_lower(Hs))
        assert abs(g[0] - r[0]) <= 1e-5 * abs(r[0]) and abs(g[1] - r[1]) <= 1e-5 * abs(r[1])


def test_edge_cases_and_errors(env):
    api, h, torch = env
    w = W.config1(0)
    Hd = torch.from_numpy(w.H32).cuda()
    # N_occ = 0 and N_occ = N (C18)
    for nocc, target in [(0.0, np.zeros((128, 128))), (128.0, np.eye(128))]:
        D, info = h.density_matrix(Hd, nocc, api.make_opts(bounds=(-1.0, 1.0), tol=1e-6, max_layers=100))
        assert np.abs(D.cpu().numpy() - target).max() <= P.TOL_D
    # max_layers reached -> flagged, D = S_max_layers
    D, info = h.density_matrix(Hd, 64.0, api.make_opts(bounds=(-1.0, 1.0), tol=1e-5, max_layers=5))
    assert info["status"] == api.SP2_NOT_CONVERGED and info["n_layers"] == 5 and info["stop_reason"] == 4
    Dref, st = O.sp2_ref(w.H32, 64.0, (-1.0, 1.0), tol=1e-5, max_layers=5)
    assert np.abs(D.cpu().numpy() - Dref).max() <= 1e-4 and info["sigma"] == st["sigma"]
    # degenerate bounds
    with pytest.raises(api.SP2Error) as e:
        h.density_matrix(Hd, 64.0, api.make_opts(bounds=(1.0, 1.0)))
    assert e.value.status == -2
    Hi = torch.eye(64, device="cuda") * 0.5
    with pytest.raises(api.SP2Error) as e:
        h.density_matrix(Hi, 32.0, api.make_opts())          # Gershgorin of a multiple of I
    assert e.value.status == -2
    with pytest.raises(api.SP2Error) as e:
        h.density_matrix(Hd, 500.0, api.make_opts(bounds=(-1.0, 1.0)))
    assert e.value.status == -1
    with pytest.raises(api.SP2Error) as e:
        h.density_matrix(torch.zeros((8192, 8192), device="cuda"), 1.0, api.make_opts(bounds=(-1.0, 1.0)))
    assert e.value.status == -4
    with pytest.raises(TypeError):
        h.density_matrix(torch.from_numpy(w.H32), 64.0)       # CPU tensor: no fallback
    # tie rule C4 on the device: 2x2 with symmetric spectrum
    H2 = torch.tensor([[0.0, 0.5], [0.5, 0.0]], device="cuda")
    D, info = h.density_matrix(H2, 1.0, api.make_opts(bounds=(-1.0, 1.0), tol=1e-7, max_layers=60))
    assert info["sigma"][0] == 1
    assert np.abs(D.cpu().numpy() - 0.5 * np.array([[1, -1], [-1, 1]])).max() <= 1e-4
    # leading dimensions larger than N on both sides
    big = torch.zeros((128, 200), device="cuda"); big[:, :128] = Hd
    out = torch.full((128, 160), 7.0, device="cuda")
    o1 = api.make_opts(bounds=(-1.0, 1.0), tol=1e-5, max_layers=60, tile_config=1)
    D2, _ = h.density_matrix(big[:, :128], 64.0, o1, out=out[:, :128])
    D1, i1 = h.density_matrix(Hd, 64.0, o1)
    assert torch.equal(D1, out[:, :128]) and float(out[:, 128:].min()) == 7.0
    # small contiguous problems with default options take the one-launch resident kernel; strided ones the tiled
    # kernels: same result within the arithmetic's noise, same branch sequence
    o0 = api.make_opts(bounds=(-1.0, 1.0), tol=1e-5, max_layers=60)
    D0, i0 = h.density_matrix(Hd, 64.0, o0)
    D3, i3 = h.density_matrix(big[:, :128], 64.0, o0)
    assert i0["launches"] == 1 and i3["launches"] > 1
    k = min(i0["n_layers"], i3["n_layers"]) - 1
    assert i0["sigma"][:k] == i3["sigma"][:k]
    assert float((D0 - D3).abs().max()) <= 1e-5 and torch.equal(D0, D0.T)


@pytest.mark.parametrize("n,tile", [(1024, 0), (3000, 1), (3000, 0)])
@pytest.mark.parametrize("auto", [False, True])
def test_tiled_kernel_bit_reproducible_and_host_entry(env, n, tile, auto):
    """The TILED layer kernel (N > 256; 128 x 128 tiles: one round at N = 1024 -- the default choice there --, three rounds
    with the round sync and the reversed K walk at N = 3000; and the default at N = 3000, 2-CTA pair tiles, two rounds): two runs give identical
    bits -- D, bounds and every per-layer trace -- with caller bounds and with the device's Gershgorin bounds, and
    the host-buffer entry point returns the same bits as the device one."""
    api, h, torch = env
    k = n // 2
    w = W.gapped_dense(n + 7, n, (-1.0, -0.15), (0.15, 1.0), k, "det", bounds=(-1.0, 1.0))
    opts = api.make_opts(bounds=None if auto else w.bounds, tol=1e-5, max_layers=100, tile_config=tile)
    Hd = torch.from_numpy(w.H32).cuda()
    D1, i1 = h.density_matrix(Hd, w.N_occ, opts)
    assert i1["launches"] > 2                                   # not the one-launch resident path
    D2, i2 = h.density_matrix(Hd, w.N_occ, opts)
    assert torch.equal(D1, D2) and i1["bounds"] == i2["bounds"]
    for key in ("trace_S", "trace_X", "trace_X_diag", "iderr", "sigma", "stop_reason"):
        assert i1[key] == i2[key], key
    Dh, ih = h.density_matrix_host(w.H32, w.N_occ, opts)
    assert np.array_equal(Dh, D1.cpu().numpy()) and ih["trace_S"] == i1["trace_S"] and ih["bounds"] == i1["bounds"]
    # the host entry point copies the lower triangle only (bands of 256 rows, N > 1024): a poisoned upper triangle of
    # the host matrix changes nothing, and the reported byte counts are those of the copies
    Hp = w.H32.copy()
    Hp[np.triu_indices(n, 1)] = np.nan
    Dp, ip = h.density_matrix_host(Hp, w.N_occ, opts)
    assert np.array_equal(Dp, Dh) and ip["trace_S"] == ih["trace_S"]
    assert ip["d2h_bytes"] == 4 * n * n
    if n > 1024:
        bands = [(r0, min(n, r0 + 256)) for r0 in range(0, n, 256)]
        assert ip["h2d_bytes"] == sum(4 * r1 * (r1 - r0) for r0, r1 in bands) < 0.6 * 4 * n * n
    else:
        assert ip["h2d_bytes"] == 4 * n * n
    P.assert_acceptance(D1.cpu().numpy().astype(np.float64), O.closed_form_density(w.Q, w.N_occ), w.N_occ, f"N={n}")


@pytest.mark.parametrize("n,tile", [(1024, 0), (2048, 0), (3000, 1), (3000, 0), (4096, 0)])
def test_persistent_launch_gives_the_graph_loop_bits(env, n, tile):
    """control = 3: ONE cooperative launch runs every layer (grid barrier between layers, the operand pairs swapped per
    layer inside the kernel) -- the same tiles in the same order as the graph's WHILE loop, so the same bits, with
    caller and with Gershgorin bounds, one to three rounds, single-CTA and pair tiles."""
    api, h, torch = env
    w = W.gapped_dense(n + 3, n, (-1.0, -0.15), (0.15, 1.0), n // 2, "persist", bounds=(-1.0, 1.0))
    Hd = torch.from_numpy(w.H32).cuda()
    for bounds in (w.bounds, None):
        o0 = api.make_opts(bounds=bounds, tol=1e-5, max_layers=100, tile_config=tile, control=0)
        o3 = api.make_opts(bounds=bounds, tol=1e-5, max_layers=100, tile_config=tile, control=3)
        D0, i0 = h.density_matrix(Hd, w.N_occ, o0)
        D3, i3 = h.density_matrix(Hd, w.N_occ, o3)
        assert i3["n_layers"] == i0["n_layers"] and i3["sigma"] == i0["sigma"] and i3["stop_reason"] == i0["stop_reason"]
        assert i3["trace_S"] == i0["trace_S"] and i3["iderr"] == i0["iderr"]
        assert torch.equal(D0, D3)
    # a solve that ends on max_layers, and the exact_diag = 0 variant
    o3 = api.make_opts(bounds=w.bounds, tol=1e-5, max_layers=7, tile_config=tile, control=3, exact_diag=0)
    o0 = api.make_opts(bounds=w.bounds, tol=1e-5, max_layers=7, tile_config=tile, control=0, exact_diag=0)
    D3, i3 = h.density_matrix(Hd, w.N_occ, o3)
    D0, i0 = h.density_matrix(Hd, w.N_occ, o0)
    assert i3["n_layers"] == 7 and i3["status"] == api.SP2_NOT_CONVERGED and torch.equal(D0, D3)


def test_round_sync_timeout_path_gives_the_same_bits(env, monkeypatch):
    """The round synchronisation of the layer kernel is an optimisation with a bounded wait: when a wait runs out
    (CTAs not co-resident) the kernel gives the sync up for the rest of the solve.  Forced here with a wait bound of
    one poll (SP2_ROUND_SYNC_SPINS, a performance toggle read at sp2_create) and a sync point every four K-blocks
    (SP2_K_INTERLEAVE): same bits as the synchronised run."""
    api, h, torch = env
    n = 3000
    w = W.gapped_dense(11, n, (-1.0, -0.15), (0.15, 1.0), n // 2, "rs", bounds=(-1.0, 1.0))
    Hd = torch.from_numpy(w.H32).cuda()
    for tile in (1, 3):
        opts = api.make_opts(bounds=w.bounds, tol=1e-5, max_layers=100, tile_config=tile)
        D0, i0 = h.density_matrix(Hd, w.N_occ, opts)
        assert h.lib.sp2_last_round_sync_broken(h._h) == 0
        monkeypatch.setenv("SP2_ROUND_SYNC_SPINS", "1")
        monkeypatch.setenv("SP2_K_INTERLEAVE", "4:4")      # a sync point every 4 K-blocks (the default chunking has
        h2 = api.Handle(n, 0, 100)                          # none at this K; the bits do not depend on it)
        monkeypatch.delenv("SP2_ROUND_SYNC_SPINS")
        monkeypatch.delenv("SP2_K_INTERLEAVE")
        D1, i1 = h2.density_matrix(Hd, w.N_occ, opts)
        broken = h2.lib.sp2_last_round_sync_broken(h2._h)
        h2.close()
        assert broken == 1, "the timeout path was not taken"
        assert torch.equal(D0, D1) and i0["trace_S"] == i1["trace_S"] and i0["sigma"] == i1["sigma"]


@pytest.mark.parametrize("n,tile", [(3000, 1), (3000, 3), (4500, 1), (5000, 3)])
def test_k_interleave_chunking_gives_the_same_bits(env, monkeypatch, n, tile):
    """The K-interleave of the layer kernel (the two rounds of an epoch walk K in alternating chunks so that their
    operand panels are shared through L2; SP2_K_INTERLEAVE = edge[:mid] K-blocks per chunk, read at sp2_create) only
    changes WHEN a tile's MMAs are issued, never their order within the tile: off (one tile after the other), the
    default chunking and two odd chunkings (chunks that do not divide K, more chunks than K-blocks at one end) must
    give identical bits.  Several epochs, a partial last epoch (a first tile without a second one), pair and
    single-CTA tiles, ragged N."""
    api, h, torch = env
    w = W.gapped_dense(n + 5, n, (-1.0, -0.15), (0.15, 1.0), n // 2, "ki", bounds=(-1.0, 1.0))
    Hd = torch.from_numpy(w.H32).cuda()
    opts = api.make_opts(bounds=w.bounds, tol=1e-5, max_layers=100, tile_config=tile)
    h0 = api.Handle(n, 0, 100)
    D0, i0 = h0.density_matrix(Hd, w.N_occ, opts)                      # default chunking
    h0.close()
    for ki in ("0", "5:3", "40:7", "1000"):
        monkeypatch.setenv("SP2_K_INTERLEAVE", ki)
        h2 = api.Handle(n, 0, 100)
        monkeypatch.delenv("SP2_K_INTERLEAVE")
        D1, i1 = h2.density_matrix(Hd, w.N_occ, opts)
        h2.close()
        assert torch.equal(D0, D1), ki
        assert i0["trace_S"] == i1["trace_S"] and i0["trace_X_diag"] == i1["trace_X_diag"] and i0["sigma"] == i1["sigma"], ki
    P.assert_acceptance(D0.cpu().numpy().astype(np.float64), O.closed_form_density(w.Q, w.N_occ), w.N_occ, f"N={n}")


def test_nonfinite_input_and_unsupported_mix_tile(env):
    """A NaN in H must surface as SP2_ERR_NONFINITE from every single-matrix entry point (standard and generalized,
    caller and Gershgorin bounds); the output mix has no enhanced-accumulation instantiation -> SP2_ERR_INVALID_ARG."""
    api, h, torch = env
    w = W.config1(0, n=384)
    Hn = torch.from_numpy(w.H32).cuda()
    Hn[100, 3] = float("nan")
    theta = np.array([[1.0, 0.0, 0.0], [-1.0, 2.0, 0.0], [1.0, 0.0, 0.0]])
    for bounds in (w.bounds, None):
        with pytest.raises(api.SP2Error) as e:
            h.density_matrix(Hn, w.N_occ, api.make_opts(bounds=bounds, tol=1e-5, max_layers=30))
        assert e.value.status == -3
        with pytest.raises(api.SP2Error) as e:
            h.generalized(Hn, theta, bounds=bounds)
        assert e.value.status == -3
    with pytest.raises(api.SP2Error) as e:
        h.generalized_mix(torch.from_numpy(w.H32).cuda(), theta, np.array([0.1, 0.2, 0.3, 0.4]), bounds=w.bounds,
                          opts=api.make_opts(tile_config=4))
    assert e.value.status == -1


def test_host_buffer_entry_point_and_determinism(env):
    api, h, torch = env
    w = W.config1(1, n=256)
    opts = api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=w.max_layers)
    Dh, info_h = h.density_matrix_host(w.H32, w.N_occ, opts)
    Dd, info_d = h.density_matrix(torch.from_numpy(w.H32).cuda(), w.N_occ, opts)
    assert np.array_equal(Dh, Dd.cpu().numpy())
    Dd2, info_d2 = h.density_matrix(torch.from_numpy(w.H32).cuda(), w.N_occ, opts)
    assert torch.equal(Dd, Dd2) and info_d["trace_S"] == info_d2["trace_S"] and info_d["iderr"] == info_d2["iderr"]


def test_literal_eq13_split_still_within_tolerance(env):
    """fp16_scale_log2 = 0 is Eq. 13 literally (X1 may fall into FP16 subnormals, reading C10)."""
    api, h, torch = env
    w = W.config1(0, n=512)
    for k in (0, 13):
        opts = api.make_opts(bounds=w.bounds, tol=w.tol, max_layers=w.max_layers, fp16_scale_log2=k)
        D, info = h.density_matrix(torch.from_numpy(w.H32).cuda(), w.N_occ, opts)
        Dref = O.closed_form_density(w.Q, w.N_occ)
        err, tr, idem = P.assert_acceptance(D.cpu().numpy().astype(np.float64), Dref, w.N_occ, f"k={k}")
        print(f"scale 2^{k}: err={err:.2e} trace={tr:.2e} idem={idem:.2e} layers={info['n_layers']}")


@pytest.fixture(scope="module")
def benv(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    h = api.Handle(256, 1024, 80)
    yield api, h, torch
    h.close()


@pytest.mark.parametrize("auto", [False, True])
def test_config5_batched_full(benv, auto):
    """BASELINE configs[4]: 1024 independent gapped H of N=256, one launch; every matrix against the closed form
    D* = Q_occ Q_occ^T, a sample of matrices against the FP64 oracle layer by layer."""
    api, h, torch = benv
    w = W.config5(0, batch=1024, n=256)
    opts = api.make_opts(bounds=None if auto else w.bounds, tol=w.tol, max_layers=w.max_layers)
    D, info = h.density_matrix_batched(torch.from_numpy(w.H32).cuda(), w.N_occ, opts)
    D = D.cpu().numpy().astype(np.float64)
    assert info["status"] == 0 and np.all(info["per_status"] == 0)
    assert info["n_layers"].min() >= 15 and info["n_layers"].max() <= (45 if auto else 30)
    for m in range(1024):
        Dstar = O.closed_form_density(w.Q[m], w.N_occ)
        assert np.abs(D[m] - Dstar).max() <= P.TOL_D, f"matrix {m}"
        assert abs(np.trace(D[m]) - w.N_occ) <= 1e-3 * w.N_occ
        assert np.array_equal(D[m], D[m].T)
    for m in (0, 1, 17, 511, 1023):
        st_g = api.batched_stats(info, m)
        bounds = w.bounds
        if auto:
            bounds = O.gershgorin_bounds(O.symmetrize_lower(w.H32[m]))
        Dref, st = O.sp2_ref(w.H32[m], w.N_occ, bounds, tol=w.tol, max_layers=w.max_layers)
        P.assert_acceptance(D[m], Dref, w.N_occ, f"matrix {m}")
        P.branch_prefix_check(st_g, st, w.N_occ)
        P.replay_check(st_g, w.H32[m], w.N_occ, bounds, eigs=w.eps[m])
        assert abs(int(info["n_layers"][m]) - st["n_layers"]) <= 2


@pytest.mark.parametrize("n,b", [(1, 3), (2, 5), (50, 7), (128, 300), (129, 4), (200, 150), (256, 149)])
def test_batched_sizes_and_per_matrix_occupation(benv, n, b):
    """Ragged N (one CTA for N<=128, a CTA pair above), batch sizes that do not divide the grid, a different
    N_occ per matrix (so branch sequences and stop layers differ across the batch)."""
    api, h, torch = benv
    rng = np.random.default_rng(n * 1000 + b)
    Hs = np.empty((b, n, n), dtype=np.float32)
    noccs = np.empty(b)
    refs = []
    for m in range(b):
        k = int(rng.integers(0, n + 1)) if n > 2 else min(m % (n + 1), n)
        if n == 1:
            Hs[m] = np.float32(rng.uniform(-0.9, 0.9))
            Dstar = np.array([[float(k)]])
        else:
            k = max(1, min(n - 1, k))
            wl = W.gapped_dense(0, n, (-1.0, -0.15), (0.15, 1.0), k, "b", bounds=(-1.0, 1.0), rng=rng)
            Hs[m] = wl.H32
            Dstar = O.closed_form_density(wl.Q, k)
        noccs[m] = k
        refs.append(Dstar)
    opts = api.make_opts(bounds=(-1.0, 1.0), tol=1e-5, max_layers=80)
    D, info = h.density_matrix_batched(torch.from_numpy(Hs).cuda(), noccs, opts)
    D = D.cpu().numpy().astype(np.float64)
    assert np.all(info["per_status"] == 0)
    for m in range(b):
        assert np.abs(D[m] - refs[m]).max() <= P.TOL_D, f"N={n} matrix {m} N_occ={noccs[m]}"
    m = b - 1
    Dref, st = O.sp2_ref(Hs[m], noccs[m], (-1.0, 1.0), tol=1e-5, max_layers=80)
    P.assert_acceptance(D[m], Dref, noccs[m])
    assert abs(int(info["n_layers"][m]) - st["n_layers"]) <= 2


def test_batched_errors(benv):
    api, h, torch = benv
    Hs = torch.zeros((4, 64, 64), device="cuda")
    Hs[1] = torch.eye(64, device="cuda")          # multiple of I: Gershgorin degenerate for this matrix only
    w = W.config1(0, n=64)
    Hs[0] = torch.from_numpy(w.H32).cuda(); Hs[2] = Hs[0]; Hs[3] = Hs[0]
    with pytest.raises(api.SP2Error) as e:
        h.density_matrix_batched(Hs, 32.0, api.make_opts(tol=1e-5, max_layers=60))
    assert e.value.status == -2
    with pytest.raises(api.SP2Error):
        h.density_matrix_batched(torch.zeros((2, 300, 300), device="cuda"), 1.0, api.make_opts(bounds=(-1.0, 1.0)))
