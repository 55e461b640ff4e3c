"""sp2_gershgorin_static: the allocation-free Gershgorin call, checked against the ordinary handle-based one.

The ordinary path (sp2_create + sp2_gershgorin) calls cudaMalloc for its workspace.  Some users of this library cannot
do that where they call from: their own memory arena already owns all of HBM, so a library's cudaMalloc fails, or they
sit in a time-step loop where the device-wide synchronisation of a cudaMalloc is not acceptable.  For them the library
has ONE entry point whose scratch is a static device array (N <= 4096, about 2.2 MB per GPU).  This file checks that it
returns what the handle path returns, on two calls in a row (the array is shared and keeps the previous call's
contents, so the second call is the one that would show stale data), and that it refuses sizes beyond its limit.

The file name sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide the parity tests.
It passes alone in a fresh process and after the rest of the suite (it owns its handle and touches no global state
other than the static array, which no other test uses)."""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W

pytestmark = pytest.mark.gpu

REL_TOL = 1e-5   # the bar of test_gershgorin_matches_oracle (reading C3)


def _close(a, b):
    return abs(a - b) <= REL_TOL * abs(b)


def test_static_scratch_gershgorin_matches_handle_path_twice_in_a_row(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    torch.cuda.set_device(0)
    lib = api.load()
    assert lib.sp2_gershgorin_static_max_n() == 4096
    assert lib.sp2_gershgorin_static_bytes() < 4 * 1024 * 1024      # "modest": a few MB per GPU
    h = api.Handle(4096, 0, 10)
    out = torch.empty(2, dtype=torch.float64, device="cuda")         # the caller's output buffer, allocated once
    try:
        # two calls in a row, the second on a SMALLER matrix so that most of the scratch still holds the first call's
        # sums; then the limit itself, a ragged size and N = 1, back to back as well
        for seed, n in ((1, 3000), (2, 1000), (3, 4096), (4, 65), (5, 1), (6, 3000), (6, 3000)):
            Hs = W.uniform_symmetric(seed, n)
            Hs[np.triu_indices(n, 1)] += 0.25        # only the lower triangle may be read
            Hd = torch.from_numpy(Hs).cuda()
            ref = h.gershgorin(Hd)                   # existing path: handle workspace from cudaMalloc
            out.fill_(float("nan"))
            api.gershgorin_static(Hd, out)
            torch.cuda.synchronize()
            got = out.cpu().numpy()
            assert _close(got[0], ref[0]) and _close(got[1], ref[1]), (n, got, ref)
            # same kernels on the same input in the same fixed summation order: the bits agree too
            assert got[0] == ref[0] and got[1] == ref[1], (n, got, ref)
            orc = O.gershgorin_bounds(O.symmetrize_lower(Hs))
            assert _close(got[0], orc[0]) and _close(got[1], orc[1]), (n, got, orc)
    finally:
        h.close()


def test_static_scratch_gershgorin_rejects_sizes_beyond_its_limit(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    torch.cuda.set_device(0)
    lib = api.load()
    n = lib.sp2_gershgorin_static_max_n() + 1
    Hd = torch.zeros((n, n), dtype=torch.float32, device="cuda")
    out = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
    st = lib.sp2_gershgorin_static(Hd.data_ptr(), n, n, out.data_ptr(), None)
    assert lib.sp2_status_string(st).decode() == "SP2_ERR_UNSUPPORTED_N"
    msg = lib.sp2_gershgorin_static_last_error().decode()
    assert "4097" in msg and "4096" in msg and "sp2_gershgorin" in msg
    with pytest.raises(RuntimeError, match="exceeds the static scratch"):
        api.gershgorin_static(Hd, out)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [7.0, 7.0]          # nothing was enqueued
    # a non-finite row poisons the bounds, as in the handle path
    Hd = torch.zeros((100, 100), dtype=torch.float32, device="cuda")
    Hd[50, 3] = float("inf")
    api.gershgorin_static(Hd, out)
    torch.cuda.synchronize()
    assert all(np.isnan(out.cpu().numpy()))
