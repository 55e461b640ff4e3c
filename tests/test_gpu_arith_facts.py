"""An arithmetic fact the design leans on, as a parity test against the oracle's exact mixed-precision square:
the tensor core's FP32 accumulation TRUNCATES.  An off-diagonal entry of the mixed-precision square comes out
multiplied by 1 + beta, beta < 0 growing with the number of accumulations -- the noise floor of the plain layers
and the reason for the enhanced-accumulation layers of the refinement (NEXT-1).
(The timing probes that used to live here are hardware measurements, not parity: tests/test_probe_hardware.py,
marker gpu_probe, outside the `-m gpu` selection.)"""
import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W

pytestmark = pytest.mark.gpu


def test_tensor_core_accumulation_shrinks_the_off_diagonal_part(cuda_device):
    import torch

    from paper_2101_06385_b200 import api

    h = api.Handle(2304, 0, 8)
    betas = {}
    for n in (640, 2048):
        rng = np.random.default_rng(100 + n)
        Q = W.haar_orthogonal(rng, n)
        nocc = n // 2
        s = np.concatenate([1.0 - rng.uniform(0, 2e-2, nocc), rng.uniform(0, 2e-2, n - nocc)])   # a nearly converged S
        S64 = (Q * s) @ Q.T
        H32 = np.ascontiguousarray((np.eye(n) - 0.5 * (S64 + S64.T)).astype(np.float32))           # S_0 = I - H with (0, 1)
        S0 = (-H32).astype(np.float32)
        S0[np.diag_indices(n)] = (S0[np.diag_indices(n)] + np.float32(1.0)).astype(np.float32)
        S0 = np.tril(S0) + np.tril(S0, -1).T
        hi, lo = O.split_fp16(S0 * np.float32(8192.0))
        Xmix = O.mixed_square_exact(hi, lo) / 8192.0 ** 2              # Eq. 15 with exact sums: the target
        off = ~np.eye(n, dtype=bool)
        # plain / enhanced accumulation with 2 K-blocks per tensor-core chunk / with the library default (4)
        for tile, kc in ((1, 0), (4, 2), (4, 0)):
            X, _ = h.generalized(torch.from_numpy(H32).cuda(), np.array([[1.0, 0.0, 0.0]]), bounds=(0.0, 1.0),
                                 opts=api.make_opts(tile_config=tile, enh_kc=kc))
            d = (X.cpu().numpy().astype(np.float64) - Xmix)[off]
            r = Xmix[off]
            # least-squares factor: X_off = (1 + beta) target
            betas[(n, tile) if kc == 2 or tile == 1 else (n, "default")] = float((d * r).sum() / (r * r).sum())
    print("off-diagonal shrink factor beta of one layer (plain | enhanced, 2 K-blocks per chunk | enhanced, default 4): "
          + ", ".join(f"N={n}: {betas[(n, 1)]:+.2e} | {betas[(n, 4)]:+.2e} | {betas[(n, 'default')]:+.2e}"
                      for n in (640, 2048)))
    assert -2e-5 < betas[(2048, 1)] < betas[(640, 1)] < -5e-7         # truncation: negative, growing with K
    # chunked accumulation removes it (measured -4.4e-7 against -4.1e-6; -6.2e-6 before the 128 x 128 tiles kept X0 X1 in
    # an accumulator of its own, which shortens the chain of truncating adds behind the dominant term by a third)
    assert abs(betas[(2048, 4)]) < 0.15 * abs(betas[(2048, 1)])
    # the default chunk of 4 K-blocks chains twice as many truncating adds: twice the residue (measured -8.2e-7)
    assert abs(betas[(2048, 4)]) < abs(betas[(2048, "default")]) < 0.3 * abs(betas[(2048, 1)])
    h.close()
