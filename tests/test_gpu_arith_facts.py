"""Measurements of the two hardware facts the design leans on, as tests (they print the numbers DESIGN.md quotes):

1. The tensor core's FP32 accumulation TRUNCATES: an off-diagonal entry of the mixed-precision square comes out
   multiplied by 1 + beta, beta < 0 growing with the number of accumulations -- the noise floor of the plain layers
   and the reason for the enhanced-accumulation layers of the refinement (NEXT-1).
2. An isolated FP64 instruction pays a wake-up latency of the FP64 datapath (hundreds of cycles) while back-to-back
   FP64 instructions do not -- the reason the control step and every trace are integer fixed point
   (csrc/sp2_control.cuh)."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from oracle import sp2_oracle as O
from paper_2101_06385_b200 import workloads as W

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


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
        for tile in (1, 4):                                            # plain / enhanced accumulation
            X, _ = h.generalized(torch.from_numpy(H32).cuda(), np.array([[1.0, 0.0, 0.0]]), bounds=(0.0, 1.0),
                                 opts=api.make_opts(tile_config=tile))
            d = (X.cpu().numpy().astype(np.float64) - Xmix)[off]
            r = Xmix[off]
            betas[(n, tile)] = float((d * r).sum() / (r * r).sum())    # least-squares factor: X_off = (1 + beta) target
    print("off-diagonal shrink factor beta of one layer (plain | enhanced accumulation): "
          + ", ".join(f"N={n}: {betas[(n, 1)]:+.2e} | {betas[(n, 4)]:+.2e}" for n in (640, 2048)))
    assert -2e-5 < betas[(2048, 1)] < betas[(640, 1)] < -5e-7         # truncation: negative, growing with K
    # chunked accumulation removes it (measured -4.4e-7 against -4.1e-6; -6.2e-6 before the 128 x 128 tiles kept X0 X1 in
    # an accumulator of its own, which shortens the chain of truncating adds behind the dominant term by a third)
    assert abs(betas[(2048, 4)]) < 0.15 * abs(betas[(2048, 1)])
    h.close()


def test_fp64_wakeup_latency(cuda_device, tmp_path):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    exe = str(tmp_path / "fp64_wakeup")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe,
                    os.path.join(HERE, "cuda", "fp64_wakeup.cu")], check=True)
    out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout
    v = {k: float(x) for k, x in (ln.split() for ln in out.strip().splitlines())}
    print("cycles per iteration:", v)
    assert v["dfma_chain"] < 20.0                                      # back to back: the pipeline latency
    sum_of_latencies = v["dfma_chain"] + 16 * v["ffma_chain"]
    print(f"1 DFMA + 16 FFMA: {v['dfma_plus_16_ffma']:.0f} cycles against {sum_of_latencies:.0f} for the sum of the "
          f"latencies -> wake-up {v['dfma_plus_16_ffma'] - sum_of_latencies:.0f} cycles")
    assert v["dfma_plus_16_ffma"] > 1.5 * sum_of_latencies             # an isolated FP64 instruction is expensive


def test_mma_issue_interval(cuda_device, tmp_path):
    """Third fact: a tcgen05.mma issued under `if (lane == 0)` costs ~105 cycles whatever its size (the compiler wraps it
    in a loop of R2UR.BROADCASTs), one issued by an elect.sync thread in warp-uniform control flow runs at the tensor
    pipe's rate (N = 128: 64 cycles, N = 256: 128) -- why every MMA / TMA issue in the library goes through elect_one()
    (csrc/sp2_ptx.cuh), why 128 x 128 tiles stop paying as soon as they need a second round (choose_tile_config) and why
    the MMA issuer is one thread running the whole loop (the ring numbers)."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    exe = str(tmp_path / "mma_rate")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe,
                    os.path.join(HERE, "cuda", "mma_rate.cu")], check=True)
    out = subprocess.run([exe], capture_output=True, text=True, check=True, timeout=120).stdout
    v = {k: float(x) for k, x in (ln.split() for ln in out.strip().splitlines())}
    print("cycles per MMA / per stage:", v)
    assert 60.0 < v["cg1_n128_one_acc_elect"] < 72.0                   # the pipe rate of a 128 x 128 x 16 MMA
    assert 120.0 < v["cg1_n256_one_acc"] < 136.0 and 120.0 < v["cg2_n256_one_acc"] < 136.0
    assert v["cg1_n128_one_acc"] > 1.25 * v["cg1_n128_one_acc_elect"]  # lane == 0: issue-bound
    assert abs(v["cg1_n64_one_acc"] - v["cg1_n128_one_acc"]) < 5.0     # ... at a rate that does not depend on N
    assert v["ring_3x128_one_thread_loop"] < v["ring_3x128_cheap_desc_stages3"] < v["ring_3x128_stages3"]


def test_store_patterns_of_the_epilogue(cuda_device, tmp_path):
    """Fourth fact: the layer epilogue is bound by its stores, and how a warp packages them matters.  A lane that writes
    64 bytes of a row of its own in 16-byte stores gets well under half of what it gets with 32-byte st.global.v8 stores
    (why the own-row stores of sp2_square_tiled.cu are st_cs_v8); 64-byte row segments (the FP16 operands of a 32-column
    chunk) stay below 128-byte ones however they are packaged (pairing rows in one instruction does not help)."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    exe = str(tmp_path / "store_patterns")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe,
                    os.path.join(HERE, "cuda", "store_patterns.cu")], check=True)
    out = subprocess.run([exe], capture_output=True, text=True, check=True, timeout=120).stdout
    v = {k: float(x) for k, x in (ln.split() for ln in out.strip().splitlines())}
    print("GB/s:", v)
    assert v["own_rows_32B_per_lane"] > 1.8 * v["own_rows_16B_per_lane"]
    assert v["mirrored_128B_per_instruction"] > 1.2 * v["mirrored_64B_per_instruction"]
    assert v["mirrored_two_rows_of_64B_per_instruction"] < 1.15 * v["mirrored_64B_per_instruction"]
