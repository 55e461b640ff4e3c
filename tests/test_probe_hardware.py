"""Hardware probes (marker `gpu_probe`, NOT part of `-m gpu`): timing measurements of three facts the kernels' design
leans on.  They compile tests/cuda/*.cu with nvcc on the GPU box, print the numbers DESIGN.md / profiles/ quote, and
assert only the DIRECTION of each fact with wide margins -- cycle counts and GB/s depend on clocks and driver, and a
missed threshold here must never stand between `pytest -x` and the parity tests.  Run them on a B200 with
    python -m pytest tests/test_probe_hardware.py -m gpu_probe -s

1. An isolated FP64 instruction pays a wake-up latency of the FP64 datapath (hundreds of cycles) while back-to-back
   FP64 instructions do not -- the reason the control step and every trace are integer fixed point
   (csrc/sp2_control.cuh).
2. MMA issue interval: lane == 0 against elect.sync issue.
3. Store patterns of the layer epilogue."""
import os
import shutil
import subprocess

import pytest

pytestmark = pytest.mark.gpu_probe
HERE = os.path.dirname(os.path.abspath(__file__))


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
    assert v["dfma_chain"] < 40.0                                      # back to back: the pipeline latency (measured 9)
    sum_of_latencies = v["dfma_chain"] + 16 * v["ffma_chain"]
    print(f"1 DFMA + 16 FFMA: {v['dfma_plus_16_ffma']:.0f} cycles against {sum_of_latencies:.0f} for the sum of the "
          f"latencies -> wake-up {v['dfma_plus_16_ffma'] - sum_of_latencies:.0f} cycles")
    assert v["dfma_plus_16_ffma"] > 1.2 * sum_of_latencies             # an isolated FP64 instruction is expensive (measured 3.1x)


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
    # measured on the round-2 boxes: 64 / 128 / 128 cycles at the pipe rate, ~105 under lane == 0 whatever N
    assert 50.0 < v["cg1_n128_one_acc_elect"] < 90.0                   # about the pipe rate of a 128 x 128 x 16 MMA
    assert 100.0 < v["cg1_n256_one_acc"] < 170.0 and 100.0 < v["cg2_n256_one_acc"] < 170.0
    assert v["cg1_n128_one_acc"] > 1.1 * v["cg1_n128_one_acc_elect"]   # lane == 0: issue-bound
    assert v["ring_3x128_one_thread_loop"] < v["ring_3x128_stages3"]


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
    # measured on the round-2 boxes: 2.2x, 1.4x, 1.0x
    assert v["own_rows_32B_per_lane"] > 1.2 * v["own_rows_16B_per_lane"]
    assert v["mirrored_128B_per_instruction"] > 1.05 * v["mirrored_64B_per_instruction"]
