"""The C-ABI library builds for sm_100a (cross-compiled, no GPU needed), loads, and exports every function that
include/sp2_b200.h declares; the ctypes structures match the header's layouts.  No compute calls here."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sp2_b200.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(sp2_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2101_06385_b200 import api, build

    build.build()
    return api.load()


def test_header_declares_the_path_calls():
    names = _declared_functions()
    for must in ("sp2_density_matrix", "sp2_generalized", "sp2_generalized_wb", "sp2_density_matrix_batched",
                 "sp2_split_fp16", "sp2_gershgorin", "sp2_create", "sp2_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2101_06385_b200 import api

    declared = _declared_functions()
    for name in declared:
        assert hasattr(lib, name), f"libsp2b200.so does not export {name}"
    assert sorted(api.EXPORTS) == declared, "api.EXPORTS and include/sp2_b200.h disagree"
    out = subprocess.run(["nm", "-D", "--defined-only", api.LIB_PATH], capture_output=True, text=True).stdout
    for name in declared:
        assert re.search(rf"\bT {name}\b", out), f"{name} is not a defined text symbol"


def test_struct_layouts_match_header():
    """Compile a tiny C program against the header with gcc and compare sizeof/offsetof with the ctypes mirror."""
    from paper_2101_06385_b200 import api

    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "sp2_b200.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\n", sizeof(sp2_layer_stat_t), offsetof(sp2_layer_stat_t, trace_X_diag),
         offsetof(sp2_layer_stat_t, sigma), offsetof(sp2_layer_stat_t, t_end_ns), sizeof(sp2_opts_t),
         offsetof(sp2_opts_t, tol), offsetof(sp2_opts_t, eps_alt), offsetof(sp2_opts_t, tile_config),
         offsetof(sp2_opts_t, accelerated), offsetof(sp2_opts_t, lumo), offsetof(sp2_opts_t, noise_kappa),
         offsetof(sp2_opts_t, enh_kc), offsetof(sp2_opts_t, trunc_tau));
  return 0; }'''
    import tempfile

    with tempfile.TemporaryDirectory() as d:
        src = os.path.join(d, "t.c")
        open(src, "w").write(prog)
        exe = os.path.join(d, "t")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), src, "-o", exe], check=True)
        got = [int(x) for x in subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()]
    L, Op = api.LayerStat, api.Opts
    want = [C.sizeof(L), L.trace_X_diag.offset, L.sigma.offset, L.t_end_ns.offset, C.sizeof(Op), Op.tol.offset,
            Op.eps_alt.offset, Op.tile_config.offset, Op.accelerated.offset, Op.lumo.offset, Op.noise_kappa.offset,
            Op.enh_kc.offset, Op.trunc_tau.offset]
    assert got == want


def test_host_only_calls_do_not_need_a_gpu(lib):
    from paper_2101_06385_b200 import api

    assert lib.sp2_version().decode().startswith("sp2b200")
    assert lib.sp2_status_string(-2).decode() == "SP2_ERR_BOUNDS_DEGENERATE"
    o = api.Opts()
    lib.sp2_default_opts(C.byref(o))
    assert o.auto_bounds == 1 and o.max_layers == 120 and o.tol == 0.0
    assert o.noise_kappa < 0 and o.enh_kc == 0 and o.trunc_tau == 0.0
    assert lib.sp2_workspace_bytes_lazy(16384) >= 3 * 16384 * 16384 * 4      # mix matrix + two staging matrices
    assert lib.sp2_workspace_bytes(16384, 0, 120) >= 3 * 16384 * 16384 * 4
    assert lib.sp2_workspace_bytes(0, 0, 120) == 0


def test_no_cpu_fallback_without_a_device(lib):
    """On a box without a GPU the product path must fail loudly, never compute on the CPU."""
    import torch

    from paper_2101_06385_b200 import api

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(api.SP2Error) as e:
        api.Handle(128, 0, 10)
    assert e.value.status == -5


def test_oracle_and_product_are_independent():
    """The oracle is test infrastructure: the package never imports it and it never imports the package; only the
    seeded input generators (workloads.py, which hold none of the method's arithmetic) serve both."""
    pkg = os.path.join(ROOT, "paper_2101_06385_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f"{f} imports the oracle"
                assert "sp2_oracle" not in src, f"{f} mentions the oracle module"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2101_06385_b200\b", src, re.M), f"{f} imports the product"
    # workloads.py: generators only -- no split, no square, no SP2 layer
    wl = open(os.path.join(pkg, "workloads.py")).read()
    for word in ("float16", "gershgorin", "@ S", "S @", "split_fp16"):
        assert word not in wl, f"workloads.py contains method arithmetic: {word}"
    # bench.py may execute the oracle only in its cpu_baseline / --impl reference legs
    bench = open(os.path.join(ROOT, "bench.py")).read()
    assert bench.count("from oracle import") == 1 and "def cpu_oracle_sample" in bench
