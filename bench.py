#!/usr/bin/env python
"""bench.py -- SP2 hot path at N=16384 (BASELINE.json configs[2]) on B200.

A "step" is one pass of the whole hot path over one synthetic Hamiltonian: Gershgorin bounds (a1), initial
affine layer + split (a2, a3), every fused SP2 layer to convergence (a4-a8, device-side control in a CUDA
graph), D copied out.  `value` = effective TFLOP/s = 6 N^3 flop-equivalents per layer ("3 FP16 GEMM-equivalents",
BASELINE.json metric) x layers / device time of the whole solve, inputs resident in HBM.  The paper's own count
(2 GEMMs, 4 N^3) and the executed count (3 N^3: three products on the symmetric half) are in `detail`.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 16384] [--bounds auto|explicit] [--impl reference]

Multi-GPU: a single large H does not shard: N ranks = N independent replicas, no collective
on the data path; value = total work / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "sp2_effective_tflops_n16384"
UNIT = "TFLOP/s (6*N^3 per layer)"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return d, "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            pass
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def _dist_setup(n_gpus: int):
    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist

        torch.cuda.set_device(local)
        dist.init_process_group("nccl" if torch.cuda.is_available() else "gloo")
    elif torch.cuda.is_available():
        torch.cuda.set_device(0)
    return rank, world, local


def _max_over_ranks(x: float, world: int) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist

    t = torch.tensor([x], dtype=torch.float64, device="cuda" if torch.cuda.is_available() else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def _barrier(world: int):
    import torch

    if world > 1:
        import torch.distributed as dist

        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def cpu_oracle_sample(w, budget_s: float = 20.0):
    """The FP64 oracle as it stands (oracle/sp2_oracle.py, NumPy dgemm on the host cores) on a bounded sample:
    whole layers of sp2_ref on the same H if one layer fits the budget, otherwise on the leading principal block
    of H of the largest size whose layer does (stated in `sample`)."""
    from oracle import sp2_oracle as O

    try:
        from threadpoolctl import threadpool_info

        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    rng = np.random.default_rng(0)
    A = rng.standard_normal((2048, 2048))
    t0 = time.perf_counter(); A @ A; dt = time.perf_counter() - t0
    gflops = 2 * 2048 ** 3 / dt / 1e9
    n = w.N
    while n > 1024 and 2.0 * n ** 3 / (gflops * 1e9) > budget_s:
        n //= 2
    layers = max(1, min(4, int(budget_s / max(1e-9, 2.0 * n ** 3 / (gflops * 1e9)))))
    Hs = np.ascontiguousarray(w.H32[:n, :n])
    bounds = w.bounds if w.bounds is not None else None
    t0 = time.perf_counter()
    _, st = O.sp2_ref(Hs, n / 2.0, (-2.5, 2.5) if bounds is None else bounds, tol=0.0, max_layers=layers)
    dt = time.perf_counter() - t0
    value = 6.0 * n ** 3 * st["n_layers"] / dt / 1e12
    sample = (f"oracle.sp2_ref FP64, {st['n_layers']} layer(s) on the "
              f"{'full' if n == w.N else 'leading principal'} {n}x{n} block of the same H, {dt:.1f} s "
              f"(host dgemm probe {gflops:.0f} GFLOP/s)")
    return {"value": value, "unit": UNIT, "cores": int(cores), "kind": "oracle", "sample": sample,
            "ms_per_layer": dt / st["n_layers"] * 1e3, "n": n}


def other_configs(api, W, torch, dev, stream, _time):
    """detail.configs: BASELINE.json configs[0], [1], [3], [4] (the headline is configs[2]) through the same C ABI:
    ms per call (CUDA events around the whole call, median of 7 after 30 ms of warm-up calls), layers, and the parity
    triple of BASELINE north_star
    -- max |X - X*|, |Tr - N_occ|, ||X^2 - X||_F / sqrt(N) -- against the CLOSED FORM each input is built for
    (Eq. 6: D* = Q_occ Q_occ^T; config 2: the LAPACK eigenprojector, FP64 on the device; config 4:
    X* = Q diag(p(eps)) Q^T with p the scalar polynomial of Eq. 17), all evaluated here in FP64 with torch / numpy."""
    out = {}
    base_time = _time

    def _time(fn, reps=7):
        # These calls last 0.2 - 5 ms: a GPU that idled through the host-side set-up of a config needs tens of
        # milliseconds of work before its clocks are back up, so warm up with 30 ms of the same call first.
        t0 = time.perf_counter()
        while time.perf_counter() - t0 < 0.03:
            fn()
        return base_time(fn, reps=reps)

    def triple(X, Xstar, nocc):
        Xd = X.double()
        return {"max_abs_err": float((Xd - Xstar).abs().max()),
                "trace_err": (float(torch.trace(Xd)) - nocc) if nocc is not None else None,
                "idempotency": (float(torch.linalg.norm(Xd @ Xd - Xd)) / np.sqrt(X.shape[-1])) if nocc is not None else None,
                "symmetric": bool(torch.equal(X, X.transpose(-1, -2)))}

    # ---- config 1: N = 128, explicit (-1, 1) and Gershgorin bounds (one launch of the resident kernel)
    w = W.config1(0)
    Hd = torch.from_numpy(w.H32).to(dev)
    Qo = torch.from_numpy(w.Q[:, : int(w.N_occ)]).to(dev)
    Dstar = Qo @ Qo.T
    h1 = api.Handle(128, 0, 120)
    for name, bnd in (("explicit", w.bounds), ("gershgorin", None)):
        o = api.make_opts(bounds=bnd, tol=w.tol, max_layers=w.max_layers)
        ms = _time(lambda: h1.density_matrix(Hd, w.N_occ, o, stream=stream))
        D, info = h1.density_matrix(Hd, w.N_occ, o, stream=stream)
        out[f"config1_N128_{name}"] = dict(ms_per_D=ms, layers=info["n_layers"], launches=info["launches"],
                                           **triple(D, Dstar, w.N_occ))
    h1.close()
    # ---- config 2: N = 2048 tight-binding-like, Gershgorin bounds
    w = W.config2(0)
    Hd = torch.from_numpy(w.H32).to(dev)
    E, V = torch.linalg.eigh(torch.tril(Hd.double()) + torch.tril(Hd.double(), -1).T)
    k = int(w.N_occ)
    Dstar = V[:, :k] @ V[:, :k].T
    h2 = api.Handle(4096, 0, 120)
    o = api.make_opts(bounds=None, tol=w.tol, max_layers=w.max_layers)
    ms = _time(lambda: h2.density_matrix(Hd, w.N_occ, o, stream=stream))
    D, info = h2.density_matrix(Hd, w.N_occ, o, stream=stream)
    t = np.diff(np.array(info["t_end_ns"], dtype=np.float64)) * 1e-3
    out["config2_N2048_tight_binding"] = dict(ms_per_D=ms, layers=info["n_layers"], us_per_layer=float(np.median(t)),
                                              executed_tflops_3N3=3.0 * 2048 ** 3 / (float(np.median(t)) * 1e-6) / 1e12,
                                              homo_lumo_gap=float(E[k] - E[k - 1]), **triple(D, Dstar, w.N_occ))
    # ---- config 4: N = 4096 generalized network, 30 layers (sigma alternating +1, -1; w_n, b_n from the seed)
    w = W.config4(0, device=dev)
    L = w.extra["layers"]
    sig = np.array([1, -1] * (L // 2 + 1))[:L]
    wt, bs = w.extra["weights"], w.extra["biases"]
    lam = (w.bounds[1] - w.eps) / (w.bounds[1] - w.bounds[0])          # eigenvalues of S_0 (Alg. 1)
    for n in range(L):                                                 # Eq. 17 on each eigenvalue (reading C19)
        lam = wt[n] * (sig[n] * lam * lam + (1 - sig[n]) * lam) + bs[n]
    Hd = torch.from_numpy(w.H32).to(dev)
    Qd = torch.from_numpy(w.Q).to(dev)
    Xstar = (Qd * torch.from_numpy(lam).to(dev)[None, :]) @ Qd.T
    ms = _time(lambda: h2.generalized_wb(Hd, sig, wt, bs, bounds=w.bounds, stream=stream))
    X, info = h2.generalized_wb(Hd, sig, wt, bs, bounds=w.bounds, stream=stream)
    tr = triple(X, Xstar, None)
    tr["trace_err"] = float(torch.trace(X.double())) - float(lam.sum())
    out["config4_N4096_generalized_30_layers"] = dict(ms_per_call=ms, layers=L, us_per_layer=ms / L * 1e3,
                                                      executed_tflops_3N3=3.0 * 4096 ** 3 * L / (ms * 1e-3) / 1e12, **tr)
    h2.close()
    del Qd, Xstar, X, Hd
    # ---- config 5: 1024 matrices of N = 256, one launch
    w = W.config5(0)
    Hd = torch.from_numpy(w.H32).to(dev)
    Qo = torch.from_numpy(np.ascontiguousarray(w.Q[:, :, : int(w.N_occ)])).to(dev)
    Dstar = Qo @ Qo.transpose(1, 2)
    h5 = api.Handle(256, 1024, 60)
    Db = torch.empty_like(Hd)
    for name, bnd in (("explicit", w.bounds), ("gershgorin", None)):
        o = api.make_opts(bounds=bnd, tol=w.tol, max_layers=w.max_layers)
        ms = _time(lambda: h5.density_matrix_batched(Hd, w.N_occ, o, out=Db, stream=stream))
        _, info = h5.density_matrix_batched(Hd, w.N_occ, o, out=Db, stream=stream)
        Dd = Db.double()
        idem = torch.linalg.norm((Dd @ Dd - Dd).reshape(1024, -1), dim=1) / 16.0
        trs = torch.diagonal(Dd, dim1=1, dim2=2).sum(1) - w.N_occ
        layers = float(info["n_layers"].mean())
        out[f"config5_1024xN256_{name}"] = dict(
            ms_per_batch=ms, matrices_per_s=1024 / (ms * 1e-3), layers_mean=layers,
            executed_tflops_3N3=3.0 * 256 ** 3 * float(info["n_layers"].sum()) / (ms * 1e-3) / 1e12,
            max_abs_err=float((Dd - Dstar).abs().max()), trace_err=float(trs.abs().max()),
            idempotency=float(idem.max()), symmetric=bool(torch.equal(Db, Db.transpose(1, 2))),
            worst_status=int(info["status"]))
    h5.close()
    return out


def next_rows_and_sweep(api, W, torch, dev, stream, _time, sustained_tflops):
    """detail.blocked_sparse_next4, detail.mix_next2, detail.size_sweep (rank 0, outside the timed step):
    the two NEXT rows that had no driver-run number, and the layer kernel's throughput against N (the paper's one
    performance figure is TFLOP/s against system size, Fig. 3)."""
    base_time = _time

    def _time(fn, reps=5):
        t0 = time.perf_counter()
        while time.perf_counter() - t0 < 0.03:          # clocks back up after host-side set-up (see other_configs)
            fn()
        return base_time(fn, reps=reps)

    h = api.Handle(16384, 0, 120)
    # ---- NEXT-4: blocked-sparse variant on the decaying chain (reading C28), tau = 1e-6, against the dense layer
    # kernel with the same 128 x 128 tiles and the tensor-core diagonal (what the sparse instantiation computes when
    # nothing is cut)
    sparse = {}
    for n in (2048, 8192, 16384):
        w = W.decaying_chain(n, n=n)
        Hd = torch.from_numpy(w.H32).to(dev)
        o_s = api.make_opts(tol=w.tol, max_layers=w.max_layers, trunc_tau=1e-6)
        o_d = api.make_opts(tol=w.tol, max_layers=w.max_layers, tile_config=1, exact_diag=0)
        o_0 = api.make_opts(tol=w.tol, max_layers=w.max_layers)
        Ds = torch.empty_like(Hd)
        ms_s = _time(lambda: h.density_matrix(Hd, w.N_occ, o_s, out=Ds, stream=stream), reps=3)
        _, i_s = h.density_matrix(Hd, w.N_occ, o_s, out=Ds, stream=stream)
        Dd = torch.empty_like(Hd)
        ms_d = _time(lambda: h.density_matrix(Hd, w.N_occ, o_d, out=Dd, stream=stream), reps=3)
        _, i_d = h.density_matrix(Hd, w.N_occ, o_d, out=Dd, stream=stream)
        ms_0 = _time(lambda: h.density_matrix(Hd, w.N_occ, o_0, out=Dd, stream=stream), reps=3)
        _, i_0 = h.density_matrix(Hd, w.N_occ, o_0, out=Dd, stream=stream)
        Dc = Ds.double()
        sparse[f"decaying_chain_N{n}"] = dict(
            ms_sparse=ms_s, layers_sparse=i_s["n_layers"], work_fraction=i_s["work_fraction"],
            us_per_layer_sparse=ms_s / i_s["n_layers"] * 1e3,
            ms_dense_same_tiles=ms_d, layers_dense_same_tiles=i_d["n_layers"],
            ms_dense_default=ms_0, layers_dense_default=i_0["n_layers"],
            max_abs_diff_sparse_vs_dense_default=float((Ds - Dd).abs().max()),
            trace_err=float(torch.trace(Dc)) - w.N_occ,
            idempotency=float(torch.linalg.norm(Dc @ Dc - Dc)) / np.sqrt(n), symmetric=bool(torch.equal(Ds, Ds.T)))
        del Hd, Ds, Dd, Dc
    sparse["what"] = ("sp2_density_matrix, Gershgorin bounds, tol 1e-5; sparse: opts.trunc_tau = 1e-6; dense_same_tiles: "
                      "tile_config = 1, exact_diag = 0; dense_default: library defaults")
    # ---- NEXT-2: output mix F~ = I - sum_i c_i E_i (Eqs. 17-18), N = 4096, 11 layers, against the scalar network on the
    # known eigenvalues through the known eigenbasis
    rng = np.random.default_rng(42)
    n, L = 4096, 11
    Q = W.haar_orthogonal(rng, n, dev)
    lam = rng.uniform(-1.0, 1.0, n)
    Qd = torch.from_numpy(Q).to(dev)
    Hs = (Qd * torch.from_numpy(lam).to(dev)[None, :]) @ Qd.T
    Hd = ((Hs + Hs.T) * 0.5).float().contiguous()
    theta = []
    for k in range(L):                                   # alternating SP2 polynomials with seeded perturbations
        b0 = (1.0, 0.0) if k % 2 else (-1.0, 2.0)
        wk = 1.0 + rng.normal(0, 0.02)
        theta.append((wk * b0[0], wk * b0[1], rng.normal(0, 0.005)))
    theta = np.array(theta)
    c = rng.normal(0, 0.05, L + 1)
    c[-1] += 1.0
    ms_m = _time(lambda: h.generalized_mix(Hd, theta, c, bounds=(-1.0, 1.0), stream=stream), reps=5)
    F, _ = h.generalized_mix(Hd, theta, c, bounds=(-1.0, 1.0), stream=stream)
    ms_g = _time(lambda: h.generalized(Hd, theta, bounds=(-1.0, 1.0), stream=stream), reps=5)
    e = (lam + 1.0) / 2.0
    acc = c[0] * e
    for k in range(L):
        e = theta[k, 0] * e * e + theta[k, 1] * e + theta[k, 2]
        acc = acc + c[k + 1] * e
    Fstar = (Qd * torch.from_numpy(1.0 - acc).to(dev)[None, :]) @ Qd.T
    mix = dict(N=n, layers=L, ms_per_call=ms_m, us_per_layer=ms_m / L * 1e3, ms_same_network_without_mix=ms_g,
               max_abs_err_vs_scalar_network=float((F.double() - Fstar).abs().max()),
               symmetric=bool(torch.equal(F, F.T)),
               what="sp2_generalized_mix, caller bounds (-1, 1), seeded theta (alternating SP2 polynomials, w = 1 + N(0, "
                    "0.02), b = N(0, 0.005)) and c; reference Q diag(1 - sum_i c_i e_i) Q^T in FP64")
    del Q, Qd, Hs, Hd, F, Fstar
    # ---- layer time against N: 10 fixed layers (sigma alternating), caller bounds, default tile choice
    sweep = []
    L = 10
    sig = np.array([1, -1] * (L // 2))
    ones, zeros = np.ones(L), np.zeros(L)
    gen = torch.Generator(device=dev)
    gen.manual_seed(1234)
    for n in (1024, 2048, 3072, 4096, 6144, 8192, 12288, 16384):
        A = torch.rand((n, n), device=dev, generator=gen) * 2.0 - 1.0
        Hd = (torch.tril(A) + torch.tril(A, -1).T).contiguous()
        del A
        r = 1.3 * float(np.sqrt(n))                      # encloses the semicircle of radius 2 sqrt(n / 3)
        ms = _time(lambda: h.generalized_wb(Hd, sig, ones, zeros, bounds=(-r, r), stream=stream), reps=5)
        X, info = h.generalized_wb(Hd, sig, ones, zeros, bounds=(-r, r), stream=stream)
        t = np.diff(np.array(info["t_end_ns"], dtype=np.float64)) * 1e-3       # device timer, layer to layer
        us = float(np.median(t))
        tf = 3.0 * n ** 3 / (us * 1e-6) / 1e12
        sweep.append(dict(N=n, us_per_layer=us, ms_per_call_10_layers=ms, executed_tflops_3N3=tf,
                          frac_of_sustained_peak=tf / sustained_tflops, finite=bool(torch.isfinite(X).all())))
        del Hd, X
    h.close()
    return sparse, mix, {"points": sweep,
                         "what": "sp2_generalized_wb, 10 layers (sigma = +1, -1, ...; w = 1, b = 0), H uniform in [-1, 1] "
                                 "symmetric, caller bounds; us_per_layer = median interval of the per-layer device "
                                 "timestamps; executed flops = 3 N^3 per layer"}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2101_06385_b200 import workloads as W

    n = args.n
    dev = None
    try:
        import torch

        dev = "cuda:0" if torch.cuda.is_available() else None
    except Exception:
        pass
    w = W.config3(args.seed, n, device=dev) if n > 4096 or dev else W.config3(args.seed, n)
    times, last = [], None
    for i in range(args.warmup + args.steps):
        last = cpu_oracle_sample(w, budget_s=max(2.0, 20.0 / max(1, args.steps + args.warmup)))
        if i >= args.warmup:
            times.append(last)
    value = float(np.mean([t["value"] for t in times]))
    ms = float(np.mean([t["ms_per_layer"] for t in times]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config3 gapped dense H N={n} (BASELINE.json configs[2]); each step = a bounded "
                                   f"sample: {last['sample']}"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle",
                             "sample": last["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n", "--size", dest="n", type=int, default=16384)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--bounds", choices=["auto", "explicit"], default="auto")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--control", type=int, default=0,
                    help="0: device-side WHILE graph (default, the product path); 2: max_layers guarded launches "
                         "(same kernels, no graph: lets ncu see every layer launch)")
    ap.add_argument("--exact-diag", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip detail.configs (BASELINE configs 1, 2, 4, 5)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch

    from paper_2101_06385_b200 import api, workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    rank, world, local = _dist_setup(args.gpus)
    dev = f"cuda:{torch.cuda.current_device()}"
    N = args.n
    peaks, peak_src = _peaks()

    # ---- synthetic input (each rank its own seed: independent replicas)
    w = W.config3(args.seed + rank, N, device=dev)
    H = torch.from_numpy(w.H32).to(dev)
    D = torch.empty_like(H)
    h = api.Handle(N, 0, 120)
    bounds = None if args.bounds == "auto" else w.bounds
    opts = api.make_opts(bounds=bounds, tol=w.tol, max_layers=w.max_layers, tile_config=args.tile,
                         control=args.control, exact_diag=args.exact_diag)
    stream = torch.cuda.current_stream()

    def solve():
        return h.density_matrix(H, w.N_occ, opts, out=D, stream=stream)

    # ---- warm-up (W >= 3: graph instantiation, clocks), then K timed steps, CUDA events on the launching stream
    for _ in range(max(3, args.warmup)):
        _, info = solve()
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    _barrier(world)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    layers_total, launches, layer_ms = 0, 0, []
    t_wall0 = time.perf_counter()
    for a, b in ev:
        a.record(stream)
        _, info = solve()
        b.record(stream)
        layers_total += info["n_layers"]
        launches += info["launches"]
        t = np.array(info["t_end_ns"], dtype=np.float64)
        layer_ms.extend(list(np.diff(t) * 1e-6))
    _barrier(world)
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    ms_steps = [a.elapsed_time(b) for a, b in ev]
    t_dev = _max_over_ranks(sum(ms_steps) * 1e-3, world)
    ms_per_step = t_dev / args.steps * 1e3
    n_layers = layers_total / args.steps
    value = world * 6.0 * N ** 3 * layers_total / t_dev / 1e12

    # ---- parity spot checks at full size on the LAST TIMED solve's D (before anything else overwrites D):
    # sampled entries of the closed form D* = Q_occ Q_occ^T, trace, exact symmetry
    Dc = D.double()
    tr = float(torch.trace(Dc).item())
    rng = np.random.default_rng(1)
    ri, ci = rng.integers(0, N, 256), rng.integers(0, N, 256)
    ri[:64] = ci[:64]                                   # a quarter of the samples on the diagonal
    Qo = w.Q[:, : int(w.N_occ)]
    ref = np.einsum("ik,ik->i", Qo[ri], Qo[ci])
    samp_err = float(np.abs(Dc[ri, ci].cpu().numpy() - ref).max())
    symmetric = bool(torch.equal(D, D.T))
    del Dc
    info_timed = info

    # ---- dominant kernel (fused layer) duration.  The layer launches sit inside the device-side WHILE graph, so CUDA
    # events cannot bracket one of them; two measurements of the same timed region instead:
    #   launch_ms              = event-timed step / layers of the step: a purely event-based UPPER bound on the average
    #                            launch (it still holds the ~0.3 % of setup kernels), used for `achieved`;
    #   launch_ms_device_timer = mean interval between consecutive layer completions (%globaltimer stamps written by
    #                            each layer's last CTA), the kernel-to-kernel period itself.
    # (Differences of separately timed solves are not used: under the 1 kW cap the clock state depends on what ran
    # just before, which biased them in both directions.)
    t_layer_ms = float(np.median(ms_steps)) / max(1.0, n_layers)
    t_layer_dev_ms = float(np.mean(layer_ms)) if layer_ms else None
    t_setup_ms = max(0.0, float(np.median(ms_steps)) - n_layers * t_layer_dev_ms) if layer_ms else None
    exec_tflops = 3.0 * N ** 3 / (t_layer_ms * 1e-3) / 1e12
    peak = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
    roofline = {"bound": "tensor", "kernel": "k_sp2_layer (fused symmetric square + epilogue)",
                "achieved": exec_tflops, "peak": peak, "unit": "TFLOP/s", "frac": exec_tflops / peak,
                "peak_source": peak_src + ": cuBLAS bf16 sustained (fp16 and bf16 share the tensor rate)",
                "algorithmic_flops_per_launch": 3.0 * N ** 3, "launch_ms": t_layer_ms,
                "launch_ms_how": "CUDA events on the launching stream: median step time / layers of the step (upper "
                                 "bound: includes the setup kernels' ~0.3 %)",
                "launch_ms_device_timer": t_layer_dev_ms, "traffic": None}
    prof = os.path.join(ROOT, "profiles", "r03_layer_traffic.json")
    if not os.path.exists(prof):
        prof = os.path.join(ROOT, "profiles", "r02_layer_traffic.json")
    if not os.path.exists(prof):
        prof = os.path.join(ROOT, "profiles", "r01_layer_traffic.json")
    if os.path.exists(prof):
        try:
            with open(prof) as f:
                roofline["traffic"] = json.load(f).get(str(N))
        except Exception:
            pass

    # ---- HBM-bound kernels of the path (a1 Gershgorin, a3 split) timed alone, and a same-run cuBLAS FP16 yardstick
    def _time(fn, reps=5):
        ts = []
        for i in range(reps + 1):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            if i:
                ts.append(a.elapsed_time(b))
        return float(np.median(ts))

    hbm_peak = float(peaks["hbm_gbs"])
    t_g = _time(lambda: h.gershgorin(H, stream=stream))
    t_s = _time(lambda: api.split_fp16(H, 13, stream=stream))
    tri_bytes = 2.0 * N * (N + 1)              # lower triangle incl. diagonal, 4 B each
    hbm_kernels = {
        "gershgorin": {"ms": t_g, "bytes_moved": tri_bytes + 8.0 * N * ((N + 63) // 64) * 2,
                       "moved_GBps": (tri_bytes + 16.0 * N * ((N + 63) // 64)) / (t_g * 1e-3) / 1e9,
                       "frac_of_measured_hbm": (tri_bytes + 16.0 * N * ((N + 63) // 64)) / (t_g * 1e-3) / 1e9 / hbm_peak,
                       "algorithmic_GBps_4B_per_element": 4.0 * N * N / (t_g * 1e-3) / 1e9,
                       "note": "reads H's lower triangle only (2 B/element) + writes/reads the per-tile row and column "
                               "sums; SURVEY 8(d) counts 4 B/element (algorithmic rate, not a utilisation); the time "
                               "includes the call's final sync + 16-byte D2H"},
        "split_fp16": {"ms": t_s, "bytes_moved": 8.0 * N * N, "moved_GBps": 8.0 * N * N / (t_s * 1e-3) / 1e9,
                       "frac_of_measured_hbm": 8.0 * N * N / (t_s * 1e-3) / 1e9 / hbm_peak,
                       "note": "4 B read + 4 B written per element; time includes two torch.empty allocations"},
        "setup_ms_bounds_affine_split_copyout": t_setup_ms,
        "setup_how": "event-timed step - layers x mean device-timer layer interval of the same steps (clamped at 0)",
    }
    yard = None
    if rank == 0:
        a16 = torch.randn(8192, 8192, device=dev).half()
        b16 = torch.randn(8192, 8192, device=dev).half()
        c16 = torch.empty_like(a16)
        for _ in range(3):
            torch.matmul(a16, b16, out=c16)
        reps = 150
        t_y = _time(lambda: [torch.matmul(a16, b16, out=c16) for _ in range(reps)], reps=2)
        yard = {"tflops": 2.0 * 8192 ** 3 * reps / (t_y * 1e-3) / 1e12,
                "what": "torch.matmul FP16 8192^3 (cuBLAS), 150 back-to-back calls (~0.13 s), same process and box"}
        del a16, b16, c16

    # ---- NEXT-1 row: final refinement (Eq. 16) + energy on the last solve's D (outside the timed step)
    refine = None
    if rank == 0:
        _, info_r = solve()
        t_r = _time(lambda: h.refine_energy(D, info_r["sigma"][-1], H, stream=stream), reps=3)
        D1, res = h.refine_energy(D, info_r["sigma"][-1], H, stream=stream)
        e_star = float(np.sort(w.eps)[: int(w.N_occ)].sum())
        refine = {"ms": t_r, "energy_err_in": res["energy_in"] - e_star, "energy_err_out": res["energy_out"] - e_star,
                  "iderr_in": res["iderr_in"], "iderr_out": res["iderr_out"],
                  "trace_minus_nocc_out": res["trace_out"] - w.N_occ,
                  "max_err_256_sampled_entries_vs_closed_form_out":
                      float(np.abs(D1.double()[ri, ci].cpu().numpy() - ref).max()),
                  "what": "sp2_refine_energy: 2 enhanced-accumulation layers (128x128 tiles, library default of 4 K-blocks "
                          "per tensor-core chunk, two-sum running pair in TMEM) + 2 Tr[XH] passes"}
        del D1
        # the caller's accuracy / speed knob: 2 K-blocks per chunk (twice the folds of the running pair; the default
        # until round 3)
        o4 = api.make_opts()
        o4.enh_kc = 2
        t_r4 = _time(lambda: h.refine_energy(D, info_r["sigma"][-1], H, stream=stream, opts=o4), reps=3)
        D4, res4 = h.refine_energy(D, info_r["sigma"][-1], H, stream=stream, opts=o4)
        refine["enh_kc_2"] = {"ms": t_r4, "energy_err_out": res4["energy_out"] - e_star, "iderr_out": res4["iderr_out"],
                              "trace_minus_nocc_out": res4["trace_out"] - w.N_occ,
                              "max_err_256_sampled_entries_vs_closed_form_out":
                                  float(np.abs(D4.double()[ri, ci].cpu().numpy() - ref).max())}
        del D4

    # ---- NEXT-3 row: accelerated Deep-NN SP2 (section V.A) with HOMO/LUMO estimates 1 % inside the known gap
    accel = None
    if rank == 0:
        es = np.sort(w.eps)
        no = int(w.N_occ)
        g = es[no] - es[no - 1]
        o_acc = api.make_opts(bounds=bounds, tol=w.tol, max_layers=w.max_layers, tile_config=args.tile,
                              control=args.control, exact_diag=args.exact_diag,
                              homo_lumo=(es[no - 1] + 0.01 * g, es[no] - 0.01 * g))
        t_a = _time(lambda: h.density_matrix(H, w.N_occ, o_acc, out=D, stream=stream), reps=3)
        _, ia = h.density_matrix(H, w.N_occ, o_acc, out=D, stream=stream)
        accel = {"ms_per_converged_D": t_a, "layers": ia["n_layers"], "layers_standard": n_layers,
                 "stop_reason": api.STOP_NAMES.get(ia["stop_reason"]),
                 "trace_minus_nocc": float(torch.trace(D.double()).item()) - w.N_occ,
                 "max_err_256_sampled_entries_vs_closed_form": float(np.abs(D.double()[ri, ci].cpu().numpy() - ref).max())}

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D + solve + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        Hh = torch.from_numpy(w.H32).pin_memory()
        Dh = torch.empty((N, N), dtype=torch.float32).pin_memory()
        h.density_matrix_host(Hh, w.N_occ, opts, out=Dh, stream=stream)
        _barrier(world)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k2, lay2 = max(1, min(args.steps, 3)), 0
        ph = []
        a.record(stream)
        for _ in range(k2):
            _, i2 = h.density_matrix_host(Hh, w.N_occ, opts, out=Dh, stream=stream)
            lay2 += i2["n_layers"]
            ph.append((i2["h2d_ms"], i2["solve_ms"], i2["d2h_ms"]))
        b.record(stream)
        torch.cuda.synchronize()
        t2 = _max_over_ranks(a.elapsed_time(b) * 1e-3, world)
        ph = np.median(np.array(ph), axis=0)
        nb_in, nb = int(i2["h2d_bytes"]), int(i2["d2h_bytes"])      # counted by the library from the copies it enqueued
        e2e = {"value": world * 6.0 * N ** 3 * lay2 / t2 / 1e12, "unit": UNIT, "ms_per_step": t2 / k2 * 1e3,
               "h2d_bytes_per_step": nb_in, "d2h_bytes_per_step": nb,
               "h2d_what": "lower triangle of H only (the library reads nothing else), in bands of 256 rows",
               "h2d_ms": float(ph[0]), "solve_ms": float(ph[1]), "d2h_ms": float(ph[2]),
               "h2d_GBps": nb_in / (ph[0] * 1e-3) / 1e9, "d2h_GBps": nb / (ph[2] * 1e-3) / 1e9,
               "phases_how": "CUDA events recorded by the library around each phase of the same calls (median)",
               "api": "sp2_density_matrix_host (pinned host buffers)"}
        del Hh, Dh

    configs = sparse4 = mix2 = sweep = None
    if rank == 0 and not args.no_configs:
        h.close()
        del H, D
        torch.cuda.empty_cache()
        configs = other_configs(api, W, torch, dev, stream, _time)
        sparse4, mix2, sweep = next_rows_and_sweep(api, W, torch, dev, stream, _time, float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])))
        h = None

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_oracle_sample(w)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f16 operands (hi/lo split), f32 accumulate",
            "data": "synthetic",
            "config": {"workload": f"config3: gapped dense symmetric H = Q diag(eps) Q^T, N={N}, N_occ={int(w.N_occ)}, "
                                   f"seed {args.seed} (BASELINE.json configs[2])",
                       "bounds": "Gershgorin on device" if bounds is None else f"explicit {bounds}",
                       "tol": w.tol, "max_layers": w.max_layers, "tile_config": args.tile, "control": args.control,
                       "exact_diag": args.exact_diag,
                       "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "single GPU",
                       "l2": "inputs (1 GiB H, 3 GiB workspace) exceed the 126 MB L2; no flush needed"},
            "detail": {"layers_per_solve": n_layers, "ms_per_converged_D": ms_per_step,
                       "ms_per_layer": t_layer_ms, "executed_tflops_3N3": exec_tflops,
                       "paper_count_tflops_4N3": 4.0 * N ** 3 / (t_layer_ms * 1e-3) / 1e12,
                       "effective_tflops_6N3_per_layer": 6.0 * N ** 3 / (t_layer_ms * 1e-3) / 1e12,
                       "frac_of_datasheet_2250": exec_tflops / 2250.0,
                       "frac_of_measured_burst": exec_tflops / float(peaks["bf16_tflops"]),
                       "stop_reason": api.STOP_NAMES.get(info_timed["stop_reason"]), "bounds_used": info_timed["bounds"],
                       "trace_minus_nocc": tr - w.N_occ, "max_err_256_sampled_entries_vs_closed_form": samp_err,
                       "D_exactly_symmetric": symmetric,
                       "frac_of_same_run_cublas_fp16": (exec_tflops / yard["tflops"]) if yard else None,
                       "cublas_fp16_yardstick": yard, "hbm_kernels": hbm_kernels, "refinement_next1": refine, "accelerated_next3": accel,
                       "blocked_sparse_next4": sparse4, "mix_next2": mix2, "size_sweep": sweep,
                       "configs": configs,
                       "paper_context": "paper: ~120 TFLOP/s on A100 (P:204), other hardware, count unstated",
                       "wall_s_timed_region": t_wall},
            "clocks": clocks, "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu,
            "gpu_launches": int(launches),
        }
        print(json.dumps(line))
    if h is not None:
        h.close()
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()


if __name__ == "__main__":
    main()
