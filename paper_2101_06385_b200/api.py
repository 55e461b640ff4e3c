"""Thin ctypes binding over libsp2b200.so (include/sp2_b200.h): argument marshalling only.

torch supplies device memory and the stream; every step of the path runs in the library's kernels.
There is no CPU fallback: a missing library or a non-CUDA tensor raises."""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsp2b200.so")

SP2_OK, SP2_NOT_CONVERGED = 0, 1
STOP_NAMES = {0: "none", 1: "iderr<=0", 2: "param_free", 3: "tol", 4: "max_layers", 5: "nonfinite", 6: "noise_floor"}
TILE_AUTO, TILE_128x128, TILE_128x256, TILE_256x256_PAIR, TILE_128x128_ENH = 0, 1, 2, 3, 4

EXPORTS = ["sp2_default_opts", "sp2_create", "sp2_destroy", "sp2_workspace_bytes", "sp2_workspace_bytes_lazy",
           "sp2_density_matrix", "sp2_density_matrix_host", "sp2_generalized", "sp2_generalized_mix", "sp2_generalized_wb",
           "sp2_density_matrix_batched", "sp2_generalized_batched", "sp2_refine_energy", "sp2_split_fp16",
           "sp2_gershgorin", "sp2_status_string", "sp2_last_cuda_error", "sp2_last_launch_count",
           "sp2_last_host_timing", "sp2_last_host_bytes", "sp2_last_round_sync_broken", "sp2_last_sparse_work", "sp2_version",
           "sp2_gershgorin_static", "sp2_gershgorin_static_max_n", "sp2_gershgorin_static_bytes",
           "sp2_gershgorin_static_last_error"]


class LayerStat(C.Structure):
    _fields_ = [("trace_S", C.c_double), ("trace_X", C.c_double), ("trace_X_diag", C.c_double),
                ("iderr", C.c_double), ("sigma", C.c_int), ("stop_reason", C.c_int), ("t_end_ns", C.c_ulonglong)]


class Opts(C.Structure):
    _fields_ = [("auto_bounds", C.c_int), ("eps_min", C.c_double), ("eps_max", C.c_double), ("tol", C.c_double),
                ("max_layers", C.c_int), ("eps_alt", C.c_double), ("fp16_scale_log2", C.c_int),
                ("control", C.c_int), ("tile_config", C.c_int), ("exact_diag", C.c_int), ("accelerated", C.c_int),
                ("homo", C.c_double), ("lumo", C.c_double), ("noise_kappa", C.c_double), ("enh_kc", C.c_int),
                ("trunc_tau", C.c_double)]


class RefineResult(C.Structure):
    _fields_ = [("energy_in", C.c_double), ("trace_in", C.c_double), ("iderr_in", C.c_double),
                ("energy_out", C.c_double), ("trace_out", C.c_double), ("iderr_out", C.c_double)]


class SP2Error(RuntimeError):
    def __init__(self, status: int, where: str):
        lib = load()
        msg = lib.sp2_status_string(status).decode()
        if status == -5:
            msg += ": " + lib.sp2_last_cuda_error().decode()
        super().__init__(f"{where}: {msg}")
        self.status = status


_lib = None


def load() -> C.CDLL:
    """Load the C-ABI library (built in-tree by __graft_entry__.build / build.py).  Raises if missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(nvcc, sm_100a). There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, ip, dp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)
    lib.sp2_default_opts.argtypes = [C.POINTER(Opts)]; lib.sp2_default_opts.restype = None
    lib.sp2_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int]; lib.sp2_create.restype = C.c_int
    lib.sp2_destroy.argtypes = [vp]; lib.sp2_destroy.restype = C.c_int
    lib.sp2_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int]; lib.sp2_workspace_bytes.restype = C.c_size_t
    lib.sp2_workspace_bytes_lazy.argtypes = [C.c_int]; lib.sp2_workspace_bytes_lazy.restype = C.c_size_t
    lib.sp2_density_matrix.argtypes = [vp, vp, C.c_int, C.c_int, C.c_double, C.POINTER(Opts), vp, C.c_int,
                                       C.POINTER(LayerStat), ip, dp, vp]
    lib.sp2_density_matrix.restype = C.c_int
    lib.sp2_density_matrix_host.argtypes = lib.sp2_density_matrix.argtypes
    lib.sp2_density_matrix_host.restype = C.c_int
    lib.sp2_generalized.argtypes = [vp, vp, C.c_int, C.c_int, dp, C.c_int, C.c_double, C.c_double,
                                    C.POINTER(Opts), vp, C.c_int, C.POINTER(LayerStat), vp]
    lib.sp2_generalized.restype = C.c_int
    lib.sp2_generalized_mix.argtypes = [vp, vp, C.c_int, C.c_int, dp, dp, C.c_int, C.c_double, C.c_double,
                                        C.POINTER(Opts), vp, C.c_int, C.POINTER(LayerStat), vp]
    lib.sp2_generalized_mix.restype = C.c_int
    lib.sp2_generalized_wb.argtypes = [vp, vp, C.c_int, C.c_int, ip, dp, dp, C.c_int, C.c_double, C.c_double,
                                       C.POINTER(Opts), vp, C.c_int, C.POINTER(LayerStat), vp]
    lib.sp2_generalized_wb.restype = C.c_int
    lib.sp2_density_matrix_batched.argtypes = [vp, vp, C.c_int, C.c_int, dp, C.c_int, dp, C.POINTER(Opts), vp,
                                               C.POINTER(LayerStat), ip, ip, vp]
    lib.sp2_density_matrix_batched.restype = C.c_int
    lib.sp2_generalized_batched.argtypes = [vp, vp, C.c_int, C.c_int, dp, C.c_int, C.c_double, C.c_double,
                                            C.POINTER(Opts), vp, C.POINTER(LayerStat), ip, vp]
    lib.sp2_generalized_batched.restype = C.c_int
    lib.sp2_refine_energy.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, vp, C.c_int, C.POINTER(Opts), vp, C.c_int,
                                      C.POINTER(RefineResult), vp]
    lib.sp2_refine_energy.restype = C.c_int
    lib.sp2_split_fp16.argtypes = [vp, C.c_int, C.c_int, vp, vp, C.c_int, C.c_int, vp]
    lib.sp2_split_fp16.restype = C.c_int
    lib.sp2_gershgorin.argtypes = [vp, vp, C.c_int, C.c_int, dp, vp]; lib.sp2_gershgorin.restype = C.c_int
    lib.sp2_status_string.argtypes = [C.c_int]; lib.sp2_status_string.restype = C.c_char_p
    lib.sp2_last_cuda_error.argtypes = []; lib.sp2_last_cuda_error.restype = C.c_char_p
    lib.sp2_last_launch_count.argtypes = [vp]; lib.sp2_last_launch_count.restype = C.c_int
    lib.sp2_last_round_sync_broken.argtypes = [vp]; lib.sp2_last_round_sync_broken.restype = C.c_int
    lib.sp2_last_host_timing.argtypes = [vp, dp]; lib.sp2_last_host_timing.restype = None
    lib.sp2_last_sparse_work.argtypes = [vp, dp]; lib.sp2_last_sparse_work.restype = None
    lib.sp2_last_host_bytes.argtypes = [vp, dp]; lib.sp2_last_host_bytes.restype = None
    lib.sp2_version.argtypes = []; lib.sp2_version.restype = C.c_char_p
    lib.sp2_gershgorin_static.argtypes = [vp, C.c_int, C.c_int, vp, vp]; lib.sp2_gershgorin_static.restype = C.c_int
    lib.sp2_gershgorin_static_max_n.argtypes = []; lib.sp2_gershgorin_static_max_n.restype = C.c_int
    lib.sp2_gershgorin_static_bytes.argtypes = []; lib.sp2_gershgorin_static_bytes.restype = C.c_size_t
    lib.sp2_gershgorin_static_last_error.argtypes = []; lib.sp2_gershgorin_static_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _stream_ptr(stream) -> int:
    import torch

    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dev_f32(t, name):
    import torch

    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.stride(-1) == 1):
        raise TypeError(f"{name} must be a CUDA float32 tensor with unit inner stride (no CPU fallback)")
    return t


def _stats_to_dict(stats, n):
    keys = ("trace_S", "trace_X", "trace_X_diag", "iderr", "sigma", "stop_reason", "t_end_ns")
    return {k: [getattr(stats[i], k) for i in range(n)] for k in keys}


def make_opts(bounds=None, tol=0.0, max_layers=120, eps_alt=0.0, fp16_scale_log2=-1, control=0, tile_config=0,
              exact_diag=1, homo_lumo=None, noise_kappa=-1.0, enh_kc=0, trunc_tau=0.0, accelerated=None) -> Opts:
    o = Opts()
    load().sp2_default_opts(C.byref(o))
    if bounds is not None:
        o.auto_bounds, o.eps_min, o.eps_max = 0, float(bounds[0]), float(bounds[1])
    o.tol, o.max_layers, o.eps_alt = float(tol), int(max_layers), float(eps_alt)
    o.fp16_scale_log2, o.control, o.tile_config = int(fp16_scale_log2), int(control), int(tile_config)
    o.exact_diag = int(exact_diag)
    o.noise_kappa, o.enh_kc, o.trunc_tau = float(noise_kappa), int(enh_kc), float(trunc_tau)
    if homo_lumo is not None:        # accelerated Deep-NN SP2 (section V.A)
        o.accelerated, o.homo, o.lumo = 1, float(homo_lumo[0]), float(homo_lumo[1])
    if accelerated is not None:      # batched call: the estimates travel as a per-matrix array
        o.accelerated = int(accelerated)
    return o


class Handle:
    """Owns the library workspace for problems up to N_max (and batches of batch_max matrices)."""

    def __init__(self, N_max: int, batch_max: int = 0, max_layers: int = 120):
        self.lib = load()
        self._h = C.c_void_p()
        self.max_layers = max_layers
        st = self.lib.sp2_create(C.byref(self._h), N_max, batch_max, max_layers)
        if st != 0:
            raise SP2Error(st, "sp2_create")

    def close(self):
        if self._h:
            self.lib.sp2_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- Alg. 1
    def density_matrix(self, H, N_occ, opts: Optional[Opts] = None, out=None, stream=None, check=True):
        import torch

        H = _dev_f32(H, "H")
        N = H.shape[0]
        opts = opts or make_opts()
        D = torch.empty((N, N), dtype=torch.float32, device=H.device) if out is None else _dev_f32(out, "out")
        stats = (LayerStat * opts.max_layers)()
        nl = C.c_int(0)
        bounds = (C.c_double * 2)()
        st = self.lib.sp2_density_matrix(self._h, H.data_ptr(), N, H.stride(0), float(N_occ), C.byref(opts),
                                         D.data_ptr(), D.stride(0), stats, C.byref(nl), bounds, _stream_ptr(stream))
        if st < 0 and check:
            raise SP2Error(st, "sp2_density_matrix")
        info = _stats_to_dict(stats, nl.value)
        info.update(status=st, n_layers=nl.value, bounds=(bounds[0], bounds[1]),
                    stop_reason=(info["stop_reason"][-1] if nl.value else 0),
                    launches=self.lib.sp2_last_launch_count(self._h))
        if opts.trunc_tau > 0.0:
            wk = (C.c_double * 2)()
            self.lib.sp2_last_sparse_work(self._h, wk)
            info["work_fraction"] = (wk[0] / wk[1]) if wk[1] > 0 else 1.0
        return D, info

    def density_matrix_host(self, H_host: np.ndarray, N_occ, opts: Optional[Opts] = None, out=None, stream=None):
        """Host buffers in, host buffers out (H2D and D2H inside the call)."""
        def _ptr(a):
            return a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr()

        if isinstance(H_host, np.ndarray):
            H_host = np.ascontiguousarray(H_host, dtype=np.float32)
        elif H_host.is_cuda or not H_host.is_contiguous():
            raise TypeError("H_host must be a contiguous host buffer (numpy array or CPU torch tensor)")
        N = H_host.shape[0]
        opts = opts or make_opts()
        D = np.empty((N, N), dtype=np.float32) if out is None else out
        stats = (LayerStat * opts.max_layers)()
        nl = C.c_int(0)
        bounds = (C.c_double * 2)()
        st = self.lib.sp2_density_matrix_host(self._h, _ptr(H_host), N, N, float(N_occ), C.byref(opts),
                                              _ptr(D), N, stats, C.byref(nl), bounds, _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_density_matrix_host")
        info = _stats_to_dict(stats, nl.value)
        ms = (C.c_double * 3)()
        self.lib.sp2_last_host_timing(self._h, ms)
        nbytes = (C.c_double * 2)()
        self.lib.sp2_last_host_bytes(self._h, nbytes)
        info.update(status=st, n_layers=nl.value, bounds=(bounds[0], bounds[1]),
                    h2d_ms=ms[0], solve_ms=ms[1], d2h_ms=ms[2], h2d_bytes=int(nbytes[0]), d2h_bytes=int(nbytes[1]))
        return D, info

    # -- generalized network
    def generalized(self, H, theta: np.ndarray, bounds=None, opts: Optional[Opts] = None, stream=None):
        import torch

        H = _dev_f32(H, "H")
        N = H.shape[0]
        theta = np.ascontiguousarray(theta, dtype=np.float64)
        L = theta.shape[0]
        X = torch.empty((N, N), dtype=torch.float32, device=H.device)
        stats = (LayerStat * L)()
        e0, e1 = (0.0, 0.0) if bounds is None else (float(bounds[0]), float(bounds[1]))
        st = self.lib.sp2_generalized(self._h, H.data_ptr(), N, H.stride(0),
                                      theta.ctypes.data_as(C.POINTER(C.c_double)), L, e0, e1,
                                      C.byref(opts) if opts is not None else None, X.data_ptr(), X.stride(0), stats,
                                      _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_generalized")
        info = _stats_to_dict(stats, L)
        info.update(status=st, n_layers=L)
        return X, info

    def generalized_mix(self, H, theta: np.ndarray, c: np.ndarray, bounds=None, opts: Optional[Opts] = None,
                        stream=None):
        """F~(H) = I - sum_i c_i S_i (Eqs. 17-18): theta [L][3], c [L+1]."""
        import torch

        H = _dev_f32(H, "H")
        N = H.shape[0]
        theta = np.ascontiguousarray(theta, dtype=np.float64)
        c = np.ascontiguousarray(c, dtype=np.float64)
        L = theta.shape[0]
        if c.shape != (L + 1,):
            raise ValueError("c must have L + 1 entries (c_0 weights S_0)")
        F = torch.empty((N, N), dtype=torch.float32, device=H.device)
        stats = (LayerStat * L)()
        e0, e1 = (0.0, 0.0) if bounds is None else (float(bounds[0]), float(bounds[1]))
        st = self.lib.sp2_generalized_mix(self._h, H.data_ptr(), N, H.stride(0),
                                          theta.ctypes.data_as(C.POINTER(C.c_double)),
                                          c.ctypes.data_as(C.POINTER(C.c_double)), L, e0, e1,
                                          C.byref(opts) if opts is not None else None, F.data_ptr(), F.stride(0),
                                          stats, _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_generalized_mix")
        info = _stats_to_dict(stats, L)
        info.update(status=st, n_layers=L)
        return F, info

    def generalized_wb(self, H, sigma: Optional[Sequence[int]], weights, biases, bounds=None,
                       opts: Optional[Opts] = None, stream=None):
        import torch

        H = _dev_f32(H, "H")
        N = H.shape[0]
        w = np.ascontiguousarray(weights, dtype=np.float64)
        b = np.ascontiguousarray(biases, dtype=np.float64)
        L = w.shape[0]
        sg = None if sigma is None else np.ascontiguousarray(sigma, dtype=np.int32)
        X = torch.empty((N, N), dtype=torch.float32, device=H.device)
        stats = (LayerStat * L)()
        e0, e1 = (0.0, 0.0) if bounds is None else (float(bounds[0]), float(bounds[1]))
        st = self.lib.sp2_generalized_wb(self._h, H.data_ptr(), N, H.stride(0),
                                         None if sg is None else sg.ctypes.data_as(C.POINTER(C.c_int)),
                                         w.ctypes.data_as(C.POINTER(C.c_double)),
                                         b.ctypes.data_as(C.POINTER(C.c_double)), L, e0, e1,
                                         C.byref(opts) if opts is not None else None, X.data_ptr(), X.stride(0),
                                         stats, _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_generalized_wb")
        info = _stats_to_dict(stats, L)
        info.update(status=st, n_layers=L)
        return X, info

    # -- final refinement + energy (Eq. 16)
    def refine_energy(self, S, last_sigma: int, H, out=None, stream=None, opts: Optional[Opts] = None):
        """D' = f_final(S) in enhanced precision and the observables of S and D' against H."""
        import torch

        S = _dev_f32(S, "S")
        H = _dev_f32(H, "H")
        N = S.shape[0]
        D = torch.empty((N, N), dtype=torch.float32, device=S.device) if out is None else _dev_f32(out, "out")
        res = RefineResult()
        st = self.lib.sp2_refine_energy(self._h, S.data_ptr(), N, S.stride(0), int(last_sigma), H.data_ptr(),
                                        H.stride(0), C.byref(opts) if opts is not None else None, D.data_ptr(),
                                        D.stride(0), C.byref(res), _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_refine_energy")
        return D, {k: getattr(res, k) for k, _ in RefineResult._fields_}

    # -- batched small-N
    def density_matrix_batched(self, H, N_occ, opts: Optional[Opts] = None, out=None, stream=None, homo_lumo=None):
        """homo_lumo: None, or a [B, 2] array of per-matrix HOMO / LUMO estimates (accelerated weights, section V.A)."""
        import torch

        H = _dev_f32(H, "H")
        if H.dim() != 3 or not H.is_contiguous():
            raise TypeError("H must be a contiguous [B, N, N] CUDA float32 tensor")
        B, N = H.shape[0], H.shape[1]
        opts = opts or make_opts()
        D = torch.empty_like(H) if out is None else out
        scalar = np.isscalar(N_occ)
        nocc = np.ascontiguousarray([N_occ] if scalar else N_occ, dtype=np.float64)
        hl = None
        if homo_lumo is not None:
            hl = np.ascontiguousarray(homo_lumo, dtype=np.float64)
            if hl.shape != (B, 2):
                raise ValueError("homo_lumo must have shape [B, 2]")
            opts.accelerated = 1
        stats = (LayerStat * (B * opts.max_layers))()
        nl = (C.c_int * B)()
        status = (C.c_int * B)()
        st = self.lib.sp2_density_matrix_batched(self._h, H.data_ptr(), N, B, nocc.ctypes.data_as(C.POINTER(C.c_double)),
                                                 1 if scalar else 0,
                                                 None if hl is None else hl.ctypes.data_as(C.POINTER(C.c_double)),
                                                 C.byref(opts), D.data_ptr(), stats, nl, status, _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_density_matrix_batched")
        n_layers = np.frombuffer(nl, dtype=np.int32).copy()
        return D, {"status": st, "n_layers": n_layers, "per_status": np.frombuffer(status, dtype=np.int32).copy(),
                   "stats": stats, "max_layers": opts.max_layers}

    def generalized_batched(self, H, theta: np.ndarray, bounds=None, opts: Optional[Opts] = None, out=None, stream=None):
        """The same L generalized layers (theta [L][3]) applied to each matrix of H [B, N, N], N <= 256."""
        import torch

        H = _dev_f32(H, "H")
        if H.dim() != 3 or not H.is_contiguous():
            raise TypeError("H must be a contiguous [B, N, N] CUDA float32 tensor")
        B, N = H.shape[0], H.shape[1]
        theta = np.ascontiguousarray(theta, dtype=np.float64)
        L = theta.shape[0]
        X = torch.empty_like(H) if out is None else out
        stats = (LayerStat * (B * L))()
        status = (C.c_int * B)()
        e0, e1 = (0.0, 0.0) if bounds is None else (float(bounds[0]), float(bounds[1]))
        st = self.lib.sp2_generalized_batched(self._h, H.data_ptr(), N, B, theta.ctypes.data_as(C.POINTER(C.c_double)),
                                              L, e0, e1, C.byref(opts) if opts is not None else None, X.data_ptr(),
                                              stats, status, _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_generalized_batched")
        return X, {"status": st, "per_status": np.frombuffer(status, dtype=np.int32).copy(), "stats": stats,
                   "max_layers": L, "n_layers": np.full(B, L, dtype=np.int32)}

    def gershgorin(self, H, stream=None):
        H = _dev_f32(H, "H")
        out = (C.c_double * 2)()
        st = self.lib.sp2_gershgorin(self._h, H.data_ptr(), H.shape[0], H.stride(0), out, _stream_ptr(stream))
        if st < 0:
            raise SP2Error(st, "sp2_gershgorin")
        return out[0], out[1]


def shard_range(n_items: int, rank: int, world: int):
    """Contiguous [start, stop) slice of a batch of independent matrices owned by `rank` of `world` processes
    (one process per GPU).  The batched path shards with no data-path collective:
    the first n_items % world ranks get one extra item."""
    if world < 1 or not (0 <= rank < world) or n_items < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_items, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def batched_stats(info, m: int):
    """Per-layer statistics of matrix m of a batched solve."""
    n = int(info["n_layers"][m])
    base = m * info["max_layers"]
    keys = ("trace_S", "trace_X", "trace_X_diag", "iderr", "sigma", "stop_reason", "t_end_ns")
    return {k: [getattr(info["stats"][base + i], k) for i in range(n)] for k in keys}


def split_fp16(X, fp16_scale_log2: int = 0, stream=None):
    """Eqs. 12-13: returns (hi, lo) as CUDA float16 tensors."""
    import torch

    X = _dev_f32(X, "X")
    N = X.shape[0]
    hi = torch.empty((N, N), dtype=torch.float16, device=X.device)
    lo = torch.empty((N, N), dtype=torch.float16, device=X.device)
    st = load().sp2_split_fp16(X.data_ptr(), N, X.stride(0), hi.data_ptr(), lo.data_ptr(), N, fp16_scale_log2,
                               _stream_ptr(stream))
    if st < 0:
        raise SP2Error(st, "sp2_split_fp16")
    return hi, lo


def gershgorin_static(H, out, stream=None):
    """Gershgorin bounds of H through sp2_gershgorin_static: the variant for callers that cannot allocate device memory
    (their own arena owns HBM, or a cudaMalloc's device-wide synchronisation is not acceptable where they call from).
    No handle: the scratch is a static device array inside the library, which limits N to sp2_gershgorin_static_max_n()
    (4096).  `out` is the CALLER's CUDA float64 tensor of 2 elements and receives {eps_min, eps_max}; nothing is
    allocated here either, and the call does not synchronise -- read `out` after synchronising `stream`.  Calls share
    the one scratch array: do not let two of them overlap on the GPU."""
    import torch

    H = _dev_f32(H, "H")
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.numel() == 2
            and out.is_contiguous()):
        raise TypeError("out must be a contiguous CUDA float64 tensor of 2 elements (the caller owns the output)")
    lib = load()
    st = lib.sp2_gershgorin_static(H.data_ptr(), H.shape[0], H.stride(0), out.data_ptr(), _stream_ptr(stream))
    if st < 0:
        raise RuntimeError(f"{lib.sp2_status_string(st).decode()}: {lib.sp2_gershgorin_static_last_error().decode()}")
    return out
