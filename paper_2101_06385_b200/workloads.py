"""Seeded synthetic inputs for the SP2 hot path (shared by tests, bench.py and smoke()).

This module holds NONE of the method's arithmetic (no SP2 layer, no split, no bounds):
it only builds Hamiltonians with a known spectrum, following the five recipes of
BASELINE.json `configs` as made concrete in SURVEY.md section 8(d) / DESIGN.md "Input recipe".
The paper itself measures on unspecified random test Hamiltonians (PAPER.md line 175, 202,
234), so these are stand-ins of the same shape (dense symmetric H with a gap at N_occ).

Every generator draws from ``numpy.random.default_rng(seed)`` (PCG64) in a fixed order,
builds H in FP64, symmetrises it and rounds ONCE to FP32; the same FP32 bytes go to the
oracle and to the CUDA path.  Orthogonal factors come from a Householder QR of a seeded
standard-normal matrix (sign-fixed so that Q is Haar distributed); for large N the QR may
run on a CUDA device through torch (harness-side plumbing only).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np


@dataclasses.dataclass
class Workload:
    """One synthetic problem.  `H32` is what both the oracle and the library receive."""

    name: str
    H32: np.ndarray                      # (N, N) or (B, N, N) float32, symmetric
    N: int
    N_occ: float
    eps: Optional[np.ndarray] = None     # known eigenvalues (FP64), occupied first; None if unknown
    Q: Optional[np.ndarray] = None       # known eigenvectors (FP64 columns), same order as eps
    bounds: Optional[tuple] = None       # explicit spectral bounds enclosing eps, or None (auto)
    tol: float = 1e-5
    max_layers: int = 120
    extra: dict = dataclasses.field(default_factory=dict)


def _sym32(H: np.ndarray) -> np.ndarray:
    H = 0.5 * (H + np.swapaxes(H, -1, -2))
    return np.ascontiguousarray(H.astype(np.float32))


def haar_orthogonal(rng: np.random.Generator, n: int, device: Optional[str] = None) -> np.ndarray:
    """Orthogonal factor of the Householder QR of an n x n standard-normal matrix, with the
    columns sign-fixed by sign(diag R).  `device` = a torch device string runs the QR there."""
    A = rng.standard_normal((n, n))
    if device is None:
        Q, R = np.linalg.qr(A)
        d = np.sign(np.diag(R))
        d[d == 0] = 1.0
        return Q * d[None, :]
    import torch

    At = torch.from_numpy(A).to(device)
    Qt, Rt = torch.linalg.qr(At)
    d = torch.sign(torch.diagonal(Rt))
    d[d == 0] = 1.0
    return (Qt * d[None, :]).cpu().numpy()


def _from_spectrum(Q: np.ndarray, eps: np.ndarray, device: Optional[str] = None) -> np.ndarray:
    if device is None:
        return (Q * eps[None, :]) @ Q.T
    import torch

    Qt = torch.from_numpy(Q).to(device)
    et = torch.from_numpy(eps).to(device)
    return ((Qt * et[None, :]) @ Qt.T).cpu().numpy()


def gapped_dense(seed: int, n: int, lo_band: tuple, hi_band: tuple, n_occ: int, name: str,
                 bounds: Optional[tuple], tol: float = 1e-5, max_layers: int = 120,
                 device: Optional[str] = None, rng: Optional[np.random.Generator] = None) -> Workload:
    """H = Q diag(eps) Q^T with n_occ eigenvalues U(lo_band) (occupied) and the rest U(hi_band)."""
    rng = np.random.default_rng(seed) if rng is None else rng
    Q = haar_orthogonal(rng, n, device)
    eps = np.concatenate([rng.uniform(lo_band[0], lo_band[1], n_occ),
                          rng.uniform(hi_band[0], hi_band[1], n - n_occ)])
    H = _from_spectrum(Q, eps, device)
    return Workload(name=name, H32=_sym32(H), N=n, N_occ=float(n_occ), eps=eps, Q=Q, bounds=bounds,
                    tol=tol, max_layers=max_layers, extra={"seed": seed})


def config1(seed: int = 0, n: int = 128) -> Workload:
    """BASELINE.json configs[0]: N=128, gap 0.2 around 0, N_occ=N/2, tol 1e-5, max 60 layers."""
    h = n // 2
    return gapped_dense(seed, n, (-1.0, -0.1), (0.1, 1.0), h, f"cfg1_gapped_N{n}", bounds=(-1.0, 1.0),
                        tol=1e-5, max_layers=60)


def config2(seed: int = 0, n_sites: int = 512) -> Workload:
    """BASELINE.json configs[1]: tight-binding-like H, n_sites uniform in a periodic cube of density
    0.1 / A^3, 4 orbitals per site, onsite -0.5 (orbitals 0,1) / +0.5 (orbitals 2,3), hopping
    -2.0 exp(-r/1.5) N(1,0.1) for r < 6 A between every inter-site orbital pair (reading C21)."""
    rng = np.random.default_rng(seed)
    L = (n_sites / 0.1) ** (1.0 / 3.0)
    pos = rng.uniform(0.0, L, (n_sites, 3))
    d = pos[:, None, :] - pos[None, :, :]
    d -= L * np.round(d / L)                       # minimum image
    r = np.sqrt((d * d).sum(-1))
    n = 4 * n_sites
    H = np.zeros((n, n))
    ia, ib = np.where(np.triu(r < 6.0, k=1))       # site pairs a < b, row-major order
    fac = rng.normal(1.0, 0.1, (ia.size, 4, 4))
    blk = -2.0 * np.exp(-r[ia, ib] / 1.5)[:, None, None] * fac
    for k in range(ia.size):
        a, b = 4 * ia[k], 4 * ib[k]
        H[a:a + 4, b:b + 4] = blk[k]
        H[b:b + 4, a:a + 4] = blk[k].T
    onsite = np.tile(np.array([-0.5, -0.5, 0.5, 0.5]), n_sites)
    H[np.arange(n), np.arange(n)] = onsite
    return Workload(name=f"cfg2_tightbinding_N{n}", H32=_sym32(H), N=n, N_occ=float(n // 2), bounds=None,
                    tol=1e-5, max_layers=120,
                    extra={"seed": seed, "box": L, "nnz_per_row": float((H != 0).sum() / n)})


def config3(seed: int = 0, n: int = 16384, device: Optional[str] = None) -> Workload:
    """BASELINE.json configs[2]: N=16384 gapped dense H, half eps U(-2,-0.05), half U(0.05,2)."""
    h = n // 2
    return gapped_dense(seed, n, (-2.0, -0.05), (0.05, 2.0), h, f"cfg3_gapped_N{n}", bounds=(-2.0, 2.0),
                        tol=1e-5, max_layers=120, device=device)


def config3_lowrank(seed: int = 0, n: int = 16384, k: int = 16) -> Workload:
    """Smoke-test stand-in for config 3: k Householder reflectors applied to diag(eps), O(k N^2).
    NOT representative (diagonal + low rank); never used for a reported number."""
    rng = np.random.default_rng(seed)
    h = n // 2
    eps = np.concatenate([rng.uniform(-2.0, -0.05, h), rng.uniform(0.05, 2.0, n - h)])
    H = np.diag(eps)
    Q = np.eye(n)
    for _ in range(k):
        v = rng.standard_normal(n)
        v /= np.linalg.norm(v)
        H -= 2.0 * np.outer(v, v @ H)
        H -= 2.0 * np.outer(H @ v, v)
        Q -= 2.0 * np.outer(v, v @ Q)     # H <- P H P with P = I - 2 v v^T symmetric, so Q <- P Q
    return Workload(name=f"cfg3_lowrank_N{n}", H32=_sym32(H), N=n, N_occ=float(h), eps=eps, Q=Q,
                    bounds=(-2.0, 2.0), tol=1e-5, max_layers=120, extra={"seed": seed, "reflectors": k})


def config4(seed: int = 0, n: int = 4096, layers: int = 30, device: Optional[str] = None) -> Workload:
    """BASELINE.json configs[3]: gapless eps ~ U(-1,1); per-layer weight w_n = 1 + N(0,0.02) and bias
    b_n = N(0,0.005).  The per-layer branch sigma_n is NOT drawn here: the harness derives it from the
    scalar recursion (reading C19) so that this module stays free of the method's arithmetic."""
    rng = np.random.default_rng(seed)
    Q = haar_orthogonal(rng, n, device)
    eps = rng.uniform(-1.0, 1.0, n)
    w = 1.0 + rng.normal(0.0, 0.02, layers)
    b = rng.normal(0.0, 0.005, layers)
    H = _from_spectrum(Q, eps, device)
    return Workload(name=f"cfg4_generalized_N{n}", H32=_sym32(H), N=n, N_occ=float(n // 2), eps=eps, Q=Q,
                    bounds=(-1.0, 1.0), tol=0.0, max_layers=layers,
                    extra={"seed": seed, "weights": w, "biases": b, "layers": layers})


def config5(seed: int = 0, batch: int = 1024, n: int = 256) -> Workload:
    """BASELINE.json configs[4]: `batch` independent gapped H of size n (gap 0.1 around 0: eps in
    U(-1,-0.05) / U(0.05,1), reading C20), N_occ = n/2, drawn sequentially from one generator."""
    rng = np.random.default_rng(seed)
    h = n // 2
    Hs = np.empty((batch, n, n), dtype=np.float32)
    Qs = np.empty((batch, n, n))
    es = np.empty((batch, n))
    for m in range(batch):
        w = gapped_dense(seed, n, (-1.0, -0.05), (0.05, 1.0), h, "", bounds=None, rng=rng)
        Hs[m], Qs[m], es[m] = w.H32, w.Q, w.eps
    return Workload(name=f"cfg5_batched_B{batch}_N{n}", H32=Hs, N=n, N_occ=float(h), eps=es, Q=Qs,
                    bounds=(-1.0, 1.0), tol=1e-5, max_layers=60, extra={"seed": seed, "batch": batch})


def uniform_symmetric(seed: int, n: int) -> np.ndarray:
    """Shape of the paper's Fig. 2 input: symmetric, H_ij uniform in [-1, 1]."""
    rng = np.random.default_rng(seed)
    A = rng.uniform(-1.0, 1.0, (n, n))
    return _sym32(np.triu(A) + np.triu(A, 1).T)


def decaying_chain(seed: int = 0, n: int = 2048, gap: float = 1.0, decay: float = 3.0, cutoff: int = 24) -> Workload:
    """A Hamiltonian WITH DECAY, the case the paper's sparse-matrix remark is about: a one-
    dimensional chain of n orbitals with alternating onsite energies -gap/2, +gap/2 and hoppings
    H_ij = -0.25 exp(-|i - j| / decay) N(1, 0.1) for 0 < |i - j| <= cutoff.  The staggered onsite term keeps a gap
    open at half filling, so the density matrix decays exponentially away from the diagonal and its far
    off-diagonal blocks are numerically zero.  N_occ = n / 2; no spectrum is known in closed form (the tests use
    LAPACK for the reference projector)."""
    rng = np.random.default_rng(seed)
    H = np.zeros((n, n))
    idx = np.arange(n)
    H[idx, idx] = np.where(idx % 2 == 0, -0.5 * gap, 0.5 * gap)
    for d in range(1, cutoff + 1):
        v = -0.25 * np.exp(-d / decay) * rng.normal(1.0, 0.1, n - d)
        H[idx[:-d], idx[:-d] + d] = v
        H[idx[:-d] + d, idx[:-d]] = v
    return Workload(name=f"decaying_chain_N{n}", H32=_sym32(H), N=n, N_occ=float(n // 2), bounds=None, tol=1e-5,
                    max_layers=120, extra={"seed": seed, "gap": gap, "decay": decay, "cutoff": cutoff})
