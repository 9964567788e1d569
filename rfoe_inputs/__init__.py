"""Seeded synthetic inputs for the RFOE hot path (shared by tests, oracle runs and bench).

This module holds NONE of the method's arithmetic: it only builds projected Hamiltonians
``H^p = Q diag(lambda) Q^T`` with a controlled spectrum (BASELINE.json configs 1-5; SURVEY.md
section 8(d) "Synthetic inputs", reading R16) and the paper's own formula matrix
(section IV; reading R12).  Neither ``oracle/`` nor the CUDA package is imported here.

Recipe (stated again in DESIGN.md):
  * lambda: i.i.d. uniform draws from ``numpy.random.default_rng(1000 + c)``, occupied group first,
    then the unoccupied group; the first/last element of each group is overwritten with the
    group's stated ends so the gap and the spread are exact.  Config 4 additionally writes a
    cluster of 0.25 % of k values within 1e-3 of each gap edge (indices 1..n of each group).
  * Q: Householder QR (LAPACK / cuSOLVER geqrf) of a seeded N(0,1) k x k matrix
    (``default_rng(2000 + c)`` on the CPU, ``torch.Generator(2000 + c)`` on the GPU for
    k >= 8192), columns sign-fixed so that diag(R) > 0.
  * H = (Q diag(lambda)) Q^T, then H <- (H + H^T)/2 so that H is bitwise symmetric.
The same bytes are handed to the oracle and to the library; ``sha256`` identifies them.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np

__all__ = ["CONFIGS", "Workload", "spectrum", "make_workload", "from_spectrum", "paper_matrix", "sha256",
           "Subspace", "make_subspace", "invariant_subspace"]


@dataclass(frozen=True)
class _Cfg:
    k: int
    nocc: int
    occ: tuple          # (lo, hi) of the occupied eigenvalues
    unocc: tuple        # (lo, hi) of the unoccupied eigenvalues
    tol: float          # stop rule A tolerance, reading R9: 1e-12 * k / 256
    cluster: int = 0    # values clustered within 1e-3 of each gap edge (config 4)


# BASELINE.json "configs" 1..5 (1-based).
CONFIGS = {
    1: _Cfg(256, 64, (-1.0, -0.2), (0.0, 2.0), 1e-12),
    2: _Cfg(2048, 1536, (-0.6, -0.05), (0.05, 1.5), 8e-12),
    3: _Cfg(8192, 6300, (-1.0, -0.01), (0.01, 3.0), 3.2e-11),
    4: _Cfg(16384, 12600, (-2.0, -0.025), (0.025, 4.0), 6.4e-11, cluster=41),
    5: _Cfg(40000, 30000, (-1.0, -0.025), (0.025, 3.0), 1.6e-10),
}


@dataclass
class Workload:
    """One seeded problem instance.  ``H``/``Q`` are numpy arrays (CPU build) or torch CUDA
    tensors (GPU build); ``lam`` is always numpy; ``lam[:nocc]`` are the occupied eigenvalues and
    column ``i`` of ``Q`` is the eigenvector of ``lam[i]``."""
    name: str
    k: int
    nocc: int
    tol: float
    lam: np.ndarray
    H: object
    Q: object = None
    meta: dict = field(default_factory=dict)

    def exact_projector(self):
        """Construction-exact P = Q_occ Q_occ^T (pin P2 of SURVEY.md section 8(c)): a closed form of the
        generator's own Q, not produced by any RFOE code."""
        Qo = self.Q[:, : self.nocc]
        return Qo @ Qo.T

    def band_energy(self) -> float:
        """sum of the occupied eigenvalues = tr(P H) for the exact projector."""
        return float(np.sum(self.lam[: self.nocc]))


def spectrum(c: int, k: int | None = None, nocc: int | None = None) -> np.ndarray:
    """Eigenvalues of config ``c`` (reading R16).  ``k``/``nocc`` may be overridden to build a
    scaled-down instance with the same value distribution (used by parity tests at odd sizes)."""
    cfg = CONFIGS[c]
    k = cfg.k if k is None else k
    nocc = cfg.nocc if nocc is None else nocc
    if not (0 < nocc < k):
        raise ValueError("need 0 < nocc < k")
    rng = np.random.default_rng(1000 + c)
    occ = rng.uniform(cfg.occ[0], cfg.occ[1], size=nocc)
    uno = rng.uniform(cfg.unocc[0], cfg.unocc[1], size=k - nocc)
    ncl = cfg.cluster if (cfg.cluster and k == cfg.k) else (max(1, k // 400) if cfg.cluster else 0)
    if ncl:
        ncl = min(ncl, nocc - 2, k - nocc - 2)
        if ncl > 0:
            occ[1 : 1 + ncl] = cfg.occ[1] - 1e-3 * rng.uniform(0.0, 1.0, size=ncl)
            uno[1 : 1 + ncl] = cfg.unocc[0] + 1e-3 * rng.uniform(0.0, 1.0, size=ncl)
    occ[0], occ[-1] = cfg.occ[0], cfg.occ[1]
    uno[0], uno[-1] = cfg.unocc[0], cfg.unocc[1]
    return np.concatenate([occ, uno])


def _haar_q_numpy(k: int, seed: int) -> np.ndarray:
    A = np.random.default_rng(seed).standard_normal((k, k))
    Q, R = np.linalg.qr(A)
    sgn = np.sign(np.diag(R))
    sgn[sgn == 0] = 1.0
    return Q * sgn[None, :]


def _haar_q_torch(k: int, seed: int, device):
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    A = torch.randn((k, k), dtype=torch.float64, device=device, generator=g)
    Q, R = torch.linalg.qr(A)
    del A
    sgn = torch.sign(torch.diagonal(R))
    sgn[sgn == 0] = 1.0
    del R
    Q.mul_(sgn[None, :])
    return Q


def from_spectrum(lam: np.ndarray, nocc: int, seed: int, *, name: str = "custom", tol: float | None = None,
                  device: str = "cpu", keep_q: bool = True) -> Workload:
    """H = Q diag(lam) Q^T with a seeded Haar-like Q, then symmetrised bitwise."""
    lam = np.asarray(lam, dtype=np.float64)
    k = lam.shape[0]
    tol = 1e-12 * max(k, 256) / 256 if tol is None else tol
    if device == "cpu":
        Q = _haar_q_numpy(k, seed)
        H = (Q * lam[None, :]) @ Q.T
        H = 0.5 * (H + H.T)
        H = np.ascontiguousarray(H)
    else:
        import torch

        Q = _haar_q_torch(k, seed, device)
        lam_d = torch.from_numpy(lam).to(device)
        H = (Q * lam_d[None, :]) @ Q.T
        H = H.add_(H.T.clone()).mul_(0.5).contiguous()
    return Workload(name=name, k=k, nocc=nocc, tol=tol, lam=lam, H=H, Q=Q if keep_q else None,
                    meta={"seed": seed, "device": device})


def make_workload(c: int, *, k: int | None = None, nocc: int | None = None, device: str | None = None,
                  keep_q: bool = True) -> Workload:
    """BASELINE.json config ``c`` (1..5).  k <= 2048 is always built with numpy on the CPU so that
    CPU-only and GPU test runs see identical bytes; larger k defaults to torch on ``cuda``."""
    cfg = CONFIGS[c]
    kk = cfg.k if k is None else k
    no = cfg.nocc if nocc is None else nocc
    if k is not None and nocc is None:
        no = max(1, min(kk - 1, round(cfg.nocc / cfg.k * kk)))
    lam = spectrum(c, kk, no)
    if device is None:
        device = "cpu" if kk <= 2048 else "cuda"
    tol = cfg.tol if kk == cfg.k else 1e-12 * max(kk, 256) / 256
    w = from_spectrum(lam, no, 2000 + c, name=f"config{c}" + ("" if kk == cfg.k else f"@k={kk}"), tol=tol,
                      device=device, keep_q=keep_q)
    w.meta["config"] = c
    return w


def paper_matrix(k: int) -> np.ndarray:
    """The paper's own synthetic H^p (section IV), reading R12 of SURVEY.md section 8(c):
    H_ij = exp(-0.5 |i-j|) sin(min(i,j)+1), 0-based indices; symmetric by construction."""
    i = np.arange(k)
    d = np.abs(i[:, None] - i[None, :]).astype(np.float64)
    m = np.minimum(i[:, None], i[None, :]).astype(np.float64)
    return np.ascontiguousarray(np.exp(-0.5 * d) * np.sin(m + 1.0))


def sha256(H) -> str:
    """SHA-256 of the raw FP64 bytes of H (numpy array or torch tensor)."""
    if not isinstance(H, np.ndarray):
        H = H.detach().cpu().numpy()
    return hashlib.sha256(np.ascontiguousarray(H).tobytes()).hexdigest()


# ---- inputs of the steps either side of the expansion (Rayleigh-Ritz before, P applied to the basis after) ----
@dataclass
class Subspace:
    """A subspace basis and the action of H on it, one state per row (k x M, row-major, pitch M).
    ``Psi`` has orthonormal rows; ``HPsi`` row j is H applied to state j; ``Psi @ HPsi.T`` equals the
    projected Hamiltonian ``w.H`` of the underlying workload up to rounding.  numpy arrays or CUDA tensors."""
    k: int
    M: int
    Psi: object
    HPsi: object
    w: Workload
    H_full: object = None      # the M x M matrix, only for the tiny explicit construction


def make_subspace(c: int, k: int, M: int, *, resid: float = 0.1, device: str = "cpu") -> Subspace:
    """Synthetic Rayleigh-Ritz input with the structure of the paper's setting (a basis of
    k states over M >> k degrees of freedom, H never formed densely).  Recipe: ``w`` = config ``c`` scaled to
    k (spectrum, gap and nocc/k kept); Psi^T = thin QR of a seeded N(0,1) M x k matrix (seed 3000+c);
    HPsi = w.H Psi + R with R a seeded N(0,1) k x M matrix (seed 4000+c) projected off span(Psi) twice and
    scaled to ``resid`` x rms(w.H Psi) -- the part of H Psi that leaves the subspace, which the projection
    must annihilate."""
    w = make_workload(c, k=k, device="cpu" if device == "cpu" else device)
    if device == "cpu":
        A = np.random.default_rng(3000 + c).standard_normal((M, k))
        Q, _ = np.linalg.qr(A)
        Psi = np.ascontiguousarray(Q.T)
        G = np.random.default_rng(4000 + c).standard_normal((k, M))
        for _ in range(2):
            G -= (G @ Psi.T) @ Psi
        HP = np.asarray(w.H) @ Psi
        G *= resid * np.sqrt(np.mean(HP * HP) / np.mean(G * G))
        HPsi = np.ascontiguousarray(HP + G)
    else:
        import torch

        g = torch.Generator(device=device)
        g.manual_seed(3000 + c)
        A = torch.randn((M, k), dtype=torch.float64, device=device, generator=g)
        Q, _ = torch.linalg.qr(A)
        del A
        Psi = Q.T.contiguous()
        del Q
        g.manual_seed(4000 + c)
        G = torch.randn((k, M), dtype=torch.float64, device=device, generator=g)
        for _ in range(2):
            G -= (G @ Psi.T) @ Psi
        H = w.H if isinstance(w.H, torch.Tensor) else torch.from_numpy(w.H).to(device)
        HP = H @ Psi
        G *= resid * float(torch.sqrt(torch.mean(HP * HP) / torch.mean(G * G)))
        HPsi = HP.add_(G).contiguous()
        del G
    return Subspace(k=k, M=M, Psi=Psi, HPsi=HPsi, w=w)


def invariant_subspace(M: int, k: int, nocc: int, seed: int, *, gap: float = 0.3) -> Subspace:
    """Tiny explicit instance: a full symmetric M x M matrix H_full = V diag(mu) V^T (mu ascending, a gap of
    ``gap`` after the nocc-th value) and a basis Psi whose rows span the invariant subspace of its k lowest
    eigenvectors, mixed by a seeded k x k rotation.  Everything downstream then has a plain definition through
    an explicit eigendecomposition of H_full: H^p has the k lowest eigenvalues, and the density is
    rho_m = sum_{i < nocc} V_mi^2."""
    rng = np.random.default_rng(seed)
    V = _haar_q_numpy(M, seed + 1)
    lo = np.sort(rng.uniform(-1.0, -gap / 2, size=nocc))
    hi = np.sort(rng.uniform(gap / 2, 2.0, size=M - nocc))
    mu = np.concatenate([lo, hi])
    H_full = (V * mu[None, :]) @ V.T
    H_full = 0.5 * (H_full + H_full.T)
    R = _haar_q_numpy(k, seed + 2)
    Psi = np.ascontiguousarray(R @ V[:, :k].T)
    HPsi = np.ascontiguousarray(Psi @ H_full)
    w = Workload(name=f"invariant(M={M},k={k})", k=k, nocc=nocc, tol=1e-12, lam=mu[:k].copy(), H=None, Q=None,
                 meta={"seed": seed, "V": V, "mu": mu})
    return Subspace(k=k, M=M, Psi=Psi, HPsi=HPsi, w=w, H_full=H_full)
