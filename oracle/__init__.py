"""CPU oracle for the RFOE hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper around ``oracle/rfoe_oracle.c`` (plain FP64 C, naive triple-loop products;
see that file's header for the passages of PAPER.md it follows and for its pins).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package; it imports nothing from ``paper_2301_04642_b200``.

Parity status: every function is pinned by tests/test_oracle_pins.py (estimate_homo_lumo: by
tests/test_oracle_homo_lumo_pins.py; project / apply / density: tests/test_oracle_subspace_pins.py; bounds_lanczos:
tests/test_oracle_lanczos_pins.py), including the FP32 product (bit for bit against a numpy.float32 loop), the
mixed schedule's phase switches, the sign rule outside [0,1] and T-RFOE against the exact Fermi-Dirac matrix.
"Parity unpinned": only the exact bit patterns of the iterates X_n (the paper prints no worked example).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rfoe_oracle.c")
_LIB = os.path.join(_HERE, "librfoe_oracle.so")

SP2, MCWEENY, SP2_MIXED, SP2_ACCEL, TRUNC, TRUNC_MIXED = 0, 1, 2, 3, 4, 5
RULE_A, RULE_B = 0, 1
MAX_STEPS = 256


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (portable flags; no FMA contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
               "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class _Run(C.Structure):
    _fields_ = [
        ("variant", C.c_int32), ("stop_rule", C.c_int32), ("max_iter", C.c_int32), ("use_bounds", C.c_int32),
        ("tol", C.c_double), ("emin", C.c_double), ("emax", C.c_double),
        ("mixed_head", C.c_double), ("mixed_reltr", C.c_double), ("homo", C.c_double), ("lumo", C.c_double),
        ("iterations", C.c_int32), ("multiplications", C.c_int32), ("mcweeny_steps", C.c_int32),
        ("fp32_steps", C.c_int32), ("converged", C.c_int32), ("pad_", C.c_int32),
        ("tr_PH", C.c_double),
        ("t", C.c_double * (MAX_STEPS + 1)), ("s", C.c_double * (MAX_STEPS + 1)),
        ("e", C.c_double * MAX_STEPS), ("reltr", C.c_double * MAX_STEPS),
        ("branch", C.c_char * (MAX_STEPS + 1)),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.rfoe_oracle_bounds.argtypes = [dp, C.c_int64, dp, dp]
        L.rfoe_oracle_bounds.restype = None
        L.rfoe_oracle_affine.argtypes = [dp, C.c_int64, C.c_double, C.c_double, dp]
        L.rfoe_oracle_affine.restype = None
        L.rfoe_oracle_trace.argtypes = [dp, C.c_int64]
        L.rfoe_oracle_trace.restype = C.c_double
        L.rfoe_oracle_sumsq.argtypes = [dp, C.c_int64]
        L.rfoe_oracle_sumsq.restype = C.c_double
        for name in ("rfoe_oracle_square", "rfoe_oracle_square_ijk"):
            f = getattr(L, name)
            f.argtypes = [dp, C.c_int64, dp]
            f.restype = None
        for name in ("rfoe_oracle_matmul", "rfoe_oracle_matmul_ijk"):
            f = getattr(L, name)
            f.argtypes = [dp, dp, C.c_int64, dp]
            f.restype = None
        for name in ("rfoe_oracle_project", "rfoe_oracle_project_full", "rfoe_oracle_apply", "rfoe_oracle_density"):
            f = getattr(L, name)
            f.argtypes = [dp, dp, C.c_int64, C.c_int64, C.c_int64, dp]
            f.restype = None
        L.rfoe_oracle_bounds_lanczos.argtypes = [dp, C.c_int64, C.c_int32, dp, dp, dp, dp]
        L.rfoe_oracle_bounds_lanczos.restype = C.c_int
        L.rfoe_oracle_square_f32.argtypes = [dp, C.c_int64, dp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.rfoe_oracle_square_f32.restype = None
        L.rfoe_oracle_is_symmetric.argtypes = [dp, C.c_int64]
        L.rfoe_oracle_is_symmetric.restype = C.c_int
        L.rfoe_oracle_expand.argtypes = [dp, C.c_int64, C.c_int64, C.POINTER(_Run), dp]
        L.rfoe_oracle_expand.restype = C.c_int
        assert L.rfoe_oracle_sizeof_run() == C.sizeof(_Run), "oracle_run_t layout mismatch"
        assert L.rfoe_oracle_max_steps() == MAX_STEPS
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _sq(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.ndim != 2 or a.shape[0] != a.shape[1]:
        raise ValueError("square FP64 matrix expected")
    return a


def bounds(H):
    """Gershgorin bounds (O1)."""
    H = _sq(H)
    lo, hi = C.c_double(), C.c_double()
    lib().rfoe_oracle_bounds(_p(H), H.shape[0], C.byref(lo), C.byref(hi))
    return lo.value, hi.value


def affine(H, emin: float, emax: float) -> np.ndarray:
    """X0 = (emax I - H)/(emax - emin) (O2)."""
    H = _sq(H)
    X = np.empty_like(H)
    lib().rfoe_oracle_affine(_p(H), H.shape[0], emin, emax, _p(X))
    return X


def trace(X) -> float:
    X = _sq(X)
    return lib().rfoe_oracle_trace(_p(X), X.shape[0])


def sumsq(X) -> float:
    X = _sq(X)
    return lib().rfoe_oracle_sumsq(_p(X), X.shape[0])


def square(X, literal: bool = False) -> np.ndarray:
    """Naive X*X, contraction index ascending.  ``literal`` = the i-j-l loop nest."""
    X = _sq(X)
    Y = np.empty_like(X)
    (lib().rfoe_oracle_square_ijk if literal else lib().rfoe_oracle_square)(_p(X), X.shape[0], _p(Y))
    return Y


def matmul(A, B, literal: bool = False) -> np.ndarray:
    A, B = _sq(A), _sq(B)
    Y = np.empty_like(A)
    (lib().rfoe_oracle_matmul_ijk if literal else lib().rfoe_oracle_matmul)(_p(A), _p(B), A.shape[0], _p(Y))
    return Y


def square_f32(X) -> np.ndarray:
    """The FP32 step's product: X rounded to binary32, binary32 products and sums, l ascending."""
    X = _sq(X)
    k = X.shape[0]
    Y = np.empty_like(X)
    xf = np.empty(k * k, dtype=np.float32)
    yf = np.empty(k * k, dtype=np.float32)
    fp = C.POINTER(C.c_float)
    lib().rfoe_oracle_square_f32(_p(X), k, _p(Y), xf.ctypes.data_as(fp), yf.ctypes.data_as(fp))
    return Y


def is_symmetric(X) -> bool:
    X = _sq(X)
    return bool(lib().rfoe_oracle_is_symmetric(_p(X), X.shape[0]))


@dataclass
class OracleResult:
    P: np.ndarray
    iterations: int
    multiplications: int
    mcweeny_steps: int
    fp32_steps: int
    converged: bool
    branch: str
    emin: float
    emax: float
    tr_PH: float
    t: np.ndarray      # t[0..iterations]
    s: np.ndarray      # s[0..iterations]
    e: np.ndarray      # e[0..iterations-1]
    reltr: np.ndarray  # reltr[0..iterations-1]


def expand(H, nocc: int, *, variant: int = SP2, tol: float = 1e-12, stop_rule: int = RULE_A, max_iter: int = 100,
           bounds_override=None, mixed_head: float = 0.0, mixed_reltr: float = 5e-4,
           homo: float = 0.0, lumo: float = 0.0) -> OracleResult:
    """The whole expansion (O1-O5): Gershgorin -> affine map -> trace-steered recursion -> P.
    variant TRUNC / TRUNC_MIXED (T-RFOE): exactly ``max_iter`` = m steps, no convergence test;
    ``converged`` then means "G_m delivered"."""
    H = _sq(H)
    k = H.shape[0]
    run = _Run()
    run.variant, run.stop_rule, run.max_iter = variant, stop_rule, max_iter
    run.tol = tol
    if bounds_override is not None:
        run.use_bounds, run.emin, run.emax = 1, float(bounds_override[0]), float(bounds_override[1])
    run.mixed_head, run.mixed_reltr, run.homo, run.lumo = mixed_head, mixed_reltr, homo, lumo
    P = np.empty_like(H)
    rc = lib().rfoe_oracle_expand(_p(H), k, nocc, C.byref(run), _p(P))
    if rc != 0:
        raise RuntimeError(f"rfoe_oracle_expand failed with code {rc}")
    n = run.iterations
    return OracleResult(
        P=P, iterations=n, multiplications=run.multiplications, mcweeny_steps=run.mcweeny_steps,
        fp32_steps=run.fp32_steps, converged=bool(run.converged), branch=run.branch.decode()[:n],
        emin=run.emin, emax=run.emax, tr_PH=run.tr_PH,
        t=np.array(run.t[: n + 1]), s=np.array(run.s[: n + 1]), e=np.array(run.e[:n]), reltr=np.array(run.reltr[:n]))


def estimate_homo_lumo(res: OracleResult, nocc: int, e_floor: float = 1e-6):
    """HOMO / LUMO estimates for A-Z-RFOE (polynomials chosen "based on HOMO ... and LUMO ... eigenvalues";
    the paper is silent on their source, reading R-HL: the history of the previous Z-RFOE run, refs. 31, 38).

    Step by step: for every step n whose occupation is settled (t_n - s_n < 3/16 and |t_n - nocc| < 1/2, reading R11) and
    whose e_n = ||X_n^2 - X_n||_F lies in [e_floor, 1/4): every eigenvalue x of X_n has x(1 - x) <= e_n, so the LUMO image
    is <= a = (1 - sqrt(1 - 4 e_n))/2 and the HOMO image is >= 1 - a.  Undo steps n-1 .. 0 ('S' x^2 -> sqrt(x);
    'L' 2x - x^2 -> 1 - sqrt(1 - x); both monotone), undo X_0 = (emax - lambda)/(emax - emin), keep the tightest pair.
    Returns (homo_est, lumo_est) with homo_est >= lambda_HOMO and lumo_est <= lambda_LUMO."""
    import math

    if any(ch not in "SL" for ch in res.branch):
        raise ValueError("history of a plain FP64 SP2 run expected")
    w = res.emax - res.emin
    homo, lumo = math.inf, -math.inf
    for n in range(res.iterations):
        t, s, e = float(res.t[n]), float(res.s[n]), float(res.e[n])
        if not (t - s < 3.0 / 16.0 and abs(t - nocc) < 0.5 and e_floor <= e < 0.25):
            continue
        a = 0.5 * (1.0 - math.sqrt(1.0 - 4.0 * e))
        x_lumo, x_homo = a, 1.0 - a
        for j in range(n - 1, -1, -1):
            if res.branch[j] == "S":
                x_lumo, x_homo = math.sqrt(x_lumo), math.sqrt(x_homo)
            else:
                x_lumo, x_homo = 1.0 - math.sqrt(1.0 - x_lumo), 1.0 - math.sqrt(1.0 - x_homo)
        lumo = max(lumo, res.emax - w * x_lumo)
        homo = min(homo, res.emax - w * x_homo)
    if not (math.isfinite(homo) and math.isfinite(lumo)):
        raise RuntimeError("no admissible step in the history")
    return homo, lumo


def square_entries(X, pairs):
    """(X X)_ij for a list of (i, j), each by the definition Y_ij = sum_l X_il X_lj with l ascending, one
    IEEE product and one IEEE sum at a time (pure-Python loop over Python floats).  Used where the full
    naive product is out of reach (k >= 8192): sampled outputs computed one by one."""
    X = np.asarray(X)
    out = []
    for i, j in pairs:
        row = X[i, :].tolist()
        col = X[:, j].tolist()
        acc = 0.0
        for a, b in zip(row, col):
            acc = acc + a * b
        out.append(acc)
    return np.array(out)


def _rect(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.ndim != 2:
        raise ValueError("k x M FP64 matrix expected")
    return a


def project(Psi, HPsi, full: bool = False) -> np.ndarray:
    """Rayleigh-Ritz step: H^p = Psi H Psi^T from Psi (k x M, one state per row) and HPsi
    (row j = H applied to state j).  Upper triangle by the definition, mirrored; ``full`` = all k^2 sums."""
    Psi, HPsi = _rect(Psi), _rect(HPsi)
    k, M = Psi.shape
    assert HPsi.shape == (k, M)
    Hp = np.empty((k, k))
    (lib().rfoe_oracle_project_full if full else lib().rfoe_oracle_project)(_p(Psi), _p(HPsi), k, M, M, _p(Hp))
    return Hp


def apply(P, Psi) -> np.ndarray:
    """Y = P Psi (the subspace density matrix applied to the basis), j ascending."""
    P, Psi = _sq(P), _rect(Psi)
    k, M = Psi.shape
    assert P.shape == (k, k)
    Y = np.empty((k, M))
    lib().rfoe_oracle_apply(_p(P), _p(Psi), k, M, M, _p(Y))
    return Y


def density(Psi, Y) -> np.ndarray:
    """rho_m = sum_i Psi_im Y_im = diag(Psi^T P Psi), i ascending."""
    Psi, Y = _rect(Psi), _rect(Y)
    k, M = Psi.shape
    assert Y.shape == (k, M)
    rho = np.empty(M)
    lib().rfoe_oracle_density(_p(Psi), _p(Y), k, M, M, _p(rho))
    return rho


def bounds_lanczos(H, m: int = 24):
    """m-step Lanczos spectral bounds (theta_min - beta_m, theta_max + beta_m); returns (emin, emax, alpha, beta)."""
    H = _sq(H)
    lo, hi = C.c_double(), C.c_double()
    a = np.zeros(64)
    b = np.zeros(65)
    steps = lib().rfoe_oracle_bounds_lanczos(_p(H), H.shape[0], int(m), C.byref(lo), C.byref(hi), _p(a), _p(b))
    return lo.value, hi.value, a[:steps].copy(), b[: steps + 1].copy()
