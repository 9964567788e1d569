"""Independent pins for the oracle (and, through it, for the CUDA path).

Nothing here calls ``oracle/`` or the CUDA library: these are the textbook objects the method must
reach -- a cyclic Jacobi eigendecomposition (north_star: "checked on tiny inputs against a Jacobi
eigendecomposition projector"), and the scalar eigenvalue-space model of the recursion (pin P5 of
SURVEY.md section 8(c)): because X_n = Q diag(x_n) Q^T in exact arithmetic, the recursion on the
eigenvalues alone predicts branch string, iteration count, t_n, s_n and e_n of the matrix run.
"""
from __future__ import annotations

import math

import numpy as np


def jacobi_eigh(A, sweeps: int = 60, tol: float = 1e-30):
    """Cyclic Jacobi eigendecomposition of a small symmetric matrix (pure Python loops).
    Returns (eigenvalues ascending, eigenvectors as columns)."""
    A = np.array(A, dtype=np.float64)
    n = A.shape[0]
    V = np.eye(n)
    for _ in range(sweeps):
        off = float(np.sum(np.triu(A, 1) ** 2))
        if off <= tol:
            break
        for p in range(n - 1):
            for q in range(p + 1, n):
                apq = A[p, q]
                if apq == 0.0:
                    continue
                theta = (A[q, q] - A[p, p]) / (2.0 * apq)
                t = math.copysign(1.0, theta) / (abs(theta) + math.sqrt(theta * theta + 1.0))
                c = 1.0 / math.sqrt(t * t + 1.0)
                s = t * c
                # A <- J^T A J with J the rotation in the (p, q) plane
                Ap, Aq = A[:, p].copy(), A[:, q].copy()
                A[:, p], A[:, q] = c * Ap - s * Aq, s * Ap + c * Aq
                Ap, Aq = A[p, :].copy(), A[q, :].copy()
                A[p, :], A[q, :] = c * Ap - s * Aq, s * Ap + c * Aq
                Vp, Vq = V[:, p].copy(), V[:, q].copy()
                V[:, p], V[:, q] = c * Vp - s * Vq, s * Vp + c * Vq
    w = np.diag(A).copy()
    order = np.argsort(w)
    return w[order], V[:, order]


def jacobi_projector(H, nocc: int):
    """P_ref = V_occ V_occ^T from the Jacobi eigenvectors of the nocc lowest eigenvalues."""
    w, V = jacobi_eigh(H)
    Vo = V[:, :nocc]
    return Vo @ Vo.T, w


def scalar_sp2(lam, nocc: int, emin: float, emax: float, *, tol: float, rule: str = "A", max_iter: int = 100):
    """Eigenvalue-space SP2 (pin P5): x_i <- (emax - lam_i)/(emax - emin), then x <- x^2 if
    the resulting trace is nearer nocc than that of 2x - x^2 (else the latter).  Returns dict(branch, iterations, t, s, e)."""
    x = (emax - np.asarray(lam, dtype=np.float64)) / (emax - emin)
    t_hist, s_hist, e_hist, branch = [float(np.sum(x))], [float(np.sum(x * x))], [], ""
    it = 0
    for _ in range(max_iter):
        t = float(np.sum(x))
        x2 = x * x
        e = float(np.sqrt(np.sum((x2 - x) ** 2)))
        # the sign that brings the trace of X_{n+1} nearer N_occ (tie -> L)
        if abs(float(np.sum(x2)) - nocc) < abs(float(np.sum(2.0 * x - x2)) - nocc):
            x = x2
            branch += "S"
        else:
            x = 2.0 * x - x2
            branch += "L"
        it += 1
        t1 = float(np.sum(x))
        e_hist.append(e)
        t_hist.append(t1)
        s_hist.append(float(np.sum(x * x)))
        reltr = abs(t1 - t) / abs(t)
        if (rule == "A" and e <= tol) or (rule == "B" and reltr <= tol):
            break
    return dict(branch=branch, iterations=it, t=np.array(t_hist), s=np.array(s_hist), e=np.array(e_hist), x=x)


def scalar_sp2_accel(lam, nocc: int, emin: float, emax: float, homo: float, lumo: float, *, tol: float,
                     rule: str = "B", max_iter: int = 100):
    """Eigenvalue-space accelerated SP2 in its *unexpanded* form (shift-and-scale, then the SP2
    polynomial): S: x <- ((1-a) + a x)^2, a = 2/(2-beta); L: y = a x, x <- 2y - y^2, a = 2/(1+bbar)."""
    w = emax - emin
    x = (emax - np.asarray(lam, dtype=np.float64)) / w
    beta, bbar = (emax - lumo) / w, (emax - homo) / w
    branch, it = "", 0
    for _ in range(max_iter):
        t = float(np.sum(x))
        e = float(np.sqrt(np.sum((x * x - x) ** 2)))
        aS, aL = 2.0 / (2.0 - beta), 2.0 / (1.0 + bbar)
        fS = lambda v, a=aS: ((1.0 - a) + a * v) ** 2
        fL = lambda v, a=aL: 2.0 * (a * v) - (a * v) ** 2
        if abs(float(np.sum(fS(x))) - nocc) < abs(float(np.sum(fL(x))) - nocc):
            f = fS
            branch += "S"
        else:
            f = fL
            branch += "L"
        x, beta, bbar = f(x), f(beta), f(bbar)
        it += 1
        t1 = float(np.sum(x))
        if (rule == "A" and e <= tol) or (rule == "B" and abs(t1 - t) / abs(t) <= tol):
            break
    return dict(branch=branch, iterations=it, x=x)


def fermi_dirac(lam, mu: float, beta: float):
    """Occupancies of the finite-temperature density matrix D = [exp(beta (H - mu I)) + I]^-1,
    in the overflow-free form (1 - tanh(z/2)) / 2."""
    return 0.5 * (1.0 - np.tanh(0.5 * beta * (np.asarray(lam, dtype=np.float64) - mu)))


def fit_fermi_dirac(lam, occ, mu0: float):
    """Least-squares (mu, beta) of the Fermi-Dirac function to occupancies ``occ`` at eigenvalues ``lam``
    (scipy.optimize.least_squares on (mu, log beta) from several starting betas).  Returns (mu, beta)."""
    from scipy.optimize import least_squares

    lam = np.asarray(lam, dtype=np.float64)
    best = None
    for b0 in (10.0, 1e2, 1e3, 1e4, 1e5):
        r = least_squares(lambda p: fermi_dirac(lam, p[0], math.exp(p[1])) - occ, [mu0, math.log(b0)],
                          xtol=1e-15, ftol=1e-15, gtol=1e-15)
        if best is None or r.cost < best.cost:
            best = r
    return float(best.x[0]), float(math.exp(best.x[1]))
