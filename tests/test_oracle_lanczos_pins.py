"""Pins for the oracle's Lanczos spectral bounds (optional replacement of Gershgorin in row A1; DESIGN.md reading
R3b; the paper only says "spectral bound estimates").  -m "not gpu"."""
import numpy as np
import pytest

import oracle
import rfoe_inputs
from tests import pins


def _hash_start(i):
    """The 32-bit start-vector hash, retyped from its definition with Python integers."""
    x = (i * 2654435761 + 0x9E3779B9) & 0xFFFFFFFF
    x ^= x >> 16
    x = (x * 0x85EBCA6B) & 0xFFFFFFFF
    x ^= x >> 13
    x = (x * 0xC2B2AE35) & 0xFFFFFFFF
    x ^= x >> 16
    return x / 4294967296.0 - 0.5


def test_full_run_reproduces_the_spectrum():
    """k steps on a k x k matrix: T_k is orthogonally similar to H, so its eigenvalues are H's (textbook property of
    the recursion; fails for a wrong sign or index anywhere in it).  alpha_0 = v0^T H v0 pins the start vector."""
    w = rfoe_inputs.from_spectrum(np.linspace(-1.0, 2.0, 10), 4, seed=3)
    lo, hi, a, b = oracle.bounds_lanczos(w.H, 10)
    assert len(a) == 10 and b[0] == 0.0
    T = np.diag(a) + np.diag(b[1:10], 1) + np.diag(b[1:10], -1)
    evT, _ = pins.jacobi_eigh(T)
    evH, _ = pins.jacobi_eigh(w.H)
    assert np.allclose(evT, evH, atol=1e-9)
    s = np.array([_hash_start(i) for i in range(10)])
    v0 = s / np.linalg.norm(s)
    assert a[0] == pytest.approx(v0 @ w.H @ v0, rel=1e-13)
    assert b[1] == pytest.approx(np.linalg.norm(w.H @ v0 - a[0] * v0), rel=1e-12)


@pytest.mark.parametrize("c,k,m", [(1, 256, 24), (2, 300, 16), (3, 333, 24), (4, 512, 32), (2, 64, 8)])
def test_bounds_enclose_the_spectrum_and_are_tight(c, k, m):
    w = rfoe_inputs.make_workload(c, k=k)
    lo, hi, a, b = oracle.bounds_lanczos(w.H, m)
    ev = np.linalg.eigvalsh(w.H)
    assert lo <= ev[0] and ev[-1] <= hi                           # the property the expansion needs
    glo, ghi = oracle.bounds(w.H)
    assert (hi - lo) < 0.5 * (ghi - glo)                          # and the point of having them
    assert (hi - lo) < 2.0 * (ev[-1] - ev[0])
    # theta_min / theta_max are the extreme eigenvalues of T_m (library routine on the returned alpha, beta)
    T = np.diag(a) + np.diag(b[1:-1], 1) + np.diag(b[1:-1], -1)
    th = np.linalg.eigvalsh(T)
    assert lo + b[-1] == pytest.approx(th[0], abs=1e-12) and hi - b[-1] == pytest.approx(th[-1], abs=1e-12)
    assert ev[0] <= th[0] and th[-1] <= ev[-1]                    # Ritz values lie inside the spectrum (Cauchy interlacing)


def test_invariant_subspace_breakdown_and_diagonal_matrix():
    # H = 2 I: every vector is an eigenvector, the recursion stops after one step with exact bounds
    lo, hi, a, b = oracle.bounds_lanczos(2.0 * np.eye(7), 5)
    assert len(a) == 1 and a[0] == pytest.approx(2.0) and b[1] == 0.0 and lo == pytest.approx(2.0) and hi == pytest.approx(2.0)
    # diagonal H with 3 distinct values: at most 3 steps
    d = np.diag([1.0, 1.0, -3.0, 5.0, 5.0, -3.0])
    lo, hi, a, b = oracle.bounds_lanczos(d, 6)
    assert len(a) == 3 and lo == pytest.approx(-3.0, abs=1e-12) and hi == pytest.approx(5.0, abs=1e-12)


def test_expansion_with_lanczos_bounds_needs_fewer_steps_and_reaches_the_same_projector():
    w = rfoe_inputs.make_workload(4, k=400)
    lo, hi, _, _ = oracle.bounds_lanczos(w.H, 24)
    r_g = oracle.expand(w.H, w.nocc, tol=w.tol)
    r_l = oracle.expand(w.H, w.nocc, tol=w.tol, bounds_override=(lo, hi))
    assert r_l.converged and r_l.iterations <= r_g.iterations - 6
    P = w.exact_projector()
    assert np.linalg.norm(r_l.P - P) / 20.0 <= 1e-12
