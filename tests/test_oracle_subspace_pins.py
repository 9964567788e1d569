"""Pins for the oracle's Rayleigh-Ritz / apply / density functions (-m "not gpu").
The paper prints neither step (PAPER.md:17, 62 state the setting), so each pin is a plain definition reached
another way: literal Python loops, an explicit eigendecomposition of the full M x M matrix (tests/pins.py
Jacobi and numpy), closed forms, and the electron-count invariant sum_m rho_m = N_occ."""
import numpy as np
import pytest

import oracle
import rfoe_inputs
from tests import pins


def test_project_literal_loops_and_transposed_operand_mistake():
    rng = np.random.default_rng(5)
    k, M = 4, 7
    Psi, Phi = rng.standard_normal((k, M)), rng.standard_normal((k, M))
    full = oracle.project(Psi, Phi, full=True)
    for i in range(k):
        for j in range(k):
            acc = 0.0
            for m in range(M):
                acc = acc + Psi[i, m] * Phi[j, m]
            assert full[i, j] == acc           # same order of the same IEEE operations: bit-exact
    up = oracle.project(Psi, Phi)
    assert np.array_equal(np.triu(up), np.triu(full)) and np.array_equal(up, up.T)
    # for a non-symmetric pair the two triangles differ, so a transposed operand (Phi Psi^T) is caught
    assert not np.allclose(full, full.T)
    # small integers: every partial sum is exact, so any summation order gives these numbers
    A = np.arange(12.0).reshape(3, 4)
    B = (np.arange(12.0).reshape(3, 4) % 5) - 2
    assert np.array_equal(oracle.project(A, B, full=True), A @ B.T)


def test_project_of_invariant_subspace_has_the_lowest_eigenvalues():
    sub = rfoe_inputs.invariant_subspace(M=40, k=12, nocc=5, seed=21)
    Hp = oracle.project(sub.Psi, sub.HPsi)
    assert oracle.is_symmetric(Hp)
    full = oracle.project(sub.Psi, sub.HPsi, full=True)
    assert np.abs(full - full.T).max() < 1e-14          # exact H^p is symmetric: the mirror only fixes rounding
    ev, _ = pins.jacobi_eigh(Hp)
    mu_full, _ = pins.jacobi_eigh(sub.H_full)           # explicit diagonalisation of the big matrix
    assert np.allclose(ev, mu_full[:12], atol=1e-12)
    assert np.allclose(ev, sub.w.meta["mu"][:12], atol=1e-12)


def test_apply_and_density_closed_forms():
    rng = np.random.default_rng(8)
    k, M = 5, 9
    Psi = rng.standard_normal((k, M))
    assert np.array_equal(oracle.apply(np.eye(k), Psi), Psi)          # P = I
    E = np.zeros((k, k)); E[1, 3] = 2.0                                # a single entry picks one row: catches P^T
    Y = oracle.apply(E, Psi)
    assert np.array_equal(Y[1], 2.0 * Psi[3]) and not Y[[0, 2, 3, 4]].any()
    P = rng.standard_normal((k, k))
    Y = oracle.apply(P, Psi)
    for i in range(k):
        for m in range(M):
            acc = 0.0
            for j in range(k):
                acc = acc + P[i, j] * Psi[j, m]
            assert Y[i, m] == acc
    rho = oracle.density(Psi, Y)
    for m in range(M):
        acc = 0.0
        for i in range(k):
            acc = acc + Psi[i, m] * Y[i, m]
        assert rho[m] == acc
    assert np.allclose(rho, np.diag(Psi.T @ P @ Psi), atol=1e-13)


@pytest.mark.parametrize("M,k,nocc,seed", [(30, 8, 3, 1), (48, 16, 9, 2), (36, 36, 10, 3)])
def test_pipeline_density_equals_explicit_diagonalisation(M, k, nocc, seed):
    """project -> expand -> apply -> density reproduces the density of the nocc lowest eigenvectors of the
    FULL matrix, obtained by explicit diagonalisation (the route the paper's method replaces)."""
    sub = rfoe_inputs.invariant_subspace(M=M, k=k, nocc=nocc, seed=seed)
    Hp = oracle.project(sub.Psi, sub.HPsi)
    res = oracle.expand(Hp, nocc, tol=1e-13)
    assert res.converged
    Y = oracle.apply(res.P, sub.Psi)
    rho = oracle.density(sub.Psi, Y)
    mu, V = pins.jacobi_eigh(sub.H_full)
    rho_ref = (V[:, :nocc] ** 2).sum(axis=1)
    assert np.abs(rho - rho_ref).max() < 1e-11
    assert abs(rho.sum() - nocc) < 1e-11                         # electron count
    D_full = sub.Psi.T @ Y                                        # density matrix in the M-dimensional space
    assert np.abs(D_full - V[:, :nocc] @ V[:, :nocc].T).max() < 1e-11
    assert abs(res.tr_PH - mu[:nocc].sum()) < 1e-11               # band energy


def test_make_subspace_recipe():
    sub = rfoe_inputs.make_subspace(2, k=24, M=200)
    Psi, HPsi = sub.Psi, sub.HPsi
    assert np.abs(Psi @ Psi.T - np.eye(24)).max() < 1e-13
    Hp = oracle.project(Psi, HPsi)
    assert np.abs(Hp - sub.w.H).max() < 1e-13                     # the residual part of H Psi is annihilated
    R = HPsi - sub.w.H @ Psi
    assert np.sqrt((R * R).mean()) > 0.05 * np.sqrt((HPsi * HPsi).mean())
    ev = np.linalg.eigvalsh(Hp)
    assert np.allclose(ev, np.sort(sub.w.lam), atol=1e-12)
