"""Pins for the CPU oracle (run with -m "not gpu").  Each test checks oracle/ against something
other than itself: a Jacobi eigendecomposition, a closed form, an invariant, brute force on a tiny
input, the scalar eigenvalue-space model, or a number the paper prints."""
import math
import os

import numpy as np
import pytest

import oracle
import rfoe_inputs
from tests import pins

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _tiny(k, nocc, seed, lo=(-1.0, -0.2), hi=(0.1, 2.0)):
    rng = np.random.default_rng(seed)
    lam = np.concatenate([rng.uniform(*lo, nocc), rng.uniform(*hi, k - nocc)])
    return rfoe_inputs.from_spectrum(lam, nocc, seed + 7, tol=1e-12)


# ---------------------------------------------------------------- O1 bounds
def test_bounds_bruteforce_and_enclose_spectrum():
    w = _tiny(24, 9, 3)
    H = w.H
    lo, hi = oracle.bounds(H)
    # brute force in pure Python
    los, his = [], []
    for i in range(24):
        r = sum(abs(H[i, j]) for j in range(24) if j != i)
        los.append(H[i, i] - r)
        his.append(H[i, i] + r)
    assert lo == min(los) and hi == max(his)
    ev, _ = pins.jacobi_eigh(H)
    assert lo <= ev[0] and ev[-1] <= hi          # Gershgorin circle theorem
    # diagonal matrix: radii vanish, bounds are the extreme diagonal entries
    d = np.diag([3.0, -2.0, 0.5])
    assert oracle.bounds(d) == (-2.0, 3.0)
    # a sign pattern that a dropped fabs() would get wrong
    A = np.array([[1.0, -4.0], [-4.0, 2.0]])
    assert oracle.bounds(A) == (-3.0, 6.0)


# ---------------------------------------------------------------- O2 affine map
def test_affine_map_closed_form():
    H = np.array([[1.0, 0.5], [0.5, -2.0]])
    X = oracle.affine(H, -3.0, 2.0)
    # occupied (low energy) -> 1: eigenvalue emin maps to 1, emax maps to 0
    assert np.array_equal(X, np.array([[(2.0 - 1.0) / 5.0, -0.5 / 5.0], [-0.5 / 5.0, (2.0 + 2.0) / 5.0]]))
    assert np.allclose(oracle.affine(np.diag([-3.0, 2.0]), -3.0, 2.0), np.diag([1.0, 0.0]))
    w = _tiny(16, 5, 11)
    lo, hi = oracle.bounds(w.H)
    ev = np.linalg.eigvalsh(oracle.affine(w.H, lo, hi))
    assert ev.min() >= 0.0 and ev.max() <= 1.0
    assert np.allclose(np.sort(ev), np.sort((hi - w.lam) / (hi - lo)), atol=1e-14)


# ---------------------------------------------------------------- O3 scalars, products
def test_scalars_and_products_against_definitions():
    rng = np.random.default_rng(5)
    X = rng.standard_normal((37, 37))
    X = X + X.T
    assert oracle.trace(X) == pytest.approx(math.fsum(np.diag(X)), rel=1e-15)
    assert oracle.sumsq(X) == pytest.approx(math.fsum((X * X).ravel()), rel=1e-14)
    # Tr(A^2) = ||A||_F^2 for symmetric A
    Y = oracle.square(X, literal=True)
    assert oracle.trace(Y) == pytest.approx(oracle.sumsq(X), rel=1e-13)
    # literal loop nest vs. pure-Python triple loop, bit for bit (3x3, non-symmetric product too)
    A = rng.standard_normal((5, 5))
    B = rng.standard_normal((5, 5))
    ref = np.zeros((5, 5))
    for i in range(5):
        for j in range(5):
            acc = 0.0
            for l in range(5):
                acc = acc + A[i, l] * B[l, j]
            ref[i, j] = acc
    assert np.array_equal(oracle.matmul(A, B, literal=True), ref)
    assert np.array_equal(oracle.matmul(A, B), ref)          # a transposed operand would fail here
    # interchanged/mirrored squaring is bit-identical to the literal one and bitwise symmetric
    for k in (1, 2, 7, 64, 193):
        Z = rng.standard_normal((k, k))
        Z = Z + Z.T
        S1, S2 = oracle.square(Z), oracle.square(Z, literal=True)
        assert np.array_equal(S1, S2) and oracle.is_symmetric(S1)
        assert np.allclose(S1, Z @ Z, rtol=0, atol=1e-12 * k)


# ---------------------------------------------------------------- P1 Jacobi projector
@pytest.mark.parametrize("k,nocc,seed", [(12, 4, 0), (33, 20, 1), (48, 47, 2), (20, 1, 3)])
def test_expand_matches_jacobi_projector(k, nocc, seed):
    w = _tiny(k, nocc, seed)
    r = oracle.expand(w.H, nocc, tol=1e-12)
    Pref, ev = pins.jacobi_projector(w.H, nocc)
    assert r.converged
    assert np.linalg.norm(r.P - Pref) <= 1e-12
    # north_star's three checks
    assert abs(np.trace(r.P) - nocc) <= 1e-11
    assert np.linalg.norm(r.P @ r.P - r.P) <= 1e-12
    assert np.linalg.norm(w.H @ r.P - r.P @ w.H) <= 1e-12
    assert r.tr_PH == pytest.approx(float(np.sum(ev[:nocc])), rel=1e-12)
    assert oracle.is_symmetric(r.P)


# ---------------------------------------------------------------- P2 construction-exact projector
def test_expand_matches_construction_projector_config1():
    w = rfoe_inputs.make_workload(1)
    r = oracle.expand(w.H, w.nocc, tol=w.tol)
    assert r.converged and r.iterations == 34      # 34 with Gershgorin bounds
    assert np.linalg.norm(r.P - w.exact_projector()) / math.sqrt(w.k) <= 1e-13
    assert abs(r.tr_PH - w.band_energy()) / abs(w.band_energy()) <= 1e-13


# ---------------------------------------------------------------- P3 invariants per step
def test_step_invariants():
    w = rfoe_inputs.make_workload(1, k=96)
    r = oracle.expand(w.H, w.nocc, tol=1e-12)
    n = r.iterations
    assert np.all(r.s[: n + 1] >= 0) and np.all(r.s <= r.t + 1e-12) and np.all(r.t <= w.k)
    # |t_{n+1} - t_n| = t_n - s_n (both branches)
    assert np.allclose(np.abs(np.diff(r.t)), (r.t[:-1] - r.s[:-1]), rtol=0, atol=1e-11)
    # branch sign: S lowers the trace, L raises it
    for i, b in enumerate(r.branch):
        assert (r.t[i + 1] <= r.t[i] + 1e-12) if b == "S" else (r.t[i + 1] >= r.t[i] - 1e-12)
        assert (b == "S") == (r.t[i] > w.nocc)
    assert abs(r.t[-1] - w.nocc) < 1e-10


# ---------------------------------------------------------------- P4 diagonal H = scalar recursion
def test_diagonal_hamiltonian_is_scalar_recursion():
    lam = np.array([-1.0, -0.7, -0.3, 0.2, 0.9, 1.4, 2.0])
    H = np.diag(lam)
    nocc = 3
    r = oracle.expand(H, nocc, tol=1e-13)
    lo, hi = lam.min(), lam.max()                  # Gershgorin is exact for a diagonal matrix
    assert (r.emin, r.emax) == (lo, hi)
    m = pins.scalar_sp2(lam, nocc, lo, hi, tol=1e-13)
    assert r.branch == m["branch"]
    assert np.array_equal(np.diag(r.P), m["x"])     # same operations on each diagonal entry
    assert np.count_nonzero(r.P - np.diag(np.diag(r.P))) == 0
    assert np.allclose(np.diag(r.P), [1, 1, 1, 0, 0, 0, 0], atol=1e-13)


def test_two_by_two_closed_form():
    # H = R diag(-1, 1) R^T, nocc = 1: P = v v^T with v the eigenvector of -1
    th = 0.3
    v = np.array([math.cos(th), math.sin(th)])
    u = np.array([-math.sin(th), math.cos(th)])
    H = -np.outer(v, v) + np.outer(u, u)
    H = 0.5 * (H + H.T)
    r = oracle.expand(H, 1, tol=1e-14)
    assert np.allclose(r.P, np.outer(v, v), atol=1e-14)


# ---------------------------------------------------------------- P5 scalar model: counts, branch strings
@pytest.mark.parametrize("c,k", [(1, 256), (2, 320), (3, 256), (4, 384)])
def test_scalar_model_predicts_matrix_run(c, k):
    w = rfoe_inputs.make_workload(c, k=k)
    r = oracle.expand(w.H, w.nocc, tol=w.tol)
    m = pins.scalar_sp2(w.lam, w.nocc, r.emin, r.emax, tol=w.tol)
    assert r.converged
    assert r.iterations == m["iterations"]
    n = r.iterations
    # the branch is unique except where t_n - nocc is at rounding level (after convergence; R10)
    decided = np.abs(r.t[:n] - w.nocc) > 1e-9
    assert decided[: n - 4].all()
    assert all(a == b for a, b, d in zip(r.branch, m["branch"], decided) if d)
    assert np.allclose(r.t, m["t"], rtol=0, atol=1e-9)
    assert np.allclose(r.s, m["s"], rtol=0, atol=1e-9)
    assert np.allclose(r.e[: n - 1], m["e"][: n - 1], rtol=1e-6, atol=1e-12)


def test_rule_b_reltr():
    w = rfoe_inputs.make_workload(1, k=128)
    r = oracle.expand(w.H, w.nocc, tol=5e-8, stop_rule=oracle.RULE_B)
    m = pins.scalar_sp2(w.lam, w.nocc, r.emin, r.emax, tol=5e-8, rule="B")
    assert r.iterations == m["iterations"] and r.branch == m["branch"]
    assert r.reltr[-1] <= 5e-8 < r.reltr[-2]
    assert np.allclose(r.reltr, np.abs(np.diff(r.t)) / np.abs(r.t[:-1]), rtol=1e-12)


# ---------------------------------------------------------------- P6 the paper's printed iteration counts
def test_paper_matrix_iteration_counts():
    """PAPER.md:92 (section IV): RelTr 5e-8 gives 'around 50' Z-RFOE and 'around 30' A-Z-RFOE
    iterations on H_ij = exp(-0.5|i-j|) sin(i+1) with N_occ ~ 0.9 k.  The golden file
    quotes the sentence; tolerance bands are ours (around = +-20 %)."""
    with open(os.path.join(GOLDEN, "paper_iteration_counts.txt")) as f:
        txt = f.read()
    z, az = [int(x) for x in txt.split("VALUES:")[1].split()[:2]]
    assert (z, az) == (50, 30)
    k = 768
    H = rfoe_inputs.paper_matrix(k)
    nocc = round(0.9 * k)
    r = oracle.expand(H, nocc, tol=5e-8, stop_rule=oracle.RULE_B, max_iter=120)
    assert r.converged and abs(r.iterations - z) <= 0.2 * z, r.iterations
    ev = np.linalg.eigvalsh(H)
    ra = oracle.expand(H, nocc, variant=oracle.SP2_ACCEL, tol=5e-8, stop_rule=oracle.RULE_B, max_iter=120,
                       homo=float(ev[nocc - 1]), lumo=float(ev[nocc]))
    assert ra.converged and abs(ra.iterations - az) <= 0.2 * az, ra.iterations
    # both reach the same projector; errors at the level the paper reports (eps1 ~ 1e-10, eps2 ~ 1e-9)
    V = np.linalg.eigh(H)[1][:, :nocc]
    Pref = V @ V.T
    for res in (r, ra):
        eps1 = np.linalg.norm(res.P - Pref) / np.linalg.norm(Pref)
        eps2 = abs(res.tr_PH - np.sum(ev[:nocc])) / abs(np.sum(ev[:nocc]))
        assert eps1 < 1e-6 and eps2 < 1e-8, (eps1, eps2)


# ---------------------------------------------------------------- variants
def test_accelerated_matches_scalar_model_and_jacobi():
    w = _tiny(40, 13, 21)
    homo, lumo = w.lam[: w.nocc].max(), w.lam[w.nocc:].min()
    r = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=1e-12, homo=homo, lumo=lumo)
    plain = oracle.expand(w.H, w.nocc, tol=1e-12)
    m = pins.scalar_sp2_accel(w.lam, w.nocc, r.emin, r.emax, homo, lumo, tol=1e-12, rule="A")
    assert r.converged and r.iterations == m["iterations"]
    assert r.branch[:-2] == m["branch"][:-2]          # last steps: t - nocc is rounding noise (R10)
    assert r.iterations < plain.iterations
    Pref, _ = pins.jacobi_projector(w.H, w.nocc)
    assert np.linalg.norm(r.P - Pref) <= 1e-11


def test_mcweeny_variant_reaches_projector():
    w = _tiny(36, 14, 8)
    r = oracle.expand(w.H, w.nocc, variant=oracle.MCWEENY, tol=1e-12)
    Pref, _ = pins.jacobi_projector(w.H, w.nocc)
    assert r.converged and r.mcweeny_steps >= 1 and "M" in r.branch
    assert r.multiplications == r.iterations + r.mcweeny_steps
    assert r.branch.rstrip("M").count("M") == 0          # SP2 phase first, then only McWeeny steps
    assert np.linalg.norm(r.P - Pref) <= 1e-12
    assert abs(np.trace(r.P) - w.nocc) <= 1e-11 and oracle.is_symmetric(r.P)
    # the McWeeny polynomial on a diagonal matrix: x -> 3x^2 - 2x^3
    x = np.array([0.95, 0.97, 0.04, 0.02])
    r2 = oracle.expand(np.diag(1.0 - x), 2, variant=oracle.MCWEENY, tol=0.0, max_iter=1,
                       bounds_override=(0.0, 1.0))
    assert r2.branch == "M"
    assert np.allclose(np.diag(r2.P), 3 * x**2 - 2 * x**3, rtol=1e-15)


def test_mixed_variant_schedule_and_accuracy():
    w = _tiny(48, 30, 4)
    r64 = oracle.expand(w.H, w.nocc, tol=1e-12)
    # paper schedule: FP32 from the start until RelTr <= 5e-4, FP64 to the end
    r = oracle.expand(w.H, w.nocc, variant=oracle.SP2_MIXED, tol=1e-12, mixed_head=0.0, mixed_reltr=5e-4)
    assert r.converged and r.fp32_steps >= 1
    assert r.branch[: r.fp32_steps].islower() and r.branch[r.fp32_steps:].isupper()
    assert r.branch.upper()[: r.fp32_steps] == r64.branch[: r.fp32_steps]
    Pref, _ = pins.jacobi_projector(w.H, w.nocc)
    err = np.linalg.norm(r.P - Pref) / math.sqrt(w.k)
    assert 1e-12 < err < 1e-4          # FP32 damage is visible but small (paper: eps1 ~ 1e-7)
    assert np.linalg.norm(r.P @ r.P - r.P) <= 1e-11


def test_truncated_expansion_is_smeared_step_function():
    """T-RFOE (Eq. 2): stopping after m steps leaves fractional occupancies; the
    intermediate G_m(H) = Q diag(g_m(lambda)) Q^T with g_m the composed scalar polynomials."""
    w = _tiny(32, 12, 17, lo=(-1.0, -0.02), hi=(0.02, 1.0))
    m_steps = 8
    r = oracle.expand(w.H, w.nocc, tol=0.0, max_iter=m_steps)
    assert r.iterations == m_steps and not r.converged
    m = pins.scalar_sp2(w.lam, w.nocc, r.emin, r.emax, tol=0.0, max_iter=m_steps)
    G = (w.Q * m["x"][None, :]) @ w.Q.T
    assert np.allclose(r.P, G, atol=1e-12)
    occ = np.linalg.eigvalsh(r.P)
    assert occ.min() > -1e-12 and occ.max() < 1 + 1e-12
    assert np.sum((occ > 1e-3) & (occ < 1 - 1e-3)) > 0          # fractional occupancies present
    # monotone in energy, like a Fermi-Dirac function
    order = np.argsort(w.lam)
    assert np.all(np.diff(m["x"][order]) <= 1e-15)


def test_bad_arguments():
    with pytest.raises(RuntimeError):
        oracle.expand(np.array([[1.0, 2.0], [3.0, 4.0]]), 1)          # not symmetric
    with pytest.raises(RuntimeError):
        oracle.expand(np.eye(3), 1)                                   # emax == emin


# ---------------------------------------------------------------- the FP32 product, bit for bit
def test_square_f32_bits():
    """The mixed variants' FP32 step: X rounded to binary32, every product and sum a binary32
    operation, l ascending -- against a literal numpy.float32 triple loop, bit for bit.  A double-accumulating
    (or FMA-contracting) version must fail: the test first checks that such versions differ on these inputs."""
    rng = np.random.default_rng(123)
    for k in (1, 2, 5, 8):
        X = rng.standard_normal((k, k))
        X = X + X.T
        xf = X.astype(np.float32)
        ref = np.zeros((k, k), dtype=np.float32)
        dbl = np.zeros((k, k))
        for i in range(k):
            for j in range(k):
                acc = np.float32(0.0)
                accd = 0.0
                for l in range(k):
                    acc = np.float32(acc + np.float32(xf[i, l] * xf[l, j]))
                    accd = accd + float(xf[i, l]) * float(xf[l, j])
                ref[i, j] = acc
                dbl[i, j] = accd
        Y = oracle.square_f32(X)
        assert np.array_equal(Y, ref.astype(np.float64))
        assert oracle.is_symmetric(Y)
        if k >= 5:
            assert not np.array_equal(ref.astype(np.float64), dbl.astype(np.float32).astype(np.float64))
            assert not np.array_equal(Y, oracle.square(X))


# ---------------------------------------------------------------- mixed schedule: where the phases switch
def test_mixed_phase_switch_on_diagonal():
    """FP32 steps until RelTr <= mixed_reltr, FP64 afterwards; optional FP64 head while
    Tr X - Tr X^2 >= mixed_head (reading R-MIX).  On a diagonal H the matrix run is the scalar recursion, so the
    positions of the lower-case (FP32) steps follow from the plain FP64 scalar model's history (pins.scalar_sp2,
    which knows nothing about phases): the FP32 phase starts at the first step n with t_n - s_n < head and the
    last FP32 step is the first one whose RelTr <= switch.  Thresholds sit far from any t_n - s_n / RelTr value."""
    rng = np.random.default_rng(31)
    k, nocc = 40, 17
    lam = np.sort(np.concatenate([rng.uniform(-1.0, -0.1, nocc), rng.uniform(0.1, 1.5, k - nocc)]))
    H = np.diag(lam)
    lo, hi = -4.0, 5.0
    m = pins.scalar_sp2(lam, nocc, lo, hi, tol=1e-12)
    gap = m["t"][:-1] - m["s"][:-1]                       # t_n - s_n, the quantity the head watches
    reltr = np.abs(np.diff(m["t"])) / np.abs(m["t"][:-1])
    n_steps = m["iterations"]
    for head, switch in [(0.0, 5e-4), (1.8, 5e-4), (0.5, 1e-6), (0.0, 0.0)]:
        # thresholds must not sit within 5 % of any history value, else FP32 noise could move the switch
        assert head == 0.0 or all(abs(g - head) > 0.05 * head for g in gap)
        assert switch == 0.0 or all(abs(r - switch) > 0.05 * switch for r in reltr)
        first = 0 if head == 0.0 else int(np.argmax(gap < head))
        if switch == 0.0:
            expected = None                              # leaves FP32 only once the trace stops moving at all
        else:
            last = next(n for n in range(first, n_steps) if reltr[n] <= switch)
            expected = "".join(ch.lower() if first <= n <= last else ch for n, ch in enumerate(m["branch"]))
        r = oracle.expand(H, nocc, variant=oracle.SP2_MIXED, tol=1e-12, bounds_override=(lo, hi),
                          mixed_head=head, mixed_reltr=switch, max_iter=60)
        if expected is None:
            nf = r.fp32_steps
            assert r.branch[:nf].islower() and r.branch[nf:].isupper() and nf >= n_steps - 4
            assert r.reltr[nf - 1] == 0.0 and np.all(r.reltr[: nf - 1] > 0.0)
            continue
        assert r.converged and r.branch == expected, (head, switch, r.branch, expected)
        assert r.fp32_steps == last - first + 1
        # FP32 steps leave FP32-level, not FP64-level, agreement with the FP64 model; FP64 steps then repair it
        assert np.allclose(np.diag(r.P), (lam < 0).astype(float), atol=1e-12)
    # the FP32 steps really are FP32: after one FP32 step every diagonal entry is a binary32 number
    r1 = oracle.expand(H, nocc, variant=oracle.TRUNC_MIXED, max_iter=1, bounds_override=(lo, hi), mixed_reltr=0.0)
    d = np.diag(r1.P)
    x0 = ((hi - lam) / (hi - lo)).astype(np.float32)
    sq = (x0 * x0).astype(np.float64)
    want = sq if r1.branch == "s" else 2.0 * ((hi - lam) / (hi - lo)) - sq
    assert r1.branch in ("s", "l") and np.array_equal(d, want)


# ---------------------------------------------------------------- sign rule outside [0,1]
def test_sign_rule_repairs_out_of_range_eigenvalue():
    """"the +/- sign is chosen to adjust the trace of X_{n+1} ... such that it converges to N_occ".
    Worked by hand on a diagonal X_0 (bounds override (0,1), so X_0 = I - H):
      * one eigenvalue at 1 + d, d = 1e-7 (as rounding noise of an FP32 phase leaves it), the rest at 0/1:
        t = N + d, Tr X^2 = N + 2d + d^2, Tr(2X - X^2) = N - d^2 -> the "+" branch 2X - X^2 lands nearer N_occ and maps
        1 + d to 1 - d^2; the naive "X^2 iff t > N_occ" would square it to 1 + 2d and double the excess every step.
      * mirror case, one eigenvalue at -d: t = N - d, Tr X^2 = N + d^2, Tr(2X - X^2) = N - 2d - d^2 -> X^2, mapping -d to d^2."""
    d = 1e-7
    for x0, first, fixed in [(np.array([1.0 + d, 1.0, 0.0, 0.0]), "L", 1.0 - d * d),
                             (np.array([1.0, 1.0, -d, 0.0]), "S", d * d)]:
        nocc = 2
        H = np.diag(1.0 - x0)
        r = oracle.expand(H, nocc, tol=1e-13, bounds_override=(0.0, 1.0), max_iter=20)
        assert r.branch[0] == first, r.branch
        assert r.t[0] == pytest.approx(float(x0.sum()), abs=1e-15)
        one = oracle.expand(H, nocc, variant=oracle.TRUNC, max_iter=1, bounds_override=(0.0, 1.0))
        i = int(np.argmax(np.abs(x0 * (1 - x0))))          # the out-of-range entry
        assert np.diag(one.P)[i] == pytest.approx(fixed, abs=1e-20 if fixed < 1e-3 else 1e-15)
        assert r.converged and r.iterations <= 3
        assert np.all(np.diag(r.P) >= 0.0) and np.all(np.diag(r.P) <= 1.0)
        assert np.allclose(np.diag(r.P), [1, 1, 0, 0], atol=1e-13)


# ---------------------------------------------------------------- A-Z-RFOE: unexpanded form, step by step
def test_accelerated_unexpanded_form_traces():
    """A-Z-RFOE (reading R-ACC) step by step in eigenvalue space: X_n = Q diag(x_n) Q^T, so Tr X_n is the
    sum of the shifted-and-scaled SP2 polynomial applied to each eigenvalue (pins.scalar_sp2_accel applies
    ((1-a) + a x)^2 and 2(ax) - (ax)^2 literally).  A dropped shift, a wrong alpha or a swapped HOMO/LUMO image
    changes t_1 already."""
    w = _tiny(28, 11, 41)
    homo, lumo = w.lam[: w.nocc].max(), w.lam[w.nocc:].min()
    r = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=1e-12, homo=homo, lumo=lumo)
    x = (r.emax - w.lam) / (r.emax - r.emin)
    beta, bbar = (r.emax - lumo) / (r.emax - r.emin), (r.emax - homo) / (r.emax - r.emin)
    for n, ch in enumerate(r.branch[:8]):
        aS, aL = 2.0 / (2.0 - beta), 2.0 / (1.0 + bbar)
        cand = {"S": ((1.0 - aS) + aS * x) ** 2, "L": 2.0 * (aL * x) - (aL * x) ** 2}
        # the branch taken is the one whose trace (summing the candidate's eigenvalues) is nearer N_occ
        assert abs(cand[ch].sum() - w.nocc) <= abs(cand["L" if ch == "S" else "S"].sum() - w.nocc)
        f = (lambda v, a=aS: ((1.0 - a) + a * v) ** 2) if ch == "S" else (lambda v, a=aL: 2.0 * (a * v) - (a * v) ** 2)
        x, beta, bbar = f(x), f(beta), f(bbar)
        assert r.t[n + 1] == pytest.approx(x.sum(), abs=1e-11)
        assert r.s[n + 1] == pytest.approx((x * x).sum(), abs=1e-11)
        # HOMO / LUMO images stay the edges of the gap in the mapped spectrum
        assert beta == pytest.approx(x[w.nocc:].max(), abs=1e-12) and bbar == pytest.approx(x[: w.nocc].min(), abs=1e-12)
    # estimates outside the spectral bounds are refused (alpha would leave (0, 2))
    with pytest.raises(RuntimeError):
        oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, homo=r.emin - 1.0, lumo=lumo)
    with pytest.raises(RuntimeError):
        oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, homo=lumo, lumo=homo)


# ---------------------------------------------------------------- T-RFOE against the exact Fermi-Dirac matrix
def test_truncated_variant_runs_exactly_m_steps():
    w = _tiny(32, 12, 17, lo=(-1.0, -0.02), hi=(0.02, 1.0))
    for m_steps in (1, 5, 9):
        r = oracle.expand(w.H, w.nocc, variant=oracle.TRUNC, max_iter=m_steps)
        old = oracle.expand(w.H, w.nocc, tol=0.0, max_iter=m_steps)          # the same arithmetic by the SP2 route
        assert r.converged and r.iterations == m_steps and not old.converged
        assert np.array_equal(r.P, old.P) and r.branch == old.branch
    # even when the expansion has long converged, T-RFOE keeps going to m (no convergence test)
    r = oracle.expand(w.H, w.nocc, variant=oracle.TRUNC, max_iter=70)
    assert r.iterations == 70 and r.converged


@pytest.mark.parametrize("k", [96, 256])
def test_truncated_expansion_vs_fermi_dirac(k):
    """D = [exp(beta (H - mu I)) + I]^-1;  PAPER.md:47-52 (Eq. 2): the truncated G_m(H) "serves as a
    smeared function" standing in for it, more steps m <-> higher beta;  PAPER.md:86: the paper's matrix with 85 %
    of the states occupied;  PAPER.md:92: eps1 ~ 1e-3 against the exact Fermi-Dirac density matrix, "around 30"
    T-RFOE iterations at 500 K.  The paper gives no m <-> beta relation (reading R-TRUNC): for each m the pair
    (mu, beta) is fitted to the occupancies of G_m by least squares and the paper's error metrics
    are taken against D_FD = V f(lambda) V^T built from numpy's eigendecomposition."""
    H = rfoe_inputs.paper_matrix(k)
    nocc = round(0.85 * k)
    lam, V = np.linalg.eigh(H)
    mu0 = 0.5 * (lam[nocc - 1] + lam[nocc])
    betas, eps1s = [], []
    for m_steps in (12, 16, 20, 24, 28, 32, 36):
        r = oracle.expand(H, nocc, variant=oracle.TRUNC, max_iter=m_steps)
        assert r.iterations == m_steps
        occ = np.einsum("ij,ij->j", V, r.P @ V)                      # v_i^T G_m v_i
        assert np.linalg.norm(r.P - (V * occ[None, :]) @ V.T) <= 1e-10   # G_m is a function of H
        assert occ.min() > -1e-9 and occ.max() < 1 + 1e-9
        assert np.all(np.diff(occ) <= 1e-9)                          # monotone in energy, like f_FD
        mu, beta = pins.fit_fermi_dirac(lam, occ, mu0)
        f = pins.fermi_dirac(lam, mu, beta)
        D = (V * f[None, :]) @ V.T
        eps1 = np.linalg.norm(r.P - D) / np.linalg.norm(D)
        eps2 = abs(r.tr_PH - float(np.sum(f * lam))) / abs(float(np.sum(f * lam)))
        assert eps1 <= 5e-3 and eps2 <= 5e-3, (m_steps, eps1, eps2)   # paper: eps1 ~ 1e-3
        assert lam[0] < mu < lam[-1]
        betas.append(beta)
        eps1s.append(eps1)
    assert all(b1 > b0 for b0, b1 in zip(betas, betas[1:]))          # more steps <-> lower temperature
    assert betas[-1] / betas[0] > 30
    assert max(eps1s) >= 1e-4                                        # a smeared stand-in, not the Fermi function itself
    # "around 30" iterations at 500 K (golden value 3): with the matrix read in Hartree, beta(500 K) = 1 / (k_B T) =
    # 631.6; the m whose fitted beta is nearest lies within +-25 % of 30 (m runs in steps of 4 here)
    with open(os.path.join(GOLDEN, "paper_iteration_counts.txt")) as fh:
        t_iters = int(fh.read().split("VALUES:")[1].split()[2])
    assert t_iters == 30
    beta_500K = 1.0 / (3.166811563e-6 * 500.0)
    m_near = (12, 16, 20, 24, 28, 32, 36)[int(np.argmin(np.abs(np.log(np.array(betas) / beta_500K))))]
    assert abs(m_near - t_iters) <= 0.25 * t_iters, (m_near, betas)
