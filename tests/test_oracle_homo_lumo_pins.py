"""Pins for oracle.estimate_homo_lumo (run with -m "not gpu"), and the library's host-only
rfoe_estimate_homo_lumo against it (no device needed: both are functions of a run's scalar history).

The estimator is checked against things other than itself: the eigenvalues the generator put into H^p, a case where
the bound is attained exactly (one interior eigenvalue), the per-step spectrum of X_n in eigenvalue space, and the
accelerated run it feeds, whose projector is compared with the construction-exact one."""
import ctypes as C
import math

import numpy as np
import pytest

import oracle
import rfoe_inputs


def _run(c, k):
    w = rfoe_inputs.make_workload(c, k=k)
    return w, oracle.expand(w.H, w.nocc, tol=w.tol)


@pytest.mark.parametrize("c,k", [(1, 256), (2, 384), (3, 320), (4, 400)])
def test_estimates_lie_inside_the_gap_and_close_to_its_edges(c, k):
    w, res = _run(c, k)
    lam_homo, lam_lumo = float(np.max(w.lam[: w.nocc])), float(np.min(w.lam[w.nocc:]))
    gap = lam_lumo - lam_homo
    homo, lumo = oracle.estimate_homo_lumo(res, w.nocc)
    slack = 1e-9 * (res.emax - res.emin)                 # rounding of X_n, carried back (DESIGN.md R-HL)
    assert lam_homo - slack <= homo < lumo <= lam_lumo + slack
    assert homo - lam_homo <= 0.05 * gap and lam_lumo - lumo <= 0.05 * gap


def test_bound_is_attained_with_a_single_interior_eigenvalue():
    """Occupied eigenvalues at eps_min (x = 1 exactly, x(1-x) = 0 at every step), one unoccupied eigenvalue inside:
    e_n = y_n (1 - y_n) exactly, so every admissible step returns the LUMO itself; mirrored for the HOMO."""
    k, nocc = 6, 4
    lam = np.array([-2.0] * nocc + [0.75, 3.0])              # unoccupied: 0.75 (interior) and eps_max (x = 0)
    res = oracle.expand(np.diag(lam), nocc, tol=1e-13, bounds_override=(-2.0, 3.0))
    _, lumo = oracle.estimate_homo_lumo(res, nocc)
    assert lumo == pytest.approx(0.75, abs=1e-12)
    lam = np.array([-2.0] * (nocc - 1) + [-0.5] + [3.0, 3.0])  # one interior occupied eigenvalue
    res = oracle.expand(np.diag(lam), nocc, tol=1e-13, bounds_override=(-2.0, 3.0))
    homo, _ = oracle.estimate_homo_lumo(res, nocc)
    assert homo == pytest.approx(-0.5, abs=1e-12)


def test_every_admissible_step_bounds_the_images_in_eigenvalue_space():
    """Brute force: push the generator's eigenvalues through the branches the run took; at each step the images of HOMO and
    LUMO must respect x(1-x) <= e_n, and the estimate must be the tightest back-mapped bound."""
    w, res = _run(2, 384)
    x = (res.emax - w.lam) / (res.emax - res.emin)
    ih, il = int(np.argmax(w.lam[: w.nocc])), w.nocc + int(np.argmin(w.lam[w.nocc:]))
    admissible = 0
    best_h, best_l = math.inf, -math.inf
    for n, ch in enumerate(res.branch):
        settled = res.t[n] - res.s[n] < 3 / 16 and abs(res.t[n] - w.nocc) < 0.5
        if settled and 1e-6 <= res.e[n] < 0.25:
            admissible += 1
            a = 0.5 * (1 - math.sqrt(1 - 4 * res.e[n]))
            assert x[il] <= a * (1 + 1e-9) and x[ih] >= 1 - a * (1 + 1e-9)
            assert np.all((x <= a * (1 + 1e-9)) | (x >= 1 - a * (1 + 1e-9)))      # two clusters, nothing between
            assert int(np.sum(x > 0.5)) == w.nocc
            # carry [a, 1-a] back by root finding on the forward polynomials instead of the closed-form inverses
            def forward(x0):
                for chj in res.branch[:n]:
                    x0 = x0 * x0 if chj == "S" else 2 * x0 - x0 * x0
                return x0
            def invert(target):
                lo, hi = 0.0, 1.0
                for _ in range(200):
                    mid = 0.5 * (lo + hi)
                    lo, hi = (mid, hi) if forward(mid) < target else (lo, mid)
                return 0.5 * (lo + hi)
            best_l = max(best_l, res.emax - (res.emax - res.emin) * invert(a))
            best_h = min(best_h, res.emax - (res.emax - res.emin) * invert(1 - a))
        x = x * x if ch == "S" else 2 * x - x * x
    assert admissible >= 3
    homo, lumo = oracle.estimate_homo_lumo(res, w.nocc)
    width = res.emax - res.emin
    assert homo == pytest.approx(best_h, abs=1e-9 * width) and lumo == pytest.approx(best_l, abs=1e-9 * width)


@pytest.mark.parametrize("c,k", [(1, 256), (3, 320)])
def test_accelerated_run_fed_with_the_estimates(c, k):
    w, res = _run(c, k)
    homo, lumo = oracle.estimate_homo_lumo(res, w.nocc)
    acc = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=w.tol, homo=homo, lumo=lumo)
    exact = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=w.tol,
                          homo=float(np.max(w.lam[: w.nocc])), lumo=float(np.min(w.lam[w.nocc:])))
    assert acc.converged and acc.iterations < res.iterations
    assert abs(acc.iterations - exact.iterations) <= 1
    assert np.linalg.norm(acc.P - w.exact_projector()) / math.sqrt(k) <= 1e-12
    assert round(np.trace(acc.P)) == w.nocc


def test_rejections():
    w = rfoe_inputs.make_workload(1)
    short = oracle.expand(w.H, w.nocc, tol=0.0, max_iter=6)          # stopped long before the occupation settles
    with pytest.raises(RuntimeError):
        oracle.estimate_homo_lumo(short, w.nocc)
    mixed = oracle.expand(w.H, w.nocc, variant=oracle.SP2_MIXED, tol=w.tol)
    with pytest.raises(ValueError):
        oracle.estimate_homo_lumo(mixed, w.nocc)


# ------------------------------------------------------------------------------------------------------------------
# host logic of the library: rfoe_estimate_homo_lumo is a function of rfoe_stats_t alone, so it runs without a GPU
def _stats_from(res, nocc, rfoe):
    st = rfoe._Stats()
    st.variant, st.iterations, st.fp32_steps, st.nocc = rfoe.SP2, res.iterations, res.fp32_steps, nocc
    st.eps_min, st.eps_max = res.emin, res.emax
    for n in range(res.iterations + 1):
        st.t[n], st.s[n] = res.t[n], res.s[n]
    for n in range(res.iterations):
        st.e[n] = res.e[n]
    st.branch = res.branch.encode()
    return st


@pytest.mark.parametrize("c,k", [(1, 256), (2, 384), (4, 400)])
def test_library_host_function_matches_oracle(c, k):
    import paper_2301_04642_b200 as rfoe

    w, res = _run(c, k)
    homo, lumo = rfoe.estimate_homo_lumo(_stats_from(res, w.nocc, rfoe))
    oh, ol = oracle.estimate_homo_lumo(res, w.nocc)
    width = res.emax - res.emin
    assert homo == pytest.approx(oh, abs=1e-10 * width) and lumo == pytest.approx(ol, abs=1e-10 * width)


def test_library_host_function_error_codes():
    import paper_2301_04642_b200 as rfoe

    w = rfoe_inputs.make_workload(1)
    res = oracle.expand(w.H, w.nocc, tol=w.tol)
    L = rfoe.load_library()
    a, b = C.c_double(), C.c_double()
    st = _stats_from(res, w.nocc, rfoe)
    assert L.rfoe_estimate_homo_lumo(None, C.byref(a), C.byref(b)) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_estimate_homo_lumo(C.byref(st), None, C.byref(b)) == rfoe.ERR_INVALID_ARG
    st.variant = rfoe.SP2_ACCEL
    assert L.rfoe_estimate_homo_lumo(C.byref(st), C.byref(a), C.byref(b)) == rfoe.ERR_UNSUPPORTED
    st = _stats_from(res, w.nocc, rfoe)
    st.branch = res.branch.lower().encode()                            # reduced-precision steps in the history
    assert L.rfoe_estimate_homo_lumo(C.byref(st), C.byref(a), C.byref(b)) == rfoe.ERR_UNSUPPORTED
    st = _stats_from(res, w.nocc, rfoe)
    st.iterations = 5                                                  # history cut before the occupation settles
    assert L.rfoe_estimate_homo_lumo(C.byref(st), C.byref(a), C.byref(b)) == rfoe.ERR_NOT_CONVERGED
    st.eps_max = st.eps_min
    assert L.rfoe_estimate_homo_lumo(C.byref(st), C.byref(a), C.byref(b)) == rfoe.ERR_INVALID_ARG
