"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (north_star, FP64 path): ||P_gpu - P_oracle||_F / sqrt(k) <= 1e-10, |tr(P H) difference| / |tr| <= 1e-11,
identical iteration counts; branch strings identical wherever t_n - nocc is above rounding level (R10).
Kernel-level products: the DMMA path and the oracle sum the same k products per element in different
orders, so |C_gpu - C_oracle| <= 4 k eps max|x|^2.
"""
import math

import numpy as np
import pytest

import oracle
import rfoe_inputs
from tests import pins

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2301_04642_b200 as rfoe  # noqa: E402

EPS = 2.0 ** -52


@pytest.fixture(scope="module")
def handle():
    h = rfoe.Rfoe(2048)
    yield h
    h.close()


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _sym(k, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    X = rng.standard_normal((k, k)) * scale
    return np.ascontiguousarray(0.5 * (X + X.T))


# ------------------------------------------------------------------ A1: Gershgorin
@pytest.mark.parametrize("k", [1, 2, 7, 64, 129, 255, 1000, 2048])
def test_bounds_parity(handle, k):
    H = _sym(k, 10 + k)
    lo, hi = handle.bounds(_dev(H))
    olo, ohi = oracle.bounds(H)
    tol = 4 * k * EPS * max(abs(olo), abs(ohi), 1.0)
    assert abs(lo - olo) <= tol and abs(hi - ohi) <= tol


# ------------------------------------------------------------------ A4 + A5: one squaring, all outputs
@pytest.mark.parametrize("k", [1, 5, 64, 128, 130, 257, 384, 777])
@pytest.mark.parametrize("coef", [(1.0, 0.0, 0.0), (-1.0, 2.0, 0.0), (1.21, -0.44, 0.04)])
def test_square_parity(handle, k, coef):
    X = _sym(k, 100 + k, scale=1.0 / math.sqrt(k))
    c2, c1, c0 = coef
    out, sc, ms = handle.square(_dev(X), c2, c1, c0)
    out = out.cpu().numpy()
    Y = oracle.square(X)
    ref = c2 * Y + c1 * X + c0 * np.eye(k)
    xmax = np.abs(X).max()
    tol = 4 * k * EPS * xmax * xmax * (abs(c2) + 1) + 4 * EPS * np.abs(ref).max()
    assert np.abs(out - ref).max() <= tol
    assert np.array_equal(out, out.T)                                  # bitwise symmetric
    rel = 1e-12
    assert sc[0] == pytest.approx(np.trace(ref), rel=rel, abs=1e-13)
    assert sc[1] == pytest.approx(np.sum(ref * ref), rel=rel)
    assert sc[2] == pytest.approx(np.sum((Y - X) ** 2), rel=rel)
    assert sc[3] == pytest.approx(np.trace(Y), rel=rel)
    assert sc[3] == pytest.approx(np.sum(X * X), rel=rel)                # Tr(X^2) = ||X||_F^2
    assert sc[4] == pytest.approx(np.sum(Y * X), rel=1e-10, abs=1e-12)
    if coef == (1.0, 0.0, 0.0):
        # exact when every product and partial sum is representable: small integers
        Xi = np.random.default_rng(k).integers(-3, 4, size=(k, k)).astype(np.float64)
        Xi = np.triu(Xi) + np.triu(Xi, 1).T
        outi, _, _ = handle.square(_dev(Xi))
        assert np.array_equal(outi.cpu().numpy(), oracle.square(Xi))


@pytest.mark.parametrize("k", [2100, 3000])
def test_square_parity_main_plus_tail_launch(k):
    """Sizes whose launch is a whole-wave main part PLUS a split-K tail (rfoe_plan_squaring: n_main > 0, slices > 1),
    ragged in both (2100 = 16*128 + 52, 3000 = 23*128 + 56): every element against the oracle, both SP2 branches."""
    nt, nm, sl, _ = rfoe.plan_squaring(k, torch.cuda.get_device_properties(0).multi_processor_count)
    assert 0 < nm < nt and sl > 1
    X = _sym(k, 100 + k, scale=1.0 / math.sqrt(k))
    Y = oracle.square(X)
    xmax = np.abs(X).max()
    with rfoe.Rfoe(k) as h:
        for c2, c1 in [(1.0, 0.0), (-1.0, 2.0)]:
            out, sc, _ = h.square(_dev(X), c2, c1, 0.0)
            out = out.cpu().numpy()
            ref = c2 * Y + c1 * X
            assert np.abs(out - ref).max() <= 8 * k * EPS * xmax * xmax + 4 * EPS * np.abs(ref).max()
            assert np.array_equal(out, out.T)
            assert sc[0] == pytest.approx(np.trace(ref), rel=1e-12)
            assert sc[1] == pytest.approx(np.sum(ref * ref), rel=1e-12)
            assert sc[2] == pytest.approx(np.sum((Y - X) ** 2), rel=1e-12)
            assert sc[3] == pytest.approx(np.sum(X * X), rel=1e-12)
        Xi = np.random.default_rng(k).integers(-3, 4, size=(k, k)).astype(np.float64)
        Xi = np.triu(Xi) + np.triu(Xi, 1).T
        outi, _, _ = h.square(_dev(Xi))
        assert np.array_equal(outi.cpu().numpy(), oracle.square(Xi))       # exact on small integers


@pytest.mark.parametrize("k", [3, 128, 200, 515])
def test_symm_product_parity(handle, k):
    X = _sym(k, 300 + k, scale=1.0 / math.sqrt(k))
    Y = oracle.square(X)                                                 # commutes with X, symmetric
    out, sc, _ = handle.symm_product(_dev(Y), _dev(X), -2.0, 3.0, 0.0)     # McWeeny: 3Y - 2YX
    out = out.cpu().numpy()
    Z = oracle.matmul(Y, X)
    ref = np.triu(3.0 * Y - 2.0 * Z)
    ref = ref + np.triu(ref, 1).T
    tol = 8 * k * EPS * np.abs(Y).max() * np.abs(X).max() + 8 * EPS * np.abs(ref).max()
    assert np.abs(out - ref).max() <= tol
    assert np.array_equal(out, out.T)
    assert sc[0] == pytest.approx(np.trace(ref), rel=1e-12)
    assert sc[1] == pytest.approx(np.sum(ref * ref), rel=1e-12)


# ------------------------------------------------------------------ whole expansions
def _check_expansion(w, res, ref, *, ptol=1e-10, etol=1e-11, inv=1.0, projector=True):
    k = w.k
    P = res.P.cpu().numpy() if hasattr(res.P, "cpu") else res.P
    assert res.converged == ref.converged
    assert res.iterations == ref.iterations
    decided = np.abs(ref.t[: ref.iterations] - w.nocc) > 1e-9 * max(1.0, k / 256)
    assert all(a == b for a, b, d in zip(res.branch, ref.branch, decided) if d), (res.branch, ref.branch)
    assert np.linalg.norm(P - ref.P) / math.sqrt(k) <= ptol
    assert np.abs(P - ref.P).max() <= ptol / 10.0            # every element, not only the norm (measured: 1e-15 .. 3e-14)
    assert abs(res.tr_PH - ref.tr_PH) / abs(ref.tr_PH) <= etol
    assert np.array_equal(P, P.T)
    assert abs(res.eps_min - ref.emin) <= 1e-12 * abs(ref.emin) and abs(res.eps_max - ref.emax) <= 1e-12 * abs(ref.emax)
    n = ref.iterations
    assert np.allclose(res.t, ref.t, rtol=0, atol=1e-9 * k / 256)
    assert np.allclose(res.s, ref.s, rtol=0, atol=1e-9 * k / 256)
    assert np.allclose(res.e[: n - 1], ref.e[: n - 1], rtol=1e-6, atol=1e-11 * k / 256)
    # north_star invariants on the GPU result, and the construction-exact projector (pin P2)
    if ref.converged and projector:          # (a truncated expansion G_m is delivered, but it is not a projector)
        # (inv loosens them for stop rule B, which stops at RelTr 5e-8 -- before P is converged to rounding)
        assert abs(np.trace(P) - w.nocc) <= 1e-9 * inv
        assert np.linalg.norm(P @ P - P) <= 1e-10 * k / 256 * inv
        H = w.H
        assert np.linalg.norm(H @ P - P @ H) <= 1e-10 * k / 256 * inv
        assert np.linalg.norm(P - w.exact_projector()) / math.sqrt(k) <= 1e-10 * inv


def test_expand_config1(handle):
    w = rfoe_inputs.make_workload(1)
    ref = oracle.expand(w.H, w.nocc, tol=w.tol)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, w.tol)
    assert res.status == rfoe.OK and res.iterations == 34
    _check_expansion(w, res, ref)


@pytest.mark.parametrize("c,k", [(1, 100), (2, 333), (3, 200), (4, 450), (5, 129)])
def test_expand_ragged_sizes(handle, c, k):
    w = rfoe_inputs.make_workload(c, k=k)
    ref = oracle.expand(w.H, w.nocc, tol=w.tol)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, w.tol)
    _check_expansion(w, res, ref)


def test_expand_rule_b(handle):
    w = rfoe_inputs.make_workload(2, k=300)
    ref = oracle.expand(w.H, w.nocc, tol=5e-8, stop_rule=oracle.RULE_B)
    handle.configure(stop_rule=rfoe.RULE_B)
    try:
        res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, 5e-8)
    finally:
        handle.configure(stop_rule=rfoe.RULE_A)
    _check_expansion(w, res, ref, inv=1e4)
    assert np.allclose(res.reltr, ref.reltr, rtol=1e-6, atol=1e-13)


def test_expand_bounds_override_and_truncated(handle):
    w = rfoe_inputs.make_workload(1, k=160)
    lo, hi = float(w.lam.min()) - 0.01, float(w.lam.max()) + 0.01
    handle.configure(bounds=(lo, hi))
    try:
        ref = oracle.expand(w.H, w.nocc, tol=w.tol, bounds_override=(lo, hi))
        res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, w.tol)
        _check_expansion(w, res, ref)
        assert res.iterations < 30
        # the MAX_ITER route: m steps of SP2 with an unreachable tolerance is a convergence FAILURE by definition
        handle.configure(max_iter=7)
        ref = oracle.expand(w.H, w.nocc, tol=0.0, max_iter=7, bounds_override=(lo, hi))
        res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, 0.0)
        assert res.status == rfoe.ERR_NOT_CONVERGED and res.iterations == 7 and res.trunc_steps == 0
        _check_expansion(w, res, ref)
        # T-RFOE proper (Eq. 2): RFOE_VARIANT_TRUNC with m steps delivers G_m and reports success
        handle.configure(max_iter=100, trunc_steps=7)
        ref = oracle.expand(w.H, w.nocc, variant=oracle.TRUNC, max_iter=7, bounds_override=(lo, hi))
        res2 = handle.expand(_dev(w.H), w.nocc, rfoe.TRUNC, 0.0)
        assert res2.status == rfoe.OK and res2.converged and res2.iterations == 7 and res2.trunc_steps == 7
        _check_expansion(w, res2, ref, projector=False)
        assert torch.equal(res2.P, res.P)
    finally:
        handle.configure(bounds=False, max_iter=100, trunc_steps=30)


@pytest.mark.parametrize("k", [384, 2048])
def test_truncated_paper_matrix_vs_oracle_and_fermi_dirac(k):
    """T-RFOE as the paper runs it: its synthetic H^p, 85 % of the states occupied, m = 30 steps.
    Against the whole oracle (every element of G_m, same branch string), and against the exact Fermi-Dirac density
    matrix D = [exp(beta (H - mu)) + I]^-1 with (mu, beta) fitted to the occupancies (reading R-TRUNC):
    eps1 at the paper's order (~1e-3), eps2 small."""
    H = rfoe_inputs.paper_matrix(k)
    nocc = round(0.85 * k)
    m_steps = 30
    ref = oracle.expand(H, nocc, variant=oracle.TRUNC, max_iter=m_steps)
    with rfoe.Rfoe(k) as h:
        h.configure(trunc_steps=m_steps)
        res = h.expand(_dev(H), nocc, rfoe.TRUNC, 0.0)
        assert res.status == rfoe.OK and res.iterations == m_steps == res.trunc_steps and res.branch == ref.branch
        G = res.P.cpu().numpy()
        assert np.linalg.norm(G - ref.P) / math.sqrt(k) <= 1e-10 and np.abs(G - ref.P).max() <= 1e-11
        assert abs(res.tr_PH - ref.tr_PH) <= 1e-11 * abs(ref.tr_PH)
        assert np.allclose(res.t, ref.t, rtol=1e-12, atol=0) and np.allclose(res.s, ref.s, rtol=1e-12, atol=0)
        lam, V = np.linalg.eigh(H)
        occ = np.einsum("ij,ij->j", V, G @ V)
        mu, beta = pins.fit_fermi_dirac(lam, occ, 0.5 * (lam[nocc - 1] + lam[nocc]))
        f = pins.fermi_dirac(lam, mu, beta)
        D = (V * f[None, :]) @ V.T
        eps1 = np.linalg.norm(G - D) / np.linalg.norm(D)
        eps2 = abs(res.tr_PH - float(np.sum(f * lam))) / abs(float(np.sum(f * lam)))
        frac = int(np.sum((occ > 1e-3) & (occ < 1 - 1e-3)))
        print(f"T-RFOE k={k} m={m_steps}: beta={beta:.4g} mu={mu:.5f} eps1={eps1:.2e} eps2={eps2:.2e} fractional={frac}")
        assert eps1 <= 5e-3 and eps2 <= 5e-3 and frac >= 3
        # mixed-precision T-RFOE: same m, reduced-precision steps until RelTr <= 5e-4
        h.configure(mixed_head=0.0, mixed_reltr=5e-4)
        mx = h.expand(_dev(H), nocc, rfoe.TRUNC_MIXED, 0.0)
        refm = oracle.expand(H, nocc, variant=oracle.TRUNC_MIXED, max_iter=m_steps, mixed_head=0.0, mixed_reltr=5e-4)
        assert mx.status == rfoe.OK and mx.iterations == m_steps and mx.fp32_steps == refm.fp32_steps >= 5
        assert [c.islower() for c in mx.branch] == [c.islower() for c in refm.branch]
        Gm = mx.P.cpu().numpy()
        e1m = np.linalg.norm(Gm - G) / np.linalg.norm(G)
        e1o = np.linalg.norm(refm.P - ref.P) / np.linalg.norm(ref.P)
        print(f"  mixed: fp32 steps {mx.fp32_steps}, eps1 vs FP64 G_m: kernel {e1m:.2e}, oracle FP32 loop {e1o:.2e}")
        # FP32-level agreement with the FP64 G_m; the kernel's reduced step is not worse than the oracle's plain FP32 loop
        assert e1m <= 1e-4 and e1m <= 3.0 * e1o + 1e-7
        assert np.linalg.norm(Gm - D) / np.linalg.norm(D) <= 5e-3


def test_expand_mcweeny(handle):
    w = rfoe_inputs.make_workload(2, k=260)
    ref = oracle.expand(w.H, w.nocc, variant=oracle.MCWEENY, tol=w.tol)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.MCWEENY, w.tol)
    assert res.mcweeny_steps == ref.mcweeny_steps >= 1 and res.multiplications == ref.multiplications
    _check_expansion(w, res, ref)


def test_expand_accelerated(handle):
    w = rfoe_inputs.make_workload(3, k=256)
    homo, lumo = float(w.lam[: w.nocc].max()), float(w.lam[w.nocc:].min())
    ref = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=w.tol, homo=homo, lumo=lumo)
    handle.configure(homo=homo, lumo=lumo)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2_ACCEL, w.tol)
    _check_expansion(w, res, ref)
    plain = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, w.tol)
    assert res.iterations < plain.iterations
    # estimates outside the spectral bounds are refused on both sides (the scaling factors would leave (0, 2))
    handle.configure(homo=res.eps_min - 1.0, lumo=lumo)
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(_dev(w.H), w.nocc, rfoe.SP2_ACCEL, w.tol)
    assert ei.value.status == rfoe.ERR_INVALID_ARG
    with pytest.raises(RuntimeError):
        oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=w.tol, homo=res.eps_min - 1.0, lumo=lumo)
    handle.configure(homo=homo, lumo=lumo)


@pytest.mark.parametrize("c,k", [(1, 256), (2, 333), (4, 450)])
def test_homo_lumo_from_sp2_history_feed_accelerated(handle, c, k):
    """Z-RFOE, then rfoe_estimate_homo_lumo on its history, then A-Z-RFOE with those estimates (reading R-HL): each side
    uses its own history and its own estimates; estimates, iteration counts and P agree."""
    w = rfoe_inputs.make_workload(c, k=k)
    ref0 = oracle.expand(w.H, w.nocc, tol=w.tol)
    oh, ol = oracle.estimate_homo_lumo(ref0, w.nocc)
    res0 = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, w.tol)
    homo, lumo = handle.estimate_homo_lumo()
    width = res0.eps_max - res0.eps_min
    assert homo == pytest.approx(oh, abs=1e-8 * width) and lumo == pytest.approx(ol, abs=1e-8 * width)
    lam_homo, lam_lumo = float(w.lam[: w.nocc].max()), float(w.lam[w.nocc:].min())
    assert lam_homo - 1e-9 * width <= homo < lumo <= lam_lumo + 1e-9 * width
    ref = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=w.tol, homo=oh, lumo=ol)
    handle.configure(homo=homo, lumo=lumo)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2_ACCEL, w.tol)
    _check_expansion(w, res, ref)
    assert res.iterations < res0.iterations
    with pytest.raises(rfoe.RfoeError) as ei:          # the history of the accelerated run itself is not accepted
        handle.estimate_homo_lumo()
    assert ei.value.status == rfoe.ERR_UNSUPPORTED


def test_expand_host_entry_point(handle):
    w = rfoe_inputs.make_workload(1, k=192)
    ref = oracle.expand(w.H, w.nocc, tol=w.tol)
    res = handle.expand_host(w.H, w.nocc, rfoe.SP2, w.tol)
    _check_expansion(w, res, ref)


def test_expand_config2_full(handle):
    w = rfoe_inputs.make_workload(2)
    ref = oracle.expand(w.H, w.nocc, tol=w.tol)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2, w.tol)
    assert res.iterations == 42
    _check_expansion(w, res, ref)


def test_expand_config2_full_mcweeny_and_accelerated(handle):
    """BASELINE config 2 at its full size (k=2048, nocc=1536) in the other two FP64 variants it names / the paper's best
    performer: McWeeny-style tail (reading R11) and A-Z-RFOE against the whole oracle run."""
    w = rfoe_inputs.make_workload(2)
    H = _dev(w.H)
    ref = oracle.expand(w.H, w.nocc, variant=oracle.MCWEENY, tol=w.tol)
    res = handle.expand(H, w.nocc, rfoe.MCWEENY, w.tol)
    assert res.mcweeny_steps == ref.mcweeny_steps >= 1 and res.multiplications == ref.multiplications
    _check_expansion(w, res, ref)
    homo, lumo = float(w.lam[: w.nocc].max()), float(w.lam[w.nocc:].min())
    ref = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=w.tol, homo=homo, lumo=lumo)
    handle.configure(homo=homo, lumo=lumo)
    res = handle.expand(H, w.nocc, rfoe.SP2_ACCEL, w.tol)
    assert res.iterations <= 24
    _check_expansion(w, res, ref)


# ------------------------------------------------------------------ errors and degenerate inputs
def test_error_paths(handle):
    w = rfoe_inputs.make_workload(1, k=64)
    H = _dev(w.H)
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(H, 0, rfoe.SP2, 1e-12)
    assert ei.value.status == rfoe.ERR_INVALID_ARG
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(H, 64, rfoe.SP2, 1e-12)
    assert ei.value.status == rfoe.ERR_INVALID_ARG
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(H, 10, 17, 1e-12)
    assert ei.value.status == rfoe.ERR_UNSUPPORTED
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(H, 10, rfoe.SP2, 1e-12, P=H)
    assert ei.value.status == rfoe.ERR_INVALID_ARG
    Hbad = H.clone()
    Hbad[3, 5] += 1e-9
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(Hbad, 10, rfoe.SP2, 1e-12)
    assert ei.value.status == rfoe.ERR_NOT_SYMMETRIC
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(torch.eye(8, dtype=torch.float64, device="cuda"), 3, rfoe.SP2, 1e-12)
    assert ei.value.status == rfoe.ERR_BAD_BOUNDS
    with pytest.raises(rfoe.RfoeError) as ei:
        rfoe.Rfoe(64).expand(torch.zeros(65, 65, dtype=torch.float64, device="cuda"), 3)
    assert ei.value.status == rfoe.ERR_INVALID_ARG
    # empty input
    empty = torch.empty((0, 0), dtype=torch.float64, device="cuda")
    for call in (lambda: handle.expand(empty, 1, rfoe.SP2, 1e-12), lambda: handle.bounds(empty), lambda: handle.square(empty)):
        with pytest.raises(rfoe.RfoeError) as ei:
            call()
        assert ei.value.status == rfoe.ERR_INVALID_ARG
    # non-finite input: the bounds are not finite
    Hnan = H.clone()
    Hnan[2, 2] = float("nan")
    with pytest.raises(rfoe.RfoeError) as ei:
        handle.expand(Hnan, 10, rfoe.SP2, 1e-12)
    assert ei.value.status == rfoe.ERR_BAD_BOUNDS        # (the bitwise symmetry check passes: same NaN pattern)
    # the handle is still usable after errors
    res = handle.expand(H, w.nocc, rfoe.SP2, w.tol)
    assert res.converged


# ------------------------------------------------------------------ A8: reduced-precision path (reported separately)
@pytest.mark.parametrize("pair", [True, False])
@pytest.mark.parametrize("k", [1, 5, 128, 130, 257, 777, 1100])
def test_square_reduced_error_bound(handle, k, pair):
    """Three-part (scaled FP16 hi / lo) product with FP32 tensor-core accumulation against the FP64 oracle product.  Bound:
    dropped Zl Zl term and 11-bit rounding of Zl: 3 * 2^-22 per product; FP32 accumulation in tensor memory, one
    truncation per 8-wide MMA block plus the in-block tree, over chunks of 256: (k/8 + 8) * 2^-23 bounds it,
    all relative to sum_l |z_il||z_lj| with Z = X - (Tr X / k) I.  Both forms of the kernel: CTA pairs (tcgen05.mma.cta_group::2,
    the default) and one CTA per tile (RFOE_OPT_REDUCED_PAIR = 0); sizes with an odd number of tiles per row end in a phantom tile."""
    X = _sym(k, 100 + k, scale=1.0 / math.sqrt(k))
    handle.configure(reduced_pair=pair)
    try:
        out, sc, ms = handle.square(_dev(X), -1.0, 2.0, 0.0, reduced=True)
    finally:
        handle.configure(reduced_pair=True)
    out = out.cpu().numpy()
    Y = oracle.square(X)
    Z = X - np.trace(X) / k * np.eye(k)
    S = np.abs(Z) @ np.abs(Z)
    bound = (3 * 2.0 ** -22 + (k / 8 + 8) * 2.0 ** -23) * S + 4 * EPS * np.abs(2 * X - Y)
    assert np.all(np.abs(out - (2.0 * X - Y)) <= bound)
    assert np.array_equal(out, out.T)
    assert sc[0] == pytest.approx(np.trace(out), rel=1e-12, abs=1e-13)       # scalars describe the matrix written
    assert sc[1] == pytest.approx(np.sum(out * out), rel=1e-12)
    assert sc[3] == pytest.approx(np.trace(Y), rel=1e-4)


@pytest.mark.parametrize("c,k", [(3, 256), (3, 640), (2, 333), (4, 450)])
def test_expand_mixed(handle, c, k):
    """Mixed variant with the FP64 head (R-MIX): north_star's reduced-precision tolerances 1e-6 / 1e-8 and
    identical iteration counts against the oracle's FP32 steps; FP32 steps occupy the same positions."""
    w = rfoe_inputs.make_workload(c, k=k)
    head = w.nocc / 512.0      # FP32 phase starts late enough for the ORACLE's own FP32 noise to stay below 1e-6
    ref = oracle.expand(w.H, w.nocc, variant=oracle.SP2_MIXED, tol=w.tol, mixed_head=head, mixed_reltr=5e-4)
    handle.configure(mixed_head=head, mixed_reltr=5e-4)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2_MIXED, w.tol)
    P = res.P.cpu().numpy()
    assert res.converged and ref.converged
    assert res.iterations == ref.iterations
    assert res.fp32_steps == ref.fp32_steps >= 2
    assert [ch.islower() for ch in res.branch] == [ch.islower() for ch in ref.branch]
    dP = np.linalg.norm(P - ref.P) / math.sqrt(k)
    dE = abs(res.tr_PH - ref.tr_PH) / abs(ref.tr_PH)
    print(f"mixed c={c} k={k}: fp32 steps {res.fp32_steps}/{res.iterations} dP={dP:.2e} dE={dE:.2e} "
          f"errP_exact={np.linalg.norm(P - w.exact_projector()) / math.sqrt(k):.2e}")
    assert dP <= 1e-6 and dE <= 1e-8
    assert np.array_equal(P, P.T)
    assert abs(np.trace(P) - w.nocc) <= 1e-9
    assert np.linalg.norm(P @ P - P) <= 1e-10 * max(1.0, k / 256)


def test_expand_mixed_single_cta_form_agrees(handle):
    """RFOE_OPT_REDUCED_PAIR = 0 (one CTA per tile, the round-1 kernel) against the default CTA-pair kernel: the same products
    in the same order per FP32 sum (the two differ in the last bits of those sums: 3e-12 on one squaring), so the whole
    mixed expansion takes the same decisions, and the two P differ by less than the reduced-precision path's own 1e-6
    (measured 3e-8: the recursion amplifies last-bit differences of the reduced steps up to their noise floor)."""
    w = rfoe_inputs.make_workload(3, k=640)
    handle.configure(mixed_head=0.0, mixed_reltr=5e-4)
    Hd = _dev(w.H)
    a = handle.expand(Hd, w.nocc, rfoe.SP2_MIXED, w.tol)
    handle.configure(reduced_pair=False)
    try:
        b = handle.expand(Hd, w.nocc, rfoe.SP2_MIXED, w.tol)
    finally:
        handle.configure(reduced_pair=True)
    assert a.converged and b.converged and a.iterations == b.iterations and a.fp32_steps == b.fp32_steps >= 2
    assert a.branch == b.branch
    assert (a.P - b.P).abs().max().item() <= 1e-6
    assert np.allclose(a.t, b.t, rtol=0, atol=1e-5) and torch.equal(b.P, b.P.T)
    Pex = _dev(w.exact_projector())
    for r in (a, b):
        assert torch.linalg.norm(r.P - Pex).item() / math.sqrt(640) <= 1e-6


def test_expand_mixed_paper_schedule(handle):
    """Paper's own schedule (FP32 from the first step until RelTr <= 5e-4): converges to a
    projector with tr P = nocc; accuracy is FP32-limited (paper: eps1 ~ 1e-7 on its matrix), reported, not 1e-6."""
    w = rfoe_inputs.make_workload(3, k=512)
    handle.configure(mixed_head=0.0, mixed_reltr=5e-4)
    res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2_MIXED, w.tol)
    ref = oracle.expand(w.H, w.nocc, variant=oracle.SP2_MIXED, tol=w.tol, mixed_head=0.0, mixed_reltr=5e-4)
    P = res.P.cpu().numpy()
    assert res.converged and res.iterations == ref.iterations and res.fp32_steps == ref.fp32_steps
    assert abs(np.trace(P) - w.nocc) <= 1e-9
    err = np.linalg.norm(P - w.exact_projector()) / math.sqrt(w.k)
    err_oracle = np.linalg.norm(ref.P - w.exact_projector()) / math.sqrt(w.k)
    print(f"paper schedule k={w.k}: errP kernel {err:.2e}, oracle FP32 loop {err_oracle:.2e}, fp32 steps {res.fp32_steps}")
    # the oracle's plain FP32 loop on the same input sets the scale (a few 1e-5 here, R-MIX): the kernel's reduced step
    # (FP16 parts, exact products) must not be worse than it, and both stay FP32-sized
    assert err <= 1.5 * err_oracle + 1e-7 and err <= 2e-4
    assert abs(res.tr_PH - w.band_energy()) / abs(w.band_energy()) <= 1e-7


def test_expand_mixed_paper_matrix_eps1():
    """mixed-precision Z-RFOE reaches eps1 ~ 1e-7, eps2 ~ 1e-9 on the paper's matrix (PAPER.md:86,
    N_occ = 0.9 k) with FP32 steps until RelTr <= 5e-4.  Stop rule A here, so that the FP32 damage is not hidden behind
    the RelTr 5e-8 stop; D_ref from an eigendecomposition, as in the paper."""
    k = 1024
    H = rfoe_inputs.paper_matrix(k)
    nocc = round(0.9 * k)
    lam, V = np.linalg.eigh(H)
    Dref = V[:, :nocc] @ V[:, :nocc].T
    eband = float(lam[:nocc].sum())
    with rfoe.Rfoe(k) as h:
        h.configure(mixed_head=0.0, mixed_reltr=5e-4)
        r64 = h.expand(_dev(H), nocc, rfoe.SP2, 4e-12)
        mx = h.expand(_dev(H), nocc, rfoe.SP2_MIXED, 4e-12)
    assert r64.converged and mx.converged and mx.fp32_steps >= 10
    e64 = np.linalg.norm(r64.P.cpu().numpy() - Dref) / math.sqrt(nocc)
    e1 = np.linalg.norm(mx.P.cpu().numpy() - Dref) / math.sqrt(nocc)
    e2 = abs(mx.tr_PH - eband) / abs(eband)
    print(f"paper matrix k={k}: eps1 fp64 {e64:.2e}, mixed {e1:.2e}, eps2 mixed {e2:.2e}, fp32 steps {mx.fp32_steps}/{mx.iterations}")
    assert e64 <= 1e-9
    assert e1 <= 2e-6 and e2 <= 1e-8          # paper: ~1e-7 / ~1e-9; a regression of the reduced kernel by 10x fails this


def test_probe_fp64_peak(handle):
    """rfoe_probe_fp64_peak: register-only DMMA issue loop; B200's FP64 tensor pipe is 128 flop/clk/SM (37.2 TFLOP/s at
    1965 MHz on 148 SMs), and no clock this part runs at takes it below 20."""
    tf = handle.probe_fp64_peak(50.0)
    print(f"FP64 DMMA issue-rate probe: {tf:.2f} TFLOP/s")
    assert 20.0 < tf < 40.0


def test_expand_mixed_truncated(handle):
    """Mixed T-RFOE: the truncated expansion G_m with reduced-precision steps; fractional
    occupancies, so the comparison with the oracle's FP32 loop is entry-wise at FP32 level, scalars likewise."""
    w = rfoe_inputs.make_workload(1, k=192)
    lo, hi = float(w.lam.min()) - 0.01, float(w.lam.max()) + 0.01
    handle.configure(bounds=(lo, hi), max_iter=9, mixed_head=0.0, mixed_reltr=0.0)
    try:
        ref = oracle.expand(w.H, w.nocc, variant=oracle.SP2_MIXED, tol=0.0, max_iter=9, bounds_override=(lo, hi),
                            mixed_head=0.0, mixed_reltr=0.0)
        res = handle.expand(_dev(w.H), w.nocc, rfoe.SP2_MIXED, 0.0)
    finally:
        handle.configure(bounds=False, max_iter=100, mixed_reltr=5e-4)
    assert res.status == rfoe.ERR_NOT_CONVERGED and res.iterations == ref.iterations == 9
    assert res.fp32_steps == ref.fp32_steps == 9 and res.branch == ref.branch
    P = res.P.cpu().numpy()
    assert np.abs(P - ref.P).max() <= 2e-5
    assert np.allclose(res.t, ref.t, rtol=0, atol=1e-3) and np.array_equal(P, P.T)


# ------------------------------------------------------------------ tiny and degenerate problems
@pytest.mark.parametrize("k,nocc", [(2, 1), (3, 1), (3, 2), (5, 4)])
def test_expand_tiny(handle, k, nocc):
    rng = np.random.default_rng(900 + 10 * k + nocc)
    A = rng.standard_normal((k, k))
    H = np.ascontiguousarray(0.5 * (A + A.T)) + np.diag(np.arange(k, dtype=np.float64))
    ref = oracle.expand(H, nocc, tol=1e-12)
    res = handle.expand(_dev(H), nocc, rfoe.SP2, 1e-12)
    assert res.converged and ref.converged and res.iterations == ref.iterations
    P = res.P.cpu().numpy()
    Pref, _ = pins.jacobi_projector(H, nocc)
    assert np.abs(P - ref.P).max() <= 1e-13 and np.abs(P - Pref).max() <= 1e-12
    assert abs(np.trace(P) - nocc) <= 1e-12


def test_expand_degenerate_fermi_level(handle):
    """No gap at the Fermi level: the eigenvalue pair straddling N_occ is degenerate, theta(mu I - H) is not a
    projector of rank N_occ and the recursion cannot converge -- both sides must say so in the same way
    (max_iter steps, NOT_CONVERGED, last iterate returned, the degenerate pair left at fractional occupation)."""
    k, nocc = 64, 20
    rng = np.random.default_rng(77)
    Q, _ = np.linalg.qr(rng.standard_normal((k, k)))
    lam = np.sort(rng.uniform(-1.0, 1.0, size=k))
    lam[nocc] = lam[nocc - 1]                                  # HOMO == LUMO
    H = (Q * lam[None, :]) @ Q.T
    H = np.ascontiguousarray(0.5 * (H + H.T))
    handle.configure(max_iter=60)
    try:
        ref = oracle.expand(H, nocc, tol=1e-12, max_iter=60)
        res = handle.expand(_dev(H), nocc, rfoe.SP2, 1e-12)
    finally:
        handle.configure(max_iter=100)
    assert not ref.converged and not res.converged and res.status == rfoe.ERR_NOT_CONVERGED
    assert res.iterations == ref.iterations == 60
    P = res.P.cpu().numpy()
    occ = np.sort(np.linalg.eigvalsh(P))
    assert np.sum((occ > 0.01) & (occ < 0.99)) >= 1            # fractional occupation survives
    assert np.allclose(res.t[:20], ref.t[:20], rtol=0, atol=1e-8)   # the trace-steered map is chaotic here: compare the head only


def test_run_to_run_bitwise(handle):
    """No FP atomics, fixed-order reductions: two runs give the same bits (P, traces, branch string), for the
    FP64 path and for the reduced-precision path."""
    w = rfoe_inputs.make_workload(4, k=515)
    H = _dev(w.H)
    for variant in (rfoe.SP2, rfoe.SP2_MIXED):
        a = handle.expand(H, w.nocc, variant, w.tol)
        Pa, ta, sa, ba = a.P.clone(), a.t.copy(), a.s.copy(), a.branch
        b = handle.expand(H, w.nocc, variant, w.tol)
        assert torch.equal(Pa, b.P) and np.array_equal(ta, b.t) and np.array_equal(sa, b.s) and ba == b.branch
        assert a.tr_PH == b.tr_PH
