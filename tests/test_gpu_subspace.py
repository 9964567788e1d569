"""GPU parity of the steps either side of the expansion against the CPU oracle, through
the C ABI: rfoe_project (Rayleigh-Ritz), rfoe_apply (Y = P Psi) and the density.
Tolerances: one product adds the same L products per element in a different association
(DMMA groups of 4, fused; K-slices) -> |dC| <= 4 L eps max|a| max|b|; bit-exact on small-integer inputs."""
import math

import numpy as np
import pytest
import torch

import oracle  # noqa: F401
import paper_2301_04642_b200 as rfoe
import rfoe_inputs

pytestmark = pytest.mark.gpu
EPS = 2.0 ** -52


@pytest.fixture(scope="module")
def handle():
    with rfoe.Rfoe(1024, device=0) as h:
        yield h


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("k,M", [(1, 2), (5, 18), (128, 512), (129, 1000), (200, 4098), (333, 20002), (640, 70000)])
def test_project_matches_oracle(handle, k, M):
    rng = np.random.default_rng(k * 7 + M)
    Psi, Phi = rng.standard_normal((k, M)), rng.standard_normal((k, M))
    ref = oracle.project(Psi, Phi)
    Hp, (tr, ss), ms = handle.project(_dev(Psi), _dev(Phi))
    Hp = Hp.cpu().numpy()
    assert np.array_equal(Hp, Hp.T)                                   # bitwise symmetric
    bound = 4 * M * EPS * np.abs(Psi).max() * np.abs(Phi).max()
    assert np.abs(Hp - ref).max() <= bound
    assert abs(tr - np.trace(ref)) <= 1e-12 * max(1.0, np.abs(np.diag(ref)).sum())
    assert abs(ss - (ref * ref).sum()) <= 1e-12 * (ref * ref).sum()


def test_project_exact_on_small_integers_and_pitched_rows(handle):
    rng = np.random.default_rng(3)
    k, M, ld = 130, 3001, 3008                                         # ragged M, padded row pitch
    Psi = rng.integers(-4, 5, size=(k, M)).astype(np.float64)
    Phi = rng.integers(-4, 5, size=(k, M)).astype(np.float64)
    bufA = torch.full((k, ld), 7.0, dtype=torch.float64, device="cuda")   # garbage in the pitch padding must be ignored
    bufB = torch.full((k, ld), -3.0, dtype=torch.float64, device="cuda")
    bufA[:, :M] = _dev(Psi)
    bufB[:, :M] = _dev(Phi)
    Hp, _, _ = handle.project(bufA[:, :M], bufB[:, :M])
    ref = oracle.project(Psi, Phi)
    assert np.array_equal(Hp.cpu().numpy(), ref)                       # all partial sums exact: any order agrees


@pytest.mark.parametrize("k,M", [(1, 2), (5, 18), (128, 512), (129, 1000), (200, 4098), (333, 2050), (640, 1538)])
def test_apply_and_density_match_oracle(handle, k, M):
    rng = np.random.default_rng(k * 11 + M)
    P = rng.standard_normal((k, k))
    P = 0.5 * (P + P.T)
    Psi = rng.standard_normal((k, M))
    Yr = oracle.apply(P, Psi)
    rr = oracle.density(Psi, Yr)
    Y, rho, ms = handle.apply(_dev(P), _dev(Psi))
    Y, rho = Y.cpu().numpy(), rho.cpu().numpy()
    bound = 4 * k * EPS * np.abs(P).max() * np.abs(Psi).max()
    assert np.abs(Y - Yr).max() <= bound
    assert np.abs(rho - rr).max() <= 4 * k * EPS * np.abs(Psi).max() * np.abs(Yr).max() + k * bound * np.abs(Psi).max()


def test_apply_exact_on_small_integers_nonsymmetric_P_and_pitched_output(handle):
    """Integer inputs make every sum exact, so the result must equal the oracle bit for bit whatever the
    contraction order; a non-symmetric P catches a transposed operand; Y has a padded pitch and an odd M."""
    rng = np.random.default_rng(9)
    k, M = 257, 1027
    P = rng.integers(-3, 4, size=(k, k)).astype(np.float64)
    Psi = rng.integers(-3, 4, size=(k, M)).astype(np.float64)
    PsiD = torch.zeros((k, M + 1), dtype=torch.float64, device="cuda")
    PsiD[:, :M] = _dev(Psi)
    Ybuf = torch.full((k, M + 5), 99.0, dtype=torch.float64, device="cuda")
    Y, rho, _ = handle.apply(_dev(P), PsiD[:, :M], out=Ybuf[:, :M])
    Yr = oracle.apply(P, Psi)
    assert np.array_equal(Y.cpu().numpy(), Yr)
    assert np.array_equal(rho.cpu().numpy(), oracle.density(Psi, Yr))
    assert bool((Ybuf[:, M:] == 99.0).all())                            # nothing written past column M


def test_pipeline_project_expand_apply_matches_oracle_and_exact_density(handle):
    """The whole chain through the C ABI on a synthetic Rayleigh-Ritz input (config 2 scaled to k=333, M=6002):
    same iteration count as the oracle chain, P / Y / rho within the north_star tolerances, electron count."""
    sub = rfoe_inputs.make_subspace(2, k=333, M=6002)
    w = sub.w
    Hp_o = oracle.project(sub.Psi, sub.HPsi)
    ro = oracle.expand(Hp_o, w.nocc, tol=w.tol)
    Yo = oracle.apply(ro.P, sub.Psi)
    rho_o = oracle.density(sub.Psi, Yo)
    Psi_d, HPsi_d = _dev(sub.Psi), _dev(sub.HPsi)
    Hp, _, _ = handle.project(Psi_d, HPsi_d)
    res = handle.expand(Hp, w.nocc, rfoe.SP2, w.tol)
    Y, rho, _ = handle.apply(res.P, Psi_d)
    assert res.converged and res.iterations == ro.iterations
    k = w.k
    assert np.linalg.norm(res.P.cpu().numpy() - ro.P) / math.sqrt(k) <= 1e-10
    assert abs(res.tr_PH - ro.tr_PH) / abs(ro.tr_PH) <= 1e-11
    assert np.abs(Y.cpu().numpy() - Yo).max() <= 1e-10
    rho = rho.cpu().numpy()
    assert np.abs(rho - rho_o).max() <= 1e-12
    assert abs(rho.sum() - w.nocc) <= 1e-9                                # electron count
    # construction-exact density: rows of Psi rotated by the generator's own occupied eigenvectors
    Qo = np.asarray(w.Q)[:, : w.nocc]
    rho_exact = ((Qo.T @ sub.Psi) ** 2).sum(axis=0)
    assert np.abs(rho - rho_exact).max() <= 1e-11


def test_bad_arguments(handle):
    Psi = torch.zeros((8, 31), dtype=torch.float64, device="cuda")      # odd pitch: TMA needs 16-byte rows
    with pytest.raises(rfoe.RfoeError) as e:
        handle.project(Psi, Psi.clone())
    assert e.value.status == rfoe.ERR_INVALID_ARG
    big = torch.zeros((2048, 4), dtype=torch.float64, device="cuda")    # k > k_max
    with pytest.raises(rfoe.RfoeError):
        handle.project(big, big.clone())


def _dot_by_definition(a, b):
    """sum_l a_l b_l, l ascending, one IEEE product and one IEEE sum at a time (Python floats)."""
    acc = 0.0
    for x, y in zip(a.tolist(), b.tolist()):
        acc = acc + x * y
    return acc


def test_fullsize_chain_bench_configuration():
    """The workload bench.py's `subspace_steps` times (config 4 spectrum at k=4096, nocc=3150, M=600000; the launch
    configuration is the same: 528 tiles x 7 K-slices, 32 x 4688 apply tiles).  The naive oracle cannot run 2 M k^2
    flops here, so: sampled entries of H^p and Y computed one by one by the definition (every tile class, the
    ragged last column block, mirrored entries), and properties that hold at any size -- H^p equals the
    generator's target matrix, bitwise symmetry, electron count, the construction-exact density."""
    k, M = 4096, 600000
    sub = rfoe_inputs.make_subspace(4, k=k, M=M, device="cuda")
    w = sub.w
    rng = np.random.default_rng(44)
    with rfoe.Rfoe(k) as h:
        Hp, (tr, ss), _ = h.project(sub.Psi, sub.HPsi)
        assert torch.equal(Hp, Hp.T)
        Hw = w.H if isinstance(w.H, torch.Tensor) else torch.from_numpy(w.H).cuda()
        assert float((Hp - Hw).abs().max()) <= 1e-13                 # Psi HPsi^T = target H^p by construction
        assert tr == pytest.approx(float(w.lam.sum()), abs=1e-9)
        pairs = [(0, 0), (k - 1, k - 1), (0, k - 1), (k - 1, 0), (130, 129), (129, 130), (2047, 2048), (4000, 77)]
        pairs += [tuple(rng.integers(0, k, size=2).tolist()) for _ in range(6)]
        amax = float(sub.Psi.abs().max()) * float(sub.HPsi.abs().max())
        for i, j in pairs:
            a, b = min(i, j), max(i, j)                              # the upper triangle is the definition
            ref = _dot_by_definition(sub.Psi[a].cpu().numpy(), sub.HPsi[b].cpu().numpy())
            assert abs(Hp[i, j].item() - ref) <= 4 * M * EPS * amax
        res = h.expand(Hp, w.nocc, rfoe.SP2, w.tol)
        assert res.converged
        Y, rho, _ = h.apply(res.P, sub.Psi)
        Pn = res.P.cpu().numpy()
        cols = [0, 1, 127, 128, M - 1, M - 2, M - 64, 599936, 599935] + rng.integers(0, M, size=6).tolist()
        rows = [0, k - 1, 128, 127, 2049] + rng.integers(0, k, size=4).tolist()
        pmax = float(np.abs(Pn).max()) * float(sub.Psi.abs().max())
        for m_ in cols:
            col = sub.Psi[:, m_].cpu().numpy()
            for i in rows:
                assert abs(Y[i, m_].item() - _dot_by_definition(Pn[i], col)) <= 4 * k * EPS * pmax
            ycol = Y[:, m_].cpu().numpy()
            assert abs(rho[m_].item() - _dot_by_definition(col, ycol)) <= 4 * k * EPS * float(np.abs(col).max() * np.abs(ycol).max())
        assert abs(float(rho.sum()) - w.nocc) <= 1e-8                  # electron count
        Qo = w.Q[:, : w.nocc] if isinstance(w.Q, torch.Tensor) else torch.from_numpy(w.Q[:, : w.nocc]).cuda()
        rho_exact = ((Qo.T @ sub.Psi) ** 2).sum(dim=0)
        assert float((rho - rho_exact).abs().max()) <= 1e-12


def test_project_apply_lanczos_are_bitwise_reproducible(handle):
    """No FP atomics anywhere: K-slices, density slices and the Lanczos sums are added in a fixed order."""
    rng = np.random.default_rng(77)
    k, M = 640, 20002
    Psi, Phi = _dev(rng.standard_normal((k, M))), _dev(rng.standard_normal((k, M)))
    P = rng.standard_normal((k, k))
    P = _dev(0.5 * (P + P.T))
    a = handle.project(Psi, Phi)[0].clone()
    ya, ra, _ = handle.apply(P, Psi)
    ya, ra = ya.clone(), ra.clone()
    la = handle.bounds_lanczos(P, 24)
    for _ in range(3):
        assert torch.equal(handle.project(Psi, Phi)[0], a)
        yb, rb, _ = handle.apply(P, Psi)
        assert torch.equal(yb, ya) and torch.equal(rb, ra)
        assert handle.bounds_lanczos(P, 24) == la
