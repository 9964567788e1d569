"""GPU parity at BASELINE.json's full sizes, in the configuration bench.py times (rfoe_expand, SP2, rule A,
Gershgorin bounds).  The naive oracle cannot run a whole expansion here (2 k^3 x 56 steps), so:
  * the O(k^2) oracle steps run in full: Gershgorin bounds, affine map, Tr X0, ||X0||_F^2 (A1, A2);
  * one squaring (A4 + A5) is checked on sampled outputs the oracle computes one by one (definition,
    l ascending) in every tile class: diagonal tiles, off-diagonal tiles, mirrored entries, last tile;
  * the whole expansion is checked through properties that hold at any size: the construction-exact
    projector Q_occ Q_occ^T (pin P2), tr P = nocc, idempotency, bitwise symmetry, band energy =
    sum of the occupied eigenvalues, and the scalar eigenvalue-space model (pin P5) for the iteration
    count and the branch string.
torch is used for the harness-side algebra only (building Q_occ Q_occ^T, norms)."""
import math
import os

import numpy as np
import pytest

import oracle
import rfoe_inputs
from tests import pins

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2301_04642_b200 as rfoe  # noqa: E402

EPS = 2.0 ** -52


def _sample_pairs(k, rng, n_each=6):
    m = (k + 127) // 128
    pairs = []
    for _ in range(n_each):
        I, J = sorted(rng.integers(0, m, size=2).tolist())
        i = min(k - 1, I * 128 + int(rng.integers(0, 128)))
        j = min(k - 1, J * 128 + int(rng.integers(0, 128)))
        pairs += [(i, j), (j, i)]                       # an entry and its mirror
        d = min(k - 1, I * 128 + int(rng.integers(0, 128)))
        pairs += [(d, d), (d, min(k - 1, d + 1))]       # inside a diagonal tile
    pairs += [(0, 0), (k - 1, k - 1), (0, k - 1), (k - 1, 0), (k - 2, k - 1)]
    return pairs


def _run_fullsize(c):
    w = rfoe_inputs.make_workload(c, device="cuda")
    k, nocc = w.k, w.nocc
    H = w.H
    Hn = H.cpu().numpy()
    with rfoe.Rfoe(k) as h:
        # ---- A1/A2 against the full oracle (O(k^2))
        lo, hi = h.bounds(H)
        olo, ohi = oracle.bounds(Hn)
        assert abs(lo - olo) <= 4 * k * EPS * abs(olo) and abs(hi - ohi) <= 4 * k * EPS * abs(ohi)
        X0 = oracle.affine(Hn, olo, ohi)
        t0, s0 = oracle.trace(X0), oracle.sumsq(X0)
        # ---- A4/A5: one squaring of X0 at full size, sampled entries by the definition
        Xd = torch.from_numpy(X0).cuda()
        out, sc, ms = h.square(Xd, -1.0, 2.0, 0.0)                                     # the L branch: 2X - X^2
        del Xd
        pairs = _sample_pairs(k, np.random.default_rng(c))
        y = oracle.square_entries(X0, pairs)
        got = np.array([out[i, j].item() for i, j in pairs])
        x = np.array([X0[i, j] for i, j in pairs])
        xmax = float(np.abs(X0).max())
        assert np.abs(got - (2.0 * x - y)).max() <= 8 * k * EPS * xmax * xmax + 4 * EPS * np.abs(x).max()
        assert torch.equal(out, out.T)
        assert sc[3] == pytest.approx(s0, rel=1e-12)                                   # Tr X^2 = ||X||_F^2
        assert sc[0] == pytest.approx(2.0 * t0 - s0, rel=1e-12)
        del out
        # ---- the expansion bench.py times
        res = h.expand(H, nocc, rfoe.SP2, w.tol)
    assert res.status == rfoe.OK and res.converged
    assert res.t[0] == pytest.approx(t0, rel=1e-13) and res.s[0] == pytest.approx(s0, rel=1e-12)
    model = pins.scalar_sp2(w.lam, nocc, res.eps_min, res.eps_max, tol=w.tol)
    assert res.iterations == model["iterations"]
    decided = np.abs(model["t"][: res.iterations] - nocc) > 1e-9 * k / 256
    assert all(a == b for a, b, d in zip(res.branch, model["branch"], decided) if d), (res.branch, model["branch"])
    assert np.allclose(res.t, model["t"], rtol=0, atol=1e-8 * k / 256)
    P = res.P
    assert torch.equal(P, P.T)
    assert abs(torch.diagonal(P).sum().item() - nocc) <= 1e-8
    Qo = w.Q[:, :nocc]
    Pex = Qo @ Qo.T
    dP = torch.linalg.norm(P - Pex).item() / math.sqrt(k)
    del Pex, Qo
    assert dP <= 1e-10, dP
    idem = torch.linalg.norm(P @ P - P).item()
    assert idem <= 1e-10 * k / 256, idem
    comm = torch.linalg.norm(H @ P - P @ H).item()
    assert comm <= 1e-10 * k / 256, comm
    assert abs(res.tr_PH - w.band_energy()) / abs(w.band_energy()) <= 1e-11
    return dict(k=k, iterations=res.iterations, dP=dP, idem=idem, comm=comm, device_ms=res.device_ms,
                square_ms=res.square_ms, branch=res.branch)


def test_fullsize_config3():
    r = _run_fullsize(3)
    print(r)


def test_fullsize_config4_headline():
    r = _run_fullsize(4)
    assert r["iterations"] == 56
    print(r)


def test_fullsize_config5():
    r = _run_fullsize(5)
    print(r)
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/config5.txt", "w") as f:
        f.write(repr(r) + "\n")


@pytest.mark.slow
@pytest.mark.parametrize("variant", ["sp2", "accel"])
@pytest.mark.parametrize("c", [3] + ([4] if os.environ.get("RFOE_FULL_ORACLE_16384") == "1" else []))
def test_full_oracle_expansion_every_element(c, variant):
    """"run the full oracle once for k=8192 and 16384 (budget it)".  The WHOLE naive oracle expansion
    (2 k^3 per squaring, host cores, minutes to hours) against the GPU expansion on the same bytes: every element of P,
    the iteration count, the branch string, the band energy and the per-step history, at the north_star tolerances.
    k=16384 only with RFOE_FULL_ORACLE_16384=1 (about two hours of host time)."""
    import time

    w = rfoe_inputs.make_workload(c, device="cuda")
    k, nocc = w.k, w.nocc
    Hn = w.H.cpu().numpy()
    accel = variant == "accel"          # A-Z-RFOE with the generator's HOMO / LUMO: about half the squarings
    homo, lumo = float(w.lam[:nocc].max()), float(w.lam[nocc:].min())
    with rfoe.Rfoe(k) as h:
        if accel:
            h.configure(homo=homo, lumo=lumo)
        res = h.expand(w.H, nocc, rfoe.SP2_ACCEL if accel else rfoe.SP2, w.tol)
    P = res.P.cpu().numpy()
    del res.P
    w.H = w.Q = None
    torch.cuda.empty_cache()
    t0 = time.perf_counter()
    if accel:
        ref = oracle.expand(Hn, nocc, variant=oracle.SP2_ACCEL, tol=w.tol, homo=homo, lumo=lumo)
    else:
        ref = oracle.expand(Hn, nocc, tol=w.tol)
    oracle_s = time.perf_counter() - t0
    assert ref.converged and res.converged and res.iterations == ref.iterations
    decided = np.abs(ref.t[: ref.iterations] - nocc) > 1e-9 * k / 256
    assert all(a == b for a, b, d in zip(res.branch, ref.branch, decided) if d), (res.branch, ref.branch)
    dP = float(np.linalg.norm(P - ref.P) / math.sqrt(k))
    dmax = float(np.abs(P - ref.P).max())
    dE = abs(res.tr_PH - ref.tr_PH) / abs(ref.tr_PH)
    assert dP <= 1e-10 and dE <= 1e-11, (dP, dE)
    assert res.eps_min == pytest.approx(ref.emin, rel=1e-13) and res.eps_max == pytest.approx(ref.emax, rel=1e-13)
    assert np.allclose(res.t, ref.t, rtol=0, atol=1e-8 * k / 256)
    assert np.allclose(res.s, ref.s, rtol=0, atol=1e-8 * k / 256)
    live = ref.e > 1e3 * EPS * k                       # above the rounding floor of e_n
    assert np.allclose(res.e[live], ref.e[live], rtol=1e-6)
    out = dict(config=c, variant=variant, k=k, iterations=ref.iterations, branch=ref.branch, dP=dP, max_abs_dP=dmax, dE=dE,
               oracle_seconds=oracle_s, oracle_threads=os.cpu_count(), gpu_ms=res.device_ms,
               oracle_tflops=ref.iterations * float(k) * k * (k + 1) / oracle_s / 1e12)
    print(out)
    os.makedirs("gpurun_out", exist_ok=True)
    with open(f"gpurun_out/full_oracle_config{c}_{variant}.txt", "w") as f:
        f.write(repr(out) + "\n")


@pytest.mark.parametrize("m", [3])
def test_headline_size_first_steps_every_element(m):
    """k=16384 (config 4, the size bench.py times): the whole naive oracle expansion would take hours of host time, so the
    first m recursion steps are run on both sides (RFOE_VARIANT_TRUNC with m steps) and EVERY element of
    X_m is compared, with the scalars of every step; both SP2 branches occur in these steps (`LLS...`).  m = 3 runs in the
    default suite (about 130 s of oracle per step on 16 host threads; round 1 ran m = 5: profiles/r01g_oracle_runs.md)."""
    import time

    w = rfoe_inputs.make_workload(4, device="cuda")
    k, nocc = w.k, w.nocc
    Hn = w.H.cpu().numpy()
    with rfoe.Rfoe(k) as h:
        h.configure(trunc_steps=m)
        res = h.expand(w.H, nocc, rfoe.TRUNC, 0.0)
    assert res.status == rfoe.OK and res.iterations == m
    X = res.P.cpu().numpy()
    del res.P
    w.H = w.Q = None
    torch.cuda.empty_cache()
    t0 = time.perf_counter()
    ref = oracle.expand(Hn, nocc, variant=oracle.TRUNC, max_iter=m)
    oracle_s = time.perf_counter() - t0
    assert ref.iterations == m and res.branch == ref.branch and len(set(ref.branch)) == 2
    xmax = float(np.abs(ref.P).max())
    dmax = float(np.abs(X - ref.P).max())
    dF = float(np.linalg.norm(X - ref.P) / math.sqrt(k))
    # m products of k terms each, errors carried through x^2 / 2x - x^2 (derivative <= 2): a generous rounding bound
    assert dmax <= (2.0 ** m) * 8 * k * EPS * xmax, (dmax, xmax)
    assert dF <= 1e-10
    assert np.allclose(res.t, ref.t, rtol=1e-12, atol=0) and np.allclose(res.s, ref.s, rtol=1e-12, atol=0)
    assert np.allclose(res.e, ref.e, rtol=1e-9, atol=0)
    assert abs(res.tr_PH - ref.tr_PH) <= 1e-11 * abs(ref.tr_PH)
    out = dict(k=k, steps=m, branch=ref.branch, max_abs_diff=dmax, frob_diff_per_sqrt_k=dF, oracle_seconds=oracle_s,
               oracle_seconds_per_squaring=oracle_s / m, oracle_threads=os.cpu_count(), gpu_ms=res.device_ms)
    print(out)
    os.makedirs("gpurun_out", exist_ok=True)
    with open(f"gpurun_out/first_steps_k16384_m{m}.txt", "w") as f:
        f.write(repr(out) + "\n")


def _run_fullsize_mixed(c):
    """Reduced-precision path (A8) at full size with the paper's schedule (FP32 steps from the start until
    RelTr <= 5e-4).  The oracle's FP32 loop cannot run here; properties that hold at any
    size: north_star's reduced-precision tolerances against the construction-exact projector (1e-6) and the
    exact band energy (1e-8), the FP64 path's iteration count and branch string, tr P = nocc, idempotency."""
    w = rfoe_inputs.make_workload(c, device="cuda")
    k, nocc = w.k, w.nocc
    Qo = w.Q[:, :nocc]
    Pex = Qo @ Qo.T
    del Qo
    with rfoe.Rfoe(k) as h:
        r64 = h.expand(w.H, nocc, rfoe.SP2, w.tol)
        its64, br64, ms64 = r64.iterations, r64.branch, r64.device_ms
        del r64
        h.configure(mixed_head=0.0, mixed_reltr=5e-4)
        res = h.expand(w.H, nocc, rfoe.SP2_MIXED, w.tol)
    assert res.status == rfoe.OK and res.converged
    assert res.iterations == its64 and res.branch.upper() == br64
    assert res.fp32_steps >= res.iterations // 2 and res.branch[: res.fp32_steps].islower()
    P = res.P
    assert torch.equal(P, P.T)
    assert abs(torch.diagonal(P).sum().item() - nocc) <= 1e-8
    dP = torch.linalg.norm(P - Pex).item() / math.sqrt(k)
    dE = abs(res.tr_PH - w.band_energy()) / abs(w.band_energy())
    idem = torch.linalg.norm(P @ P - P).item()
    assert dP <= 1e-6 and dE <= 1e-8 and idem <= 1e-10 * k / 256, (dP, dE, idem)
    return dict(k=k, iterations=res.iterations, fp32_steps=res.fp32_steps, dP=dP, dE=dE, idem=idem,
                device_ms=res.device_ms, fp64_device_ms=ms64, branch=res.branch)


def test_fullsize_config3_mixed():
    print(_run_fullsize_mixed(3))


def test_fullsize_config4_mixed():
    print(_run_fullsize_mixed(4))


def test_paper_workload_k8192():
    """NEXT-3: the paper's own synthetic H^p (reading R12), N_occ = 0.9 k, RelTr 5e-8 (stop rule B,
    PAPER.md:92), k = 8192 (the smallest size the paper runs).  D_ref comes from an explicit
    eigendecomposition, as in the paper (ELPA there, torch.linalg.eigh here -- harness only); error metrics
    eps1 = ||D - D_ref||_F / ||D_ref||_F and eps2 = |Tr(D H) - Tr(D_ref H)| / |Tr(D_ref H)|.
    Paper: "around 50" Z-RFOE and "around 30" A-Z-RFOE iterations, eps1 ~ 1e-10, eps2 ~ 1e-9 (FP64),
    eps1 ~ 1e-7, eps2 ~ 1e-9 (mixed)."""
    k = 8192
    Hn = rfoe_inputs.paper_matrix(k)
    H = torch.from_numpy(Hn).cuda()
    nocc = round(0.9 * k)
    lam, V = torch.linalg.eigh(H)
    Vo = V[:, :nocc]
    Dref = Vo @ Vo.T
    del V, Vo
    homo, lumo, eband = lam[nocc - 1].item(), lam[nocc].item(), lam[:nocc].sum().item()
    nref = torch.linalg.norm(Dref).item()
    assert nref == pytest.approx(math.sqrt(nocc), rel=1e-9)                      # R14: ||D_ref||_F = sqrt(N_occ)

    def eps(r):
        return torch.linalg.norm(r.P - Dref).item() / nref, abs(r.tr_PH - eband) / abs(eband)

    out = {}
    with rfoe.Rfoe(k) as h:
        h.configure(stop_rule=rfoe.RULE_B)
        z = h.expand(H, nocc, rfoe.SP2, 5e-8)
        out["Z-RFOE"] = (z.iterations, *eps(z), z.device_ms)
        model = pins.scalar_sp2(lam.cpu().numpy(), nocc, z.eps_min, z.eps_max, tol=5e-8, rule="B")
        assert z.converged and z.iterations == model["iterations"] and 45 <= z.iterations <= 60
        assert out["Z-RFOE"][1] <= 1e-5 and out["Z-RFOE"][2] <= 1e-6              # limited by the RelTr stop, not by rounding
        h.configure(homo=homo, lumo=lumo)
        a = h.expand(H, nocc, rfoe.SP2_ACCEL, 5e-8)
        out["A-Z-RFOE"] = (a.iterations, *eps(a), a.device_ms)
        assert a.converged and 26 <= a.iterations <= 34
        assert out["A-Z-RFOE"][1] <= 1e-9 and out["A-Z-RFOE"][2] <= 1e-9
        h.configure(mixed_head=0.0, mixed_reltr=5e-4)
        m = h.expand(H, nocc, rfoe.SP2_MIXED, 5e-8)
        out["Z-RFOE mixed"] = (m.iterations, *eps(m), m.device_ms)
        assert m.converged and m.iterations == z.iterations and m.fp32_steps >= 20
        assert out["Z-RFOE mixed"][1] <= 1e-5 and out["Z-RFOE mixed"][2] <= 1e-6
    print({k_: tuple(float(f"{v:.3g}") for v in vs) for k_, vs in out.items()})


def _paper_matrix_cuda(k, block=4096):
    """rfoe_inputs.paper_matrix (reading R12) built on the GPU in row blocks (same formula)."""
    H = torch.empty((k, k), dtype=torch.float64, device="cuda")
    j = torch.arange(k, device="cuda", dtype=torch.float64)
    for r0 in range(0, k, block):
        i = j[r0:r0 + block]
        H[r0:r0 + block] = torch.exp(-0.5 * (i[:, None] - j[None, :]).abs()) * torch.sin(torch.minimum(i[:, None], j[None, :]) + 1.0)
    return H


@pytest.mark.slow
def test_paper_workload_k65536():
    """The paper's largest problem (k = 65536) on ONE B200: 34 GB per FP64 matrix.
    No eigendecomposition reference at this size; properties only: the scalar-model-free invariants
    tr D = N_occ, bitwise symmetry, idempotency, commutation with H, and A-Z-RFOE reaching the same D as Z-RFOE."""
    k = 65536
    nocc = round(0.9 * k)
    H = _paper_matrix_cuda(k)
    assert torch.allclose(H[:512, :512], torch.from_numpy(rfoe_inputs.paper_matrix(512)).cuda(), rtol=1e-13, atol=1e-300)
    out = {}
    with rfoe.Rfoe(k) as h:
        h.configure(stop_rule=rfoe.RULE_B, check_symmetry=True)
        z = h.expand(H, nocc, rfoe.SP2, 5e-8)
        Pz = z.P
        fl = 2.0 * k * (512 * 513 // 2) * 128 * 128
        out["Z-RFOE"] = dict(steps=z.iterations, seconds=z.device_ms / 1e3, tflops=z.iterations * fl / (z.device_ms * 1e-3) / 1e12)
        assert z.converged and 45 <= z.iterations <= 66
        assert abs(torch.diagonal(Pz).sum().item() - nocc) <= 1e-3          # RelTr 5e-8 of 59k stops ~3e-3 away at most
    # the handle (two 34 GB work matrices) is gone: room for the checks
    PP = Pz @ Pz
    idem = torch.linalg.norm(PP - Pz).item()
    del PP
    HP = H @ Pz
    comm = torch.linalg.norm(HP - HP.T).item()
    del HP
    out["Z-RFOE"].update(idem=idem, comm=comm, trace_err=abs(torch.diagonal(Pz).sum().item() - nocc))
    assert torch.equal(Pz, Pz.T) and idem <= 1e-2 and comm <= 1e-2
    # ---- the paper's mixed-precision Z-RFOE on the same problem: reduced-precision squarings until
    # RelTr <= 5e-7 (late switch), FP64 to 5e-8; Pz waits on the host meanwhile (34 GB per matrix)
    Pz_host = Pz.cpu()
    z.P = None                      # the result object holds the other reference to the 34 GB matrix
    del Pz
    torch.cuda.empty_cache()
    with rfoe.Rfoe(k) as h:
        h.configure(stop_rule=rfoe.RULE_B, mixed_head=0.0, mixed_reltr=5e-7)
        mres = h.expand(H, nocc, rfoe.SP2_MIXED, 5e-8)
        Pm = mres.P
        out["mixed Z-RFOE (late switch)"] = dict(steps=mres.iterations, reduced=mres.fp32_steps, seconds=mres.device_ms / 1e3,
                                                 speedup=z.device_ms / mres.device_ms)
        assert mres.converged and abs(mres.iterations - z.iterations) <= 2
    del H
    torch.cuda.empty_cache()
    Pz = Pz_host.cuda()
    eps1 = (torch.linalg.norm(Pm - Pz) / torch.linalg.norm(Pz)).item()          # the paper's eps_1 against the FP64 run
    out["mixed Z-RFOE (late switch)"].update(eps1_vs_fp64=eps1, trace_err=abs(torch.diagonal(Pm).sum().item() - nocc))
    print(out)
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/paper_k65536.txt", "w") as f:
        f.write(repr(out) + "\n")
    # RelTr 5e-8 stops both runs ~1e-4 short of idempotency on this matrix (gap ~2e-5 of a width 3.7: idem above), so two
    # differently rounded runs agree to that level, not to the 1e-7 the paper quotes for its (unstated) sizes
    assert eps1 <= 5e-4 and torch.equal(Pm, Pm.T)
