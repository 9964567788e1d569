"""The whole recursion in one persistent launch (csrc/resident.cuh; RFOE_OPT_RESIDENT, the default for k <= 4096)
against (a) the CPU oracle at the north_star tolerances, (b) the launch-per-step path of the same library, (c) itself.

The persistent kernel cuts a step into equal runs of 16-wide contraction slices per SM (stream-K), so a tile's sum over
the contraction index is associated differently from the launch-per-step path: the two agree to rounding, not to the
bit.  What IS bitwise: two runs of the same path (fixed-order sums everywhere), and every decision taken from the
sums -- iteration count and branch string are identical on all three."""
import math

import numpy as np
import pytest

import oracle
import rfoe_inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2301_04642_b200 as rfoe  # noqa: E402


def _dev(a):
    if isinstance(a, torch.Tensor):
        return a.cuda()
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("c,k", [(1, 2), (1, 5), (1, 100), (5, 129), (1, 256), (2, 333), (4, 515), (3, 777), (3, 1024),
                                 (2, 1500), (2, 2048)])
def test_resident_vs_oracle_and_stepwise(c, k):
    if k >= 16:
        w = rfoe_inputs.make_workload(c, k=k)
        H, nocc, tol = w.H, w.nocc, w.tol
    else:
        rng = np.random.default_rng(50 + k)
        A = rng.standard_normal((k, k))
        H = np.ascontiguousarray(0.5 * (A + A.T)) + np.diag(np.arange(k, dtype=np.float64))
        nocc, tol = max(1, k // 2), 1e-12
    ref = oracle.expand(H, nocc, tol=tol)
    Hd = _dev(H)
    with rfoe.Rfoe(k) as h:
        res = h.expand(Hd, nocc, rfoe.SP2, tol)
        again = h.expand(Hd, nocc, rfoe.SP2, tol)
        h.configure(resident=False)
        step = h.expand(Hd, nocc, rfoe.SP2, tol)
    assert res.resident and again.resident and not step.resident
    assert res.gpu_launches <= 12 < step.gpu_launches           # the host is out of the loop
    # (a) the oracle
    P = res.P.cpu().numpy()
    assert res.status == rfoe.OK and res.converged == ref.converged and res.iterations == ref.iterations
    decided = np.abs(ref.t[: ref.iterations] - nocc) > 1e-9 * max(1.0, k / 256)
    assert all(a == b for a, b, d in zip(res.branch, ref.branch, decided) if d), (res.branch, ref.branch)
    assert np.linalg.norm(P - ref.P) / math.sqrt(k) <= 1e-10 and np.abs(P - ref.P).max() <= 1e-11
    assert abs(res.tr_PH - ref.tr_PH) <= 1e-11 * abs(ref.tr_PH)
    assert np.array_equal(P, P.T)
    assert np.allclose(res.t, ref.t, rtol=0, atol=1e-9 * max(1.0, k / 256)) and np.allclose(res.s, ref.s, rtol=0, atol=1e-9 * max(1.0, k / 256))
    n = ref.iterations
    assert np.allclose(res.e[: n - 1], ref.e[: n - 1], rtol=1e-6, atol=1e-11 * max(1.0, k / 256))
    assert abs(np.trace(P) - nocc) <= 1e-9
    # (b) the launch-per-step path: same decisions, same matrix to rounding
    assert step.iterations == res.iterations
    assert all(a == b_ for a, b_, d in zip(step.branch, res.branch, decided) if d), (step.branch, res.branch)
    Ps = step.P.cpu().numpy()
    assert np.abs(P - Ps).max() <= 1e-12
    assert np.allclose(res.t, step.t, rtol=1e-13, atol=1e-13) and np.allclose(res.s, step.s, rtol=1e-13, atol=1e-13)
    assert res.eps_min == step.eps_min and res.eps_max == step.eps_max and res.t[0] == step.t[0] and res.s[0] == step.s[0]
    # (c) itself: bitwise
    assert torch.equal(res.P, again.P) and np.array_equal(res.t, again.t) and np.array_equal(res.s, again.s)
    assert np.array_equal(res.e, again.e) and res.tr_PH == again.tr_PH and res.branch == again.branch


def test_resident_variants_and_options():
    """A-Z-RFOE, T-RFOE, stop rule B, bounds override and the Lanczos bounds through the persistent kernel."""
    w = rfoe_inputs.make_workload(3, k=640)
    Hd = _dev(w.H)
    homo, lumo = float(w.lam[: w.nocc].max()), float(w.lam[w.nocc:].min())
    with rfoe.Rfoe(640) as h:
        h.configure(homo=homo, lumo=lumo)
        ref = oracle.expand(w.H, w.nocc, variant=oracle.SP2_ACCEL, tol=w.tol, homo=homo, lumo=lumo)
        res = h.expand(Hd, w.nocc, rfoe.SP2_ACCEL, w.tol)
        assert res.resident and res.iterations == ref.iterations and res.branch[:-3] == ref.branch[:-3]
        assert np.abs(res.P.cpu().numpy() - ref.P).max() <= 1e-11
        h.configure(trunc_steps=11)
        ref = oracle.expand(w.H, w.nocc, variant=oracle.TRUNC, max_iter=11)
        res = h.expand(Hd, w.nocc, rfoe.TRUNC, 0.0)
        assert res.resident and res.status == rfoe.OK and res.iterations == 11 == res.trunc_steps and res.branch == ref.branch
        assert np.abs(res.P.cpu().numpy() - ref.P).max() <= 1e-12
        h.configure(stop_rule=rfoe.RULE_B)
        ref = oracle.expand(w.H, w.nocc, tol=5e-8, stop_rule=oracle.RULE_B)
        res = h.expand(Hd, w.nocc, rfoe.SP2, 5e-8)
        assert res.resident and res.iterations == ref.iterations and res.branch == ref.branch
        assert np.abs(res.P.cpu().numpy() - ref.P).max() <= 1e-11 and np.allclose(res.reltr, ref.reltr, rtol=1e-6, atol=1e-13)
        lo, hi = float(w.lam.min()) - 0.01, float(w.lam.max()) + 0.01
        h.configure(stop_rule=rfoe.RULE_A, bounds=(lo, hi))
        ref = oracle.expand(w.H, w.nocc, tol=w.tol, bounds_override=(lo, hi))
        res = h.expand(Hd, w.nocc, rfoe.SP2, w.tol)
        assert res.resident and res.iterations == ref.iterations and (res.eps_min, res.eps_max) == (lo, hi)
        assert np.abs(res.P.cpu().numpy() - ref.P).max() <= 1e-11
        h.configure(bounds=False, max_iter=5)
        res = h.expand(Hd, w.nocc, rfoe.SP2, w.tol)                   # max_iter reached: NOT_CONVERGED, stats complete
        assert res.resident and res.status == rfoe.ERR_NOT_CONVERGED and res.iterations == 5 and len(res.e) == 5


def test_resident_errors_are_settled_on_the_device():
    """Bad input stops the enqueued sequence by itself (control_begin); the host reports it after its single sync."""
    w = rfoe_inputs.make_workload(1, k=300)
    Hd = _dev(w.H)
    with rfoe.Rfoe(300) as h:
        bad = Hd.clone()
        bad[7, 200] += 1e-9
        with pytest.raises(rfoe.RfoeError) as ei:
            h.expand(bad, w.nocc, rfoe.SP2, w.tol)
        assert ei.value.status == rfoe.ERR_NOT_SYMMETRIC
        with pytest.raises(rfoe.RfoeError) as ei:
            h.expand(torch.eye(300, dtype=torch.float64, device="cuda"), 10, rfoe.SP2, 1e-12)
        assert ei.value.status == rfoe.ERR_BAD_BOUNDS
        nan = Hd.clone()
        nan[5, 5] = float("nan")
        with pytest.raises(rfoe.RfoeError) as ei:
            h.expand(nan, w.nocc, rfoe.SP2, w.tol)
        assert ei.value.status == rfoe.ERR_BAD_BOUNDS
        h.configure(homo=-1e3, lumo=0.0)
        with pytest.raises(rfoe.RfoeError) as ei:
            h.expand(Hd, w.nocc, rfoe.SP2_ACCEL, w.tol)
        assert ei.value.status == rfoe.ERR_INVALID_ARG
        res = h.expand(Hd, w.nocc, rfoe.SP2, w.tol)                   # the handle is fine afterwards
        assert res.converged and res.resident


@pytest.mark.parametrize("k", [1800, 2048, 2304, 2600])
def test_resident_finisher_form_vs_band_form(k):
    """k = 1792 ... 2816: a tile cut between SMs is finished by its first holder, from registers, with the other holders' parts
    arriving through the operand ring (csrc/resident_fin.cuh; one grid barrier per step) -- against the band form
    (RFOE_OPT_RESIDENT = 2: all parts to the workspace, finished in 16-row bands after a barrier), which adds the same parts in
    the same order: X_{n+1} agrees bit for bit step by step until the trace reaches nocc to rounding; the tile records are
    summed from differently shaped partial sums, so t_n differs in its last bits and an undecided late step may take the
    other (equally valid) branch.  Both against the construction-exact projector."""
    w = rfoe_inputs.make_workload(2, k=k)
    Hd = _dev(w.H)
    with rfoe.Rfoe(k) as h:
        fin = h.expand(Hd, w.nocc, rfoe.SP2, w.tol)
        again = h.expand(Hd, w.nocc, rfoe.SP2, w.tol)
        h.configure(resident=2)
        band = h.expand(Hd, w.nocc, rfoe.SP2, w.tol)
        h.configure(trunc_steps=6)
        b6 = h.expand(Hd, w.nocc, rfoe.TRUNC, 0.0)
        h.configure(resident=1)
        f6 = h.expand(Hd, w.nocc, rfoe.TRUNC, 0.0)
    assert fin.resident and band.resident and fin.converged and band.converged and fin.iterations == band.iterations
    assert torch.equal(f6.P, b6.P)                                     # six steps, all decided: the same bits
    assert torch.equal(fin.P, again.P) and np.array_equal(fin.t, again.t)     # run to run: bitwise
    decided = np.abs(band.t[: band.iterations] - w.nocc) > 1e-9 * max(1.0, k / 256)
    assert all(a == b for a, b, d in zip(fin.branch, band.branch, decided) if d)
    assert (fin.P - band.P).abs().max().item() <= 1e-12 and torch.equal(fin.P, fin.P.T)
    assert np.allclose(fin.t, band.t, rtol=1e-13, atol=1e-11) and np.allclose(fin.e[:-3], band.e[:-3], rtol=1e-6, atol=1e-12)
    Pex = _dev(w.exact_projector())
    for r in (fin, band):
        assert torch.linalg.norm(r.P - Pex).item() / math.sqrt(k) <= 1e-10
    print(f"k={k}: finisher form {fin.device_ms:.3f} ms, band form {band.device_ms:.3f} ms, {fin.iterations} steps, phases (us/step) "
          f"{[round(x * 1e3 / fin.iterations, 1) for x in fin.resident_phase_ms]}")


@pytest.mark.parametrize("k", [3000, 4096])
def test_resident_largest_sizes_vs_stepwise(k):
    """The upper end of the persistent path (several whole tiles per SM plus split ones): against the launch-per-step
    path and the construction-exact projector (the oracle would need minutes here; k = 2048 above is the largest
    whole-oracle case)."""
    w = rfoe_inputs.make_workload(2, k=k, device="cuda")
    H = w.H if isinstance(w.H, torch.Tensor) else _dev(w.H)
    with rfoe.Rfoe(k) as h:
        res = h.expand(H, w.nocc, rfoe.SP2, w.tol)
        h.configure(resident=False)
        step = h.expand(H, w.nocc, rfoe.SP2, w.tol)
    assert res.resident and res.converged and res.iterations == step.iterations and res.branch[:-3] == step.branch[:-3]
    assert (res.P - step.P).abs().max().item() <= 1e-12 and torch.equal(res.P, res.P.T)
    Q = w.Q if isinstance(w.Q, torch.Tensor) else _dev(w.Q)
    Pex = Q[:, : w.nocc] @ Q[:, : w.nocc].T
    assert torch.linalg.norm(res.P - Pex).item() / math.sqrt(k) <= 1e-10
    print(f"k={k}: resident {res.device_ms:.3f} ms, launch-per-step {step.device_ms:.3f} ms, {res.iterations} steps")
