"""GPU parity of the optional Lanczos spectral bounds (rfoe_bounds_lanczos, RFOE_OPT_LANCZOS_STEPS) with the oracle.
Tolerance: both sides run the same recursion from the same start vector with different summation orders (warp
shuffles, FMA); rounding differences of ~k eps per product are amplified mildly over m <= 32 steps, the converged
extreme Ritz values and beta_m stay within 1e-9 of the spectral width (measured: <= 1e-12)."""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_2301_04642_b200 as rfoe
import rfoe_inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("c,k,m", [(1, 256, 24), (2, 333, 16), (3, 640, 24), (4, 1024, 32), (1, 5, 3), (2, 129, 8), (3, 2048, 24)])
def test_bounds_match_oracle_and_enclose(c, k, m):
    w = rfoe_inputs.make_workload(c, k=k)
    olo, ohi, _, _ = oracle.bounds_lanczos(w.H, m)
    with rfoe.Rfoe(k) as h:
        lo, hi = h.bounds_lanczos(torch.from_numpy(w.H).cuda(), m)
    width = ohi - olo
    assert abs(lo - olo) <= 1e-9 * width and abs(hi - ohi) <= 1e-9 * width
    ev = np.linalg.eigvalsh(w.H)
    assert lo <= ev[0] and ev[-1] <= hi


def test_breakdown_on_device():
    with rfoe.Rfoe(16) as h:
        lo, hi = h.bounds_lanczos((2.0 * torch.eye(7, dtype=torch.float64)).cuda(), 5)
        assert lo == pytest.approx(2.0) and hi == pytest.approx(2.0)
        d = torch.diag(torch.tensor([1.0, 1.0, -3.0, 5.0, 5.0, -3.0], dtype=torch.float64)).cuda()
        lo, hi = h.bounds_lanczos(d, 6)
        assert lo == pytest.approx(-3.0, abs=1e-12) and hi == pytest.approx(5.0, abs=1e-12)
        with pytest.raises(rfoe.RfoeError):
            h.bounds_lanczos(d, 0)


@pytest.mark.parametrize("c,k", [(2, 333), (4, 777)])
def test_expand_with_lanczos_bounds_matches_oracle(c, k):
    w = rfoe_inputs.make_workload(c, k=k)
    olo, ohi, _, _ = oracle.bounds_lanczos(w.H, 24)
    ref = oracle.expand(w.H, w.nocc, tol=w.tol, bounds_override=(olo, ohi))
    ref_g = oracle.expand(w.H, w.nocc, tol=w.tol)
    with rfoe.Rfoe(k) as h:
        h.configure(lanczos_steps=24)
        res = h.expand(torch.from_numpy(w.H).cuda(), w.nocc, rfoe.SP2, w.tol)
    assert res.converged and res.iterations == ref.iterations and res.iterations < ref_g.iterations
    assert np.linalg.norm(res.P.cpu().numpy() - ref.P) / math.sqrt(k) <= 1e-10
    assert abs(res.tr_PH - ref.tr_PH) / abs(ref.tr_PH) <= 1e-11


def test_fullsize_config4_lanczos_bounds():
    """k=16384: the bounds enclose the spectrum the generator prescribed ([-2, 4]), are within 1.6x of its width, and
    the expansion needs about 39 instead of 56 squarings and reaches the construction-exact projector."""
    w = rfoe_inputs.make_workload(4, device="cuda")
    with rfoe.Rfoe(w.k) as h:
        lo, hi = h.bounds_lanczos(w.H, 24)
        assert lo <= -2.0 and hi >= 4.0 and (hi - lo) <= 1.6 * 6.0
        h.configure(lanczos_steps=24)
        res = h.expand(w.H, w.nocc, rfoe.SP2, w.tol)
        assert res.converged and 34 <= res.iterations <= 42
        Qo = w.Q[:, : w.nocc]
        errP = float(torch.linalg.norm(res.P - Qo @ Qo.T)) / math.sqrt(w.k)
        assert errP <= 1e-10
        assert abs(res.tr_PH - w.band_energy()) / abs(w.band_energy()) <= 1e-11
        print(f"lanczos bounds [{lo:.4f}, {hi:.4f}], {res.iterations} squarings, {res.device_ms:.1f} ms, errP {errP:.2e}")
