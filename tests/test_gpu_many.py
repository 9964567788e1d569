"""rfoe_expand_many: independent problems side by side on one GPU (one handle, stream and host thread each) give, problem
by problem, bitwise the P of a lone rfoe_expand call and the oracle's result within the north_star tolerances."""
import math

import numpy as np
import pytest

import oracle
import rfoe_inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2301_04642_b200 as rfoe  # noqa: E402


def _problems():
    out = []
    for c, k in [(1, 100), (2, 333), (3, 200), (4, 450), (1, 256), (2, 130), (3, 64), (4, 257), (1, 5), (2, 512)]:
        w = rfoe_inputs.make_workload(c, k=k)
        out.append((w, torch.from_numpy(w.H).cuda()))
    return out


@pytest.mark.parametrize("n_handles", [1, 3, 16])
def test_many_equals_lone_calls_bitwise_and_oracle(n_handles):
    probs = _problems()
    handles = [rfoe.Rfoe(512) for _ in range(n_handles)]
    try:
        res = rfoe.expand_many(handles, [(H, w.nocc, w.tol) for w, H in probs])
        assert len(res) == len(probs)
        with rfoe.Rfoe(512) as lone:
            for (w, H), r in zip(probs, res):
                one = lone.expand(H, w.nocc, rfoe.SP2, w.tol)
                assert r.converged and r.iterations == one.iterations and r.branch == one.branch
                assert torch.equal(r.P, one.P)                                    # the same path, bit for bit
                assert r.tr_PH == one.tr_PH and np.array_equal(r.t, one.t) and np.array_equal(r.e, one.e)
        for (w, H), r in list(zip(probs, res))[:4]:
            ref = oracle.expand(w.H, w.nocc, tol=w.tol)
            assert r.iterations == ref.iterations
            assert np.linalg.norm(r.P.cpu().numpy() - ref.P) / math.sqrt(w.k) <= 1e-10
            assert abs(r.tr_PH - ref.tr_PH) <= 1e-11 * abs(ref.tr_PH)
    finally:
        for h in handles:
            h.close()


def test_many_variants_status_and_errors():
    probs = _problems()[:5]
    handles = [rfoe.Rfoe(512) for _ in range(2)]
    try:
        # accelerated variant with per-handle options; a capped run reports NOT_CONVERGED per problem without raising
        w, H = probs[1]
        for h in handles:
            h.configure(max_iter=5)
        res = rfoe.expand_many(handles, [(H, w.nocc, 0.0)] * 3)
        assert [r.status for r in res] == [rfoe.ERR_NOT_CONVERGED] * 3 and all(r.iterations == 5 for r in res)
        assert torch.equal(res[0].P, res[1].P) and torch.equal(res[0].P, res[2].P)
        for h in handles:
            h.configure(max_iter=100)
        assert rfoe.expand_many(handles, []) == []
        with pytest.raises(rfoe.RfoeError) as ei:                                   # nocc out of range in problem 1 only
            rfoe.expand_many(handles, [(H, w.nocc, w.tol), (H, w.k, w.tol)])
        assert ei.value.status == rfoe.ERR_INVALID_ARG and "problem 1" in str(ei.value)
        with pytest.raises(rfoe.RfoeError) as ei:                                   # the same handle twice
            rfoe.expand_many([handles[0], handles[0]], [(H, w.nocc, w.tol)])
        assert ei.value.status == rfoe.ERR_INVALID_ARG
    finally:
        for h in handles:
            h.close()
