"""The C ABI used from plain C (no Python, no torch in the process): tests/abi_client.c builds the paper's synthetic
H^p, runs Z-RFOE through rfoe_create / rfoe_bounds / rfoe_expand / rfoe_get_stats / rfoe_destroy with
cudaMalloc'ed buffers and its own stream, and writes P; the oracle runs on the same matrix."""
import math
import subprocess

import numpy as np
import pytest

import oracle
import rfoe_inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("k", [200, 777])
def test_c_client_matches_oracle(tmp_path, k):
    from tests import abi_client_build

    exe = abi_client_build.build(tmp_path)
    nocc = round(0.9 * k)                                   # "N_occ around 90 %" (reading R13)
    tol = 1e-12 * max(1.0, k / 256)
    out_bin = tmp_path / "P.bin"
    out = subprocess.run([exe, "expand", str(k), str(nocc), repr(tol), str(out_bin)], check=True, capture_output=True,
                         text=True, timeout=300).stdout
    kv = dict(p.split("=", 1) for p in out.split())
    H = rfoe_inputs.paper_matrix(k)
    ref = oracle.expand(H, nocc, tol=tol)
    P = np.fromfile(out_bin, dtype=np.float64).reshape(k, k)
    assert int(kv["status"]) == 0 and int(kv["converged"]) == 1
    assert int(kv["iterations"]) == ref.iterations and len(kv["branch"]) == ref.iterations
    for n, (a, b) in enumerate(zip(kv["branch"], ref.branch)):  # identical wherever t_n - nocc is above rounding level (R10)
        assert a == b or abs(ref.t[n] - nocc) <= 1e-9 * max(1.0, k / 256), n
    lo, hi = oracle.bounds(H)
    for key, val in (("eps_min", lo), ("bounds_min", lo), ("eps_max", hi), ("bounds_max", hi)):
        assert float(kv[key]) == pytest.approx(val, rel=1e-13)
    assert np.linalg.norm(P - ref.P) / math.sqrt(k) <= 1e-10
    assert abs(float(kv["tr_PH"]) - ref.tr_PH) <= 1e-11 * abs(ref.tr_PH)
    assert np.array_equal(P, P.T) and round(float(kv["t_last"])) == nocc
    # k <= 4096: the recursion is one persistent launch (stats.resident); otherwise at least one launch per step
    assert int(kv["launches"]) >= (5 if int(kv["resident"]) else ref.iterations)
    oh, ol = oracle.estimate_homo_lumo(ref, nocc)
    assert int(kv["hl_status"]) == 0
    assert float(kv["homo"]) == pytest.approx(oh, abs=1e-8 * (hi - lo)) and float(kv["lumo"]) == pytest.approx(ol, abs=1e-8 * (hi - lo))
