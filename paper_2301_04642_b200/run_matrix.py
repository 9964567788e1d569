"""Run matrix of DESIGN.md section 8 / SURVEY.md section 8(d): every BASELINE.json config through the C ABI in each
variant that applies, with timing and accuracy against the construction-exact projector.

    python -m paper_2301_04642_b200.run_matrix [--configs 1 2 3 4] [--markdown]

Harness code: torch builds the inputs (rfoe_inputs) and the reference projector Q_occ Q_occ^T; every step
of the expansions runs in librfoe.  Prints one row per (config, run)."""
from __future__ import annotations

import argparse
import math
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main() -> int:
    import torch

    import paper_2301_04642_b200 as rfoe
    import rfoe_inputs

    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[1, 2, 3, 4])
    ap.add_argument("--markdown", action="store_true")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("run_matrix: no CUDA device -- there is no CPU fallback")
    sep = " | " if args.markdown else "  "
    cols = ["config", "k", "run", "steps", "mults", "reduced", "ms", "TFLOP/s", "errP", "dE", "status"]
    print(sep.join(cols))
    if args.markdown:
        print(sep.join("---" for _ in cols))
    for c in args.configs:
        w = rfoe_inputs.make_workload(c, device="cuda")
        k, nocc = w.k, w.nocc
        H = w.H if isinstance(w.H, torch.Tensor) else torch.from_numpy(w.H).cuda()
        Q = w.Q if isinstance(w.Q, torch.Tensor) else torch.from_numpy(w.Q).cuda()
        Pex = Q[:, :nocc] @ Q[:, :nocc].T
        del Q
        w.Q = None
        eband = w.band_energy()
        m = (k + 127) // 128
        fl_sq = 2.0 * (m * 128) * (m * (m + 1) // 2) * 128 * 128
        lam = w.lam
        homo, lumo = float(lam[:nocc].max()), float(lam[nocc:].min())
        runs = [("SP2 rule A, Gershgorin (normative)", rfoe.SP2, w.tol, {}),
                ("SP2 rule B RelTr 5e-8 (paper's criterion)", rfoe.SP2, 5e-8, dict(stop_rule=rfoe.RULE_B)),
                ("SP2 rule A, exact spectral bounds", rfoe.SP2, w.tol, dict(bounds=(float(lam.min()), float(lam.max())))),
                ("SP2 rule A, Lanczos bounds (24 steps, on the device)", rfoe.SP2, w.tol, dict(lanczos_steps=24)),
                ("mixed (late switch 5e-7) + Lanczos bounds", rfoe.SP2_MIXED, w.tol, dict(lanczos_steps=24, mixed_head=0.0, mixed_reltr=5e-7)),
                ("A-Z-RFOE (accelerated), exact HOMO/LUMO", rfoe.SP2_ACCEL, w.tol, dict(homo=homo, lumo=lumo)),
                ("A-Z-RFOE, HOMO/LUMO estimated from the normative run's history", rfoe.SP2_ACCEL, w.tol, "estimated"),
                ("McWeeny-style tail", rfoe.MCWEENY, w.tol, {}),
                ("mixed, paper schedule (reduced until RelTr 5e-4)", rfoe.SP2_MIXED, w.tol, dict(mixed_head=0.0, mixed_reltr=5e-4))]
        with rfoe.Rfoe(k) as h:
            for name, variant, tol, opts in runs:
                h.configure(stop_rule=rfoe.RULE_A, bounds=False, mixed_head=0.0, mixed_reltr=5e-4, lanczos_steps=0)
                if opts == "estimated":                              # rfoe_estimate_homo_lumo on the first row's history
                    opts = dict(homo=est[0], lumo=est[1])
                h.configure(**opts)
                r = None
                for _ in range(2):                                   # second run is the timed one (warm)
                    r = h.expand(H, nocc, variant, tol)
                if name.endswith("(normative)"):
                    est = h.estimate_homo_lumo()
                P = r.P
                err = torch.linalg.norm(P - Pex).item() / math.sqrt(k)
                dE = abs(r.tr_PH - eband) / abs(eband)
                tf = r.multiplications * fl_sq / (r.device_ms * 1e-3) / 1e12
                row = [str(c), str(k), name, str(r.iterations), str(r.multiplications), str(r.fp32_steps), f"{r.device_ms:.2f}",
                       f"{tf:.1f}", f"{err:.2e}", f"{dE:.1e}", "ok" if r.converged else "not converged"]
                print(sep.join(row), flush=True)
                del P, r
        del H, Pex
        torch.cuda.empty_cache()
    return 0


if __name__ == "__main__":
    sys.exit(main())
