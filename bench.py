#!/usr/bin/env python
"""bench.py -- one JSON line for the RFOE hot path on B200.

A *step* is one whole expansion through the C ABI (``rfoe_expand``): symmetry check, Gershgorin
bounds (A1), affine map (A2), the trace-steered recursion of symmetric FP64 squarings with the fused
epilogue (A3-A6, ~56 squarings at k=16384) and the output pass with tr(P H).  Workload: BASELINE.json
config 4 (k=16384, nocc=12600), the configuration the metric is quoted on; synthetic seeded input
(rfoe_inputs), resident in HBM before the timed region.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

N > 1 (torchrun): the path does not shard inside one expansion in this build ("replicas only",
DESIGN.md): every rank expands its own H^p, no data-path collective, weak scaling; `value` is the
whole-job aggregate.  `--impl reference` times the CPU oracle (oracle/) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FP64 TFLOP/s over a whole RFOE expansion (executed flops of the symmetric squarings / expansion time)"
UNIT = "TFLOP/s"
TILE = 128

# FP64 tensor-pipe peak.  MEASURED_PEAKS.json has no FP64 entry and the profiling
# guide lists no FP64 nominal, so the denominator is MEASURED BY THIS RUN: rfoe_probe_fp64_peak, a register-only
# DMMA.8x8x4 issue loop on every SM (`roofline.peak` = `peak_measured`), right after the timed region.  The derived
# figure 148 SMs x 64 DFMA/clk/SM x 2 x 1.965 GHz is reported beside it as `peak_derived`, and a cuBLAS Dgemm
# (torch.matmul, FP64) as context.
FP64_PEAK_DERIVED_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
FP64_PEAK_TFLOPS = FP64_PEAK_DERIVED_TFLOPS

# dram__bytes_read.sum + dram__bytes_write.sum of one sym_square_kernel launch, from the `ncu --set full` captures
# summarised in profiles/ (ncu cannot run inside a timed bench: the figure is quoted, with its source, not re-measured).
NCU_TRAFFIC_BYTES = {16384: (24.629606e9 + 2.129160e9, "profiles/r02c_sym_square_k16384.md")}


def fp64_peaks(h, torch, stream, n_gemm=8192):
    """The FP64 denominators, measured now on this device: the library's DMMA issue-rate probe (~300 ms) and, as context,
    cuBLAS Dgemm through torch.matmul (2 n^3 flops, best of 3 after a warm-up)."""
    probe = h.probe_fp64_peak(300.0, stream=stream)
    a = torch.randn((n_gemm, n_gemm), dtype=torch.float64, device="cuda")
    b = torch.randn((n_gemm, n_gemm), dtype=torch.float64, device="cuda")
    c = torch.empty_like(a)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = float("inf")
    for i in range(4):
        e0.record(stream)
        torch.matmul(a, b, out=c)
        e1.record(stream)
        torch.cuda.synchronize()
        if i:
            best = min(best, e0.elapsed_time(e1))
    del a, b, c
    return probe, 2.0 * n_gemm ** 3 / (best * 1e-3) / 1e12


def executed_flops_per_squaring(k: int) -> float:
    """2 * k_padded * n_t * T^2: the FMA-flops the squaring kernel issues (upper-triangle tiles only)."""
    m = (k + TILE - 1) // TILE
    n_t = m * (m + 1) // 2
    return 2.0 * (m * TILE) * n_t * TILE * TILE


def oracle_flops_per_squaring(k: int) -> float:
    """The oracle's symmetric product computes j >= i only: k(k+1)/2 dot products of length k."""
    return float(k) * k * (k + 1)


# --------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """`nvidia-smi ... -lms 200` (the recipe's clocks line) for one GPU while the timed region runs."""

    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_id: str):
        self.gpu_id = gpu_id
        self.proc = None
        self.path = None

    def start(self):
        fd, self.path = tempfile.mkstemp(prefix="rfoe_clocks_", suffix=".csv")
        os.close(fd)
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", self.gpu_id, f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "200", "-f", self.path], stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None
        return self

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "power_w_max": None, "power_w_mean": None, "samples": 0, "reasons": []}
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
        try:
            rows = [r.split(",") for r in open(self.path).read().strip().splitlines() if r.strip()]
            os.unlink(self.path)
        except OSError:
            rows = []
        sm, smax, pw, reasons = [], [], [], set()
        for r in rows:
            r = [x.strip() for x in r]
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); smax.append(float(r[2])); pw.append(float(r[3]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, r[5:9]):
                if val == "Active":
                    reasons.add(name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(smax), power_w_max=max(pw), power_w_mean=statistics.fmean(pw),
                       samples=len(sm),
                       reasons=sorted(reasons))
        return out


# --------------------------------------------------------------------------------------- oracle legs
def oracle_sample(config: int, k_sample: int):
    """One bounded sample of the workload for the CPU oracle: the same construction (spectrum shape,
    nocc/k, gap, Haar-rotated dense H) scaled down to k_sample so that a whole expansion is ~10-30 s of
    CPU work.  The metric is a rate (TFLOP/s), so the sample's value is directly comparable; the naive
    loop gets slower, not faster, at larger k (cache), so the sample flatters the oracle if anything."""
    import oracle
    import rfoe_inputs

    w = rfoe_inputs.make_workload(config, k=k_sample, device="cpu", keep_q=False)
    t0 = time.perf_counter()
    ref = oracle.expand(w.H, w.nocc, tol=w.tol)
    dt = time.perf_counter() - t0
    flops = ref.iterations * oracle_flops_per_squaring(w.k)
    return dt, flops, ref.iterations, w


def cpu_threads() -> int:
    env = os.environ.get("OMP_NUM_THREADS")
    if env and env.isdigit():
        return int(env)
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def run_reference(args) -> int:
    """--impl reference: the oracle, as it stands, on the host cores; each step one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import rfoe_inputs

    cfg = rfoe_inputs.CONFIGS[args.config]
    for _ in range(args.warmup):
        oracle_sample(args.config, args.cpu_k)
    tot_t = tot_f = 0.0
    its = 0
    for _ in range(args.steps):
        dt, fl, its, w = oracle_sample(args.config, args.cpu_k)
        tot_t += dt
        tot_f += fl
    value = tot_f / tot_t / 1e12
    sample = (f"config {args.config} construction scaled to k={w.k}, nocc={w.nocc}: one full SP2 expansion per step "
              f"({its} squarings, stop rule A tol {w.tol:.3g}); oracle flops = k^2(k+1) per squaring")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tot_t / max(args.steps, 1) * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json config {args.config}: k={cfg.k}, nocc={cfg.nocc}, SP2, Gershgorin bounds",
                   "sampled_as": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------ our arm
def whole_job_rate(ms_local: float, flops_per_rank: float, device="cpu"):
    """Replicas-only aggregation: every rank did `flops_per_rank` of independent work;
    the job's time is the MAX over ranks of the device-timed region, the job's work is the SUM.
    Returns (ms_max, TFLOP/s of the whole job).  Works on any backend (gloo on CPU in the tests)."""
    import torch
    import torch.distributed as dist

    ms = torch.tensor([ms_local], dtype=torch.float64, device=device)
    fl = torch.tensor([flops_per_rank], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        dist.all_reduce(fl, op=dist.ReduceOp.SUM)
    ms_max = float(ms.item())
    return ms_max, float(fl.item()) / (ms_max * 1e-3) / 1e12


def run_ours(args) -> int:
    import torch
    import torch.distributed as dist

    import paper_2301_04642_b200 as rfoe
    import rfoe_inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1 or args.shard:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29537")
        dist.init_process_group("nccl", device_id=dev, rank=rank, world_size=world)

    def barrier():
        if world > 1:
            dist.barrier(device_ids=[local])
        torch.cuda.synchronize()

    if args.only_subspace:          # profiling aid: only the separately reported NEXT-4 chain, one JSON line
        if rank == 0:
            with rfoe.Rfoe(args.subspace_k, device=local) as h2:
                print(json.dumps({"subspace_steps": subspace_report(h2, rfoe, rfoe_inputs, args, dev, torch.cuda.current_stream())}),
                      flush=True)
        return 0
    cfg = rfoe_inputs.CONFIGS[args.config]
    # every rank owns an independent problem of the same configuration (replicas; no data-path collective)
    want_reduced = (world == 1 and not args.no_reduced and not args.shard)
    w = rfoe_inputs.make_workload(args.config, device=str(dev) if cfg.k > 2048 else "cpu", keep_q=want_reduced)
    H = w.H if isinstance(w.H, torch.Tensor) else torch.from_numpy(w.H).to(dev)
    k, nocc, tol = w.k, w.nocc, w.tol
    P = torch.empty_like(H)
    stream = torch.cuda.current_stream()
    h = rfoe.Rfoe(k, device=local)

    shard = bool(args.shard)
    if shard and world > 1:
        dist.broadcast(H, src=0)         # one problem, the same bytes on every rank

    if args.shard == "p2p":
        # CUDA IPC handles of the work buffers, exchanged over the process group; every rank must agree on the outcome
        ok = 1
        try:
            h.shard_connect()
        except rfoe.RfoeError as e:
            if e.status != rfoe.ERR_NO_PEER_ACCESS:
                raise
            ok = 0
            why = str(e)
        if world > 1:
            flag = torch.tensor([ok], device=dev)
            dist.all_reduce(flag, op=dist.ReduceOp.MIN)
            ok = int(flag.item())
        if not ok:
            if rank == 0:
                print("bench.py: --shard p2p: a peer GPU's buffers cannot be mapped (no P2P access"
                      + (": " + why if "why" in dir() else "") + "); falling back to --shard allgather", file=sys.stderr)
            args.shard = "allgather"

    def p2p_barrier(stream_ptr):         # every rank's enqueued work complete, then a cross-rank barrier
        stream.synchronize()
        if world > 1:
            dist.barrier(device_ids=[local])
        return 0

    def step():
        if args.shard == "p2p":    # ONE expansion over all ranks, exchange fused into the epilogue
            return h.expand_sharded_p2p(H, nocc, rfoe.SP2, tol, P=P, barrier=p2p_barrier, stream=stream)
        if shard:                  # the same with pack + one NCCL all-gather + unpack per step
            return h.expand_sharded(H, nocc, rfoe.SP2, tol, P=P, rank=rank, world=world, stream=stream)
        return h.expand(H, nocc, rfoe.SP2, tol, P=P, stream=stream)

    # ---- device-resident arm: W warm-up steps, then exactly K timed steps
    res = None
    for _ in range(args.warmup):
        res = step()
    gpu_id = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid).replace("GPU-", "")
    sampler = ClockSampler(gpu_id)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sq_ms = sq_n = launches = 0
    barrier()
    sampler.start()
    ev0.record(stream)
    for _ in range(args.steps):
        res = step()
        sq_ms += res.square_ms
        sq_n += res.square_launches
        launches += res.gpu_launches
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_local = ev0.elapsed_time(ev1)
    if not (res.converged and abs(float(torch.diagonal(P).sum().item()) - nocc) < 1e-6):
        raise SystemExit(f"bench.py: expansion did not converge to a projector (status {res.status})")
    iters = res.iterations
    fl_sq = executed_flops_per_squaring(k)
    fl_step = iters * fl_sq
    ms_total, value = whole_job_rate(ms_local, args.steps * fl_step / (world if shard else 1), dev)

    # ---- end-to-end arm: host buffers through rfoe_expand_host (H2D of H^p and D2H of P inside the timed region)
    Hh = torch.empty((k, k), dtype=torch.float64, pin_memory=True)
    Hh.copy_(H)
    Ph = torch.empty((k, k), dtype=torch.float64, pin_memory=True)
    h.expand_host(Hh, nocc, rfoe.SP2, tol, P=Ph, stream=stream)          # warm-up (allocates the staging buffers)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        r2 = h.expand_host(Hh, nocc, rfoe.SP2, tol, P=Ph, stream=stream)
        launches_e2e = r2.gpu_launches
    e1.record(stream)
    barrier()
    ms2, e2e_value = whole_job_rate(e0.elapsed_time(e1), args.steps * r2.iterations * fl_sq, dev)
    if shard:     # the host-buffer arm runs per-rank replicas; a sharded job is one expansion, so quote one rank's rate
        e2e_value /= world
    assert abs(float(Ph.diagonal().sum()) - nocc) < 1e-6

    if rank == 0:
        avg_launch_ms = sq_ms / max(sq_n, 1)
        fl_launch = fl_sq / (world if shard else 1)      # a sharded launch squares 1/world of the tiles
        achieved = fl_launch / (avg_launch_ms * 1e-3) / 1e12
        # the denominator, measured by this run (outside the timed region, device still warm), with its own clock sample
        psamp = ClockSampler(gpu_id).start()
        peak_probe, dgemm_tf = fp64_peaks(h, torch, stream)
        pclk = psamp.stop()
        traffic = NCU_TRAFFIC_BYTES.get(k)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json config {args.config}: k={k}, nocc={nocc}, SP2, stop rule A tol {tol:.3g}, "
                                   "Gershgorin bounds, H^p = Q diag(lambda) Q^T seeded",
                       "parallelism": (f"sharded ({args.shard}): one expansion over {world} GPUs, tile ranges, "
                                        + ("epilogue stores to every rank over peer memory + one barrier per step" if args.shard == "p2p"
                                           else "one NCCL all-gather per step") if shard
                                       else "replicas only: one independent expansion per GPU, no collective"),
                       "l2": f"inputs larger than L2 (each matrix {8.0 * k * k / 1e6:.0f} MB vs 126 MB L2); no flush needed",
                       "squarings_per_expansion": iters, "branch": res.branch},
            "seconds_per_expansion": ms_total / args.steps / 1e3,
            "gemm_equiv_tflops": (1 if shard else world) * args.steps * iters * 2.0 * k ** 3 / (ms_total * 1e-3) / 1e12,
            "square_share_of_step": sq_ms / ms_total if world == 1 else None,
            "roofline": {"bound": "tensor", "kernel": "sym_square_kernel<0> (FP64 DMMA.8x8x4)", "achieved": achieved,
                         "peak": peak_probe, "unit": "TFLOP/s", "frac": achieved / peak_probe,
                         "traffic": traffic[0] if traffic else None, "traffic_source": traffic[1] if traffic else None,
                         "avg_launch_ms": avg_launch_ms, "launches_timed": sq_n, "flops_per_launch": fl_launch,
                         "peak_measured": peak_probe, "peak_derived": FP64_PEAK_DERIVED_TFLOPS,
                         "frac_of_derived": achieved / FP64_PEAK_DERIVED_TFLOPS, "cublas_dgemm_tflops": dgemm_tf,
                         "peak_clocks": {"sm_mhz": pclk["sm_mhz"], "reasons": pclk["reasons"], "power_w_max": pclk["power_w_max"]},
                         "peak_source": "measured by this run: rfoe_probe_fp64_peak (register-only DMMA.8x8x4 issue loop, 8 warps x 32 "
                                        "accumulators per SM, ~300 ms) right after the timed region; peak_derived = 148 SM x 64 DFMA/clk "
                                        "x 2 x 1.965 GHz; cublas_dgemm_tflops = torch.matmul FP64 8192^3 (context); MEASURED_PEAKS.json "
                                        "has no FP64 entry"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * k * k, "d2h_bytes_per_step": 8 * k * k,
                    "ms_per_step": ms2 / args.steps},
            "gpu_launches": launches,
            "clocks": {"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"], "reasons": clocks["reasons"],
                       "power_w_max": clocks["power_w_max"], "samples": clocks["samples"]},
        }
        if clocks.get("power_w_mean"):
            # the paper's energy metric is TDP x time, an upper bound; here: mean board power sampled by
            # nvidia-smi during the timed region x seconds per expansion
            sec = ms_total / args.steps / 1e3
            line["energy"] = {"mean_power_w": clocks["power_w_mean"], "joules_per_expansion": clocks["power_w_mean"] * sec,
                              "wh_per_expansion": clocks["power_w_mean"] * sec / 3600.0,
                              "gflops_per_watt": value * 1e3 / clocks["power_w_mean"]}
        if world == 1 and not shard:
            line["hbm_kernels"] = hbm_report(h, H, stream)
            line["lanczos_bounds"] = lanczos_report(h, rfoe, w, H, P, stream, ms_total / args.steps)
        if world == 1 and not shard and not args.no_many:
            line["small_configs_single_expand"] = small_configs_report(rfoe, rfoe_inputs, local, peak_probe)
            line["many_small_problems"] = many_report(rfoe, rfoe_inputs, local)
        if want_reduced:
            line["reduced_precision"] = reduced_report(h, rfoe, w, H, P, stream, ms_total / args.steps)
        if world == 1 and not args.no_subspace and k <= 16384:   # 59 GB of basis + generator temporaries: not beside config 5
            del Hh, Ph
            with rfoe.Rfoe(args.subspace_k, device=local) as h2:
                line["subspace_steps"] = subspace_report(h2, rfoe, rfoe_inputs, args, dev, stream)
        if world == 1 and not args.no_cpu_baseline:
            dt, fl, its, ws = oracle_sample(args.config, args.cpu_k)
            line["cpu_baseline"] = {
                "value": fl / dt / 1e12, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "seconds": dt,
                "sample": f"config {args.config} construction scaled to k={ws.k}, nocc={ws.nocc}: one full SP2 expansion "
                          f"({its} squarings); oracle flops = k^2(k+1) per squaring"}
        print(json.dumps(line), flush=True)
    h.close()
    if dist.is_initialized():
        dist.destroy_process_group()
    return 0


def small_configs_report(rfoe, rfoe_inputs, local, peak_tflops):
    """BASELINE configs 1 and 2 (k=256, k=2048) as ONE rfoe_expand each -- the call north_star specifies -- on the default
    path (the whole recursion in one persistent launch, RFOE_OPT_RESIDENT) and on the launch-per-step path, CUDA-event time
    of the best of 5 warm runs; executed-flop rate against the probe's FP64 peak."""
    import torch

    out = {}
    for c in (1, 2):
        w = rfoe_inputs.make_workload(c)
        H = torch.from_numpy(w.H).cuda(local)
        P = torch.empty_like(H)
        fl = executed_flops_per_squaring(w.k)
        row = {}
        with rfoe.Rfoe(w.k, device=local) as h:
            for name, resident in (("resident", True), ("launch_per_step", False)):
                h.configure(resident=resident)
                best = None
                for i in range(7):
                    r = h.expand(H, w.nocc, rfoe.SP2, w.tol, P=P)
                    if i >= 2 and (best is None or r.device_ms < best.device_ms):
                        best = r
                tf = best.iterations * fl / (best.device_ms * 1e-3) / 1e12
                row[name] = {"ms_per_expansion": best.device_ms, "squarings": best.iterations,
                             "us_per_step": best.device_ms / best.iterations * 1e3, "tflops_executed": tf,
                             "frac_of_fp64_peak": tf / peak_tflops, "gpu_launches": best.gpu_launches,
                             "converged": bool(best.converged)}
                if resident:
                    row[name]["phase_us_per_step"] = [x / best.iterations * 1e3 for x in best.resident_phase_ms]
        out[f"config{c}_k{w.k}"] = row
    return out


def many_report(rfoe, rfoe_inputs, local):
    """Reported separately ("throughput over independent H^p (k-points, spins)"): BASELINE configs 1 and 2 are too
    small to fill the chip one at a time; rfoe_expand_many runs independent copies side by side on one GPU (one handle,
    stream and host thread each).  Wall-clock rate of a batch after one warm batch, against the lone-handle rate."""
    import time

    import torch

    out = {}
    for c, n_handles, n_problems in ((1, 16, 128), (2, 4, 32)):
        w = rfoe_inputs.make_workload(c)
        H = torch.from_numpy(w.H).cuda(local)
        m = (w.k + TILE - 1) // TILE
        rates = {}
        for nh in (1, n_handles):
            handles = [rfoe.Rfoe(w.k, device=local) for _ in range(nh)]
            streams = [torch.cuda.Stream() for _ in range(nh)]
            Ps = [torch.empty_like(H) for _ in range(n_problems)]
            probs = [(H, w.nocc, w.tol, Ps[j]) for j in range(n_problems)]
            rfoe.expand_many(handles, probs, rfoe.SP2, streams)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            res = rfoe.expand_many(handles, probs, rfoe.SP2, streams)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            rates[nh] = n_problems / dt
            its = res[0].iterations
            for hh in handles:
                hh.close()
            del Ps, probs, res
        out[f"config{c}_k{w.k}"] = {
            "handles": n_handles, "problems": n_problems, "squarings_per_expansion": its,
            "expansions_per_s": rates[n_handles], "expansions_per_s_one_handle": rates[1],
            "speedup": rates[n_handles] / rates[1],
            "tflops_executed": rates[n_handles] * its * executed_flops_per_squaring(w.k) / 1e12,
            "timing": "host wall clock around one rfoe_expand_many batch (device idle before and after)"}
    return out


def hbm_report(h, H, stream):
    """HBM GB/s of the bound kernels, live: rfoe_bounds = gershgorin_rows_kernel (8 k^2 bytes read) + a
    one-block reduction, CUDA events around the call (best of 5), against the measured copy peak."""
    import torch

    k = H.shape[0]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = float("inf")
    for _ in range(5):
        torch.cuda.synchronize()
        e0.record(stream)
        h.bounds(H, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    peak = None
    try:
        peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs")
    except (OSError, ValueError):
        pass
    gbs = 8.0 * k * k / (best * 1e-3) / 1e9
    return {"rfoe_bounds_ms": best, "gershgorin_gbs": gbs, "peak_gbs": peak, "frac": gbs / peak if peak else None,
            "note": "whole rfoe_bounds call (rows kernel + reduction + 16-byte D2H); per-kernel figures: profiles/r02_launches_k16384.md"}


def lanczos_report(h, rfoe, w, H, P, stream, fp64_ms, m=24):
    """Information beside the normative Gershgorin run ("iteration count ... with tight bounds"): the
    same FP64 expansion with the optional m-step Lanczos bounds (rfoe_bounds_lanczos, reading R3b)."""
    import torch

    k = w.k
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h.bounds_lanczos(H, m, stream=stream)
    torch.cuda.synchronize()
    e0.record(stream)
    lo, hi = h.bounds_lanczos(H, m, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_b = e0.elapsed_time(e1)
    h.configure(lanczos_steps=m)
    h.expand(H, w.nocc, rfoe.SP2, w.tol, P=P, stream=stream)
    torch.cuda.synchronize()
    e0.record(stream)
    r = h.expand(H, w.nocc, rfoe.SP2, w.tol, P=P, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    h.configure(lanczos_steps=0)
    return {"steps": m, "eps_min": lo, "eps_max": hi, "bounds_ms": ms_b,
            "matvec_gbs": m * 8.0 * k * k / (ms_b * 1e-3) / 1e9, "seconds_per_expansion": ms / 1e3,
            "squarings": r.iterations, "converged": bool(r.converged), "speedup_vs_gershgorin": fp64_ms / ms,
            "trace_error": abs(float(torch.diagonal(P).sum()) - w.nocc)}


_scratch = {}


def H_scratch(like):
    """a second matrix of the same shape (rfoe_square needs out != X); kept between calls"""
    import torch

    key = (tuple(like.shape), like.device)
    if key not in _scratch:
        _scratch.clear()
        _scratch[key] = torch.empty_like(like)
    return _scratch[key]


def reduced_report(h, rfoe, w, H, P, stream, fp64_ms):
    """Row A8, reported separately from the FP64 headline: the same workload through RFOE_VARIANT_SP2_MIXED with
    the paper's schedule (reduced-precision squarings -- three FP16-part products on tcgen05 -- from the first step until
    RelTr <= 5e-4, FP64 afterwards).  Accuracy is measured against the construction-exact
    projector Q_occ Q_occ^T and the exact band energy (harness algebra in torch)."""
    import torch

    k, nocc = w.k, w.nocc
    Q = w.Q if isinstance(w.Q, torch.Tensor) else torch.from_numpy(w.Q).to(H.device)
    Qo = Q[:, :nocc]
    Pex = Qo @ Qo.T
    h.configure(mixed_head=0.0, mixed_reltr=5e-4)
    h.expand(H, nocc, rfoe.SP2_MIXED, w.tol, P=P, stream=stream)                    # warm-up (allocates the FP32 copies)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    r = h.expand(H, nocc, rfoe.SP2_MIXED, w.tol, P=P, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    err = torch.linalg.norm(P - Pex).item() / math.sqrt(k)
    eband = w.band_energy()
    # same path with the switch to FP64 moved from the paper's RelTr <= 5e-4 to 5e-7
    h.configure(mixed_head=0.0, mixed_reltr=5e-7)
    h.expand(H, nocc, rfoe.SP2_MIXED, w.tol, P=P, stream=stream)
    torch.cuda.synchronize()
    e0.record(stream)
    r_late = h.expand(H, nocc, rfoe.SP2_MIXED, w.tol, P=P, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_late = e0.elapsed_time(e1)
    late = {"switch_reltr": 5e-7, "seconds_per_expansion": ms_late / 1e3, "speedup_vs_fp64": fp64_ms / ms_late,
            "iterations": r_late.iterations, "reduced_steps": r_late.fp32_steps, "converged": bool(r_late.converged),
            "errP_vs_exact_projector": torch.linalg.norm(P - Pex).item() / math.sqrt(k),
            "rel_band_energy_error": abs(r_late.tr_PH - eband) / abs(eband)}
    h.configure(mixed_reltr=5e-4)
    # one reduced squaring (split pass + product kernel) of the final P, in both forms of the kernel, interleaved
    sq = {"pair": [], "single_cta": []}
    for it in range(6):
        for name, flag in (("single_cta", False), ("pair", True)):
            h.configure(reduced_pair=flag)
            _, _, ms_sq = h.square(P, -1.0, 2.0, 0.0, out=H_scratch(P), stream=stream, reduced=True)
            if it:
                sq[name].append(ms_sq)
    h.configure(reduced_pair=True)
    flops3 = 3.0 * executed_flops_per_squaring(k)
    squaring = {name: {"ms": sorted(v)[len(v) // 2], "tflops_executed_f16": flops3 / (sorted(v)[len(v) // 2] * 1e-3) / 1e12} for name, v in sq.items()}
    _scratch.clear()
    squaring["note"] = ("rfoe_square_reduced on the converged P, CUDA events around split pass + product kernel, median of 5; pair = "
                        "tcgen05.mma.cta_group::2 (default), single_cta = RFOE_OPT_REDUCED_PAIR 0; a kernel timed alone, not the "
                        "power-capped sustained rate of the expansion above")
    return {"variant": "SP2_MIXED, paper schedule (reduced precision until RelTr <= 5e-4)", "dtype": "3xFP16 parts (tcgen05 kind::f16, FP32 accumulate, FP64 epilogue) + f64",
            "reduced_squaring": squaring,
            "seconds_per_expansion": ms / 1e3, "speedup_vs_fp64": fp64_ms / ms, "iterations": r.iterations,
            "reduced_steps": r.fp32_steps, "converged": bool(r.converged),
            "errP_vs_exact_projector": err, "rel_band_energy_error": abs(r.tr_PH - eband) / abs(eband),
            "tolerances": {"errP": 1e-6, "band_energy": 1e-8}, "late_switch": late}


def subspace_report(h, rfoe, rfoe_inputs, args, dev, stream):
    """SURVEY.md 8(f) NEXT-4, reported separately from the headline: the steps either side of the expansion on a
    synthetic Rayleigh-Ritz input with the paper's proportions (N is 0.1-0.5 % of M; the subspace is
    ~1.3 N): the config's spectrum scaled to k = 4096 (nocc = 3150), M = 600000 degrees of freedom.
    rfoe_project (H^p = Psi HPsi^T) -> rfoe_expand -> rfoe_apply (Y = P Psi, rho = diag(Psi^T P Psi)), each timed
    with CUDA events on the launching stream; checks against the generator's own closed forms (harness algebra)."""
    import torch

    k, M = args.subspace_k, args.subspace_m
    sub = rfoe_inputs.make_subspace(args.config, k=k, M=M, device=str(dev))
    w = sub.w
    Hp = torch.empty((k, k), dtype=torch.float64, device=dev)
    P = torch.empty_like(Hp)
    Y = torch.empty_like(sub.Psi)
    m = (k + TILE - 1) // TILE
    fl_proj = 2.0 * M * (m * (m + 1) // 2) * TILE * TILE            # executed: upper tiles only
    fl_apply = 2.0 * M * float(m * TILE) ** 2                        # executed: P zero-padded to tiles
    out = {"workload": f"config {args.config} spectrum scaled to k={k}, nocc={w.nocc}; M={M} (nocc/M = {100.0 * w.nocc / M:.2f} %); "
                       "Psi = thin QR of seeded N(0,1), HPsi = H^p Psi + 10 % out-of-subspace residual",
           "bytes_resident": 3 * 8 * k * M}
    ms_p = ms_a = tot_e = None
    for it in range(2):                                              # first pass warms up (workspaces, tile maps)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        torch.cuda.synchronize()
        e[0].record(stream)
        _, (tr, ss), ms_p = h.project(sub.Psi, sub.HPsi, out=Hp, stream=stream)
        e[1].record(stream)
        res = h.expand(Hp, w.nocc, rfoe.SP2, w.tol, P=P, stream=stream)
        e[2].record(stream)
        _, rho, ms_a = h.apply(P, sub.Psi, out=Y, density=True, stream=stream)
        e[3].record(stream)
        torch.cuda.synchronize()
        tot_p, tot_e, tot_a = e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2]), e[2].elapsed_time(e[3])
    Hw = w.H if isinstance(w.H, torch.Tensor) else torch.from_numpy(w.H).to(dev)
    Q = w.Q if isinstance(w.Q, torch.Tensor) else torch.from_numpy(w.Q).to(dev)
    Qo = Q[:, : w.nocc]
    rho_exact = ((Qo.T @ sub.Psi) ** 2).sum(dim=0)
    out.update({
        "project": {"kernel": "sym_square_kernel<2> + project_reduce_kernel", "ms": ms_p, "ms_call": tot_p,
                    "tflops_executed": fl_proj / ms_p / 1e9, "frac_fp64_peak_derived": fl_proj / ms_p / 1e9 / FP64_PEAK_TFLOPS,
                    "max_abs_err_vs_construction": float((Hp - Hw).abs().max()), "bitwise_symmetric": bool(torch.equal(Hp, Hp.T))},
        "expand": {"ms": tot_e, "iterations": res.iterations, "converged": bool(res.converged)},
        "apply": {"kernel": "apply_kernel (+ density kernels in ms_call)", "ms": ms_a, "ms_call": tot_a,
                  "tflops_executed": fl_apply / ms_a / 1e9, "frac_fp64_peak_derived": fl_apply / ms_a / 1e9 / FP64_PEAK_TFLOPS,
                  "electron_count_error": abs(float(rho.sum()) - w.nocc),
                  "max_abs_density_err_vs_construction": float((rho - rho_exact).abs().max())},
        "seconds_chain": (tot_p + tot_e + tot_a) / 1e3,
    })
    return out


def run_matrix(args) -> int:
    """--run-matrix: the run matrix of SURVEY.md section 8(d) / DESIGN.md section 8 -- every BASELINE.json config through the
    C ABI in each variant that applies, CUDA-event time of the second (warm) run, accuracy against the construction-exact
    projector (harness algebra in torch).  Prints one table row per (config, run); not a bench line."""
    import torch

    import paper_2301_04642_b200 as rfoe
    import rfoe_inputs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py --run-matrix: no CUDA device -- there is no CPU fallback")
    sep = " | " if args.markdown else "  "
    cols = ["config", "k", "run", "steps", "mults", "reduced", "resident", "ms", "TFLOP/s", "errP", "dE", "status"]
    print(sep.join(cols))
    if args.markdown:
        print(sep.join("---" for _ in cols))
    for c in args.matrix_configs:
        w = rfoe_inputs.make_workload(c, device="cuda")
        k, nocc = w.k, w.nocc
        H = w.H if isinstance(w.H, torch.Tensor) else torch.from_numpy(w.H).cuda()
        Q = w.Q if isinstance(w.Q, torch.Tensor) else torch.from_numpy(w.Q).cuda()
        Pex = Q[:, :nocc] @ Q[:, :nocc].T
        del Q
        w.Q = None
        eband = w.band_energy()
        fl_sq = executed_flops_per_squaring(k)
        lam = w.lam
        homo, lumo = float(lam[:nocc].max()), float(lam[nocc:].min())
        runs = [("SP2 rule A, Gershgorin (normative)", rfoe.SP2, w.tol, {}),
                ("the same, one launch sequence per step (RFOE_OPT_RESIDENT = 0)", rfoe.SP2, w.tol, dict(resident=False)),
                ("SP2 rule B RelTr 5e-8 (paper's criterion)", rfoe.SP2, 5e-8, dict(stop_rule=rfoe.RULE_B)),
                ("SP2 rule A, exact spectral bounds", rfoe.SP2, w.tol, dict(bounds=(float(lam.min()), float(lam.max())))),
                ("SP2 rule A, Lanczos bounds (24 steps, on the device)", rfoe.SP2, w.tol, dict(lanczos_steps=24)),
                ("mixed (late switch 5e-7) + Lanczos bounds", rfoe.SP2_MIXED, w.tol, dict(lanczos_steps=24, mixed_head=0.0, mixed_reltr=5e-7)),
                ("A-Z-RFOE (accelerated), exact HOMO/LUMO", rfoe.SP2_ACCEL, w.tol, dict(homo=homo, lumo=lumo)),
                ("A-Z-RFOE, HOMO/LUMO estimated from the normative run's history", rfoe.SP2_ACCEL, w.tol, "estimated"),
                ("McWeeny-style tail", rfoe.MCWEENY, w.tol, {}),
                ("mixed, paper schedule (reduced until RelTr 5e-4)", rfoe.SP2_MIXED, w.tol, dict(mixed_head=0.0, mixed_reltr=5e-4)),
                ("T-RFOE, m = 30 (fractional occupancies: errP is the distance to the zero-temperature projector)", rfoe.TRUNC, 0.0,
                 dict(trunc_steps=30)),
                ("mixed T-RFOE, m = 30", rfoe.TRUNC_MIXED, 0.0, dict(trunc_steps=30, mixed_head=0.0, mixed_reltr=5e-4))]
        est = None
        with rfoe.Rfoe(k) as h:
            for name, variant, tol, opts in runs:
                h.configure(stop_rule=rfoe.RULE_A, bounds=False, mixed_head=0.0, mixed_reltr=5e-4, lanczos_steps=0, resident=True)
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
                row = [str(c), str(k), name, str(r.iterations), str(r.multiplications), str(r.fp32_steps), "yes" if r.resident else "no",
                       f"{r.device_ms:.3f}", f"{tf:.1f}", f"{err:.2e}", f"{dE:.1e}", "ok" if r.converged else "not converged"]
                print(sep.join(row), flush=True)
                del P, r
        del H, Pex
        torch.cuda.empty_cache()
    return 0


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-k", type=int, default=2048, help="size of the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-reduced", action="store_true", help="skip the separately reported reduced-precision run")
    ap.add_argument("--shard", nargs="?", const="p2p", default=None, choices=["p2p", "allgather"],
                    help="N > 1: shard ONE expansion over the ranks (strong scaling) instead of independent replicas; p2p (default): "
                         "epilogue stores to all ranks' memory over NVLink + one barrier per step; allgather: NCCL all-gather per step")
    ap.add_argument("--no-many", action="store_true", help="skip the separately reported many-small-problems run")
    ap.add_argument("--no-subspace", action="store_true", help="skip the separately reported Rayleigh-Ritz / apply steps")
    ap.add_argument("--only-subspace", action="store_true", help="run only the Rayleigh-Ritz / apply chain (ncu captures)")
    ap.add_argument("--subspace-k", type=int, default=4096)
    ap.add_argument("--subspace-m", type=int, default=600000)
    ap.add_argument("--run-matrix", action="store_true", help="print the run matrix (every config x variant) instead of the bench line")
    ap.add_argument("--matrix-configs", type=int, nargs="+", default=[1, 2, 3, 4])
    ap.add_argument("--markdown", action="store_true")
    args = ap.parse_args()
    if args.run_matrix:
        return run_matrix(args)
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
