"""GPU test of the sharded expansion (rfoe_expand_sharded) on ONE GPU.

Only one GPU is available to the tests, so the g ranks run as g host threads of one process, each with its own
librfoe handle and CUDA stream; the exchange callback is host-synchronous (stream sync, thread barrier,
device-to-device copies, stream sync, barrier), so no kernel ever waits on another kernel.  What is checked is what
the design promises: every rank's P is BITWISE the single-GPU P, with the same iteration count, branch string and
scalars, and the single-GPU result is itself compared with the CPU oracle at the north_star tolerances."""
import math
import threading

import numpy as np
import pytest
import torch

import oracle
import paper_2301_04642_b200 as rfoe
import rfoe_inputs

pytestmark = pytest.mark.gpu


class _LocalWorld:
    """All-gather between g threads sharing one device."""

    def __init__(self, g):
        self.g = g
        self.bar = threading.Barrier(g, timeout=120)
        self.send = [None] * g

    def allgather_for(self, rank):
        def ag(send_ptr, recv_ptr, nbytes, stream_ptr):
            st = torch.cuda.ExternalStream(stream_ptr) if stream_ptr else torch.cuda.default_stream()
            st.synchronize()                                   # my send block is complete
            self.send[rank] = torch.as_tensor(rfoe._DevBytes(send_ptr, nbytes), device="cuda")
            self.bar.wait()
            recv = torch.as_tensor(rfoe._DevBytes(recv_ptr, nbytes * self.g), device="cuda")
            with torch.cuda.stream(st):
                for r in range(self.g):
                    recv[r * nbytes:(r + 1) * nbytes].copy_(self.send[r])
            st.synchronize()
            self.bar.wait()                                    # nobody reuses a send block before all have copied it
            return 0
        return ag


def _run_sharded(H, nocc, variant, tol, g, configure=None):
    world = _LocalWorld(g)
    out, errs = [None] * g, []

    def work(rank):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st), rfoe.Rfoe(H.shape[0]) as h:
                if configure:
                    h.configure(**configure)
                out[rank] = h.expand_sharded(H, nocc, variant, tol, rank=rank, world=g, allgather=world.allgather_for(rank),
                                             stream=st)
                st.synchronize()
        except BaseException as e:  # noqa: BLE001
            errs.append(e)
            world.bar.abort()

    th = [threading.Thread(target=work, args=(r,)) for r in range(g)]
    [t.start() for t in th]
    [t.join(300) for t in th]
    if errs:
        raise errs[0]
    return out


@pytest.mark.parametrize("c,k,g", [(1, 200, 2), (2, 333, 3), (3, 640, 2), (2, 130, 5), (1, 100, 4)])
def test_sharded_equals_single_gpu_bitwise(c, k, g):
    w = rfoe_inputs.make_workload(c, k=k)
    H = torch.from_numpy(w.H).cuda()
    with rfoe.Rfoe(k) as h:
        h.configure(resident=False)      # the sharded run reproduces the bits of the launch-per-step path (same tiles, same order)
        one = h.expand(H, w.nocc, rfoe.SP2, w.tol)
    ref = oracle.expand(w.H, w.nocc, tol=w.tol)
    assert one.iterations == ref.iterations
    assert np.linalg.norm(one.P.cpu().numpy() - ref.P) / math.sqrt(k) <= 1e-10
    res = _run_sharded(H, w.nocc, rfoe.SP2, w.tol, g)
    for r in res:
        assert r.converged and r.iterations == one.iterations and r.branch == one.branch
        assert torch.equal(r.P, one.P)                                     # bitwise
        assert np.array_equal(r.t, one.t) and np.array_equal(r.s, one.s) and np.array_equal(r.e, one.e)
        assert r.tr_PH == one.tr_PH


def test_sharded_world1_and_accelerated_and_truncated():
    w = rfoe_inputs.make_workload(2, k=333)
    H = torch.from_numpy(w.H).cuda()
    homo, lumo = float(w.lam[: w.nocc].max()), float(w.lam[w.nocc:].min())
    with rfoe.Rfoe(333) as h:
        h.configure(homo=homo, lumo=lumo, resident=False)
        one = h.expand(H, w.nocc, rfoe.SP2_ACCEL, w.tol)
    assert torch.equal(_run_sharded(H, w.nocc, rfoe.SP2_ACCEL, w.tol, 1, dict(homo=homo, lumo=lumo))[0].P, one.P)
    for r in _run_sharded(H, w.nocc, rfoe.SP2_ACCEL, w.tol, 2, dict(homo=homo, lumo=lumo)):
        assert r.iterations == one.iterations and torch.equal(r.P, one.P)
    with rfoe.Rfoe(333) as h:                                              # T-RFOE: m = 12 steps, no stop test
        h.configure(max_iter=12, resident=False)
        trunc = h.expand(H, w.nocc, rfoe.SP2, 0.0)
    for r in _run_sharded(H, w.nocc, rfoe.SP2, 0.0, 3, dict(max_iter=12)):
        assert r.iterations == 12 and not r.converged and torch.equal(r.P, trunc.P)


def test_sharded_rejects_unsupported_variants_and_failing_exchange():
    w = rfoe_inputs.make_workload(1, k=100)
    H = torch.from_numpy(w.H).cuda()
    with rfoe.Rfoe(100) as h:
        with pytest.raises(rfoe.RfoeError) as e:
            h.expand_sharded(H, w.nocc, rfoe.MCWEENY, w.tol, rank=0, world=1, allgather=lambda *a: 0)
        assert e.value.status == rfoe.ERR_UNSUPPORTED
        with pytest.raises(rfoe.RfoeError):
            h.expand_sharded(H, w.nocc, rfoe.SP2, w.tol, rank=2, world=2, allgather=lambda *a: 0)
        with pytest.raises(ZeroDivisionError):                            # an exception in the callback surfaces in Python
            h.expand_sharded(H, w.nocc, rfoe.SP2, w.tol, rank=0, world=1, allgather=lambda *a: 1 // 0)


# ---------------------------------------------------------------------------------------------------------------
# the exchange fused into the squaring kernel: epilogue stores go to every rank's X_{n+1} (peer memory)
def _run_p2p_threads(H, nocc, variant, tol, g, configure=None):
    """g ranks as threads of this process: raw device pointers stand in for peer-mapped ones (same GPU)."""
    bar = threading.Barrier(g, timeout=120)
    handles = [rfoe.Rfoe(H.shape[0]) for _ in range(g)]
    ptrs = [p for h in handles for p in h.shard_local_ptrs()]
    out, errs = [None] * g, []

    def work(rank):
        try:
            torch.cuda.set_device(0)
            h = handles[rank]
            h.shard_set_peers(rank, g, ptrs)
            if configure:
                h.configure(**configure)
            st = torch.cuda.Stream()

            def barrier(stream_ptr):
                st.synchronize()
                bar.wait()
                return 0

            with torch.cuda.stream(st):
                out[rank] = h.expand_sharded_p2p(H, nocc, variant, tol, barrier=barrier, stream=st)
                st.synchronize()
        except BaseException as e:  # noqa: BLE001
            errs.append(e)
            bar.abort()

    th = [threading.Thread(target=work, args=(r,)) for r in range(g)]
    [t.start() for t in th]
    [t.join(300) for t in th]
    [h.close() for h in handles]
    if errs:
        raise errs[0]
    return out


@pytest.mark.parametrize("c,k,g", [(1, 200, 2), (2, 333, 3), (3, 640, 2), (2, 130, 5), (3, 1024, 4), (1, 100, 1)])
def test_p2p_sharded_equals_single_gpu_bitwise(c, k, g):
    w = rfoe_inputs.make_workload(c, k=k)
    H = torch.from_numpy(w.H).cuda()
    with rfoe.Rfoe(k) as h:
        h.configure(resident=False)
        one = h.expand(H, w.nocc, rfoe.SP2, w.tol)
    for r in _run_p2p_threads(H, w.nocc, rfoe.SP2, w.tol, g):
        assert r.converged and r.iterations == one.iterations and r.branch == one.branch
        assert torch.equal(r.P, one.P)
        assert np.array_equal(r.t, one.t) and np.array_equal(r.s, one.s) and np.array_equal(r.e, one.e)


def _ipc_worker(rank, world, port, k, c, out):
    import os
    import torch.distributed as dist

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    w = rfoe_inputs.make_workload(c, k=k)
    H = torch.from_numpy(w.H).cuda()
    with rfoe.Rfoe(k) as h:
        h.shard_connect()
        first = h.expand_sharded_p2p(H, w.nocc, rfoe.SP2, w.tol)
        P_first = first.P.clone()
        # a second expansion straight after the first, one rank late: the entry barrier of rfoe_expand_sharded_p2p must keep
        # the early rank's first stores out of buffers the late rank's previous call could still be reading
        if rank == 1:
            import time
            time.sleep(0.05)
        res = h.expand_sharded_p2p(H, w.nocc, rfoe.SP2, w.tol)
        torch.cuda.synchronize()
        out[f"repeat{rank}"] = bool(torch.equal(res.P, P_first)) and res.branch == first.branch
        dist.barrier()
        if rank == 0:
            h.configure(resident=False)
            one = h.expand(H, w.nocc, rfoe.SP2, w.tol)
            out["single"] = (one.iterations, one.branch)
            out["equal"] = bool(torch.equal(one.P, res.P))
        out[rank] = (res.iterations, res.branch, bool(res.converged), float(torch.diagonal(res.P).sum()))
        dist.barrier()
    dist.destroy_process_group()


def test_p2p_sharded_two_processes_ipc_handles():
    """One process per rank, CUDA IPC handles exchanged over torch.distributed (gloo), both ranks on the one GPU the
    test box has: exercises rfoe_shard_ipc_export / _import and the default barrier."""
    import socket

    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    k, c, world = 333, 2, 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_ipc_worker, args=(world, port, k, c, out), nprocs=world, join=True)
        res = dict(out)
    w = rfoe_inputs.make_workload(c, k=k)
    assert res["equal"] and res["repeat0"] and res["repeat1"]      # the second of two back-to-back calls gives the same bits
    for r in range(world):
        it, br, conv, tr = res[r]
        assert conv and (it, br) == res["single"] and abs(tr - w.nocc) < 1e-9
