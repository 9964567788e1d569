"""Host logic of the sharded expansion on CPU: the tile partition
(rfoe_shard_range, a host-only C call) single-process and across a world_size-2 gloo group."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("n_tiles,world", [(1, 1), (1, 4), (3, 2), (10, 4), (528, 8), (8256, 8), (8256, 7), (49141, 6)])
def test_shard_ranges_partition_the_tile_list(n_tiles, world):
    import paper_2301_04642_b200 as rfoe

    c_max = -(-n_tiles // world)
    nxt = 0
    for r in range(world):
        b, c = rfoe.shard_range(n_tiles, r, world)
        assert b == min(r * c_max, n_tiles)            # rank r's block starts at r * c_max in the gathered buffer
        assert b == nxt or c == 0
        assert 0 <= c <= c_max
        nxt = b + c
    assert nxt == n_tiles
    with pytest.raises(rfoe.RfoeError):
        rfoe.shard_range(n_tiles, world, world)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_tiles, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2301_04642_b200 as rfoe

    b, c = rfoe.shard_range(n_tiles, rank, world)
    # the exchange step in miniature: every rank contributes a block of c_max slots holding the global indices of
    # its tiles (padding = -1); the gathered buffer must list 0..n_tiles-1 in order, padding only at the end
    c_max = -(-n_tiles // world)
    send = torch.full((c_max,), -1, dtype=torch.int64)
    send[:c] = torch.arange(b, b + c)
    recv = torch.empty((world * c_max,), dtype=torch.int64)
    dist.all_gather_into_tensor(recv, send)
    out[rank] = recv.tolist()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n_tiles", [5, 528])
def test_gathered_layout_is_global_tile_order_world2(n_tiles):
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, n_tiles, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    got = res[0]
    assert got[:n_tiles] == list(range(n_tiles))
    assert all(v == -1 for v in got[n_tiles:])


def test_squaring_launch_plan():
    """Host logic of the split-K tail: whole waves for the main kernel, a tail only
    where the cycle model gains >= 1.5 %, slices that cover the contraction."""
    import paper_2301_04642_b200 as rfoe

    for k in (1, 100, 256, 1000, 1024, 2048, 4096, 8192, 16384, 40000, 65536):
        nt, nm, sl, per = rfoe.plan_squaring(k)
        m = -(-k // 128)
        kt = m * 128 // 16
        assert nt == m * (m + 1) // 2 and 0 <= nm <= nt
        if sl == 1:
            assert nm == nt and per == kt                 # plain launch
        else:
            assert nm % 148 == 0 and nt - nm > 0          # the main kernel runs whole waves only
            assert per >= 16 and sl * per >= kt and (sl - 1) * per < kt
    assert rfoe.plan_squaring(16384)[2] == 1              # the headline size keeps the plain launch (measured: no gain)
    assert rfoe.plan_squaring(40000)[2] == 1
    nt, nm, sl, per = rfoe.plan_squaring(8192)            # 2080 tiles = 14.05 waves: the 8 left-over tiles are split 16-way
    assert (nt, nm, sl, per) == (2080, 2072, 16, 32)
    assert rfoe.plan_squaring(4096)[:3] == (528, 444, 7)
    with pytest.raises(rfoe.RfoeError):
        rfoe.plan_squaring(0)


def _ipc_layout_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2301_04642_b200 as rfoe

    # stand-ins for the four 64-byte CUDA IPC handles of a rank (W0, W1, records of even / odd steps): byte (q, i) of
    # rank r is 64 r + 16 q + (i % 16), so that every position of the gathered buffer names its source
    mine = bytes((64 * rank + 16 * q + (i % 16)) & 0xFF for q in range(4) for i in range(rfoe.IPC_HANDLE_BYTES))
    out[rank] = rfoe.gather_ipc_handles(mine)
    try:
        rfoe.gather_ipc_handles(mine[:-1])
        out[f"err{rank}"] = False
    except ValueError:
        out[f"err{rank}"] = True
    dist.barrier()
    dist.destroy_process_group()


def test_ipc_handle_gather_layout_world2():
    """rfoe_shard_ipc_import reads `world x 4 x 64` bytes, rank-major (include/rfoe.h): the buffer shard_connect builds over
    the process group must have exactly that order, on every rank."""
    import paper_2301_04642_b200 as rfoe

    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_ipc_layout_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    hb = rfoe.IPC_HANDLE_BYTES
    assert res[0] == res[1] and len(res[0]) == world * 4 * hb
    for r in range(world):
        for q in range(4):
            seg = res[0][(4 * r + q) * hb:(4 * r + q + 1) * hb]
            assert seg == bytes((64 * r + 16 * q + (i % 16)) & 0xFF for i in range(hb))
    assert res["err0"] and res["err1"]
