"""Host logic of the persistent-kernel paths (csrc/resident.cuh, resident_small.cuh) on CPU: which path a
size takes and, for the stream-K kernel, that the ranges of chunk units partition the step and that the table of split tiles
says exactly what a brute-force walk over the ranges says.  rfoe_plan_resident is a host-only C call (no device)."""
import pytest

import paper_2301_04642_b200 as rfoe


@pytest.mark.parametrize("k,path,grid", [(1, 1, 10), (128, 1, 10), (256, 1, 36), (512, 1, 136), (513, 2, 55), (1024, 2, 136),
                                          (1025, 3, 148), (2048, 3, 148), (4096, 3, 148), (4097, 0, 0), (16384, 0, 0)])
def test_which_path(k, path, grid):
    d = rfoe.plan_resident(k, 148)
    assert (d["path"], d["grid"]) == (path, grid)
    m = -(-k // 128)
    if path in (0, 3):
        assert d["n_tiles"] == m * (m + 1) // 2
    else:
        bm = 32 if path == 1 else 64
        mt = m * 128 // bm
        assert d["n_tiles"] == mt * (mt + 1) // 2 == d["grid"]          # one output tile per CTA, all co-resident


def test_small_kernel_needs_one_sm_per_tile():
    assert rfoe.plan_resident(512, 132)["path"] == 0                     # 136 tiles do not fit 132 SMs: launch per step
    assert rfoe.plan_resident(256, 36)["path"] == 1
    with pytest.raises(rfoe.RfoeError):
        rfoe.plan_resident(0, 148)
    with pytest.raises(rfoe.RfoeError):
        rfoe.plan_resident(256, 0)


@pytest.mark.parametrize("sm", [148, 132, 64, 7])
@pytest.mark.parametrize("k", [1100, 1536, 2048, 2100, 3000, 3333, 4096])
def test_stream_k_ranges_partition_the_step(k, sm):
    d = rfoe.plan_resident(k, sm)
    assert d["path"] == 3
    G, KT, nt, bnd = d["grid"], d["kt"], d["n_tiles"], d["boundaries"]
    U = nt * KT
    assert G == min(sm, U) and KT == -(-k // 128) * 128 // 16
    assert bnd[0] == 0 and bnd[-1] == U and len(bnd) == G + 1
    assert all(b1 > b0 for b0, b1 in zip(bnd, bnd[1:]))                  # no empty range
    lens = [b1 - b0 for b0, b1 in zip(bnd, bnd[1:])]
    # equal cost: chunk counts differ by at most one epilogue's worth per whole tile held (+1 for rounding)
    whole_per_cta = [sum(1 for t in range(b0 // KT, -(-b1 // KT)) if t * KT >= b0 and (t + 1) * KT <= b1) for b0, b1 in zip(bnd, bnd[1:])]
    cost10 = [ln + 10 * w for ln, w in zip(lens, whole_per_cta)]
    assert max(lens) - min(lens) <= 1 or max(cost10) - min(cost10) <= 11
    # brute force: who holds what
    holders = {t: [] for t in range(nt)}
    for b in range(G):
        for t in range(bnd[b] // KT, (bnd[b + 1] - 1) // KT + 1):
            holders[t].append(b)
    split = {t: (b0, n) for t, b0, n in d["split_tiles"]}
    assert d["n_split"] == len(split)
    # a boundary between two CTAs cuts at most one tile: fewer split tiles than CTAs, hence at most ONE 16-row fix-up band per
    # warp (8 bands per split tile, 8 warps per CTA) -- resident.cuh's FIX phase relies on it
    assert d["n_split"] < G
    for t in range(nt):
        hs = holders[t]
        assert hs == list(range(hs[0], hs[0] + len(hs)))                 # consecutive CTAs
        if len(hs) == 1:
            assert t not in split                                        # whole tile: register epilogue
        else:
            assert split[t] == (hs[0], len(hs))                          # finished in the fix-up phase: first holder, count
            # the first holder's segment starts the tile, every later one continues it (the slot rule of resident.cuh)
            assert bnd[hs[0]] <= t * KT and all(bnd[b] > t * KT for b in hs[1:])
    # every chunk unit of every tile is covered exactly once
    assert sum(lens) == U
