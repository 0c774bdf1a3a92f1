"""Host logic of the work decomposition (no GPU): the stream-K cut of the pair space that the pairwise kernels follow
(hawkes_plan_segments restates on the host what worker w of a kernel does), for one GPU and for an evaluation sharded
across ranks -- every (tile, streamed event) pair exactly once, loads balanced, partial slots dense per tile and rank."""
import numpy as np
import pytest

import paper_2103_03348_b200 as hp

TILE = 256
# modelled cost per streamed event of the non-symmetric pass 1 (csrc/hawkes.cu W_ALL / W_HEAD, gradient level) and of
# pass 2 (W2_PLAIN past the tile's own events, W2_OWN for its own -- masked -- ones, 16 W2_PLAIN per tile)
W_ALL, W_HEAD = 46, 33
W2_PLAIN, W2_OWN = 4, 5


def expected_range(n, pass_, sym, I):
    i0, i1 = I * TILE, min(n, (I + 1) * TILE)
    if pass_ == 2:
        return i0, n                      # a source tile streams the targets from its own first event on
    return (0, i1) if sym else (0, n)     # symmetric pass 1: up to the end of the tile; dense: every source


@pytest.mark.parametrize("n,workers,world", [(1, 3, 1), (255, 4, 2), (256, 4, 2), (1000, 7, 2), (1281, 5, 3),
                                             (23422, 444, 1), (23422, 444, 8), (250000, 444, 8)])
@pytest.mark.parametrize("pass_,sym", [(1, True), (1, False), (2, False)])
def test_cut_covers_every_pair_once_and_balances(n, workers, world, pass_, sym):
    n_tiles = (n + TILE - 1) // TILE
    per_tile = {}
    loads = []
    for r in range(world):
        seg = hp.plan_segments(n, pass_, 1, sym, workers * world, r * workers, (r + 1) * workers)
        load = 0
        slots = {}
        for w, I, jb, je, slot in seg:
            assert r * workers <= w < (r + 1) * workers and 0 <= I < n_tiles and jb <= je
            per_tile.setdefault(int(I), []).append((int(jb), int(je)))
            slots.setdefault(int(I), []).append(int(slot))
            i0, i1 = I * TILE, min(n, (I + 1) * TILE)
            if pass_ == 2:
                own = max(0, min(je, i1) - max(jb, i0))
                load += W2_OWN * own + W2_PLAIN * (je - jb - own) + (16 * W2_PLAIN if jb == i0 else 0)
            elif sym:
                load += je - jb
            else:                         # the dense pass 1 weighs sources before the tile's end higher
                load += W_ALL * (je - jb) + W_HEAD * max(0, min(je, i1) - jb)
        for I, sl in slots.items():       # a rank's partial slots of a tile: 0, 1, 2, ... in worker order
            assert sl == list(range(len(sl))), (I, sl)
        loads.append(load)
    assert sorted(per_tile) == list(range(n_tiles))
    for I, ranges in per_tile.items():
        lo, hi = expected_range(n, pass_, sym, I)
        pos = lo
        for jb, je in sorted(ranges):
            assert jb == pos, (I, ranges)
            pos = je
        assert pos == hi, (I, ranges)
    if world > 1 and n >= 20000:          # equal chunks of the cost axis: the ranks' loads agree to within two chunks + 1 %
        assert max(loads) - min(loads) <= 2.0 * sum(loads) / (workers * world) + 0.01 * sum(loads) / world + 1


def test_plan_segments_rejects_bad_arguments():
    lib = hp.load()
    assert lib.hawkes_plan_segments(0, 1, 0, 1, 4, 0, 4, None, 0) == hp.ERR_ARG
    assert lib.hawkes_plan_segments(100, 3, 0, 1, 4, 0, 4, None, 0) == hp.ERR_ARG
    assert lib.hawkes_plan_segments(100, 1, 0, 1, 4, 0, 4, None, 8) == hp.ERR_ARG     # rows wanted, no buffer
    assert lib.hawkes_plan_segments(100, 1, 0, 1, 4, 0, 4, None, 0) > 0                # counting only
    assert hp.load().hawkes_shard_part_doubles(1000, hp.WANT_GRAD, 1) == 6 * 1024
    assert hp.load().hawkes_shard_part_doubles(1000, hp.WANT_GRAD, 2) == 2 * 1024
