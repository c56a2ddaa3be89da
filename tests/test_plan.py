"""Host logic of the launch planner (nbk_plan, no GPU): the stream-K cut of the (i-tile, j-tile)
pair list must cover every pair exactly once, fit the partial-row storage a context allocates,
and respect the kernel's shape constraints -- for the BASELINE.json sizes and for ragged ones.
The planner generalises the paper's split-j rule for small i-blocks."""
import itertools

import pytest

from paper_0707_0438_b200 import binding as nb

SIZES = [(1, 1), (1, 16384), (32, 16384), (256, 16384), (2048, 16384), (16384, 16384),
         (1024, 1024), (131072, 131072), (1048576, 1048576), (65536, 65536), (37, 1000),
         (5000, 4999), (100000, 3), (4096, 64), (1 << 20, 64), (7, 1 << 20)]


@pytest.mark.parametrize("n_i,n_j", SIZES)
@pytest.mark.parametrize("sms,force_i", [(148, 0), (148, 1), (148, 2), (148, 4), (132, 0), (1, 0)])
def test_plan_invariants(n_i, n_j, sms, force_i):
    p = nb.nbk_plan(n_i, n_j, sms, force_i)
    I, W = p["i_per_thread"], p["threads"] // 32
    assert I in (1, 2, 4) and (force_i == 0 or I == force_i)
    assert W == {1: 16, 2: 12, 4: 8}[I]
    wj, tj, ti = p["j_split_warps"], p["j_tile"], p["i_tile"]
    assert W % wj == 0 and tj in (64, 128, 256) and (tj // wj) % 4 == 0
    assert ti == (W // wj) * 32 * I
    assert p["i_tiles"] == -(-n_i // ti) and p["j_tiles"] == -(-n_j // tj)
    P, G = p["pairs"], p["grid"]
    assert P == p["i_tiles"] * p["j_tiles"] and 1 <= G <= min(sms, P)
    # contiguous ranges [k*P/G, (k+1)*P/G) tile [0, P) without gap or overlap, sizes differ by <= 1
    starts = [k * P // G for k in range(G + 1)]
    assert starts[0] == 0 and starts[-1] == P
    sizes = [b - a for a, b in zip(starts, starts[1:])]
    assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1
    # no CTA touches more i-tiles than max_segments rows were reserved for
    njt = p["j_tiles"]
    touched = max((b - 1) // njt - a // njt + 1 for a, b in zip(starts, starts[1:]))
    assert touched <= p["max_segments"]
    assert p["partial_floats"] == G * p["max_segments"] * ti * 8
    assert p["partial_floats"] <= p["partial_floats_bound"]


def test_plan_fills_the_machine_for_block_steps():
    """Small i-blocks ('If n is smaller than 4096 ...') still get >= 148 work units."""
    for n_i in (1, 32, 256, 2048):
        p = nb.nbk_plan(n_i, 16384, 148, 0)
        assert p["grid"] >= 128, (n_i, p)
    p = nb.nbk_plan(131072, 131072, 148, 0)
    assert p["grid"] == 148 and p["i_per_thread"] == 4 and p["j_split_warps"] == 1


def test_plan_rejects_bad_arguments():
    for args in [(0, 1, 148, 0), (1, 0, 148, 0), (1, 1, 0, 0), (1, 1, 148, 3)]:
        with pytest.raises(nb.NbkError):
            nb.nbk_plan(*args)
