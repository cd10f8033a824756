"""`-m "not gpu"`: the host logic that shares the flattened (proposal tile, bin) space among the CTAs of the fused kernel
(csrc/gw_internal.h `segment_at`, exported host-only as gw_plan_cta_segments).  The kernel runs the same inline
arithmetic, so what is checked here is what fixes the summation order on the GPU."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def segs():
    from paper_1904_02863_b200.csrc import build as csrc_build
    csrc_build.build()
    from paper_1904_02863_b200 import binding

    def all_segments(n_tiles, n_bins, n_ctas):
        return [binding.plan_cta_segments(n_tiles, n_bins, n_ctas, k) for k in range(n_ctas)]
    return all_segments


CASES = [(16, 8113, 296), (16, 8113, 148), (16, 8113, 144), (4, 259585, 296), (1, 1043457, 296), (256, 8113, 296),
         (3, 1601, 296), (1, 37, 5), (7, 10, 70), (7, 10, 69), (5, 3, 15), (2, 100, 1), (32, 3937, 288), (88, 1601, 3520)]


@pytest.mark.parametrize("n_tiles,n_bins,n_ctas", CASES)
def test_segments_partition_every_tile_in_order(segs, n_tiles, n_bins, n_ctas):
    per_cta = segs(n_tiles, n_bins, n_ctas)
    by_tile = {t: [] for t in range(n_tiles)}
    sizes, slots = [], []
    for k, rows in enumerate(per_cta):
        sizes.append(int((rows[:, 2] - rows[:, 1]).sum()) if len(rows) else 0)
        last_tile = -1
        for tile, j0, j1, index, count, slot in rows:
            assert 0 <= j0 < j1 <= n_bins and tile > last_tile          # a CTA walks tiles in ascending order
            last_tile = tile
            by_tile[int(tile)].append((int(j0), int(j1), int(index), int(count), int(slot), k))
            slots.append(int(slot))
    # equal shares: no CTA has more than one bin above the smallest share
    assert sum(sizes) == n_tiles * n_bins and max(sizes) - min(sizes) <= 1
    assert len(set(slots)) == len(slots) and max(slots) < n_ctas + n_tiles   # unique partial-sum slots within bound
    for t, lst in by_tile.items():
        # ascending bins, contiguous cover of [0, n_bins), consistent (index, count), consecutive slots and CTAs
        assert lst[0][0] == 0 and lst[-1][1] == n_bins
        for i, (j0, j1, index, count, slot, k) in enumerate(lst):
            assert index == i and count == len(lst)
            if i:
                assert j0 == lst[i - 1][1] and slot == lst[i - 1][4] + 1 and k == lst[i - 1][5] + 1


@pytest.mark.parametrize("n_tiles,n_bins,n_chunks", [(16, 8113, 9), (3, 1601, 40), (4, 259585, 74), (1, 1000, 7)])
def test_aligned_grid_reproduces_equal_chunks(segs, n_tiles, n_bins, n_chunks):
    """n_ctas = n_tiles * n_chunks gives every tile the chunks [floor(c M / n), floor((c + 1) M / n)) of round 1."""
    per_cta = segs(n_tiles, n_bins, n_tiles * n_chunks)
    for k, rows in enumerate(per_cta):
        t, c = divmod(k, n_chunks)
        assert rows.tolist() == [[t, c * n_bins // n_chunks, (c + 1) * n_bins // n_chunks, c, n_chunks, k + t]]


def test_random_grids(segs):
    rng = np.random.Generator(np.random.PCG64(7))
    for _ in range(60):
        n_tiles, n_bins = int(rng.integers(1, 40)), int(rng.integers(1, 3000))
        n_ctas = int(rng.integers(1, min(600, n_tiles * n_bins) + 1))
        test_segments_partition_every_tile_in_order(segs, n_tiles, n_bins, n_ctas)


def test_rejects_bad_arguments():
    from paper_1904_02863_b200 import binding
    lib = binding.load_library()
    assert lib.gw_plan_cta_segments(0, 10, 4, 0, 0, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_plan_cta_segments(2, 10, 4, 4, 0, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_plan_cta_segments(2, 10, 4, 0, 0, None) == 1
    assert lib.gw_plan_cta_segments(1 << 40, 1 << 30, 1 << 20, 0, 0, None) == binding.GW_ERR_INVALID_ARG
