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

    def all_segments(n_tiles, n_bins, n_ctas, boundary_bins=0):
        return [binding.plan_cta_segments(n_tiles, n_bins, n_ctas, k, boundary_bins=boundary_bins) for k in range(n_ctas)]
    return all_segments


CASES = [(16, 8113, 296), (16, 8113, 148), (16, 8113, 144), (4, 259585, 296), (1, 1043457, 296), (256, 8113, 296),
         (3, 1601, 296), (1, 37, 5), (7, 10, 70), (7, 10, 69), (5, 3, 15), (2, 100, 1), (32, 3937, 288), (88, 1601, 3520)]


@pytest.mark.parametrize("n_tiles,n_bins,n_ctas", CASES)
def test_segments_partition_every_tile_in_order(segs, n_tiles, n_bins, n_ctas, boundary_bins=0):
    per_cta = segs(n_tiles, n_bins, n_ctas, boundary_bins)
    by_tile = {t: [] for t in range(n_tiles)}
    sizes, slots = [], []
    for k, rows in enumerate(per_cta):
        sizes.append(int((rows[:, 2] - rows[:, 1]).sum()) if len(rows) else 0)
        last_tile = -1
        for tile, j0, j1, index, count, slot in rows:
            assert 0 <= j0 <= j1 <= n_bins and tile > last_tile         # a CTA walks tiles in ascending order
            assert j0 < j1 or (boundary_bins > 0 and j0 == j1 == n_bins)   # no bins only behind a tile's last bin
            last_tile = tile
            by_tile[int(tile)].append((int(j0), int(j1), int(index), int(count), int(slot), k))
            slots.append(int(slot))
    # equal shares: no CTA has more than one bin above the smallest share; with boundary bins a CTA has up to that many
    # bins less for every tile boundary its range touches, and never more than the plain share
    assert sum(sizes) == n_tiles * n_bins
    if boundary_bins == 0:
        assert max(sizes) - min(sizes) <= 1
    else:
        tile_len = n_bins + boundary_bins
        work = n_tiles * tile_len - boundary_bins                     # no boundary positions behind the last tile
        for k in range(n_ctas):
            w0, w1 = k * work // n_ctas, (k + 1) * work // n_ctas
            touched = (w1 - 1) // tile_len - w0 // tile_len + 1 if w1 > w0 else 0
            assert (w1 - w0) - touched * boundary_bins <= sizes[k] <= w1 - w0
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


@pytest.mark.parametrize("n_tiles,n_bins,n_ctas,boundary_bins", [(16, 8113, 148, 30), (16, 8113, 296, 30), (64, 8113, 296, 30),
                                                                 (256, 8113, 296, 30), (4, 259585, 296, 30), (7, 10, 69, 3),
                                                                 (5, 3, 14, 1), (3, 1601, 296, 200), (9, 50, 4, 40)])
def test_boundary_bins_keep_the_partition(segs, n_tiles, n_bins, n_ctas, boundary_bins):
    """Boundary bins (consecutive tiles separated by positions without work) only move the segment ends: every
    (tile, bin) is still swept exactly once, in order, with consistent counts and slots; a range that only touches a tile's
    boundary positions is a segment of no bins, counted like any other."""
    test_segments_partition_every_tile_in_order(segs, n_tiles, n_bins, n_ctas, boundary_bins)


def test_boundary_bins_shorten_the_crossing_cta(segs):
    """C1's balanced grid: the CTAs whose range crosses a tile boundary sweep 30 bins less than the others."""
    per_cta = segs(16, 8113, 148, 30)
    sizes = np.array([int((r[:, 2] - r[:, 1]).sum()) for r in per_cta])
    two = np.array([len(r) == 2 and r[0, 2] > r[0, 1] and r[1, 2] > r[1, 1] for r in per_cta])
    full = sizes.max()                    # the share of a CTA whose range touches no boundary positions
    assert two.sum() >= 10 and np.all(np.abs(sizes[two] - (full - 30)) <= 1) and sizes.min() >= full - 31
    assert (sizes >= full - 1).sum() >= 148 - 12 - 8      # a range that merely ends or starts in boundary positions is rare


def test_random_grids_with_boundary_bins(segs):
    rng = np.random.Generator(np.random.PCG64(11))
    for _ in range(60):
        n_tiles, n_bins = int(rng.integers(1, 40)), int(rng.integers(1, 3000))
        n_ctas = int(rng.integers(1, min(600, n_tiles * n_bins) + 1))
        test_segments_partition_every_tile_in_order(segs, n_tiles, n_bins, n_ctas, int(rng.integers(1, 200)))


def test_rejects_bad_arguments():
    from paper_1904_02863_b200 import binding
    lib = binding.load_library()
    assert lib.gw_plan_cta_segments(0, 10, 0, 4, 0, 0, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_plan_cta_segments(2, 10, 0, 4, 4, 0, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_plan_cta_segments(2, 10, -1, 4, 0, 0, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_plan_cta_segments(2, 10, 0, 4, 0, 0, None) == 1
    assert lib.gw_plan_cta_segments(1 << 40, 1 << 30, 0, 1 << 20, 0, 0, None) == binding.GW_ERR_INVALID_ARG
