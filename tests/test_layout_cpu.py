"""Host logic of the bank layout, through the host-only C-ABI call
spiir_layout_probe: every filter gets exactly one slot inside its own template's warp tiles, padding is
what the tile size demands, lanes are dealt so that shared-memory loads avoid bank conflicts, and a
template's layout does not depend on its position in the bank."""
import numpy as np
import pytest

import spiir_inputs


@pytest.fixture(scope="module")
def pkg():
    import __graft_entry__ as entry
    entry.build()
    import paper_1602_05573_b200 as p
    return p


def tiles_of(counts, F):
    per = 32 * F
    return [(-(-k // per)) for k in counts]


@pytest.mark.parametrize("F,W", [(2, 32), (4, 16), (4, 32), (8, 8), (8, 16), (16, 8)])
@pytest.mark.parametrize("NC", [1, 2, 4])
def test_slots_are_a_partial_permutation_inside_each_template(pkg, F, W, NC):
    counts = [1, 31, 32, 33, 64, 100, 255, 256, 257, 700, 5000, 3]
    inp = spiir_inputs.make_random_bank(77, counts, 8, d_max=300)
    slots, st = pkg.spiir_layout_probe(inp.offsets, inp.delays, F, W, NC)
    nt = tiles_of(counts, F)
    assert st["n_warp_tiles"] == sum(nt) and st["n_slots"] == sum(nt) * 32 * F
    assert len(set(slots.tolist())) == slots.size                      # one slot per filter
    first = np.concatenate([[0], np.cumsum(nt)]) * 32 * F
    for t, k in enumerate(counts):
        s = slots[inp.offsets[t]:inp.offsets[t + 1]]
        assert s.min() >= first[t] and s.max() < first[t + 1]          # inside its own tiles
    assert st["padding_fraction"] == pytest.approx(1 - sum(counts) / st["n_slots"])
    assert 1.0 <= st["avg_conflict_degree"] <= 32 / NC


@pytest.mark.parametrize("NC,bound", [(1, 1.55), (2, 1.35), (4, 1.22)])
def test_dealing_keeps_uniform_random_delays_nearly_conflict_free(pkg, NC, bound):
    # cfg3-like template sizes and delays; an undealt warp of 32 random delays has degree ~3.4 (NC = 1)
    inp = spiir_inputs.make_config(3, n_templates=64, n_samples=8)
    _, st = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, NC)
    assert st["padding_fraction"] == 0.0
    assert st["avg_conflict_degree"] < bound
    # measure the phases directly from the slots: lanes of one load phase must mostly have distinct keys
    slots, _ = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, NC)
    d_of_slot = np.full(int(st["n_slots"]), -1, np.int64)
    d_of_slot[slots] = inp.delays
    P = 32 // NC
    key = (-(-d_of_slot // NC)) % P
    deg = [np.bincount(ph, minlength=P).max() for ph in key.reshape(-1, P)]
    assert np.mean(deg) == pytest.approx(st["avg_conflict_degree"], rel=1e-12)


def test_structured_delays_are_conflict_free(pkg):
    inp = spiir_inputs.make_config(2, n_templates=8, n_samples=8)      # chirp bank: consecutive delays
    for NC in (1, 2, 4):
        _, st = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, NC)
        assert st["avg_conflict_degree"] < 1.2


def test_layout_of_a_template_is_independent_of_its_position(pkg):
    inp = spiir_inputs.make_random_bank(5, [256, 100, 512, 33, 1024], 8, d_max=2000)
    perm = np.array([3, 0, 4, 2, 1])
    a, _ = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, 2)
    pin = inp.select_templates(perm)
    b, _ = pkg.spiir_layout_probe(pin.offsets, pin.delays, 8, 16, 2)
    nt = tiles_of(np.diff(inp.offsets), 8)
    base_a = np.concatenate([[0], np.cumsum(nt)]) * 256
    base_b = np.concatenate([[0], np.cumsum(np.array(nt)[perm])]) * 256
    for j, t in enumerate(perm):
        rel_a = a[inp.offsets[t]:inp.offsets[t + 1]] - base_a[t]
        rel_b = b[pin.offsets[j]:pin.offsets[j + 1]] - base_b[j]
        assert np.array_equal(rel_a, rel_b)


def test_work_list_counts(pkg):
    # 4096 x 1024 filters, F = 8, W = 16: 4 warp tiles per template, 4 templates per CTA item
    off = np.arange(0, 129) * 1024
    d = (np.arange(128 * 1024) * 7919 % 16384).astype(np.int32)
    _, st = pkg.spiir_layout_probe(off, d, 8, 16, 2)
    assert st["n_warp_tiles"] == 512 and st["n_cta_items"] == 32 and st["n_rounds"] == 32
    # a template larger than a CTA gets an item of its own with several rounds
    _, st = pkg.spiir_layout_probe(np.array([0, 10000]), np.zeros(10000, np.int32), 8, 16, 1)
    assert st["n_warp_tiles"] == 40 and st["n_cta_items"] == 1 and st["n_rounds"] == 3


def test_small_templates_pack_into_shared_tiles(pkg):
    counts = [32, 17, 8, 1, 32, 30, 2, 25, 64, 33, 700, 12, 128, 129]
    inp = spiir_inputs.make_random_bank(9, counts, 8, d_max=300)
    plain, st0 = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, 2, False)
    slots, st = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, 2, True)
    assert st0["segmented"] == 0 and st["segmented"] == 1 and st["uniform_groups"] == 0
    assert st["n_slots"] <= 0.5 * st0["n_slots"]
    assert len(set(slots.tolist())) == slots.size
    F = 8
    tile = slots // (32 * F)
    lane = slots % 32
    for t, k in enumerate(counts):
        s = slice(inp.offsets[t], inp.offsets[t + 1])
        if k <= 16 * F:
            w = next(w for w in (4, 8, 16) if w * F >= k)
            assert len(set(tile[s].tolist())) == 1                      # one tile
            lo = lane[s].min() // w * w
            assert lane[s].min() >= lo and lane[s].max() < lo + w        # inside one aligned segment of w lanes
        else:
            assert len(set(tile[s].tolist())) == -(-k // (32 * F))
    # 32 and 17 filters (4 lanes) share a tile; the class change to 8 filters (4 lanes too) keeps sharing; 64 -> 8 lanes opens a new one
    assert tile[inp.offsets[0]] == tile[inp.offsets[1]] == tile[inp.offsets[2]]
    assert tile[inp.offsets[8]] != tile[inp.offsets[7]]


def test_shared_tile_segments_are_dealt_by_conflict_key(pkg):
    """Inside a segment the filters of one register slot are read by one load phase: they are dealt by conflict key, not by
    position in delay order (uniform delays D / K_t apart are a multiple of the bank-group period as often as not)."""
    def brute_degree(offsets, delays, slots, F, NC):
        """mean over load phases (32 / NC consecutive lanes of one register slot) of the largest key multiplicity"""
        P = 32 // NC
        key = (delays.astype(np.int64) + NC - 1) // NC % P
        phase = slots // 32 * NC + slots % 32 // P                     # (tile, slot) row x phase within the row
        deg = []
        for ph in np.unique(phase):
            deg.append(np.bincount(key[phase == ph], minlength=P).max())
        return float(np.mean(deg))
    for kt, limit in ((64, 1.7), (128, 1.55), (100, 1.55)):
        inp = spiir_inputs.make_random_bank(5, [kt] * 256, 8, d_max=2047)
        slots, st = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, 4, True)
        assert st["segmented"] == 1
        assert st["avg_conflict_degree"] == pytest.approx(brute_degree(inp.offsets, inp.delays, slots, 8, 4), abs=1e-9)
        assert st["avg_conflict_degree"] <= limit, (kt, st["avg_conflict_degree"])      # by position in delay order: 1.9
    # regular spacing, the worst case of dealing by position: 64 filters 32 samples apart all have the same key
    off = np.arange(0, 65 * 64, 64)
    d = np.tile(np.arange(64, dtype=np.int32) * 32, 64)
    slots, st = pkg.spiir_layout_probe(off, d, 8, 16, 4, True)
    assert st["avg_conflict_degree"] == 8.0                            # nothing to deal: one key class
    d = np.tile(np.arange(64, dtype=np.int32) * 33, 64)                # keys 0..7 cyclically: perfect phases exist
    slots, st = pkg.spiir_layout_probe(off, d, 8, 16, 4, True)
    assert st["avg_conflict_degree"] <= 1.15
    # the arrangement of a template does not depend on where it sits in the bank
    inp = spiir_inputs.make_random_bank(6, [64, 20, 64, 33, 64], 8, d_max=900)
    a, _ = pkg.spiir_layout_probe(inp.offsets, inp.delays, 8, 16, 4, True)
    perm = np.array([2, 3, 4, 0, 1])
    inp2 = inp.select_templates(perm)
    b, _ = pkg.spiir_layout_probe(inp2.offsets, inp2.delays, 8, 16, 4, True)
    F = 8
    for new_t, old_t in enumerate(perm):
        sa = a[inp.offsets[old_t]:inp.offsets[old_t + 1]]
        sb = b[inp2.offsets[new_t]:inp2.offsets[new_t + 1]]
        w = next(w for w in (4, 8, 16, 32) if w * F >= sa.size)
        # same register slot and same lane within the segment for every filter
        assert np.array_equal(sa // 32 % F, sb // 32 % F) and np.array_equal(sa % 32 % w, sb % 32 % w)


def test_probe_validates_arguments(pkg):
    with pytest.raises(pkg.SpiirError):
        pkg.spiir_layout_probe(np.array([0, 2]), np.array([0, -1], np.int32))
    with pytest.raises(pkg.SpiirError):
        pkg.spiir_layout_probe(np.array([0, 2]), np.zeros(2, np.int32), 3, 16, 1)
    with pytest.raises(pkg.SpiirError):
        pkg.spiir_layout_probe(np.array([0, 2]), np.zeros(2, np.int32), 8, 16, 3)
