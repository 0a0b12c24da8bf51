"""Host logic of the pair kernels' work decomposition (CPU only, no CUDA call): vn_plan_farfield returns what
vn_farfield would launch; the walk over unordered pairs of super-tiles documented in include/vesnet_farfield.h is
replayed here and must visit every unordered pair exactly once, with equal work per block."""
import itertools

import pytest

import paper_2606_25569_b200 as vn

SHAPES = [(1, 1), (2, 1), (16, 32), (3, 129), (7, 1000), (256, 128), (1000, 128), (2000, 128), (8000, 128),
          (1030, 1), (9, 1024), (5, 1025), (513, 8)]


def walk(n_st):
    """List of (target super-tile, source super-tile, both_directions) the kernel visits."""
    out = []
    for I in range(n_st):
        S = (n_st - 1) // 2
        if n_st % 2 == 0 and I < n_st // 2:
            S += 1
        out.append((I, I, False))
        out += [(I, (I + s) % n_st, True) for s in range(1, S + 1)]
    return out


@pytest.mark.parametrize("prec", [vn.VN_F32, vn.VN_F64])
@pytest.mark.parametrize("nves,npts", SHAPES)
def test_plan_is_consistent(nves, npts, prec):
    p = vn.vn_plan_farfield(nves, npts, prec)
    P = nves * npts
    assert p["tile"] == 128 and p["super_tile"] == p["tile"] * p["tiles_per_super_tile"]
    assert p["n_super_tiles"] == -(-P // p["super_tile"]) and p["n_chunks"] >= 1
    # every chunk of the longest list keeps at least one tile
    longest = p["tiles_per_super_tile"] * (p["n_super_tiles"] // 2 + 1)
    assert p["n_chunks"] <= longest


@pytest.mark.parametrize("n_st", list(range(1, 40)) + [125, 250, 1000])
def test_walk_visits_every_unordered_pair_once(n_st):
    seen = {}
    per_block = {}
    for I, J, both in walk(n_st):
        key = (min(I, J), max(I, J))
        seen[key] = seen.get(key, 0) + 1
        per_block[I] = per_block.get(I, 0) + 1
        assert both == (I != J)
    assert set(seen) == set(itertools.combinations_with_replacement(range(n_st), 2))
    assert all(v == 1 for v in seen.values())
    assert max(per_block.values()) - min(per_block.values()) <= 1          # equal work per block (up to one super-tile)


def test_plan_fills_the_device_in_waves():
    """The chunk count is chosen against the number of resident blocks: large problems get many more blocks than
    slots (smooth tail), small ones still get at least one block per two slots."""
    slots = 148 * 3
    for nves in (256, 1000, 2000, 8000):
        p = vn.vn_plan_farfield(nves, 128, vn.VN_F32, slots)
        blocks = p["n_super_tiles"] * p["n_chunks"]
        assert blocks >= slots // 2
        if nves >= 2000:
            assert blocks >= 8 * slots
    assert vn.lib().vn_plan_farfield(0, 4, vn.VN_F32, slots, None) == vn.VN_ERR_INVALID_ARG


def test_chunk_length_follows_the_measured_model():
    """choose_sym_split: chunks of t = sqrt(0.12 W) tiles, W = tiles of work per resident-block
    slot; the fp64 kernel caps t at the ring depth (4 stages)."""
    slots = 148 * 3

    def tiles_per_chunk(nves, prec):
        p = vn.vn_plan_farfield(nves, 128, prec, slots)
        n_st = p["n_super_tiles"]
        longest = p["tiles_per_super_tile"] * ((n_st - 1) // 2 + (1 if n_st % 2 == 0 else 0) + 1)
        W = n_st * longest / slots
        return -(-longest // p["n_chunks"]), W

    for nves in (256, 1000, 2000, 8000):
        t, W = tiles_per_chunk(nves, vn.VN_F32)
        assert abs(t - max(1.0, (0.12 * W) ** 0.5)) <= 1.0
        t64, _ = tiles_per_chunk(nves, vn.VN_F64)
        assert 1 <= t64 <= 4
    assert tiles_per_chunk(256, vn.VN_F32)[0] == 1 and tiles_per_chunk(8000, vn.VN_F32)[0] == 33
