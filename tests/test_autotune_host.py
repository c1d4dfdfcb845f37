"""Host logic of the auto-tuner (no GPU): candidate tiles."""
from paper_1212_0785_b200 import autotune


def test_force_tiles_divide_fill_the_block_and_prefer_long_rows():
    for dims, limit in [((32, 32, 32, 64), 128), ((32, 32, 32, 64), 256), ((48, 48, 48, 96), 128), ((4, 4, 4, 4), 128),
                        ((6, 4, 2, 8), 256)]:
        tiles = autotune.force_tiles(dims, limit)
        assert tiles and len(tiles) <= 16
        top = max(t[0] * t[1] * t[2] * t[3] for t in tiles)
        assert top <= limit
        for t in tiles:
            assert t[0] % 2 == 0 and all(d % x == 0 for d, x in zip(dims, t))
            # block-filling tiles, or whole-row tiles within 3/4 of them (48-wide lattices)
            assert t[0] * t[1] * t[2] * t[3] == top or (t[0] == dims[0] and t[0] * t[1] * t[2] * t[3] >= 0.75 * top)
        full = [t for t in tiles if t[0] * t[1] * t[2] * t[3] == top]
        assert full[0][0] == max(t[0] for t in full) or full[0][0] >= 32
    assert any(t[0] == 48 for t in autotune.force_tiles((48, 48, 48, 96), 128))
    assert autotune.force_tiles((32, 32, 32, 64), 128)[0][0] == 32
    assert autotune.force_tiles((2, 2, 2, 2), 1) == []
