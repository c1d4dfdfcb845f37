"""Host logic of the auto-tuner (no GPU): candidate tiles."""
from paper_1212_0785_b200 import autotune


def test_force_tiles_divide_fill_the_block_and_prefer_long_rows():
    for dims, limit in [((32, 32, 32, 64), 128), ((32, 32, 32, 64), 256), ((48, 48, 48, 96), 128), ((4, 4, 4, 4), 128),
                        ((6, 4, 2, 8), 256)]:
        tiles = autotune.force_tiles(dims, limit)
        assert tiles and len(tiles) <= 12
        sizes = {t[0] * t[1] * t[2] * t[3] for t in tiles}
        assert len(sizes) == 1 and sizes.pop() <= limit
        for t in tiles:
            assert t[0] % 2 == 0 and all(d % x == 0 for d, x in zip(dims, t))
        assert tiles[0][0] == max(t[0] for t in tiles) or tiles[0][0] >= 32
    assert autotune.force_tiles((32, 32, 32, 64), 128)[0][0] == 32
    assert autotune.force_tiles((2, 2, 2, 2), 1) == []
