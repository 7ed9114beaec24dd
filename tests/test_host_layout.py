"""CPU-only: host-side logic of the marker binning layout (lbm_query_layout needs no GPU) and of the
seeded workload generators.  The invariants below are what the chunk / tile kernels rely on
(DESIGN.md section 5); they are checked by brute force over every lattice width."""
import numpy as np


def _blocks(nx, lay):
    """block index of every cell as the kernels compute it: min(x >> 3, nbx - 1)"""
    return np.minimum(np.arange(nx) >> 3, lay["x_blocks"] - 1)


def test_x_blocks_every_width():
    from paper_1904_02108_b200 import api
    for nx in range(4, 400):
        lay = api.query_layout(nx, 8, 8)
        assert lay["block_width"] == 8 and lay["tile_rows"] == 4
        blk = _blocks(nx, lay)
        widths = np.bincount(blk)
        assert len(widths) == lay["x_blocks"] and (widths > 0).all()
        if nx >= 8:
            # every block at least 4 wide, all but the last exactly 8, the last at most 11
            assert (widths[:-1] == 8).all() and 4 <= widths[-1] <= 11
        # a chunk window = block + 3 cells must fit the profile pitch, which never exceeds the maximum
        assert lay["entries"] == max(widths.max(), 8) + 3 <= lay["entries_max"]
        # four consecutive cells (the source cells of one target cell), periodic, meet at most two blocks
        if nx >= 14:
            for x in range(nx):
                src = [(x + 1 - j) % nx for j in range(4)]
                assert len(set(blk[src])) <= 2
        assert lay["mask_words_per_row"] == (nx + 31) // 32


def test_tiles_cover_the_rows():
    from paper_1904_02108_b200 import api
    for n in range(4, 70):
        lay = api.query_layout(16, n, 2 * n + 1)
        assert lay["tiles_y"] == -(-n // 4) and lay["tiles_z"] == -(-(2 * n + 1) // 4)


def test_workload_generators_are_seeded_and_sized():
    from paper_1904_02108_b200 import workloads
    counts = {"W1": 240, "W3": 15360, "W3lit": 7680, "W3x4": 61440, "P1": 3936, "P6": 6 * 3936, "P18": 18 * 3936}
    for name, n in counts.items():
        a, b = workloads.get(name, 0), workloads.get(name, 0)
        assert a.n_markers == n
        for x, y in zip(a.bodies, b.bodies):
            assert np.array_equal(x.pos, y.pos) and np.array_equal(x.axis, y.axis)
    c = workloads.get("W3", 1)
    assert not np.array_equal(c.bodies[0].pos, workloads.get("W3", 0).bodies[0].pos)
    # walls: every stencil of W3 stays inside the box over a full turn (R17)
    w3 = workloads.get("W3")
    r = np.linalg.norm(w3.bodies[0].pos - w3.bodies[0].center, axis=1).max()
    assert 64 - r >= 1 and 64 + r <= 128 - 3
    # the paper-shaped bodies sit inside the 160 x 160 x 320 box with their stencils
    for name in ("P1", "P6", "P18"):
        w = workloads.get(name)
        assert (w.nx, w.ny, w.nz) == (160, 160, 320) and w.bodies[0].area[0] == 1.0
