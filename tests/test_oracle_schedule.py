"""Pins for the sub-sweep schedule (Eq. 8, Eqs. 9-22, Table 1, Fig. 2 remark)."""
import itertools
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _brute(nx, ny, nz, S):
    return sum(1 for i in range(nx) for j in range(ny) for k in range(nz) if i + j + k == S)


def test_eq9_equals_brute_force_all_small_meshes(orc):
    for nx, ny, nz in itertools.product(range(1, 8), repeat=3):
        tot = 0
        for S in range(nx + ny + nz - 2):
            p = orc.wavefront_size(nx, ny, nz, S)
            assert p == _brute(nx, ny, nz, S), (nx, ny, nz, S)
            tot += p
        assert tot == nx * ny * nz


def test_c_and_python_eq9_agree(orc):
    lib = orc._lib()
    for (nx, ny, nz) in [(8, 8, 8), (32, 32, 32), (5, 9, 3), (256, 256, 128), (1, 1, 7)]:
        for S in range(nx + ny + nz - 2):
            assert lib.orc_wavefront_size(nx, ny, nz, S) == orc.wavefront_size(nx, ny, nz, S)


def test_table1_rows(orc):
    rows = [tuple(int(v) for v in l.split()) for l in open(os.path.join(GOLD, "table1_subsweep4.txt"))
            if l.strip() and not l.startswith("#")]
    n = 6                                     # any cube with N > 4 shows the full 15-voxel sub-sweep
    off, cell_of = orc.schedule(n, n, n, 0)
    cells = cell_of[off[4]:off[5]]
    assert len(cells) == 15 == len(rows)
    for (idx, ix, iy, iz), c in zip(rows, cells):
        assert (c % n, (c // n) % n, c // (n * n)) == (ix, iy, iz), idx
        assert ix + iy + iz == 4


def test_growth_and_last_subsweep(orc):
    # PAPER.md:68 "three voxels ... After those three, six"; Fig. 2: S = 14 holds one voxel
    assert [orc.wavefront_size(8, 8, 8, S) for S in range(3)] == [1, 3, 6]
    for dims in [(5, 6, 6), (4, 4, 9), (7, 7, 3)]:            # any mesh with nx+ny+nz = 17
        assert sum(dims) == 17
        assert orc.wavefront_size(*dims, 14) == 1
        off, _ = orc.schedule(*dims, 0)
        assert len(off) - 1 == 15 and off[-1] - off[-2] == 1


@pytest.mark.parametrize("dims", [(4, 4, 4), (3, 5, 2), (1, 6, 4), (7, 2, 2)])
@pytest.mark.parametrize("octant", range(8))
def test_schedule_is_a_valid_upwind_order(orc, dims, octant):
    nx, ny, nz = dims
    off, cell_of = orc.schedule(nx, ny, nz, octant)
    assert sorted(cell_of.tolist()) == list(range(nx * ny * nz))          # a permutation
    plane_of = np.empty(nx * ny * nz, dtype=int)
    for S in range(len(off) - 1):
        plane_of[cell_of[off[S]:off[S + 1]]] = S
    sx, sy, sz = (-1 if octant & 1 else 1), (-1 if octant & 2 else 1), (-1 if octant & 4 else 1)
    for c in range(nx * ny * nz):
        i, j, k = c % nx, (c // nx) % ny, c // (nx * ny)
        for (iu, ju, ku) in [(i - sx, j, k), (i, j - sy, k), (i, j, k - sz)]:
            if 0 <= iu < nx and 0 <= ju < ny and 0 <= ku < nz:
                assert plane_of[iu + nx * (ju + ny * ku)] == plane_of[c] - 1


def test_schedule_full_size_counts(orc):
    # SURVEY §8 size table: planes per octant and max P(S) of the five configs
    for dims, planes, pmax in [((8, 8, 8), 22, 48), ((32, 32, 32), 94, 768), ((64, 64, 64), 190, 3072),
                               ((128, 128, 64), 318, 7168), ((256, 256, 128), 638, 28672)]:
        ps = [orc.wavefront_size(*dims, S) for S in range(sum(dims) - 2)]
        assert len(ps) == planes and max(ps) == pmax and sum(ps) == dims[0] * dims[1] * dims[2]
