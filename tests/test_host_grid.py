"""Host logic of libtdpd.so without a GPU: the static grid tables of the pair kernel (tdpd_host_grid) against an
independent numpy construction, and a static check that the product path never touches the oracle or the reference."""
import os
import re

import numpy as np
import pytest

import tdpd_workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def T():
    from paper_1611_06163_b200 import build
    build.build()
    import paper_1611_06163_b200 as T
    return T


def _morton(x, y, z):
    code = 0
    for b in range(10):
        code |= ((x >> b) & 1) << (3 * b) | ((y >> b) & 1) << (3 * b + 1) | ((z >> b) & 1) << (3 * b + 2)
    return code


@pytest.mark.parametrize("box", [(10, 10, 10), (13, 11, 8), (40, 20, 20), (5, 5, 5), (32, 32, 32)])
def test_neighbour_runs_cover_the_27_cell_stencil_once(T, box):
    p = W.fluid_params(box, 3.0, seed=1)
    g = T.host_grid(p)
    nc = g["ncell"]
    assert list(nc) == [int(np.floor(np.float32(b) / np.float32(1.58))) for b in box]      # R-bin: floor(L / r_cc)
    ncells = int(nc.prod())
    # Morton rank = position of the cell in the sorted list of interleaved codes
    codes = np.array([_morton(i % nc[0], (i // nc[0]) % nc[1], i // (nc[0] * nc[1])) for i in range(ncells)])
    rank = np.empty(ncells, np.int64)
    rank[np.argsort(codes, kind="stable")] = np.arange(ncells)
    assert np.array_equal(g["cell_rank"], rank)
    cell_of_rank = np.argsort(rank)
    off, first, meta = g["seg_off"], g["seg_first"], g["seg_meta"]
    assert off[0] == 0 and off[-1] == len(first) and np.all(np.diff(off.astype(np.int64)) >= 1)
    for r in range(ncells):
        lin = cell_of_rank[r]
        c = np.array([lin % nc[0], (lin // nc[0]) % nc[1], lin // (nc[0] * nc[1])])
        want = {}
        for k in range(27):
            d = np.array([k % 3 - 1, (k // 3) % 3 - 1, k // 9 - 1])
            q = c + d
            w = np.where(q < 0, -1, np.where(q >= nc, 1, 0))
            q = q - w * nc
            want[int(rank[(q[2] * nc[1] + q[1]) * nc[0] + q[0]])] = (tuple(q // 2), tuple(w))
        got = {}
        sizes = []
        for s in range(off[r], off[r + 1]):
            m = int(meta[s]) & 15
            w = tuple(((int(meta[s]) >> (4 + 2 * a)) & 3) - 1 for a in range(3))
            sizes.append(m)
            for t in range(m):                      # rank-consecutive cells of the run
                rk = int(first[s]) + t
                assert rk not in got
                got[rk] = w
        assert sizes == sorted(sizes, reverse=True)   # longest runs first
        assert set(got) == set(want)                  # the 27 neighbours (fewer distinct cells never occur: n >= 3)
        for s in range(off[r], off[r + 1]):           # one block and one periodic image per run
            m = int(meta[s]) & 15
            blocks = {want[int(first[s]) + t][0] for t in range(m)}
            wraps = {want[int(first[s]) + t][1] for t in range(m)}
            assert len(blocks) == 1 and len(wraps) == 1 and wraps == {got[int(first[s])]}
    if all(n % 2 == 0 and n >= 4 for n in nc):        # interior pattern of an even grid: 8 + 4 + 2 + 2 + 2 + 9 x 1
        assert np.all(np.diff(off.astype(np.int64)) == 14)


def test_product_never_touches_the_oracle_or_the_reference():
    pkg = os.path.join(ROOT, "paper_1611_06163_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "libtdpd_oracle" not in src and "tdpd_oracle.c" not in src, f
                assert "/root/reference" not in src or f.endswith((".cu", ".cuh", ".h")), f   # citations in comments only
    for f in ("bench.py", "__graft_entry__.py"):
        assert "/root/reference" not in open(os.path.join(ROOT, f)).read()
