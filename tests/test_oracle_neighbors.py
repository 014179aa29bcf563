"""Pins for the oracle's neighbour sets (Eq.2; readings R7-R9)."""
import itertools

import numpy as np

import gnep_synth as gs
from cases import golden
from oracle import gnep_oracle as orc


def _spec(rcR, rcA):
    d = dict(gs.MODEL_SPECS[0]); d["rc_radial"] = rcR; d["rc_angular"] = rcA
    return orc.make_spec(d)


def _python_brute(pos, cell, rc, nimg=3):
    """Independent statement of Eq.2 with periodic images: plain numpy over +-nimg images."""
    n = len(pos)
    rows = []
    shifts = list(itertools.product(range(-nimg, nimg + 1), repeat=3))
    for i in range(n):
        row = []
        for j in range(n):
            for s in shifts:
                if j == i and s == (0, 0, 0):
                    continue
                d = pos[j] - pos[i] + s[0] * cell[0] + s[1] * cell[1] + s[2] * cell[2]
                if d @ d < rc * rc:
                    row.append((j,) + s)
        rows.append(sorted(row))
    return rows


def _rows(ob, which):
    rptr, j, sh, r = ob.neighbors(which)
    return [[(int(j[p]),) + tuple(int(v) for v in sh[p]) for p in range(rptr[i], rptr[i + 1])]
            for i in range(ob.N)], r, rptr


def test_brute_force_small_triclinic_multi_image():
    rng = np.random.default_rng(7)
    cell = np.array([[5.0, 0.0, 0.0], [1.2, 4.6, 0.0], [-0.7, 0.9, 5.3]])
    pos = rng.uniform(0.02, 0.98, size=(9, 3)) @ cell
    sp = _spec(6.0, 3.5)          # rc > cell heights: several images of the same atom, self images
    ob = orc.Batch(sp, [0, 9], pos, cell.reshape(1, 9), np.zeros(9, np.int32))
    for which, rc in ((0, 6.0), (1, 3.5)):
        rows, r, rptr = _rows(ob, which)
        assert rows == _python_brute(pos, cell, rc)
        assert any(row.count and any(e[0] == i for e in row) for i, row in enumerate(rows)) or which == 1
        # stored r_ij equals r_j + shift - r_i
        for i, row in enumerate(rows):
            for k, e in enumerate(row):
                d = pos[e[0]] - pos[i] + e[1] * cell[0] + e[2] * cell[1] + e[3] * cell[2]
                np.testing.assert_allclose(r[rptr[i] + k], d, atol=1e-13)


def test_pair_symmetry_and_angular_sublist():
    b = gs.make_batch(0)
    sp = orc.make_spec(gs.MODEL_SPECS[0])
    ob = orc.Batch(sp, b["atom_offsets"], b["positions"], b["cells"], b["types"])
    rows, _, _ = _rows(ob, 0)
    s = set((i,) + e for i, row in enumerate(rows) for e in row)
    for (i, j, a, b_, c) in s:
        assert (j, i, -a, -b_, -c) in s
    rows_a, _, _ = _rows(ob, 1)
    for ra, rr in zip(rows_a, rows):
        assert set(ra) <= set(rr) and ra == sorted(ra)
    # neighbours never cross structures
    off = b["atom_offsets"]
    for i, row in enumerate(rows):
        sidx = np.searchsorted(off, i, side="right") - 1
        assert all(off[sidx] <= e[0] < off[sidx + 1] for e in row)


def test_simple_cubic_shell_counts():
    a, n = 2.0, 3
    g = np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3) * a + 0.25
    cell = np.eye(3) * n * a
    shells = [int(v) for v in golden("sc_shells")]
    for k in range(1, 7):
        rc = a * np.sqrt(k + 0.5)
        ob = orc.Batch(_spec(rc, 1.0), [0, len(g)], g, cell.reshape(1, 9), np.zeros(len(g), np.int32))
        rptr = ob.neighbors(0)[0]
        assert np.all(np.diff(rptr) == sum(shells[:k]))


def test_wrap_by_lattice_vectors_is_invisible():
    b = gs.make_batch(0, n_structs=1)
    sp = orc.make_spec(gs.MODEL_SPECS[0])
    ob = orc.Batch(sp, b["atom_offsets"], b["positions"], b["cells"], b["types"])
    rng = np.random.default_rng(8)
    cell = b["cells"][0].reshape(3, 3)
    moved = b["positions"] + rng.integers(-2, 3, size=(64, 3)) @ cell     # exact for this cubic cell
    ob2 = orc.Batch(sp, b["atom_offsets"], moved, b["cells"], b["types"])
    np.testing.assert_array_equal(ob.positions(), ob2.positions())
    for which in (0, 1):
        for x, y in zip(ob.neighbors(which), ob2.neighbors(which)):
            np.testing.assert_array_equal(x, y)


def test_empty_and_isolated():
    sp = _spec(3.0, 2.0)
    ob = orc.Batch(sp, [0, 1], np.array([[1.0, 1.0, 1.0]]), (np.eye(3) * 10).reshape(1, 9), np.zeros(1, np.int32))
    assert ob.num_pairs(0) == 0 and ob.num_pairs(1) == 0
    # one atom in a cell smaller than the cutoff sees its own images (R7): 6 at distance L=2.5 < 3
    ob = orc.Batch(sp, [0, 1], np.array([[1.0, 1.0, 1.0]]), (np.eye(3) * 2.5).reshape(1, 9), np.zeros(1, np.int32))
    assert ob.num_pairs(0) == 6 and ob.num_pairs(1) == 0
