"""Pins for the oracle's neighbour sets (brute force, symmetry, counts)."""
import numpy as np
import pytest

import gen
import oracle
from np_pairform import edges_bruteforce


def test_cell_equals_bruteforce_small_box(cfg1):
    # config 1: box 9.86 < 2(rc+skin) = 14 -> one cell per dimension, duplicate images present
    R = cfg1["rc"] + cfg1["skin"]
    a = oracle.neighbors(cfg1["pos"], cfg1["box"], R, "cell")
    b = oracle.neighbors(cfg1["pos"], cfg1["box"], R, "brute")
    assert a.shape == b.shape and (a == b).all()
    # an atom and an image of the same atom both neighbours of some i (A-12)
    key = a[:, 0].astype(np.int64) * 1000 + a[:, 1]
    assert len(np.unique(key)) < len(key)


@pytest.mark.parametrize("n_mol,R", [(60, 4.0), (150, 5.5), (260, 6.5)])
def test_cell_equals_bruteforce_multi_cell(n_mol, R):
    c = gen.make_config(2, n_mol=n_mol, geometry_only=True)   # 2..3 cells per dimension
    a = oracle.neighbors(c["pos"], c["box"], R, "cell")
    b = oracle.neighbors(c["pos"], c["box"], R, "brute")
    assert (a == b).all()


def test_matches_independent_numpy_enumeration(cfg1):
    R = 7.0
    rows = oracle.neighbors(cfg1["pos"], cfg1["box"], R, "cell")
    ii, jj, dd = edges_bruteforce(cfg1["pos"], cfg1["box"], R)
    assert len(ii) == len(rows)
    # compare (i, j) multisets and the multiset of edge lengths reconstructed from the shifts
    Lb = cfg1["box"].reshape(3, 3).diagonal()
    d_rows = cfg1["pos"][rows[:, 1]] + rows[:, 2:5] * Lb - cfg1["pos"][rows[:, 0]]
    np.testing.assert_allclose(np.sort((d_rows ** 2).sum(1)), np.sort((dd ** 2).sum(1)), rtol=0, atol=1e-9)
    k1 = np.sort(rows[:, 0].astype(np.int64) * 100000 + rows[:, 1])
    k2 = np.sort(ii.astype(np.int64) * 100000 + jj)
    assert (k1 == k2).all()


def test_symmetry_and_no_self(cfg1):
    rows = oracle.neighbors(cfg1["pos"], cfg1["box"], 7.0)
    s = {tuple(r) for r in rows.tolist()}
    assert len(s) == len(rows)                       # unique
    for (i, j, a, b, c) in s:
        assert (j, i, -a, -b, -c) in s               # (i,j,S) in E <=> (j,i,-S) in E
        assert not (i == j and a == 0 and b == 0 and c == 0)


def test_unwrapped_positions_give_caller_frame_shifts(cfg1):
    rng = np.random.default_rng(5)
    Lb = cfg1["box"].reshape(3, 3).diagonal()
    k = rng.integers(-2, 3, size=cfg1["pos"].shape)
    pos2 = cfg1["pos"] + k * Lb                       # same system, atoms moved by lattice vectors
    R = 7.0
    r1 = oracle.neighbors(cfg1["pos"], cfg1["box"], R)
    r2 = oracle.neighbors(pos2, cfg1["box"], R)
    assert len(r1) == len(r2)
    # edge vectors rebuilt from the caller-frame shifts are within R in both frames
    for rows, p in ((r1, cfg1["pos"]), (r2, pos2)):
        d = p[rows[:, 1]] + rows[:, 2:5] * Lb - p[rows[:, 0]]
        assert ((d ** 2).sum(1) < R * R + 1e-9).all()
    # and map onto each other: S2 = S1 - k_j + k_i
    s1 = {tuple(r) for r in r1.tolist()}
    s2 = {(i, j, a + k[j][0] - k[i][0], b + k[j][1] - k[i][1], c + k[j][2] - k[i][2]) for (i, j, a, b, c) in r2.tolist()}
    assert s1 == s2


def test_density_count_and_fcc_shells():
    c = gen.make_config(4, ncell=4, geometry_only=True)     # 256 atoms, box 14.44
    pos, _ = gen.fcc_lattice(4, 3.61, 0.0, 0)
    rows = oracle.neighbors(pos, c["box"], 5.0)
    # perfect fcc a=3.61: shells at 2.553 (12), 3.61 (6), 4.421 (24) inside 5.0; 5.105 outside
    assert len(rows) == 256 * 42
    rows = oracle.neighbors(pos, c["box"], 6.0)             # + 12 at 5.105 + 24 at 5.708
    assert len(rows) == 256 * 78


def test_box_errors(cfg1):
    with pytest.raises(ValueError):
        oracle.neighbors(cfg1["pos"], cfg1["box"], 10.0)    # box < R
    tric = cfg1["box"].copy(); tric[1] = 0.3
    with pytest.raises(ValueError):
        oracle.neighbors(cfg1["pos"], tric, 7.0)            # non-orthorhombic unsupported


@pytest.mark.parametrize("which", ["cfg1", "w260", "slab"])
def test_selected_rows_equal_the_bruteforce_rows(which, cfg1):
    """oracle.neighbor_rows (rows of selected atoms only; used for sampled pair-set parity on systems whose
    full list does not fit the host) against the O(N^2 27) brute-force list, unwrapped positions included."""
    if which == "cfg1":
        pos, box, R = cfg1["pos"] + np.array([31.0, -17.0, 5.5]), cfg1["box"], cfg1["rc"] + cfg1["skin"]
    elif which == "w260":
        c = gen.make_config(2, n_mol=260, geometry_only=True); pos, box, R = c["pos"], c["box"], 6.5
    else:
        c = gen.make_config(5, n_mol=300, geometry_only=True); pos, box, R = c["pos"], c["box"], 8.0
    full = oracle.neighbors(pos, box, R, "brute")
    sel = np.unique(np.random.default_rng(4).integers(0, len(pos), 40))
    rows, row_ptr = oracle.neighbor_rows(pos, box, R, sel)
    want = full[np.isin(full[:, 0], sel)]
    assert rows.shape == want.shape and (rows == want).all()
    assert row_ptr[-1] == len(rows) and (np.diff(row_ptr) == [(full[:, 0] == i).sum() for i in sel]).all()
