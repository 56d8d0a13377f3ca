"""Pins of the oracle on triclinic cells (reading B-9): lower-triangular lattice
a = (ax, 0, 0), b = (bx, by, 0), c = (cx, cy, cz). What fixes the answer here is geometry, not the oracle: the set of
(i, j, S) with |r_j + S.box - r_i| < R over ALL lattice translations, and the fact that a crystal does not care which
unit cell describes it."""
import numpy as np
import pytest

import gen
import oracle


def tric_box(L, xy, xz, yz, Ly=None, Lz=None):
    Ly = L if Ly is None else Ly; Lz = L if Lz is None else Lz
    return np.array([L, 0, 0, xy, Ly, 0, xz, yz, Lz], dtype=np.float64)


def enumerate_all_translations(pos, box9, R, smax=3):
    """Independent of any wrapping: caller positions as they are, S in {-smax..smax}^3."""
    H = np.asarray(box9).reshape(3, 3)
    out = set()
    N = len(pos)
    rng = range(-smax, smax + 1)
    for sa in rng:
        for sb in rng:
            for sc in rng:
                sh = sa * H[0] + sb * H[1] + sc * H[2]
                d = pos[None, :, :] + sh - pos[:, None, :]
                m = (d ** 2).sum(-1) < R * R
                if sa == sb == sc == 0:
                    m &= ~np.eye(N, dtype=bool)
                for i, j in zip(*np.nonzero(m)):
                    out.add((int(i), int(j), sa, sb, sc))
    return out


@pytest.mark.parametrize("case", ["mild", "strong", "negative", "outside"])
def test_neighbor_set_equals_enumeration_over_all_translations(case):
    rng = np.random.default_rng(11)
    box = {"mild": tric_box(9.0, 1.5, -1.0, 2.0), "strong": tric_box(11.0, 5.0, 4.5, -5.0, 10.0, 9.5),
           "negative": tric_box(9.5, -3.0, 2.5, -2.0), "outside": tric_box(9.0, 2.0, 1.0, -1.5)}[case]
    H = box.reshape(3, 3)
    n = 60
    s = rng.random((n, 3))
    if case == "outside":
        s = s * 5.0 - 2.0                          # atoms up to two periods outside the cell: caller-frame shifts
    pos = s @ H
    R = 4.2
    want = enumerate_all_translations(pos, box, R, smax=5 if case == "outside" else 3)
    for mode in ("cell", "brute"):
        rows = oracle.neighbors(pos, box, R, mode)
        got = {tuple(r) for r in rows.tolist()}
        assert len(got) == len(rows)
        assert got == want, (mode, len(got), len(want))
    # symmetric
    assert all((j, i, -a, -b, -c) in want for (i, j, a, b, c) in want)


def test_cell_equals_bruteforce_multi_cell_triclinic():
    rng = np.random.default_rng(12)
    box = tric_box(21.0, 6.0, -4.0, 5.0, 19.0, 23.0)      # 3 x 3 x 4 cells at R = 5.5
    pos = rng.random((700, 3)) @ box.reshape(3, 3) + np.array([3.0, -40.0, 11.0])
    a = oracle.neighbors(pos, box, 5.5, "cell")
    b = oracle.neighbors(pos, box, 5.5, "brute")
    assert a.shape == b.shape and (a == b).all()
    sel = np.unique(rng.integers(0, len(pos), 30))
    rows, row_ptr = oracle.neighbor_rows(pos, box, 5.5, sel)
    want = b[np.isin(b[:, 0], sel)]
    assert rows.shape == want.shape and (rows == want).all()


def test_box_checks_triclinic():
    pos = np.random.default_rng(1).random((10, 3)) * 8.0
    # distance between the faces spanned by b and c: L / sqrt(1 + (xy/Ly)^2) for a pure xy tilt
    box = tric_box(8.0, 8.0, 0.0, 0.0)
    with pytest.raises(ValueError):
        oracle.neighbors(pos, box, 6.0)                    # 8 / sqrt(2) = 5.66 < 6
    assert len(oracle.neighbors(pos, box, 5.6)) > 0
    up = tric_box(8.0, 0.0, 0.0, 0.0); up[2] = 0.5         # an upper-triangular entry: not in the accepted form
    with pytest.raises(ValueError):
        oracle.neighbors(pos, up, 5.0)


def test_energy_forces_do_not_depend_on_the_choice_of_cell():
    """The same periodic structure described by the cubic cell (a, b, c) and by the sheared cells (a, b + a, c) and
    (a, b - a, c + a): E, F and the virial agree; so do per-atom energies."""
    cfg = gen.make_config(1)                                # 96 atoms, cubic 9.86, rc 6: images matter
    L = cfg["box"][0]
    # shrink the cutoff radius of the comparison so that the sheared cells stay wide enough (L / sqrt(2) ... >= rc)
    w = gen.make_weights(S=2, T=2, L=2, n_gauss=6, n_orb=gen.n_orb_default(6, 2), H=(16, 12), Hc=(10, 14), rc=4.4,
                         nbar=30.0, seed=77, wc_gain=[1.5, 1.5], c_gain=[1.5], e_scale=2.0, radial_jitter=0.1)
    blob = gen.pack_blob(w)
    ref = oracle.energy_forces(blob, cfg["species"], cfg["pos"], cfg["box"])
    for box in (tric_box(L, L, 0.0, 0.0), tric_box(L, -L, L, 0.0)):
        r = oracle.energy_forces(blob, cfg["species"], cfg["pos"], box)
        assert abs(r["E"] - ref["E"]) < 1e-10 * max(1.0, abs(ref["E"]))
        np.testing.assert_allclose(r["F"], ref["F"], atol=1e-10 * max(1.0, np.abs(ref["F"]).max()))
        np.testing.assert_allclose(r["Ei"], ref["Ei"], atol=1e-10)
        np.testing.assert_allclose(r["virial"], ref["virial"], atol=1e-9 * max(1.0, np.abs(ref["virial"]).max()))


def test_forces_and_shear_virial_by_finite_differences_in_a_triclinic_cell():
    rng = np.random.default_rng(21)
    w = gen.make_weights(S=2, T=2, L=2, n_gauss=5, n_orb=gen.n_orb_default(5, 2), H=(12, 10), Hc=(9, 11), rc=3.6,
                         nbar=12.0, seed=5, wc_gain=[2.0, 2.0], c_gain=[2.0], e_scale=3.0, radial_jitter=0.15)
    blob = gen.pack_blob(w)
    box = tric_box(8.0, 2.5, -1.5, 2.0, 7.5, 8.5)
    n = 40
    pos = rng.random((n, 3)) @ box.reshape(3, 3)
    sp = rng.integers(0, 2, n).astype(np.int32)
    r = oracle.energy_forces(blob, sp, pos, box)
    h = 1e-5
    for i, d in [(0, 0), (7, 1), (23, 2)]:
        pp, pm = pos.copy(), pos.copy()
        pp[i, d] += h; pm[i, d] -= h
        ep = oracle.energy_forces(blob, sp, pp, box, forces=False)["E"]
        em = oracle.energy_forces(blob, sp, pm, box, forces=False)["E"]
        assert abs(-(ep - em) / (2 * h) - r["F"][i, d]) < 2e-7 * max(1.0, np.abs(r["F"]).max())
    # homogeneous deformation x' = x + eps * y (keeps the lattice lower-triangular): dE/d eps = -virial[y][x]
    for (src, dst) in [(1, 0), (2, 0), (2, 1)]:
        Es = []
        for sgn in (+1, -1):
            D = np.eye(3); D[src, dst] = sgn * h
            Es.append(oracle.energy_forces(blob, sp, pos @ D, (box.reshape(3, 3) @ D).reshape(9), forces=False)["E"])
        dE = (Es[0] - Es[1]) / (2 * h)
        assert abs(-dE - r["virial"][src, dst]) < 1e-6 * max(1.0, np.abs(r["virial"]).max()), (src, dst)
    np.testing.assert_allclose(r["virial"], r["virial"].T, atol=1e-9 * np.abs(r["virial"]).max())
    assert np.abs(r["F"].sum(0)).max() < 1e-10 * max(1.0, np.abs(r["F"]).max()) * n
