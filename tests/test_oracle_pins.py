"""Pins for the oracle's energy / force / virial (SURVEY.md 8(c) "What pins each part").

Nothing here compares the oracle with itself through the same formula: the references are
an independent NumPy pair-form (tests/np_pairform.py), closed forms typed out below,
finite differences, and symmetry / locality properties the paper states
(PAPER.md:23, :43, :49, :76, :92).
"""
import numpy as np
import pytest

import gen
import oracle
import np_pairform

BIG = np.diag([200.0, 200.0, 200.0]).reshape(9)


def small_model(S=2, T=3, L=3, n_gauss=5, H=(12, 10), Hc=(9, 11), rc=3.5, seed=77, n_orb=None, radial_jitter=0.15):
    """Radial tables differ per (layer, species) by 15-30 % so that their indexing (A-3) is visible."""
    n_orb = gen.n_orb_default(n_gauss, L) if n_orb is None else n_orb
    w = gen.make_weights(S=S, T=T, L=L, n_gauss=n_gauss, n_orb=n_orb, H=H, Hc=Hc, rc=rc, nbar=12.0, seed=seed,
                         radial_jitter=radial_jitter)
    return w, gen.pack_blob(w)


def cluster(n, spread, seed, S=2, centre=(100.0, 100.0, 100.0)):
    rng = np.random.default_rng(seed)
    pos = np.asarray(centre) + spread * rng.standard_normal((n, 3))
    return pos, rng.integers(0, S, n).astype(np.int32)


# ------------------------------------------------------------------ whole-E pins vs the pair form
def test_pairform_config0(cfg0):
    r = oracle.energy_forces(cfg0["blob"], cfg0["species"], cfg0["pos"], cfg0["box"], forces=False, dumps=True)
    E, Ei, rhos, cs = np_pairform.energy(cfg0["weights"], cfg0["species"], cfg0["pos"], cfg0["box"], True)
    for t in range(cfg0["T"]):
        np.testing.assert_allclose(r["rho"][t], rhos[t], rtol=1e-10, atol=1e-12)
        np.testing.assert_allclose(r["c"][t], cs[t], rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(r["Ei"], Ei, rtol=1e-10, atol=1e-12)
    assert abs(r["E"] - E) < 1e-10 * max(1.0, abs(E))


def test_pairform_config1_duplicate_images(cfg1):
    r = oracle.energy_forces(cfg1["blob"], cfg1["species"], cfg1["pos"], cfg1["box"], forces=False)
    E, Ei, _, _ = np_pairform.energy(cfg1["weights"], cfg1["species"], cfg1["pos"], cfg1["box"], True)
    np.testing.assert_allclose(r["Ei"], Ei, rtol=1e-9, atol=1e-11)


def test_pairform_L3_T3_mixed_widths():
    w, blob = small_model()
    pos, sp = cluster(30, 2.0, 3)
    r = oracle.energy_forces(blob, sp, pos, BIG, forces=False, dumps=True)
    E, Ei, rhos, cs = np_pairform.energy(w, sp, pos, BIG, True)
    np.testing.assert_allclose(r["Ei"], Ei, rtol=1e-10, atol=1e-12)
    for t in range(3):
        np.testing.assert_allclose(r["rho"][t], rhos[t], rtol=1e-9, atol=1e-12)


# ------------------------------------------------------------------ closed forms
def test_dimer_closed_form():
    """b[n,a] = c_j[n] exp(-alpha (r-r_n)^2) (1+cos(pi r/rc))/2 x^lx y^ly z^lz, typed by hand."""
    w, blob = small_model(T=1, L=3, n_gauss=6)
    d = np.array([0.7, -1.1, 1.9])
    pos = np.array([[100.0, 100.0, 100.0], [100.0, 100.0, 100.0] + d])
    sp = np.array([0, 1], dtype=np.int32)
    r = oracle.energy_forces(blob, sp, pos, BIG, forces=False, dumps=True)
    lxyz, mu = oracle.monomials(3)
    assert len(lxyz) == 20 and mu.sum() == 1 + 3 + 9 + 27          # sum_a mu_a = 3^l per l
    rr = np.linalg.norm(d)
    for i, j, dv in ((0, 1, d), (1, 0, -d)):
        rad = w["c0"][sp[j]] * np.exp(-w["alpha"][0, sp[j]] * (rr - w["rcen"][0, sp[j]]) ** 2) \
            * 0.5 * (1 + np.cos(np.pi * rr / w["rc"]))
        ang = np.array([dv[0] ** a * dv[1] ** b * dv[2] ** c for a, b, c in lxyz])
        np.testing.assert_allclose(r["b"][0, i], np.outer(rad, ang), rtol=1e-13, atol=1e-15)
        # A-3 (PAPER.md:35 "G_j ... of the jth neighbor atom", :38): the radial table is the NEIGHBOUR's row.
        # With the centre's row instead the value is different (the rows differ by >= 15 %), so this pin can fail.
        rad_i = w["c0"][sp[j]] * np.exp(-w["alpha"][0, sp[i]] * (rr - w["rcen"][0, sp[i]]) ** 2) \
            * 0.5 * (1 + np.cos(np.pi * rr / w["rc"]))
        assert np.abs(np.outer(rad_i, ang) - r["b"][0, i]).max() > 1e-3 * np.abs(r["b"][0, i]).max()


def test_dimer_second_layer_uses_its_own_tables():
    """T = 2 dimer: b^1_i[n,a] = c^1_j[n] R_n(r; t=1, s_j) A_a typed by hand from the layer-1 rows of the radial
    tables and the oracle's own c^1 (the MLP output, pinned by the pair form and the matmul pins). The rows of
    layer 0 give a different value: the layer index of the tables (A-3) is pinned."""
    w, blob = small_model(T=2, L=2, n_gauss=6)
    assert np.abs(w["rcen"][1] / np.where(w["rcen"][0] == 0, 1, w["rcen"][0]) - 1)[:, 1:].min() > 0.02
    d = np.array([-0.9, 1.3, 0.8])
    pos = np.array([[100.0, 100.0, 100.0], [100.0, 100.0, 100.0] + d])
    sp = np.array([1, 0], dtype=np.int32)
    r = oracle.energy_forces(blob, sp, pos, BIG, forces=False, dumps=True)
    lxyz, _ = oracle.monomials(2)
    rr = np.linalg.norm(d)
    fc = 0.5 * (1 + np.cos(np.pi * rr / w["rc"]))
    for i, j, dv in ((0, 1, d), (1, 0, -d)):
        ang = np.array([dv[0] ** a * dv[1] ** b * dv[2] ** c for a, b, c in lxyz])
        for t_tab, same in ((1, True), (0, False)):
            rad = r["c"][1, j] * np.exp(-w["alpha"][t_tab, sp[j]] * (rr - w["rcen"][t_tab, sp[j]]) ** 2) * fc
            ok = np.allclose(r["b"][1, i], np.outer(rad, ang), rtol=1e-12, atol=1e-15)
            assert ok == same, (i, t_tab)


def test_pairform_T2_layer_tables_differ():
    """Whole-E pin on a model whose layer-0 and layer-1 tables (and species rows) differ: the independent NumPy
    pair form, which reads alpha[t][s_j] / rcen[t][s_j] as the blob docstring lays them out."""
    w, blob = small_model(T=2, L=2, n_gauss=6, radial_jitter=0.2)
    pos, sp = cluster(24, 1.7, 13)
    r = oracle.energy_forces(blob, sp, pos, BIG, forces=False, dumps=True)
    E, Ei, rhos, cs = np_pairform.energy(w, sp, pos, BIG, True)
    np.testing.assert_allclose(r["Ei"], Ei, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(r["rho"][1], rhos[1], rtol=1e-9, atol=1e-12)
    # the same weights with every row equal to row (0, 0) give a different energy: the test can see the indexing
    w2 = dict(w); w2["rcen"] = np.broadcast_to(w["rcen"][0, 0], w["rcen"].shape).copy()
    w2["alpha"] = np.broadcast_to(w["alpha"][0, 0], w["alpha"].shape).copy()
    r2 = oracle.energy_forces(gen.pack_blob(w2), sp, pos, BIG, forces=False)
    assert np.abs(r2["Ei"] - r["Ei"]).max() > 1e-4 * np.abs(r["Ei"]).max()


def test_cutoff_function_limits():
    w, blob = small_model(T=1, L=0, n_gauss=4)
    sp = np.array([0, 0], dtype=np.int32)

    def b_at(r):
        pos = np.array([[50.0, 50.0, 50.0], [50.0 + r, 50.0, 50.0]])
        return oracle.energy_forces(blob, sp, pos, BIG, forces=False, dumps=True)["b"][0, 0, :, 0]
    rc = w["rc"]
    # f_c -> 1 at r -> 0: b_n -> c0_n exp(-alpha r_n^2)
    np.testing.assert_allclose(b_at(1e-9), w["c0"][0] * np.exp(-w["alpha"][0, 0] * w["rcen"][0, 0] ** 2), rtol=1e-8)
    # f_c(rc) = 0 and f_c'(rc) = 0: b ~ (pi eps / 2 rc)^2 near the cutoff; zero beyond
    eps = 1e-4
    ratio = b_at(rc - eps) / (w["c0"][0] * np.exp(-w["alpha"][0, 0] * (rc - eps - w["rcen"][0, 0]) ** 2))
    np.testing.assert_allclose(ratio, (np.pi * eps / (2 * rc)) ** 2, rtol=1e-6)
    assert (b_at(rc + 1e-9) == 0).all()


def test_mlp_against_numpy_matmul():
    """Isolated atoms: b = 0 -> rho = 0 -> E_i = MLP_s(0); library matmul on the same blob."""
    w, blob = small_model(T=1)
    pos = np.array([[10.0, 10, 10], [60.0, 60, 60], [120.0, 120, 120]])
    sp = np.array([0, 1, 0], dtype=np.int32)
    r = oracle.energy_forces(blob, sp, pos, BIG, forces=False)
    for i in range(3):
        m = w["mlp"][0][sp[i]]
        h1 = np_pairform.silu(m["b1"]); h2 = np_pairform.silu(h1 @ m["W2"] + m["b2"])
        np.testing.assert_allclose(r["Ei"][i], (h2 @ m["W3"] + m["b3"])[0], rtol=1e-13)


def test_identity_contraction_is_plain_eann_descriptor():
    """n_orb = N_phi (L+1), Wc = identity per (n,l): rho[(n,l)] = sum_{|a|=l} mu_a b[n,a]^2 (A-1)."""
    L, nphi = 2, 4
    w, _ = small_model(T=1, L=L, n_gauss=nphi, n_orb=nphi * (L + 1))
    w["Wc"][:] = 0
    for l in range(L + 1):
        for n in range(nphi):
            w["Wc"][0, l, n, l * nphi + n] = 1.0
    blob = gen.pack_blob(w)
    pos, sp = cluster(12, 1.5, 9)
    r = oracle.energy_forces(blob, sp, pos, BIG, forces=False, dumps=True)
    rho_pair = np_pairform.energy(w, sp, pos, BIG, True)[2][0]
    np.testing.assert_allclose(r["rho"][0], rho_pair, rtol=1e-10, atol=1e-13)
    assert (r["rho"][0] >= 0).all()


# ------------------------------------------------------------------ forces and virial
def fd_force(blob, sp, pos, box, i, d, h=1e-4):
    p = pos.copy(); p[i, d] += h
    ep = oracle.energy_forces(blob, sp, p, box, forces=False)["E"]
    p[i, d] -= 2 * h
    em = oracle.energy_forces(blob, sp, p, box, forces=False)["E"]
    return -(ep - em) / (2 * h)


@pytest.mark.parametrize("which", ["cfg0", "L3T3"])
def test_forces_vs_central_differences(which, cfg0):
    if which == "cfg0":
        blob, sp, pos, box = cfg0["blob"], cfg0["species"], cfg0["pos"], cfg0["box"]
    else:
        _, blob = small_model()
        pos, sp = cluster(25, 1.8, 21); box = BIG
    r = oracle.energy_forces(blob, sp, pos, box)
    rng = np.random.default_rng(0)
    scale = max(1.0, np.abs(r["F"]).max())
    for _ in range(12):
        i, d = int(rng.integers(len(pos))), int(rng.integers(3))
        assert abs(fd_force(blob, sp, pos, box, i, d) - r["F"][i, d]) < 2e-7 * scale
    assert np.abs(r["F"].sum(0)).max() < 1e-10 * scale * len(pos)      # sum_k F_k = 0


def test_pairform_fd_matches_oracle_force(cfg0):
    """One force component from finite differences of the independent NumPy energy."""
    w, sp, pos, box = cfg0["weights"], cfg0["species"], cfg0["pos"], cfg0["box"]
    F = oracle.energy_forces(cfg0["blob"], sp, pos, box)["F"]
    h = 1e-4
    for i, d in ((3, 0), (10, 2)):
        p = pos.copy(); p[i, d] += h; ep = np_pairform.energy(w, sp, p, box)
        p[i, d] -= 2 * h; em = np_pairform.energy(w, sp, p, box)
        assert abs(-(ep - em) / (2 * h) - F[i, d]) < 2e-7 * max(1.0, np.abs(F).max())


def test_virial_diagonal_strain_periodic(cfg0):
    blob, sp, pos, box = cfg0["blob"], cfg0["species"], cfg0["pos"], cfg0["box"]
    vir = oracle.energy_forces(blob, sp, pos, box)["virial"]
    eps = 1e-5
    for a in range(3):
        Es = []
        for sgn in (+1, -1):
            scale = np.ones(3); scale[a] += sgn * eps
            Es.append(oracle.energy_forces(blob, sp, pos * scale, (box.reshape(3, 3) * scale).reshape(9), forces=False)["E"])
        dE = (Es[0] - Es[1]) / (2 * eps)
        assert abs(-dE - vir[a, a]) < 1e-6 * max(1.0, np.abs(vir).max())
    np.testing.assert_allclose(vir, vir.T, atol=1e-9 * np.abs(vir).max())


def test_virial_cluster_identity_and_zero_torque():
    _, blob = small_model()
    pos, sp = cluster(20, 1.6, 4)
    r = oracle.energy_forces(blob, sp, pos, BIG)
    # isolated cluster: virial = sum_i r_i (x) F_i, net force and net torque vanish
    np.testing.assert_allclose(r["virial"], pos.T @ r["F"], atol=1e-9 * max(1, np.abs(r["virial"]).max()))
    assert np.abs(np.cross(pos, r["F"]).sum(0)).max() < 1e-9 * max(1, np.abs(r["F"]).max()) * 100


# ------------------------------------------------------------------ symmetry
def test_translation_and_permutation(cfg0):
    blob, sp, pos, box = cfg0["blob"], cfg0["species"], cfg0["pos"], cfg0["box"]
    r0 = oracle.energy_forces(blob, sp, pos, box)
    r1 = oracle.energy_forces(blob, sp, pos + np.array([3.21, -17.7, 40.123]), box)   # left unwrapped
    assert abs(r0["E"] - r1["E"]) < 1e-10 * max(1, abs(r0["E"]))
    np.testing.assert_allclose(r0["F"], r1["F"], atol=1e-9)
    perm = np.random.default_rng(1).permutation(len(pos))
    r2 = oracle.energy_forces(blob, sp[perm], pos[perm], box)
    assert abs(r0["E"] - r2["E"]) < 1e-10 * max(1, abs(r0["E"]))
    np.testing.assert_allclose(r0["F"][perm], r2["F"], atol=1e-10)


def random_orthogonal(seed, improper):
    q, _ = np.linalg.qr(np.random.default_rng(seed).standard_normal((3, 3)))
    if (np.linalg.det(q) < 0) != improper:
        q[:, 0] *= -1
    return q


@pytest.mark.parametrize("improper", [False, True])
def test_rotation_isolated_cluster(improper):
    _, blob = small_model()
    pos, sp = cluster(22, 1.7, 8)
    r0 = oracle.energy_forces(blob, sp, pos, BIG, dumps=True)
    Q = random_orthogonal(11, improper)
    c0 = np.array([100.0, 100, 100])
    r1 = oracle.energy_forces(blob, sp, (pos - c0) @ Q.T + c0, BIG, dumps=True)
    assert abs(r0["E"] - r1["E"]) < 1e-10 * max(1, abs(r0["E"]))
    np.testing.assert_allclose(r0["F"] @ Q.T, r1["F"], atol=1e-9)
    np.testing.assert_allclose(r0["rho"], r1["rho"], rtol=1e-9, atol=1e-12)      # every rho[m] invariant
    np.testing.assert_allclose(Q @ r0["virial"] @ Q.T, r1["virial"], atol=1e-8)


def test_cubic_group_ops_periodic(cfg1):
    blob, sp, pos, box = cfg1["blob"], cfg1["species"], cfg1["pos"], cfg1["box"]
    r0 = oracle.energy_forces(blob, sp, pos, box)
    for axes, signs in (((1, 2, 0), (1, 1, 1)), ((0, 2, 1), (-1, 1, 1)), ((2, 1, 0), (1, -1, -1))):
        Q = np.zeros((3, 3))
        for r_, (c_, s_) in enumerate(zip(axes, signs)):
            Q[r_, c_] = s_
        r1 = oracle.energy_forces(blob, sp, pos @ Q.T, box)        # cubic box maps onto itself
        assert abs(r0["E"] - r1["E"]) < 1e-10 * max(1, abs(r0["E"]))
        np.testing.assert_allclose(r0["F"] @ Q.T, r1["F"], atol=1e-9)


def test_supercell_2x2x2(cfg1):
    blob, sp, pos, box = cfg1["blob"], cfg1["species"], cfg1["pos"], cfg1["box"]
    Lb = box.reshape(3, 3).diagonal()
    r0 = oracle.energy_forces(blob, sp, pos, box)
    shifts = np.array([[a, b, c] for a in (0, 1) for b in (0, 1) for c in (0, 1)]) * Lb
    pos8 = (pos[None] + shifts[:, None]).reshape(-1, 3)
    r8 = oracle.energy_forces(blob, np.tile(sp, 8), pos8, (2 * box.reshape(3, 3)).reshape(9))
    assert abs(r8["E"] - 8 * r0["E"]) < 1e-9 * max(1, abs(r0["E"]))
    np.testing.assert_allclose(r8["F"], np.tile(r0["F"], (8, 1)), atol=1e-9)
    np.testing.assert_allclose(r8["virial"], 8 * r0["virial"], atol=1e-7)


# ------------------------------------------------------------------ locality
def test_additivity_of_distant_clusters():
    w, blob = small_model(T=3)
    A, sa = cluster(10, 1.5, 1, centre=(40.0, 40, 40))
    B, sb = cluster(12, 1.5, 2, centre=(40.0 + 5 * 1.5 + 3 * w["rc"] + 15, 40, 40))
    ea = oracle.energy_forces(blob, sa, A, BIG); eb = oracle.energy_forces(blob, sb, B, BIG)
    eab = oracle.energy_forces(blob, np.concatenate([sa, sb]), np.vstack([A, B]), BIG)
    assert abs(eab["E"] - ea["E"] - eb["E"]) < 1e-11
    np.testing.assert_allclose(eab["F"], np.vstack([ea["F"], eb["F"]]), atol=1e-12)


@pytest.mark.parametrize("T", [1, 2, 3])
def test_receptive_field_is_T_times_rc(T):
    """A chain with spacing 0.8 rc (so atom k > T is also farther than T*rc from atom 0): atom 0 feels atom k iff k <= T (information moves one
    neighbour shell per layer). Moving atom k > T leaves E_0 bit-identical in
    the maths; moving atom k = T changes it."""
    w, blob = small_model(T=T, S=1, L=2)
    step = 0.8 * w["rc"]
    n = T + 3
    pos = np.array([[20.0 + step * k, 30.0 + 0.1 * k, 30.0 - 0.07 * k * k] for k in range(n)])
    sp = np.zeros(n, dtype=np.int32)
    e0 = oracle.energy_forces(blob, sp, pos, BIG)["Ei"][0]
    for k in range(1, n):
        p = pos.copy(); p[k] += np.array([0.0, 0.21, -0.13])
        ek = oracle.energy_forces(blob, sp, p, BIG)["Ei"][0]
        if k <= T:
            assert abs(ek - e0) > 100 * np.spacing(abs(e0)), f"atom {k} within T hops must matter"
        else:
            assert ek == e0, f"atom {k} beyond T*rc must not matter"


def test_perfect_fcc_symmetry():
    c = gen.make_config(4, ncell=4, T=2)
    pos, sp = gen.fcc_lattice(4, 3.61, 0.0, 0)
    r = oracle.energy_forces(c["blob"], sp, pos, c["box"], dumps=True)
    assert np.abs(r["F"]).max() < 1e-10                      # F = 0 by inversion symmetry
    assert np.ptp(r["Ei"]) < 1e-12 * max(1, abs(r["Ei"][0]))  # all sites equivalent
    lxyz, _ = oracle.monomials(c["L"])
    odd = (lxyz.sum(1) % 2) == 1
    assert np.abs(r["b"][:, :, :, odd]).max() < 1e-12        # odd-l sums cancel
    # virial of a cubic crystal is isotropic
    v = r["virial"]
    assert abs(v[0, 0] - v[1, 1]) < 1e-9 and abs(v[0, 1]) < 1e-9


# ------------------------------------------------------------------ blob validation
def test_blob_validation(cfg0):
    blob = cfg0["blob"]
    info = oracle.blob_info(blob)
    assert len(blob) == gen.blob_layout(info["S"], info["T"], info["L"], info["n_gauss"], info["n_orb"],
                                        info["H1c"], info["H2c"], info["H1e"], info["H2e"])
    assert (info["H1c"], info["H2c"], info["H1e"], info["H2e"]) == (16, 16, 32, 16)   # Table S1 shapes
    for bad in (blob[:-8], blob + b"\0" * 8, b"XXXXXXXX" + blob[8:], blob[:40]):
        with pytest.raises(ValueError):
            oracle.blob_info(bad)


def test_oracle_regression_guard():
    """Frozen oracle outputs (tests/golden/make_golden.py); regression only, not an external pin."""
    import json, os
    with open(os.path.join(os.path.dirname(__file__), "golden", "oracle_regression.json")) as f:
        gold = json.load(f)
    for k in (0, 1):
        cfg = gen.make_config(k)
        r = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
        g = gold[str(k)]
        assert abs(r["E"] - g["E"]) < 1e-9 * max(1, abs(g["E"]))
        np.testing.assert_allclose(r["F"][:3], g["F_first3"], atol=1e-9)
        assert len(oracle.neighbors(cfg["pos"], cfg["box"], cfg["rc"] + cfg["skin"])) == g["n_list_edges"]
