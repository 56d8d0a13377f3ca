"""GPU parity on triclinic cells (reading B-9): exact pair sets and E / F / virial
against the oracle, whose triclinic arithmetic is pinned in tests/test_oracle_triclinic.py."""
import numpy as np
import pytest

import gen
import oracle
from gpu_util import check_parity, gpu_rows

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def R():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import __graft_entry__ as ge
    ge.build()
    import paper_2505_06711_b200 as R
    return R


def unit_force_cfg(k, **kw):
    """Config k with the energy layer rescaled (oracle only) until rms|F| = 1 eV/A, as the recipe of SURVEY.md 8(d)
    prescribes: the calibrated gains of gen/calib.json belong to the orthorhombic geometry of each config."""
    cfg = gen.make_config(k, **kw)
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    g = dict(cfg["gains"]); g["e"] = g.get("e", 1.0) / np.sqrt((ref["F"] ** 2).sum(1).mean())
    return gen.make_config(k, gains=g, **kw)


def tric_cfg(case):
    if case == "w_small":   # one cell per direction, duplicate images, strong tilt
        return gen.make_config(1, tilt=(2.0, -1.5, 2.5))
    if case == "w300":      # 2 cells per direction
        return gen.make_config(2, n_mol=300, tilt=(4.0, -3.0, 5.0))
    if case == "w1024":     # 3 cells per direction, negative and positive tilts
        return gen.make_config(2, tilt=(-9.0, 6.0, 8.0))
    if case == "w700_L3":   # config 3 shapes (L = 3, 16 Gaussians)
        return unit_force_cfg(3, n_mol=700, tilt=(5.0, 4.0, -6.0))
    if case == "fcc7":      # the same fcc crystal in a sheared cell: tilts are multiples of the lattice constant
        return gen.make_config(4, ncell=7, T=3, tilt=(2 * 3.61, -3.61, 3 * 3.61))
    if case == "slab":      # vacuum gap: empty cells
        return unit_force_cfg(5, n_mol=400, tilt=(3.0, 0.0, 0.0))
    if case == "outside":   # atoms several periods outside the cell: caller-frame shifts
        cfg = gen.make_config(1, tilt=(2.0, -1.5, 2.5))
        k = np.random.default_rng(3).integers(-2, 3, size=cfg["pos"].shape)
        cfg["pos"] = cfg["pos"] + k @ cfg["box"].reshape(3, 3)
        return cfg
    raise KeyError(case)


@pytest.mark.parametrize("case", ["w_small", "w300", "w1024", "fcc7", "slab", "outside"])
def test_neighbor_pair_sets_exact_triclinic(R, case):
    cfg = tric_cfg(case)
    m = R.Reann.from_config(cfg)
    m.build_neighbors(cfg["pos"], cfg["box"])
    rows = gpu_rows(m)
    ref = oracle.neighbors(cfg["pos"], cfg["box"], cfg["rc"] + cfg["skin"], "cell")
    assert rows.shape == ref.shape
    assert (rows == ref).all()
    m.close()


@pytest.mark.parametrize("case", ["w_small", "w300", "w700_L3", "fcc7", "slab", "outside"])
def test_energy_forces_virial_parity_triclinic(R, case):
    cfg = tric_cfg(case)
    m = R.Reann.from_config(cfg)
    m.build_neighbors(cfg["pos"], cfg["box"])
    out = m.energy_forces(cfg["pos"], cfg["box"])
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    check_parity(out, ref, m.n, "triclinic " + case)
    assert np.abs(m.atomic_energies() - ref["Ei"]).max() <= 4e-6 * max(1.0, np.abs(ref["Ei"]).max())
    m.close()


def test_same_crystal_in_cubic_and_sheared_cell(R):
    """The same periodic structure (thermally displaced fcc) in its cubic cell (a, b, c) and in the sheared cell
    (a, b + a, c - a): the same list lengths and, within the FP32 gates, the same energy and forces."""
    a = gen.make_config(4, ncell=7, T=2)
    L = a["box"][0]
    b = gen.make_config(4, ncell=7, T=2, tilt=(L, -L, 0.0))
    res = []
    for cfg in (a, b):
        m = R.Reann.from_config(cfg)
        m.build_neighbors(cfg["pos"], cfg["box"])
        E, F, V = m.energy_forces(cfg["pos"], cfg["box"])
        res.append((E, F, V, m.stats()["n_edges_list"], m.stats()["n_edges_rc"]))
        m.close()
    assert res[0][3] == res[1][3] and res[0][4] == res[1][4]
    assert abs(res[0][0] - res[1][0]) / a["pos"].shape[0] < 2e-6      # each within 1e-6 eV/atom of the exact value
    assert np.abs(res[0][1] - res[1][1]).max() < 5e-4
    assert np.abs(res[0][2] - res[1][2]).max() < 1e-4 * max(np.abs(res[0][2]).max(), a["pos"].shape[0])


def test_md_with_rebuilds_in_a_triclinic_cell(R):
    import torch
    from oracle import md as omd
    cfg = tric_cfg("w_small")
    n = len(cfg["pos"])
    acc = 1e-3 * gen.configs.ACC_UNIT
    vel0 = gen.maxwell_boltzmann(cfg["masses"], 300.0, cfg["seed_vel"]) * 6.0
    force_fn = lambda p: (lambda r: (r["E"], r["F"]))(oracle.energy_forces(cfg["blob"], cfg["species"], p, cfg["box"]))
    ref = omd.md_run(force_fn, cfg["pos"], vel0, cfg["masses"], 30, 0.5, acc)
    m = R.Reann.from_config(cfg)
    pos = torch.tensor(cfg["pos"], device="cuda"); vel = torch.tensor(vel0, device="cuda")
    inv_m = torch.tensor(1.0 / cfg["masses"], device="cuda")
    F = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    st = m.md_run(pos, vel, inv_m, cfg["box"], 30, 0.5, acc, F=F)
    assert st["n_rebuilds"] >= 2
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < 1e-5 and np.abs(F.cpu().numpy() - ref["F"]).max() < 5e-4
    m.close()


def test_box_errors_triclinic(R):
    cfg = gen.make_config(1)
    m = R.Reann.from_config(cfg)
    L = cfg["box"][0]
    thin = cfg["box"].copy(); thin[3] = 1.2 * L              # faces spanned by b, c come closer than rc + skin
    with pytest.raises(R.ReannError) as e:
        m.build_neighbors(cfg["pos"], thin)
    assert e.value.code == R.REANN_ERR_BOX
    up = cfg["box"].copy(); up[5] = 0.3
    with pytest.raises(R.ReannError) as e:
        m.build_neighbors(cfg["pos"], up)
    assert e.value.code == R.REANN_ERR_UNSUPPORTED
    m.close()
