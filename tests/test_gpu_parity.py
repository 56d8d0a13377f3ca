"""GPU parity tests: the CUDA path (through the C ABI) against the float64 oracle on the same
seeded inputs. Tolerances: BASELINE.json north_star (energy 1e-6 eV/atom relative, forces
5e-4 eV/A max-abs, FP32 path); neighbour sets exact."""
import numpy as np
import pytest

import gen
import oracle
from gpu_util import E_TOL_REL, F_TOL, check_parity, gpu_rows, open_cluster

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def R():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import __graft_entry__ as ge
    ge.build()
    import paper_2505_06711_b200 as R
    return R


def small_cfg(S=2, T=3, L=3, n_gauss=5, H=(12, 10), Hc=(9, 11), rc=3.5, skin=0.5, n=60, box=14.0, seed=5,
              radial_jitter=0.15):
    """Radial tables differ per (layer, neighbour species) by 15-30 % (reading A-3 is visible to the parity)."""
    rng = np.random.default_rng(seed)
    w = gen.make_weights(S=S, T=T, L=L, n_gauss=n_gauss, n_orb=gen.n_orb_default(n_gauss, L), H=H, Hc=Hc, rc=rc,
                         nbar=12.0, seed=seed + 1, wc_gain=[2.0] * T, c_gain=[2.0] * (T - 1), e_scale=3.0,
                         radial_jitter=radial_jitter)
    return dict(pos=rng.random((n, 3)) * box, species=rng.integers(0, S, n).astype(np.int32),
                box=np.diag([box] * 3).reshape(9), rc=rc, skin=skin, T=T, L=L, n_gauss=n_gauss, blob=gen.pack_blob(w),
                weights=w)


def run(R, cfg, pos=None):
    m = R.Reann.from_config(cfg)
    p = cfg["pos"] if pos is None else pos
    m.build_neighbors(p, cfg["box"])
    out = m.energy_forces(p, cfg["box"])
    return m, out


# ------------------------------------------------------------------ neighbour sets, exact
@pytest.mark.parametrize("case", ["cfg0", "cfg1", "w150", "w260", "w1024", "fcc6", "slab", "unwrapped"])
def test_neighbor_pair_sets_exact(R, case):
    if case == "cfg0": cfg = gen.make_config(0)
    elif case == "cfg1": cfg = gen.make_config(1)             # box < 2(rc+skin): duplicate images
    elif case == "w150": cfg = gen.make_config(2, n_mol=150)  # 2 cells per dimension
    elif case == "w260": cfg = gen.make_config(2, n_mol=260)
    elif case == "w1024": cfg = gen.make_config(2)            # 3 cells per dimension, 3072 atoms
    elif case == "fcc6": cfg = gen.make_config(4, ncell=6)
    elif case == "slab": cfg = gen.make_config(5, n_mol=400)  # vacuum gap: empty cells
    else:
        cfg = gen.make_config(1)
        k = np.random.default_rng(3).integers(-2, 3, size=cfg["pos"].shape)
        cfg["pos"] = cfg["pos"] + k * cfg["box"].reshape(3, 3).diagonal()
    m = R.Reann.from_config(cfg)
    m.build_neighbors(cfg["pos"], cfg["box"])
    rows = gpu_rows(m)
    ref = oracle.neighbors(cfg["pos"], cfg["box"], cfg["rc"] + cfg["skin"], "cell")
    assert rows.shape == ref.shape
    assert (rows == ref).all()
    st = m.stats()
    assert st["n_edges_list"] == len(ref) and st["n_ext"] >= st["n_atoms"]
    m.close()


# ------------------------------------------------------------------ energy / forces / virial
@pytest.mark.parametrize("case", ["cfg0", "cfg0j", "cfg1", "cfg2", "cfg2j", "cfg3r", "cfg3rj", "cfg4r_T1", "cfg4r_T3",
                                  "cfg4r_T6", "cfg5r", "small_L3", "small_L0", "small_L1_S1", "small_n4", "small_n12"])
def test_energy_forces_virial_parity(R, case):
    """`j` cases: radial tables that differ per (layer, neighbour species) -- with identical rows (the BASELINE
    recipe) an indexing mistake in the edge kernels (s_j -> s_i, t -> 0) would be invisible."""
    if case.startswith("cfg") and case[3:].isdigit(): cfg = gen.make_config(int(case[3:]))
    elif case == "cfg0j": cfg = gen.make_config(0, radial_jitter=0.15)
    elif case == "cfg2j": cfg = gen.make_config(2, n_mol=300, radial_jitter=0.1)   # N_phi = 16, L = 2: mma.sync edge forward
    elif case == "cfg3rj": cfg = gen.make_config(3, n_mol=500, radial_jitter=0.1)  # N_phi = 16, L = 3
    elif case == "cfg3r": cfg = gen.make_config(3, n_mol=700)         # L=3, 16 Gaussians, ragged tiles
    elif case.startswith("cfg4r"): cfg = gen.make_config(4, ncell=7, T=int(case[-1]))
    elif case == "cfg5r": cfg = gen.make_config(5, n_mol=900)
    elif case == "small_L3": cfg = small_cfg()
    elif case == "small_L0": cfg = small_cfg(L=0, n_gauss=8, T=2)
    elif case == "small_L1_S1": cfg = small_cfg(L=1, S=1, n_gauss=16, T=2, H=(64, 32), Hc=(16, 128))
    elif case == "small_n4": cfg = small_cfg(L=2, n_gauss=3, T=4)
    else: cfg = small_cfg(L=3, n_gauss=11, T=2, H=(100, 20), Hc=(33, 65))
    m, out = run(R, cfg)
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    check_parity(out, ref, m.n, case)
    # per-atom energies: E_i carries FP32 rounding of a value of order |E_i|: 4e-6 * max(1, |E_i|)
    Ei = m.atomic_energies()
    assert np.abs(Ei - ref["Ei"]).max() <= 4e-6 * max(1.0, np.abs(ref["Ei"]).max())
    m.close()


def test_edge_cases_empty_single_and_isolated(R):
    cfg = small_cfg(n=1)
    m, (E, F, vir) = run(R, cfg)                       # one atom: no edges, E = MLP(0), F = 0
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    assert abs(E - ref["E"]) <= 1e-6 * max(1, abs(ref["E"])) and np.abs(F).max() == 0 and np.abs(vir).max() == 0
    m.close()
    cfg = small_cfg(n=0)
    m, (E, F, vir) = run(R, cfg)                       # empty system
    assert E == 0.0 and F.shape == (0, 3)
    m.close()
    cfg = small_cfg(n=65, box=60.0)                    # dilute: most rows empty, one ragged dense tile
    m, out = run(R, cfg)
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    check_parity(out, ref, m.n, "dilute")
    m.close()


def test_bitwise_determinism_and_host_device_equivalence(R):
    import torch
    cfg = gen.make_config(2, n_mol=300)
    m = R.Reann.from_config(cfg)
    m.build_neighbors(cfg["pos"], cfg["box"])
    E0, F0, V0 = m.energy_forces(cfg["pos"], cfg["box"])
    for _ in range(2):
        E1, F1, V1 = m.energy_forces(cfg["pos"], cfg["box"])
        assert E1 == E0 and (F1 == F0).all() and (V1 == V0).all()
    m.build_neighbors(cfg["pos"], cfg["box"])            # rebuild: same list, same bits
    E1, F1, V1 = m.energy_forces(cfg["pos"], cfg["box"])
    assert E1 == E0 and (F1 == F0).all()
    m2 = R.Reann.from_config(cfg)                        # fresh handle, device pointers
    pos = torch.tensor(cfg["pos"], device="cuda")
    E = torch.zeros(1, dtype=torch.float64, device="cuda"); F = torch.zeros((m.n, 3), dtype=torch.float64, device="cuda")
    V = torch.zeros(9, dtype=torch.float64, device="cuda")
    m2.build_neighbors(pos, cfg["box"])
    m2.energy_forces(pos, cfg["box"], E, F, V)
    torch.cuda.synchronize()
    assert E.item() == E0 and (F.cpu().numpy() == F0).all() and (V.cpu().numpy().reshape(3, 3) == V0).all()
    m.close(); m2.close()


def test_skin_logic_stale_list_and_automatic_rebuild(R):
    cfg = gen.make_config(2, n_mol=300)                  # skin = 2.0
    rng = np.random.default_rng(9)
    m = R.Reann.from_config(cfg)
    m.build_neighbors(cfg["pos"], cfg["box"])
    step = rng.standard_normal(cfg["pos"].shape)
    step *= 0.9 / np.linalg.norm(step, axis=1, keepdims=True)     # every atom moves 0.9 A < skin/2
    pos1 = cfg["pos"] + step
    out_stale = m.energy_forces(pos1, cfg["box"])
    assert m.stats()["n_rebuilds"] == 1                           # stale but valid list was used
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], pos1, cfg["box"])
    check_parity(out_stale, ref, m.n, "stale list")
    m.build_neighbors(pos1, cfg["box"])
    out_fresh = m.energy_forces(pos1, cfg["box"])
    assert abs(out_fresh[0] - out_stale[0]) / m.n <= E_TOL_REL and np.abs(out_fresh[1] - out_stale[1]).max() <= F_TOL
    n_before = m.stats()["n_rebuilds"]
    pos2 = pos1.copy(); pos2[17] += np.array([0.0, 1.05, 0.0])    # one atom beyond skin/2 -> rebuild inside the call
    out2 = m.energy_forces(pos2, cfg["box"])
    assert m.stats()["n_rebuilds"] == n_before + 1
    check_parity(out2, oracle.energy_forces(cfg["blob"], cfg["species"], pos2, cfg["box"]), m.n, "auto rebuild")
    box2 = cfg["box"] * 1.01                                      # box change -> rebuild
    out3 = m.energy_forces(pos2, box2)
    assert m.stats()["n_rebuilds"] == n_before + 2
    check_parity(out3, oracle.energy_forces(cfg["blob"], cfg["species"], pos2, box2), m.n, "box change")
    m.close()


def test_unwrapped_positions_and_permutation(R):
    cfg = gen.make_config(1)
    m, (E0, F0, _) = run(R, cfg)
    rng = np.random.default_rng(2)
    k = rng.integers(-3, 4, size=cfg["pos"].shape)
    pos_u = cfg["pos"] + k * cfg["box"].reshape(3, 3).diagonal()
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], pos_u, cfg["box"])
    m1, out1 = run(R, cfg, pos_u)
    check_parity(out1, ref, m.n, "unwrapped")
    perm = rng.permutation(m.n)
    cfgp = dict(cfg); cfgp["pos"] = cfg["pos"][perm]; cfgp["species"] = cfg["species"][perm].copy()
    m2, (E2, F2, _) = run(R, cfgp)
    assert abs(E2 - E0) / m.n <= E_TOL_REL and np.abs(F2 - F0[perm]).max() <= F_TOL
    for x in (m, m1, m2): x.close()


def test_error_codes(R):
    cfg = gen.make_config(1)
    m = R.Reann.from_config(cfg)
    with pytest.raises(R.ReannError) as e:
        m.energy_forces(cfg["pos"], cfg["box"])
    assert e.value.code == R.REANN_ERR_NO_NEIGHBORS
    with pytest.raises(R.ReannError) as e:
        m.build_neighbors(cfg["pos"], cfg["box"] * 0.5)            # 4.93 < rc + skin
    assert e.value.code == R.REANN_ERR_BOX
    tric = cfg["box"].copy(); tric[1] = 0.5
    with pytest.raises(R.ReannError) as e:
        m.build_neighbors(cfg["pos"], tric)
    assert e.value.code == R.REANN_ERR_UNSUPPORTED
    m.close()
    with pytest.raises(R.ReannError) as e:
        R.reann_create(cfg["blob"], cfg["species"], cfg["rc"], cfg["skin"], cfg["T"] + 1, cfg["L"], cfg["n_gauss"])
    assert e.value.code == R.REANN_ERR_WEIGHTS
    with pytest.raises(R.ReannError) as e:
        R.reann_create(cfg["blob"][:-8], cfg["species"], cfg["rc"], cfg["skin"], cfg["T"], cfg["L"], cfg["n_gauss"])
    assert e.value.code == R.REANN_ERR_WEIGHTS
    bad = cfg["species"].copy(); bad[3] = 7
    with pytest.raises(R.ReannError) as e:
        R.reann_create(cfg["blob"], bad, cfg["rc"], cfg["skin"], cfg["T"], cfg["L"], cfg["n_gauss"])
    assert e.value.code == R.REANN_ERR_ARG


def test_md_trajectory_config2(R):
    """Config 2: velocity Verlet (0.5 fs, 300 K) on the device; parity at step 0, at every rebuild and
    at the end by feeding the GPU positions to the oracle; rebuild steps equal the host-side skin rule."""
    import torch
    cfg = gen.make_config(2)
    n = len(cfg["pos"])
    m = R.Reann.from_config(cfg)
    pos = torch.tensor(cfg["pos"], device="cuda")
    # 8x thermal speeds so that several skin-triggered rebuilds fall inside 40 steps; the integrator uses
    # forces scaled by 1e-3 (the random-weight potential has close contacts with |F| of hundreds of eV/A,
    # unscaled dynamics would blow up within a few steps). The E+F evaluation under test is unaffected.
    vel = torch.tensor(gen.maxwell_boltzmann(cfg["masses"], 300.0, cfg["seed_vel"]) * 8.0, device="cuda")
    acc = 1e-3 * gen.configs.ACC_UNIT
    inv_m = torch.tensor(1.0 / cfg["masses"], device="cuda")
    E = torch.zeros(1, dtype=torch.float64, device="cuda"); F = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    m.build_neighbors(pos, cfg["box"])
    m.energy_forces(pos, cfg["box"], E, F)
    pos_build = pos.cpu().numpy().copy()
    expected_rebuilds, checked = 1, 0
    for step in range(40):
        m.verlet(pos, vel, F, inv_m, 0.5, acc, True)
        p = pos.cpu().numpy()
        moved = ((p - pos_build) ** 2).sum(1).max() > (0.5 * cfg["skin"]) ** 2
        m.energy_forces(pos, cfg["box"], E, F)
        m.verlet(pos, vel, F, inv_m, 0.5, acc, False)
        if moved:
            expected_rebuilds += 1
            pos_build = p.copy()
        assert m.stats()["n_rebuilds"] == expected_rebuilds, step
        if moved or step in (0, 39):
            ref = oracle.energy_forces(cfg["blob"], cfg["species"], p, cfg["box"])
            check_parity((E.item(), F.cpu().numpy(), None), ref, n, f"md step {step}")
            checked += 1
    assert expected_rebuilds >= 2 and checked >= 3
    m.close()


def test_full_size_config3_sampled(R):
    """Config 3 at full size (192 000 atoms, the bench launch configuration): E_i and F_k of sampled
    atoms against the oracle on an open cluster cut around them (exact by the receptive field T*rc,
    PAPER.md:23), plus global invariants."""
    cfg = gen.make_config(3)
    m, (E, F, vir) = run(R, cfg)
    n = m.n
    Ei = m.atomic_energies()
    assert abs(Ei.sum() - E) <= 1e-9 * max(1.0, abs(E))
    assert np.abs(F.sum(0)).max() <= 1e-6 * n                     # sum_k F_k = 0 up to FP32 rounding
    assert np.abs(vir - vir.T).max() <= 2e-5 * max(np.abs(vir).max(), n)
    st = m.stats()
    assert st["n_edges_rc"] > 80 * n and st["n_edges_list"] > 190 * n
    T, rc = cfg["T"], cfg["rc"]
    centre = cfg["pos"][12345]
    r_f, r_e = 4.0, 4.0 + T * rc                                   # forces inside r_f; E_i inside r_e
    sel, cpos, cbox = open_cluster(cfg["pos"], cfg["species"], cfg["box"], centre, r_f + 2 * T * rc + 0.5)
    ref = oracle.energy_forces(cfg["blob"], cfg["species"][sel], cpos, cbox)
    d = np.linalg.norm(cpos - cpos[np.nonzero(sel == 12345)[0][0]], axis=1)
    in_e, in_f = d < r_e, d < r_f
    assert in_f.sum() >= 10 and in_e.sum() >= 1000
    assert np.abs(Ei[sel][in_e] - ref["Ei"][in_e]).max() <= 4e-6 * max(1.0, np.abs(ref["Ei"][in_e]).max())
    assert np.abs(F[sel][in_f] - ref["F"][in_f]).max() <= F_TOL
    m.close()


def test_full_size_config4_sampled(R):
    """Config 4 at full size (4 000 000 fcc atoms, T = 3 of the sweep): sampled E_i / F_k against the oracle on an
    open cluster (receptive field T*rc), the per-atom neighbour count of the perturbed lattice,
    and global invariants."""
    cfg = gen.make_config(4, T=3)
    m, (E, F, vir) = run(R, cfg)
    n = m.n
    assert n == 4_000_000
    Ei = m.atomic_energies()
    assert abs(Ei.sum() - E) <= 1e-9 * max(1.0, abs(E))
    assert np.abs(F.sum(0)).max() <= 1e-6 * n
    st = m.stats()
    assert 77.5 * n < st["n_edges_list"] < 78.5 * n              # shells 12+6+24+12+24 within rc+skin = 6 A
    assert 42 * n < st["n_edges_rc"] < 48 * n
    T, rc = cfg["T"], cfg["rc"]
    k0 = 2_345_678
    centre = cfg["pos"][k0]
    r_f, r_e = 3.0, 3.0 + T * rc
    sel, cpos, cbox = open_cluster(cfg["pos"], cfg["species"], cfg["box"], centre, r_f + 2 * T * rc + 0.5)
    ref = oracle.energy_forces(cfg["blob"], cfg["species"][sel], cpos, cbox)
    d = np.linalg.norm(cpos - cpos[np.nonzero(sel == k0)[0][0]], axis=1)
    in_e, in_f = d < r_e, d < r_f
    assert in_f.sum() >= 10 and in_e.sum() >= 1000
    assert np.abs(Ei[sel][in_e] - ref["Ei"][in_e]).max() <= 4e-6 * max(1.0, np.abs(ref["Ei"][in_e]).max())
    assert np.abs(F[sel][in_f] - ref["F"][in_f]).max() <= F_TOL
    m.close()


@pytest.mark.parametrize("env", [{"REANN_EDGE": "mma", "REANN_EDGE_FWD": "simt"}, {"REANN_DENSE": "simt"}],
                         ids=["edge_bwd_mma+edge_fwd_simt", "dense_simt"])
def test_non_default_kernel_variants_parity(env):
    """The kernels behind the library's environment switches: REANN_EDGE=mma (mma.sync 3xTF32 edge
    backward) with REANN_EDGE_FWD=simt (FP32 ALU edge forward), and REANN_DENSE=simt (FP32 ALU GEMM chain). The
    switches are read once per process, hence the subprocess. Same parity gates as the default kernels."""
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = (
        "import sys; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
        "import gen, oracle\nimport paper_2505_06711_b200 as R\nfrom gpu_util import check_parity\n"
        "for k, kw in ((3, dict(n_mol=700)), (2, dict(n_mol=300))):\n"
        "    cfg = gen.make_config(k, **kw)\n"
        "    m = R.Reann.from_config(cfg); m.build_neighbors(cfg['pos'], cfg['box'])\n"
        "    out = m.energy_forces(cfg['pos'], cfg['box'])\n"
        "    ref = oracle.energy_forces(cfg['blob'], cfg['species'], cfg['pos'], cfg['box'])\n"
        "    check_parity(out, ref, m.n, 'variant cfg%%d' %% k); m.close()\n" % (root, os.path.join(root, "tests")))
    r = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, **env), capture_output=True, text=True,
                       timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("[parity] variant") == 2


def test_stash_chunks_memory_limited_path(R, monkeypatch):
    """Config 5 needs the kappa stash in chunks of atoms to fit 180 GB; REANN_STASH_CHUNKS forces the same code
    path on a small system: parity with the oracle, and the same result as the unchunked run up to the
    summation order of cbar."""
    cfg = gen.make_config(5, n_mol=900)
    m1, (E1, F1, V1) = run(R, cfg)
    m1.close()
    monkeypatch.setenv("REANN_STASH_CHUNKS", "3")
    m3, out3 = run(R, cfg)
    ref = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    check_parity(out3, ref, m3.n, "stash chunks = 3")
    E3, F3, V3 = out3
    assert abs(E3 - E1) <= 1e-9 * max(1.0, abs(E1)) * m3.n
    assert np.abs(F3 - F1).max() <= 2e-5 and np.abs(V3 - V1).max() <= 1e-5 * max(1.0, np.abs(V1).max())
    E3b, F3b, _ = m3.energy_forces(cfg["pos"], cfg["box"])       # deterministic for a fixed chunk count
    assert E3b == E3 and (F3b == F3).all()
    m3.close()
