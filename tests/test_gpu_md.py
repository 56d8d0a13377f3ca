"""GPU parity of reann_md_run (device-resident velocity Verlet + Nose-Hoover) against the NumPy
driver oracle/md.py fed with the float64 oracle's forces: same seeded start, trajectories compared at the end."""
import numpy as np
import pytest

import gen
import oracle
from oracle import md as omd

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def R():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import __graft_entry__ as ge
    ge.build()
    import paper_2505_06711_b200 as R
    return R


def setup(cfg, speed, fscale=1e-3):
    # forces enter the integrator scaled by 1e-3 (the random-weight potential has close contacts with |F| of
    # hundreds of eV/A; see test_md_trajectory_config2) -- the same acc_unit on both sides
    acc = fscale * gen.configs.ACC_UNIT
    vel = gen.maxwell_boltzmann(cfg["masses"], 300.0, cfg["seed_vel"]) * speed
    force_fn = lambda p: (lambda r: (r["E"], r["F"]))(oracle.energy_forces(cfg["blob"], cfg["species"], p, cfg["box"]))
    return acc, vel, force_fn


@pytest.mark.parametrize("mode", ["nvt", "nve"])
def test_md_run_matches_oracle_driver(R, mode):
    import torch
    cfg = gen.make_config(1)                       # 96 atoms, skin 1 A
    n = len(cfg["pos"])
    acc, vel0, force_fn = setup(cfg, 6.0)          # fast atoms: skin-triggered rebuilds inside the run
    ke0 = omd.kinetic_energy(vel0, cfg["masses"], acc)
    kT = 0.25 * ke0 / (1.5 * n) if mode == "nvt" else 0.0     # target: a quarter of the initial temperature
    n_steps, dt, tau = 40, 0.5, 10.0
    ref = omd.md_run(force_fn, cfg["pos"], vel0, cfg["masses"], n_steps, dt, acc, T_K=kT / omd.KB_EV, tau=tau)

    m = R.Reann.from_config(cfg)
    pos = torch.tensor(cfg["pos"], device="cuda"); vel = torch.tensor(vel0, device="cuda")
    inv_m = torch.tensor(1.0 / cfg["masses"], device="cuda")
    F = torch.zeros((n, 3), dtype=torch.float64, device="cuda"); vir = torch.zeros(9, dtype=torch.float64, device="cuda")
    st = m.md_run(pos, vel, inv_m, cfg["box"], n_steps, dt, acc, kT=kT, tau=tau, F=F, virial=vir)
    torch.cuda.synchronize()
    dp = np.abs(pos.cpu().numpy() - ref["pos"]).max()
    dv = np.abs(vel.cpu().numpy() - ref["vel"]).max()
    dF = np.abs(F.cpu().numpy() - ref["F"]).max()
    print(f"[md {mode}] max|dpos|={dp:.2e} A max|dvel|={dv:.2e} A/fs max|dF|={dF:.2e} xi={st['xi']:.6f}/{ref['xi']:.6f} "
          f"vxi={st['vxi']:.6e}/{ref['vxi']:.6e} KE={st['kinetic']:.6f}/{ref['KE']:.6f} rebuilds={st['n_rebuilds']}")
    # FP32 forces (<= 5e-4 eV/A off) integrated over 20 fs with the scaled acc_unit: positions agree far below 1e-5 A
    assert dp < 1e-5 and dv < 1e-6 and dF < 5e-4
    assert st["n_steps_done"] == n_steps and st["n_rebuilds"] >= 2
    assert abs(st["kinetic"] - ref["KE"]) < 1e-6 * max(1.0, ref["KE"])
    assert abs(st["potential"] - ref["PE"]) < 1e-6 * n * max(1.0, abs(ref["PE"]) / n)
    assert abs(st["conserved"] - ref["conserved"][-1]) < 2e-6 * n * max(1.0, abs(ref["PE"]) / n)
    if mode == "nvt":
        assert abs(st["xi"] - ref["xi"]) < 1e-8 + 1e-6 * abs(ref["xi"]) and abs(st["vxi"] - ref["vxi"]) < 1e-9 + 1e-6 * abs(ref["vxi"])
        assert ref["KE"] < 0.9 * ke0          # the thermostat did act
    else:
        assert st["xi"] == 0.0 and st["vxi"] == 0.0
    m.close()


def test_config2_protocol_100_steps_300K(R):
    """BASELINE.json config 2: 1024 H2O, 100 velocity-Verlet steps of 0.5 fs from a seeded Maxwell-Boltzmann start at
    300 K, skin-triggered rebuilds inside the run; the whole trajectory against the oracle driver (same scaled
    acc_unit on both sides, see setup())."""
    import torch
    cfg = gen.make_config(2)
    n = len(cfg["pos"])
    # forces scaled by 1e-4 as in bench.py: displacements stay thermal (with 1e-3 the close contacts of the random-weight
    # potential fling atoms 4 A within 50 fs and the trajectory is no longer comparable)
    acc, vel0, force_fn = setup(cfg, 1.0, 1e-4)
    ref = omd.md_run(force_fn, cfg["pos"], vel0, cfg["masses"], 100, 0.5, acc)
    m = R.Reann.from_config(cfg)
    pos = torch.tensor(cfg["pos"], device="cuda"); vel = torch.tensor(vel0, device="cuda")
    inv_m = torch.tensor(1.0 / cfg["masses"], device="cuda")
    F = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    st = m.md_run(pos, vel, inv_m, cfg["box"], 100, 0.5, acc, F=F)
    disp = np.sqrt(((ref["pos"] - cfg["pos"]) ** 2).sum(1)).max()
    dp = np.abs(pos.cpu().numpy() - ref["pos"]).max(); dv = np.abs(vel.cpu().numpy() - ref["vel"]).max()
    dF = np.abs(F.cpu().numpy() - ref["F"]).max()
    print(f"[md cfg2] 100 steps: max displacement {disp:.2f} A, rebuilds {st['n_rebuilds']}, max|dpos|={dp:.2e} max|dvel|={dv:.2e} max|dF|={dF:.2e}")
    assert disp > 0.5 * cfg["skin"] and st["n_rebuilds"] >= 2       # the initial build and at least one triggered by the skin rule
    assert dp < 1e-5 and dv < 1e-6 and dF < 5e-4
    assert abs(st["potential"] - ref["PE"]) < 1e-6 * n * max(1.0, abs(ref["PE"]) / n)
    m.close()


def test_md_run_continuation_equals_one_run(R):
    """Two calls of 15 + 25 steps (thermostat state passed on) == one call of 40 steps, bit for bit: the second
    call re-evaluates the forces at its start positions, which are the ones the first call ended with."""
    import torch
    cfg = gen.make_config(1)
    n = len(cfg["pos"])
    acc, vel0, _ = setup(cfg, 3.0)
    kT = 0.5 * omd.kinetic_energy(vel0, cfg["masses"], acc) / (1.5 * n)
    outs = []
    for split in ((40,), (15, 25)):
        m = R.Reann.from_config(cfg)
        pos = torch.tensor(cfg["pos"], device="cuda"); vel = torch.tensor(vel0, device="cuda")
        inv_m = torch.tensor(1.0 / cfg["masses"], device="cuda")
        F = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
        xi = vxi = 0.0
        for k in split:
            st = m.md_run(pos, vel, inv_m, cfg["box"], k, 0.5, acc, kT=kT, tau=15.0, F=F, xi=xi, vxi=vxi)
            xi, vxi = st["xi"], st["vxi"]
        outs.append((pos.cpu().numpy(), vel.cpu().numpy(), xi, vxi))
        m.close()
    assert np.abs(outs[0][0] - outs[1][0]).max() < 1e-9 and np.abs(outs[0][1] - outs[1][1]).max() < 1e-10
    assert abs(outs[0][2] - outs[1][2]) < 1e-12 and abs(outs[0][3] - outs[1][3]) < 1e-13


def test_md_run_rejects_host_pointers(R):
    cfg = gen.make_config(1)
    m = R.Reann.from_config(cfg)
    n = len(cfg["pos"])
    with pytest.raises(R.ReannError) as e:
        m.md_run(cfg["pos"].copy(), np.zeros((n, 3)), 1.0 / cfg["masses"], cfg["box"], 1, 0.5, 1e-3, F=np.zeros((n, 3)))
    assert e.value.code == R.REANN_ERR_ARG
    m.close()
