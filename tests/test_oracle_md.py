"""Pins of oracle/md.py (the NumPy MD driver that checks reann_md_run): facts fixed by the mathematics of the
integrator, not by the oracle itself."""
import numpy as np

from oracle import md

ACC = 9.648533e-3


def harmonic(k):
    return lambda x: (0.5 * k * float((x * x).sum()), -k * x)


def quartic_chain(n, seed=0):
    """n particles on a ring with anharmonic nearest-neighbour springs plus an on-site quartic well (smooth,
    non-integrable): a force field the thermostat tests can run on without the REANN oracle."""
    rng = np.random.default_rng(seed)
    x0 = rng.standard_normal((n, 3)) * 0.1

    def f(x):
        d = x - np.roll(x, 1, axis=0)
        r2 = (d * d).sum(1)
        pe = float((0.5 * r2 + 0.25 * r2 * r2).sum() + 0.05 * (x ** 4).sum())
        gd = (1.0 + r2)[:, None] * d
        F = -(gd - np.roll(gd, -1, axis=0)) - 0.2 * x ** 3
        return pe, F
    return x0, f


def test_velocity_verlet_exact_discrete_solution_of_the_harmonic_oscillator():
    # velocity Verlet on x'' = -w^2 x with x0 = 1, v0 = 0 gives x_n = cos(n theta), cos(theta) = 1 - (w dt)^2 / 2
    k, m, dt, n = 2.5, 3.0, 0.7, 57
    w2 = k * ACC / m
    theta = np.arccos(1.0 - 0.5 * w2 * dt * dt)
    out = md.md_run(harmonic(k), np.array([[1.0, 0.0, 0.0]]), np.zeros((1, 3)), np.array([m]), n, dt, ACC)
    assert abs(out["pos"][0, 0] - np.cos(n * theta)) < 1e-12
    # and the matching velocity: v_n = -(sin(n theta) / sin(theta)) w^2 dt (1 - (w dt)^2 / 4)
    v_exact = -np.sin(n * theta) / np.sin(theta) * w2 * dt * (1.0 - 0.25 * w2 * dt * dt)
    assert abs(out["vel"][0, 0] - v_exact) < 1e-12


def test_force_function_finite_difference():
    x0, f = quartic_chain(5, 1)
    pe, F = f(x0)
    h = 1e-6
    for idx in [(0, 0), (2, 1), (4, 2)]:
        xp, xm = x0.copy(), x0.copy()
        xp[idx] += h; xm[idx] -= h
        assert abs(-(f(xp)[0] - f(xm)[0]) / (2 * h) - F[idx]) < 1e-8


def test_time_reversibility_with_thermostat():
    n = 12
    x0, f = quartic_chain(n, 2)
    rng = np.random.default_rng(3)
    m = rng.uniform(1.0, 16.0, n)
    v0 = rng.standard_normal((n, 3)) * 0.02
    a = md.md_run(f, x0, v0, m, 40, 0.5, ACC, T_K=300.0, tau=20.0)
    b = md.md_run(f, a["pos"], -a["vel"], m, 40, 0.5, ACC, T_K=300.0, tau=20.0, xi=a["xi"], vxi=-a["vxi"])
    assert np.abs(b["pos"] - x0).max() < 1e-10
    assert np.abs(b["vel"] + v0).max() < 1e-12
    assert abs(b["vxi"]) < 1e-13


def test_conserved_quantity_converges_with_second_order():
    n = 16
    x0, f = quartic_chain(n, 4)
    rng = np.random.default_rng(5)
    m = rng.uniform(1.0, 16.0, n)
    v0 = rng.standard_normal((n, 3)) * 0.03
    errs = []
    for dt, steps in ((1.0, 100), (0.5, 200), (0.25, 400)):
        out = md.md_run(f, x0, v0, m, steps, dt, ACC, T_K=500.0, tau=25.0)
        h0 = md.kinetic_energy(v0, m, ACC) + f(x0)[0]
        errs.append(np.abs(out["conserved"] - h0).max())
    assert errs[0] > 0 and 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0, errs


def test_thermostat_fixed_point_and_direction():
    n = 8
    rng = np.random.default_rng(6)
    m = rng.uniform(1.0, 16.0, n)
    v = rng.standard_normal((n, 3))
    T = 300.0
    g, kT = 3.0 * n, md.KB_EV * T
    v *= np.sqrt(0.5 * g * kT / md.kinetic_energy(v, m, ACC))        # KE = g kT / 2 exactly: G = 0
    v1 = v.copy()
    xi, vxi = md.nose_hoover_half_step(v1, m, 0.0, 0.0, 0.25, g, kT, g * kT * 100.0, ACC)
    assert np.abs(v1 - v).max() < 1e-15 and abs(vxi) < 1e-15 and xi == 0.0
    v2 = 2.0 * v                                                       # too hot: friction positive, velocities shrink
    xi, vxi = md.nose_hoover_half_step(v2, m, 0.0, 0.0, 0.25, g, kT, g * kT * 100.0, ACC)
    assert vxi > 0 and np.all(np.abs(v2) < np.abs(2.0 * v) + 1e-300) and xi > 0
    # off switch: T_K <= 0 is plain velocity Verlet (thermostat state untouched)
    x0, f = quartic_chain(n, 7)
    out = md.md_run(f, x0, v, m, 5, 0.5, ACC, T_K=0.0)
    assert out["xi"] == 0.0 and out["vxi"] == 0.0


def test_thermostat_drives_kinetic_energy_to_target():
    n = 32
    x0, f = quartic_chain(n, 8)
    rng = np.random.default_rng(9)
    m = np.full(n, 4.0)
    T = 400.0
    g, kT = 3.0 * n, md.KB_EV * T
    v0 = rng.standard_normal((n, 3))
    v0 *= np.sqrt(2.0 * (0.5 * g * kT) / md.kinetic_energy(v0, m, ACC))   # start at twice the target temperature
    kes, x, v, xi, vxi = [], x0, v0, 0.0, 0.0
    for _ in range(60):
        out = md.md_run(f, x, v, m, 50, 1.0, ACC, T_K=T, tau=30.0, xi=xi, vxi=vxi)
        x, v, xi, vxi = out["pos"], out["vel"], out["xi"], out["vxi"]
        kes.append(out["KE"])
    mean_late = np.mean(kes[20:])
    assert abs(mean_late - 0.5 * g * kT) < 0.25 * 0.5 * g * kT, (mean_late, 0.5 * g * kT)
