"""oracle/md.py -- TEST INFRASTRUCTURE ONLY (imported by tests/, never by the product path).

Plain NumPy float64 molecular dynamics driver used to check `reann_md_run` (the
paper runs its potentials in NVT molecular dynamics at 300 K, with the MD
driver of section 4.2). The paper does not print the integrator (it uses LAMMPS), so the
reading taken here (B-8) is the textbook one:

  * velocity Verlet:            v += dt/2 a(x);  x += dt v;  a = F(x)/m;  v += dt/2 a(x)
  * Nose-Hoover thermostat (one thermostat variable xi with "velocity" vxi), applied as a half step
    before and after the velocity-Verlet step (the Trotter splitting of Martyna, Tuckerman, Tobias and
    Klein, Mol. Phys. 87, 1117 (1996), with one thermostat and no higher-order sub-stepping):
        dv/dt = -vxi v,   dvxi/dt = (2 KE - g kB T) / Q,   dxi/dt = vxi,   Q = g kB T tau^2
    half step of length h = dt/2:  vxi += h/2 G(KE);  v *= exp(-h vxi) (so KE *= exp(-2 h vxi));
                                   xi += h vxi;  vxi += h/2 G(KE)
  * g = 3 N degrees of freedom; conserved quantity H' = KE + PE + Q vxi^2 / 2 + g kB T xi.

Units: Angstrom, fs, amu, eV; `acc_unit` converts eV/(Angstrom amu) to Angstrom/fs^2, so
KE [eV] = sum m v^2 / (2 acc_unit). T_K <= 0 switches the thermostat off (NVE).

Pins (tests/test_oracle_md.py): the exact discrete solution of velocity Verlet for a harmonic oscillator,
time reversibility, second-order convergence of H', the fixed point of the thermostat half step.
"""
from __future__ import annotations

import numpy as np

KB_EV = 8.617333e-5   # eV/K (same constant as gen/configs.py: an input convention, not method arithmetic)


def kinetic_energy(vel: np.ndarray, masses: np.ndarray, acc_unit: float) -> float:
    return float((masses[:, None] * vel * vel).sum() / (2.0 * acc_unit))


def nose_hoover_half_step(vel, masses, xi, vxi, h, g, kT, Q, acc_unit):
    """One thermostat half step of length h (in place on vel); returns (xi, vxi)."""
    ke2 = 2.0 * kinetic_energy(vel, masses, acc_unit)
    vxi = vxi + 0.5 * h * (ke2 - g * kT) / Q
    s = np.exp(-h * vxi)
    vel *= s
    ke2 *= s * s
    xi = xi + h * vxi
    vxi = vxi + 0.5 * h * (ke2 - g * kT) / Q
    return xi, vxi


def md_run(force_fn, pos, vel, masses, n_steps, dt, acc_unit, T_K=0.0, tau=100.0, xi=0.0, vxi=0.0, F0=None):
    """n_steps of (thermostatted) velocity Verlet. force_fn(pos) -> (PE, F[N,3]).
    Returns dict(pos, vel, F, PE, KE, xi, vxi, conserved=[H' after every step])."""
    pos = np.array(pos, dtype=np.float64)
    vel = np.array(vel, dtype=np.float64)
    masses = np.asarray(masses, dtype=np.float64)
    n = len(masses)
    g = 3.0 * n
    nvt = T_K > 0.0
    kT = KB_EV * T_K if nvt else 0.0
    Q = g * kT * tau * tau if nvt else 1.0
    if F0 is None:
        PE, F = force_fn(pos)
    else:
        PE, F = None, np.array(F0, dtype=np.float64)
    inv_m = (acc_unit / masses)[:, None]
    conserved = []
    for _ in range(int(n_steps)):
        if nvt:
            xi, vxi = nose_hoover_half_step(vel, masses, xi, vxi, 0.5 * dt, g, kT, Q, acc_unit)
        vel += 0.5 * dt * F * inv_m
        pos += dt * vel
        PE, F = force_fn(pos)
        F = np.asarray(F, dtype=np.float64)
        vel += 0.5 * dt * F * inv_m
        if nvt:
            xi, vxi = nose_hoover_half_step(vel, masses, xi, vxi, 0.5 * dt, g, kT, Q, acc_unit)
        ke = kinetic_energy(vel, masses, acc_unit)
        conserved.append(ke + PE + (0.5 * Q * vxi * vxi + g * kT * xi if nvt else 0.0))
    return dict(pos=pos, vel=vel, F=F, PE=PE, KE=kinetic_energy(vel, masses, acc_unit), xi=xi, vxi=vxi,
                conserved=np.array(conserved))
