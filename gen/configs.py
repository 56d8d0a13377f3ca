"""Geometry recipes for the five BASELINE.json configs (+ small unit configs).

Stand-ins for the paper's workloads (solid Ag, liquid water):
the datasets and trained models are not available, so only the *shape* is kept
(fcc metal; water at 1 g/cm^3; 96 ... 10^7 atoms). Recipe: SURVEY.md section 8(d).

Seeds: geometry 1000+k, weights 2000+k, velocities 3000+k for config k.
"""
from __future__ import annotations

import json
import os

import numpy as np

# 18.015 g/mol at 1.0 g/cm^3 -> Angstrom^3 per molecule
_VOL_PER_H2O = 18.015 / 6.02214076e23 * 1e24

MASS = {"O": 15.999, "H": 1.008, "M": 107.8682}  # amu ("M": the fcc metal, Ag-like)
KB_EV = 8.617333e-5            # eV/K
ACC_UNIT = 9.648533e-3         # 1 eV/(Angstrom amu) in Angstrom/fs^2

CONFIGS = {
    # k: recipe. nbar = expected neighbours within rc (used only to scale random weights)
    0: dict(name="unit-tableS1", kind="water", n_mol=16, box=None, rc=3.8, skin=0.5, T=2, L=2,
            n_gauss=7, H=(32, 16), Hc=(16, 16), nbar=23.0),            # PAPER.md:267-271 shapes
    1: dict(name="tiny-water-96", kind="water", n_mol=32, box=9.86, rc=6.0, skin=1.0, T=2, L=2,
            n_gauss=8, H=(64, 64), nbar=90.7),
    2: dict(name="bulk-water-3072", kind="water", n_mol=1024, box=31.29, rc=6.0, skin=2.0, T=3, L=2,
            n_gauss=16, H=(128, 128), nbar=90.7),
    3: dict(name="large-water-192000", kind="water", n_mol=64000, box=124.17, rc=6.0, skin=2.0, T=3,
            L=3, n_gauss=16, H=(128, 128), nbar=90.7),
    4: dict(name="fcc-4M", kind="fcc", ncell=100, a=3.61, sigma=0.1, rc=5.0, skin=1.0, T=3, L=2,
            n_gauss=12, H=(64, 64), nbar=44.7),
    # NEXT-4 of SURVEY.md 8(f): multi-element solid, the shape of the paper's HEA workload (Fig. 7b: 576
    # atoms per GPU; :116: five elements): fcc with `S` randomly assigned species
    6: dict(name="hea-fcc", kind="hea", ncell=6, a=3.6, sigma=0.08, S=5, rc=6.0, skin=1.0, T=2, L=2, n_gauss=8,
            H=(64, 64), nbar=78.0),
    5: dict(name="water-slab-10M", kind="slab", n_mol=3333333, box=463.7, gap=30.0, rc=6.0, skin=2.0,
            T=3, L=2, n_gauss=16, H=(128, 128), nbar=90.7),
}


def _random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """Uniform random rotations from normalised 4-Gaussian quaternions -> [n,3,3]."""
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def water_box(n_mol: int, box_xyz, seed: int, fill_z: float | None = None):
    """n_mol rigid H2O (O-H 0.96 A, 104.5 deg): uniform random centres (the O site),
    uniform random orientation, + N(0, 0.05 A) jitter per coordinate.
    Atom order O,H,H per molecule; species O=0, H=1. `fill_z`: molecules only in z in [0, fill_z)."""
    rng = np.random.default_rng(seed)
    box_xyz = np.asarray(box_xyz, dtype=np.float64)
    span = box_xyz.copy()
    if fill_z is not None:
        span[2] = fill_z
    centres = rng.random((n_mol, 3)) * span
    R = _random_rotations(rng, n_mol)
    half = np.deg2rad(104.5) / 2
    h_local = 0.96 * np.array([[np.sin(half), np.cos(half), 0.0], [-np.sin(half), np.cos(half), 0.0]])
    pos = np.empty((n_mol, 3, 3))
    pos[:, 0, :] = centres
    pos[:, 1, :] = centres + R @ h_local[0]
    pos[:, 2, :] = centres + R @ h_local[1]
    pos = pos.reshape(-1, 3)
    pos += 0.05 * rng.standard_normal(pos.shape)
    species = np.tile(np.array([0, 1, 1], dtype=np.int32), n_mol)
    return pos, species


def fcc_lattice(ncell: int, a: float, sigma: float, seed: int):
    """fcc, ncell^3 conventional cells, + N(0, sigma) per coordinate; one species."""
    rng = np.random.default_rng(seed)
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]], dtype=np.float64)
    g = np.arange(ncell, dtype=np.float64)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    pos = ((cells + basis[None, :, :]) * a).reshape(-1, 3)
    if sigma > 0:
        pos = pos + sigma * rng.standard_normal(pos.shape)
    species = np.zeros(len(pos), dtype=np.int32)
    return pos, species


def maxwell_boltzmann(masses: np.ndarray, temp_K: float, seed: int) -> np.ndarray:
    """Velocities in Angstrom/fs, centre-of-mass velocity removed."""
    rng = np.random.default_rng(seed)
    sig = np.sqrt(KB_EV * temp_K / masses * ACC_UNIT)  # sqrt(kT/m) in A/fs
    v = rng.standard_normal((len(masses), 3)) * sig[:, None]
    v -= (masses[:, None] * v).sum(0) / masses.sum()
    return v


def _calib_table() -> dict:
    path = os.path.join(os.path.dirname(__file__), "calib.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f)
    return {}


def make_config(k: int, T: int | None = None, n_mol: int | None = None, ncell: int | None = None,
                geometry_only: bool = False, gains: dict | None = None, radial_jitter: float = 0.0,
                n_species: int | None = None, tilt: tuple | None = None) -> dict:
    """Build config k. Overrides (T, n_mol, ncell) give same-density replicas / the T sweep.

    tilt = (xy, xz, yz) in Angstrom (tests of the triclinic path, NEXT-4): lattice vectors a = (Lx, 0, 0),
    b = (xy, Ly, 0), c = (xz, yz, Lz). Water: the molecules' fractional coordinates are kept, so the density is that of
    the orthorhombic recipe; fcc: the Cartesian positions are kept (choose tilts that are multiples of the lattice
    constant to describe the same crystal).

    radial_jitter > 0 (tests only): per-(layer, species) radial tables, see make_weights.

    Returns dict with pos[N,3] f64, species[N] i32, box[9] f64 (row-major lattice), masses[N],
    hyper-parameters, and (unless geometry_only) the weights blob (bytes)."""
    from .weights import make_weights, pack_blob, n_orb_default

    r = dict(CONFIGS[k])
    if T is not None:
        r["T"] = T
    seed_g, seed_w = 1000 + k, 2000 + k
    if r["kind"] in ("water", "slab"):
        nm = n_mol if n_mol is not None else r["n_mol"]
        if r["kind"] == "water":
            if n_mol is None and r["box"] is not None:
                Lb = r["box"]
            else:
                Lb = float((nm * _VOL_PER_H2O) ** (1.0 / 3.0))
            box = np.array([Lb, Lb, Lb])
            pos, species = water_box(nm, box, seed_g)
        else:
            d = r["box"] if n_mol is None else float((nm * _VOL_PER_H2O) ** (1.0 / 3.0))
            box = np.array([d, d, d + r["gap"]])
            pos, species = water_box(nm, box, seed_g, fill_z=d)
        S = 2
        masses = np.where(species == 0, MASS["O"], MASS["H"])
    else:
        nc = ncell if ncell is not None else r["ncell"]
        pos, species = fcc_lattice(nc, r["a"], r["sigma"], seed_g)
        box = np.array([nc * r["a"]] * 3)
        S = int(r.get("S", 1)) if n_species is None else int(n_species)
        if S > 1:
            species = np.random.default_rng(seed_g + 500).integers(0, S, len(pos)).astype(np.int32)
        masses = np.full(len(pos), MASS["M"])
    box9 = np.diag(box).reshape(9).copy()
    if tilt is not None:
        box9[3], box9[6], box9[7] = float(tilt[0]), float(tilt[1]), float(tilt[2])
        if r["kind"] in ("water", "slab"):
            centre = pos.reshape(-1, 3, 3)[:, :1, :]                   # the O site carries the molecule
            moved = (centre / box) @ box9.reshape(3, 3)
            pos = (pos.reshape(-1, 3, 3) - centre + moved).reshape(-1, 3)
    out = dict(k=k, name=r["name"], pos=pos, species=species, box=box9,
               masses=masses, rc=r["rc"], skin=r["skin"], T=r["T"], L=r["L"], n_gauss=r["n_gauss"],
               H=r["H"], S=S, nbar=r["nbar"], n_orb=n_orb_default(r["n_gauss"], r["L"]),
               seed_vel=3000 + k)
    if not geometry_only:
        g = gains if gains is not None else _calib_table().get(f"{k}:{r['T']}", {})
        w = make_weights(S=S, T=r["T"], L=r["L"], n_gauss=r["n_gauss"], n_orb=out["n_orb"],
                         H=r["H"], Hc=r.get("Hc", r["H"]), rc=r["rc"], nbar=r["nbar"], seed=seed_w,
                         e_scale=g.get("e", 1.0), wc_gain=g.get("wc"), c_gain=g.get("c"),
                         radial_jitter=radial_jitter)
        out["weights"] = w
        out["blob"] = pack_blob(w)
        out["gains"] = g
    return out
