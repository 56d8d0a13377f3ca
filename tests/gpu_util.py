"""Helpers for the GPU parity tests (calls go through the C ABI via the thin binding)."""
import numpy as np

import oracle

E_TOL_REL = 1e-6      # |E_gpu - E_orc| / N <= 1e-6 * max(1 eV, |E_orc| / N)   (north_star; A-17)
F_TOL = 5e-4          # max |dF| eV/A in the FP32 path                          (north_star)
VIR_TOL_REL = 1e-4    # see check_parity


def gpu_rows(model):
    """Sorted (i, j, Sx, Sy, Sz) rows of the library's neighbour list, caller frame."""
    row_ptr, j, sh = model.neighbors()
    i = np.repeat(np.arange(model.n, dtype=np.int32), np.diff(row_ptr))
    rows = np.column_stack([i, j, sh.astype(np.int32)]).astype(np.int32)
    order = np.lexsort((rows[:, 4], rows[:, 3], rows[:, 2], rows[:, 1], rows[:, 0]))
    return rows[order]


def check_parity(res_gpu, ref, n, what=""):
    E, F, vir = res_gpu
    dE = abs(E - ref["E"]) / max(n, 1)
    assert dE <= E_TOL_REL * max(1.0, abs(ref["E"]) / max(n, 1)), f"{what}: |dE|/N = {dE:.3e}"
    if n:
        dF = np.abs(F - ref["F"]).max()
        assert dF <= F_TOL, f"{what}: max|dF| = {dF:.3e}"
    if vir is not None:
        # The virial is not in north_star's tolerance list. It is a force-weighted sum
        # (-sum_e r_e (x) g_e), so it gets the same relative class as the forces, made stricter:
        # F_TOL / rms|F| ~ 5e-4 relative for forces -> 1e-4 relative here, of max(|virial|, 1 eV/atom).
        scale = max(np.abs(ref["virial"]).max(), float(n))
        dV = np.abs(vir - ref["virial"]).max()
        assert dV <= VIR_TOL_REL * scale, f"{what}: virial {dV:.3e} vs {VIR_TOL_REL * scale:.3e}"
    print(f"[parity] {what}: n={n} |dE|/N={dE:.2e} (E/N={ref['E'] / max(n, 1):.3f}) max|dF|="
          f"{(np.abs(F - ref['F']).max() if n else 0):.2e} rmsF={(np.sqrt((ref['F'] ** 2).sum(1).mean()) if n else 0):.2f}"
          + (f" dVir/scale={np.abs(vir - ref['virial']).max() / max(np.abs(ref['virial']).max(), float(n), 1.0):.2e}" if vir is not None else ""))


def open_cluster(pos, species, box9, centre, radius):
    """Atoms (with periodic images unfolded by minimum image w.r.t. `centre`) within `radius` of
    `centre`; needs box >= 2*radius. Returns (indices, positions in a big open box, big box)."""
    Lb = np.asarray(box9).reshape(3, 3).diagonal()
    assert (Lb >= 2 * radius).all()
    d = pos - centre
    d -= np.round(d / Lb) * Lb
    sel = np.nonzero((d ** 2).sum(1) < radius * radius)[0]
    big = 2 * radius + 40.0
    return sel, d[sel] + big / 2, np.diag([big] * 3).reshape(9)
