"""Thin Python binding of libreann_b200.so (include/reann.h): argument marshalling only.

Every step of the energy/force path runs inside the CUDA library; there is no Python or CPU
fallback -- importing works without a GPU (so the C ABI can be inspected), but any call that
needs the library raises if it has not been built, and reann_create fails without a device.

Arrays may be NumPy arrays (host pointers) or torch CUDA tensors (device pointers); they must be
contiguous and of the dtype the header states (pos/E/F/virial float64, species int32).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libreann_b200.so")

REANN_OK, REANN_ERR_ARG, REANN_ERR_WEIGHTS, REANN_ERR_BOX, REANN_ERR_NO_NEIGHBORS, REANN_ERR_CUDA, \
    REANN_ERR_OOM, REANN_ERR_UNSUPPORTED = range(8)

EXPORTS = ["reann_create", "reann_build_neighbors", "reann_energy_forces", "reann_destroy", "reann_last_error",
           "reann_get_neighbors", "reann_get_neighbor_rows", "reann_get_stats", "reann_set_profiling", "reann_set_stream",
           "reann_get_atomic_energies", "reann_verlet", "reann_set_halo", "reann_step_begin", "reann_step_forward",
           "reann_coeff_get", "reann_coeff_set", "reann_step_backward", "reann_cbar_get", "reann_cbar_add", "reann_step_end",
           "reann_md_run", "reann_row_ptr_noalloc"]
REANN_NOALLOC_MAX_ROWS = 1 << 24


class ReannError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"reann error {code}: {text}")
        self.code = code


class MdState(ctypes.Structure):
    _fields_ = [("xi", ctypes.c_double), ("vxi", ctypes.c_double), ("forces_valid", ctypes.c_int64), ("kinetic", ctypes.c_double),
                ("potential", ctypes.c_double), ("conserved", ctypes.c_double), ("n_steps_done", ctypes.c_int64),
                ("n_rebuilds", ctypes.c_int64)]


class Stats(ctypes.Structure):
    _fields_ = [("n_atoms", ctypes.c_int64), ("n_ext", ctypes.c_int64), ("n_edges_list", ctypes.c_int64),
                ("n_edges_rc", ctypes.c_int64), ("n_rebuilds", ctypes.c_int64), ("n_calls", ctypes.c_int64),
                ("n_launches", ctypes.c_int64), ("ms_build", ctypes.c_double), ("ms_prep", ctypes.c_double),
                ("ms_edge_fwd", ctypes.c_double), ("ms_dense_fwd", ctypes.c_double), ("ms_gather", ctypes.c_double),
                ("ms_dense_bwd", ctypes.c_double), ("ms_edge_bwd", ctypes.c_double),
                ("ms_rev_gather", ctypes.c_double), ("ms_output", ctypes.c_double),
                ("n_profiled_calls", ctypes.c_int64), ("bytes_device", ctypes.c_size_t),
                ("ms_rev_gather_t0", ctypes.c_double), ("stash_chunks", ctypes.c_int64)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load the CUDA library; fail loudly if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2505_06711_b200._build` "
                               "or __graft_entry__.build(); there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double
        L.reann_create.restype = ctypes.c_int
        L.reann_create.argtypes = [ctypes.POINTER(vp), vp, ctypes.c_size_t, vp, i64, dbl, dbl, ctypes.c_int,
                                   ctypes.c_int, ctypes.c_int]
        L.reann_build_neighbors.restype = ctypes.c_int
        L.reann_build_neighbors.argtypes = [vp, vp, vp]
        L.reann_energy_forces.restype = ctypes.c_int
        L.reann_energy_forces.argtypes = [vp, vp, vp, vp, vp, vp]
        L.reann_destroy.restype = None
        L.reann_destroy.argtypes = [vp]
        L.reann_last_error.restype = ctypes.c_char_p
        L.reann_last_error.argtypes = [vp]
        L.reann_get_neighbors.restype = ctypes.c_int
        L.reann_get_neighbors.argtypes = [vp, ctypes.POINTER(i64), vp, vp, vp]
        L.reann_get_neighbor_rows.restype = ctypes.c_int
        L.reann_get_neighbor_rows.argtypes = [vp, i64, vp, vp, vp, vp]
        L.reann_get_stats.restype = ctypes.c_int
        L.reann_get_stats.argtypes = [vp, ctypes.POINTER(Stats)]
        L.reann_set_profiling.restype = ctypes.c_int
        L.reann_set_profiling.argtypes = [vp, ctypes.c_int]
        L.reann_set_stream.restype = ctypes.c_int
        L.reann_set_stream.argtypes = [vp, vp]
        L.reann_get_atomic_energies.restype = ctypes.c_int
        L.reann_get_atomic_energies.argtypes = [vp, vp]
        for name, args in (("reann_set_halo", [vp, vp]), ("reann_step_begin", [vp, vp, vp, ctypes.c_int]),
                           ("reann_step_forward", [vp, ctypes.c_int]), ("reann_coeff_get", [vp, ctypes.c_int, i64, vp, vp]),
                           ("reann_coeff_set", [vp, ctypes.c_int, i64, vp, vp]), ("reann_step_backward", [vp, ctypes.c_int]),
                           ("reann_cbar_get", [vp, i64, vp, vp]), ("reann_cbar_add", [vp, i64, vp, vp]),
                           ("reann_step_end", [vp, vp, vp, vp])):
            getattr(L, name).restype = ctypes.c_int
            getattr(L, name).argtypes = args
        L.reann_verlet.restype = ctypes.c_int
        L.reann_verlet.argtypes = [vp, vp, vp, vp, vp, dbl, dbl, ctypes.c_int]
        L.reann_md_run.restype = ctypes.c_int
        L.reann_md_run.argtypes = [vp, vp, vp, vp, vp, i64, dbl, dbl, dbl, dbl, vp, vp, ctypes.POINTER(MdState)]
        L.reann_row_ptr_noalloc.restype = ctypes.c_int
        L.reann_row_ptr_noalloc.argtypes = [vp, i64, vp, vp]
        _lib = L
    return _lib


def _ptr(x, dtype=None):
    """Address of a NumPy array / torch tensor / bytes object; None -> NULL."""
    if x is None:
        return None
    if isinstance(x, (bytes, bytearray)):
        return ctypes.cast(ctypes.c_char_p(bytes(x)), ctypes.c_void_p)
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"] or (dtype is not None and x.dtype != dtype):
            raise TypeError(f"need a C-contiguous array of dtype {dtype}, got {x.dtype}")
        return ctypes.c_void_p(x.ctypes.data)
    if hasattr(x, "data_ptr"):  # torch tensor (host or device)
        if not x.is_contiguous():
            raise TypeError("need a contiguous tensor")
        return ctypes.c_void_p(x.data_ptr())
    if isinstance(x, int):
        return ctypes.c_void_p(x)
    raise TypeError(f"cannot marshal {type(x)}")


def _check(h, code):
    if code != REANN_OK:
        raise ReannError(code, lib().reann_last_error(h).decode())


def _box(box) -> np.ndarray:
    b = np.ascontiguousarray(np.asarray(box, dtype=np.float64).reshape(-1))
    if b.size == 3:
        b = np.diag(b).reshape(9).copy()
    if b.size != 9:
        raise TypeError("box must have 3 or 9 entries")
    return b


# ---- the three calls of the boundary, same names as the C ABI ----
def reann_create(weights: bytes, species, rc: float, skin: float, T: int, L: int, n_gauss: int):
    h = ctypes.c_void_p()
    wbuf = ctypes.create_string_buffer(bytes(weights), len(weights))
    n = int(species.shape[0])
    code = lib().reann_create(ctypes.byref(h), ctypes.cast(wbuf, ctypes.c_void_p), len(weights),
                              _ptr(species, np.int32), n, float(rc), float(skin), int(T), int(L), int(n_gauss))
    _check(None, code)
    return h


def reann_build_neighbors(h, pos, box):
    b = _box(box)
    _check(h, lib().reann_build_neighbors(h, _ptr(pos, np.float64), _ptr(b)))


def reann_energy_forces(h, pos, box, E, F, virial=None):
    b = _box(box)
    _check(h, lib().reann_energy_forces(h, _ptr(pos, np.float64), _ptr(b), _ptr(E, np.float64), _ptr(F, np.float64),
                                        _ptr(virial, np.float64)))


def reann_destroy(h):
    lib().reann_destroy(h)


def reann_get_stats(h) -> dict:
    s = Stats()
    _check(h, lib().reann_get_stats(h, ctypes.byref(s)))
    return {k: getattr(s, k) for k, _ in Stats._fields_}


def reann_get_neighbors(h, n_atoms: int):
    """-> (row_ptr[n_atoms+1], j[E], shift[E,3]) in caller order / caller frame."""
    n = ctypes.c_int64(0)
    _check(h, lib().reann_get_neighbors(h, ctypes.byref(n), None, None, None))
    row_ptr = np.zeros(n_atoms + 1, dtype=np.int64)
    j = np.zeros(max(n.value, 1), dtype=np.int32)
    sh = np.zeros((max(n.value, 1), 3), dtype=np.int8)
    _check(h, lib().reann_get_neighbors(h, ctypes.byref(n), _ptr(row_ptr), _ptr(j), _ptr(sh)))
    return row_ptr, j[:n.value], sh[:n.value]


def reann_row_ptr_noalloc(counts, n_rows: int, row_ptr, cuda_stream=None) -> None:
    """row_ptr[0] = 0, row_ptr[i+1] = counts[0] + ... + counts[i] on the device, allocating nothing (reann.h):
    counts int32 [n_rows] and row_ptr int64 [n_rows+1] are DEVICE tensors / addresses of the caller."""
    _check(None, lib().reann_row_ptr_noalloc(_ptr(counts), int(n_rows), _ptr(row_ptr), _ptr(cuda_stream)))


def reann_get_neighbor_rows(h, atoms):
    """-> (row_ptr[len(atoms)+1], j[E], shift[E,3]) of the selected atoms, caller order / caller frame."""
    atoms = np.ascontiguousarray(atoms, dtype=np.int64)
    row_ptr = np.zeros(len(atoms) + 1, dtype=np.int64)
    _check(h, lib().reann_get_neighbor_rows(h, len(atoms), _ptr(atoms), _ptr(row_ptr), None, None))
    n = int(row_ptr[-1])
    j = np.zeros(max(n, 1), dtype=np.int32)
    sh = np.zeros((max(n, 1), 3), dtype=np.int8)
    _check(h, lib().reann_get_neighbor_rows(h, len(atoms), _ptr(atoms), _ptr(row_ptr), _ptr(j), _ptr(sh)))
    return row_ptr, j[:n], sh[:n]


class Reann:
    """Convenience wrapper around one handle (host NumPy in, NumPy out unless tensors are given)."""

    def __init__(self, weights: bytes, species, rc, skin, T, L, n_gauss):
        self.species = np.ascontiguousarray(species, dtype=np.int32)
        self.n = int(self.species.shape[0])
        self.n_gauss = int(n_gauss)
        self.h = reann_create(weights, self.species, rc, skin, T, L, n_gauss)

    @classmethod
    def from_config(cls, cfg: dict) -> "Reann":
        return cls(cfg["blob"], cfg["species"], cfg["rc"], cfg["skin"], cfg["T"], cfg["L"], cfg["n_gauss"])

    def build_neighbors(self, pos, box):
        reann_build_neighbors(self.h, pos, box)

    def energy_forces(self, pos, box, E=None, F=None, virial=None, want_virial=True):
        """With E/F/virial None: host outputs are allocated and returned as (E, F, virial)."""
        if E is None and F is None:
            E = np.zeros(1); F = np.zeros((self.n, 3)); virial = np.zeros(9) if want_virial else None
            reann_energy_forces(self.h, pos, box, E, F, virial)
            return float(E[0]), F, (virial.reshape(3, 3) if virial is not None else None)
        reann_energy_forces(self.h, pos, box, E, F, virial)
        return E, F, virial

    def atomic_energies(self) -> np.ndarray:
        out = np.zeros(self.n)
        _check(self.h, lib().reann_get_atomic_energies(self.h, _ptr(out)))
        return out

    def neighbors(self):
        return reann_get_neighbors(self.h, self.n)

    def neighbor_rows(self, atoms):
        return reann_get_neighbor_rows(self.h, atoms)

    def stats(self) -> dict:
        return reann_get_stats(self.h)

    def set_profiling(self, on: bool):
        _check(self.h, lib().reann_set_profiling(self.h, int(on)))

    def set_stream(self, stream_ptr: int):
        _check(self.h, lib().reann_set_stream(self.h, ctypes.c_void_p(stream_ptr)))

    # ---- one rank of a decomposed run (include/reann.h, reann_step_*; driver: decomp.energy_forces_decomposed) ----
    def set_halo(self, is_halo):
        a = None if is_halo is None else np.ascontiguousarray(is_halo, dtype=np.uint8)
        _check(self.h, lib().reann_set_halo(self.h, _ptr(a)))

    def step_begin(self, pos, box, want_virial=True):
        _check(self.h, lib().reann_step_begin(self.h, _ptr(pos, np.float64), _ptr(_box(box)), int(want_virial)))

    def step_forward(self, t: int):
        _check(self.h, lib().reann_step_forward(self.h, int(t)))

    def step_backward(self, t: int):
        _check(self.h, lib().reann_step_backward(self.h, int(t)))

    def _rows(self, fn, idx, rows=None, t=None):
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        out = np.zeros((len(idx), self.n_gauss), dtype=np.float32) if rows is None else np.ascontiguousarray(rows, dtype=np.float32)
        args = (self.h,) + (() if t is None else (int(t),)) + (len(idx), _ptr(idx), _ptr(out))
        _check(self.h, fn(*args))
        return out

    def coeff_get(self, t, idx): return self._rows(lib().reann_coeff_get, idx, None, t)
    def coeff_set(self, t, idx, rows): self._rows(lib().reann_coeff_set, idx, rows, t)
    def cbar_get(self, idx): return self._rows(lib().reann_cbar_get, idx)
    def cbar_add(self, idx, rows): self._rows(lib().reann_cbar_add, idx, rows)

    def step_end(self, want_virial=True):
        E = np.zeros(1); F = np.zeros((self.n, 3)); vir = np.zeros(9) if want_virial else None
        _check(self.h, lib().reann_step_end(self.h, _ptr(E), _ptr(F), _ptr(vir)))
        return float(E[0]), F, (vir.reshape(3, 3) if want_virial else None)

    def verlet(self, pos, vel, F, inv_mass, dt, acc_unit, drift: bool):
        _check(self.h, lib().reann_verlet(self.h, _ptr(pos), _ptr(vel), _ptr(F), _ptr(inv_mass), float(dt),
                                          float(acc_unit), int(drift)))

    def md_run(self, pos, vel, inv_mass, box, n_steps, dt, acc_unit, kT=0.0, tau=100.0, F=None, virial=None, xi=0.0, vxi=0.0,
               forces_valid=False):
        """reann_md_run on device tensors (pos, vel advanced in place); returns the thermostat / energy record."""
        st = MdState(xi=float(xi), vxi=float(vxi), forces_valid=int(bool(forces_valid)))
        _check(self.h, lib().reann_md_run(self.h, _ptr(pos), _ptr(vel), _ptr(inv_mass), _ptr(_box(box)), int(n_steps),
                                          float(dt), float(acc_unit), float(kT), float(tau), _ptr(F), _ptr(virial),
                                          ctypes.byref(st)))
        return {k: getattr(st, k) for k, _ in MdState._fields_}

    def close(self):
        if self.h is not None:
            reann_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
