"""ctypes binding of the float64 CPU oracle (oracle/reann_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs. Never import this from
paper_2505_06711_b200/ (the product path) and never import that package from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "reann_oracle.c")
_LIB = os.path.join(_HERE, "libreann_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-ffp-contract=off: SURVEY.md 8(c) A-15)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        c_dp = ctypes.POINTER(ctypes.c_double)
        c_ip = ctypes.POINTER(ctypes.c_int32)
        L.oracle_neighbors.restype = ctypes.c_int64
        L.oracle_neighbors.argtypes = [c_dp, ctypes.c_int64, c_dp, ctypes.c_double, ctypes.c_int,
                                       c_ip, ctypes.c_int64]
        L.oracle_neighbor_rows.restype = ctypes.c_int64
        L.oracle_neighbor_rows.argtypes = [c_dp, ctypes.c_int64, c_dp, ctypes.c_double, ctypes.POINTER(ctypes.c_int64),
                                           ctypes.c_int64, ctypes.POINTER(ctypes.c_int64), c_ip, ctypes.c_int64]
        L.oracle_energy_forces.restype = ctypes.c_int
        L.oracle_energy_forces.argtypes = [ctypes.c_void_p, ctypes.c_size_t, c_ip, ctypes.c_int64, c_dp,
                                           c_dp, ctypes.c_int, c_dp, c_dp, c_dp, c_dp, c_dp, c_dp, c_dp,
                                           ctypes.c_int]
        L.oracle_blob_info.restype = ctypes.c_int
        L.oracle_blob_info.argtypes = [ctypes.c_void_p, ctypes.c_size_t, c_ip, c_dp]
        L.oracle_monomials.restype = ctypes.c_int
        L.oracle_monomials.argtypes = [ctypes.c_int, c_ip, c_dp]
        L.oracle_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)) if a is not None else None


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def neighbors(pos, box9, R, mode="cell") -> np.ndarray:
    """Sorted rows (i, j, Sx, Sy, Sz), caller frame; mode 'cell' or 'brute' (O(N^2 27))."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    box9 = np.ascontiguousarray(box9, dtype=np.float64).reshape(9)
    N = pos.shape[0]
    m = 1 if mode == "cell" else 0
    n = lib().oracle_neighbors(_dp(pos), N, _dp(box9), float(R), m, None, 0)
    if n < 0:
        raise ValueError(f"oracle_neighbors error {-n}")
    rows = np.zeros((max(n, 1), 5), dtype=np.int32)
    n2 = lib().oracle_neighbors(_dp(pos), N, _dp(box9), float(R), m, _ip(rows), n)
    assert n2 == n
    return rows[:n]


def neighbor_rows(pos, box9, R, sel):
    """Sorted rows (i, j, Sx, Sy, Sz) of the atoms `sel` (strictly ascending) only, and row_ptr[len(sel)+1]:
    the same pair test as neighbors() over the cell list; for systems whose full list is too large."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    box9 = np.ascontiguousarray(box9, dtype=np.float64).reshape(9)
    sel = np.ascontiguousarray(sel, dtype=np.int64)
    i64p = ctypes.POINTER(ctypes.c_int64)
    row_ptr = np.zeros(len(sel) + 1, dtype=np.int64)
    n = lib().oracle_neighbor_rows(_dp(pos), pos.shape[0], _dp(box9), float(R), sel.ctypes.data_as(i64p), len(sel),
                                   row_ptr.ctypes.data_as(i64p), None, 0)
    if n < 0:
        raise ValueError(f"oracle_neighbor_rows error {-n}")
    rows = np.zeros((max(n, 1), 5), dtype=np.int32)
    n2 = lib().oracle_neighbor_rows(_dp(pos), pos.shape[0], _dp(box9), float(R), sel.ctypes.data_as(i64p), len(sel),
                                    row_ptr.ctypes.data_as(i64p), _ip(rows), n)
    assert n2 == n
    return rows[:n], row_ptr


def blob_info(blob: bytes) -> dict:
    out = np.zeros(10, dtype=np.int32)
    rc = ctypes.c_double(0)
    code = lib().oracle_blob_info(blob, len(blob), _ip(out), ctypes.byref(rc))
    if code:
        raise ValueError(f"oracle_blob_info error {code}")
    keys = ["S", "T", "L", "n_gauss", "n_orb", "H1c", "H2c", "H1e", "H2e", "Na"]
    d = {k: int(v) for k, v in zip(keys, out)}
    d["rc"] = rc.value
    return d


def monomials(L: int):
    lxyz = np.zeros((56, 3), dtype=np.int32)
    mu = np.zeros(56)
    n = lib().oracle_monomials(L, _ip(lxyz), _dp(mu))
    return lxyz[:n].copy(), mu[:n].copy()


def energy_forces(blob: bytes, species, pos, box9, forces=True, dumps=False, nthreads=0) -> dict:
    """E (eV), F [N,3] (eV/A), virial [3,3] (eV), Ei [N]; with dumps=True also c, b, rho per layer."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    species = np.ascontiguousarray(species, dtype=np.int32)
    box9 = np.ascontiguousarray(box9, dtype=np.float64).reshape(9)
    N = pos.shape[0]
    info = blob_info(blob)
    E = ctypes.c_double(0)
    F = np.zeros((N, 3)) if forces else None
    vir = np.zeros(9) if forces else None
    Ei = np.zeros(N)
    c = b = rho = None
    if dumps:
        T, nphi, Na, norb = info["T"], info["n_gauss"], info["Na"], info["n_orb"]
        c = np.zeros((T, N, nphi)); b = np.zeros((T, N, nphi, Na)); rho = np.zeros((T, N, norb))
    code = lib().oracle_energy_forces(blob, len(blob), _ip(species), N, _dp(pos), _dp(box9),
                                      1 if forces else 0, ctypes.byref(E), _dp(F), _dp(vir), _dp(Ei),
                                      _dp(c), _dp(b), _dp(rho), int(nthreads))
    if code:
        raise ValueError(f"oracle_energy_forces error {code}")
    out = dict(E=E.value, Ei=Ei)
    if forces:
        out["F"] = F
        out["virial"] = vir.reshape(3, 3)
    if dumps:
        out.update(c=c, b=b, rho=rho)
    return out
