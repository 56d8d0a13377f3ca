"""Random weights and the weights-blob byte layout.

Blob (little-endian; every real is float64 so both implementations read the same numbers):

  header, 64 bytes:
    char  magic[8] = "REANNB2\\0"
    u32   version (=1), S, T, L, n_gauss, n_orb, H1c, H2c, H1e, H2e, act (0 = SiLU), pad (=0)
    f64   rc
  then float64 arrays, C order, back to back:
    r_center[T][S][n_gauss]     centre of primitive n, indexed by the NEIGHBOUR's species
    alpha   [T][S][n_gauss]     width parameter of exp(-alpha (r - r_center)^2)
    c0      [S][n_gauss]        layer-0 orbital coefficients per species
    Wc      [T][L+1][n_gauss][n_orb]   contraction weights
    for t in 0..T-1, for s in 0..S-1:
       W1[n_orb][H1], b1[H1], W2[H1][H2], b2[H2], W3[H2][out], b3[out]
       with (H1,H2,out) = (H1c,H2c,n_gauss) for t < T-1 and (H1e,H2e,1) for t = T-1.

H1c/H2c: hidden widths of the coefficient networks (the paper's "MPNN structure"),
H1e/H2e: of the energy network ("atomic NN structure"), PAPER.md:265-271 (Table S1).
"""
from __future__ import annotations

import struct

import numpy as np

MAGIC = b"REANNB2\x00"
HEADER_BYTES = 64


def n_monomials(L: int) -> int:
    return (L + 1) * (L + 2) * (L + 3) // 6


def n_orb_default(n_gauss: int, L: int) -> int:
    """The paper's feature count N_phi (N_phi+1) (L+1) / 2."""
    return n_gauss * (n_gauss + 1) * (L + 1) // 2


def make_weights(S, T, L, n_gauss, n_orb, H, rc, nbar, seed, Hc=None, e_scale=1.0, wc_gain=None,
                 c_gain=None, radial_jitter=0.0) -> dict:
    """Seeded weights: r_n = n rc/(N-1), alpha = 1/(2 Delta^2) with Delta = rc/(N-1);
    c0 ~ N(0,1); Wc[t] ~ wc_gain[t] N(0,1) rc^-l / sqrt(N nbar); MLP Xavier-normal, biases
    N(0, 0.1^2); last layer of coefficient network t multiplied by c_gain[t]; the energy
    network's last layer by e_scale. The gains (gen/calib.json, written by
    oracle/calibrate.py) keep rho^t and c^t of order one in every layer, so that every term
    of the backward pass carries weight in the parity tests.

    radial_jitter > 0 (tests only; the BASELINE configs keep identical rows, as their recipe says):
    every (layer t, species s) row of r_center / alpha is scaled by its own seeded factor
    (1 + j (1 + u))^(+-1), u ~ U[0,1), j = radial_jitter (10-20 % for j = 0.1; drawn from a separate
    stream so that no other weight changes), so that reading A-3 -- tables indexed by layer and by
    the NEIGHBOUR's species -- is visible to the pins and the parity tests."""
    rng = np.random.default_rng(seed)
    Hc = H if Hc is None else Hc
    delta = rc / (n_gauss - 1) if n_gauss > 1 else rc
    rcen = np.broadcast_to(np.arange(n_gauss) * delta, (T, S, n_gauss)).copy()
    alpha = np.full((T, S, n_gauss), 1.0 / (2.0 * delta * delta))
    if radial_jitter > 0:
        jr = np.random.default_rng(seed + 7777)
        for arr in (rcen, alpha):
            f = (1.0 + radial_jitter * (1.0 + jr.random((T, S)))) ** jr.choice([-1.0, 1.0], size=(T, S))
            arr *= f[:, :, None]
    c0 = rng.standard_normal((S, n_gauss))
    Wc = rng.standard_normal((T, L + 1, n_gauss, n_orb))
    for l in range(L + 1):
        Wc[:, l] *= rc ** (-l) / np.sqrt(n_gauss * nbar)
    if wc_gain is not None:
        for t in range(T):
            Wc[t] *= wc_gain[t]
    mlps = []
    for t in range(T):
        last = t == T - 1
        H1, H2 = (H if last else Hc)
        out = 1 if last else n_gauss
        per_s = []
        for _s in range(S):
            def xavier(fi, fo):
                return rng.standard_normal((fi, fo)) * np.sqrt(2.0 / (fi + fo))
            W1, b1 = xavier(n_orb, H1), 0.1 * rng.standard_normal(H1)
            W2, b2 = xavier(H1, H2), 0.1 * rng.standard_normal(H2)
            W3, b3 = xavier(H2, out), 0.1 * rng.standard_normal(out)
            if last:
                W3, b3 = W3 * e_scale, b3 * e_scale
            elif c_gain is not None:
                W3, b3 = W3 * c_gain[t], b3 * c_gain[t]
            per_s.append(dict(W1=W1, b1=b1, W2=W2, b2=b2, W3=W3, b3=b3))
        mlps.append(per_s)
    return dict(S=S, T=T, L=L, n_gauss=n_gauss, n_orb=n_orb, H1c=Hc[0], H2c=Hc[1], H1e=H[0],
                H2e=H[1], act=0, rc=float(rc), rcen=rcen, alpha=alpha, c0=c0, Wc=Wc, mlp=mlps)


def pack_blob(w: dict) -> bytes:
    head = MAGIC + struct.pack("<12I", 1, w["S"], w["T"], w["L"], w["n_gauss"], w["n_orb"],
                               w["H1c"], w["H2c"], w["H1e"], w["H2e"], w["act"], 0)
    head += struct.pack("<d", w["rc"])
    assert len(head) == HEADER_BYTES
    parts = [head]
    for key in ("rcen", "alpha", "c0", "Wc"):
        parts.append(np.ascontiguousarray(w[key], dtype="<f8").tobytes())
    for per_s in w["mlp"]:
        for m in per_s:
            for key in ("W1", "b1", "W2", "b2", "W3", "b3"):
                parts.append(np.ascontiguousarray(m[key], dtype="<f8").tobytes())
    return b"".join(parts)


def blob_layout(S, T, L, n_gauss, n_orb, H1c, H2c, H1e, H2e) -> int:
    """Total byte size implied by a header (for validation tests)."""
    n = 2 * T * S * n_gauss + S * n_gauss + T * (L + 1) * n_gauss * n_orb
    for t in range(T):
        H1, H2, out = (H1e, H2e, 1) if t == T - 1 else (H1c, H2c, n_gauss)
        n += S * (n_orb * H1 + H1 + H1 * H2 + H2 + H2 * out + out)
    return HEADER_BYTES + 8 * n
