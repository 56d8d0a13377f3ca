"""Independent NumPy evaluation of the REANN energy, used ONLY to pin the oracle.

It shares no code with oracle/ or the CUDA path and does not use Cartesian monomials or
multinomial coefficients at all. By the multinomial theorem

    sum_{|a|=l} l!/(lx!ly!lz!) ( sum_j w_j r_j^a )^2  =  sum_{j,k} w_j w_k (r_j . r_k)^l ,

so Eq. 1 with the contraction of SURVEY.md 8(c) A-1 becomes, per atom i,

    rho_i[m] = sum_l  sum_{j,k}  w^l_j[m] w^l_k[m] (r_ij . r_ik)^l ,
    w^l_j[m] = sum_n Wc[t][l][n][m] c_j[n] exp(-alpha_n (r_ij - r_n)^2) (1 + cos(pi r_ij / rc))/2 .

Edges come from an explicit O(N^2 * 27) image loop; the MLP is plain matmul.
"""
import numpy as np


def edges_bruteforce(pos, box, R):
    """All (i, j, S) with |r_j + S*box - r_i| < R, S in {-1,0,1}^3 over wrapped coordinates."""
    Lb = np.asarray(box, dtype=np.float64).reshape(3, 3).diagonal()
    xw = pos - np.floor(pos / Lb) * Lb
    out_i, out_j, out_d = [], [], []
    N = len(pos)
    for sx in (-1, 0, 1):
        for sy in (-1, 0, 1):
            for sz in (-1, 0, 1):
                sh = np.array([sx, sy, sz]) * Lb
                d = xw[None, :, :] + sh - xw[:, None, :]          # [i, j, 3]
                d2 = (d ** 2).sum(-1)
                mask = d2 < R * R
                if sx == 0 and sy == 0 and sz == 0:
                    mask &= ~np.eye(N, dtype=bool)
                ii, jj = np.nonzero(mask)
                out_i.append(ii); out_j.append(jj); out_d.append(d[ii, jj])
    return np.concatenate(out_i), np.concatenate(out_j), np.concatenate(out_d)


def silu(z):
    return z / (1.0 + np.exp(-z))


def energy(w, species, pos, box, return_all=False):
    """E and per-layer rho, c via the pair form. `w`: the dict from gen.make_weights."""
    T, L, rc = w["T"], w["L"], w["rc"]
    N = len(pos)
    ei, ej, ed = edges_bruteforce(pos, box, rc)
    er = np.sqrt((ed ** 2).sum(-1))
    fc = 0.5 * (1.0 + np.cos(np.pi * er / rc))
    c = w["c0"][species]                                   # [N, nphi]
    rhos, cs = [], [c]
    for t in range(T):
        sj = species[ej]
        radial = np.exp(-w["alpha"][t][sj] * (er[:, None] - w["rcen"][t][sj]) ** 2) * fc[:, None]
        X = c[ej] * radial                                 # [E, nphi]
        rho = np.zeros((N, w["n_orb"]))
        for i in range(N):
            sel = ei == i
            Xi, ri = X[sel], ed[sel]
            gram = ri @ ri.T
            for l in range(L + 1):
                Wl = Xi @ w["Wc"][t][l]                    # [K, n_orb]
                rho[i] += np.einsum("jm,jk,km->m", Wl, gram ** l, Wl)
        rhos.append(rho)
        out = np.zeros((N, 1 if t == T - 1 else w["n_gauss"]))
        for s in range(w["S"]):
            m = w["mlp"][t][s]
            sel = species == s
            h1 = silu(rho[sel] @ m["W1"] + m["b1"])
            h2 = silu(h1 @ m["W2"] + m["b2"])
            out[sel] = h2 @ m["W3"] + m["b3"]
        if t < T - 1:
            c = out
            cs.append(c)
        else:
            Ei = out[:, 0]
    if return_all:
        return Ei.sum(), Ei, rhos, cs
    return Ei.sum()
