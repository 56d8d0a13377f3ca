"""Host-side bookkeeping of a spatially decomposed run (groundwork for NEXT-1 of SURVEY.md 8(f)).

The paper's scheme (Fig. 3-4a): the box is cut into sub-domains, one per process; a process owns
the atoms of its sub-domain (local atoms, LAs) and keeps copies of the atoms of other sub-domains that lie within
the cutoff (+ skin) of it (ghost atoms, GAs). Per message-passing layer the owners send the GAs' coefficients
c^{t+1} forward and receive the gradients dE/dc^t of their atoms back.

This module holds no arithmetic of the method: it builds index lists (slabs along one axis, ghost copies with
their periodic shift, per-peer send / receive orders) and moves rows between ranks with torch.distributed
point-to-point calls; the per-layer work runs in the CUDA library (reann_step_* calls of include/reann.h).
With NVLink the two exchanges become peer stores from the gather kernels; here they go through
host buffers so that the logic can be tested with the gloo backend.
"""
from __future__ import annotations

import numpy as np


class SlabPartition:
    """Slabs of equal width along `axis`; rank r owns wrapped coordinates [r L / W, (r + 1) L / W).

    Attributes (per rank, after build()):
      local      global indices of the LAs (ascending)
      ghost_src  global index of every GA copy;  ghost_shift  its periodic shift along `axis` (-1, 0, +1)
      ghost_rank owner rank of every GA copy
      pos_loc    positions of LAs then GAs in the rank's own box (`box_loc`): the slab plus a margin of 2 R on either
                 side along `axis` (R = rc + skin), so that no periodic image along that axis is within R
      send[p]    positions (into `local`) of the LAs that rank p holds as GAs, in p's ghost order
      recv[p]    positions (into the ghost list) of the GAs owned by rank p, in the same order
    """

    def __init__(self, pos, box9, R, world, axis=0):
        self.pos = np.asarray(pos, dtype=np.float64)
        self.Lb = np.asarray(box9, dtype=np.float64).reshape(3, 3).diagonal().copy()
        self.R, self.world, self.axis = float(R), int(world), int(axis)
        L = self.Lb[axis]
        if L / world < R:
            raise ValueError("slab width below rc + skin: ghosts would come from beyond the adjacent slabs")
        self.xw = self.pos[:, axis] - np.floor(self.pos[:, axis] / L) * L
        self.owner = np.minimum((self.xw / (L / world)).astype(np.int64), world - 1)

    def ghosts_of(self, rank):
        """(global index, shift) of every ghost copy of `rank`, ordered by (shift, index)."""
        L, W, R = self.Lb[self.axis], self.world, self.R
        lo, hi = rank * L / W, (rank + 1) * L / W
        src, shf = [], []
        for s in (-1, 0, 1):
            x = self.xw + s * L
            m = (x >= lo - R) & (x < hi + R)
            if s == 0:
                m &= self.owner != rank
            idx = np.nonzero(m)[0]
            src.append(idx); shf.append(np.full(len(idx), s, dtype=np.int64))
        return np.concatenate(src), np.concatenate(shf)

    def build(self, rank):
        L, W, R, ax = self.Lb[self.axis], self.world, self.R, self.axis
        lo, hi = rank * L / W, (rank + 1) * L / W
        self.rank = rank
        self.local = np.nonzero(self.owner == rank)[0]
        self.ghost_src, self.ghost_shift = self.ghosts_of(rank)
        self.ghost_rank = self.owner[self.ghost_src]
        n_loc = len(self.local)
        p = np.vstack([self.pos[self.local], self.pos[self.ghost_src]])
        x = np.concatenate([self.xw[self.local], self.xw[self.ghost_src] + self.ghost_shift * L])
        p[:, ax] = x - (lo - 2.0 * R)                       # slab at [2R, 2R + width), ghosts within R of it
        self.pos_loc = p
        Lloc = self.Lb.copy(); Lloc[ax] = (hi - lo) + 4.0 * R
        self.box_loc = np.diag(Lloc).reshape(9).copy()
        self.is_halo = np.concatenate([np.zeros(n_loc, np.uint8), np.ones(len(self.ghost_src), np.uint8)])
        self.index_loc = np.concatenate([self.local, self.ghost_src])      # global index of every atom of the handle
        glob2loc = -np.ones(len(self.pos), dtype=np.int64)
        glob2loc[self.local] = np.arange(n_loc)
        self.recv, self.send = {}, {}
        for peer in range(W):
            if peer == rank:
                continue
            self.recv[peer] = np.nonzero(self.ghost_rank == peer)[0]           # my ghosts owned by peer, my ghost order
            src_p, _ = self.ghosts_of(peer)                                      # peer's ghosts, peer's ghost order
            self.send[peer] = glob2loc[src_p[self.owner[src_p] == rank]]         # my LAs among them, in peer's order
        return self


def _exchange(dist, rank, world, out_rows: dict, in_counts: dict, width: int):
    """Send out_rows[p] (float32 [n_p, width]) to every peer p and receive in_counts[p] rows from it (gloo / CPU
    tensors, non-blocking point-to-point)."""
    import torch
    reqs, got = [], {}
    for p in range(world):
        if p == rank:
            continue
        buf = torch.empty((in_counts[p], width), dtype=torch.float32)
        got[p] = buf
        if in_counts[p]:
            reqs.append(dist.irecv(buf, src=p))
        if len(out_rows[p]):
            reqs.append(dist.isend(torch.from_numpy(np.ascontiguousarray(out_rows[p], dtype=np.float32)), dst=p))
    for r in reqs:
        r.wait()
    return {p: b.numpy() for p, b in got.items()}


def forward_exchange(dist, part: SlabPartition, rows_of_locals):
    """The paper's forward message: rows (e.g. c^t) of my LAs go to the ranks that hold them as GAs; returns the rows
    of my GAs, ghost order. rows_of_locals(idx) -> float32 [len(idx), width] for positions into `local`."""
    W, rank = part.world, part.rank
    out = {p: rows_of_locals(part.send[p]) for p in part.send}
    width = next((o.shape[1] for o in out.values() if len(o)), 0)
    if width == 0:                                           # nothing to send: take the width from a probe
        width = rows_of_locals(np.zeros(0, dtype=np.int64)).shape[1]
    got = _exchange(dist, rank, W, out, {p: len(part.recv[p]) for p in part.recv}, width)
    rows = np.zeros((len(part.ghost_src), width), dtype=np.float32)
    for p, r in got.items():
        rows[part.recv[p]] = r
    return rows


def backward_exchange(dist, part: SlabPartition, rows_of_ghosts):
    """The paper's backward message: rows (e.g. dE/dc^t, or force contributions) accumulated on my GAs go back to
    their owners; returns the sum of what the other ranks accumulated on copies of my LAs, [n_local, width]."""
    W, rank = part.world, part.rank
    rows_of_ghosts = np.asarray(rows_of_ghosts, dtype=np.float32)
    width = rows_of_ghosts.shape[1]
    out = {p: rows_of_ghosts[part.recv[p]] for p in part.recv}
    got = _exchange(dist, rank, W, out, {p: len(part.send[p]) for p in part.send}, width)
    acc = np.zeros((len(part.local), width), dtype=np.float64)
    for p, r in got.items():
        np.add.at(acc, part.send[p], r.astype(np.float64))   # an LA may have several ghost copies on one peer
    return acc


def energy_forces_decomposed(dist, model, part: SlabPartition, T: int, n_gauss: int, want_virial=True):
    """One E/F(/virial) evaluation of the whole system by `world` ranks, each with the handle `model` over
    part.pos_loc (LAs then GAs, reann_set_halo(part.is_halo) done). Returns (E_total, F of my LAs [n_local, 3],
    virial_total [3, 3]); E and the virial are all-reduced."""
    import torch
    n_loc, n_gh = len(part.local), len(part.ghost_src)
    loc_idx = np.arange(n_loc, dtype=np.int64)
    gh_idx = n_loc + np.arange(n_gh, dtype=np.int64)
    model.step_begin(part.pos_loc, part.box_loc, want_virial)
    for t in range(T):
        if t >= 1:      # forward message: c^t of my ghosts from their owners
            rows = forward_exchange(dist, part, lambda sel: model.coeff_get(t, loc_idx[sel]) if len(sel)
                                    else np.zeros((0, n_gauss), np.float32))
            if n_gh:
                model.coeff_set(t, gh_idx, rows)
        model.step_forward(t)
    for t in range(T - 1, -1, -1):
        if t < T - 1:   # backward message: dE/dc^{t+1} accumulated on my ghosts goes to the owners
            mine = backward_exchange(dist, part, model.cbar_get(gh_idx) if n_gh else np.zeros((0, n_gauss), np.float32))
            if n_loc:
                model.cbar_add(loc_idx, mine.astype(np.float32))
        model.step_backward(t)
    E, F, vir = model.step_end(want_virial)
    F_loc = F[:n_loc] + backward_exchange(dist, part, F[n_loc:].astype(np.float32))   # forces on other ranks' atoms
    tot = torch.tensor([E] + (list(vir.reshape(-1)) if want_virial else [0.0] * 9), dtype=torch.float64)
    dist.all_reduce(tot)
    return float(tot[0]), F_loc, tot[1:].numpy().reshape(3, 3)
