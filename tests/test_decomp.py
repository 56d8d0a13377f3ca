"""Spatial decomposition (groundwork for NEXT-1; Fig. 3-4): the host-side bookkeeping of
paper_2505_06711_b200/decomp.py on CPU -- single-process checks against the oracle's neighbour sets and a
world_size-2 gloo run of the two messages of the paper -- and, on the GPU box, the layer-by-layer C-ABI calls
(reann_step_*) driven by two ranks against the single-handle result."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

import gen
import oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn(script_path, world, timeout):
    port = free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE=str(world), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script_path)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=timeout) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, o + e
    return [json.loads(o.strip().splitlines()[-1]) for o, _ in outs]


@pytest.mark.parametrize("world,axis", [(2, 0), (3, 2)])
def test_rank_local_pair_sets_cover_the_global_set_exactly(world, axis):
    """Every rank sees complete neighbour lists of its local atoms ("complete neighbor lists of LAs"):
    the rows of the local atoms in the rank's own box (LAs + ghost copies), mapped back to global indices, are the
    rows of the global periodic system -- as multisets of (i, j, edge vector)."""
    from paper_2505_06711_b200.decomp import SlabPartition
    cfg = gen.make_config(2, n_mol=400, geometry_only=True)        # box 22.9 A
    pos = cfg["pos"] + np.array([3.3, -40.0, 7.7])                  # unwrapped
    R = 6.5
    Lb = cfg["box"].reshape(3, 3).diagonal()
    glob = oracle.neighbors(pos, cfg["box"], R)
    def key(i, j, d):
        return np.column_stack([i, j, np.round(d * 1e6)]).astype(np.int64)
    dg = pos[glob[:, 1]] + glob[:, 2:5] * Lb - pos[glob[:, 0]]
    want = key(glob[:, 0], glob[:, 1], dg)
    want = want[np.lexsort(want.T[::-1])]
    got = []
    n_owned = 0
    for r in range(world):
        part = SlabPartition(pos, cfg["box"], R, world, axis).build(r)
        n_loc = len(part.local)
        n_owned += n_loc
        assert (part.is_halo[:n_loc] == 0).all() and (part.is_halo[n_loc:] == 1).all()
        rows = oracle.neighbors(part.pos_loc, part.box_loc, R)
        rows = rows[rows[:, 0] < n_loc]                             # centred on local atoms
        Ll = part.box_loc.reshape(3, 3).diagonal()
        d = part.pos_loc[rows[:, 1]] + rows[:, 2:5] * Ll - part.pos_loc[rows[:, 0]]
        got.append(key(part.index_loc[rows[:, 0]], part.index_loc[rows[:, 1]], d))
    assert n_owned == len(pos)                                      # every atom has exactly one owner
    got = np.vstack(got)
    got = got[np.lexsort(got.T[::-1])]
    assert got.shape == want.shape and (got == want).all()


WORKER_MSG = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch.distributed as dist, gen
from paper_2505_06711_b200.decomp import SlabPartition, forward_exchange, backward_exchange
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg = gen.make_config(2, n_mol=400, geometry_only=True)
part = SlabPartition(cfg["pos"], cfg["box"], 6.5, world, 0).build(rank)
feat = lambda g: np.stack([g * 1.0, g * 0.5 + 1, np.sin(g)], 1).astype(np.float32)      # a "feature" of the global index
rows = forward_exchange(dist, part, lambda sel: feat(part.local[sel]))
ok_fwd = bool(np.array_equal(rows, feat(part.ghost_src)))                                 # ghost features == owner features
# backward: every ghost copy carries (1, global index); owners must receive (number of copies, copies * index)
back = backward_exchange(dist, part, np.stack([np.ones(len(part.ghost_src)), part.ghost_src.astype(np.float64)], 1))
copies = np.zeros(len(cfg["pos"]))
for r in range(world):
    if r != rank:
        src, _ = part.ghosts_of(r)
        np.add.at(copies, src[part.owner[src] == rank], 1.0)
ok_bwd = bool(np.allclose(back[:, 0], copies[part.local]) and np.allclose(back[:, 1], copies[part.local] * part.local))
dist.barrier()
print(json.dumps({{"rank": rank, "ok_fwd": ok_fwd, "ok_bwd": ok_bwd, "n_local": int(len(part.local)),
                  "n_ghost": int(len(part.ghost_src)), "n_multi": int((copies > 1).sum())}}))
dist.destroy_process_group()
"""


def test_forward_and_backward_messages_gloo_world2(tmp_path):
    """The two messages of the paper over gloo, world_size 2: after the forward message every ghost row equals its
    owner's row (otherwise "errors propagate"); the backward message returns to every owner the sum
    over all ghost copies of its atom."""
    script = tmp_path / "worker.py"
    script.write_text(WORKER_MSG.format(root=ROOT))
    outs = spawn(script, 2, 180)
    assert all(o["ok_fwd"] and o["ok_bwd"] for o in outs)
    assert sum(o["n_local"] for o in outs) == 1200 and all(o["n_ghost"] > 0 for o in outs)


WORKER_GPU = r"""
import os, sys, json
sys.path.insert(0, {root!r}); sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch, torch.distributed as dist, gen
import paper_2505_06711_b200 as R
from paper_2505_06711_b200.decomp import SlabPartition, energy_forces_decomposed
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)                                   # both ranks share the one GPU of the box; exchanges on the host
cfg = gen.make_config({k}, **{kw!r})
part = SlabPartition(cfg["pos"], cfg["box"], cfg["rc"] + cfg["skin"], world, 0).build(rank)
m = R.Reann(cfg["blob"], cfg["species"][part.index_loc], cfg["rc"], cfg["skin"], cfg["T"], cfg["L"], cfg["n_gauss"])
m.set_halo(part.is_halo)
m.build_neighbors(part.pos_loc, part.box_loc)
E, F_loc, vir = energy_forces_decomposed(dist, m, part, cfg["T"], cfg["n_gauss"])
E2, F_loc2, _ = energy_forces_decomposed(dist, m, part, cfg["T"], cfg["n_gauss"])     # a second step: same bits
out = dict(rank=rank, E=E, same=bool(E2 == E and (F_loc2 == F_loc).all()), n_local=int(len(part.local)), n_ghost=int(len(part.ghost_src)))
F = np.zeros((len(cfg["pos"]), 3)); F[part.local] = F_loc
Ft = torch.from_numpy(F); dist.all_reduce(Ft)
if rank == 0:
    ms = R.Reann.from_config(cfg); ms.build_neighbors(cfg["pos"], cfg["box"])
    Es, Fs, Vs = ms.energy_forces(cfg["pos"], cfg["box"])
    n = len(cfg["pos"])
    out.update(dE=abs(E - Es) / n, Escale=max(1.0, abs(Es) / n), dF=float(np.abs(Ft.numpy() - Fs).max()),
               dV=float(np.abs(vir - Vs).max()), Vscale=float(max(np.abs(Vs).max(), n)))
dist.barrier()
print(json.dumps(out))
dist.destroy_process_group()
"""


@pytest.mark.gpu
@pytest.mark.parametrize("k,kw", [(2, dict(n_mol=500)), (6, {})], ids=["water-T3", "hea-T2"])
def test_two_ranks_equal_the_single_handle_result(tmp_path, k, kw):
    """The paper's per-layer exchange between two ranks (each a handle over its slab + ghost copies, messages through
    host buffers / gloo) against one handle over the whole periodic system: E, F and the virial within the FP32 gates
    ("energies and forces ... are identical" across implementations)."""
    import __graft_entry__ as ge
    ge.build()
    script = tmp_path / "worker.py"
    script.write_text(WORKER_GPU.format(root=ROOT, k=k, kw=kw))
    outs = spawn(script, 2, 600)
    o = [x for x in outs if x["rank"] == 0][0]
    print("[decomposed]", o)
    assert all(x["same"] for x in outs) and all(x["n_ghost"] > 0 for x in outs)
    assert o["dE"] <= 1e-6 * o["Escale"] and o["dF"] <= 5e-4 and o["dV"] <= 1e-4 * o["Vscale"]
