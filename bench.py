#!/usr/bin/env python
"""bench.py -- MD atom-steps/s of the REANN energy+force hot path on B200 (BASELINE.json metric).

One "step" = one MD step of the synthetic workload (velocity Verlet with a Nose-Hoover thermostat at 300 K):
thermostat half step, half kick + drift, one energy+force evaluation (skin check, rebuild when triggered,
T forward layers, reverse pass, outputs), half kick, thermostat half step. All of it runs in this repo's CUDA
kernels behind the C ABI (reann_md_run for the timed region).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference]

The path does not shard ("replicas only"): with --gpus N every rank runs an
independent replica of the same workload ("scaling": "weak"); no data-path collective exists.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import gen  # noqa: E402

METRIC = "MD atom-steps/s (E+F per step)"
UNIT = "atom-steps/s"
FP32_FMA_LANES_PER_SM = 128
N_SM = 148


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "_source": "fallback"}


def max_over_ranks(value: float, device: str = "cuda") -> float:
    """Replicas only: the one cross-rank step of the bench is the max of the per-rank
    device times, so that `value` = (units all ranks processed) / (slowest rank's time)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(n_units_per_rank: int, steps: int, ms_total_local: float, world: int, device: str = "cuda"):
    """(whole-job units/s, ms per step) from each rank's locally timed region."""
    ms = max_over_ranks(ms_total_local, device)
    return world * n_units_per_rank * steps / (ms * 1e-3), ms / steps


def csrc_sha() -> str:
    """sha256 (first 16 hex digits) over the CUDA sources: ties an ncu capture to the kernels it was taken on."""
    import hashlib
    d = os.path.join(ROOT, "paper_2505_06711_b200", "csrc")
    hsh = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            with open(os.path.join(d, f), "rb") as fh:
                hsh.update(f.encode() + b"\0" + fh.read())
    return hsh.hexdigest()[:16]


def load_traffic(k: int) -> tuple[dict, str]:
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture) of
    the kernel groups, from the newest committed profiles/r*_dram_traffic.csv. A capture is only reported for the
    config it was taken on AND when its `# csrc_sha=` line equals the hash of the current kernel sources; otherwise
    `traffic` is null and the note says which capture is stale."""
    pdir = os.path.join(ROOT, "profiles")
    files = sorted(f for f in os.listdir(pdir) if f.endswith("_dram_traffic.csv")) if os.path.isdir(pdir) else []
    if not files:
        return {}, "no capture committed"
    out, sha = {}, None
    with open(os.path.join(pdir, files[-1])) as f:
        for line in f:
            if line.startswith("# csrc_sha="):
                sha = line.split("=", 1)[1].strip()
            if line.startswith("#") or not line.strip():
                continue
            group, cfg, nbytes = line.strip().split(",")[:3]
            if group != "group" and int(cfg) == k:
                out[group] = float(nbytes)
    if sha != csrc_sha():
        return {}, f"profiles/{files[-1]} was captured on kernel sources {sha}, current sources are {csrc_sha()}: stale, not reported"
    return out, f"profiles/{files[-1]} (csrc_sha {sha})"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx, self.rows, self.proc = gpu_index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.idx), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def wait_first(self, timeout_s: float):
        t0 = time.time()
        while self.proc is not None and not self.rows and time.time() - t0 < timeout_s:
            time.sleep(0.02)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip().split(", "))

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.strip().lower() == "active":
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_baseline(k: int, budget_atoms: int) -> dict:
    """The oracle, as it stands, on a same-density replica of config k (bounded sample)."""
    import oracle
    base = gen.CONFIGS[k]
    if base["kind"] == "fcc":
        nc = max(4, int(round((budget_atoms / 4) ** (1 / 3))))
        cfg = gen.make_config(k, ncell=min(nc, base["ncell"]))
    else:
        cfg = gen.make_config(k, n_mol=min(base["n_mol"], max(32, budget_atoms // 3)))
    n = len(cfg["pos"])
    t0 = time.perf_counter()
    oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"])
    dt = time.perf_counter() - t0
    return {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"1 E+F evaluation of a {n}-atom same-density replica of config {k} ({cfg['name']}), "
                      f"{dt:.2f} s, float64, OpenMP", "seconds": dt, "atoms": n}


def run_reference(args):
    """--impl reference: the float64 CPU oracle (there is no other reference implementation; tier note)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    for _ in range(min(args.warmup, 1)):
        cpu_baseline(args.config, args.ref_atoms)          # builds the oracle, touches the caches
    times, atoms, cb = [], 0, None
    for _ in range(args.steps):
        cb = cpu_baseline(args.config, args.ref_atoms)
        times.append(cb["seconds"])
        atoms = cb["atoms"]
    value = atoms * len(times) / sum(times)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {args.config} ({gen.CONFIGS[args.config]['name']}), bounded sample: "
                                   f"{atoms}-atom same-density replica per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cb["cores"], "kind": "oracle", "sample": cb["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number 1..5 (default 3: large water)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-atoms", type=int, default=24000, help="atoms of the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--T", type=int, default=None, help="override the number of layers (config 4 sweep)")
    ap.add_argument("--mlp-mode", default="fp32", choices=["fp32", "tf32"],
                    help="fp32 (default, 3xTF32 tensor-core GEMMs at FP32-class accuracy, the headline) or tf32 (plain TF32 "
                         "GEMMs, one accumulator per GEMM; tolerance restated in DESIGN.md section 2)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.mlp_mode == "tf32":
        os.environ["REANN_MLP_MODE"] = "tf32"      # read by the library once, at reann_create

    import torch
    import torch.distributed as dist
    import paper_2505_06711_b200 as R

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cfg = gen.make_config(args.config, T=args.T)
    cfg["vel"] = gen.maxwell_boltzmann(cfg["masses"], 300.0, cfg["seed_vel"])
    n = len(cfg["pos"])
    K, W = args.steps, max(args.warmup, 3)
    # The random-weight potential is not a physical liquid: forces on the randomly placed molecules are
    # ~5 eV/A rms (hundreds of eV/A where molecules overlap) and would heat the system within a few steps. The integrator therefore uses forces
    # scaled by 1e-4 so that displacements stay thermal (300 K) and the skin-triggered rebuild cadence
    # is that of an equilibrated liquid. The E+F evaluation that is timed is unaffected.
    dt_fs, acc = 0.5, 1e-4 * gen.configs.ACC_UNIT
    kT_300 = gen.configs.KB_EV * 300.0 * gen.configs.ACC_UNIT / acc     # 300 K in the integrator's (force-scaled) energy unit
    m = R.Reann.from_config(cfg)
    stream = torch.cuda.current_stream()
    m.set_stream(stream.cuda_stream)
    pos = torch.tensor(cfg["pos"], device="cuda")
    vel = torch.tensor(cfg["vel"], device="cuda")
    inv_m = torch.tensor(1.0 / cfg["masses"], device="cuda")
    E = torch.zeros(1, dtype=torch.float64, device="cuda")
    F = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    box = cfg["box"]

    vir = torch.zeros(9, dtype=torch.float64, device="cuda")

    def md_step():
        m.verlet(pos, vel, F, inv_m, dt_fs, acc, True)
        m.energy_forces(pos, box, E, F, vir)               # the full boundary call: E, F and the virial
        m.verlet(pos, vel, F, inv_m, dt_fs, acc, False)

    def timed(fn, reps=1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    # nvidia-smi takes a few hundred ms to attach to the driver and holds up CUDA calls while it does: start it
    # before the warm-up and wait for its first sample, so that only its periodic queries fall in the timed region
    sampler = ClockSampler(local_rank)
    sampler.start()
    m.build_neighbors(pos, box)
    m.energy_forces(pos, box, E, F, vir)
    # ---- "single evaluation incl. build" (BASELINE config 3; SURVEY 8(d) timing protocol): median of 5 ----
    t_build = sorted(timed(lambda: m.build_neighbors(pos, box)) for _ in range(5))[2]
    t_single = sorted(timed(lambda: (m.build_neighbors(pos, box), m.energy_forces(pos, box, E, F, vir))) for _ in range(5))[2]
    # warm-up through the same call as the timed region (same pointers: the CUDA graph of the evaluation is captured here)
    md_kw = dict(kT=kT_300, tau=100.0, F=F, virial=vir)
    md = m.md_run(pos, vel, inv_m, box, W, dt_fs, acc, **md_kw)
    torch.cuda.synchronize()
    sampler.wait_first(5.0)
    md = m.md_run(pos, vel, inv_m, box, 2, dt_fs, acc, xi=md["xi"], vxi=md["vxi"], forces_valid=True, **md_kw)
    torch.cuda.synchronize()
    sampler.rows.clear()

    # ---------------- device-resident timed region (profiling OFF: the production path) ----------------
    m.set_profiling(False)
    s0 = m.stats()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    # K steps of NVT MD (NVT at 300 K) in ONE library call: positions, velocities, forces and the
    # thermostat stay on the device (reann_md_run); F holds the forces at pos from the warm-up steps
    md = m.md_run(pos, vel, inv_m, box, K, dt_fs, acc, xi=md["xi"], vxi=md["vxi"], forces_valid=True, **md_kw)
    ev1.record(stream)
    torch.cuda.synchronize()
    ms_total = ev0.elapsed_time(ev1)
    value, ms_step = aggregate_throughput(n, K, ms_total, world)
    if world > 1:
        dist.barrier()
    ms_total = ms_step * K
    clocks = sampler.stop()
    s1 = m.stats()

    # ---------------- second, separate pass with per-group CUDA events (one more host sync per step) ----------------
    Kp = max(3, min(K, 20))
    m.set_profiling(True)
    p0 = m.stats()
    ms_prof = timed(md_step, Kp)
    p1 = m.stats()
    m.set_profiling(False)

    # ---------------- end-to-end leg: host buffers through the C ABI ----------------
    # replay: positions of an MD trajectory advanced on the host side of the boundary (pinned memory);
    # every step copies pos H2D inside reann_energy_forces and E, F, virial back D2H.
    pos_h = torch.empty((n, 3), dtype=torch.float64).pin_memory()
    F_h = torch.empty((n, 3), dtype=torch.float64).pin_memory()
    E_h = torch.empty(1, dtype=torch.float64).pin_memory()
    V_h = torch.empty(9, dtype=torch.float64).pin_memory()
    pos_h.copy_(pos.cpu()); vel_t = vel.cpu().clone()
    kick = (dt_fs * acc / torch.tensor(cfg["masses"]))[:, None].expand(n, 3).contiguous()   # [n, 3], full step
    pos_np, F_np, E_np, V_np = pos_h.numpy(), F_h.numpy(), E_h.numpy(), V_h.numpy()
    m.energy_forces(pos_np, box, E_np, F_np, V_np)
    m.energy_forces(pos_np, box, E_np, F_np, V_np)            # second call: the graph over the staging buffers exists
    vel_t.addcmul_(F_h, kick, value=0.5)                      # v(t + dt/2): leapfrog form of velocity Verlet from here on
    Ke = max(3, min(K, 25))
    torch.cuda.synchronize()
    # three consecutive segments of Ke steps of the same trajectory, the median segment is reported: a host-side
    # hiccup (seen once in six runs: one 80 ms gap in a 25-step wall-clock segment) does not decide the number
    seg = []
    for _ in range(3):
        t0 = time.perf_counter()
        for _ in range(Ke):                                   # host-side integrator (the caller's job in e2e use; torch CPU ops, all host cores)
            pos_h.add_(vel_t, alpha=dt_fs)                    # x(t + dt)
            m.energy_forces(pos_np, box, E_np, F_np, V_np)    # H2D pos, kernels, D2H E/F/virial, stream sync
            vel_t.addcmul_(F_h, kick)                         # v(t + 3dt/2): the two half kicks on the same forces in one pass
        seg.append(max_over_ranks(time.perf_counter() - t0))
    t_e2e = sorted(seg)[1]
    e2e = {"value": world * n * Ke / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(n * 24),
           "d2h_bytes_per_step": int(n * 24 + 8 + 72), "steps": Ke, "segments_s": [round(x, 5) for x in seg],
           "protocol": "median of 3 consecutive segments of `steps` steps"}

    if rank == 0:
        peaks = load_peaks()
        ncalls = max(1, p1["n_profiled_calls"] - p0["n_profiled_calls"])
        groups = {g: (p1[g] - p0[g]) / ncalls for g in ("ms_prep", "ms_edge_fwd", "ms_dense_fwd", "ms_gather",
                                                        "ms_dense_bwd", "ms_edge_bwd", "ms_rev_gather",
                                                        "ms_rev_gather_t0", "ms_output")}
        T, nphi, L = cfg["T"], cfg["n_gauss"], cfg["L"]
        nphip = (nphi + 3) // 4 * 4
        Na = gen.n_monomials(L)
        E_rc, E_list, n_ext = s1["n_edges_rc"], s1["n_edges_list"], s1["n_ext"]
        H1, H2 = cfg["H"]
        n_q = gen.n_orb_default(nphi, L)
        # Algorithmic work PER LAUNCH and launches per step of every kernel group (SURVEY.md 8(d) per-unit figures x
        # units): 1 FMA = 2 flop. dense groups = contraction (radial-pair form) + MLP GEMMs;
        # n_out is N_phi for the T-1 coefficient layers and 1 for the last. rev_gather has two launch kinds: layers
        # t >= 1 read rev (4 B) + kappa_e (4 N_phi B) per edge and write cbar (the g_e stash is summed over the layers
        # by k_edge_bwd and gathered once); the t = 0 launch reads rev + the summed g_e (c^0 is constant,
        # PAPER.md:76) and writes nothing per atom but the forces.
        nout_avg = ((T - 1) * nphi + 1) / T
        dense_flops = 2.0 * n * (n_q * H1 + H1 * H2 + H2 * nout_avg)
        work = {"ms_edge_fwd": ("alu", 2.0 * E_rc * nphi * Na, T), "ms_edge_bwd": ("alu", 4.0 * E_rc * nphi * Na, T),
                "ms_dense_fwd": ("tensor", dense_flops, T), "ms_dense_bwd": ("tensor", dense_flops, T),
                "ms_rev_gather_t0": ("hbm", float(E_rc) * (4 + 16) + n * 24.0, 1)}
        if T > 1:
            work["ms_rev_gather"] = ("hbm", float(E_rc) * (4 * nphip + 4) + n * (4.0 * nphip + 8), T - 1)
        sm_max = peaks.get("sm_max_mhz", 1965.0)
        alu_peak = N_SM * FP32_FMA_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        # TF32 peak = measured BF16 dense peak x the guide's nominal TF32/BF16 ratio (1.13 / 2.25 PFLOP/s);
        # the sustained figure, because the kernel is timed inside a long step
        tf32_peak = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]) * 0.5
        peak_of = {"alu": (alu_peak, "TFLOP/s", f"148 SM x 128 FP32 FMA lanes x 2 x {sm_max:.0f} MHz ({peaks['_source']} max SM clock)"),
                   "tensor": (tf32_peak, "TFLOP/s", f"0.5 x {peaks['_source']} sustained BF16 cuBLAS peak (TF32 nominal ratio)"),
                   "hbm": (peaks["hbm_gbs"], "GB/s", f"{peaks['_source']} HBM copy bandwidth")}
        traffic, traffic_note = load_traffic(args.config)

        def roof(g):
            bound, amount, launches = work[g]
            ms = groups[g] / launches
            peak, unit, src = peak_of[bound]
            ach = amount / (ms * 1e-3) / (1e9 if bound == "hbm" else 1e12) if ms > 0 else 0.0
            return {"bound": bound, "kernel": g.replace("ms_", ""), "achieved": ach, "peak": peak, "unit": unit,
                    "frac": ach / peak, "traffic": traffic.get(g.replace("ms_", "")), "peak_source": src,
                    "ms_per_launch": ms, "launches_per_step": launches,
                    "algorithmic_per_launch": amount, "algorithmic_unit": "bytes" if bound == "hbm" else "flop"}

        dom = max(work, key=lambda g: groups[g])
        roofline = roof(dom)
        roofline["traffic_source"] = traffic_note
        roofline["ms_per_step_by_group"] = {k.replace("ms_", ""): v for k, v in groups.items()}
        roofline["ms_per_step_by_group"]["note"] = (f"separate profiled pass of {Kp} steps at {ms_prof:.3f} ms/step "
                                                    "(per-group CUDA events add one host sync per step); `value` is timed with profiling off")
        roofline["other_kernels"] = [roof(g) for g in work if g != dom]
        # neighbour build (A1-A3), per rebuild: HBM bound; algorithmic bytes = positions in (24 B/atom) + ext records
        # (32 B each) + CSR col and rev written (4 + 4 B per list entry) + row_ptr (8 B/atom)
        nb_bytes = 24.0 * n + 32.0 * n_ext + 8.0 * E_list + 8.0 * n
        roofline["other_kernels"].append({"bound": "hbm", "kernel": "neighbor_build", "achieved": nb_bytes / (t_build * 1e-3) / 1e9,
                                          "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": nb_bytes / (t_build * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                          "traffic": traffic.get("neighbor_build"),   # k_nbr<count> + k_nbr<fill> + k_rev of the capture
                                          "peak_source": peak_of["hbm"][2], "ms_per_launch": t_build,
                                          "launches_per_step": (s1["n_rebuilds"] - s0["n_rebuilds"]) / K,
                                          "algorithmic_per_launch": nb_bytes, "algorithmic_unit": "bytes"})
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if args.mlp_mode == "fp32" else "tf32 (MLP GEMMs), f32 elsewhere", "data": "synthetic",
                "config": {"workload": f"config {args.config}: {cfg['name']} ({n} atoms, rc={cfg['rc']}, skin={cfg['skin']}, "
                                       f"T={T}, L={L}, n_gauss={nphi}, MLP {H1}x{H2}), velocity Verlet 0.5 fs + Nose-Hoover NVT 300 K (tau 100 fs), "
                                       f"device-resident reann_md_run",
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": "working set (compact edge list + stash, >300 MB) exceeds the 126 MB L2; no flush needed",
                           "virial": True, "profiling_in_timed_region": False, "mlp_mode": args.mlp_mode,
                           "rebuilds_in_timed_region": s1["n_rebuilds"] - s0["n_rebuilds"],
                           "md": {"kinetic_eV": md["kinetic"], "potential_eV": md["potential"], "xi": md["xi"], "vxi": md["vxi"]},
                           "n_edges_rc": E_rc, "n_edges_list": E_list, "n_ext": n_ext,
                           "stash_chunks": s1["stash_chunks"], "device_bytes": s1["bytes_device"]},
                "single_eval": {"ms": t_single, "value": n / (t_single * 1e-3), "unit": UNIT, "ms_build": t_build,
                                "what": "reann_build_neighbors + one reann_energy_forces (E, F, virial), device pointers, median of 5"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": s1["n_launches"] - s0["n_launches"],
                "roofline": roofline}
        if not args.no_cpu_baseline:
            cb = cpu_baseline(args.config, args.ref_atoms)
            line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
        print(json.dumps(line))
    m.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
