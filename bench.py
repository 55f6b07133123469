#!/usr/bin/env python
"""bench.py — ANI energy+forces throughput of the dhp hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 4]

A "step" is one pass of the whole hot path (neighbour search, AEV, 8-network MLP forward and
transpose-backward, AEV backward -> E, F) over one synthetic system.  Default workload: BASELINE.json
configs[3], the 98 000-atom biosystem the north_star targets are quoted on.  Prints ONE JSON line.

  value   atoms*evals/s, inputs resident in HBM, CUDA events over exactly K steps, max over ranks
  e2e     same metric through dhp_ani_energy_forces_host: pinned host buffers, H2D + D2H inside
  roofline  the dominant kernel (k_mlp_fused, tensor-bound): algorithmic FLOPs / device time of the timed (burst) loop vs the
            measured BURST bf16 peak; `frac` counts a product once, `issued_frac` the 3 MMAs issued per product
  roofline_mlp_phase / roofline_kernels   the same for the whole MLP phase and for every kernel group (HBM-bound ones vs copy bandwidth)
  cpu_baseline  the fp64 oracle, as it stands, on a bounded sample of the same workload (rank 0, N=1)
  parity_sample  that oracle sample against dhp_ani_energy_forces_partial over the same central atoms (|dE|/n, max |dF|)
  energy_only_ms_per_step, md, sustained   the energy-only call, the multiple-timestep driver with list reuse, and the same
                loop run for ~1 s (power-capped steady state) with its clocks, beside the headline
With N > 1 every rank evaluates its own replica of the system (independent problems, no collective on
the data path): weak scaling; --shard slab decomposes ONE system over the ranks instead (strong scaling).
--impl reference times the oracle itself.
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

from paper_2207_14276_b200 import workloads as W  # noqa: E402

METRIC = "ani_energy_forces_atoms_evals_per_s"
UNIT = "atoms*evals/s"
NS_PER_DAY_PER_EVAL_PER_S = 0.5e-6 * 86400.0      # 0.5 fs step
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r3_traffic_98k.csv")


def traffic_98k():
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per launch at configs[3], read from the committed summary of
    the `ncu --set full` capture of this same command (profiles/r3_traffic_98k.csv; profiles/r3_README.md names the command
    and the commit it was taken at).  Returns {} when the file is missing: `traffic` is then null, never a stale constant."""
    out = {}
    try:
        with open(TRAFFIC_FILE) as f:
            for line in f:
                line = line.strip()
                if not line or line.startswith("#") or line.startswith("key,"):
                    continue
                key, rd, wr = line.split(",")[:3]
                out[key] = out.get(key, 0.0) + float(rd) + float(wr)
    except OSError:
        pass
    return out


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw"

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 6 for i in range(4) if r[2 + i].lower().startswith("active")})
        pw = [float(r[6]) for r in self.rows if len(r) >= 7 and r[6].replace(".", "").isdigit()]
        self.power_w = float(max(pw)) if pw else None           # peak board power seen while sampling
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def oracle_sample_rate(system, params, blob, target_s: float = 15.0, seed: int = 0):
    """Oracle throughput (atoms*evals/s) on a bounded random sample of central atoms of `system`."""
    import oracle
    rng = np.random.default_rng(seed)
    n_try = min(system.n_atoms, 4 * oracle.num_threads())
    centres = rng.choice(system.n_atoms, n_try, replace=False).astype(np.int32)
    t0 = time.perf_counter()
    Ea, Fo, _ = oracle.energy_forces(system.pos, system.species, system.box, params, blob, system.n_models, centres=centres,
                                     mol_offsets=system.mol_offsets)
    dt = time.perf_counter() - t0
    n = n_try
    for _ in range(3):          # the probe over-estimates the per-atom cost (thread start-up): refine until ~target_s
        n = int(min(system.n_atoms, max(n_try, n * target_s / max(dt, 1e-3))))
        centres = rng.choice(system.n_atoms, n, replace=False).astype(np.int32)
        t0 = time.perf_counter()
        Ea, Fo, _ = oracle.energy_forces(system.pos, system.species, system.box, params, blob, system.n_models, centres=centres,
                                         mol_offsets=system.mol_offsets)
        dt = time.perf_counter() - t0
        if dt >= 0.6 * target_s or n == system.n_atoms:
            break
    return n / dt, n, dt, oracle.num_threads(), centres, Ea, Fo


def run_reference(args, system, params, blob):
    """--impl reference: the oracle as it stands on the host cores; each step a bounded sample."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    rng = np.random.default_rng(0)
    probe = min(system.n_atoms, 4 * oracle.num_threads())
    t0 = time.perf_counter()
    oracle.energy_forces(system.pos, system.species, system.box, params, blob, system.n_models,
                         centres=rng.choice(system.n_atoms, probe, replace=False).astype(np.int32),
                         mol_offsets=system.mol_offsets)
    per_atom = (time.perf_counter() - t0) / probe
    budget = 120.0 / max(1, args.steps + args.warmup)           # whole run within a few minutes
    n = int(max(oracle.num_threads(), min(system.n_atoms, budget / per_atom)))
    times = []
    for it in range(args.warmup + args.steps):
        centres = rng.choice(system.n_atoms, n, replace=False).astype(np.int32)
        t0 = time.perf_counter()
        oracle.energy_forces(system.pos, system.species, system.box, params, blob, system.n_models, centres=centres,
                             mol_offsets=system.mol_offsets)
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    total = sum(times)
    value = n * args.steps / total
    sample = f"{n} random central atoms of {system.name} per step (energies + the forces they exert), fp64, brute-force neighbours"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, system), "n_atoms": system.n_atoms, "n_models": system.n_models},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "ns_per_day_at_0.5fs": value / system.n_atoms * NS_PER_DAY_PER_EVAL_PER_S,
    }))


def workload_name(cfg: int, system) -> str:
    return f"BASELINE.json configs[{cfg - 1}]: {system.name}, {system.n_atoms} atoms, {system.n_models}-network ensemble"


def _ensure_built():
    """The libraries are built in-tree and git-ignored: a checkout without them builds them once (no CPU fallback exists)."""
    from paper_2207_14276_b200 import build as cuda_build
    from oracle import build as oracle_build
    if not os.path.exists(cuda_build.LIB):
        cuda_build.build(force=True)
    if not os.path.exists(oracle_build.LIB):
        oracle_build.build(force=True)


def main():
    _ensure_built()
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="dhp", choices=["dhp", "reference"])
    ap.add_argument("--config", type=int, default=4, help="1-based BASELINE.json config (default 4 = configs[3], 98k atoms)")
    ap.add_argument("--mlp", default="auto", choices=["auto", "simt", "tensor", "fp16"])
    ap.add_argument("--model", default="ani2x", choices=["ani2x", "ani1x"],
                    help="ani1x: the ANI-1x / ANI-1ccx shape of PAPER.md L87 / L159 on the same geometry (species H, C, N, O - the few S "
                         "become O; Rcr 5.2 Å, 4 x 8 angular grid, 384 features, 384-160-128-96-1 networks loaded zero-padded)")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: 'replicas' = one independent system per GPU (weak scaling, the default the contract asks for); "
                         "'slab' = ONE system, central atoms partitioned into spatial slabs, positions all-gathered, partial F reduce-scattered, E all-reduced over NCCL (strong scaling)")
    ap.add_argument("--simulate-world", type=int, default=0,
                    help="ONE GPU: time dhp_ani_energy_forces_partial for each of W slab masks of the system in turn (what each of W "
                         "ranks would run under --shard slab) and report the per-rank times and the strong-scaling ceiling "
                         "t_full / max_r t_r they predict; no collective is timed")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-md", action="store_true", help="skip the multiple-timestep driver measurement")
    ap.add_argument("--no-sustained", action="store_true", help="skip the ~1 s sustained-rate loop")
    ap.add_argument("--md-steps", type=int, default=40)
    ap.add_argument("--skin", type=float, default=1.0, help="Verlet skin (A) of the MD measurement")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "dhp" else args.warmup

    params = W.default_params()
    system = W.make_system(args.config)
    blob = W.make_weights(system.n_models)
    if args.model == "ani1x":
        params = W.ani1x_params()
        sp1 = system.species.copy()
        sp1[sp1 > W.O] = W.O                                   # S, F, Cl -> O: ANI-1x covers H, C, N, O
        system = W.System(system.name + "+ani1x", system.pos, sp1, system.box, system.mol_offsets, system.n_models)
        blob = W.embed_ani1x(W.make_weights_ani1x(system.n_models), system.n_models)
    if args.impl == "reference":
        run_reference(args, system, params, blob)
        return

    import torch
    import torch.distributed as dist
    from paper_2207_14276_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl dhp needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    d = B.Dhp(system.n_atoms, max_mols=system.n_mol, params=params, device=dev)
    d.dhp_set_mlp_mode({"auto": B.MLP_AUTO, "simt": B.MLP_SIMT, "tensor": B.MLP_TENSOR, "fp16": B.MLP_TENSOR_FP16}[args.mlp])
    w = d.dhp_weights_load(blob, system.n_models)
    tensor_path = d.dhp_tensor_path_available() and args.mlp != "simt"
    # each rank its own replica, positions jittered per step (N(0, 0.01^2) A^2) so nothing is trivially cached
    n_sets = 4
    pos_sets = [torch.from_numpy(W.jitter(system, 0.01, 100 + 17 * rank + k)).to(dev) for k in range(n_sets)]
    species = torch.from_numpy(system.species).to(dev)
    mol = None if system.mol_offsets is None else torch.from_numpy(system.mol_offsets).to(dev)
    n_mol = system.n_mol
    E = torch.empty(max(1, n_mol), dtype=torch.float64, device=dev)
    F = torch.empty((system.n_atoms, 3), dtype=torch.float32, device=dev)

    slab = args.shard == "slab" and system.mol_offsets is None
    if slab:
        # one system over all ranks: every rank holds all positions (same jitter seeds on every rank), owns the
        # central atoms of one equal-count slab and an index range of atoms; a step is the exchange SURVEY.md §8(e) specifies, on
        # the kernels' stream: all-gather of the owned positions, the partial call, reduce-scatter of the partial forces (each
        # rank ends up with the total force on the atoms it owns), 8-byte all-reduce of E
        from paper_2207_14276_b200 import shard
        pos_sets = [torch.from_numpy(W.jitter(system, 0.01, 100 + k)).to(dev) for k in range(n_sets)]
        masks = [shard.slab_mask_device(p_, system.box, world, rank) for p_ in pos_sets]
        ex = shard.Exchange(shard.owner_bounds(system.n_atoms, world), dev)
        F_part = torch.empty_like(F)

    def step(k):
        if slab:
            p_ = pos_sets[k % n_sets]
            ex.all_gather_positions(p_)
            d.dhp_ani_energy_forces_partial(p_, system.box, species, w, masks[k % n_sets], mol, E=E, F=F_part)
            ex.reduce_scatter_forces(F_part, F)
            ex.all_reduce_energy(E)
        else:
            d.dhp_ani_energy_forces(pos_sets[k % n_sets], system.box, species, w, mol, E=E, F=F)

    # set-up, not warm-up: the library builds the CUDA graph of an argument set on its second sighting, so every rotating
    # position buffer is passed twice here and no graph construction can fall into the warm-up or the timed region
    for k in range(2 * n_sets):
        step(k)
    for k in range(args.warmup):
        step(k)
    barrier()
    assert d.dhp_status() == 0, "device status word set during warm-up"

    # ---- device-resident timing --------------------------------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    l0 = d.dhp_launch_count()
    g0 = d.dhp_graph_replays()
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    for k in range(args.steps):
        step(k)
    ev1.record(stream)
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = d.dhp_launch_count() - l0
    graph_replays = d.dhp_graph_replays() - g0
    # per-phase CUDA events in a second pass over the same K steps: the events sit between the kernels, so small systems
    # (whose call is otherwise replayed as one CUDA graph) take the plain enqueue path while they are on
    d.dhp_profile_enable(True)
    d.dhp_profile_reset()
    for k in range(args.steps):
        step(k)
    phase_ms, calls = d.dhp_profile_read()
    d.dhp_profile_enable(False)
    n_row_tiles, n_active_blocks = d.dhp_debug_tile_blocks()
    clocks = sampler.stop() if rank == 0 else None
    assert d.dhp_status() == 0

    # ---- sustained rate: the same loop for ~1 s, long enough for the board's power management to settle (the 20-step
    # headline is a 50 ms burst); reported beside the headline with the clocks and power sampled during it -------------
    sustained = None
    if not args.no_sustained:
        n_sus = max(args.steps, int(1000.0 / max(ms_total / args.steps, 1e-3)))
        s2 = ClockSampler(local)
        if rank == 0:
            s2.start()
        barrier()
        d.dhp_profile_enable(True)
        d.dhp_profile_reset()
        ev0.record(stream)
        for k in range(n_sus):
            step(k)
        ev1.record(stream)
        barrier()
        ms_sus = ev0.elapsed_time(ev1) / n_sus
        ph_sus, calls_sus = d.dhp_profile_read()
        d.dhp_profile_enable(False)
        if rank == 0:
            c2 = s2.stop()
            atoms_s = system.n_atoms * (1 if slab else world)
            sustained = {"ms_per_step": ms_sus, "steps": n_sus, "value": atoms_s / (ms_sus * 1e-3), "unit": UNIT,
                         "ns_per_day_at_0.5fs": NS_PER_DAY_PER_EVAL_PER_S / (ms_sus * 1e-3),
                         "phase_ms": {k: v / max(calls_sus, 1) for k, v in ph_sus.items()},
                         "sm_mhz": c2["sm_mhz"], "reasons": c2["reasons"],
                         "power_w": getattr(s2, "power_w", None), "samples": c2.get("samples"),
                         "note": "steady state of a long run (board power management settled): the number an MD run gets"}

    # ---- strong-scaling prediction without a multi-GPU node: every slab's partial call on this one GPU -------------------
    simulated = None
    if args.simulate_world > 1 and system.mol_offsets is None and world == 1:
        from paper_2207_14276_b200 import shard
        Wn = args.simulate_world
        per_rank, per_phase = [], []
        for r in range(Wn):
            # the mask is derived inside the timed region on the first of every `mask_every` = 10 steps, as shard.ShardedMd does
            m_r = [shard.slab_mask_device(p_, system.box, Wn, r) for p_ in pos_sets]
            for k in range(3):
                d.dhp_ani_energy_forces_partial(pos_sets[k % n_sets], system.box, species, w, m_r[k % n_sets], mol, E=E, F=F)
            barrier()
            d.dhp_profile_enable(True)
            d.dhp_profile_reset()
            ev0.record(stream)
            for k in range(args.steps):
                if k % 10 == 0:
                    m_r[k % n_sets] = shard.slab_mask_device(pos_sets[k % n_sets], system.box, Wn, r)
                d.dhp_ani_energy_forces_partial(pos_sets[k % n_sets], system.box, species, w, m_r[k % n_sets], mol, E=E, F=F)
            ev1.record(stream)
            barrier()
            phr, cr = d.dhp_profile_read()
            d.dhp_profile_enable(False)
            per_rank.append(ev0.elapsed_time(ev1) / args.steps)
            per_phase.append({k_: v_ / max(cr, 1) for k_, v_ in phr.items()})
        t_full = ms_total / args.steps
        simulated = {"world": Wn, "ms_per_rank": per_rank, "phase_ms_slowest_rank": per_phase[int(np.argmax(per_rank))],
                     "ms_full_call_one_gpu": t_full, "predicted_speedup_ceiling": t_full / max(per_rank),
                     "predicted_parallel_efficiency_ceiling": t_full / max(per_rank) / Wn,
                     "exchange_bytes_per_rank_per_step": {"all_gather_positions": system.n_atoms * 12,
                                                          "reduce_scatter_forces": system.n_atoms * 12},
                     "note": "per-rank device time of the masked call measured on ONE GPU (slab mask refreshed every 10 steps inside "
                             "the timed loop); the NVLink exchange (2 x 1.2 MB per step) is not included - unmeasured at N > 1"}

    # ---- energy-only call (a1-a3), same inputs, device-resident ---------------------------------
    for k in range(2 * n_sets):            # every argument set twice: graphs are built on the second sighting
        d.dhp_ani_energy(pos_sets[k % n_sets], system.box, species, w, mol, E=E)
    barrier()
    ev0.record(stream)
    for k in range(args.steps):
        d.dhp_ani_energy(pos_sets[k % n_sets], system.box, species, w, mol, E=E)
    ev1.record(stream)
    barrier()
    ms_energy_only = ev0.elapsed_time(ev1) / args.steps

    # ---- the hot path inside the multiple-timestep driver (Eqs. 8-9): RESPA outer step 0.5 fs, 2 inner steps,
    # water O-H bonds in the inner loop, neighbour-list reuse with a 1 A skin; reported beside the headline, not in it ----
    md_out = None
    if system.mol_offsets is None and not args.no_md:
        mdi = W.md_inputs(system)
        d.dhp_set_skin(args.skin)
        hmd = d.dhp_md_create(mdi.inv_mass, mdi.bonds, mdi.bond_k, mdi.bond_r0) if len(mdi.bonds) else d.dhp_md_create(mdi.inv_mass)
        pos_md = torch.from_numpy(system.pos.copy()).to(dev)
        vel_md = torch.from_numpy(mdi.vel.copy()).to(dev)
        E_md = torch.empty(3, dtype=torch.float64, device=dev)
        d.dhp_md_run(hmd, pos_md, vel_md, system.box, species, w, 0.5, 2, 3, E_out=E_md)
        barrier()
        r0, l0m = d.dhp_nlist_rebuild_count(), d.dhp_launch_count()
        ev0.record(stream)
        d.dhp_md_run(hmd, pos_md, vel_md, system.box, species, w, 0.5, 2, args.md_steps, E_out=E_md)
        ev1.record(stream)
        barrier()
        ms_md = ev0.elapsed_time(ev1) / args.md_steps
        assert d.dhp_status() == 0
        md_out = {"ms_per_outer_step": ms_md, "outer_steps": args.md_steps, "dt_fs": 0.5, "n_inner": 2, "n_bonds": int(len(mdi.bonds)),
                  "skin_A": args.skin, "full_list_builds": d.dhp_nlist_rebuild_count() - r0,
                  "launches_per_step": (d.dhp_launch_count() - l0m) / args.md_steps,
                  "ns_per_day": 0.5e-6 * 86400.0 / (ms_md * 1e-3),
                  "note": "random-init networks: forces are ~5x larger than a trained model's, so atoms leave the skin sooner"}
        d.dhp_md_destroy(hmd)
        # the same evaluation loop as the headline (positions jittered by 0.01 A around one structure) with the skin on:
        # one full build, then every call filters the candidate list
        for k in range(3):
            step(k)
        barrier()
        d.dhp_profile_enable(True)
        d.dhp_profile_reset()
        r0 = d.dhp_nlist_rebuild_count()
        ev0.record(stream)
        for k in range(args.steps):
            step(k)
        ev1.record(stream)
        barrier()
        ph_reuse, calls_reuse = d.dhp_profile_read()
        d.dhp_profile_enable(False)
        md_out["list_reuse_only"] = {"ms_per_step": ev0.elapsed_time(ev1) / args.steps, "nlist_ms": ph_reuse["nlist"] / max(calls_reuse, 1),
                                     "full_list_builds": d.dhp_nlist_rebuild_count() - r0}
        d.dhp_set_skin(0.0)

    # ---- end to end through the host entry point -----------------------------------------------------
    pos_h = [torch.from_numpy(W.jitter(system, 0.01, 500 + 17 * rank + k)).pin_memory() for k in range(n_sets)]
    sp_h = torch.from_numpy(system.species).pin_memory()
    mol_h = None if system.mol_offsets is None else torch.from_numpy(system.mol_offsets).pin_memory()
    E_h = torch.empty(max(1, n_mol), dtype=torch.float64).pin_memory()
    F_h = torch.empty((system.n_atoms, 3), dtype=torch.float32).pin_memory()
    for k in range(3):
        d.dhp_ani_energy_forces_host(pos_h[k % n_sets], system.box, sp_h, w, mol_h, E=E_h, F=F_h)
    barrier()
    t0 = time.perf_counter()
    for k in range(args.steps):
        d.dhp_ani_energy_forces_host(pos_h[k % n_sets], system.box, sp_h, w, mol_h, E=E_h, F=F_h)
    barrier()
    e2e_s = time.perf_counter() - t0
    h2d = system.n_atoms * 12 + system.n_atoms * 4 + (0 if mol_h is None else mol_h.numel() * 4)
    d2h = max(1, n_mol) * 8 + system.n_atoms * 12

    times = torch.tensor([ms_total, e2e_s * 1e3], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
    ms_total, e2e_ms = float(times[0]), float(times[1])

    if rank == 0:
        pk = peaks()
        atoms_all = system.n_atoms * (1 if slab else world)
        value = atoms_all * args.steps / (ms_total * 1e-3)
        e2e_value = atoms_all * args.steps / (e2e_ms * 1e-3)
        ph = {k: v / max(calls, 1) for k, v in phase_ms.items()}            # ms per launch, CUDA events on the ctx stream
        ph["mlp"] = ph["mlp_g1"] + ph["mlp_mid"] + ph["mlp_b1"]
        N, M = system.n_atoms, system.n_models
        passes = (1 if args.mlp == "fp16" else 3) if tensor_path else 1
        # The timed region is a burst (K steps, ~50 ms at the default K = 20): the phase times are divided by the BURST bf16
        # peak.  The ~1 s `sustained` loop below carries its own phase times and is divided by the SUSTAINED peak.
        peak_t, peak_kind = pk["bf16_tflops"], "burst"
        # algorithmic FLOPs (forward + input gradient) per atom and network, by kernel; one product = one multiply-add
        f_g1_dense = 2.0 * 1008 * 256
        f_mid = 2.0 * (256 * 192 + 192 * 160 + 160 + 160 * 192 + 192 * 256)
        # G1 visits / B1 produces only the 64-wide feature blocks that are non-zero for the row tile: the zero blocks are
        # not work of the method (absent neighbour species), so the ALGORITHMIC count is over the active blocks only; the
        # dense-K figure is reported under its own key
        rows_pad = 128.0 * max(n_row_tiles, 1)
        act = n_active_blocks / max(n_row_tiles, 1)                        # active blocks per tile (of 16)
        f_g1 = 2.0 * 64 * 256 * act                                        # per atom and network
        # MMAs actually issued (3 passes per product, padded rows included)
        i_g1 = passes * 2.0 * M * 128.0 * 64 * 256 * n_active_blocks
        i_mid = passes * 2.0 * M * rows_pad * (256 * 192 + 192 * 160 + 160 * 192 + 192 * 256)

        def tensor_entry(name, ms, alg_flop, issued_flop, traffic, dense_flop=None, peak=None, kind=None):
            peak = peak or peak_t
            ach = alg_flop / (ms * 1e-3) / 1e12
            e = {"kernel": name, "bound": "tensor", "achieved": ach, "peak": peak, "peak_kind": kind or peak_kind, "unit": "TFLOP/s",
                 "frac": ach / peak, "traffic": traffic, "ms_per_launch": ms, "algorithmic_flop_per_launch": alg_flop,
                 "issued_tflops": issued_flop / (ms * 1e-3) / 1e12, "issued_frac": issued_flop / (ms * 1e-3) / 1e12 / peak}
            if dense_flop is not None:
                e["dense_k_tflops"] = dense_flop / (ms * 1e-3) / 1e12     # counts the skipped zero blocks: NOT a utilisation
            return e

        def hbm_entry(name, ms, bytes_per_atom, traffic, note, floor_us=None, compact_bytes_per_atom=None):
            # `frac` divides the survey's per-atom figure (§8(d): fp32 rows with every feature column, 4 x 1008 B + the list
            # reads) by the kernel time.  The kernel moves less than that: fp16 hi / lo planes of the ACTIVE feature blocks
            # only (`traffic` is what DRAM saw).  `frac_compacted` uses the survey's second figure, the row without the columns
            # of absent species.  Neither says how busy the kernel is - these kernels are bound on chip - which is what
            # `time_over_arithmetic_floor` is for.
            ach = bytes_per_atom * N / (ms * 1e-3) / 1e9
            e = {"kernel": name, "bound": "hbm", "achieved": ach, "peak": pk["hbm_gbs"], "unit": "GB/s",
                 "frac": ach / pk["hbm_gbs"], "traffic": traffic, "ms_per_launch": ms,
                 "algorithmic_bytes_per_launch": bytes_per_atom * N,
                 "note": note + "; `frac` counts the survey's dense fp32 row bytes, not the bytes the kernel moves (see `traffic`); "
                                "the number that says how far the kernel is from its limit is `time_over_arithmetic_floor`"}
            if compact_bytes_per_atom is not None:
                e["compacted_bytes_per_launch"] = compact_bytes_per_atom * N
                e["frac_compacted"] = compact_bytes_per_atom * N / (ms * 1e-3) / 1e9 / pk["hbm_gbs"]
            if floor_us is not None:                                      # the kernel's real floor is arithmetic, not bytes
                e["arithmetic_floor_us"] = floor_us
                e["time_over_arithmetic_floor"] = ms * 1e3 / floor_us
            return e

        tr = traffic_98k() if (args.config == 4 and tensor_path) else {}
        scale_n = N / 98000.0
        kernels = []
        # default: G1 runs inside the fused chain kernel (k_mlp_fused; DHP_TC_FUSE=0 keeps G1 and k_mlp_mid as two launches)
        fused_g1 = tensor_path and os.environ.get("DHP_TC_FUSE", "1") != "0" and args.mlp != "simt"
        n_mlp_kernels = 2 if fused_g1 else 3
        if tensor_path and fused_g1:
            kernels += [tensor_entry("k_mlp_fused (G1+G2+G3+out+B3+B2 in one kernel: AEV planes -> E_i, d1)", ph["mlp_g1"] + ph["mlp_mid"],
                                     (f_g1 + f_mid) * M * N, i_g1 + i_mid, tr.get("fused"), (f_g1_dense + f_mid) * M * N),
                        tensor_entry("k_gemm_tc2<GRAD,N-skip> (B1: d1 -> dE/dAEV) + energy reduction", ph["mlp_b1"], f_g1 * M * N, i_g1, tr.get("b1"),
                                     f_g1_dense * M * N)]
        elif tensor_path:
            kernels += [tensor_entry("k_gemm_tc<CELU,K-skip> (G1: AEV -> h1)", ph["mlp_g1"], f_g1 * M * N, i_g1, tr.get("g1"), f_g1_dense * M * N),
                        tensor_entry("k_mlp_mid (G2+G3+out+B3+B2 fused: h1 -> E_i, d1)", ph["mlp_mid"], f_mid * M * N, i_mid, tr.get("mid")),
                        tensor_entry("k_gemm_tc<GRAD,N-skip> (B1: d1 -> dE/dAEV) + energy reduction", ph["mlp_b1"], f_g1 * M * N, i_g1, tr.get("b1"),
                                     f_g1_dense * M * N)]
        # arithmetic floors at configs[3]: a1 386 candidate tests x ~12 fp64 ops per atom; a2 3.3 k MUFU
        # ops per atom at 16 / clk / SM; a5 about twice a2's arithmetic
        kernels += [hbm_entry("nlist (a1: all kernels)", ph["nlist"], 264.0, tr.get("nlist"), "working set is L2-resident; instruction-bound",
                              11.0 * scale_n),
                    hbm_entry("k_aev_fwd (a2)", ph["aev_fwd"], 4256.0, tr.get("aev_fwd"), "L1 / shared-memory pipe and issue-bound; the floor that binds is MUFU, not HBM", 69.0 * scale_n,
                              2464.0),
                    hbm_entry("k_aev_bwd + k_unsort_forces (a5)", ph["aev_bwd"], 4268.0, tr.get("aev_bwd"), "L1 / shared-memory pipe bound", 140.0 * scale_n, 2476.0)]
        if tensor_path:
            roof = dict(max(kernels[:n_mlp_kernels], key=lambda k: k["ms_per_launch"]))          # the dominant kernel of the step
            roof["peak_source"] = f"{pk['source']} {peak_kind} bf16 peak (fp16 operands, same rate); the timed loop is a burst"
            roof["arithmetic"] = ("fp16 operands, 1 tcgen05 MMA per product, fp32 accumulate (opt-in mixed precision, outside the parity bar)"
                                  if args.mlp == "fp16" else "fp16 two-term split, 3 tcgen05 MMAs per product, fp32 accumulate: `frac` counts one "
                                  "product once (ceiling 1/3), `issued_frac` counts the MMAs issued")
            if fused_g1:
                tsum = (tr["fused"] + tr["b1"]) if {"fused", "b1"} <= set(tr) else None
            else:
                tsum = (tr["g1"] + tr["mid"] + tr["b1"]) if {"g1", "mid", "b1"} <= set(tr) else None
            mlp_phase = tensor_entry("MLP phase (k_mlp_fused + B1)" if fused_g1 else "MLP phase (G1 + k_mlp_mid + B1)", ph["mlp"], (2 * f_g1 + f_mid) * M * N, 2 * i_g1 + i_mid, tsum,
                                     (2 * f_g1_dense + f_mid) * M * N)
            mlp_phase.update({"row_tiles": n_row_tiles, "active_feature_blocks_per_tile": act})
            if sustained is not None and sustained.get("phase_ms"):
                sp = sustained["phase_ms"]
                sustained["roofline"] = tensor_entry(roof["kernel"], sp["mlp_g1"] + sp["mlp_mid"] if "k_mlp_fused" in roof["kernel"] else
                                                     sp["mlp_mid"] if "k_mlp_mid" in roof["kernel"] else sp["mlp_b1"] if "B1" in roof["kernel"] else sp["mlp_g1"],
                                                     roof["algorithmic_flop_per_launch"],
                                                     roof["issued_tflops"] * roof["ms_per_launch"] * 1e9, roof["traffic"],
                                                     peak=pk["bf16_tflops_sustained"], kind="sustained")
        else:
            flops = (2 * f_g1_dense + f_mid) * M * N
            roof = tensor_entry("mlp_simt (fp32 FFMA scaffold; tensor path not in use)", ph["mlp"], flops, flops, None)
            mlp_phase = roof
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if slab else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(args.config, system), "n_atoms": system.n_atoms,
                       "n_models": system.n_models, "parallelism": (f"one system, central atoms in {world} slab(s), all-gather of owned positions + reduce-scatter of partial F + all-reduce of E over NCCL" if slab
                                       else f"{world} independent replica(s), one per GPU"),
                       "l2": "per-step working set (AEV planes, dE/dAEV and activation buffers, > 1 GB) exceeds the 126 MB L2; "
                             "positions rotate over 4 jittered copies",
                       "mlp": "tensor" if tensor_path else "simt"},
            "ns_per_day_at_0.5fs": value / atoms_all * NS_PER_DAY_PER_EVAL_PER_S,   # per replica
            "evals_per_s_per_gpu": value / atoms_all,
            "phase_ms": ph,
            "gpu_launches": int(launches), "graph_replays": int(graph_replays),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": e2e_ms / args.steps},
            "energy_only_ms_per_step": ms_energy_only, "md": md_out, "sustained": sustained, "simulated_world": simulated,
            "roofline": roof,
            "roofline_mlp_phase": mlp_phase,
            "roofline_kernels": kernels,
        }
        if world == 1 and not args.no_cpu_baseline:
            rate, n, dt, cores, centres, Ea, Fo = oracle_sample_rate(system, params, blob)
            out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": f"{n} random central atoms of {system.name} (energies + the forces they exert) "
                                             f"in {dt:.1f} s, fp64, brute-force neighbours"}
            # the same sample through the library (partial evaluation over exactly these central atoms, unjittered
            # positions): parity of this launch configuration at full size, beside the timing
            mask = torch.zeros(system.n_atoms, dtype=torch.uint8, device=dev)
            mask[torch.from_numpy(centres.astype(np.int64)).to(dev)] = 1
            pos0 = torch.from_numpy(system.pos).to(dev)
            Ec, Fc = d.dhp_ani_energy_forces_partial(pos0, system.box, species, w, mask, mol)
            torch.cuda.synchronize()
            ea = d.dhp_debug_atomic_energy().cpu().numpy()
            out["parity_sample"] = {"central_atoms": int(n), "abs_dE_per_atom": float(abs(Ec.sum().item() - Ea.sum()) / n),
                                    "max_abs_dE_atom": float(np.abs(ea[centres] - Ea).max()),
                                    "max_abs_dF": float(np.abs(Fc.cpu().numpy() - Fo).max()),
                                    "bars": {"abs_dE_per_atom": 1e-6, "max_abs_dF": 5e-5}, "status": int(d.dhp_status())}
        print(json.dumps(out))
    d.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
