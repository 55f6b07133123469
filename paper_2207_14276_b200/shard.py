"""Host-side sharding of the hot path over one process per GPU.

The path shards in two ways, and neither needs a data-path collective inside the kernels:

* independent problems (BASELINE.json configs[4], batched replicas; `bench.py --gpus N` replicas): every rank
  evaluates whole molecules / whole systems; results are gathered, nothing is reduced;
* one large system: the energy is a sum of local atomic terms, so the *central atoms* are
  partitioned into spatial slabs, every rank sees all positions (all-gather; 1.6 MB at 98 k atoms), accumulates
  the forces its centres exert on every atom, and the partial forces / energies are summed (reduce-scatter or
  all-reduce).  No AEV is computed twice — the redundancy the paper's halo scheme pays for (L194).

This module holds only index arithmetic and `torch.distributed` plumbing (gloo on CPU, nccl on GPUs); it contains
none of the method's arithmetic and does not import the oracle.
"""
from __future__ import annotations

from typing import Optional, Tuple

import numpy as np


def shard_range(n_units: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous balanced split of `n_units` into `world` parts: [lo, hi) of `rank` (sizes differ by at most 1)."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_molecules(mol_offsets: np.ndarray, world: int, rank: int):
    """Batched replicas: (mol_lo, mol_hi, atom_lo, atom_hi, local_offsets) of this rank's whole molecules.

    `local_offsets` (int32, starts at 0) is what the rank passes as `mol_offsets` with `pos[atom_lo:atom_hi]`."""
    off = np.asarray(mol_offsets, dtype=np.int64)
    m_lo, m_hi = shard_range(off.size - 1, world, rank)
    a_lo, a_hi = int(off[m_lo]), int(off[m_hi])
    return m_lo, m_hi, a_lo, a_hi, (off[m_lo:m_hi + 1] - a_lo).astype(np.int32)


def slab_owner(pos: np.ndarray, box: Optional[np.ndarray], world: int, axis: int = 0) -> np.ndarray:
    """Owner rank of every atom as a *central* atom: equal-count slabs along `axis`.

    Periodic coordinates are wrapped into [0, L) first so that a slab is a contiguous region of the cell; ties are
    broken by atom index (stable sort), which makes the partition deterministic and identical on every rank."""
    x = np.asarray(pos, dtype=np.float64)[:, axis]
    if box is not None:
        L = float(box[axis])
        x = x - L * np.floor(x / L)
    order = np.argsort(x, kind="stable")
    owner = np.empty(x.size, dtype=np.int32)
    for r in range(world):
        lo, hi = shard_range(x.size, world, r)
        owner[order[lo:hi]] = r
    return owner


def slab_centres(pos: np.ndarray, box: Optional[np.ndarray], world: int, rank: int, axis: int = 0) -> np.ndarray:
    """Ascending int32 indices of the atoms whose atomic energy (and the forces it generates) `rank` evaluates."""
    return np.nonzero(slab_owner(pos, box, world, axis) == rank)[0].astype(np.int32)


# ---- torch.distributed plumbing (the process group is the caller's: gloo on CPU, nccl on GPUs) ---------------------
def max_over_ranks(values, group=None):
    """Element-wise MAX over ranks of a 1-D sequence of floats (device time per phase, ms): every multi-GPU number is
    the slowest rank's."""
    import torch
    import torch.distributed as dist
    t = torch.as_tensor(list(values), dtype=torch.float64)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
        t = t.to(dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return [float(v) for v in t.cpu()]


def gather_molecule_energies(E_local, n_mol: int, group=None):
    """Independent problems: concatenate the per-molecule energies of all ranks in rank order (shard_range order)."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    sizes = [shard_range(n_mol, world, r) for r in range(world)]
    width = max(hi - lo for lo, hi in sizes)
    buf = torch.zeros(width, dtype=torch.float64, device=E_local.device)
    lo, hi = sizes[rank]
    buf[: hi - lo] = E_local[: hi - lo]
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf, group=group)
    return torch.cat([parts[r][: sizes[r][1] - sizes[r][0]] for r in range(world)])


def sum_partial_forces(E_partial, F_partial, group=None):
    """One large system, slab-partitioned centres: total E and F = sums of the ranks' partial results (in place)."""
    import torch.distributed as dist
    dist.all_reduce(F_partial, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(E_partial, op=dist.ReduceOp.SUM, group=group)
    return E_partial, F_partial


# ---- device side: one large system over N GPUs -------------------------------
def slab_mask_device(pos, box, world: int, rank: int, axis: int = 0):
    """`slab_owner(...) == rank` evaluated with torch ops on the device that holds `pos` (fp32 [N, 3]): the uint8
    central-atom mask `dhp_ani_energy_forces_partial` takes.  Same rule as `slab_owner` (wrap into [0, L), stable
    sort, equal counts), so every rank derives the same partition from the same positions.  Index arithmetic only."""
    import torch
    x = pos[:, axis].to(torch.float64)
    if box is not None:
        L = float(box[axis])
        x = x - L * torch.floor(x / L)
    order = torch.argsort(x, stable=True)
    lo, hi = shard_range(int(x.numel()), world, rank)
    mask = torch.zeros(x.numel(), dtype=torch.uint8, device=pos.device)
    mask[order[lo:hi]] = 1
    return mask


def ani_energy_forces_sharded(dhp, pos, box, species, weights, central, mol_offsets=None, group=None):
    """One evaluation of a system whose central atoms are partitioned over the ranks of `group`.

    Every rank holds all positions (after an MD step: all-gather of the owned slices, 1.6 MB at 98 k atoms), runs
    a1-a5 for its own central atoms only (`central`, from `slab_mask_device`) and the partial energies and forces
    are summed over ranks - one all-reduce of F (1.2 MB) and one of E (8 B) on NCCL, enqueued on the stream the
    kernels ran on, no host synchronisation.  Returns the total (E, F), identical on every rank."""
    import torch.distributed as dist
    E, F = dhp.dhp_ani_energy_forces_partial(pos, box, species, weights, central, mol_offsets)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(F, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(E, op=dist.ReduceOp.SUM, group=group)
    return E, F
