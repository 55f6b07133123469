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


# ---- the exchange SURVEY.md §8(e) specifies: all-gather of owned positions, reduce-scatter of partial forces ----------
def owner_bounds(n_atoms: int, world: int, unit: int = 1, first_unit_atom: int = 0) -> np.ndarray:
    """Index ranges of the atoms each rank OWNS for integration: [bounds[r], bounds[r+1]).  Ownership is by atom index
    (fixed for a run - it decides who integrates an atom and who receives its total force), independent of the spatial
    slabs that decide who evaluates an atom as a CENTRE.  Cuts fall on multiples of `unit` atoms counted from
    `first_unit_atom` (3 for the waters of the generators, so that no O-H bond is split between two ranks)."""
    b = np.empty(world + 1, dtype=np.int64)
    b[0], b[world] = 0, n_atoms
    for r in range(1, world):
        cut = shard_range(n_atoms, world, r)[0]
        if unit > 1 and cut > first_unit_atom:
            cut = first_unit_atom + (cut - first_unit_atom) // unit * unit
        b[r] = cut
    if np.any(np.diff(b) < 0):
        raise ValueError("bad ownership bounds")
    return b


class Exchange:
    """Padded layout for collectives with equal chunks: rank r's atoms [bounds[r], bounds[r+1]) occupy rows
    [r * chunk, r * chunk + len_r) of a [world * chunk, 3] buffer.  Index arithmetic and torch.distributed calls only.
    The collectives run whenever a process group of `world` ranks exists - also a group of ONE rank, where they are the
    identity: that is the only way the NCCL branch (reduce_scatter_tensor / all_gather_into_tensor on CUDA tensors) can be
    executed on a one-GPU box.  Without a process group (world must then be 1) the calls are plain copies.  The padded
    buffers are allocated on first use and kept, so that a step allocates nothing."""

    def __init__(self, bounds, device, group=None):
        import torch
        import torch.distributed as dist
        self.torch, self.dist, self.group = torch, dist, group
        self.bounds = np.asarray(bounds, dtype=np.int64)
        self.world = int(self.bounds.size - 1)
        self.n = int(self.bounds[-1])
        self.chunk = int(max(1, np.diff(self.bounds).max()))
        have_pg = dist.is_available() and dist.is_initialized()
        if have_pg and dist.get_world_size(group) != self.world:
            raise ValueError(f"bounds describe {self.world} ranks, the process group has {dist.get_world_size(group)}")
        if not have_pg and self.world != 1:
            raise ValueError("more than one rank needs an initialised process group")
        self.rank = dist.get_rank(group) if have_pg else 0
        self.live = have_pg
        self.backend = dist.get_backend(group) if have_pg else None
        to_pad = np.full(self.world * self.chunk, self.n, dtype=np.int64)          # padding rows read the extra zero row
        to_atom = np.empty(self.n, dtype=np.int64)
        for r in range(self.world):
            lo, hi = int(self.bounds[r]), int(self.bounds[r + 1])
            to_pad[r * self.chunk: r * self.chunk + hi - lo] = np.arange(lo, hi)
            to_atom[lo:hi] = r * self.chunk + np.arange(hi - lo)
        self.to_pad = torch.from_numpy(to_pad).to(device)
        self.to_atom = torch.from_numpy(to_atom).to(device)
        self.lo, self.hi = int(self.bounds[self.rank]), int(self.bounds[self.rank + 1])
        self._buf = {}

    def _buffers(self, like):
        """(padded [world*chunk, 3], chunk [chunk, 3], extended [n + 1, 3] with a zero last row) for like's dtype / device."""
        key = (like.dtype, like.device)
        if key not in self._buf:
            t = self.torch
            self._buf[key] = (t.empty((self.world * self.chunk, 3), dtype=like.dtype, device=like.device),
                              t.zeros((self.chunk, 3), dtype=like.dtype, device=like.device),
                              t.zeros((self.n + 1, 3), dtype=like.dtype, device=like.device))
        return self._buf[key]

    def reduce_scatter_forces(self, F_partial, F_total):
        """F_total[lo:hi] = sum over ranks of F_partial[lo:hi] (the rows this rank owns); other rows are left alone.
        NCCL: one reduce-scatter of the padded buffer (1.2 MB / world per rank at 98 k atoms); gloo (CPU tests) has no
        reduce-scatter, there the same result comes from an all-reduce and a slice."""
        t = self.torch
        if not self.live:
            F_total[self.lo:self.hi] = F_partial[self.lo:self.hi]
            return F_total
        padded, out, ext = self._buffers(F_partial)
        ext[: self.n] = F_partial                                                   # the last row stays zero
        t.index_select(ext, 0, self.to_pad, out=padded)
        if self.backend == "nccl":
            self.dist.reduce_scatter_tensor(out, padded, op=self.dist.ReduceOp.SUM, group=self.group)
        else:
            self.dist.all_reduce(padded, op=self.dist.ReduceOp.SUM, group=self.group)
            out = padded[self.rank * self.chunk:(self.rank + 1) * self.chunk]
        F_total[self.lo:self.hi] = out[: self.hi - self.lo]
        return F_total

    def all_gather_positions(self, pos):
        """Every rank has integrated its own rows of `pos` [N, 3]; afterwards every rank holds all rows (in place)."""
        t = self.torch
        if not self.live:
            return pos
        full, mine, ext = self._buffers(pos)
        mine[: self.hi - self.lo] = pos[self.lo:self.hi]                            # rows beyond the own count stay zero
        self.dist.all_gather_into_tensor(full, mine, group=self.group)
        t.index_select(full, 0, self.to_atom, out=ext[: self.n])
        pos.copy_(ext[: self.n])
        return pos

    def all_reduce_energy(self, E):
        if self.live:
            self.dist.all_reduce(E, op=self.dist.ReduceOp.SUM, group=self.group)
        return E


class ShardedMd:
    """The multiple-timestep driver over `world` ranks.

    Every rank owns an index range of atoms (it integrates them) and, per evaluation, a spatial slab of CENTRAL atoms (it
    evaluates their atomic energies and the forces they exert).  One outer step:
        dhp_md_open   (own atoms: half kick with the slow force, inner loop with the own bonds)
        all-gather    positions
        dhp_ani_energy_forces_partial over the own slab (mask refreshed every `mask_every` steps: the argsort is on the
                      list-rebuild cadence, not on every step)
        reduce-scatter of the partial forces -> total slow force of the own atoms; all-reduce of E (8 bytes)
        dhp_md_close  (own atoms: second half kick)
    `dhp` is a binding.Dhp (or, in the CPU tests, a stand-in with the same four methods)."""

    def __init__(self, dhp, weights, species, box, bounds, inv_mass, bonds=None, bond_k=None, bond_r0=None,
                 mask_every: int = 10, group=None, dtype=None):
        import torch
        self.torch = torch
        self.dhp, self.weights, self.species, self.box = dhp, weights, species, box
        self.ex = Exchange(bounds, species.device, group)
        lo, hi = self.ex.lo, self.ex.hi
        if bonds is not None and len(bonds):
            b = np.asarray(bonds)
            own = (b[:, 0] >= lo) & (b[:, 0] < hi)
            if np.any(own != ((b[:, 1] >= lo) & (b[:, 1] < hi))):
                raise ValueError("a bond is split between two ranks: cut the ownership ranges at molecule boundaries")
            bonds, bond_k, bond_r0 = b[own], np.asarray(bond_k)[own], np.asarray(bond_r0)[own]
        self.md = dhp.dhp_md_create(inv_mass, bonds if bonds is not None and len(bonds) else None,
                                    bond_k if bonds is not None and len(bonds) else None,
                                    bond_r0 if bonds is not None and len(bonds) else None)
        self.mask_every, self.steps_since_mask, self.mask = int(mask_every), 0, None
        self.F_total = torch.zeros((self.ex.n, 3), dtype=dtype or torch.float32, device=species.device)
        # outputs of the partial call and the mask live in buffers that are allocated once: the library replays a captured graph
        # only when a call's pointers repeat (include/dhp.h: dhp_graph_replays), and a step should not allocate anyway
        self.F_part = torch.zeros((self.ex.n, 3), dtype=dtype or torch.float32, device=species.device)
        self.E = torch.zeros(1, dtype=torch.float64, device=species.device)
        self.primed = False

    def _slow(self, pos):
        if self.mask is None or self.steps_since_mask >= self.mask_every:
            m = slab_mask_device(pos, self.box, self.ex.world, self.ex.rank)
            if self.mask is None:
                self.mask = m
            else:
                self.mask.copy_(m)                       # same address: the argument set of the partial call does not change
            self.steps_since_mask = 0
        self.steps_since_mask += 1
        self.dhp.dhp_ani_energy_forces_partial(pos, self.box, self.species, self.weights, self.mask, E=self.E, F=self.F_part)
        self.ex.reduce_scatter_forces(self.F_part, self.F_total)
        self.ex.all_reduce_energy(self.E)

    def run(self, pos, vel, dt: float, n_inner: int, n_steps: int):
        """`n_steps` outer steps in place on pos / vel [N, 3] (all rows of pos are current on every rank on return; only
        the own rows of vel are).  Returns the total E_ANI at the final positions (identical on every rank)."""
        lo, hi = self.ex.lo, self.ex.hi
        if not self.primed:
            self._slow(pos)
            self.primed = True
        for _ in range(n_steps):
            self.dhp.dhp_md_open(self.md, pos, vel, self.box, self.F_total, dt, n_inner, lo, hi)
            self.ex.all_gather_positions(pos)
            self._slow(pos)
            self.dhp.dhp_md_close(self.md, vel, self.F_total, dt, n_inner, lo, hi)
        return self.E
