"""Host-side multi-process logic on CPU: world_size 2, gloo backend, 127.0.0.1 rendezvous.

No GPU here, so the per-rank compute is played by the fp64 oracle (tests may use it); what is under test is the
sharding arithmetic and the gather / reduce plumbing of `paper_2207_14276_b200.shard`: the sharded result must equal
the single-process one, units must be covered exactly once, timing is the max over ranks.
"""
import os
import socket

import numpy as np
import pytest

from paper_2207_14276_b200 import shard
from paper_2207_14276_b200 import workloads as W

WORLD = 2


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_range_covers_every_unit_once():
    for n in (0, 1, 2, 7, 1024, 98000):
        for world in (1, 2, 3, 8):
            parts = [shard.shard_range(n, world, r) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(4, 2, 2)


def test_shard_molecules_keeps_molecules_whole():
    s = W.replicas_1024x30(n_mol=11)
    seen = []
    for r in range(3):
        m_lo, m_hi, a_lo, a_hi, off = shard.shard_molecules(s.mol_offsets, 3, r)
        assert off[0] == 0 and off[-1] == a_hi - a_lo and np.all(np.diff(off) == 30)
        assert a_lo == s.mol_offsets[m_lo] and a_hi == s.mol_offsets[m_hi]
        seen += list(range(m_lo, m_hi))
    assert seen == list(range(11))


def test_slab_owner_is_a_balanced_partition_and_periodic_wrap_invariant():
    s = W.make_system(1)
    own = shard.slab_owner(s.pos, s.box, 4)
    assert sorted(np.bincount(own, minlength=4)) == [72, 72, 72, 72]
    cs = [shard.slab_centres(s.pos, s.box, 4, r) for r in range(4)]
    assert np.array_equal(np.sort(np.concatenate(cs)), np.arange(s.n_atoms))
    # whole-box shifts do not move an atom to another slab: positions on a 2^-10 grid in a 16 Å box, so that the shift
    # by 3 L is exact in fp32 and the partition must be EQUAL, not approximately equal
    box = np.array([16.0, 16.0, 16.0], np.float32)
    q = (np.round(np.mod(s.pos.astype(np.float64), 16.0) * 1024) / 1024).astype(np.float32)
    own = shard.slab_owner(q, box, 4)
    shifted = q.copy()
    shifted[::5, 0] += np.float32(48.0)
    shifted[1::7, 0] -= np.float32(32.0)
    delta = shifted[:, 0].astype(np.float64) - q[:, 0].astype(np.float64)
    assert set(np.unique(delta)) <= {0.0, 48.0, -32.0, 16.0} and np.count_nonzero(delta) > 80     # exact whole-box shifts
    assert np.array_equal(shard.slab_owner(shifted, box, 4), own)


def _worker(rank, port, results):
    import torch
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        params = W.default_params()
        blob = W.make_weights(1)
        # (1) independent problems: molecules sharded, energies gathered in order
        s = W.replicas_1024x30(n_mol=7)
        m_lo, m_hi, a_lo, a_hi, off = shard.shard_molecules(s.mol_offsets, WORLD, rank)
        Ea, Fa, _ = oracle.energy_forces(s.pos[a_lo:a_hi], s.species[a_lo:a_hi], None, params, blob, 1, mol_offsets=off)
        E_local = torch.from_numpy(np.add.reduceat(Ea, off[:-1].astype(np.int64)))
        E_all = shard.gather_molecule_energies(E_local, 7).numpy()
        # (2) one system, central atoms in slabs: partial forces and energies summed
        w = W.make_system(1)
        centres = shard.slab_centres(w.pos, w.box, WORLD, rank)
        Ec, Fc, _ = oracle.energy_forces(w.pos, w.species, w.box, params, blob, 1, centres=centres)
        E_part = torch.tensor([Ec.sum()], dtype=torch.float64)
        F_part = torch.from_numpy(Fc.copy())
        shard.sum_partial_forces(E_part, F_part)
        # (2b) the same through shard.ani_energy_forces_sharded with the device-side slab rule (torch ops, here on
        # CPU tensors) and a stand-in context whose partial call is played by the oracle
        class OracleCtx:
            def dhp_ani_energy_forces_partial(self, pos, box, species, weights, central, mol_offsets=None):
                c = np.nonzero(central.numpy())[0].astype(np.int32)
                Ec, Fc, _ = oracle.energy_forces(pos.numpy(), species.numpy(), box, params, weights, 1, centres=c)
                return torch.tensor([Ec.sum()], dtype=torch.float64), torch.from_numpy(Fc.copy())
        pos_t, sp_t = torch.from_numpy(w.pos), torch.from_numpy(w.species)
        mask = shard.slab_mask_device(pos_t, w.box, WORLD, rank)
        assert np.array_equal(np.nonzero(mask.numpy())[0], centres)
        E_sh, F_sh = shard.ani_energy_forces_sharded(OracleCtx(), pos_t, w.box, sp_t, blob, mask)
        assert abs(E_sh.item() - E_part.item()) <= 1e-12 and np.max(np.abs(F_sh.numpy() - F_part.numpy())) <= 1e-14
        # (3) timing: slowest rank
        t = shard.max_over_ranks([1.0 + rank, 5.0 - rank])
        if rank == 0:
            results.put((E_all, E_part.numpy(), F_part.numpy(), t, len(centres)))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_sharded_results_equal_single_process():
    import torch.multiprocessing as mp
    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, port, q)) for r in range(WORLD)]
    for p in procs:
        p.start()
    E_all, E_sum, F_sum, t, n_c0 = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    params = W.default_params()
    blob = W.make_weights(1)
    s = W.replicas_1024x30(n_mol=7)
    Eo, _ = oracle.total_energy_forces(W.System(s.name, s.pos, s.species, None, s.mol_offsets, 1), params, blob)
    assert np.allclose(E_all, Eo, rtol=0, atol=1e-12)
    w = W.make_system(1)
    Ew, Fw = oracle.total_energy_forces(w, params, blob)
    assert n_c0 == w.n_atoms // 2
    assert abs(E_sum[0] - Ew[0]) <= 1e-10
    assert np.max(np.abs(F_sum - Fw)) <= 1e-12
    assert t == [2.0, 5.0]


# ---- the exchange of SURVEY.md §8(e) and the sharded multiple-timestep step ---------------------------------------------
def test_owner_bounds_cut_at_molecule_boundaries():
    b = shard.owner_bounds(98000, 8)
    assert b[0] == 0 and b[-1] == 98000 and np.all(np.diff(b) > 0) and np.diff(b).max() - np.diff(b).min() <= 1
    b = shard.owner_bounds(23558, 4, unit=3, first_unit_atom=11084)          # waters start after 11 084 protein atoms
    assert all(c <= 11084 or (c - 11084) % 3 == 0 for c in b[1:-1])
    s = W.make_system(1)
    m = W.md_inputs(s)
    b = shard.owner_bounds(s.n_atoms, 2, unit=3)
    for i, j in m.bonds:
        assert np.searchsorted(b, i, side="right") == np.searchsorted(b, j, side="right")   # no bond is split


class _OracleDhp:
    """CPU stand-in for binding.Dhp in the gloo tests: the four calls ShardedMd makes, played in fp64 by the oracles
    (tests may use them).  What is under test is shard.py's ownership / mask / exchange logic, not this class."""

    def __init__(self, params, blob, n_models):
        self.params, self.blob, self.n_models = params, blob, n_models

    def dhp_md_create(self, inv_mass, bonds=None, bond_k=None, bond_r0=None):
        return {"w": np.asarray(inv_mass, np.float64)[:, None], "bonds": bonds, "k": bond_k, "r0": bond_r0, "Ff": None}

    def _fast(self, md, x, box):
        from oracle import md_oracle as M
        if md["bonds"] is None:
            return np.zeros_like(x)
        return M.bond_energy_forces(x, box, md["bonds"], md["k"], md["r0"])[1]

    def dhp_ani_energy_forces_partial(self, pos, box, species, weights, central, mol_offsets=None, E=None, F=None):
        import torch
        import oracle
        c = np.nonzero(central.numpy())[0].astype(np.int32)
        Ec, Fc, _ = oracle.energy_forces(pos.numpy(), species.numpy(), box, self.params, self.blob, self.n_models, centres=c)
        Eo, Fo = torch.tensor([Ec.sum()], dtype=torch.float64), torch.from_numpy(Fc.copy())
        if E is None or F is None:
            return Eo, Fo
        E.copy_(Eo); F.copy_(Fo)                            # the caller's buffers, as binding.Dhp fills them
        return E, F

    def dhp_md_open(self, md, pos, vel, box, F_slow, dt, n_inner, lo, hi):
        x, v, w = pos.numpy(), vel.numpy(), md["w"]
        if md["bonds"] is None:
            n_inner = 1
        d = dt / n_inner
        if md["Ff"] is None:
            md["Ff"] = self._fast(md, x, box)
        v[lo:hi] += 0.5 * dt * w[lo:hi] * F_slow.numpy()[lo:hi]
        for _ in range(n_inner):
            v[lo:hi] += 0.5 * d * w[lo:hi] * md["Ff"][lo:hi]
            x[lo:hi] += d * v[lo:hi]
            md["Ff"] = self._fast(md, x, box)          # own bonds only touch own atoms
            v[lo:hi] += 0.5 * d * w[lo:hi] * md["Ff"][lo:hi]

    def dhp_md_close(self, md, vel, F_slow, dt, n_inner, lo, hi):
        vel.numpy()[lo:hi] += 0.5 * dt * md["w"][lo:hi] * F_slow.numpy()[lo:hi]


def _md_worker(rank, port, results):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        params = W.default_params()
        blob = W.make_weights(1)
        s = W.make_system(1)
        mdi = W.md_inputs(s)
        bounds = shard.owner_bounds(s.n_atoms, WORLD, unit=3)
        pos = torch.from_numpy(s.pos.astype(np.float64))
        vel = torch.from_numpy(mdi.vel.astype(np.float64))
        # the exchange alone: reduce-scatter of partial forces and all-gather of owned rows
        ex = shard.Exchange(bounds, pos.device)
        part = torch.from_numpy(np.random.default_rng(rank).normal(size=(s.n_atoms, 3)))
        tot = torch.zeros_like(part)
        ex.reduce_scatter_forces(part, tot)
        want = sum(np.random.default_rng(r).normal(size=(s.n_atoms, 3)) for r in range(WORLD))
        assert np.allclose(tot.numpy()[ex.lo:ex.hi], want[ex.lo:ex.hi], atol=1e-14)
        assert np.all(tot.numpy()[:ex.lo] == 0) and np.all(tot.numpy()[ex.hi:] == 0)
        scr = torch.full((s.n_atoms, 3), float(rank) + 1.0, dtype=torch.float64)
        ex.all_gather_positions(scr)
        for r in range(WORLD):
            assert np.all(scr.numpy()[bounds[r]:bounds[r + 1]] == r + 1.0)
        # two outer steps of the sharded driver (2 inner steps, O-H bonds, slab masks refreshed every step)
        drv = shard.ShardedMd(_OracleDhp(params, blob, 1), blob, torch.from_numpy(s.species), s.box, bounds,
                              mdi.inv_mass, mdi.bonds, mdi.bond_k, mdi.bond_r0, mask_every=1, dtype=torch.float64)
        E = drv.run(pos, vel, 0.5, 2, 2)
        own = vel.numpy()[ex.lo:ex.hi].copy()
        allv = [torch.zeros_like(vel) for _ in range(WORLD)]
        dist.all_gather(allv, vel)
        if rank == 0:
            v = np.concatenate([allv[r].numpy()[bounds[r]:bounds[r + 1]] for r in range(WORLD)])
            results.put((pos.numpy().copy(), v, float(E.item())))
        del own
    finally:
        dist.destroy_process_group()


def test_world2_gloo_sharded_md_steps_equal_the_single_process_oracle_trajectory():
    import torch.multiprocessing as mp
    import oracle
    from oracle import md_oracle as M
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_md_worker, args=(r, port, q)) for r in range(WORLD)]
    for p in procs:
        p.start()
    x_sh, v_sh, E_sh = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    params = W.default_params()
    blob = W.make_weights(1)
    s = W.make_system(1)
    mdi = W.md_inputs(s)

    def slow(x):
        Ea, F, _ = oracle.energy_forces(x, s.species, s.box, params, blob, 1)
        return Ea.sum(), F

    def fast(x):
        return M.bond_energy_forces(x, s.box, mdi.bonds, mdi.bond_k, mdi.bond_r0)

    x, v, (E_s, _, _) = M.respa_run(s.pos, mdi.vel, mdi.inv_mass, slow, fast, 0.5, 2, 2)
    assert np.max(np.abs(x_sh - x)) <= 1e-11 and np.max(np.abs(v_sh - v)) <= 1e-11
    assert abs(E_sh - E_s) <= 1e-9
