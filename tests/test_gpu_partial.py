"""Partial evaluation over a subset of central atoms (include/dhp.h: dhp_ani_energy_forces_partial) — the device-side
building block of the multi-GPU decomposition.  Each partial result is
checked against the oracle restricted to the same centres, and the partial results of a partition must add up to
the full result."""
import numpy as np
import pytest

import oracle
from paper_2207_14276_b200 import shard
from paper_2207_14276_b200 import workloads as W

pytestmark = pytest.mark.gpu

E_TOL_PER_ATOM = 1e-6
F_TOL = 5e-5


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2207_14276_b200 import binding
    return binding


@pytest.mark.parametrize("name,world", [("water96", 2), ("mix600", 3), ("ligand50", 2)])
@pytest.mark.parametrize("mode", [1, 2])
def test_slab_partials_match_oracle_and_sum_to_full(torch, B, params, name, world, mode):
    s = {"water96": lambda: W.make_system(1), "ligand50": lambda: W.make_system(2),
         "mix600": lambda: W.small_periodic_mix(600, 18.3, seed=77, n_models=2)}[name]()
    blob = W.make_weights(s.n_models)
    d = B.Dhp(s.n_atoms, params=params)
    d.dhp_set_mlp_mode(mode)
    w = d.dhp_weights_load(blob, s.n_models)
    pos, sp, _ = B.to_device(s)
    Esum, Fsum, seen = 0.0, np.zeros((s.n_atoms, 3)), np.zeros(s.n_atoms, dtype=int)
    for r in range(world):
        mask = shard.slab_mask_device(pos, s.box, world, r)
        centres = shard.slab_centres(s.pos, s.box, world, r)
        assert np.array_equal(np.nonzero(mask.cpu().numpy())[0], centres)       # device rule == host rule
        E, F = d.dhp_ani_energy_forces_partial(pos, s.box, sp, w, mask)
        torch.cuda.synchronize()
        assert d.dhp_status() == 0
        Ea, Fo, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, s.n_models, centres=centres)
        assert abs(E.item() - Ea.sum()) / len(centres) <= E_TOL_PER_ATOM
        assert np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
        ea = d.dhp_debug_atomic_energy().cpu().numpy()
        assert np.all(ea[np.setdiff1d(np.arange(s.n_atoms), centres)] == 0.0)  # non-central atoms have no row
        Esum += E.item()
        Fsum += F.cpu().numpy()
        seen[centres] += 1
    assert np.all(seen == 1)
    Eo, Fo = oracle.total_energy_forces(s, params, blob)
    assert abs(Esum - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(Fsum - Fo)) <= F_TOL
    # NULL mask = the full call
    E, F = d.dhp_ani_energy_forces_partial(pos, s.box, sp, w, None)
    torch.cuda.synchronize()
    assert abs(E.item() - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM and np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
    d.close()


def test_empty_and_single_centre_masks(torch, B, params):
    s = W.small_periodic_mix(600, 18.3, seed=77, n_models=1)
    blob = W.make_weights(1)
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(blob, 1)
    pos, sp, _ = B.to_device(s)
    mask = torch.zeros(s.n_atoms, dtype=torch.uint8, device="cuda")
    E, F = d.dhp_ani_energy_forces_partial(pos, s.box, sp, w, mask)       # no centre at all: E = 0, F = 0
    torch.cuda.synchronize()
    assert d.dhp_status() == 0 and E.item() == 0.0 and np.all(F.cpu().numpy() == 0.0)
    mask[17] = 1                                                           # one centre: its own local environment
    E, F = d.dhp_ani_energy_forces_partial(pos, s.box, sp, w, mask)
    torch.cuda.synchronize()
    Ea, Fo, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 1, centres=np.array([17], np.int32))
    assert abs(E.item() - Ea[0]) <= E_TOL_PER_ATOM and np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
    rp, _ = oracle.pairs(s.pos, s.box, params.rcr)
    touched = np.nonzero(np.abs(F.cpu().numpy()).sum(1))[0]
    assert len(touched) <= rp[18] - rp[17] + 1                             # only atom 17 and its neighbours feel a force
    d.close()


def test_partial_with_molecules(torch, B, params):
    """Batched replicas: a mask that selects whole molecules gives exactly those molecules' energies and forces."""
    s = W.replicas_1024x30(n_mol=12)
    blob = W.make_weights(8)
    d = B.Dhp(s.n_atoms, max_mols=12, params=params)
    w = d.dhp_weights_load(blob, 8)
    pos, sp, mol = B.to_device(s)
    mask = torch.zeros(s.n_atoms, dtype=torch.uint8, device="cuda")
    mask[30 * 3: 30 * 7] = 1
    E, F = d.dhp_ani_energy_forces_partial(pos, None, sp, w, mask, mol)
    torch.cuda.synchronize()
    E, F = E.cpu().numpy(), F.cpu().numpy()
    Eo, Fo = oracle.total_energy_forces(s, params, blob)
    sel = np.zeros(12, bool)
    sel[3:7] = True
    assert np.all(E[~sel] == 0.0) and np.max(np.abs(E[sel] - Eo[sel])) / 30 <= E_TOL_PER_ATOM
    assert np.all(F[:90] == 0.0) and np.all(F[210:] == 0.0) and np.max(np.abs(F[90:210] - Fo[90:210])) <= F_TOL
    d.close()


def test_sharded_call_on_a_one_rank_nccl_group(torch, B, params):
    """The NCCL plumbing of shard.ani_energy_forces_sharded on the one GPU there is: world_size 1 (no peer to wait on)."""
    import socket
    import torch.distributed as dist
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1)
    try:
        s = W.make_system(1)
        blob = W.make_weights(1)
        d = B.Dhp(s.n_atoms, params=params)
        w = d.dhp_weights_load(blob, 1)
        pos, sp, _ = B.to_device(s)
        mask = shard.slab_mask_device(pos, s.box, dist.get_world_size(), dist.get_rank())
        assert int(mask.sum()) == s.n_atoms
        E, F = shard.ani_energy_forces_sharded(d, pos, s.box, sp, w, mask)
        dist.all_reduce(F)                                   # world 1: identity, but it runs through NCCL on the stream
        torch.cuda.synchronize()
        Eo, Fo = oracle.total_energy_forces(s, params, blob)
        assert abs(E.item() - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM and np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
        d.close()
    finally:
        dist.destroy_process_group()


def test_config4_slab_partial_call_at_full_size(torch, B, params):
    """The launch configuration a rank of an 8-GPU run executes: configs[3], 98 000 atoms, 8 networks, with
    the central-atom mask of ONE of 8 spatial slabs - k_pairs skips 7/8 of the cells, the AEV / MLP kernels walk the row
    tiles of a ragged 12 250-atom subset.  Slabs 0 and 5: E, every force component and the lists of the central atoms
    against the oracle restricted to the same centres.  Then the same call as shard.ShardedMd issues it on every step:
    list reuse on, positions rewritten in place, mask kept - third call (reused list, replayed graph) against the oracle."""
    s = W.make_system(4)
    blob = W.make_weights(8)
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(blob, 8)
    pos, sp, _ = B.to_device(s)
    d.dhp_nlist_build(pos, s.box, sp)                          # the list handle is a token of the context (include/dhp.h)
    rows = {rc: oracle.pairs(s.pos, s.box, rc) for rc in (params.rcr, params.rca)}
    E = torch.empty(1, dtype=torch.float64, device="cuda")
    F = torch.empty((s.n_atoms, 3), dtype=torch.float32, device="cuda")
    for r in (0, 5):
        mask = shard.slab_mask_device(pos, s.box, 8, r)
        centres = shard.slab_centres(s.pos, s.box, 8, r)
        assert len(centres) == 12250 and np.array_equal(np.nonzero(mask.cpu().numpy())[0], centres)
        d.dhp_ani_energy_forces_partial(pos, s.box, sp, w, mask, E=E, F=F)
        torch.cuda.synchronize()
        assert d.dhp_status() == 0
        Ea, Fo, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 8, centres=centres)
        assert abs(E.item() - Ea.sum()) / len(centres) <= E_TOL_PER_ATOM
        assert np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
        # lists of the call: the canonical rows for the central atoms, nothing for the others
        rp, col, rpa, cola = (a.cpu().numpy() for a in d.dhp_nlist_export())
        central = np.zeros(s.n_atoms, bool)
        central[centres] = True
        for got_rp, got_col, rc in ((rp, col, params.rcr), (rpa, cola, params.rca)):
            rpo, colo = rows[rc]
            cnt = np.where(central, np.diff(rpo), 0)
            assert np.array_equal(np.diff(got_rp.astype(np.int64)), cnt)
            keep = np.repeat(central, np.diff(rpo))
            assert np.array_equal(got_col, colo[keep])
    # list reuse + graph replay + mask together (slab 5's mask, as between two mask refreshes of ShardedMd)
    d.dhp_set_skin(1.0)
    r0, g0 = d.dhp_nlist_rebuild_count(), d.dhp_graph_replays()
    for k in range(3):
        q = W.jitter(s, 0.01, 900 + k)
        pos.copy_(torch.from_numpy(q).cuda())
        d.dhp_ani_energy_forces_partial(pos, s.box, sp, w, mask, E=E, F=F)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    assert d.dhp_nlist_rebuild_count() - r0 == 1 and d.dhp_graph_replays() - g0 >= 1
    Ea, Fo, _ = oracle.energy_forces(q, s.species, s.box, params, blob, 8, centres=centres)
    assert abs(E.item() - Ea.sum()) / len(centres) <= E_TOL_PER_ATOM
    assert np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
    d.close()
