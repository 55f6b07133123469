"""Verlet-skin reuse of the neighbour list (include/dhp.h: dhp_set_skin; "atomic positions do not move
much between two time-steps").  The list of EVERY call must still be the canonical one, bit for bit, whether the call
rebuilt the cell grid or filtered the candidate list of an earlier build; energies and forces keep their tolerances."""
import numpy as np
import pytest

import oracle
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


SYSTEMS = {
    "water96": lambda: W.make_system(1),                                   # 2 cells per edge (per-pair minimum image)
    "ligand50": lambda: W.make_system(2),                                  # open boundary
    "mix1500": lambda: W.small_periodic_mix(1500, 24.8, seed=5, n_models=1),
    "replicas16": lambda: W.replicas_1024x30(n_mol=16),                    # one "cell" per molecule
}


def lists_equal(d, q, s, params):
    rp, col, rpa, cola = d.dhp_nlist_export()
    rpo, colo = oracle.pairs(q, s.box, params.rcr, s.mol_offsets)
    ok = np.array_equal(rp.cpu().numpy(), rpo) and np.array_equal(col.cpu().numpy(), colo)
    rpo, colo = oracle.pairs(q, s.box, params.rca, s.mol_offsets)
    return ok and np.array_equal(rpa.cpu().numpy(), rpo) and np.array_equal(cola.cpu().numpy(), colo)


@pytest.mark.parametrize("name", list(SYSTEMS))
def test_lists_stay_bit_exact_under_reuse_and_rebuild_when_needed(torch, B, params, name):
    s = SYSTEMS[name]()
    d = B.Dhp(s.n_atoms, max_mols=max(s.n_mol, 0), params=params)
    d.dhp_set_skin(1.0)
    _, sp, mol = B.to_device(s)
    rng = np.random.default_rng(11)
    q = s.pos.copy()
    drift = np.zeros_like(q)
    for it in range(6):
        d.dhp_nlist_build(torch.from_numpy(q).cuda(), s.box, sp, mol)
        assert d.dhp_status() == 0
        assert lists_equal(d, q, s, params), f"iteration {it}"
        assert d.dhp_nlist_rebuild_count() == 1                         # every step stayed within skin / 2 = 0.5 A
        step = rng.normal(0.0, 0.03, q.shape)
        drift += step
        assert np.sqrt((drift ** 2).sum(1)).max() < 0.45
        q = (s.pos.astype(np.float64) + drift).astype(np.float32)
    # one atom jumps by more than skin / 2: the device-side check must force a full build
    q[3] += np.array([0.4, 0.4, 0.0], np.float32)
    d.dhp_nlist_build(torch.from_numpy(q).cuda(), s.box, sp, mol)
    assert lists_equal(d, q, s, params)
    assert d.dhp_nlist_rebuild_count() == 2
    if s.box is not None:                                                 # re-wrapping by a box vector looks like a big move
        q[5] += np.array([s.box[0], 0, 0], np.float32)
        d.dhp_nlist_build(torch.from_numpy(q).cuda(), s.box, sp, mol)
        assert lists_equal(d, q, s, params) and d.dhp_nlist_rebuild_count() == 3
    # a species change invalidates the candidate list as well
    n0 = d.dhp_nlist_rebuild_count()
    sp2 = sp.clone()
    sp2[0] = (int(sp2[0]) + 1) % 7
    d.dhp_nlist_build(torch.from_numpy(q).cuda(), s.box, sp2, mol)
    assert d.dhp_nlist_rebuild_count() == n0 + 1
    # skin off again: plain rebuilds, counter gone
    d.dhp_set_skin(0.0)
    d.dhp_nlist_build(torch.from_numpy(q).cuda(), s.box, sp, mol)
    assert lists_equal(d, q, s, params) and d.dhp_nlist_rebuild_count() == 0
    d.close()


@pytest.mark.parametrize("name", ["water96", "mix1500", "replicas16"])
@pytest.mark.parametrize("mode", [1, 2])
def test_energy_forces_on_a_reused_list(torch, B, params, name, mode):
    s = SYSTEMS[name]()
    blob = W.make_weights(s.n_models)
    d = B.Dhp(s.n_atoms, max_mols=max(s.n_mol, 0), params=params)
    d.dhp_set_mlp_mode(mode)
    d.dhp_set_skin(0.8)
    w = d.dhp_weights_load(blob, s.n_models)
    pos, sp, mol = B.to_device(s)
    d.dhp_ani_energy_forces(pos, s.box, sp, w, mol)                        # full build
    rng = np.random.default_rng(2)
    q = (s.pos + rng.normal(0.0, 0.08, s.pos.shape)).astype(np.float32)    # well inside skin / 2
    E, F = d.dhp_ani_energy_forces(torch.from_numpy(q).cuda(), s.box, sp, w, mol)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0 and d.dhp_nlist_rebuild_count() == 1
    s2 = W.System(s.name, q, s.species, s.box, s.mol_offsets, s.n_models)
    Eo, Fo = oracle.total_energy_forces(s2, params, blob)
    per = s.n_atoms if s.mol_offsets is None else np.diff(s.mol_offsets)
    assert np.max(np.abs(E.cpu().numpy() - Eo) / per) <= E_TOL_PER_ATOM
    assert np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
    # masked (partial) calls do not share a candidate list with unmasked ones
    mask = torch.ones(s.n_atoms, dtype=torch.uint8, device="cuda")
    mask[::2] = 0
    E2, F2 = d.dhp_ani_energy_forces_partial(torch.from_numpy(q).cuda(), s.box, sp, w, mask, mol)
    torch.cuda.synchronize()
    assert d.dhp_nlist_rebuild_count() == 2
    centres = np.nonzero(mask.cpu().numpy())[0].astype(np.int32)
    Ea, Fc, _ = oracle.energy_forces(q, s.species, s.box, params, blob, s.n_models, centres=centres, mol_offsets=s.mol_offsets)
    assert abs(E2.sum().item() - Ea.sum()) / len(centres) <= E_TOL_PER_ATOM and np.max(np.abs(F2.cpu().numpy() - Fc)) <= F_TOL
    d.close()


def test_reuse_at_full_size(torch, B, params):
    """configs[2] (23 558 atoms): candidate filtering at a size that spans many cells and row tiles."""
    s = W.make_system(3)
    d = B.Dhp(s.n_atoms, params=params)
    d.dhp_set_skin(1.0)
    _, sp, mol = B.to_device(s)
    d.dhp_nlist_build(torch.from_numpy(s.pos).cuda(), s.box, sp, mol)
    q = W.jitter(s, 0.05, 9)
    d.dhp_nlist_build(torch.from_numpy(q).cuda(), s.box, sp, mol)
    assert d.dhp_status() == 0 and d.dhp_nlist_rebuild_count() == 1
    assert lists_equal(d, q, s, params)
    d.close()
