"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element.

Tolerances (BASELINE.json north_star; derivations in DESIGN.md §Tolerances):
  pair lists  bit-exact (canonical CSR);
  energy      |E_gpu - E_oracle| / N <= 1e-6 Hartree per atom (per molecule for batched replicas);
  forces      max |dF| <= 5e-5 Hartree/Å;
  AEV rows    |dG| <= 2e-5 absolute (fp32 evaluation of O(1..10) sums; intermediate, not a north_star bar);
  dE/dG rows  |dg| <= 2e-5 absolute.
"""
import numpy as np
import pytest

import oracle
from paper_2207_14276_b200 import workloads as W

pytestmark = pytest.mark.gpu

E_TOL_PER_ATOM = 1e-6
F_TOL = 5e-5
AEV_TOL = 2e-5
GRAD_TOL = 2e-5


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2207_14276_b200 import binding
    return binding


@pytest.fixture(scope="module")
def blob8():
    return W.make_weights(8)


def make_ctx(B, system, params, extra_atoms=0):
    return B.Dhp(system.n_atoms + extra_atoms, max_mols=max(system.n_mol, 0), params=params)


def csr_equal(rp_g, col_g, rp_o, col_o):
    rp_g = rp_g.cpu().numpy().astype(np.int64)
    col_g = col_g.cpu().numpy()
    return np.array_equal(rp_g, rp_o) and np.array_equal(col_g, col_o)


SYSTEMS = {
    "water96": lambda: W.make_system(1),
    "ligand50": lambda: W.make_system(2),
    "mix600": lambda: W.small_periodic_mix(600, 18.3, seed=77, n_models=2),
    "mix1500": lambda: W.small_periodic_mix(1500, 24.8, seed=5, n_models=1),
    "replicas16": lambda: W.replicas_1024x30(n_mol=16),
}


# ------------------------------------------------------------------------------------------- a1
@pytest.mark.parametrize("name", list(SYSTEMS))
def test_pair_lists_bit_exact_small(torch, B, params, name):
    s = SYSTEMS[name]()
    d = make_ctx(B, s, params)
    pos, sp, mol = B.to_device(s)
    d.dhp_nlist_build(pos, s.box, sp, mol)
    assert d.dhp_status() == 0
    rp, col, rpa, cola = d.dhp_nlist_export()
    rpo, colo = oracle.pairs(s.pos, s.box, params.rcr, s.mol_offsets)
    assert csr_equal(rp, col, rpo, colo)
    rpo, colo = oracle.pairs(s.pos, s.box, params.rca, s.mol_offsets)
    assert csr_equal(rpa, cola, rpo, colo)
    d.close()


@pytest.mark.parametrize("name", ["water96", "ligand50", "replicas16"])
def test_small_systems_through_the_general_path(torch, B, params, blob8, name, monkeypatch):
    """Systems of <= 320 atoms normally take the single-block list build; DHP_NO_SMALL_PATH=1 sends them through the
    cell-list kernels instead, which keeps those kernels' small-box branches under test: two cells per periodic edge with
    the per-pair minimum image (water96), the bounding-box grid of open boundaries (ligand50), one cell per molecule
    (replicas16).  Lists bit-exact, energies and forces inside the bars, on both paths."""
    monkeypatch.setenv("DHP_NO_SMALL_PATH", "1")
    s = SYSTEMS[name]()
    d = make_ctx(B, s, params)
    pos, sp, mol = B.to_device(s)
    d.dhp_nlist_build(pos, s.box, sp, mol)
    assert d.dhp_status() == 0
    rp, col, rpa, cola = d.dhp_nlist_export()
    rpo, colo = oracle.pairs(s.pos, s.box, params.rcr, s.mol_offsets)
    assert csr_equal(rp, col, rpo, colo)
    rpo, colo = oracle.pairs(s.pos, s.box, params.rca, s.mol_offsets)
    assert csr_equal(rpa, cola, rpo, colo)
    d.close()
    d, E, F = run_gpu(B, torch, s, params, blob8)              # AUTO: tensor path on B200
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: s.n_models * 7 * W.PARAMS_PER_NET])
    per = s.n_atoms if s.mol_offsets is None else np.diff(s.mol_offsets)
    assert np.max(np.abs(E - Eo) / per) <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


@pytest.mark.parametrize("cfg", [3, 5, 4])
def test_pair_lists_bit_exact_full_size(torch, B, params, cfg):
    s = W.make_system(cfg)
    d = make_ctx(B, s, params)
    pos, sp, mol = B.to_device(s)
    d.dhp_nlist_build(pos, s.box, sp, mol)
    assert d.dhp_status() == 0
    rp, col, rpa, cola = d.dhp_nlist_export()
    rpo, colo = oracle.pairs(s.pos, s.box, params.rcr, s.mol_offsets)
    assert csr_equal(rp, col, rpo, colo)
    rpo, colo = oracle.pairs(s.pos, s.box, params.rca, s.mol_offsets)
    assert csr_equal(rpa, cola, rpo, colo)
    d.close()


def test_pair_list_positions_outside_box_and_two_cells_per_edge(torch, B, params):
    """configs[0] has 2 cells per edge (Q19); shifting atoms by whole boxes must change nothing (Q3)."""
    s = W.make_system(1)
    q = s.pos.copy()
    q[::3] += s.box[0] * 2
    q[1::7, 1] -= s.box[1] * 3
    d = make_ctx(B, s, params)
    pos = torch.from_numpy(q).cuda()
    sp = torch.from_numpy(s.species).cuda()
    d.dhp_nlist_build(pos, s.box, sp)
    rp, col, _, _ = d.dhp_nlist_export()
    rpo, colo = oracle.pairs(q, s.box, params.rcr)
    assert csr_equal(rp, col, rpo, colo)
    d.close()


# ------------------------------------------------------------------------------------------- a2..a5
def run_gpu(B, torch, s, params, blob, mode=None):
    d = make_ctx(B, s, params)
    if mode is not None:
        d.dhp_set_mlp_mode(mode)
    w = d.dhp_weights_load(blob[: s.n_models * 7 * W.PARAMS_PER_NET], s.n_models)
    pos, sp, mol = B.to_device(s)
    E, F = d.dhp_ani_energy_forces(pos, s.box, sp, w, mol)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    return d, E.cpu().numpy(), F.cpu().numpy()


def mlp_modes(B):
    return [B.MLP_SIMT, B.MLP_TENSOR]


@pytest.mark.parametrize("name", ["water96", "ligand50", "mix600", "replicas16"])
@pytest.mark.parametrize("mode", [1, 2, 3])
def test_energy_forces_small(torch, B, params, blob8, name, mode):
    s = SYSTEMS[name]()
    probe = make_ctx(B, s, params)
    if mode >= B.MLP_TENSOR and not probe.dhp_tensor_path_available():
        probe.close()
        pytest.skip("tensor path not available in this build")
    probe.close()
    d, E, F = run_gpu(B, torch, s, params, blob8, mode)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: s.n_models * 7 * W.PARAMS_PER_NET])
    per = s.n_atoms if s.mol_offsets is None else np.diff(s.mol_offsets)
    assert np.max(np.abs(E - Eo) / per) <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    # intermediates: AEV rows, dE/dG rows, atomic energies
    G = d.dhp_debug_aev().cpu().numpy()
    Go = oracle.aev(s.pos, s.species, s.box, params, mol_offsets=s.mol_offsets)
    assert np.max(np.abs(G - Go)) <= AEV_TOL
    Ea, _, go = oracle.energy_forces(s.pos, s.species, s.box, params, blob8[: s.n_models * 7 * W.PARAMS_PER_NET],
                                     s.n_models, mol_offsets=s.mol_offsets, want_dEdG=True)
    # dE/dG is produced only for the 64-wide feature blocks that are non-zero somewhere in the atom's 128-row tile
    # (the others multiply identically-zero dG/dr and are skipped; the export reads them as 0)
    g = d.dhp_debug_grad().cpu().numpy()
    close = np.abs(g - go) <= GRAD_TOL
    assert np.all(close | ((g == 0) & (Go == 0)))
    assert np.all(close[Go != 0])
    ea = d.dhp_debug_atomic_energy().cpu().numpy()
    assert np.max(np.abs(ea - Ea)) <= 2e-5
    # properties
    assert np.abs(F.sum(0)).max() < 1e-3
    d.close()


def test_energy_forces_config3_full(torch, B, params, blob8):
    """23 558 atoms, 8 networks: every force component and the total energy against the oracle."""
    s = W.make_system(3)
    d, E, F = run_gpu(B, torch, s, params, blob8)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8)
    assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


def sampled_check(B, torch, s, params, blob, n_energy=256, n_force=24, seed=0):
    d, E, F = run_gpu(B, torch, s, params, blob)
    rng = np.random.default_rng(seed)
    ea = d.dhp_debug_atomic_energy().cpu().numpy()
    centres = rng.choice(s.n_atoms, n_energy, replace=False).astype(np.int32)
    Ea, _, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, s.n_models, centres=centres,
                                    mol_offsets=s.mol_offsets)
    assert np.max(np.abs(ea[centres] - Ea)) <= 2e-5
    # mean signed error of the sampled atomic energies bounds the per-atom error of the total
    assert abs(np.mean(ea[centres] - Ea)) <= E_TOL_PER_ATOM
    pos_d, sp_d, mol_d = B.to_device(s)
    d.dhp_nlist_build(pos_d, s.box, sp_d, mol_d)
    rpt, colt, _, _ = d.dhp_nlist_export()
    rp, col = rpt.cpu().numpy(), colt.cpu().numpy()
    atoms = rng.choice(s.n_atoms, n_force, replace=False)
    for a in atoms:
        cs = np.concatenate([[a], col[rp[a]:rp[a + 1]]]).astype(np.int32)
        _, Fa, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, s.n_models, centres=cs,
                                        mol_offsets=s.mol_offsets)
        assert np.max(np.abs(F[a] - Fa[a])) <= F_TOL
    assert np.abs(F.sum(0)).max() < 2e-2      # sum F = 0 up to fp32 accumulation over N atoms
    d.close()
    return E, F


def test_energy_forces_config4_sampled(torch, B, params, blob8):
    sampled_check(B, torch, W.make_system(4), params, blob8)


def test_energy_forces_config5_sampled_molecules(torch, B, params, blob8):
    s = W.make_system(5)
    d, E, F = run_gpu(B, torch, s, params, blob8)
    rng = np.random.default_rng(1)
    for m in rng.choice(1024, 24, replace=False):
        sl = slice(30 * m, 30 * m + 30)
        Em, Fm, _ = oracle.energy_forces(s.pos[sl], s.species[sl], None, params, blob8, 8)
        assert abs(E[m] - Em.sum()) / 30 <= E_TOL_PER_ATOM
        assert np.max(np.abs(F[sl] - Fm)) <= F_TOL
    d.close()


@pytest.mark.parametrize("name", ["water96", "mix600", "replicas16"])
@pytest.mark.parametrize("mode", [1, 2, 3])
def test_energy_only_call(torch, B, params, blob8, name, mode):
    """dhp_ani_energy (a1-a3 only; reweighting needs energies, not gradients) against the oracle and
    against the energy of the full call."""
    s = SYSTEMS[name]()
    blob = blob8[: s.n_models * 7 * W.PARAMS_PER_NET]
    d = make_ctx(B, s, params)
    d.dhp_set_mlp_mode(mode)
    w = d.dhp_weights_load(blob, s.n_models)
    pos, sp, mol = B.to_device(s)
    for _ in range(2):                                   # twice: the second call starts from the first one's barrier phases
        E = d.dhp_ani_energy(pos, s.box, sp, w, mol)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    Eo, _ = oracle.total_energy_forces(s, params, blob)
    per = s.n_atoms if s.mol_offsets is None else np.diff(s.mol_offsets)
    assert np.max(np.abs(E.cpu().numpy() - Eo) / per) <= E_TOL_PER_ATOM
    E2, F2 = d.dhp_ani_energy_forces(pos, s.box, sp, w, mol)   # a full call after an energy-only call still works
    torch.cuda.synchronize()
    _, Fo = oracle.total_energy_forces(s, params, blob)
    assert np.max(np.abs(E2.cpu().numpy() - Eo) / per) <= E_TOL_PER_ATOM
    assert np.max(np.abs(F2.cpu().numpy() - Fo)) <= F_TOL
    d.close()


@pytest.mark.parametrize("name", ["water96", "mix600"])
def test_mixed_precision_mode_error_is_bounded_and_documented(torch, B, params, blob8, name):
    """DHP_MLP_TENSOR_FP16 (one fp16 MMA per product; the paper's mixed-precision option) is an opt-in
    trade: measured on B200 |dE|/N = 4e-6 .. 1e-5 Hartree and max |dF| = 3e-4 .. 4e-4 Hartree/Å, i.e.
    5-10x outside the parity bars that every other mode meets.  The test pins that order of magnitude from both sides:
    the mode must stay usable (errors well below the force scale of 0.1 Hartree/Å) and must never be mistaken for a
    mode that meets the bar."""
    s = SYSTEMS[name]()
    probe = make_ctx(B, s, params)
    ok = probe.dhp_tensor_path_available()
    probe.close()
    if not ok:
        pytest.skip("tensor path not available in this build")
    d, E, F = run_gpu(B, torch, s, params, blob8, B.MLP_TENSOR_FP16)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: s.n_models * 7 * W.PARAMS_PER_NET])
    dE, dF = abs(E[0] - Eo[0]) / s.n_atoms, np.max(np.abs(F - Fo))
    assert dE <= 5e-5 and dF <= 2e-3
    assert dF > F_TOL                     # if this ever passes the bar, make it the default and delete this test
    d.close()


@pytest.mark.parametrize("name", ["water96", "mix600", "replicas16"])
def test_two_launch_g1_and_middle_kernels(torch, B, params, blob8, name, monkeypatch):
    """The default tensor path runs G1 inside the fused chain kernel (k_mlp_fused: h1 never becomes an HBM operand).
    DHP_TC_FUSE=0 keeps the earlier pair of launches (G1 = k_gemm_tc with the AEV planes in the tiled operand layout, then
    k_mlp_mid): same arithmetic, same bars - and the energy-only call on that path."""
    monkeypatch.setenv("DHP_TC_FUSE", "0")
    s = SYSTEMS[name]()
    probe = make_ctx(B, s, params)
    ok = probe.dhp_tensor_path_available()
    probe.close()
    if not ok:
        pytest.skip("tensor path not available in this build")
    d, E, F = run_gpu(B, torch, s, params, blob8, B.MLP_TENSOR)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: s.n_models * 7 * W.PARAMS_PER_NET])
    per = s.n_atoms if s.mol_offsets is None else np.diff(s.mol_offsets)
    assert np.max(np.abs(E - Eo) / per) <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


def test_host_entry_point_matches_device_entry_point(torch, B, params, blob8):
    s = SYSTEMS["mix600"]()
    d, E, F = run_gpu(B, torch, s, params, blob8)
    w = d.dhp_weights_load(blob8[: 2 * 7 * W.PARAMS_PER_NET], 2)
    Eh, Fh = d.dhp_ani_energy_forces_host(s.pos, s.box, s.species, w)
    assert abs(Eh[0] - E[0]) <= 1e-6 * s.n_atoms and np.max(np.abs(Fh - F)) <= 1e-5
    d.close()


# ------------------------------------------------------------------------------------------- edge cases
def test_empty_single_and_isolated(torch, B, params, blob8):
    d = B.Dhp(64, params=params)
    w = d.dhp_weights_load(blob8[: 7 * W.PARAMS_PER_NET], 1)
    # empty
    pos = torch.empty((0, 3), dtype=torch.float32, device="cuda")
    sp = torch.empty((0,), dtype=torch.int32, device="cuda")
    E, F = d.dhp_ani_energy_forces(pos, None, sp, w)
    torch.cuda.synchronize()
    assert E.item() == 0.0 and F.shape == (0, 3)
    # one atom, and two atoms farther apart than Rcr: G = 0, E_i = NN(0), F = 0 (Q15)
    for p in ([[0.0, 0.0, 0.0]], [[0.0, 0.0, 0.0], [9.0, 0.0, 0.0]]):
        p = np.array(p, np.float32)
        s = np.array([1, 3][: len(p)], np.int32)
        E, F = d.dhp_ani_energy_forces(torch.from_numpy(p).cuda(), None, torch.from_numpy(s).cuda(), w)
        torch.cuda.synchronize()
        Eo, Fo, _ = oracle.energy_forces(p, s, None, params, blob8[: 7 * W.PARAMS_PER_NET], 1)
        assert abs(E.item() - Eo.sum()) <= 1e-6 * len(p)
        assert np.all(F.cpu().numpy() == 0.0) and np.all(Fo == 0.0)
    d.close()


def test_dense_cluster_more_than_32_angular_neighbours(torch, B, params, blob8):
    """> 32 atoms inside Rca of one centre exercises the multi-block rounds of the AEV kernels."""
    rng = np.random.default_rng(4)
    pts = [np.zeros(3)]
    while len(pts) < 60:
        c = rng.uniform(-3.0, 3.0, 3)
        if np.linalg.norm(c) <= 3.0 and min(np.linalg.norm(c - p) for p in pts) >= 0.8:
            pts.append(c)
    pos = np.array(pts, np.float32)
    sp = rng.integers(0, 7, len(pts)).astype(np.int32)
    s = W.System("dense", pos, sp, None, None, 1)
    rp, _ = oracle.pairs(pos, None, params.rca)
    assert np.diff(rp).max() > 40
    d, E, F = run_gpu(B, torch, s, params, blob8)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: 7 * W.PARAMS_PER_NET])
    # measured on B200 (round 2): |dE|/N = 1.4e-7, max|dF| = 3.9e-6 with max|F| = 0.98 and up to 59 angular neighbours:
    # the north_star bars hold here too
    assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


def test_error_codes(torch, B, params, blob8):
    d = B.Dhp(32, params=params)
    w = d.dhp_weights_load(blob8[: 7 * W.PARAMS_PER_NET], 1)
    pos = torch.zeros((4, 3), dtype=torch.float32, device="cuda")
    pos[:, 0] = torch.arange(4) * 1.1
    sp = torch.tensor([0, 1, 2, 3], dtype=torch.int32, device="cuda")
    with pytest.raises(B.DhpError, match="-3"):         # periodic edge < 2 Rcr
        d.dhp_ani_energy_forces(pos, np.array([10.0, 20.0, 20.0], np.float32), sp, w)
    with pytest.raises(B.DhpError, match="-2"):         # more atoms than the context holds
        big = torch.zeros((33, 3), dtype=torch.float32, device="cuda")
        d.dhp_ani_energy_forces(big, None, torch.zeros(33, dtype=torch.int32, device="cuda"), w)
    bad = torch.tensor([0, 1, 9, 3], dtype=torch.int32, device="cuda")
    d.dhp_ani_energy_forces(pos, None, bad, w)
    assert d.dhp_status() == -4                          # species outside 0..6, reported by the status word
    d.dhp_ani_energy_forces(pos, None, sp, w)
    assert d.dhp_status() == 0
    with pytest.raises(B.DhpError):                      # blob size must match n_models
        d.dhp_weights_load(blob8[: 7 * W.PARAMS_PER_NET], 2)
    d.close()


def test_rows_are_ordered_by_feature_block_class(torch, B, params, blob8):
    """Work accounting of the block-skipping GEMMs: a water-only system touches 3 of the 16 feature blocks in every
    tile (HH+HO, OO+HC, radial); in the mixed box rows are ordered by block class inside a species group, so the mean
    number of active blocks per tile stays well below the all-species count."""
    s = W.make_system(1)
    d, _, _ = run_gpu(B, torch, s, params, blob8)
    tiles, blocks = d.dhp_debug_tile_blocks()
    assert tiles == 4 and blocks == 12                     # 192 H -> 2 tiles, 96 O -> 1 tile + 1 padding tile (groups are
                                                           # aligned to tile PAIRS and a pair shares its mask)
    d.close()
    s = W.make_system(3)
    d, _, _ = run_gpu(B, torch, s, params, blob8)
    tiles, blocks = d.dhp_debug_tile_blocks()
    assert tiles >= 23558 // 128 and 3.0 <= blocks / tiles <= 8.0
    d.close()


def test_launch_counter_and_profile(torch, B, params, blob8):
    s = SYSTEMS["mix600"]()
    d = make_ctx(B, s, params)
    w = d.dhp_weights_load(blob8[: 2 * 7 * W.PARAMS_PER_NET], 2)
    pos, sp, mol = B.to_device(s)
    n0 = d.dhp_launch_count()
    d.dhp_profile_enable(True)
    d.dhp_profile_reset()
    for _ in range(3):
        d.dhp_ani_energy_forces(pos, s.box, sp, w)
    ms, calls = d.dhp_profile_read()
    assert calls == 3 and all(v > 0 for v in ms.values())
    assert d.dhp_launch_count() - n0 >= 3 * 10
    d.close()


def test_status_is_sticky_until_read(torch, B, params, blob8):
    """the per-call status word is cleared at the start of every hot call, so a fault at an intermediate call
    of an unsynchronised sequence used to be lost.  The library now folds every call's word into a sticky one that only
    dhp_status() clears."""
    d = B.Dhp(32, params=params)
    w = d.dhp_weights_load(blob8[: 7 * W.PARAMS_PER_NET], 1)
    pos = torch.zeros((4, 3), dtype=torch.float32, device="cuda")
    pos[:, 0] = torch.arange(4) * 1.1
    good = torch.tensor([0, 1, 2, 3], dtype=torch.int32, device="cuda")
    bad = torch.tensor([0, 1, 9, 3], dtype=torch.int32, device="cuda")
    d.dhp_ani_energy_forces(pos, None, good, w)
    d.dhp_ani_energy_forces(pos, None, bad, w)           # fault in the middle of a sequence ...
    d.dhp_ani_energy_forces(pos, None, good, w)
    d.dhp_ani_energy_forces(pos, None, good, w)
    assert d.dhp_status() == -4                           # ... is still reported
    assert d.dhp_status() == 0                            # and reading clears it
    with pytest.raises(B.DhpError):                       # the binding refuses buffers the C ABI would misread
        d.dhp_ani_energy_forces(pos, None, good.to(torch.int64), w)
    with pytest.raises(B.DhpError):
        d.dhp_ani_energy_forces(pos.double(), None, good, w)
    with pytest.raises(B.DhpError):
        d.dhp_ani_energy_forces(torch.zeros((4, 6), dtype=torch.float32, device="cuda")[:, ::2], None, good, w)
    d.close()


@pytest.mark.parametrize("skin", [0.0, 1.0])
def test_capacity_fault_in_the_middle_of_an_md_run_is_reported(torch, B, params, blob8, skin):
    """dhp_md_run enqueues n calls without a host sync.  Atoms of infinite mass (inv_mass = 0: ballistic
    motion) fly towards the origin; after a few outer steps every atom has more neighbours than a list row holds
    (192), the rows are truncated and the call flags CAPACITY - which must survive to the dhp_status() after the run,
    with and without list reuse (a truncated candidate list must also force the next call to rebuild)."""
    rng = np.random.default_rng(12)
    n = 420
    pts = np.empty((0, 3))
    while pts.shape[0] < n:                                            # ~0.1 atoms / Å^3 in a 10 Å sphere
        c = rng.uniform(-10, 10, 3)
        if np.linalg.norm(c) <= 10 and (pts.shape[0] == 0 or np.linalg.norm(pts - c, axis=1).min() >= 1.2):
            pts = np.concatenate([pts, c[None]])
    pos0 = pts.astype(np.float32)
    sp = rng.integers(0, 4, n).astype(np.int32)
    vel0 = (-0.16 * pts).astype(np.float32)                            # Å/fs, towards the origin
    d = B.Dhp(n, params=params)
    w = d.dhp_weights_load(blob8[: 7 * W.PARAMS_PER_NET], 1)
    if skin:
        d.dhp_set_skin(skin)
    md = d.dhp_md_create(np.zeros(n, np.float32))
    pos, vel = torch.from_numpy(pos0.copy()).cuda(), torch.from_numpy(vel0.copy()).cuda()
    spd = torch.from_numpy(sp).cuda()
    # ballistic: r(t) = r0 (1 - 0.16 t / fs).  2 steps: scale 0.84, ~95 neighbours per atom - no fault yet
    d.dhp_md_run(md, pos, vel, None, spd, w, 0.5, 1, 2)
    assert d.dhp_status() == 0                                         # and the sticky word stays clear
    d.dhp_md_run(md, pos, vel, None, spd, w, 0.5, 1, 5)                # scale 0.44: ~12 x the density, rows overflow
    # expand again so that the LAST calls of the sequence are clean: only the sticky word can know about the fault
    vel.mul_(-1.0)
    d.dhp_md_run(md, pos, vel, None, spd, w, 0.5, 1, 7)
    E_last, F_last = d.dhp_ani_energy_forces(pos, None, spd, w)
    torch.cuda.synchronize()
    assert d.dhp_status() == -2
    assert d.dhp_status() == 0
    # and the state after the fault is sound: the list of the final (dilute again) positions is the canonical one
    d.dhp_nlist_build(pos, None, spd)
    rp, col, _, _ = d.dhp_nlist_export()
    rpo, colo = oracle.pairs(pos.cpu().numpy(), None, params.rcr)
    assert csr_equal(rp, col, rpo, colo)
    assert d.dhp_status() == 0
    d.dhp_md_destroy(md)
    d.close()


@pytest.mark.parametrize("n_atoms", [300, 420])
def test_capacity_and_species_fault_in_the_same_call(torch, B, params, blob8, n_atoms):
    """a species fault must not hide a capacity fault of the same call (the library derives "the candidate list was
    truncated" from the word reading CAPACITY), and a fault raised by the LAST call is reported once, not on every read.
    A ball at ~12 x liquid density overflows every list row; one atom carries species 9.  Both list paths (<= 320 atoms: the
    three-launch path; above: cell list), with list reuse on."""
    rng = np.random.default_rng(31)
    pts = np.empty((0, 3))
    while pts.shape[0] < n_atoms:
        c = rng.uniform(-4.4, 4.4, 3)
        if np.linalg.norm(c) <= 4.4 and (pts.shape[0] == 0 or np.linalg.norm(pts - c, axis=1).min() >= 0.5):
            pts = np.concatenate([pts, c[None]])
    sp = rng.integers(0, 4, n_atoms).astype(np.int32)
    bad = sp.copy()
    bad[n_atoms // 2] = 9
    d = B.Dhp(n_atoms, params=params)
    d.dhp_set_skin(1.0)
    w = d.dhp_weights_load(blob8[: 7 * W.PARAMS_PER_NET], 1)
    pos = torch.from_numpy(pts.astype(np.float32)).cuda()
    d.dhp_ani_energy_forces(pos, None, torch.from_numpy(bad).cuda(), w)
    assert d.dhp_status() == -2                           # capacity, although the species fault is raised first (binning)
    assert d.dhp_status() == 0                            # read once
    d.dhp_ani_energy_forces(pos, None, torch.from_numpy(sp).cuda(), w)
    assert d.dhp_status() == -2                           # still too dense, species fine
    assert d.dhp_status() == 0
    # dilute again (x 2.3: liquid density): a clean call with the canonical list
    pos2 = (pos * 2.3).contiguous()
    spd = torch.from_numpy(sp).cuda()
    d.dhp_ani_energy_forces(pos2, None, spd, w)
    assert d.dhp_status() == 0
    d.dhp_nlist_build(pos2, None, spd)
    rp, col, _, _ = d.dhp_nlist_export()
    rpo, colo = oracle.pairs(pos2.cpu().numpy(), None, params.rcr)
    assert csr_equal(rp, col, rpo, colo)
    d.close()


@pytest.mark.parametrize("name", ["ligand50", "water96", "replicas8"])
def test_small_systems_replay_a_captured_graph(torch, B, params, blob8, name):
    """Small systems (the hybrid scheme's per-step call) are captured into a CUDA graph on the second
    call with a given argument set (the first only records the set and runs as a plain enqueue) and replayed afterwards.  The replays must give the oracle's answer for the CURRENT
    contents of the buffers (positions are rewritten in place between calls), count as replays, and a different buffer
    must not be served by a stale graph."""
    s = W.replicas_1024x30(n_mol=8) if name == "replicas8" else SYSTEMS[name]()     # 240 atoms in 8 molecules: still "small"
    blob = blob8[: s.n_models * 7 * W.PARAMS_PER_NET]
    d = make_ctx(B, s, params)
    w = d.dhp_weights_load(blob, s.n_models)
    pos, sp, mol = B.to_device(s)
    n_mol = max(1, s.n_mol)
    E = torch.empty(n_mol, dtype=torch.float64, device="cuda")
    F = torch.empty((s.n_atoms, 3), dtype=torch.float32, device="cuda")
    per = s.n_atoms if s.mol_offsets is None else np.diff(s.mol_offsets)
    rng = np.random.default_rng(3)
    q = s.pos.copy()
    r0 = d.dhp_graph_replays()
    for it in range(4):
        pos.copy_(torch.from_numpy(q).cuda())                 # same buffer, new contents
        d.dhp_ani_energy_forces(pos, s.box, sp, w, mol, E=E, F=F)
        torch.cuda.synchronize()
        assert d.dhp_status() == 0
        s2 = W.System(s.name, q, s.species, s.box, s.mol_offsets, s.n_models)
        Eo, Fo = oracle.total_energy_forces(s2, params, blob)
        assert np.max(np.abs(E.cpu().numpy() - Eo) / per) <= E_TOL_PER_ATOM
        assert np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
        q = (q.astype(np.float64) + rng.normal(0, 0.02, q.shape)).astype(np.float32)
    assert d.dhp_graph_replays() - r0 == 3                    # first call plain; the capture call is served by the new graph too
    l0 = d.dhp_launch_count()
    d.dhp_ani_energy_forces(pos, s.box, sp, w, mol, E=E, F=F)
    assert d.dhp_launch_count() - l0 >= 6                     # replayed kernels are counted
    # a different position buffer is a different graph, not a stale replay
    pos2 = torch.from_numpy(s.pos).cuda()
    E2, F2 = d.dhp_ani_energy_forces(pos2, s.box, sp, w, mol)
    torch.cuda.synchronize()
    Eo, Fo = oracle.total_energy_forces(s, params, blob)
    assert np.max(np.abs(E2.cpu().numpy() - Eo) / per) <= E_TOL_PER_ATOM and np.max(np.abs(F2.cpu().numpy() - Fo)) <= F_TOL
    # energy-only and masked calls go through the same mechanism
    Ee = d.dhp_ani_energy(pos2, s.box, sp, w, mol)
    Ee = d.dhp_ani_energy(pos2, s.box, sp, w, mol, E=Ee)
    torch.cuda.synchronize()
    assert np.max(np.abs(Ee.cpu().numpy() - Eo) / per) <= E_TOL_PER_ATOM
    d.close()


def test_graph_replay_of_a_large_system_and_its_switch_off_under_changing_arguments(torch, B, params, blob8):
    """Systems above the small-system limit are replayed too (the cell-list path's 17 kernels as one graph).  Replays must
    give the oracle's answer for the current buffer contents; a caller whose argument set changes every call (here: the box)
    makes the library fall back to plain enqueues by itself - results unchanged either way."""
    s = SYSTEMS["mix600"]()
    blob = blob8[: s.n_models * 7 * W.PARAMS_PER_NET]
    d = make_ctx(B, s, params)
    w = d.dhp_weights_load(blob, s.n_models)
    pos, sp, mol = B.to_device(s)
    E = torch.empty(1, dtype=torch.float64, device="cuda")
    F = torch.empty((s.n_atoms, 3), dtype=torch.float32, device="cuda")
    rng = np.random.default_rng(11)
    q = s.pos.copy()
    r0 = d.dhp_graph_replays()
    for it in range(3):
        pos.copy_(torch.from_numpy(q).cuda())
        d.dhp_ani_energy_forces(pos, s.box, sp, w, mol, E=E, F=F)
        torch.cuda.synchronize()
        assert d.dhp_status() == 0
        Eo, Fo = oracle.total_energy_forces(W.System(s.name, q, s.species, s.box, s.mol_offsets, s.n_models), params, blob)
        assert abs(E.item() - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM and np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
        q = (q.astype(np.float64) + rng.normal(0, 0.02, q.shape)).astype(np.float32)
    assert d.dhp_graph_replays() - r0 == 2                    # first call plain, second captures and replays
    # a new box on every call: no argument set is ever seen twice, so nothing is captured or replayed
    r1 = d.dhp_graph_replays()
    box = np.array(s.box, dtype=np.float64)
    for it in range(40):
        b = (box * (1.0 + 1e-4 * (it + 1))).astype(np.float32)
        d.dhp_ani_energy_forces(pos, b, sp, w, mol, E=E, F=F)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    assert d.dhp_graph_replays() - r1 == 0
    Eo, Fo = oracle.total_energy_forces(W.System(s.name, pos.cpu().numpy(), s.species, b, s.mol_offsets, s.n_models), params, blob)
    assert abs(E.item() - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM and np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
    d.close()


def test_graph_table_does_not_thrash_under_rotating_buffers(torch, B, params, blob8):
    """A caller that rotates more position buffers than the table has keys (8), or that gets fresh E / F buffers on every
    call, never sees the same argument set twice in the table: every call is a plain enqueue, no graph is built and thrown
    away.  Six rotating buffers fit: from the second round on every call is a replay.  Results are the oracle's either way."""
    s = SYSTEMS["ligand50"]()
    blob = blob8[: s.n_models * 7 * W.PARAMS_PER_NET]
    Eo, Fo = oracle.total_energy_forces(s, params, blob)
    d = make_ctx(B, s, params)
    w = d.dhp_weights_load(blob, s.n_models)
    _, sp, mol = B.to_device(s)
    E = torch.empty(1, dtype=torch.float64, device="cuda")
    F = torch.empty((s.n_atoms, 3), dtype=torch.float32, device="cuda")
    bufs = [torch.from_numpy(s.pos).cuda() for _ in range(10)]
    r0 = d.dhp_graph_replays()
    for it in range(30):
        d.dhp_ani_energy_forces(bufs[it % 10], s.box, sp, w, mol, E=E, F=F)
    assert d.dhp_graph_replays() - r0 == 0
    keep = []
    for it in range(12):                                      # new E / F every call (kept alive: no address comes back)
        keep.append(d.dhp_ani_energy_forces(bufs[0], s.box, sp, w, mol))
    assert d.dhp_graph_replays() - r0 == 0
    for it in range(18):
        d.dhp_ani_energy_forces(bufs[it % 6], s.box, sp, w, mol, E=E, F=F)
    torch.cuda.synchronize()
    assert d.dhp_graph_replays() - r0 == 12
    assert d.dhp_status() == 0
    assert abs(E.item() - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM and np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
    d.close()


def test_graph_replay_can_be_switched_off(torch, B, params, blob8, monkeypatch):
    monkeypatch.setenv("DHP_NO_GRAPH", "1")
    s = SYSTEMS["ligand50"]()
    d, E, F = run_gpu(B, torch, s, params, blob8)
    assert d.dhp_graph_replays() == 0
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: s.n_models * 7 * W.PARAMS_PER_NET])
    assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM and np.max(np.abs(F - Fo)) <= F_TOL
    d.close()
