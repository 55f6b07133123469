"""Full-size and edge-case parity of the CUDA path (through the C ABI) against the fp64 oracle.

Round-2 additions ("What's weak" #2): the headline configs[3] and configs[4] compared over EVERY atom /
molecule, AEV and dE/dG rows at a size where the class-ordered rows and the dynamic tile scheduler are in play, and the
method's edge cases: an orthorhombic box with three different edges, a pair at exactly R = Rc (Eq. 3, PAPER.md L70:
"R <= Rc", zero contribution), near-collinear triplets (SURVEY.md §7 hard part 2), ensembles of 3 and 5 networks.
Bars are north_star's: lists bit-exact, |dE|/N <= 1e-6 Hartree, max |dF| <= 5e-5 Hartree/Å.
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


def run_gpu(B, torch, s, params, blob, mode=None, max_atoms=None):
    d = B.Dhp(max_atoms or s.n_atoms, max_mols=max(s.n_mol, 0), params=params)
    if mode is not None:
        d.dhp_set_mlp_mode(mode)
    w = d.dhp_weights_load(blob[: s.n_models * 7 * W.PARAMS_PER_NET], s.n_models)
    pos, sp, mol = B.to_device(s)
    E, F = d.dhp_ani_energy_forces(pos, s.box, sp, w, mol)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    return d, E.cpu().numpy(), F.cpu().numpy()


def lists_equal(B, d, s, params):
    pos, sp, mol = B.to_device(s)
    d.dhp_nlist_build(pos, s.box, sp, mol)
    assert d.dhp_status() == 0
    rp, col, rpa, cola = d.dhp_nlist_export()
    for got_rp, got_col, rc in ((rp, col, params.rcr), (rpa, cola, params.rca)):
        rpo, colo = oracle.pairs(s.pos, s.box, rc, s.mol_offsets)
        assert np.array_equal(got_rp.cpu().numpy().astype(np.int64), rpo)
        assert np.array_equal(got_col.cpu().numpy(), colo)


# ------------------------------------------------------------------------------------------- full size
def test_config4_full_energy_and_every_force(torch, B, params, blob8):
    """configs[3], the headline workload: 98 000 atoms, 8 networks, in the launch configuration bench.py times.
    The total energy through k_energy_reduce and all 294 000 force components against the oracle (about half a
    minute of oracle on 16 cores)."""
    s = W.make_system(4)
    d, E, F = run_gpu(B, torch, s, params, blob8)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8)
    assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    ea = d.dhp_debug_atomic_energy().cpu().numpy()
    Ea, _, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob8, 8,
                                    centres=np.arange(0, s.n_atoms, 97, dtype=np.int32))
    assert np.max(np.abs(ea[::97] - Ea)) <= 2e-5
    d.close()


def test_config5_full_all_molecules(torch, B, params, blob8):
    """configs[4]: all 1 024 molecules, per-molecule energies and every force."""
    s = W.make_system(5)
    d, E, F = run_gpu(B, torch, s, params, blob8)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8)
    assert E.shape == (1024,)
    assert np.max(np.abs(E - Eo)) / 30 <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


def test_config3_aev_and_grad_rows_elementwise(torch, B, params, blob8):
    """a2 and a4 in isolation at a size with ~190 row tiles, class-ordered rows and the dynamic tile scheduler:
    every AEV entry and every dE/dG entry of configs[2] (23 558 atoms) against the oracle."""
    s = W.make_system(3)
    d, E, F = run_gpu(B, torch, s, params, blob8)
    G = d.dhp_debug_aev().cpu().numpy()
    g = d.dhp_debug_grad().cpu().numpy()
    Ea, Fo, go = oracle.energy_forces(s.pos, s.species, s.box, params, blob8, 8, want_dEdG=True)
    Go = oracle.aev(s.pos, s.species, s.box, params)
    assert np.max(np.abs(G - Go)) <= AEV_TOL
    close = np.abs(g - go) <= GRAD_TOL
    # dE/dG exists only for the feature blocks that are active in the atom's row tile; the rest multiply dG/dr = 0
    assert np.all(close | ((g == 0) & (Go == 0)))
    assert np.all(close[Go != 0])
    ea = d.dhp_debug_atomic_energy().cpu().numpy()
    assert np.max(np.abs(ea - Ea)) <= 2e-5
    assert abs(E[0] - Ea.sum()) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


# ------------------------------------------------------------------------------------------- edge cases
@pytest.mark.parametrize("n,box", [(900, (17.3, 21.9, 24.6)), (300, (10.3, 13.0, 22.5))])
def test_orthorhombic_box_three_different_edges(torch, B, params, blob8, n, box):
    """include/dhp.h promises orthorhombic cells: lists bit-exact and E/F inside the bars with three different edges
    (the second box has 2 cells along two axes and 4 along the third; 300 atoms take the single-block path)."""
    s = W.small_periodic_ortho(n, box, seed=78 + n)
    d, E, F = run_gpu(B, torch, s, params, blob8)
    lists_equal(B, d, s, params)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: s.n_models * 7 * W.PARAMS_PER_NET])
    assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


def _tie_system(periodic, extra):
    """Atom 1 sits at EXACTLY R = Rcr from atom 0 and atom 2 at exactly Rca (fp32 inputs, axis-aligned so the fp64
    predicate R^2 <= rc^2 is an exact tie); atoms 3 / 4 one ulp beyond.  `extra` random atoms fill the box so that the
    general (cell list) path runs when asked to."""
    rcr, rca = np.float32(5.1), np.float32(3.5)
    base = np.array([[1.0, 1.0, 1.0]], np.float32)
    pts = [base[0],
           base[0] + np.array([rcr, 0, 0], np.float32),
           base[0] + np.array([0, rca, 0], np.float32),
           base[0] + np.array([0, 0, np.nextafter(rcr, np.float32(9))], np.float32),
           base[0] + np.array([0, -np.nextafter(rca, np.float32(9)), 0], np.float32)]
    # the sums above round in fp32; rebuild the partners so that the DIFFERENCE is exactly rc
    pts[1] = np.array([np.float32(1.0) + rcr, 1.0, 1.0], np.float32)
    pts[2] = np.array([1.0, np.float32(1.0) + rca, 1.0], np.float32)
    rng = np.random.default_rng(5)
    L = 24.0
    allp = list(pts)
    while len(allp) < 5 + extra:
        c = rng.uniform(0, L, 3).astype(np.float32)
        if min(np.linalg.norm(c.astype(np.float64) - p.astype(np.float64)) for p in allp) >= 1.0:
            allp.append(c)
    pos = np.array(allp, np.float32)
    sp = rng.integers(0, 7, len(allp)).astype(np.int32)
    box = np.array([L, L, L], np.float32) if periodic else None
    return W.System("tie", pos, sp, box, None, 1)


@pytest.mark.parametrize("periodic,extra,general", [(False, 0, False), (False, 40, True), (True, 700, False)])
def test_pair_at_exactly_the_cutoff(torch, B, params, blob8, periodic, extra, general, monkeypatch):
    """Eq. 3 is "R <= Rc": a pair at exactly Rc IS in the list (Q2) and contributes exactly 0.  The
    fp32-prefilter -> fp64-decision path of k_pairs / k_refilter / k_nlist_small exists for this tie."""
    if general:
        monkeypatch.setenv("DHP_NO_SMALL_PATH", "1")
    s = _tie_system(periodic, extra)
    x = s.pos.astype(np.float64)
    # the construction really is a tie (and one ulp beyond is not)
    assert (x[1, 0] - x[0, 0]) == float(np.float32(5.1)) and (x[2, 1] - x[0, 1]) == float(np.float32(3.5))
    rpo, colo = oracle.pairs(s.pos, s.box, params.rcr)
    assert 1 in colo[rpo[0]:rpo[1]] and 3 not in colo[rpo[0]:rpo[1]]
    rpa, cola = oracle.pairs(s.pos, s.box, params.rca)
    assert 2 in cola[rpa[0]:rpa[1]] and 4 not in cola[rpa[0]:rpa[1]]
    d, E, F = run_gpu(B, torch, s, params, blob8)
    lists_equal(B, d, s, params)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: 7 * W.PARAMS_PER_NET])
    assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


@pytest.mark.parametrize("theta", [1e-3, 5e-4, 2.5e-4])
def test_near_collinear_triplet(torch, B, params, blob8, theta):
    """SURVEY.md §7 hard part 2: for theta <~ 1e-3 rad sqrt(1 - cos^2) loses the angular gradient in fp32; the kernels
    use |r_ij x r_ik| (Q7).  A centre with two neighbours `theta` apart (and a few bystanders), near-collinear both on
    the same side (theta ~ 0) and on opposite sides (theta ~ pi)."""
    for flip in (1.0, -1.0):
        pos = np.array([[0, 0, 0], [1.0, 0, 0],
                        [flip * 1.3 * np.cos(theta), 1.3 * np.sin(theta), 0],
                        [0.3, 1.4, 0.8], [-0.9, -0.7, 1.1], [0.2, -1.5, -0.6], [1.9, 1.1, -0.4]], np.float64)
        s = W.System("collinear", pos.astype(np.float32), np.array([1, 0, 3, 2, 0, 3, 0], np.int32), None, None, 1)
        d, E, F = run_gpu(B, torch, s, params, blob8)
        Eo, Fo = oracle.total_energy_forces(s, params, blob8[: 7 * W.PARAMS_PER_NET])
        assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
        assert np.max(np.abs(F - Fo)) <= F_TOL
        G = d.dhp_debug_aev().cpu().numpy()
        assert np.max(np.abs(G - oracle.aev(s.pos, s.species, None, params))) <= AEV_TOL
        d.close()


@pytest.mark.parametrize("n_models", [3, 5, 7])
def test_ensemble_sizes_on_the_tensor_path(torch, B, params, blob8, n_models):
    """n_models in {2..7} (Eq. 2 ensemble mean, Q11) on the tensor path: the network loop of G1 / k_mlp_mid and the
    K = n_models * 256 contraction of B1."""
    s = W.small_periodic_mix(600, 18.3, seed=77, n_models=n_models)
    probe = B.Dhp(8, params=params)
    ok = probe.dhp_tensor_path_available()
    probe.close()
    if not ok:
        pytest.skip("tensor path not available in this build")
    d, E, F = run_gpu(B, torch, s, params, blob8, B.MLP_TENSOR)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: n_models * 7 * W.PARAMS_PER_NET])
    assert abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F - Fo)) <= F_TOL
    d.close()


def test_collinear_cusp_sensitivity_is_bounded(torch, B, params, blob8):
    """Eq. 5 has a cusp at theta = 0 / pi (theta = |angle| >= 0 and dE/dtheta != 0 there): the direction of the angular
    gradient, e = (r_ik^ - c r_ij^)/s, changes by delta/theta when an input moves by delta.  The oracle takes the fp32
    positions as exact; the kernels round each displacement once to fp32 (2^-24 relative), so their e is off by about
    1e-7 / theta.  DESIGN.md §7: inside the bars down to theta ~ 2.5e-4 rad (previous test; the 98 k box has
    theta_min ~ 5e-4), beyond that the error grows as 1/theta but stays bounded and finite - at theta = 1e-5 it was
    measured at 6.8e-4 Hartree/Å on the two collinear atoms, everything else inside the bars.  This test pins that
    behaviour: no NaN / Inf, energy inside its bar, force error below 1e-7 / theta x |F|-scale, other atoms inside F_TOL."""
    theta = 1e-5
    pos = np.array([[0, 0, 0], [1.0, 0, 0], [1.3 * np.cos(theta), 1.3 * np.sin(theta), 0],
                    [0.3, 1.4, 0.8], [-0.9, -0.7, 1.1], [0.2, -1.5, -0.6], [1.9, 1.1, -0.4]], np.float64)
    s = W.System("cusp", pos.astype(np.float32), np.array([1, 0, 3, 2, 0, 3, 0], np.int32), None, None, 1)
    d, E, F = run_gpu(B, torch, s, params, blob8)
    Eo, Fo = oracle.total_energy_forces(s, params, blob8[: 7 * W.PARAMS_PER_NET])
    assert np.all(np.isfinite(F)) and abs(E[0] - Eo[0]) / s.n_atoms <= E_TOL_PER_ATOM
    err = np.abs(F - Fo)
    assert err.max() <= 2e-3                                   # ~ (1e-7 / 3e-5) x |dE/dtheta| / R
    assert err[3:].max() <= F_TOL                              # atoms not on the line are unaffected
    assert np.abs(F.sum(0)).max() < 1e-5                       # Newton's third law survives the cusp
    d.close()


# ------------------------------------------------------------------------------------------- ANI-1x shape (row f3)
@pytest.mark.parametrize("mode", [1, 2])
def test_ani1x_shape_four_species_box(torch, B, blob8, mode):
    """SURVEY.md §8(f3), PAPER.md L87 / L159: the ANI-1x / ANI-1ccx shape - species H, C, N, O, Rcr = 5.2 Å (L73),
    4 x 8 angular grid, 384 features, networks 384 -> 160 -> 128 -> 96 -> 1 (reading R4) - through the same
    library: `dhp_params` selects the grid, the narrow networks are loaded zero-padded (workloads.embed_ani1x).  Lists
    bit-exact at the 5.2 Å cutoff, AEV / dE/dG rows, E and F against the oracle, SIMT and tensor paths."""
    p1x = W.ani1x_params()
    s = W.small_periodic_mix(900, 21.0, seed=31, n_models=2, hcno_only=True)
    blob = W.embed_ani1x(W.make_weights_ani1x(2), 2)
    d = B.Dhp(s.n_atoms, params=p1x)
    if mode == 2 and not d.dhp_tensor_path_available():
        d.close()
        pytest.skip("tensor path not available in this build")
    d.dhp_set_mlp_mode(mode)
    w = d.dhp_weights_load(blob, 2)
    pos, sp, mol = B.to_device(s)
    E, F = d.dhp_ani_energy_forces(pos, s.box, sp, w)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    Ea, Fo, go = oracle.energy_forces(s.pos, s.species, s.box, p1x, blob, 2, want_dEdG=True)
    assert abs(E.item() - Ea.sum()) / s.n_atoms <= E_TOL_PER_ATOM
    assert np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL
    G = d.dhp_debug_aev().cpu().numpy()
    Go = oracle.aev(s.pos, s.species, s.box, p1x)
    assert np.max(np.abs(G - Go)) <= AEV_TOL
    fmap = W.ani1x_feature_map()
    off = np.ones(1008, bool)
    off[fmap] = False
    assert np.all(G[:, off] == 0.0)                              # only the 384 ANI-1x features exist
    g = d.dhp_debug_grad().cpu().numpy()
    close = np.abs(g - go) <= GRAD_TOL
    assert np.all(close | ((g == 0) & (Go == 0))) and np.all(close[Go != 0])
    lists_equal(B, d, s, p1x)
    d.close()


def test_ani1x_params_are_validated(torch, B):
    import dataclasses
    p = W.ani1x_params()
    bad = dataclasses.replace(p, shf_z=p.shf_z[:4])              # 4 x 4: not one of the two grids
    with pytest.raises(B.DhpError):
        B.Dhp(16, params=bad)


def test_random_systems_sizes_and_ensembles(torch, B, params, blob8):
    """Seeded sweep over system size (40 .. 3 500 atoms: the single-block list path, a handful of row tiles, tens of tiles
    with ragged tails for every species) and ensemble size (1 .. 8): every call - repeated three times on the same context,
    so that replayed graphs, the chain kernel's ping-pong tensor-memory maps and its per-SM scratch tiles are reused - and
    the energy-only call must land inside the north_star bars."""
    rng = np.random.default_rng(123)
    for it in range(16):
        n = int(rng.integers(40, 3500))
        n_models = int(rng.integers(1, 9))
        edge = max((n / 0.1) ** (1.0 / 3.0), 10.5)
        s = W.small_periodic_mix(n, float(edge), seed=int(rng.integers(1, 10**6)), n_models=n_models)
        blob = blob8[: n_models * 7 * W.PARAMS_PER_NET]
        d = B.Dhp(s.n_atoms, params=params)
        w = d.dhp_weights_load(blob, n_models)
        pos, sp, mol = B.to_device(s)
        E = torch.empty(1, dtype=torch.float64, device="cuda")
        F = torch.empty((n, 3), dtype=torch.float32, device="cuda")
        for _ in range(3):
            d.dhp_ani_energy_forces(pos, s.box, sp, w, mol, E=E, F=F)
        Ee = d.dhp_ani_energy(pos, s.box, sp, w, mol)
        torch.cuda.synchronize()
        assert d.dhp_status() == 0
        Eo, Fo = oracle.total_energy_forces(s, params, blob)
        assert abs(E.item() - Eo[0]) / n <= E_TOL_PER_ATOM, (it, n, n_models)
        assert abs(Ee.item() - Eo[0]) / n <= E_TOL_PER_ATOM, (it, n, n_models)
        assert np.max(np.abs(F.cpu().numpy() - Fo)) <= F_TOL, (it, n, n_models)
        d.close()
