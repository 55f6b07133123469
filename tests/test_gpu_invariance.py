"""Properties of the CUDA path that hold at any size and need no oracle value (the energy is a sum
of atomic terms over local environments): invariance of E under whole-box translation, relabelling of atoms and - for
open boundaries - rigid rotation, with forces that permute / rotate accordingly; periodic images give the same
answer; sum of forces = 0.  Run on configs[0], configs[1] and at full size on configs[2] (23 558 atoms)."""
import numpy as np
import pytest

from paper_2207_14276_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2207_14276_b200 import binding
    return binding


def evaluate(d, torch, w, pos, species, box):
    E, F = d.dhp_ani_energy_forces(torch.from_numpy(np.ascontiguousarray(pos, dtype=np.float32)).cuda(), box,
                                   torch.from_numpy(np.ascontiguousarray(species, dtype=np.int32)).cuda(), w)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    return E.item(), F.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("cfg", [1, 3])
def test_periodic_translation_images_and_relabelling(torch, B, params, cfg):
    s = W.make_system(cfg)
    blob = W.make_weights(s.n_models)
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(blob, s.n_models)
    n = s.n_atoms
    # fp32 evaluation: per-atom energies carry ~1e-7 relative rounding that changes with the summation order
    e_tol, f_tol = 2e-7 * n, 2e-5
    E0, F0 = evaluate(d, torch, w, s.pos, s.species, s.box)
    assert np.abs(F0.sum(0)).max() < 2e-2
    # (1) whole-box images of some atoms: identical neighbourhoods
    q = s.pos.copy()
    q[::3, 0] += s.box[0]
    q[1::5, 2] -= 2 * s.box[2]
    E1, F1 = evaluate(d, torch, w, q, s.species, s.box)
    assert abs(E1 - E0) <= e_tol and np.abs(F1 - F0).max() <= f_tol
    # (2) rigid translation by an arbitrary vector (positions leave [0, L))
    t = np.array([3.217, -11.03, 0.55], np.float32)
    E2, F2 = evaluate(d, torch, w, s.pos + t, s.species, s.box)
    assert abs(E2 - E0) <= e_tol and np.abs(F2 - F0).max() <= f_tol
    # (3) relabelling: a random permutation of the atoms permutes the forces
    perm = np.random.default_rng(5).permutation(n)
    E3, F3 = evaluate(d, torch, w, s.pos[perm], s.species[perm], s.box)
    assert abs(E3 - E0) <= e_tol and np.abs(F3 - F0[perm]).max() <= f_tol
    # (4) cubic symmetry: swapping the x and y axes of a cubic cell
    E4, F4 = evaluate(d, torch, w, s.pos[:, [1, 0, 2]], s.species, s.box)
    assert abs(E4 - E0) <= e_tol and np.abs(F4 - F0[:, [1, 0, 2]]).max() <= f_tol
    d.close()


def test_open_boundary_rotation_translation_and_torque(torch, B, params):
    s = W.make_system(2)
    blob = W.make_weights(s.n_models)
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(blob, s.n_models)
    E0, F0 = evaluate(d, torch, w, s.pos, s.species, None)
    assert np.abs(F0.sum(0)).max() < 1e-4
    assert np.abs(np.cross(s.pos.astype(np.float64), F0).sum(0)).max() < 2e-3          # no net torque on an isolated molecule
    rng = np.random.default_rng(8)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    t = np.array([40.0, -7.0, 13.0])
    q = (s.pos.astype(np.float64) @ Q.T + t).astype(np.float32)
    E1, F1 = evaluate(d, torch, w, q, s.species, None)
    # the rotated coordinates are re-rounded to fp32 (1e-6 A at |x| ~ 40), forces ~ 0.1 Ha/A with gradients ~ 1 Ha/A^2
    assert abs(E1 - E0) <= 1e-5 and np.abs(F1 - F0 @ Q.T).max() <= 5e-5
    d.close()
