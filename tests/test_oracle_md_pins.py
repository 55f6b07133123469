"""Pins of oracle/md_oracle.py (the fp64 RESPA / velocity-Verlet oracle of the multiple-timestep driver, PAPER.md
§2.3.5, Eqs. 8-9) against what the mathematics fixes, independently of the CUDA path:

* velocity Verlet on a harmonic oscillator has the closed-form solution u_n = u_0 cos(n phi), cos(phi) = 1 - (w d)^2/2
  (Stoermer recurrence u_{n+1} - 2 u_n + u_{n-1} = -(w d)^2 u_n with the Verlet start u_1 = u_0 cos(phi));
* n_inner = 1 is velocity Verlet with the summed force; the scheme is time-reversible and second order;
* the bond force is minus the gradient of the bond energy (central differences) and sums to zero.
"""
import numpy as np

import oracle
from oracle import md_oracle as M
from paper_2207_14276_b200 import workloads as W


def _dimer(u0=0.11, r0=0.9572):
    pos = np.array([[0.0, 0.0, 0.0], [r0 + u0, 0.0, 0.0]])
    inv_mass = np.array([W.ACCEL_PER_FORCE / 15.999, W.ACCEL_PER_FORCE / 1.008])
    bonds = np.array([[0, 1]], np.int32)
    return pos, inv_mass, bonds


def test_bond_force_is_minus_gradient_and_sums_to_zero():
    rng = np.random.default_rng(0)
    pos = rng.uniform(0, 6.0, (7, 3))
    box = np.array([6.0, 6.0, 6.0])
    bonds = np.array([[0, 1], [1, 2], [3, 6], [4, 5]], np.int32)
    k = np.array([1.4, 0.7, 2.0, 0.3])
    r0 = np.array([0.9, 1.1, 1.5, 2.0])
    E, F = M.bond_energy_forces(pos, box, bonds, k, r0)
    assert np.abs(F.sum(0)).max() < 1e-13
    h = 1e-5
    for a in range(7):
        for c in range(3):
            p, m = pos.copy(), pos.copy()
            p[a, c] += h
            m[a, c] -= h
            g = (M.bond_energy_forces(p, box, bonds, k, r0)[0] - M.bond_energy_forces(m, box, bonds, k, r0)[0]) / (2 * h)
            assert abs(F[a, c] + g) < 1e-8
    # closed form: one bond stretched by u along x
    pos2, _, b2 = _dimer(u0=0.2)
    E2, F2 = M.bond_energy_forces(pos2, None, b2, np.array([1.434]), np.array([0.9572]))
    assert abs(E2 - 0.5 * 1.434 * 0.04) < 1e-15 and abs(F2[1, 0] + 1.434 * 0.2) < 1e-14 and abs(F2[0, 0] - 1.434 * 0.2) < 1e-14


def test_velocity_verlet_harmonic_closed_form_fast_and_slow_slots():
    k, r0, u0 = 1.434, 0.9572, 0.11
    pos, inv_mass, bonds = _dimer(u0, r0)
    vel = np.zeros_like(pos)
    w2 = k * inv_mass.sum()                              # relative coordinate: u'' = -k (1/m1 + 1/m2) u
    bond = lambda x: M.bond_energy_forces(x, None, bonds, np.array([k]), np.array([r0]))
    zero = lambda x: (0.0, np.zeros_like(x))
    # (a) the bond in the FAST slot, nothing slow: 4 inner steps of d = 0.05 per outer step
    d, n_inner, n_steps = 0.05, 4, 9
    x, v, E = M.respa_run(pos, vel, inv_mass, zero, bond, d * n_inner, n_inner, n_steps)
    phi = np.arccos(1.0 - 0.5 * w2 * d * d)
    u = np.linalg.norm(x[1] - x[0]) - r0
    assert abs(u - u0 * np.cos(n_inner * n_steps * phi)) < 1e-13
    # (b) the bond in the SLOW slot, nothing fast: velocity Verlet with dt
    dt = 0.07
    x, v, E = M.respa_run(pos, vel, inv_mass, bond, None, dt, 1, 13)
    phi = np.arccos(1.0 - 0.5 * w2 * dt * dt)
    assert abs(np.linalg.norm(x[1] - x[0]) - r0 - u0 * np.cos(13 * phi)) < 1e-13
    # centre of mass stays put (v0 = 0), kinetic + potential energy stays within O(dt^2) of the start
    m = 1.0 / inv_mass
    assert np.abs((x * m[:, None]).sum(0) - (pos * m[:, None]).sum(0)).max() < 1e-12
    E0 = 0.5 * k * u0 * u0
    assert abs(E[0] + E[2] - E0) < 0.5 * w2 * dt * dt * E0


def test_n_inner_one_is_velocity_verlet_with_the_summed_force():
    k1, k2, r0 = 0.9, 0.5, 0.9572
    pos, inv_mass, bonds = _dimer(0.08, r0)
    vel = np.array([[0.001, 0.0, 0.002], [-0.01, 0.004, 0.0]])
    f1 = lambda x: M.bond_energy_forces(x, None, bonds, np.array([k1]), np.array([r0]))
    f2 = lambda x: M.bond_energy_forces(x, None, bonds, np.array([k2]), np.array([r0]))
    both = lambda x: M.bond_energy_forces(x, None, bonds, np.array([k1 + k2]), np.array([r0]))
    xa, va, _ = M.respa_run(pos, vel, inv_mass, f1, f2, 0.1, 1, 7)
    xb, vb, _ = M.respa_run(pos, vel, inv_mass, both, None, 0.1, 1, 7)
    assert np.abs(xa - xb).max() < 1e-14 and np.abs(va - vb).max() < 1e-14


def _water_problem():
    s = W.make_system(1)
    params = W.default_params()
    blob = W.make_weights(1)
    md = W.md_inputs(s)
    slow = lambda x: (lambda E, F: (float(E.sum()), F.astype(np.float64)))(
        *oracle.energy_forces(x.astype(np.float32), s.species, s.box, params, blob, 1)[:2])
    fast = lambda x: M.bond_energy_forces(x, s.box, md.bonds, md.bond_k.astype(np.float64), md.bond_r0.astype(np.float64))
    return s, md, slow, fast


def test_md_inputs_shapes_and_thermal_scale():
    s, md, _, _ = _water_problem()
    assert md.bonds.shape == (192, 2) and np.all(s.species[md.bonds[:, 0]] == W.O) and np.all(s.species[md.bonds[:, 1]] == W.H)
    d = s.pos[md.bonds[:, 1]] - s.pos[md.bonds[:, 0]]
    d -= s.box * np.rint(d / s.box)
    assert np.abs(np.linalg.norm(d, axis=1) - 0.9572).max() < 1e-4            # the generator's O-H distance
    T = 2.0 * M.kinetic_energy(md.vel, md.inv_mass) / (3 * s.n_atoms * W.KB_HARTREE)
    assert 240.0 < T < 360.0                                                  # 288 atoms: +-10 % of 300 K is > 3 sigma
    m = 1.0 / md.inv_mass
    assert np.abs((md.vel * m[:, None]).sum(0)).max() / m.sum() < 1e-8


def test_respa_with_the_ani_oracle_is_time_reversible_and_second_order():
    s, md, slow, fast = _water_problem()
    # The oracle rounds positions to fp32 on entry (it reads the fp32 inputs of the workloads), so reversibility holds to
    # that rounding, not to fp64 round-off
    x1, v1, E1 = M.respa_run(s.pos, md.vel, md.inv_mass, slow, fast, 0.2, 2, 3)
    x0, v0, _ = M.respa_run(x1, -v1, md.inv_mass, slow, fast, 0.2, 2, 3)
    assert np.abs(x0 - s.pos).max() < 2e-6 and np.abs(v0 + md.vel).max() < 2e-6
    # total energy error after a fixed time shrinks ~4x when every timestep is halved
    E_start = slow(s.pos.astype(np.float64))[0] + fast(s.pos.astype(np.float64))[0] + M.kinetic_energy(md.vel, md.inv_mass)
    errs = []
    for dt, n in ((0.2, 2), (0.1, 4)):
        _, _, E = M.respa_run(s.pos, md.vel, md.inv_mass, slow, fast, dt, 2, n)
        errs.append(abs(sum(E) - E_start))
    assert errs[1] < 0.45 * errs[0]


def test_md_inputs_find_the_waters_of_every_generator():
    """The fast force of the driver is the O-H bonds of the generators' waters; a protein box whose
    name the helper does not recognise would silently get none (round-1 bug: "proteinbox23k" vs "protein23k")."""
    s = W.make_system(3)
    m = W.md_inputs(s)
    assert len(m.bonds) > 0 and len(m.bonds) % 2 == 0
    # every bond is an O-H pair at the TIP3P length (minimum image)
    d = s.pos[m.bonds[:, 1]].astype(np.float64) - s.pos[m.bonds[:, 0]].astype(np.float64)
    L = float(s.box[0])
    d -= L * np.rint(d / L)
    assert np.all(s.species[m.bonds[:, 0]] == W.O) and np.all(s.species[m.bonds[:, 1]] == W.H)
    assert np.abs(np.sqrt((d * d).sum(1)) - W.OH_BOND).max() < 1e-4
    # the waters are everything outside the protein-like sphere: 3 atoms per 2 bonds
    n_prot = s.n_atoms - 3 * (len(m.bonds) // 2)
    assert 0.40 < n_prot / s.n_atoms < 0.55
    assert len(W.md_inputs(W.make_system(1)).bonds) == 2 * 96
