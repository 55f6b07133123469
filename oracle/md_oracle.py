"""fp64 CPU oracle of the multiple-timestep driver (TEST INFRASTRUCTURE, like everything under oracle/).

What it follows: PAPER.md §2.3.5 (L198-208).  The potential is split into a cheap, quickly varying part evaluated
every inner timestep (Eq. 8: the bonded terms) and an expensive, slowly varying part evaluated every outer timestep
(Eq. 9: the neural-network term), integrated with RESPA; the paper's reference integrator is velocity Verlet
(L144, L208).  The paper names the scheme (its ref. 63) without printing the update formulas; the reading used here
(reading R1) is the standard symmetric (Trotter) factorisation of one outer step of length dt with n
inner steps of length d = dt / n:

    v += (dt/2) a_slow(x)
    repeat n times:  v += (d/2) a_fast(x);  x += d v;  v += (d/2) a_fast(x)
    v += (dt/2) a_slow(x)

with a = inv_mass * F.  For n = 1 this is velocity Verlet with the force F_slow + F_fast.  The fast part here is a
set of harmonic bonds E = sum_b 1/2 k_b (r_b - r0_b)^2 (a stand-in for the bonded terms; AMOEBA is out of scope).
The slow force is passed in as a callable, so the integrator can be pinned on problems with closed-form solutions
(tests/test_oracle_md_pins.py) independently of the ANI oracle.

Plain numpy, written step by step in the order above; no fusion of half kicks.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import numpy as np


def bond_energy_forces(pos: np.ndarray, box: Optional[np.ndarray], bonds: np.ndarray, k: np.ndarray,
                       r0: np.ndarray) -> Tuple[float, np.ndarray]:
    """E = sum_b 1/2 k_b (|r_j - r_i| - r0_b)^2 and F = -dE/dr (minimum image in a periodic box), fp64."""
    pos = np.asarray(pos, dtype=np.float64)
    F = np.zeros_like(pos)
    E = 0.0
    for b in range(len(bonds)):
        i, j = int(bonds[b][0]), int(bonds[b][1])
        d = pos[j] - pos[i]
        if box is not None:
            L = np.asarray(box, dtype=np.float64)
            d = d - L * np.rint(d / L)
        r = float(np.sqrt(d @ d))
        dr = r - float(r0[b])
        E += 0.5 * float(k[b]) * dr * dr
        g = float(k[b]) * dr * d / r          # dE/dr_j
        F[j] -= g
        F[i] += g
    return E, F


def kinetic_energy(vel: np.ndarray, inv_mass: np.ndarray) -> float:
    """sum_i 1/2 m_i v_i^2 with m_i = 1 / inv_mass_i (Hartree when v is in Å/fs and inv_mass in (Å/fs^2)/(Hartree/Å))."""
    v = np.asarray(vel, dtype=np.float64)
    return float(0.5 * np.sum((v * v).sum(1) / np.asarray(inv_mass, dtype=np.float64)))


def respa_run(pos: np.ndarray, vel: np.ndarray, inv_mass: np.ndarray, slow: Callable[[np.ndarray], Tuple[float, np.ndarray]],
              fast: Optional[Callable[[np.ndarray], Tuple[float, np.ndarray]]], dt: float, n_inner: int, n_steps: int):
    """n_steps outer steps.  `slow(x)` / `fast(x)` return (energy, forces [N,3]).  Returns x, v, (E_slow, E_fast, E_kin)
    at the end.  fp64 throughout."""
    x = np.array(pos, dtype=np.float64)
    v = np.array(vel, dtype=np.float64)
    w = np.asarray(inv_mass, dtype=np.float64)[:, None]
    if fast is None:
        n_inner = 1
    d = dt / n_inner
    E_s, F_s = slow(x)
    E_f, F_f = fast(x) if fast is not None else (0.0, np.zeros_like(x))
    for _ in range(n_steps):
        v = v + 0.5 * dt * w * F_s
        for _ in range(n_inner):
            v = v + 0.5 * d * w * F_f
            x = x + d * v
            if fast is not None:
                E_f, F_f = fast(x)
            v = v + 0.5 * d * w * F_f
        E_s, F_s = slow(x)
        v = v + 0.5 * dt * w * F_s
    return x, v, (E_s, E_f, kinetic_energy(v, inv_mass))
