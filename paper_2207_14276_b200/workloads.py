"""Seeded synthetic inputs shared by the CUDA path and the fp64 oracle.

This module holds NONE of the method's arithmetic (no cutoff function, no symmetry
function, no network): it only draws geometries, species and random weights, and
packs the hyper-parameters that BASELINE.json configs[0] fixes.  Both the product
path (`paper_2207_14276_b200.binding`) and the test oracle (`oracle/`) read the
fp32 arrays produced here and nothing else.

The five systems stand in for the paper's benchmark structures (§2.3.1:
DHFR 23 558 atoms, M^pro 98 500 atoms, water boxes) and for the solute of the hybrid
scheme (Eq. 7), whose coordinate files are not available; shapes,
densities and compositions come from BASELINE.json `configs` and SURVEY.md §8(d).

All geometry is built in fp64 with numpy `default_rng` (PCG64) and rounded ONCE to fp32.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np
from scipy.spatial import cKDTree

# species order: H, C, N, O, S, F, Cl = 0..6
SPECIES = ("H", "C", "N", "O", "S", "F", "Cl")
H, C, N, O, S, F, CL = range(7)
N_SPECIES = 7

# network shape (BASELINE.json configs[0]): 1008 -> 256 -> 192 -> 160 -> 1
N_RAD_SHIFTS = 16
N_ANG_SHIFTS = 8
N_ANG_SECTIONS = 4
AEV_RADIAL = N_SPECIES * N_RAD_SHIFTS                                   # 112
AEV_ANGULAR = (N_SPECIES * (N_SPECIES + 1) // 2) * N_ANG_SHIFTS * N_ANG_SECTIONS  # 896
AEV_DIM = AEV_RADIAL + AEV_ANGULAR                                      # 1008
LAYERS = (AEV_DIM, 256, 192, 160, 1)
PARAMS_PER_NET = sum(LAYERS[i] * LAYERS[i + 1] + LAYERS[i + 1] for i in range(4))  # 338689

GEOMETRY_SEEDS = {1: 1001, 2: 1002, 3: 1003, 4: 1004, 5: 1005}
WEIGHT_SEED = 2001
MIN_DIST = 0.95          # Å, BASELINE.json configs[2]
OH_BOND = 0.9572         # Å, TIP3P geometry
HOH_ANGLE_DEG = 104.52


@dataclasses.dataclass(frozen=True)
class AniParams:
    """Hyper-parameters as fp32 values (what both sides read).  BASELINE.json configs[0]."""
    rcr: np.float32
    rca: np.float32
    eta_r: np.float32
    eta_a: np.float32
    zeta: np.float32
    celu_alpha: np.float32
    shf_r: np.ndarray   # [16] f32
    shf_a: np.ndarray   # [8]  f32
    shf_z: np.ndarray   # [4]  f32


def default_params() -> AniParams:
    """ANI-2x-shaped AEV parameters of BASELINE.json configs[0]."""
    shf_r = (0.8 + 0.2625 * np.arange(N_RAD_SHIFTS, dtype=np.float64)).astype(np.float32)
    shf_a = (0.8 + 0.3375 * np.arange(N_ANG_SHIFTS, dtype=np.float64)).astype(np.float32)
    shf_z = ((2.0 * np.arange(N_ANG_SECTIONS, dtype=np.float64) + 1.0) * math.pi / 8.0).astype(np.float32)
    return AniParams(rcr=np.float32(5.1), rca=np.float32(3.5), eta_r=np.float32(19.7),
                     eta_a=np.float32(12.5), zeta=np.float32(14.1), celu_alpha=np.float32(0.1),
                     shf_r=shf_r, shf_a=shf_a, shf_z=shf_z)


def ani1x_params() -> AniParams:
    """ANI-1x / ANI-1ccx-shaped AEV parameters ("ANI-1x ... H, C, N, and O"; L73: "R_c ... fixed to 5.2 Å").
    The paper prints no other value; eta / shift values are those of the published ANI-1x model (Smith et al., ANI-1x
    data set / TorchANI `ani-1x_8x` parameter file; reading R4): 16 radial shifts 0.9 + 0.26875 m, EtaR 16;
    angular grid 4 ShfA (0.9 + 0.65 a) x 8 ShfZ ((2k+1) pi/16), EtaA 8, Zeta 32; Rca 3.5 Å.  Species H, C, N, O = 0..3 of
    the library's species order, so the 384-entry ANI-1x AEV is a sub-vector of the 1008-entry layout."""
    shf_r = (0.9 + 0.26875 * np.arange(N_RAD_SHIFTS, dtype=np.float64)).astype(np.float32)
    shf_a = (0.9 + 0.65 * np.arange(4, dtype=np.float64)).astype(np.float32)
    shf_z = ((2.0 * np.arange(8, dtype=np.float64) + 1.0) * math.pi / 16.0).astype(np.float32)
    return AniParams(rcr=np.float32(5.2), rca=np.float32(3.5), eta_r=np.float32(16.0), eta_a=np.float32(8.0),
                     zeta=np.float32(32.0), celu_alpha=np.float32(0.1), shf_r=shf_r, shf_a=shf_a, shf_z=shf_z)


# ANI-1x network shape (reading R4: the published model's hydrogen network, used here for all four elements):
ANI1X_SPECIES = 4
ANI1X_AEV_DIM = ANI1X_SPECIES * N_RAD_SHIFTS + (ANI1X_SPECIES * (ANI1X_SPECIES + 1) // 2) * 32     # 64 + 320 = 384
ANI1X_LAYERS = (ANI1X_AEV_DIM, 160, 128, 96, 1)
ANI1X_PARAMS_PER_NET = sum(ANI1X_LAYERS[i] * ANI1X_LAYERS[i + 1] + ANI1X_LAYERS[i + 1] for i in range(4))


def make_weights_ani1x(n_models: int, seed: int = WEIGHT_SEED + 1) -> np.ndarray:
    """Flat fp32 blob of the NATIVE ANI-1x shape: for e: for s in H,C,N,O: W1[160][384], b1, W2[128][160], b2,
    W3[96][128], b3, W4[1][96], b4 (same initialisation rule as `make_weights`)."""
    rng = np.random.default_rng(seed)
    out = np.empty(n_models * ANI1X_SPECIES * ANI1X_PARAMS_PER_NET, dtype=np.float32)
    p = 0
    for _e in range(n_models):
        for _s in range(ANI1X_SPECIES):
            for l in range(4):
                fan_in, fan_out = ANI1X_LAYERS[l], ANI1X_LAYERS[l + 1]
                w = rng.standard_normal(fan_in * fan_out) * (1.0 / math.sqrt(fan_in))
                out[p:p + w.size] = w.astype(np.float32); p += w.size
                b = rng.standard_normal(fan_out) * 0.1
                out[p:p + b.size] = b.astype(np.float32); p += b.size
    assert p == out.size
    return out


def split_net_ani1x(blob: np.ndarray, e: int, s: int):
    p = (e * ANI1X_SPECIES + s) * ANI1X_PARAMS_PER_NET
    out = []
    for l in range(4):
        fan_in, fan_out = ANI1X_LAYERS[l], ANI1X_LAYERS[l + 1]
        out.append(blob[p:p + fan_in * fan_out].reshape(fan_out, fan_in)); p += fan_in * fan_out
        out.append(blob[p:p + fan_out]); p += fan_out
    return tuple(out)


def ani1x_feature_map() -> np.ndarray:
    """Position of each of the 384 ANI-1x features (radial [s_j][m], then angular [pair(u<=v) of 4][a][z]) inside the
    1008-entry layout of the library (radial [s_j of 7][m], angular [pairidx of 7][32]).  Index arithmetic only."""
    idx = []
    for sj in range(ANI1X_SPECIES):
        idx += [N_RAD_SHIFTS * sj + m for m in range(N_RAD_SHIFTS)]
    for u in range(ANI1X_SPECIES):
        for v in range(u, ANI1X_SPECIES):
            p7 = N_SPECIES * u - u * (u - 1) // 2 + (v - u)
            idx += [AEV_RADIAL + 32 * p7 + q for q in range(32)]
    return np.asarray(idx, dtype=np.int64)


def embed_ani1x(blob1x: np.ndarray, n_models: int) -> np.ndarray:
    """An ANI-1x-shaped ensemble as a blob of the library's fixed layout (7 species, 1008 -> 256 -> 192 -> 160 -> 1):
    each small matrix sits in the top-left corner of its big one (W1's columns scattered by `ani1x_feature_map`),
    everything else - including all parameters of S, F, Cl - is zero.  Padding units see z = 0, CELU(0) = 0, and feed zero
    weights, so the embedded network computes exactly the native one and its input gradient.  Marshalling only."""
    fmap = ani1x_feature_map()
    out = np.zeros(n_models * N_SPECIES * PARAMS_PER_NET, dtype=np.float32)
    for e in range(n_models):
        for s in range(ANI1X_SPECIES):
            small = split_net_ani1x(blob1x, e, s)
            big = split_net(out, e, s)
            W1s, W1b = small[0], big[0]
            W1b[:W1s.shape[0], fmap] = W1s
            big[1][:small[1].size] = small[1]
            for l in (1, 2, 3):
                Ws, Wb = small[2 * l], big[2 * l]
                Wb[:Ws.shape[0], :Ws.shape[1]] = Ws
                big[2 * l + 1][:small[2 * l + 1].size] = small[2 * l + 1]
    return out


@dataclasses.dataclass
class System:
    """One synthetic input: fp32 positions [N,3], int32 species [N], optional cubic box edge,
    optional molecule offsets [n_mol+1] (pairs never cross molecules), ensemble size."""
    name: str
    pos: np.ndarray
    species: np.ndarray
    box: Optional[np.ndarray]          # f32 [3] or None (open boundary)
    mol_offsets: Optional[np.ndarray]  # i32 [n_mol+1] or None
    n_models: int

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_mol(self) -> int:
        return 0 if self.mol_offsets is None else int(self.mol_offsets.shape[0] - 1)


# --------------------------------------------------------------------------------------
# weights
# --------------------------------------------------------------------------------------
def make_weights(n_models: int, seed: int = WEIGHT_SEED) -> np.ndarray:
    """Flat fp32 blob, layout of SURVEY.md §8(b): for e: for s: W1[256][1008], b1[256],
    W2[192][256], b2[192], W3[160][192], b3[160], W4[1][160], b4[1]; row-major [out][in].
    W ~ Normal(0, variance 1/fan_in); b ~ Normal(0, 0.1^2)."""
    rng = np.random.default_rng(seed)
    out = np.empty(n_models * N_SPECIES * PARAMS_PER_NET, dtype=np.float32)
    p = 0
    for _e in range(n_models):
        for _s in range(N_SPECIES):
            for l in range(4):
                fan_in, fan_out = LAYERS[l], LAYERS[l + 1]
                w = rng.standard_normal(fan_in * fan_out) * (1.0 / math.sqrt(fan_in))
                out[p:p + w.size] = w.astype(np.float32); p += w.size
                b = rng.standard_normal(fan_out) * 0.1
                out[p:p + b.size] = b.astype(np.float32); p += b.size
    assert p == out.size
    return out


def split_net(blob: np.ndarray, e: int, s: int):
    """Views (W1,b1,W2,b2,W3,b3,W4,b4) of network (model e, species s) inside the blob."""
    p = (e * N_SPECIES + s) * PARAMS_PER_NET
    out = []
    for l in range(4):
        fan_in, fan_out = LAYERS[l], LAYERS[l + 1]
        out.append(blob[p:p + fan_in * fan_out].reshape(fan_out, fan_in)); p += fan_in * fan_out
        out.append(blob[p:p + fan_out]); p += fan_out
    return tuple(out)


# --------------------------------------------------------------------------------------
# geometry helpers (no method arithmetic)
# --------------------------------------------------------------------------------------
def _random_unit(rng, n=None):
    v = rng.standard_normal(3 if n is None else (n, 3))
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _water_from_o(o, rng):
    """O position(s) [...,3] -> (O,H,H) with TIP3P geometry and random orientation."""
    o = np.atleast_2d(o)
    n = o.shape[0]
    e1 = _random_unit(rng, n)
    t = _random_unit(rng, n)
    e2 = t - (t * e1).sum(-1, keepdims=True) * e1
    e2 /= np.linalg.norm(e2, axis=-1, keepdims=True)
    half = math.radians(HOH_ANGLE_DEG) / 2.0
    h1 = o + OH_BOND * (math.cos(half) * e1 + math.sin(half) * e2)
    h2 = o + OH_BOND * (math.cos(half) * e1 - math.sin(half) * e2)
    return np.stack([o, h1, h2], axis=1)   # [n,3,3]


def _min_image(d, L):
    return d - L * np.rint(d / L)


def water_box_96(seed: int = GEOMETRY_SEEDS[1]) -> System:
    """configs[0]: 96 H2O in a cubic periodic 14.2 Å box."""
    rng = np.random.default_rng(seed)
    L = 14.2
    sites = []
    for i in range(5):
        for j in range(5):
            for k in range(4):
                sites.append(((i + 0.5) * L / 5, (j + 0.5) * L / 5, (k + 0.5) * L / 4))
    sites = np.array(sites[:96])
    sites = sites + rng.uniform(-0.25, 0.25, size=sites.shape)
    placed = np.empty((0, 3))
    for m in range(96):
        while True:
            mol = _water_from_o(sites[m], rng)[0]
            if placed.shape[0] == 0:
                break
            d = _min_image(mol[:, None, :] - placed[None, :, :], L)
            if np.sqrt((d * d).sum(-1)).min() >= MIN_DIST:
                break
        placed = np.concatenate([placed, mol], axis=0)
    species = np.tile(np.array([O, H, H], dtype=np.int32), 96)
    return System("water96", placed.astype(np.float32), species,
                  np.array([L, L, L], dtype=np.float32), None, n_models=1)


def _random_walk_molecule(rng, n_atoms: int, radius: Optional[float]) -> np.ndarray:
    """Connected random walk: each new atom at U(1.0,1.6) Å from a uniformly chosen placed atom,
    >= 1.0 Å from all placed atoms, optionally inside `radius` of the origin."""
    pts = np.zeros((n_atoms, 3))
    n = 1
    while n < n_atoms:
        parent = rng.integers(0, n)
        r = rng.uniform(1.0, 1.6)
        cand = pts[parent] + r * _random_unit(rng)
        if radius is not None and np.linalg.norm(cand) > radius:
            continue
        if np.sqrt(((pts[:n] - cand) ** 2).sum(-1)).min() < 1.0:
            continue
        pts[n] = cand
        n += 1
    return pts


def ligand_50(seed: int = GEOMETRY_SEEDS[2]) -> System:
    """configs[1]: 50-atom solute C16 H24 N4 O4 S1 F1, open boundary, 8 networks."""
    rng = np.random.default_rng(seed)
    pts = _random_walk_molecule(rng, 50, 12.0)
    species = np.array([C] * 16 + [H] * 24 + [N] * 4 + [O] * 4 + [S] * 1 + [F] * 1, dtype=np.int32)
    rng.shuffle(species)
    return System("ligand50", pts.astype(np.float32), species, None, None, n_models=8)


def _rsa_fill(rng, L, placed, n_units, propose, unit_size):
    """Random sequential addition of `n_units` rigid units (`unit_size` atoms each) into a periodic
    cube: a unit is accepted iff all its atoms are >= MIN_DIST (minimum image) from every
    previously accepted atom.  Proposals are drawn in batches; acceptance inside a batch is
    sequential in draw order, so the result is a deterministic function of the seed."""
    out = [placed] if placed.shape[0] else []
    n_done = 0
    all_pts = placed.copy()
    while n_done < n_units:
        batch = max(256, min(8192, 2 * (n_units - n_done)))
        cand = propose(rng, batch)                        # [batch, unit_size, 3]
        flat = np.mod(cand.reshape(-1, 3), L)
        flat[flat >= L] = 0.0
        ok = np.ones(batch, dtype=bool)
        if all_pts.shape[0]:
            tree = cKDTree(np.mod(all_pts, L), boxsize=L)
            cnt = tree.query_ball_point(flat, MIN_DIST - 1e-12, return_length=True)
            ok &= (cnt.reshape(batch, unit_size) == 0).all(axis=1)
        btree = cKDTree(flat, boxsize=L)
        pairs = btree.query_pairs(MIN_DIST - 1e-12, output_type="ndarray")
        conflicts = [[] for _ in range(batch)]
        for a, b in pairs:
            ua, ub = a // unit_size, b // unit_size
            if ua != ub:
                lo, hi = (ua, ub) if ua < ub else (ub, ua)
                conflicts[hi].append(lo)
        accepted = np.zeros(batch, dtype=bool)
        for u in range(batch):
            if n_done >= n_units:
                break
            if not ok[u]:
                continue
            if any(accepted[v] for v in conflicts[u]):
                continue
            accepted[u] = True
            n_done += 1
        new = cand[accepted].reshape(-1, 3)
        out.append(new)
        all_pts = np.concatenate([all_pts, new], axis=0)
    return np.concatenate(out, axis=0) if out else np.empty((0, 3))


def protein_in_water(n_atoms: int, L: float, sphere_radius: float, seed: int, name: str) -> System:
    """configs[2]/[3]: protein-like sphere (H .50, C .31, N .09, O .095, S .005) at the box centre,
    random-orientation TIP3P-geometry water outside it, min distance 0.95 Å."""
    rng = np.random.default_rng(seed)
    rho = n_atoms / L ** 3
    n_prot = int(round(rho * 4.0 / 3.0 * math.pi * sphere_radius ** 3))
    while (n_atoms - n_prot) % 3 != 0:
        n_prot += 1
    n_wat = (n_atoms - n_prot) // 3
    centre = np.array([L / 2, L / 2, L / 2])

    def propose_prot(rng, m):
        # uniform in the sphere by rejection from the bounding cube
        pts = np.empty((0, 3))
        while pts.shape[0] < m:
            c = rng.uniform(-sphere_radius, sphere_radius, size=(2 * m, 3))
            c = c[(c * c).sum(-1) <= sphere_radius ** 2]
            pts = np.concatenate([pts, c], axis=0)
        return (pts[:m] + centre)[:, None, :]

    def propose_wat(rng, m):
        o = np.empty((0, 3))
        while o.shape[0] < m:
            c = rng.uniform(0.0, L, size=(2 * m, 3))
            c = c[((c - centre) ** 2).sum(-1) > sphere_radius ** 2]
            o = np.concatenate([o, c], axis=0)
        return _water_from_o(o[:m], rng)

    prot = _rsa_fill(rng, L, np.empty((0, 3)), n_prot, propose_prot, 1)
    prot_species = rng.choice(np.array([H, C, N, O, S], dtype=np.int32), size=n_prot,
                              p=[0.50, 0.31, 0.09, 0.095, 0.005]).astype(np.int32)
    everything = _rsa_fill(rng, L, prot, n_wat, propose_wat, 3)
    species = np.concatenate([prot_species, np.tile(np.array([O, H, H], dtype=np.int32), n_wat)])
    assert everything.shape[0] == n_atoms == species.shape[0]
    return System(name, everything.astype(np.float32), species.astype(np.int32),
                  np.array([L, L, L], dtype=np.float32), None, n_models=8)


def protein_box_23k(seed: int = GEOMETRY_SEEDS[3]) -> System:
    return protein_in_water(23558, 62.2, 30.0, seed, "protein23k")


def biosystem_98k(seed: int = GEOMETRY_SEEDS[4]) -> System:
    return protein_in_water(98000, 99.7, 45.0, seed, "biosystem98k")


def replicas_1024x30(seed: int = GEOMETRY_SEEDS[5], n_mol: int = 1024) -> System:
    """configs[4]: 1 024 independent 30-atom molecules C10 H14 N2 O3 Cl1, open boundary."""
    base = np.array([C] * 10 + [H] * 14 + [N] * 2 + [O] * 3 + [CL] * 1, dtype=np.int32)
    pos = np.empty((n_mol * 30, 3))
    species = np.empty(n_mol * 30, dtype=np.int32)
    children = np.random.SeedSequence(seed).spawn(n_mol)
    for m in range(n_mol):
        rng = np.random.default_rng(children[m])
        pos[30 * m:30 * m + 30] = _random_walk_molecule(rng, 30, None)
        sp = base.copy()
        rng.shuffle(sp)
        species[30 * m:30 * m + 30] = sp
    mol_offsets = (30 * np.arange(n_mol + 1)).astype(np.int32)
    return System("replicas1024x30", pos.astype(np.float32), species, None, mol_offsets, n_models=8)


def make_system(config: int) -> System:
    """1-based config number of BASELINE.json (`config n` = configs[n-1])."""
    return {1: water_box_96, 2: ligand_50, 3: protein_box_23k,
            4: biosystem_98k, 5: replicas_1024x30}[config]()


def small_periodic_mix(n_atoms: int = 600, L: float = 18.3, seed: int = 77, n_models: int = 2, hcno_only: bool = False) -> System:
    """A small periodic 5-species box at the density of configs[2] (~0.098 Å^-3), used by parity
    tests that need several cells/tiles and a ragged tail at a size the oracle finishes in seconds."""
    rng = np.random.default_rng(seed)

    def propose(rng, m):
        return rng.uniform(0.0, L, size=(m, 1, 3))

    pts = _rsa_fill(rng, L, np.empty((0, 3)), n_atoms, propose, 1)
    species = rng.choice(np.array([H, C, N, O, S], dtype=np.int32), size=n_atoms,
                         p=[0.50, 0.31, 0.09, 0.095, 0.005]).astype(np.int32)
    if hcno_only:                                  # ANI-1x covers H, C, N, O: the few S become O
        species[species == S] = O
    return System(f"mix{n_atoms}", pts.astype(np.float32), species,
                  np.array([L, L, L], dtype=np.float32), None, n_models=n_models)


def small_periodic_ortho(n_atoms: int = 900, box=(17.3, 21.9, 24.6), seed: int = 78, n_models: int = 2) -> System:
    """A periodic ORTHORHOMBIC box with three different edges (include/dhp.h: "cubic/orthorhombic periodic edges") at
    roughly the density of configs[2]: random sequential addition with the 0.95 Å minimum distance (minimum image per
    axis), all 7 species.  Edge-case input of the parity tests; no arithmetic of the method."""
    rng = np.random.default_rng(seed)
    L = np.asarray(box, dtype=np.float64)
    pts = np.empty((0, 3))
    while pts.shape[0] < n_atoms:
        c = rng.uniform(0.0, 1.0, size=3) * L
        if pts.shape[0]:
            d = pts - c
            d -= L * np.rint(d / L)
            if (d * d).sum(-1).min() < MIN_DIST ** 2:
                continue
        pts = np.concatenate([pts, c[None, :]], axis=0)
    species = rng.choice(np.arange(7, dtype=np.int32), size=n_atoms,
                         p=[0.46, 0.28, 0.08, 0.09, 0.03, 0.03, 0.03]).astype(np.int32)
    return System(f"ortho{n_atoms}", pts.astype(np.float32), species, L.astype(np.float32), None, n_models=n_models)


def jitter(system: System, sigma: float, seed: int) -> np.ndarray:
    """Positions displaced by N(0, sigma^2) per coordinate (timing protocol)."""
    rng = np.random.default_rng(seed)
    return (system.pos.astype(np.float64) + rng.normal(0.0, sigma, system.pos.shape)).astype(np.float32)


# --------------------------------------------------------------------------------------
# inputs of the multiple-timestep driver: masses, water O-H bonds, thermal velocities
# --------------------------------------------------------------------------------------
AMU_MASS = np.array([1.008, 12.011, 14.007, 15.999, 32.06, 18.998, 35.45])   # H C N O S F Cl
ACCEL_PER_FORCE = 0.2625499639     # (Å/fs^2) per (Hartree/Å/amu): 4.3597447222e-18 J / 1e-10 m / 1.6605390666e-27 kg
KB_HARTREE = 3.166811563e-6        # Boltzmann constant, Hartree/K


@dataclasses.dataclass
class MdInputs:
    inv_mass: np.ndarray   # f32 [N]  (Å/fs^2)/(Hartree/Å)
    bonds: np.ndarray      # i32 [n_bonds, 2]
    bond_k: np.ndarray     # f32 [n_bonds] Hartree/Å^2 (E = 1/2 k (r - r0)^2)
    bond_r0: np.ndarray    # f32 [n_bonds] Å
    vel: np.ndarray        # f32 [N, 3] Å/fs


def md_inputs(system: System, temperature: float = 300.0, seed: int = 4001, n_protein: Optional[int] = None) -> MdInputs:
    """Masses of the 7 elements; harmonic O-H bonds (k = 1.434 Hartree/Å^2, i.e. 450 kcal/mol/Å^2 in the k (r - r0)^2
    convention; r0 = 0.9572 Å) for every water of the system - the generators above lay waters out as consecutive
    (O, H, H) triples after `n_protein` leading atoms (0 for water96; derived from the recipe for the protein boxes
    when not given); Maxwell-Boltzmann velocities at `temperature` with the centre-of-mass motion removed."""
    n = system.n_atoms
    if n_protein is None:
        n_protein = 0
        if system.name in ("protein23k", "biosystem98k"):
            L = float(system.box[0])
            radius = 30.0 if system.name == "protein23k" else 45.0
            n_protein = int(round(n / L ** 3 * 4.0 / 3.0 * math.pi * radius ** 3))
            while (n - n_protein) % 3 != 0:
                n_protein += 1
        elif system.name != "water96":
            n_protein = n                      # no waters known: no bonds
    sp = system.species
    bonds = []
    for base in range(n_protein, n - 2, 3):
        if sp[base] == O and sp[base + 1] == H and sp[base + 2] == H:
            bonds += [(base, base + 1), (base, base + 2)]
    bonds = np.array(bonds, dtype=np.int32).reshape(-1, 2)
    mass = AMU_MASS[sp]
    rng = np.random.default_rng(seed)
    sigma = np.sqrt(KB_HARTREE * temperature * ACCEL_PER_FORCE / mass)          # Å/fs per component
    vel = rng.normal(0.0, 1.0, (n, 3)) * sigma[:, None]
    vel -= (vel * mass[:, None]).sum(0) / mass.sum()
    return MdInputs((ACCEL_PER_FORCE / mass).astype(np.float32), bonds, np.full(len(bonds), 1.434, np.float32),
                    np.full(len(bonds), 0.9572, np.float32), vel.astype(np.float32))
