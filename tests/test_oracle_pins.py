"""Pins of the fp64 oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself through a retyped formula: the expected values are
closed-form numbers stored in tests/golden/ (cited there), library routines (scipy cKDTree for the
pair sets, torch autograd for the network), invariances, and central finite differences.
Runs with -m "not gpu".
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2207_14276_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    with open(os.path.join(HERE, "golden", "aev_closed_form.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split()
            out[k] = float(v)
    return out


G = golden()
RAD = 112


def pairidx(u, v):
    u, v = min(u, v), max(u, v)
    return 7 * u - u * (u - 1) // 2 + (v - u)


def trimer(r1, r2, theta):
    return np.array([[0, 0, 0], [r1, 0, 0], [r2 * math.cos(theta), r2 * math.sin(theta), 0]], dtype=np.float32)


# ------------------------------------------------------------------ layout / feature count
def test_feature_count():
    assert oracle.AEV_DIM == 7 * 16 + 28 * 32 == 1008 == W.AEV_DIM
    assert oracle.NET_PARAMS == W.PARAMS_PER_NET == 338689


def test_nonzero_columns_follow_present_species(params):
    s = W.make_system(1)                                    # H/O only -> 16*2 + 32*3 = 128 columns
    a = oracle.aev(s.pos, s.species, s.box, params)
    assert int((a != 0).any(axis=0).sum()) == 128
    s = W.small_periodic_mix(300, 14.5)                     # 5 species -> 16*5 + 32*15 = 560
    a = oracle.aev(s.pos, s.species, s.box, params)
    nz = (a != 0).any(axis=0)
    assert int(nz.sum()) <= 560
    present = sorted(set(s.species.tolist()))
    for sp in range(7):
        blk = nz[16 * sp:16 * sp + 16]
        assert blk.any() == (sp in present)


# ------------------------------------------------------------------ radial (Eq. 3, Eq. 4)
@pytest.mark.parametrize("sj", [0, 3, 6])
def test_dimer_radial_closed_form(params, sj):
    pos = np.array([[0, 0, 0], [1.0, 0, 0]], dtype=np.float32)
    sp = np.array([1, sj], dtype=np.int32)
    a = oracle.aev(pos, sp, None, params)
    blk = a[0, 16 * sj:16 * sj + 16]
    for m in range(5):
        assert blk[m] == pytest.approx(G[f"rad_R1.0_m{m}"], rel=2e-6)
    mask = np.ones(1008, bool)
    mask[16 * sj:16 * sj + 16] = False
    assert np.all(a[0, mask] == 0.0)                        # everything else is exactly zero
    # the other atom sees species 1 at the same distance
    assert np.allclose(a[1, 16:32], blk, rtol=0, atol=1e-15)


def test_radial_at_shift_equals_cutoff(params):
    # at R = ShfR_0 the Gaussian is 1 and the entry is f_c(R)
    r = float(params.shf_r[0])
    a = oracle.aev(np.array([[0, 0, 0], [0, r, 0]], dtype=np.float32), np.array([0, 0], np.int32), None, params)
    assert a[0, 0] == pytest.approx(G["fc_0.8_rc5.1"], rel=1e-6)
    # f_c(Rc/2) = 1/2 exactly: at R = 2.55 entry m has Gaussian g_m, ratio to R-independent golden f_c
    a = oracle.aev(np.array([[0, 0, 0], [0, 0, 2.55]], dtype=np.float32), np.array([0, 0], np.int32), None, params)
    m = 7                                                   # ShfR_7 = 2.6375
    expect = 0.5 * math.exp(-19.7 * (2.55 - 2.6375) ** 2)
    assert a[0, m] == pytest.approx(expect, rel=2e-6)


def test_cutoff_decay_and_exclusion(params):
    sp = np.array([0, 0], np.int32)
    prev = None
    for r in (5.0, 5.05, 5.09, 5.099):
        a = oracle.aev(np.array([[0, 0, 0], [r, 0, 0]], dtype=np.float32), sp, None, params)
        tot = a[0].sum()
        assert tot > 0
        if prev is not None:
            assert tot < prev
        prev = tot
    assert prev < 1e-6
    a = oracle.aev(np.array([[0, 0, 0], [5.1001, 0, 0]], dtype=np.float32), sp, None, params)
    assert np.all(a == 0.0)


# ------------------------------------------------------------------ angular (Eq. 5)
def test_trimer_isosceles_peak(params):
    r = float(params.shf_a[2])
    for z in range(4):
        th = float(params.shf_z[z])
        a = oracle.aev(trimer(r, r, th), np.array([1, 0, 0], np.int32), None, params)
        blk = a[0, RAD + 32 * pairidx(0, 0):RAD + 32 * pairidx(0, 0) + 32].reshape(8, 4)
        assert blk[2, z] == pytest.approx(G["ang_iso_R1.475"], rel=5e-6)
        assert blk[2, z] == blk[2].max()


@pytest.mark.parametrize("sj,sk", [(0, 0), (0, 3), (3, 0), (4, 6), (6, 4)])
def test_trimer_general_closed_form(params, sj, sk):
    a = oracle.aev(trimer(1.0, 1.2, math.radians(100.0)), np.array([2, sj, sk], np.int32), None, params)
    p = pairidx(sj, sk)
    blk = a[0, RAD + 32 * p:RAD + 32 * p + 32].reshape(8, 4)
    for q in range(2):
        for z in range(4):
            assert blk[q, z] == pytest.approx(G[f"ang_gen_a{q}_z{z}"], rel=5e-6)
    ang = a[0, RAD:].copy()
    ang[32 * p:32 * p + 32] = 0
    assert np.all(ang == 0.0)


def test_angular_uses_only_the_angular_cutoff(params):
    # k at 3.6 Å > Rca: no angular term at all, but a radial one
    a = oracle.aev(trimer(1.0, 3.6, 1.0), np.array([0, 0, 0], np.int32), None, params)
    assert np.all(a[0, RAD:] == 0.0) and a[0, :16].sum() > 0


# ------------------------------------------------------------------ pair list
def kd_pairs(pos, box, rc):
    from scipy.spatial import cKDTree
    p = pos.astype(np.float64)
    if box is not None:
        L = float(box[0])
        p = p - L * np.floor(p / L)
        p[p >= L] -= L
        t = cKDTree(p, boxsize=L)
    else:
        t = cKDTree(p)
    pr = t.query_pairs(rc, output_type="ndarray")
    return set(map(tuple, pr)) | set(map(tuple, pr[:, ::-1]))


def kd_pairs_ortho(pos, box, rc):
    """Periodic k-d tree with one edge PER AXIS (scipy's own minimum image): the independent statement of the oracle's
    orthorhombic branch (pair_r2: d -= L_axis * rint(d / L_axis))."""
    from scipy.spatial import cKDTree
    L = np.asarray(box, dtype=np.float64)
    p = pos.astype(np.float64)
    p = p - L * np.floor(p / L)
    p = np.where(p >= L, p - L, p)
    pr = cKDTree(p, boxsize=L).query_pairs(rc, output_type="ndarray")
    return set(map(tuple, pr)) | set(map(tuple, pr[:, ::-1]))


@pytest.mark.parametrize("n,box", [(900, (17.3, 21.9, 24.6)), (300, (10.3, 13.0, 22.5)), (400, (22.5, 10.3, 13.0))])
@pytest.mark.parametrize("rc", [5.1, 3.5])
def test_pairs_orthorhombic_box_match_kdtree(params, n, box, rc):
    """every other pin uses a cubic box, so `L = box[0]` for all three axes in pair_r2 passed them all.  Three
    different edges, the short one on different axes (10.3 Å is barely 2 Rcr: most pairs along it cross the boundary)."""
    s = W.small_periodic_ortho(n, box, seed=78 + n)
    shift = np.array([0.0, 2.0, -1.0], np.float32) * s.box            # whole-box shifts per axis: atoms outside [0, L)
    pos = s.pos.copy()
    pos[::5] += shift
    rp, col = oracle.pairs(pos, s.box, rc)
    mine = {(i, int(j)) for i in range(s.n_atoms) for j in col[rp[i]:rp[i + 1]]}
    assert mine == kd_pairs_ortho(pos, s.box, float(np.float32(rc)))
    # a cubic box with the first edge is a different list: the test distinguishes the two
    assert mine != kd_pairs(pos, s.box, float(np.float32(rc)))


def test_energy_forces_follow_an_axis_permutation_of_an_orthorhombic_box(params):
    """Relabelling the axes (x, y, z) -> (z, x, y) of positions AND box is a symmetry of Eqs. 2-5 with per-axis minimum image:
    same energies, forces with permuted components.  A per-axis mix-up anywhere (pairs, AEV displacements, force
    back-substitution) breaks it because the three edges differ."""
    s = W.small_periodic_ortho(240, (10.3, 13.0, 18.1), seed=91, n_models=1)
    blob = W.make_weights(1)
    Ea, Fa, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 1)
    perm = [2, 0, 1]
    Eb, Fb, _ = oracle.energy_forces(np.ascontiguousarray(s.pos[:, perm]), s.species, np.ascontiguousarray(s.box[perm]), params, blob, 1)
    assert np.max(np.abs(Ea - Eb)) <= 1e-12
    assert np.max(np.abs(Fa[:, perm] - Fb)) <= 1e-11
    assert np.abs(Fa).max() > 1e-3                                     # not a trivially empty system


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("periodic", [False, True])
def test_pair_at_exactly_the_cutoff_is_in_the_list_one_ulp_beyond_is_not(params, axis, periodic):
    """Eq. 3 is "R <= Rc" (reading Q2): the tie is inclusive, at both cutoffs, in the oracle itself (the GPU half
    of this statement lives in test_gpu_parity_full.py).  Separations are exact in fp32: 1.0 + float32(rc) is representable."""
    box = np.array([23.0, 26.0, 29.0], np.float32) if periodic else None
    for rc in (params.rcr, params.rca):
        rcf = np.float32(rc)
        e = np.zeros(3, np.float32); e[axis] = 1.0
        at, beyond = np.float32(1.0) + rcf, np.nextafter(np.float32(1.0) + rcf, np.float32(100.0))
        assert np.float64(at) - 1.0 == np.float64(rcf) and np.float64(beyond) - 1.0 > np.float64(rcf)
        base = np.ones(3, np.float32)
        pos = np.stack([base, base + (at - 1) * e, base - (beyond - 1) * e]).astype(np.float32)
        assert np.float64(pos[1, axis]) - 1.0 == np.float64(rcf) and 1.0 - np.float64(pos[2, axis]) > np.float64(rcf)
        rp, col = oracle.pairs(pos, box, float(rc))
        assert list(col[rp[0]:rp[1]]) == [1]                           # the tie is kept, one ulp beyond is not
        assert list(col[rp[1]:rp[2]]) == [0] and rp[3] == rp[2]


@pytest.mark.parametrize("cfg,rc", [(1, 5.1), (1, 3.5), (2, 5.1), (2, 3.5)])
def test_pairs_match_kdtree(params, cfg, rc):
    s = W.make_system(cfg)
    rp, col = oracle.pairs(s.pos, s.box, rc)
    mine = {(i, int(j)) for i in range(s.n_atoms) for j in col[rp[i]:rp[i + 1]]}
    assert mine == kd_pairs(s.pos, s.box, float(np.float32(rc)))
    for i in range(s.n_atoms):                              # canonical form: ascending columns
        assert np.all(np.diff(col[rp[i]:rp[i + 1]]) > 0)


def test_pairs_medium_box_and_image_shift(params):
    s = W.small_periodic_mix(1500, 24.8, seed=5)
    rp, col = oracle.pairs(s.pos, s.box, 5.1)
    mine = {(i, int(j)) for i in range(s.n_atoms) for j in col[rp[i]:rp[i + 1]]}
    assert mine == kd_pairs(s.pos, s.box, float(np.float32(5.1)))
    assert rp[-1] / s.n_atoms == pytest.approx(s.n_atoms / 24.8 ** 3 * 4 / 3 * math.pi * 5.1 ** 3, rel=0.05)
    pos2 = s.pos.copy()                                     # shifting by a power-of-two-friendly whole box
    Lbox = W.System("x", s.pos, s.species, np.array([16.0] * 3, np.float32), None, 1)
    q = (s.pos % 16.0).astype(np.float32)
    rp1, col1 = oracle.pairs(q, Lbox.box, 5.1)
    q2 = q.copy(); q2[::3, 0] += 16.0; q2[1::3, 2] -= 32.0  # exact in fp32
    rp2, col2 = oracle.pairs(q2, Lbox.box, 5.1)
    assert np.array_equal(rp1, rp2) and np.array_equal(col1, col2)


def test_pairs_never_cross_molecules(params):
    s = W.replicas_1024x30(n_mol=6)
    rp, col = oracle.pairs(s.pos, None, 5.1, mol_offsets=s.mol_offsets)
    for i in range(s.n_atoms):
        assert np.all(col[rp[i]:rp[i + 1]] // 30 == i // 30)
    # each molecule alone gives the same rows
    for m in range(6):
        rpm, colm = oracle.pairs(s.pos[30 * m:30 * m + 30], None, 5.1)
        for a in range(30):
            i = 30 * m + a
            assert np.array_equal(col[rp[i]:rp[i + 1]] - 30 * m, colm[rpm[a]:rpm[a + 1]])


# ------------------------------------------------------------------ network
def torch_mlp(aev_rows, species, blob, n_models, alpha):
    import torch
    torch.set_num_threads(4)
    x = torch.tensor(aev_rows, dtype=torch.float64, requires_grad=True)
    total = []
    for r in range(x.shape[0]):
        acc = 0.0
        for e in range(n_models):
            W1, b1, W2, b2, W3, b3, W4, b4 = [torch.tensor(np.asarray(t), dtype=torch.float64)
                                              for t in W.split_net(blob, e, int(species[r]))]
            h = torch.nn.functional.celu(torch.nn.functional.linear(x[r], W1, b1), alpha)
            h = torch.nn.functional.celu(torch.nn.functional.linear(h, W2, b2), alpha)
            h = torch.nn.functional.celu(torch.nn.functional.linear(h, W3, b3), alpha)
            acc = acc + torch.nn.functional.linear(h, W4, b4)[0]
        total.append(acc / n_models)
    E = torch.stack(total)
    E.sum().backward()
    return E.detach().numpy(), x.grad.numpy()


def test_mlp_matches_torch_autograd(params):
    rng = np.random.default_rng(3)
    blob = W.make_weights(2, seed=11)
    s = W.make_system(2)
    rows = oracle.aev(s.pos, s.species, None, params)[:14]
    rows[3] = 0.0                                           # isolated atom: G = 0 is a valid input (Q15)
    rows[4] = rng.uniform(0, 1, 1008)                       # dense row
    sp = np.array([0, 1, 2, 3, 4, 5, 6, 0, 1, 2, 3, 4, 5, 6], np.int32)
    E, g = oracle.mlp(rows, sp, blob, 2, params)
    Et, gt = torch_mlp(rows, sp, blob, 2, float(np.float32(0.1)))
    assert np.allclose(E, Et, rtol=0, atol=1e-12)
    assert np.allclose(g, gt, rtol=0, atol=1e-12)


def test_mlp_linear_regime_and_ensemble(params):
    blob = W.make_weights(1, seed=12).copy()
    x = np.random.default_rng(0).uniform(0, 1, (3, 1008))
    s = 3
    W1, b1, W2, b2, W3, b3, W4, b4 = W.split_net(blob, 0, s)
    b1[:] = 5.0; b2[:] = 60.0; b3[:] = 1500.0               # every pre-activation positive -> CELU = identity
    E, g = oracle.mlp(x, np.full(3, s, np.int32), blob, 1, params)
    A1, A2, A3, A4 = [np.asarray(t, np.float64) for t in (W1, W2, W3, W4)]
    z1 = x @ A1.T + b1; z2 = z1 @ A2.T + b2; z3 = z2 @ A3.T + b3
    assert z1.min() > 0 and z2.min() > 0 and z3.min() > 0
    lin = A4 @ A3 @ A2 @ A1
    const = (A4 @ (A3 @ (A2 @ b1.astype(np.float64) + b2) + b3) + b4)[0]
    assert np.allclose(E, x @ lin[0] + const, rtol=1e-13, atol=1e-12)
    assert np.allclose(g, np.broadcast_to(lin[0], g.shape), rtol=1e-12, atol=1e-14)
    # E is linear in the output bias
    b4[:] += 0.25
    E2, _ = oracle.mlp(x, np.full(3, s, np.int32), blob, 1, params)
    assert np.allclose(E2 - E, 0.25, atol=1e-12)
    # 8 identical models == 1 model
    blob8 = np.tile(blob, 8)
    E8, g8 = oracle.mlp(x, np.full(3, s, np.int32), blob8, 8, params)
    E1, g1 = oracle.mlp(x, np.full(3, s, np.int32), blob, 1, params)
    assert np.allclose(E8, E1, atol=1e-13) and np.allclose(g8, g1, atol=1e-14)


def test_celu_special_values(params):
    # a network reduced to one CELU: W1 picks feature 0 into unit 0 with huge-negative others
    blob = np.zeros(7 * W.PARAMS_PER_NET, np.float32)
    W1, b1, W2, b2, W3, b3, W4, b4 = W.split_net(blob, 0, 0)
    W1[0, 0] = 1.0; b2[:] = 1.0; b3[:] = 1.0                # layers 2,3 output CELU(1)=1 constants
    W2[0, 0] = 1.0; W3[0, 0] = 1.0; W4[0, 0] = 1.0
    # E = CELU(CELU(CELU(x) + 1) + 1): for x=-0.05: inner h=celu(-0.05); then positive -> identity
    for key, xval in (("celu_-0.05", -0.05), ("celu_-1", -1.0)):
        x = np.zeros((1, 1008)); x[0, 0] = xval
        E, g = oracle.mlp(x, np.zeros(1, np.int32), blob, 1, params)
        assert E[0] - 2.0 == pytest.approx(G[key], rel=2e-6)
    # derivative is continuous (= 1) at 0
    for xval in (-1e-9, 1e-9):
        x = np.zeros((1, 1008)); x[0, 0] = xval
        _, g = oracle.mlp(x, np.zeros(1, np.int32), blob, 1, params)
        assert g[0, 0] == pytest.approx(1.0, abs=1e-7)


# ------------------------------------------------------------------ forces
def energy_only(s, pos, params, blob):
    E, _, _ = oracle.energy_forces(pos, s.species, s.box, params, blob, s.n_models, mol_offsets=s.mol_offsets)
    return E.sum()


@pytest.mark.parametrize("cfg", [2, 1])
def test_forces_equal_minus_finite_difference_gradient(params, cfg):
    s = W.make_system(cfg)
    blob = W.make_weights(s.n_models)
    _, F, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, s.n_models)
    rng = np.random.default_rng(cfg)
    h = 2.0 ** -16                                           # E is C^1 (CELU'' and f_c'' jump), see next test
    for a in rng.choice(s.n_atoms, 4, replace=False):
        for c in range(3):
            # positions are fp32 inputs; perturb in fp32 and use the realised step
            pp = s.pos.copy(); pm = s.pos.copy()
            pp[a, c] += np.float32(h); pm[a, c] -= np.float32(h)
            step = float(pp[a, c]) - float(pm[a, c])
            fd = -(energy_only(s, pp, params, blob) - energy_only(s, pm, params, blob)) / step
            assert fd == pytest.approx(F[a, c], abs=2e-7, rel=2e-6)


def test_fd_error_shrinks_with_step(params):
    """E is only C^1 (CELU'' jumps at 0, f_c'' jumps at Rc), so the central-difference error falls
    between first and second order in h; it must shrink monotonically towards the analytic force."""
    s = W.make_system(2)
    blob = W.make_weights(8)
    _, F, _ = oracle.energy_forces(s.pos, s.species, None, params, blob, 8)
    a, c = 7, 1
    errs = []
    for h in (2.0 ** -6, 2.0 ** -9, 2.0 ** -12, 2.0 ** -15):
        pp = s.pos.copy(); pm = s.pos.copy()
        pp[a, c] += np.float32(h); pm[a, c] -= np.float32(h)
        step = float(pp[a, c]) - float(pm[a, c])
        fd = -(energy_only(s, pp, params, blob) - energy_only(s, pm, params, blob)) / step
        errs.append(abs(fd - F[a, c]))
    assert errs[0] > errs[1] > errs[2] > errs[3]
    assert errs[3] < 1e-6 and errs[0] / errs[3] > 8.0 ** 3


def test_forces_sum_to_zero_and_no_torque(params):
    s = W.make_system(2)
    blob = W.make_weights(8)
    _, F, _ = oracle.energy_forces(s.pos, s.species, None, params, blob, 8)
    assert np.abs(F.sum(0)).max() < 1e-12
    assert np.abs(np.cross(s.pos.astype(np.float64), F).sum(0)).max() < 1e-11
    s = W.make_system(1)
    blob = W.make_weights(1)
    _, F, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 1)
    assert np.abs(F.sum(0)).max() < 1e-12


def test_invariances_open_boundary(params):
    s = W.make_system(2)
    blob = W.make_weights(8)
    E0, F0, _ = oracle.energy_forces(s.pos, s.species, None, params, blob, 8)
    # exact operations in fp32: translation by a power of two after scaling positions to a 2^-10 grid
    q = (np.round(s.pos.astype(np.float64) * 1024) / 1024).astype(np.float32)
    E0, F0, _ = oracle.energy_forces(q, s.species, None, params, blob, 8)
    Et, Ft, _ = oracle.energy_forces(q + np.float32(8.0), s.species, None, params, blob, 8)
    assert np.allclose(Et, E0, atol=1e-13) and np.allclose(Ft, F0, atol=1e-13)
    # rotation by 90 deg about z and axis relabelling (exact in fp32)
    R = np.array([[0, -1, 0], [1, 0, 0], [0, 0, 1]], dtype=np.float32)
    Er, Fr, _ = oracle.energy_forces(q @ R.T, s.species, None, params, blob, 8)
    assert np.allclose(Er, E0, atol=1e-12) and np.allclose(Fr, F0 @ R.T.astype(np.float64), atol=1e-12)
    # relabelling atoms (any permutation of the atom order) permutes E_atom and F
    perm = np.random.default_rng(0).permutation(s.n_atoms)
    Ep, Fp, _ = oracle.energy_forces(q[perm], s.species[perm], None, params, blob, 8)
    assert np.allclose(Ep, E0[perm], atol=1e-12) and np.allclose(Fp, F0[perm], atol=1e-12)
    # generic rotation (inexact in fp32 -> compare at fp32 input resolution)
    th = 0.7
    Rg = np.array([[math.cos(th), -math.sin(th), 0], [math.sin(th), math.cos(th), 0], [0, 0, 1]])
    qr = (q.astype(np.float64) @ Rg.T).astype(np.float32)
    Eg, Fg, _ = oracle.energy_forces(qr, s.species, None, params, blob, 8)
    assert abs(Eg.sum() - E0.sum()) < 1e-4 and np.abs(Fg - F0 @ Rg.T).max() < 1e-3


def test_invariances_periodic(params):
    s = W.make_system(1)
    blob = W.make_weights(1)
    L = np.float32(16.0)                                      # power-of-two box so that image shifts are exact
    q = (np.round(s.pos.astype(np.float64) * 256) / 256).astype(np.float32)
    box = np.array([L, L, L], np.float32)
    E0, F0, _ = oracle.energy_forces(q, s.species, box, params, blob, 1)
    q2 = q.copy(); q2[::2] += L; q2[1::5, 1] -= 2 * L
    E1, F1, _ = oracle.energy_forces(q2, s.species, box, params, blob, 1)
    assert np.allclose(E1, E0, atol=1e-13) and np.allclose(F1, F0, atol=1e-13)
    E2, F2, _ = oracle.energy_forces(q[:, [2, 0, 1]], s.species, box, params, blob, 1)   # axis permutation
    assert np.allclose(E2, E0, atol=1e-12) and np.allclose(F2, F0[:, [2, 0, 1]], atol=1e-12)


def test_dimer_force_vanishes_smoothly_at_cutoff(params):
    blob = W.make_weights(1)
    sp = np.array([0, 3], np.int32)
    mags = []
    for r in (5.0, 5.05, 5.09, 5.0999):
        _, F, _ = oracle.energy_forces(np.array([[0, 0, 0], [r, 0, 0]], np.float32), sp, None, params, blob, 1)
        assert abs(F[0, 0] + F[1, 0]) < 1e-15 and np.all(F[:, 1:] == 0)
        mags.append(abs(F[0, 0]))
    assert mags[0] > mags[1] > mags[2] > mags[3] and mags[3] < 1e-7
    _, F, _ = oracle.energy_forces(np.array([[0, 0, 0], [5.1001, 0, 0]], np.float32), sp, None, params, blob, 1)
    assert np.all(F == 0.0)


def test_partial_centres_give_exact_forces_on_interior_atom(params):
    """The sampled-force check used at full size: F_a only needs the centres within Rcr of a."""
    s = W.small_periodic_mix(400, 16.0, seed=9, n_models=2)
    blob = W.make_weights(2)
    _, F, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 2)
    rp, col = oracle.pairs(s.pos, s.box, 5.1)
    a = 17
    centres = np.concatenate([[a], col[rp[a]:rp[a + 1]]]).astype(np.int32)
    _, Fa, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 2, centres=centres)
    assert np.allclose(Fa[a], F[a], atol=1e-13)


def test_partial_centres_are_additive_and_local(params):
    """Eq. 2: E is a sum of atomic terms, so the oracle restricted to a subset of central atoms - the
    ground truth of the partial-evaluation (multi-GPU) tests - must be additive over any partition of the atoms, give the
    same atomic energies as the full evaluation, and a single centre may push only itself and its neighbours."""
    s = W.small_periodic_mix(300, 15.0, seed=3, n_models=1)
    blob = W.make_weights(1)
    E, F, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 1)
    rng = np.random.default_rng(1)
    owner = rng.integers(0, 3, s.n_atoms)
    Esum, Fsum = 0.0, np.zeros_like(F)
    for r in range(3):
        c = np.nonzero(owner == r)[0].astype(np.int32)
        Ec, Fc, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 1, centres=c)
        assert np.allclose(Ec, E[c], atol=1e-14)                 # the same atomic energies, centre by centre
        Esum += Ec.sum()
        Fsum += Fc
    assert abs(Esum - E.sum()) < 1e-11 and np.abs(Fsum - F).max() < 1e-12
    rp, col = oracle.pairs(s.pos, s.box, 5.1)
    _, F1, _ = oracle.energy_forces(s.pos, s.species, s.box, params, blob, 1, centres=np.array([42], np.int32))
    touched = set(np.nonzero(np.abs(F1).sum(1))[0])
    assert touched <= set(col[rp[42]:rp[43]]) | {42}
    assert np.abs(F1.sum(0)).max() < 1e-13                       # Newton's third law holds centre by centre


def test_batched_molecules_are_independent(params):
    s = W.replicas_1024x30(n_mol=4)
    blob = W.make_weights(8)
    E, F = oracle.total_energy_forces(s, params, blob)
    assert E.shape == (4,)
    for m in range(4):
        Em, Fm, _ = oracle.energy_forces(s.pos[30 * m:30 * m + 30], s.species[30 * m:30 * m + 30], None, params, blob, 8)
        assert Em.sum() == pytest.approx(E[m], abs=1e-12)
        assert np.allclose(Fm, F[30 * m:30 * m + 30], atol=1e-13)


# ------------------------------------------------------------------ composition (Eq. 2; ensemble L159, Q11)
@pytest.mark.parametrize("cfg", [2, 1])
def test_energy_forces_composes_mlp_of_aev(params, cfg):
    """`energy_forces` has its own ensemble loop (network selection by the central atom's species, 1/n_models on E and
    on dE/dG).  `oracle.mlp` is tied to torch autograd above and `oracle.aev` to the closed forms, so
    energy_forces == mlp(aev) pins "one network per element" and the ensemble mean (L159, Q11):
    a dropped 1/n_models or a wrong network index fails here."""
    s = W.make_system(cfg)
    blob = W.make_weights(s.n_models)
    E, _, g = oracle.energy_forces(s.pos, s.species, s.box, params, blob, s.n_models, want_dEdG=True)
    rows = oracle.aev(s.pos, s.species, s.box, params)
    E2, g2 = oracle.mlp(rows, s.species, blob, s.n_models, params)
    assert np.allclose(E, E2, rtol=0, atol=1e-12)
    assert np.allclose(g, g2, rtol=0, atol=1e-12)
    # and against torch autograd directly on a few centres of different species (not through oracle.mlp)
    pick = [int(np.nonzero(s.species == sp)[0][0]) for sp in sorted(set(s.species.tolist()))]
    Et, gt = torch_mlp(rows[pick], s.species[pick], blob, s.n_models, float(np.float32(0.1)))
    assert np.allclose(E[pick], Et, rtol=0, atol=1e-12)
    assert np.allclose(g[pick], gt, rtol=0, atol=1e-12)


def test_forces_follow_from_dEdG_by_finite_differences_of_the_aev(params):
    """F = -sum_i g_i . dG_i/dr with g_i from the (pinned) network gradient: contract oracle.mlp's dE/dG with central
    finite differences of oracle.aev rows - the chain rule of centre_forces without using energy_forces' own energy."""
    s = W.make_system(2)
    blob = W.make_weights(8)
    _, F, _ = oracle.energy_forces(s.pos, s.species, None, params, blob, 8)
    rows = oracle.aev(s.pos, s.species, None, params)
    _, g = oracle.mlp(rows, s.species, blob, 8, params)
    h = 2.0 ** -14
    for a, c in ((5, 0), (23, 2)):
        pp = s.pos.copy(); pm = s.pos.copy()
        pp[a, c] += np.float32(h); pm[a, c] -= np.float32(h)
        step = float(pp[a, c]) - float(pm[a, c])
        dG = (oracle.aev(pp, s.species, None, params) - oracle.aev(pm, s.species, None, params)) / step
        assert -(g * dG).sum() == pytest.approx(F[a, c], abs=5e-7, rel=5e-6)
