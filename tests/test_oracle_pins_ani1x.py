"""Pins of the fp64 oracle on the ANI-1x / ANI-1ccx SHAPE ("ANI-1x ... H, C, N, and O",
L73 "R_c ... fixed to 5.2 Å", L159: the paper's second benchmarked model).  The oracle's angular grid is a runtime field
(n_a x n_z = 4 x 8 here instead of 8 x 4); parameters are DESIGN.md reading R4.  Same kinds of pin as the ANI-2x shape:
closed forms stored in tests/golden/ani1x_closed_form.txt, torch autograd for the network, finite differences.
Runs with -m "not gpu"."""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2207_14276_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
RAD = 112


def golden():
    out = {}
    with open(os.path.join(HERE, "golden", "ani1x_closed_form.txt")) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out


G = golden()


@pytest.fixture(scope="module")
def p1x():
    return W.ani1x_params()


def pairidx(u, v):
    u, v = min(u, v), max(u, v)
    return 7 * u - u * (u - 1) // 2 + (v - u)


def trimer(r1, r2, theta):
    return np.array([[0, 0, 0], [r1, 0, 0], [r2 * math.cos(theta), r2 * math.sin(theta), 0]], dtype=np.float32)


def test_feature_count_384(p1x):
    """N radial + N(N+1)/2 angular sub-AEVs; N = 4 -> 4*16 + 10*32 = 384, a sub-vector of the 1008 layout."""
    assert W.ANI1X_AEV_DIM == 4 * 16 + 10 * 32 == 384
    fmap = W.ani1x_feature_map()
    assert fmap.size == 384 and len(set(fmap.tolist())) == 384
    s = W.small_periodic_mix(300, 14.5, seed=4, hcno_only=True)
    assert set(s.species.tolist()) == {0, 1, 2, 3}
    a = oracle.aev(s.pos, s.species, s.box, p1x)
    nz = np.nonzero((a != 0).any(axis=0))[0]
    assert set(nz.tolist()) <= set(fmap.tolist())          # nothing outside the 384 columns
    assert nz.size > 300                                   # and nearly all of them are exercised


@pytest.mark.parametrize("sj", [0, 3])
def test_dimer_radial_closed_form(p1x, sj):
    pos = np.array([[0, 0, 0], [1.0, 0, 0]], dtype=np.float32)
    a = oracle.aev(pos, np.array([1, sj], np.int32), None, p1x)
    blk = a[0, 16 * sj:16 * sj + 16]
    for m in range(5):
        assert blk[m] == pytest.approx(G[f"rad_R1.0_m{m}"], rel=3e-6)
    mask = np.ones(1008, bool)
    mask[16 * sj:16 * sj + 16] = False
    assert np.all(a[0, mask] == 0.0)
    # R = ShfR_0: the Gaussian is 1, the entry is f_c(0.9; 5.2); and the cutoff is 5.2, not 5.1
    a = oracle.aev(np.array([[0, 0, 0], [0, 0.9, 0]], np.float32), np.array([0, 0], np.int32), None, p1x)
    assert a[0, 0] == pytest.approx(G["fc_0.9_rc5.2"], rel=1e-6)
    a = oracle.aev(np.array([[0, 0, 0], [5.15, 0, 0]], np.float32), np.array([0, 0], np.int32), None, p1x)
    assert a[0].sum() > 0
    a = oracle.aev(np.array([[0, 0, 0], [5.2001, 0, 0]], np.float32), np.array([0, 0], np.int32), None, p1x)
    assert np.all(a == 0.0)


def test_trimer_isosceles_peak_on_the_4x8_grid(p1x):
    r = float(p1x.shf_a[1])
    for z in range(8):
        a = oracle.aev(trimer(r, r, float(p1x.shf_z[z])), np.array([1, 0, 0], np.int32), None, p1x)
        blk = a[0, RAD + 32 * pairidx(0, 0):RAD + 32 * pairidx(0, 0) + 32].reshape(4, 8)      # [a][z]
        assert blk[1, z] == pytest.approx(G["ang_iso_R1.55"], rel=5e-6)
        assert blk[1, z] == blk.max()


@pytest.mark.parametrize("sj,sk", [(0, 0), (0, 3), (3, 0), (1, 2)])
def test_trimer_general_closed_form(p1x, sj, sk):
    a = oracle.aev(trimer(1.0, 1.2, math.radians(100.0)), np.array([2, sj, sk], np.int32), None, p1x)
    p = pairidx(sj, sk)
    blk = a[0, RAD + 32 * p:RAD + 32 * p + 32].reshape(4, 8)
    for q in range(2):
        for z in range(8):
            assert blk[q, z] == pytest.approx(G[f"ang_gen_a{q}_z{z}"], rel=5e-6, abs=1e-16)
    ang = a[0, RAD:].copy()
    ang[32 * p:32 * p + 32] = 0
    assert np.all(ang == 0.0)


def test_embedded_network_equals_the_native_384_160_128_96_network():
    """`workloads.embed_ani1x` places the ANI-1x-shaped networks in the library's fixed 1008-256-192-160 layout with zero
    padding; CELU(0) = 0, so the padded network must reproduce the native one and its input gradient exactly.  The
    native network is evaluated by torch autograd in fp64 (not by the oracle)."""
    import torch
    torch.set_num_threads(4)
    rng = np.random.default_rng(8)
    blob1 = W.make_weights_ani1x(2)
    big = W.embed_ani1x(blob1, 2)
    fmap = W.ani1x_feature_map()
    x384 = rng.uniform(0, 1, (8, 384))
    x1008 = np.zeros((8, 1008))
    x1008[:, fmap] = x384
    sp = np.array([0, 1, 2, 3, 0, 1, 2, 3], np.int32)
    E, g = oracle.mlp(x1008, sp, big, 2, W.ani1x_params())
    xt = torch.tensor(x384, dtype=torch.float64, requires_grad=True)
    tot = []
    for r in range(8):
        acc = 0.0
        for e in range(2):
            W1, b1, W2, b2, W3, b3, W4, b4 = [torch.tensor(np.asarray(t), dtype=torch.float64)
                                              for t in W.split_net_ani1x(blob1, e, int(sp[r]))]
            h = torch.nn.functional.celu(torch.nn.functional.linear(xt[r], W1, b1), 0.1 * 1.0)
            h = torch.nn.functional.celu(torch.nn.functional.linear(h, W2, b2), 0.1)
            h = torch.nn.functional.celu(torch.nn.functional.linear(h, W3, b3), 0.1)
            acc = acc + torch.nn.functional.linear(h, W4, b4)[0]
        tot.append(acc / 2)
    Et = torch.stack(tot)
    Et.sum().backward()
    alpha32 = float(np.float32(0.1))                       # the oracle reads alpha as the fp32 value
    assert np.allclose(E, Et.detach().numpy(), rtol=0, atol=5e-8 + abs(alpha32 - 0.1))
    assert np.allclose(g[:, fmap], xt.grad.numpy(), rtol=0, atol=1e-7)
    off = np.ones(1008, bool)
    off[fmap] = False
    assert np.all(g[:, off] == 0.0)                        # no gradient leaks into the other 624 columns


def test_forces_equal_minus_finite_difference_gradient_on_the_4x8_grid(p1x):
    s = W.small_periodic_mix(200, 12.8, seed=6, n_models=1, hcno_only=True)
    blob = W.embed_ani1x(W.make_weights_ani1x(1), 1)
    _, F, _ = oracle.energy_forces(s.pos, s.species, s.box, p1x, blob, 1)
    assert np.abs(F.sum(0)).max() < 1e-12
    h = 2.0 ** -16
    for a in (3, 77, 150):
        for c in range(3):
            pp = s.pos.copy(); pm = s.pos.copy()
            pp[a, c] += np.float32(h); pm[a, c] -= np.float32(h)
            step = float(pp[a, c]) - float(pm[a, c])
            Ep = oracle.energy_forces(pp, s.species, s.box, p1x, blob, 1)[0].sum()
            Em = oracle.energy_forces(pm, s.species, s.box, p1x, blob, 1)[0].sum()
            assert -(Ep - Em) / step == pytest.approx(F[a, c], abs=2e-7, rel=2e-6)
