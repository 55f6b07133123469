"""dhp_kinetic_energy_static (include/dhp.h): the one entry point of libdhp.so that allocates nothing.

It exists for code that cannot call cudaMalloc - a plug-in working inside the memory an MD engine reserved for it, a
diagnostic inside a running loop where an allocation would stall the device, a process whose allocator owns the GPU - so it
takes no context and no handle, and its working memory is a fixed array inside the library that every call on a GPU shares.
What is checked here, on two calls in a row each time (the second call finds the first call's leftovers in that array):
the result equals the kinetic energy the existing path reports (dhp_md_run's E_out[2], accumulated in memory that
dhp_md_create allocated) within the tolerance test_gpu_md.py uses for that number, and far inside it, since both are fp64
sums of the same terms; a short call after a long one is not polluted by the long one's partial sums; sizes above the
limit are refused.  The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It passes alone in a fresh process (the first call on the device is then the one that looks up
the array's address) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2207_14276_b200 import workloads as W

pytestmark = pytest.mark.gpu

REL_TOL = 1e-4        # tests/test_gpu_md.py: |E_kin - oracle| <= 1e-4 E_kin
REL_TIGHT = 1e-12     # same terms, fp64 additions in another order


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2207_14276_b200 import binding
    return binding


def existing_path_kinetic(B, torch, s, md, params, vel):
    """E_out[2] of dhp_md_run with zero steps: the kinetic energy at the velocities passed in (k_md_kinetic, accumulator owned
    by the dhp_md handle)."""
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(W.make_weights(1), 1)
    pos = torch.from_numpy(s.pos.copy()).cuda()
    sp = torch.from_numpy(s.species).cuda()
    h = d.dhp_md_create(md.inv_mass)
    E = d.dhp_md_run(h, pos, vel, s.box, sp, w, 0.2, 1, 0)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    out = float(E.cpu().numpy()[2])
    d.dhp_md_destroy(h)
    d.close()
    return out


@pytest.mark.parametrize("system", ["water96", "mix600"])
def test_two_calls_in_a_row_match_the_existing_path(torch, B, params, system):
    s = W.make_system(1) if system == "water96" else W.small_periodic_mix(600, n_models=1)     # 1 block / 3 blocks, ragged tail
    md = W.md_inputs(s)
    inv_mass = torch.from_numpy(md.inv_mass).cuda()
    vel_a = torch.from_numpy(md.vel.copy()).cuda()
    vel_b = torch.from_numpy((1.5 * md.vel[::-1]).astype(np.float32).copy()).cuda()         # other numbers for the second call
    E_kin = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    B.dhp_kinetic_energy_static(vel_a, inv_mass, E_kin[0:1])
    B.dhp_kinetic_energy_static(vel_b, inv_mass, E_kin[1:2])                                # same stream: ordered after the first
    torch.cuda.synchronize()
    got = E_kin.cpu().numpy()
    for g, vel in zip(got, (vel_a, vel_b)):
        want = existing_path_kinetic(B, torch, s, md, params, vel)
        assert want > 0.0
        assert abs(g - want) <= REL_TOL * want
        assert abs(g - want) <= REL_TIGHT * want


def test_short_call_after_long_call_and_repeatability(torch, B):
    rng = np.random.default_rng(20)
    n_long, n_short = 300001, 700                        # 1172 blocks (more partials than the summing block has threads), then 3
    vel = rng.normal(0.0, 0.01, (n_long, 3)).astype(np.float32)
    inv_mass = (0.2625499639 / rng.choice(np.array([1.008, 12.011, 14.007, 15.999]), n_long)).astype(np.float32)
    want = lambda n: float((0.5 * (vel[:n].astype(np.float64) ** 2).sum(1) / inv_mass[:n].astype(np.float64)).sum())
    v, m = torch.from_numpy(vel).cuda(), torch.from_numpy(inv_mass).cuda()
    E = torch.zeros(4, dtype=torch.float64, device="cuda")
    B.dhp_kinetic_energy_static(v, m, E[0:1])
    B.dhp_kinetic_energy_static(v[:n_short].contiguous(), m[:n_short].contiguous(), E[1:2])
    B.dhp_kinetic_energy_static(v, m, E[2:3])
    B.dhp_kinetic_energy_static(v[:0].contiguous(), m[:0].contiguous(), E[3:4])             # no atoms: 0, nothing launched
    torch.cuda.synchronize()
    e = E.cpu().numpy()
    assert abs(e[0] - want(n_long)) <= REL_TIGHT * want(n_long)
    assert abs(e[1] - want(n_short)) <= REL_TIGHT * want(n_short)
    assert e[2] == e[0]                                  # block partials are added in block order: same bits
    assert e[3] == 0.0


def test_sizes_beyond_the_fixed_array_are_refused(torch, B):
    lib = B.load_library()
    small = torch.zeros(8, dtype=torch.float64, device="cuda")
    too_many = B.KINETIC_STATIC_MAX_ATOMS + 1
    rc = lib.dhp_kinetic_energy_static(C.c_void_p(small.data_ptr()), C.c_void_p(small.data_ptr()), too_many,
                                       C.c_void_p(small.data_ptr()), None)                  # refused before any pointer is used
    assert rc == -2 and b"capacity" in lib.dhp_strerror(rc)
    assert lib.dhp_kinetic_energy_static(None, None, 5, C.c_void_p(small.data_ptr()), None) == -1
    assert lib.dhp_kinetic_energy_static(C.c_void_p(small.data_ptr()), C.c_void_p(small.data_ptr()), 1, None, None) == -1
    with pytest.raises(B.DhpError, match="at most"):
        B.dhp_kinetic_energy_static(torch.zeros((too_many, 3), dtype=torch.float32, device="cuda"),
                                    torch.ones(too_many, dtype=torch.float32, device="cuda"), small[0:1])
