"""The multiple-timestep driver (include/dhp.h: dhp_md_run; §2.3.5, Eqs. 8-9) against the fp64 oracle
integrator oracle/md_oracle.py driven by the fp64 ANI oracle: same inputs, same number of steps, trajectories compared
atom by atom.  Tolerances: the GPU integrates in fp32 (positions ~ 15 Å: 1 ulp = 1e-6 Å, a handful of roundings per
step), forces carry <= 5e-5 Hartree/Å (measured ~ 2e-6) x inv_mass 0.26 x dt: |dx| <= 2e-5 Å, |dv| <= 5e-6 Å/fs after
ten inner steps."""
import numpy as np
import pytest

import oracle
from oracle import md_oracle as M
from paper_2207_14276_b200 import workloads as W

pytestmark = pytest.mark.gpu

X_TOL, V_TOL = 2e-5, 5e-6


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2207_14276_b200 import binding
    return binding


def oracle_run(s, md, params, blob, dt, n_inner, n_steps, bonds=True):
    slow = lambda x: (lambda E, F: (float(E.sum()), F.astype(np.float64)))(
        *oracle.energy_forces(x.astype(np.float32), s.species, s.box, params, blob, s.n_models)[:2])
    fast = (lambda x: M.bond_energy_forces(x, s.box, md.bonds, md.bond_k.astype(np.float64), md.bond_r0.astype(np.float64))) \
        if bonds and len(md.bonds) else None
    return M.respa_run(s.pos, md.vel, md.inv_mass, slow, fast, dt, n_inner, n_steps)


def gpu_run(B, torch, s, md, params, blob, dt, n_inner, chunks, skin=0.0, mode=None, bonds=True):
    d = B.Dhp(s.n_atoms, params=params)
    if mode is not None:
        d.dhp_set_mlp_mode(mode)
    if skin:
        d.dhp_set_skin(skin)
    w = d.dhp_weights_load(blob, s.n_models)
    pos = torch.from_numpy(s.pos.copy()).cuda()
    vel = torch.from_numpy(md.vel.copy()).cuda()
    sp = torch.from_numpy(s.species).cuda()
    h = d.dhp_md_create(md.inv_mass, md.bonds, md.bond_k, md.bond_r0) if bonds and len(md.bonds) else d.dhp_md_create(md.inv_mass)
    for n in chunks:
        E = d.dhp_md_run(h, pos, vel, s.box, sp, w, dt, n_inner, n)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    out = pos.cpu().numpy(), vel.cpu().numpy(), E.cpu().numpy(), d.dhp_nlist_rebuild_count()
    d.dhp_md_destroy(h)
    d.close()
    return out


@pytest.mark.parametrize("mode", [1, 2])
def test_respa_trajectory_water96(torch, B, params, mode):
    s = W.make_system(1)
    blob = W.make_weights(1)
    md = W.md_inputs(s)
    xo, vo, Eo = oracle_run(s, md, params, blob, 0.2, 2, 5)
    x, v, E, _ = gpu_run(B, torch, s, md, params, blob, 0.2, 2, [5], mode=mode)
    assert np.abs(x - xo).max() <= X_TOL and np.abs(v - vo).max() <= V_TOL
    assert abs(E[0] - Eo[0]) / s.n_atoms <= 1e-6                       # E_ANI at the final positions
    assert abs(E[1] - Eo[1]) <= 1e-5 + 1e-4 * abs(Eo[1])               # bond energy (fp32 distances)
    assert abs(E[2] - Eo[2]) <= 1e-4 * Eo[2]                           # kinetic energy
    # the forces at the current positions are carried between runs: 3 + 2 steps == 5 steps
    x2, v2, E2, _ = gpu_run(B, torch, s, md, params, blob, 0.2, 2, [3, 2], mode=mode)
    assert np.abs(x2 - xo).max() <= X_TOL and np.abs(v2 - vo).max() <= V_TOL
    # with list reuse: same trajectory, one full build for the 6 evaluations
    x3, v3, E3, nb = gpu_run(B, torch, s, md, params, blob, 0.2, 2, [5], skin=1.0, mode=mode)
    assert nb == 1
    assert np.abs(x3 - xo).max() <= X_TOL and np.abs(v3 - vo).max() <= V_TOL and abs(E3[0] - Eo[0]) / s.n_atoms <= 1e-6


def test_velocity_verlet_without_bonds_mixed_box(torch, B, params):
    """No fast part: plain velocity Verlet (the paper's benchmark integrator) on a 7-species periodic box."""
    s = W.small_periodic_mix(600, 18.3, seed=77, n_models=2)
    blob = W.make_weights(2)
    md = W.md_inputs(s)
    assert len(md.bonds) == 0
    xo, vo, Eo = oracle_run(s, md, params, blob, 0.1, 1, 4)
    x, v, E, nb = gpu_run(B, torch, s, md, params, blob, 0.1, 3, [4], skin=0.6)      # n_inner is ignored without bonds
    assert nb == 1
    assert np.abs(x - xo).max() <= X_TOL and np.abs(v - vo).max() <= V_TOL
    assert abs(E[0] - Eo[0]) / s.n_atoms <= 1e-6 and E[1] == 0.0 and abs(E[2] - Eo[2]) <= 1e-4 * Eo[2]


def test_long_run_rebuilds_when_atoms_leave_the_skin(torch, B, params):
    """40 outer steps with a thin skin: the device-side displacement check must trigger rebuilds on its own, and the
    final state must still match a run without any reuse."""
    s = W.make_system(1)
    blob = W.make_weights(1)
    md = W.md_inputs(s, temperature=600.0)
    x0, v0, E0, _ = gpu_run(B, torch, s, md, params, blob, 0.25, 1, [40], bonds=False)
    x1, v1, E1, nb = gpu_run(B, torch, s, md, params, blob, 0.25, 1, [40], skin=0.1, bonds=False)
    assert 2 <= nb <= 41
    assert np.abs(x1 - x0).max() <= 1e-4 and abs(E1[0] - E0[0]) / s.n_atoms <= 1e-6
    print(f"rebuilds with skin 0.1 over 40 steps: {nb}; max |x - x0| = {np.abs(x1 - s.pos).max():.3f} A")


def test_nve_energy_conservation_and_time_reversal(torch, B, params):
    """Properties that need no oracle value: the total energy E_ANI + E_bonds + E_kin of an NVE run fluctuates at O(dt^2)
    (second-order symplectic scheme: halving the timestep must shrink the error about fourfold), and integrating forward,
    flipping the velocities and integrating the same number of steps returns to the start (to fp32 round-off)."""
    s = W.make_system(1)
    blob = W.make_weights(1)
    md = W.md_inputs(s)
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(blob, 1)
    sp = torch.from_numpy(s.species).cuda()
    h = d.dhp_md_create(md.inv_mass, md.bonds, md.bond_k, md.bond_r0)

    def run(dt, n_outer, pos0, vel0):
        pos = torch.from_numpy(pos0.copy()).cuda()
        vel = torch.from_numpy(vel0.copy()).cuda()
        d.dhp_md_reset(h)
        E0 = d.dhp_md_run(h, pos, vel, s.box, sp, w, dt, 2, 0).cpu().numpy().sum()
        worst = 0.0
        for _ in range(n_outer // 4):
            E = d.dhp_md_run(h, pos, vel, s.box, sp, w, dt, 2, 4).cpu().numpy().sum()
            worst = max(worst, abs(E - E0))
        return worst, pos.cpu().numpy(), vel.cpu().numpy()

    e1, x1, v1 = run(0.2, 40, s.pos, md.vel)            # 8 fs
    e2, _, _ = run(0.1, 80, s.pos, md.vel)              # the same 8 fs at half the timestep
    kin0 = M.kinetic_energy(md.vel, md.inv_mass)
    print(f"NVE water96, 8 fs: max |dE_tot| = {e1:.3e} Ha (dt 0.2 fs), {e2:.3e} Ha (dt 0.1 fs); E_kin(0) = {kin0:.3e} Ha")
    assert e2 < 0.5 * e1 and e1 < 0.2 * kin0
    _, x0, v0 = run(0.2, 40, x1, -v1)
    assert np.abs(x0 - s.pos).max() < 5e-4 and np.abs(v0 + md.vel).max() < 5e-5
    d.dhp_md_destroy(h)
    d.close()


def test_argument_errors_of_the_driver_and_the_skin(torch, B, params):
    s = W.make_system(1)
    md = W.md_inputs(s)
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(W.make_weights(1), 1)
    for bad in (-0.1, 4.5, float("nan")):
        with pytest.raises(B.DhpError, match="-1"):
            d.dhp_set_skin(bad)
    with pytest.raises(B.DhpError, match="-2"):                       # more atoms than the context holds
        d.dhp_md_create(np.ones(s.n_atoms + 1, np.float32))
    with pytest.raises(B.DhpError, match="-1"):                       # bonds without force constants
        import ctypes as C
        h = C.c_void_p()
        rc = d.lib.dhp_md_create(d.ctx, s.n_atoms, C.c_void_p(md.inv_mass.ctypes.data), C.c_void_p(md.bonds.ctypes.data), None, None,
                                 len(md.bonds), C.byref(h))
        B._check(rc, d.ctx)
    h = d.dhp_md_create(md.inv_mass, md.bonds, md.bond_k, md.bond_r0)
    pos = torch.from_numpy(s.pos.copy()).cuda()
    vel = torch.from_numpy(md.vel.copy()).cuda()
    sp = torch.from_numpy(s.species).cuda()
    for dt, n_inner, n_steps in ((0.0, 1, 1), (0.5, 0, 1), (0.5, 1, -1)):
        with pytest.raises(B.DhpError, match="-1"):
            d.dhp_md_run(h, pos, vel, s.box, sp, w, dt, n_inner, n_steps)
    E = d.dhp_md_run(h, pos, vel, s.box, sp, w, 0.5, 1, 0)            # zero steps: energies of the initial state
    torch.cuda.synchronize()
    assert np.isfinite(E.cpu().numpy()).all() and np.array_equal(pos.cpu().numpy(), s.pos)
    d.dhp_md_destroy(h)
    d.close()


def test_sharded_driver_on_one_rank_equals_the_oracle_trajectory(torch, B, params):
    """shard.ShardedMd (dhp_md_open -> all-gather -> dhp_ani_energy_forces_partial over the own slab -> reduce-scatter ->
    dhp_md_close) on the one GPU there is: world size 1 takes the same code path with the collectives
    reduced to copies, and must reproduce the oracle trajectory like dhp_md_run does.  (World size 2 runs on gloo with an
    oracle-backed stand-in: tests/test_shard_gloo.py.)"""
    from paper_2207_14276_b200 import shard
    s = W.make_system(1)
    md = W.md_inputs(s)
    blob = W.make_weights(1)
    d = B.Dhp(s.n_atoms, params=params)
    w = d.dhp_weights_load(blob, 1)
    pos = torch.from_numpy(s.pos.copy()).cuda()
    vel = torch.from_numpy(md.vel.copy()).cuda()
    sp = torch.from_numpy(s.species).cuda()
    drv = shard.ShardedMd(d, w, sp, s.box, shard.owner_bounds(s.n_atoms, 1, unit=3), md.inv_mass, md.bonds, md.bond_k, md.bond_r0,
                          mask_every=2)
    E = drv.run(pos, vel, 0.5, 2, 3)
    E = drv.run(pos, vel, 0.5, 2, 2)
    torch.cuda.synchronize()
    assert d.dhp_status() == 0
    xo, vo, (Es, _, _) = oracle_run(s, md, params, blob, 0.5, 2, 5)
    assert np.max(np.abs(pos.cpu().numpy() - xo)) <= X_TOL and np.max(np.abs(vel.cpu().numpy() - vo)) <= V_TOL
    assert abs(E.item() - Es) / s.n_atoms <= 1e-6
    # an owned sub-range: only those rows move
    pos2 = torch.from_numpy(s.pos.copy()).cuda()
    vel2 = torch.from_numpy(md.vel.copy()).cuda()
    h = d.dhp_md_create(md.inv_mass)
    F = torch.from_numpy(np.random.default_rng(5).normal(size=(s.n_atoms, 3)).astype(np.float32)).cuda()
    d.dhp_md_open(h, pos2, vel2, s.box, F, 0.5, 1, 30, 90)
    with pytest.raises(B.DhpError):                         # close completes the step open began: same dt, same n_inner
        d.dhp_md_close(h, vel2, F, 0.25, 1, 30, 90)
    d.dhp_md_close(h, vel2, F, 0.5, 1, 30, 90)
    with pytest.raises(B.DhpError):                         # nothing is open any more
        d.dhp_md_close(h, vel2, F, 0.5, 1, 30, 90)
    with pytest.raises(B.DhpError):                         # buffers the C ABI would misread
        d.dhp_md_open(h, pos2.double(), vel2, s.box, F, 0.5, 1, 30, 90)
    torch.cuda.synchronize()
    moved = np.nonzero(np.abs(pos2.cpu().numpy() - s.pos).sum(1))[0]
    assert moved.min() == 30 and moved.max() == 89
    dv = vel2.cpu().numpy() - md.vel
    assert np.all(dv[:30] == 0) and np.all(dv[90:] == 0)
    assert np.allclose(dv[30:90], 0.5 * md.inv_mass[30:90, None] * F.cpu().numpy()[30:90], rtol=1e-5, atol=5e-9)   # fp32 rounding of v
    with pytest.raises(B.DhpError):
        d.dhp_md_open(h, pos2, vel2, s.box, F, 0.5, 1, 90, 30)
    d.dhp_md_destroy(h)
    d.close()


def test_sharded_driver_on_a_one_rank_nccl_group(torch, B, params):
    """The NCCL branch of shard.Exchange - reduce_scatter_tensor and all_gather_into_tensor on CUDA tensors, on the stream the
    kernels run on - executed on the one GPU there is: on a process group of ONE rank both collectives are legal and are the
    identity.  First the exchange alone, then shard.ShardedMd on that group with list reuse on (partial call + Verlet skin +
    graph replay together, what every step of a sharded run does) against the oracle trajectory."""
    import socket
    import torch.distributed as dist
    from paper_2207_14276_b200 import shard
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    assert not dist.is_initialized()
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1)
    try:
        s = W.make_system(1)
        md = W.md_inputs(s)
        blob = W.make_weights(1)
        bounds = shard.owner_bounds(s.n_atoms, 1, unit=3)
        ex = shard.Exchange(bounds, torch.device("cuda:0"))
        assert ex.live and ex.backend == "nccl" and ex.chunk == s.n_atoms
        rng = np.random.default_rng(8)
        part = torch.from_numpy(rng.normal(size=(s.n_atoms, 3)).astype(np.float32)).cuda()
        tot = torch.zeros_like(part)
        for _ in range(2):                                    # second call: the kept buffers
            ex.reduce_scatter_forces(part, tot)
            assert torch.equal(tot, part)
        x = torch.from_numpy(rng.normal(size=(s.n_atoms, 3)).astype(np.float32)).cuda()
        x0 = x.clone()
        ex.all_gather_positions(x)
        assert torch.equal(x, x0)
        e = torch.tensor([1.25], dtype=torch.float64, device="cuda")
        assert ex.all_reduce_energy(e).item() == 1.25
        # the driver on the same group
        d = B.Dhp(s.n_atoms, params=params)
        d.dhp_set_skin(1.0)
        w = d.dhp_weights_load(blob, 1)
        pos = torch.from_numpy(s.pos.copy()).cuda()
        vel = torch.from_numpy(md.vel.copy()).cuda()
        sp = torch.from_numpy(s.species).cuda()
        drv = shard.ShardedMd(d, w, sp, s.box, bounds, md.inv_mass, md.bonds, md.bond_k, md.bond_r0, mask_every=2)
        r0 = d.dhp_graph_replays()
        E = drv.run(pos, vel, 0.5, 2, 5)
        torch.cuda.synchronize()
        assert d.dhp_status() == 0
        assert d.dhp_graph_replays() - r0 >= 3                # same E / F / mask addresses every step: the call is replayed
        assert 1 <= d.dhp_nlist_rebuild_count() < 6           # the list was reused on some steps at least
        xo, vo, (Es, _, _) = oracle_run(s, md, params, blob, 0.5, 2, 5)
        assert np.max(np.abs(pos.cpu().numpy() - xo)) <= X_TOL and np.max(np.abs(vel.cpu().numpy() - vo)) <= V_TOL
        assert abs(E.item() - Es) / s.n_atoms <= 1e-6
        d.close()
    finally:
        dist.destroy_process_group()
