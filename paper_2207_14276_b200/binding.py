"""Thin ctypes binding over the C ABI of libdhp.so (include/dhp.h) — argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; PyTorch is used here only to own
device memory and the stream.  There is NO CPU fallback: if the library is missing or no CUDA device is
present, calls raise.  Function names are those of the C ABI; `Dhp` is a small convenience object that
keeps a context and marshals torch tensors / numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libdhp.so")

N_PHASES = 6
PHASES = ("nlist", "aev_fwd", "mlp_g1", "mlp_mid", "mlp_b1", "aev_bwd")
MLP_AUTO, MLP_SIMT, MLP_TENSOR, MLP_TENSOR_LAYERWISE, MLP_TENSOR_FP16 = 0, 1, 2, 3, 4
OK = 0

# every symbol include/dhp.h declares: (name, restype, argtypes)
_vp, _i64, _i32, _f32 = C.c_void_p, C.c_int64, C.c_int, C.c_float
SYMBOLS = {
    "dhp_create": (C.c_int, [C.POINTER(_vp), _vp, _i64, _i64, _vp]),
    "dhp_destroy": (C.c_int, [_vp]),
    "dhp_weights_load": (C.c_int, [_vp, _vp, _i64, _i32, C.POINTER(_vp)]),
    "dhp_weights_free": (C.c_int, [_vp, _vp]),
    "dhp_nlist_build": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _vp, _i64, _f32, C.POINTER(_vp)]),
    "dhp_set_skin": (C.c_int, [_vp, _f32]),
    "dhp_nlist_rebuild_count": (_i64, [_vp]),
    "dhp_nlist_sizes": (C.c_int, [_vp, _vp, C.POINTER(_i64), C.POINTER(_i64)]),
    "dhp_nlist_export": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "dhp_ani_energy_forces": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _vp, _i64, _vp, _i32, _vp, _vp]),
    "dhp_ani_energy_forces_partial": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _vp, _i64, _vp, _i32, _vp, _vp, _vp]),
    "dhp_ani_energy": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _vp, _i64, _vp, _i32, _vp]),
    "dhp_ani_energy_forces_host": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _vp, _i64, _vp, _i32, _vp, _vp]),
    "dhp_md_create": (C.c_int, [_vp, _i64, _vp, _vp, _vp, _vp, _i64, C.POINTER(_vp)]),
    "dhp_md_destroy": (C.c_int, [_vp, _vp]),
    "dhp_md_reset": (C.c_int, [_vp, _vp]),
    "dhp_md_run": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _i32, _f32, _i32, _i32, _vp]),
    "dhp_md_open": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _f32, _i32, _i64, _i64]),
    "dhp_md_close": (C.c_int, [_vp, _vp, _vp, _vp, _f32, _i32, _i64, _i64]),
    "dhp_kinetic_energy_static": (C.c_int, [_vp, _vp, _i64, _vp, _vp]),
    "dhp_status": (C.c_int, [_vp]),
    "dhp_set_mlp_mode": (C.c_int, [_vp, _i32]),
    "dhp_tensor_path_available": (C.c_int, [_vp]),
    "dhp_debug_aev": (C.c_int, [_vp, _vp]),
    "dhp_debug_grad": (C.c_int, [_vp, _vp]),
    "dhp_debug_atomic_energy": (C.c_int, [_vp, _vp]),
    "dhp_debug_tile_blocks": (C.c_int, [_vp, C.POINTER(_i64), C.POINTER(_i64)]),
    "dhp_profile_enable": (C.c_int, [_vp, _i32]),
    "dhp_profile_reset": (C.c_int, [_vp]),
    "dhp_profile_read": (C.c_int, [_vp, C.POINTER(C.c_double), C.POINTER(_i64)]),
    "dhp_launch_count": (_i64, [_vp]),
    "dhp_graph_replays": (_i64, [_vp]),
    "dhp_strerror": (C.c_char_p, [_i32]),
    "dhp_last_cuda_error": (C.c_char_p, [_vp]),
    "dhp_version": (C.c_char_p, []),
}


class DhpParams(C.Structure):
    _fields_ = [("rcr", _f32), ("rca", _f32), ("eta_r", _f32), ("eta_a", _f32), ("zeta", _f32), ("celu_alpha", _f32),
                ("shf_r", _f32 * 16), ("shf_a", _f32 * 8), ("shf_z", _f32 * 8), ("n_shf_a", C.c_int32), ("n_shf_z", C.c_int32)]


class DhpError(RuntimeError):
    pass


_lib = None


def load_library() -> C.CDLL:
    """dlopen libdhp.so and bind every declared symbol.  Raises if the library was not built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise DhpError(f"{LIB_PATH} not found: build it with `python -m paper_2207_14276_b200.build` "
                           "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)          # AttributeError if the symbol is not exported
            fn.restype = res
            fn.argtypes = args
        version = lib.dhp_version().decode()
        if "[extra flags:" in version and os.environ.get("DHP_ALLOW_EXPERIMENT") != "1":
            raise DhpError(f"{LIB_PATH} is an experiment build ({version}): some of those macros give wrong results by design. "
                           "Rebuild without DHP_NVCC_EXTRA (python -m paper_2207_14276_b200.build), or set DHP_ALLOW_EXPERIMENT=1")
        _lib = lib
    return _lib


def _check(rc: int, ctx=None):
    if rc != OK:
        lib = load_library()
        msg = lib.dhp_strerror(rc).decode()
        if ctx is not None and rc == -6:
            msg += ": " + lib.dhp_last_cuda_error(ctx).decode()
        raise DhpError(f"dhp error {rc}: {msg}")


def _dptr(t) -> Optional[int]:
    """Device (or host) address of a torch tensor / numpy array, or None."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _check_inputs(torch, device, pos, species, mol_offsets=None, host: bool = False):
    """The C ABI reads raw addresses: refuse anything it would misread (wrong dtype, a strided view, the wrong device)
    instead of returning garbage with DHP_OK.  `host`: buffers of the host entry point (numpy or CPU tensors)."""
    def one(name, a, dtype_np, dtype_t, shape_tail):
        if isinstance(a, np.ndarray):
            if not host:
                raise DhpError(f"{name}: a numpy array was passed to a device-pointer call")
            ok = a.dtype == dtype_np and a.flags["C_CONTIGUOUS"]
        else:
            ok = a.dtype == dtype_t and a.is_contiguous() and ((a.device.type == "cpu") if host else (a.device == device))
        if not ok or tuple(a.shape[1:]) != shape_tail:
            raise DhpError(f"{name} must be a contiguous {dtype_np.__name__} array of shape [N{', 3' if shape_tail else ''}] "
                           f"{'in host memory' if host else f'on {device}'}")
    one("pos", pos, np.float32, torch.float32, (3,))
    one("species", species, np.int32, torch.int32, ())
    n = int(pos.shape[0])
    if int(species.shape[0]) != n:
        raise DhpError("species must have one entry per atom")
    if mol_offsets is not None:
        one("mol_offsets", mol_offsets, np.int32, torch.int32, ())
        if int(mol_offsets.shape[0]) < 2:
            raise DhpError("mol_offsets needs n_mol + 1 >= 2 entries")
        if host and (int(mol_offsets[0]) != 0 or int(mol_offsets[-1]) != n):     # values of device tables are not read here:
            raise DhpError("mol_offsets must start at 0 and end at n_atoms")      # that would synchronise the hot call


KINETIC_STATIC_MAX_ATOMS = 1048576      # DHP_KINETIC_STATIC_MAX_ATOMS of include/dhp.h


def dhp_kinetic_energy_static(vel, inv_mass, E_kin, stream=None):
    """Kinetic energy sum_i 1/2 |v_i|^2 / inv_mass_i (Hartree) of cuda tensors vel fp32 [N, 3] and inv_mass fp32 [N], written
    into the caller's cuda tensor E_kin (fp64, one element) - the entry point for code that must not allocate device memory
    (an MD engine's plug-in working inside the engine's own reservation, a diagnostic inside a running loop where a
    cudaMalloc would stall the device, a process whose allocator owns the GPU).  Neither the library nor this wrapper
    allocates: no context, no handle, the result goes where the caller says, and the working memory is a fixed array
    inside libdhp.so - which is why N is limited to KINETIC_STATIC_MAX_ATOMS and why calls that could overlap on one GPU
    must be ordered by the caller (they share that array).  `stream`: a torch.cuda.Stream, or None for torch's current
    stream; the tensors' device is made current for the call.  Asynchronous.  Make the first call on a device outside any
    stream capture: it looks up the array's address.  See include/dhp.h."""
    import torch
    lib = load_library()
    for name, a, dt, shape in (("vel", vel, torch.float32, (int(inv_mass.shape[0]), 3)), ("inv_mass", inv_mass, torch.float32, None),
                               ("E_kin", E_kin, torch.float64, None)):
        if not (a.is_cuda and a.dtype == dt and a.is_contiguous() and a.device == vel.device):
            raise DhpError(f"{name} must be a contiguous {dt} cuda tensor on {vel.device}")
        if shape is not None and tuple(a.shape) != shape:
            raise DhpError(f"{name} must have shape {list(shape)}")
    n = int(inv_mass.shape[0])
    if inv_mass.dim() != 1 or E_kin.numel() < 1:
        raise DhpError("inv_mass must be [N] and E_kin must hold one fp64")
    if n > KINETIC_STATIC_MAX_ATOMS:
        raise DhpError(f"dhp_kinetic_energy_static handles at most {KINETIC_STATIC_MAX_ATOMS} atoms (its working memory is a "
                       f"fixed array inside the library), got {n}")
    with torch.cuda.device(vel.device):
        st = torch.cuda.current_stream() if stream is None else stream
        _check(lib.dhp_kinetic_energy_static(_vp(_dptr(vel)), _vp(_dptr(inv_mass)), n, _vp(_dptr(E_kin)), _vp(st.cuda_stream)))
    return E_kin


def make_params(p) -> DhpParams:
    """`workloads.AniParams` (fp32 values) -> C struct."""
    q = DhpParams()
    q.rcr, q.rca, q.eta_r, q.eta_a = float(p.rcr), float(p.rca), float(p.eta_r), float(p.eta_a)
    q.zeta, q.celu_alpha = float(p.zeta), float(p.celu_alpha)
    for i in range(16):
        q.shf_r[i] = float(p.shf_r[i])
    q.n_shf_a, q.n_shf_z = len(p.shf_a), len(p.shf_z)          # 8 x 4 (ANI-2x shape) or 4 x 8 (ANI-1x shape)
    for i in range(q.n_shf_a):
        q.shf_a[i] = float(p.shf_a[i])
    for i in range(q.n_shf_z):
        q.shf_z[i] = float(p.shf_z[i])
    return q


class Dhp:
    """One context (workspace for `max_atoms`, bound to the current torch CUDA stream)."""

    def __init__(self, max_atoms: int, max_mols: int = 0, params=None, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise DhpError("no CUDA device: the dhp hot path has no CPU fallback")
        self.torch = torch
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device)
        self._params = make_params(params) if params is not None else None
        self.rcr = float(self._params.rcr) if self._params is not None else float(np.float32(5.1))
        ctx = _vp()
        _check(self.lib.dhp_create(C.byref(ctx), C.byref(self._params) if self._params is not None else None,
                                   int(max_atoms), int(max_mols), _vp(self.stream.cuda_stream)))
        self.ctx = ctx
        self.max_atoms, self.max_mols = int(max_atoms), int(max_mols)
        self._weights = []
        self._nlist = None
        self._n = 0

    # ---- lifetime
    def close(self):
        if getattr(self, "ctx", None):
            for w in self._weights:
                self.lib.dhp_weights_free(self.ctx, w)
            self._weights = []
            self.lib.dhp_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- C ABI, same names
    def dhp_weights_load(self, blob, n_models: int):
        """blob: numpy fp32 (host) or torch cuda fp32 tensor with 338689*7*n_models values."""
        if isinstance(blob, np.ndarray):
            blob = np.ascontiguousarray(blob, dtype=np.float32)
            n = blob.size
        else:
            blob = blob.contiguous()
            n = blob.numel()
        h = _vp()
        _check(self.lib.dhp_weights_load(self.ctx, _vp(_dptr(blob)), int(n), int(n_models), C.byref(h)), self.ctx)
        self._weights.append(h)
        h.n_models = int(n_models)
        return h

    def dhp_nlist_build(self, pos, box, species, mol_offsets=None):
        """pos/species/mol_offsets: cuda tensors (fp32 [N,3], int32 [N], int32 [n_mol+1]); box: host fp32[3] or None."""
        _check_inputs(self.torch, self.device, pos, species, mol_offsets)
        n = int(pos.shape[0])
        boxh = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
        n_mol = 0 if mol_offsets is None else int(mol_offsets.shape[0]) - 1
        h = _vp()
        _check(self.lib.dhp_nlist_build(self.ctx, _vp(_dptr(pos)), _vp(_dptr(boxh)), _vp(_dptr(species)), n,
                                        _vp(_dptr(mol_offsets)), n_mol, C.c_float(self.rcr), C.byref(h)), self.ctx)
        self._nlist, self._n = h, n
        return h

    def dhp_set_skin(self, skin: float):
        _check(self.lib.dhp_set_skin(self.ctx, C.c_float(float(skin))), self.ctx)

    def dhp_nlist_rebuild_count(self) -> int:
        return int(self.lib.dhp_nlist_rebuild_count(self.ctx))

    def dhp_nlist_sizes(self):
        a, b = _i64(), _i64()
        _check(self.lib.dhp_nlist_sizes(self.ctx, self._nlist, C.byref(a), C.byref(b)), self.ctx)
        return int(a.value), int(b.value)

    def dhp_nlist_export(self):
        """Canonical CSR (caller numbering, ascending columns): (row_ptr, col, row_ptr_ang, col_ang) int32 cuda tensors."""
        t = self.torch
        nnz, nnz_a = self.dhp_nlist_sizes()
        rp = t.empty(self._n + 1, dtype=t.int32, device=self.device)
        col = t.empty(max(nnz, 1), dtype=t.int32, device=self.device)
        rpa = t.empty(self._n + 1, dtype=t.int32, device=self.device)
        cola = t.empty(max(nnz_a, 1), dtype=t.int32, device=self.device)
        _check(self.lib.dhp_nlist_export(self.ctx, self._nlist, _vp(_dptr(rp)), _vp(_dptr(col)), _vp(_dptr(rpa)),
                                         _vp(_dptr(cola))), self.ctx)
        t.cuda.synchronize(self.device)
        return rp, col[:nnz], rpa, cola[:nnz_a]

    def dhp_ani_energy_forces(self, pos, box, species, weights, mol_offsets=None, E=None, F=None):
        """Device-pointer hot call.  Returns (E fp64 [max(1,n_mol)], F fp32 [N,3]) cuda tensors; asynchronous."""
        t = self.torch
        _check_inputs(t, self.device, pos, species, mol_offsets)
        n = int(pos.shape[0])
        boxh = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
        n_mol = 0 if mol_offsets is None else int(mol_offsets.shape[0]) - 1
        if E is None:
            E = t.empty(max(1, n_mol), dtype=t.float64, device=self.device)
        if F is None:
            F = t.empty((n, 3), dtype=t.float32, device=self.device)
        _check(self.lib.dhp_ani_energy_forces(self.ctx, _vp(_dptr(pos)), _vp(_dptr(boxh)), _vp(_dptr(species)), n,
                                              _vp(_dptr(mol_offsets)), n_mol, weights, weights.n_models,
                                              _vp(_dptr(E)), _vp(_dptr(F))), self.ctx)
        self._n = n
        return E, F

    def dhp_ani_energy_forces_partial(self, pos, box, species, weights, central, mol_offsets=None, E=None, F=None):
        """Partial evaluation over the atoms with central[i] != 0 (cuda uint8 [N], or None = all): E_c and the force
        F_c = -dE_c/dr on ALL atoms.  Over a partition of the atoms the results add up to the full call's."""
        t = self.torch
        _check_inputs(t, self.device, pos, species, mol_offsets)
        n = int(pos.shape[0])
        boxh = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
        n_mol = 0 if mol_offsets is None else int(mol_offsets.shape[0]) - 1
        if central is not None and (central.dtype != t.uint8 or int(central.shape[0]) != n):
            raise DhpError("central must be a uint8 tensor with one entry per atom")
        if E is None:
            E = t.empty(max(1, n_mol), dtype=t.float64, device=self.device)
        if F is None:
            F = t.empty((n, 3), dtype=t.float32, device=self.device)
        _check(self.lib.dhp_ani_energy_forces_partial(self.ctx, _vp(_dptr(pos)), _vp(_dptr(boxh)), _vp(_dptr(species)), n,
                                                      _vp(_dptr(mol_offsets)), n_mol, weights, weights.n_models,
                                                      _vp(_dptr(central)), _vp(_dptr(E)), _vp(_dptr(F))), self.ctx)
        self._n = n
        return E, F

    def dhp_ani_energy(self, pos, box, species, weights, mol_offsets=None, E=None):
        """Energy-only device-pointer call (a1, a2, a3).  Returns E fp64 [max(1,n_mol)] cuda tensor; asynchronous."""
        t = self.torch
        _check_inputs(t, self.device, pos, species, mol_offsets)
        n = int(pos.shape[0])
        boxh = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
        n_mol = 0 if mol_offsets is None else int(mol_offsets.shape[0]) - 1
        if E is None:
            E = t.empty(max(1, n_mol), dtype=t.float64, device=self.device)
        _check(self.lib.dhp_ani_energy(self.ctx, _vp(_dptr(pos)), _vp(_dptr(boxh)), _vp(_dptr(species)), n,
                                       _vp(_dptr(mol_offsets)), n_mol, weights, weights.n_models, _vp(_dptr(E))), self.ctx)
        self._n = n
        return E

    def dhp_ani_energy_forces_host(self, pos, box, species, weights, mol_offsets=None, E=None, F=None):
        """Host-buffer call (numpy arrays or pinned torch CPU tensors): copies in, kernels, copies out, one sync."""
        _check_inputs(self.torch, self.device, pos, species, mol_offsets, host=True)
        n = int(pos.shape[0])
        boxh = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
        n_mol = 0 if mol_offsets is None else int(mol_offsets.shape[0]) - 1
        if E is None:
            E = np.empty(max(1, n_mol), dtype=np.float64)
        if F is None:
            F = np.empty((n, 3), dtype=np.float32)
        _check(self.lib.dhp_ani_energy_forces_host(self.ctx, _vp(_dptr(pos)), _vp(_dptr(boxh)), _vp(_dptr(species)), n,
                                                   _vp(_dptr(mol_offsets)), n_mol, weights, weights.n_models,
                                                   _vp(_dptr(E)), _vp(_dptr(F))), self.ctx)
        self._n = n
        return E, F

    # ---- multiple-timestep driver (Eqs. 8-9)
    def dhp_md_create(self, inv_mass, bonds=None, bond_k=None, bond_r0=None):
        """inv_mass fp32 [N]; bonds int32 [n_bonds,2], bond_k / bond_r0 fp32 [n_bonds] (numpy or cuda tensors)."""
        def prep(a, dt):
            if a is None:
                return None
            return np.ascontiguousarray(a, dtype=dt) if isinstance(a, np.ndarray) else a.contiguous()
        inv_mass, bonds = prep(inv_mass, np.float32), prep(bonds, np.int32)
        bond_k, bond_r0 = prep(bond_k, np.float32), prep(bond_r0, np.float32)
        nb = 0 if bonds is None else int(bonds.shape[0])
        h = _vp()
        _check(self.lib.dhp_md_create(self.ctx, int(inv_mass.shape[0]), _vp(_dptr(inv_mass)), _vp(_dptr(bonds)),
                                      _vp(_dptr(bond_k)), _vp(_dptr(bond_r0)), nb, C.byref(h)), self.ctx)
        return h

    def dhp_md_destroy(self, md):
        _check(self.lib.dhp_md_destroy(self.ctx, md), self.ctx)

    def dhp_md_reset(self, md):
        _check(self.lib.dhp_md_reset(self.ctx, md), self.ctx)

    def dhp_md_run(self, md, pos, vel, box, species, weights, dt: float, n_inner: int, n_steps: int, E_out=None):
        """n_steps outer steps in place on the cuda tensors pos, vel.  Returns E_out (fp64 [3] cuda: E_ANI, E_bonds, E_kin)."""
        t = self.torch
        _check_inputs(t, self.device, pos, species)
        boxh = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
        if E_out is None:
            E_out = t.empty(3, dtype=t.float64, device=self.device)
        _check(self.lib.dhp_md_run(self.ctx, md, _vp(_dptr(pos)), _vp(_dptr(vel)), _vp(_dptr(boxh)), _vp(_dptr(species)),
                                   weights, weights.n_models, C.c_float(float(dt)), int(n_inner), int(n_steps),
                                   _vp(_dptr(E_out))), self.ctx)
        self._n = int(pos.shape[0])
        return E_out

    def _check_rows3(self, **arrays):
        """fp32 [N, 3] cuda tensors of this context's device, contiguous, all with the same N (the C ABI reads raw addresses)."""
        t, n = self.torch, None
        for name, a in arrays.items():
            ok = (hasattr(a, "is_cuda") and a.device == self.device and a.dtype == t.float32 and a.is_contiguous()
                  and a.dim() == 2 and int(a.shape[1]) == 3 and (n is None or int(a.shape[0]) == n))
            if not ok:
                raise DhpError(f"{name} must be a contiguous float32 tensor of shape [N, 3] on {self.device}")
            n = int(a.shape[0])

    def dhp_md_open(self, md, pos, vel, box, F_slow, dt: float, n_inner: int, lo: int, hi: int):
        """First half kick + inner loop (all but its last fast half kick, see include/dhp.h) for the owned atoms [lo, hi),
        in place on the cuda tensors pos, vel."""
        self._check_rows3(pos=pos, vel=vel, F_slow=F_slow)
        boxh = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
        _check(self.lib.dhp_md_open(self.ctx, md, _vp(_dptr(pos)), _vp(_dptr(vel)), _vp(_dptr(boxh)), _vp(_dptr(F_slow)),
                                    C.c_float(float(dt)), int(n_inner), int(lo), int(hi)), self.ctx)

    def dhp_md_close(self, md, vel, F_slow, dt: float, n_inner: int, lo: int, hi: int):
        """The pending fast half kick and the second slow half kick for the owned atoms [lo, hi); dt and n_inner must be those
        of the dhp_md_open this call completes."""
        self._check_rows3(vel=vel, F_slow=F_slow)
        _check(self.lib.dhp_md_close(self.ctx, md, _vp(_dptr(vel)), _vp(_dptr(F_slow)), C.c_float(float(dt)), int(n_inner),
                                     int(lo), int(hi)), self.ctx)

    def dhp_status(self) -> int:
        return int(self.lib.dhp_status(self.ctx))

    def dhp_set_mlp_mode(self, mode: int):
        _check(self.lib.dhp_set_mlp_mode(self.ctx, int(mode)), self.ctx)

    def dhp_tensor_path_available(self) -> bool:
        return bool(self.lib.dhp_tensor_path_available(self.ctx))

    def _debug(self, fn, ncol):
        t = self.torch
        out = t.empty((self._n, ncol), dtype=t.float32, device=self.device)
        _check(fn(self.ctx, _vp(_dptr(out))), self.ctx)
        return out

    def dhp_debug_aev(self):
        return self._debug(self.lib.dhp_debug_aev, 1008)

    def dhp_debug_grad(self):
        return self._debug(self.lib.dhp_debug_grad, 1008)

    def dhp_debug_atomic_energy(self):
        return self._debug(self.lib.dhp_debug_atomic_energy, 1)[:, 0]

    def dhp_debug_tile_blocks(self):
        """(row tiles, active 64-wide feature blocks summed over tiles) of the last call."""
        a, b = _i64(), _i64()
        _check(self.lib.dhp_debug_tile_blocks(self.ctx, C.byref(a), C.byref(b)), self.ctx)
        return int(a.value), int(b.value)

    def dhp_profile_enable(self, on: bool):
        _check(self.lib.dhp_profile_enable(self.ctx, 1 if on else 0), self.ctx)

    def dhp_profile_reset(self):
        _check(self.lib.dhp_profile_reset(self.ctx), self.ctx)

    def dhp_profile_read(self):
        ms = (C.c_double * N_PHASES)()
        n = _i64()
        _check(self.lib.dhp_profile_read(self.ctx, ms, C.byref(n)), self.ctx)
        return {PHASES[i]: float(ms[i]) for i in range(N_PHASES)}, int(n.value)

    def dhp_launch_count(self) -> int:
        return int(self.lib.dhp_launch_count(self.ctx))

    def dhp_graph_replays(self) -> int:
        return int(self.lib.dhp_graph_replays(self.ctx))


def to_device(system, device="cuda:0"):
    """Upload a `workloads.System` once: (pos, species, mol_offsets) cuda tensors."""
    import torch
    pos = torch.from_numpy(np.ascontiguousarray(system.pos)).to(device)
    species = torch.from_numpy(np.ascontiguousarray(system.species)).to(device)
    mol = None if system.mol_offsets is None else torch.from_numpy(np.ascontiguousarray(system.mol_offsets)).to(device)
    return pos, species, mol
