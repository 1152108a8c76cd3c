"""Thin ctypes binding of include/gridff.h — argument marshalling only; every step of the path runs in the CUDA kernels
of csrc/libgridff.so.  PyTorch supplies device memory and the stream, nothing else.

There is NO CPU fallback: importing this module without the built library raises, and every compute call returns
GRIDFF_ECUDA (raised as GridffError) without a CUDA device.

Function names follow the C-ABI (gridff_build_grid, gridff_eval, gridff_run_replicas, ...); `Grid` and `Molecule` are small
owners that keep the caller-side device buffers alive next to the opaque handles.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libgridff.so")

if not os.path.exists(LIB_PATH):
    raise ImportError("paper_2508_15522_b200: csrc/libgridff.so is missing - build it with "
                      "`python -m paper_2508_15522_b200.csrc.build` (there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)

OK, EINVAL, EUNSUPPORTED, ESIZE, ECUDA = 0, -1, -2, -3, -4
CH_PAULI, CH_LONDON, CH_COULOMB, CH_ZERO = 0, 1, 2, 3
LAYOUT_ZFAST, LAYOUT_BRICK = 0, 1


class GridffError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("gridff error %d: %s" % (code, msg))
        self.code = code


class GridDesc(C.Structure):
    _fields_ = [("Lx", C.c_double), ("Ly", C.c_double), ("z_ref", C.c_double), ("z_lo", C.c_double), ("z_hi", C.c_double),
                ("spacing", C.c_double), ("alpha", C.c_double), ("r_cut", C.c_double),
                ("n_channels", C.c_int), ("channel", C.c_int * 4), ("layout", C.c_int), ("l2_persist", C.c_int), ("morse_window", C.c_int)]


class Topology(C.Structure):
    _fields_ = [("n_atoms", C.c_int), ("mass", C.c_void_p), ("coef", C.c_void_p),
                ("q", C.c_void_p), ("lj_e", C.c_void_p), ("lj_R", C.c_void_p),
                ("n_bonds", C.c_int), ("bond", C.c_void_p), ("bond_k_r0", C.c_void_p),
                ("n_angles", C.c_int), ("angle", C.c_void_p), ("angle_k_t0", C.c_void_p),
                ("n_tors", C.c_int), ("tors", C.c_void_p), ("tors_k_n_p0", C.c_void_p),
                ("excl", C.c_void_p),
                ("n_rot", C.c_int), ("rot_bond", C.c_void_p), ("rot_mask", C.c_void_p), ("ref_pos", C.c_void_p)]


class Integrator(C.Structure):
    _fields_ = [("kind", C.c_int), ("n_steps", C.c_int), ("dt", C.c_float), ("f_tol", C.c_float),
                ("dt_max", C.c_float), ("f_inc", C.c_float), ("f_dec", C.c_float), ("a_start", C.c_float), ("f_a", C.c_float),
                ("n_min", C.c_int), ("max_step", C.c_float), ("restart", C.c_int), ("seed", C.c_ulonglong),
                ("z_ref", C.c_float), ("place_z_lo", C.c_float), ("place_z_hi", C.c_float), ("place_z_min", C.c_float),
                ("clash", C.c_float), ("variant", C.c_int),
                ("temperature", C.c_float), ("gamma", C.c_float), ("step0", C.c_uint), ("n_scan", C.c_int),
                ("fixed_mask", C.c_ulonglong), ("scan_dx", C.c_float * 3)]


class Hopping(C.Structure):
    _fields_ = [("n_cycles", C.c_int), ("cycle0", C.c_int), ("md_steps", C.c_int), ("md_dt", C.c_float),
                ("temperature", C.c_float), ("gamma", C.c_float), ("relax_steps", C.c_int), ("relax_dt", C.c_float),
                ("f_tol", C.c_float), ("dt_max", C.c_float), ("max_step", C.c_float), ("e_tol", C.c_float), ("rmsd_tol", C.c_float),
                ("seed", C.c_ulonglong), ("fixed_mask", C.c_ulonglong)]


_vp, _sz, _ll, _i = C.c_void_p, C.c_size_t, C.c_longlong, C.c_int
_P = C.POINTER
_SIG = {
    "gridff_last_error": (C.c_char_p, []),
    "gridff_version": (_i, []),
    "gridff_grid_dims": (_i, [_P(GridDesc), _P(_i * 3), _P(C.c_double * 3), _P(C.c_double * 3)]),
    "gridff_grid_bytes": (_i, [_P(GridDesc), _i, _P(_sz), _P(_sz)]),
    "gridff_build_grid": (_i, [_P(GridDesc), _i, _vp, _vp, _vp, _vp, _vp, _sz, _vp, _sz, _vp, _P(_vp)]),
    "gridff_grid_from_samples": (_i, [_P(GridDesc), _vp, _vp, _sz, _vp, _sz, _vp, _P(_vp)]),
    "gridff_grid_export": (_i, [_vp, _vp, _vp]),
    "gridff_grid_info": (_i, [_vp, _P(_i * 3), _P(C.c_double * 3), _P(C.c_double * 3), _P(_i), _P(_i)]),
    "gridff_free_grid": (_i, [_vp]),
    "gridff_derive_bytes": (_sz, [_vp, _i]),
    "gridff_grid_derive": (_i, [_vp, _i, _vp, _sz, _vp, _P(_vp)]),
    "gridff_atom_coefs": (_i, [C.c_double, _i, _vp, _vp, _vp, _vp]),
    "gridff_eval": (_i, [_vp, _ll, _vp, _vp, _vp, _vp, _vp]),
    "gridff_eval_variant": (_i, [_vp, _ll, _vp, _vp, _vp, _vp, _i, _vp]),
    "gridff_eval_binned_work_bytes": (_sz, [_vp, _ll]),
    "gridff_eval_binned": (_i, [_vp, _ll, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "gridff_eval_binned_noalloc_max_bytes": (_sz, []),
    "gridff_eval_binned_noalloc": (_i, [_vp, _ll, _vp, _vp, _vp, _vp, _vp]),
    "gridff_eval_work_bytes": (_sz, [_ll]),
    "gridff_eval_host": (_i, [_vp, _ll, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "gridff_molecule_bytes": (_sz, [_P(Topology)]),
    "gridff_create_molecule": (_i, [_P(Topology), _vp, _sz, _vp, _P(_vp)]),
    "gridff_free_molecule": (_i, [_vp]),
    "gridff_run_replicas": (_i, [_vp, _vp, _P(Integrator), _i, _vp, _vp, _vp, _vp, _vp, _vp, _i, _vp, _vp]),
    "gridff_run_scan": (_i, [_vp, _vp, _P(Integrator), _i, _vp, _vp, _vp, _vp, _vp, _vp]),
    "gridff_hopping_work_bytes": (_sz, [_vp, _i]),
    "gridff_minima_hopping": (_i, [_vp, _vp, _P(Hopping), _i, _vp, _vp, _i, _vp, _vp, _vp, _sz, _vp]),
    "gridff_unique_filter": (_i, [_vp, _vp, _i, _vp, _vp, _vp, _vp, C.c_float, C.c_float, _i, _vp, _i, _vp, _vp, _vp, _vp]),
    "gridff_run_work_bytes": (_sz, [_vp, _i]),
    "gridff_run_replicas_host": (_i, [_vp, _vp, _P(Integrator), _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "gridff_probe_read": (_i, [_vp, _sz, _i, _i, _vp, _vp]),
    "gridff_launch_count": (_ll, []),
}
for _name, (_res, _args) in _SIG.items():
    _f = getattr(_lib, _name)
    _f.restype = _res
    _f.argtypes = _args
EXPORTS = sorted(_SIG)


def gridff_last_error():
    return _lib.gridff_last_error().decode()


def _check(rc):
    if rc != OK:
        raise GridffError(rc, gridff_last_error())


def gridff_version():
    return int(_lib.gridff_version())


def gridff_launch_count():
    return int(_lib.gridff_launch_count())


def _stream(stream=None):
    if stream is None:
        if not torch.cuda.is_available():
            return None            # the library call itself will fail with GRIDFF_ECUDA
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dptr(t):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    return C.c_void_p(t.data_ptr())


def _hptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def make_desc(Lx, Ly, z_ref, z_lo, z_hi, spacing, alpha, channels, r_cut=17.0, layout=LAYOUT_ZFAST, l2_persist=0, morse_window=0):
    d = GridDesc()
    d.Lx, d.Ly, d.z_ref, d.z_lo, d.z_hi, d.spacing, d.alpha, d.r_cut = Lx, Ly, z_ref, z_lo, z_hi, spacing, alpha, r_cut
    d.n_channels = len(channels)
    for k in range(4):
        d.channel[k] = int(channels[k]) if k < len(channels) else CH_ZERO
    d.layout, d.l2_persist, d.morse_window = int(layout), int(l2_persist), int(morse_window)
    return d


def gridff_grid_dims(desc):
    dims, h, org = (C.c_int * 3)(), (C.c_double * 3)(), (C.c_double * 3)()
    _check(_lib.gridff_grid_dims(C.byref(desc), C.byref(dims), C.byref(h), C.byref(org)))
    return tuple(dims), tuple(h), tuple(org)


def gridff_grid_bytes(desc, n_sub):
    a, b = C.c_size_t(0), C.c_size_t(0)
    _check(_lib.gridff_grid_bytes(C.byref(desc), int(n_sub), C.byref(a), C.byref(b)))
    return a.value, b.value


class Grid:
    """Owner of the opaque gridff_grid handle and of the device store it points into."""

    def __init__(self, handle, desc, store):
        self.handle, self.desc, self.store = handle, desc, store

    def info(self):
        dims, h, org = (C.c_int * 3)(), (C.c_double * 3)(), (C.c_double * 3)()
        nch, lay = C.c_int(0), C.c_int(0)
        _check(_lib.gridff_grid_info(self.handle, C.byref(dims), C.byref(h), C.byref(org), C.byref(nch), C.byref(lay)))
        return dict(dims=tuple(dims), h=tuple(h), origin=tuple(org), n_channels=nch.value, layout=lay.value)

    def free(self):
        if self.handle is not None:
            _lib.gridff_free_grid(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def _alloc(nbytes):
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device="cuda")


def gridff_build_grid(desc, sub_pos, sub_e, sub_R, sub_q=None, stream=None, keep_scratch=False):
    """substrate arrays: host float64.  Returns a Grid (store tensor owned by it)."""
    pos = np.ascontiguousarray(sub_pos, dtype=np.float64).reshape(-1, 3)
    n = len(pos)
    e = None if sub_e is None else np.ascontiguousarray(sub_e, dtype=np.float64)
    R = None if sub_R is None else np.ascontiguousarray(sub_R, dtype=np.float64)
    q = None if sub_q is None else np.ascontiguousarray(sub_q, dtype=np.float64)
    sb, wb = gridff_grid_bytes(desc, n)
    if not torch.cuda.is_available():
        raise GridffError(ECUDA, "no CUDA device (there is no CPU fallback)")
    store, scratch = _alloc(sb), _alloc(wb)
    out = C.c_void_p(None)
    _check(_lib.gridff_build_grid(C.byref(desc), n, _hptr(pos), _hptr(e), _hptr(R), _hptr(q),
                                  _dptr(store), store.numel(), _dptr(scratch), scratch.numel(), _stream(stream), C.byref(out)))
    g = Grid(out, desc, store)
    if keep_scratch:
        g.scratch = scratch
    else:
        torch.cuda.current_stream().synchronize()      # scratch may be released once the build has finished
    return g


def gridff_grid_from_samples(desc, d_samples, stream=None):
    """d_samples: CUDA float32 tensor [nx][ny][nz][n_channels]."""
    sb, wb = gridff_grid_bytes(desc, 0)
    store, scratch = _alloc(sb), _alloc(wb)
    out = C.c_void_p(None)
    _check(_lib.gridff_grid_from_samples(C.byref(desc), _dptr(d_samples), _dptr(store), store.numel(), _dptr(scratch), scratch.numel(),
                                         _stream(stream), C.byref(out)))
    torch.cuda.current_stream().synchronize()
    return Grid(out, desc, store)


LAYOUT_HALF, LAYOUT_TRILINEAR = 2, 3
LAYOUT_MBRICK, LAYOUT_MBRICK2, LAYOUT_MBRICK8 = 4, 5, 6       # 2x2x2-node bricks, 1 / 2 / 8 shifted copies (stores beyond the L2)


def gridff_grid_derive(parent, layout, stream=None):
    """derived store: LAYOUT_HALF (fp16 coefficients), LAYOUT_TRILINEAR (the paper's foil) or LAYOUT_MBRICK / MBRICK2 / MBRICK8 (the fp32
    coefficients in 128-byte bricks for stores beyond the L2); gridff_eval only."""
    nbytes = int(_lib.gridff_derive_bytes(parent.handle, int(layout)))
    store = _alloc(nbytes)
    out = C.c_void_p(None)
    _check(_lib.gridff_grid_derive(parent.handle, int(layout), _dptr(store), store.numel(), _stream(stream), C.byref(out)))
    return Grid(out, parent.desc, store)


def gridff_grid_export(grid, stream=None):
    info = grid.info()
    nx, ny, nz = info["dims"]
    out = torch.empty((nx, ny, nz, info["n_channels"]), dtype=torch.float32, device="cuda")
    _check(_lib.gridff_grid_export(grid.handle, _dptr(out), _stream(stream)))
    return out


def gridff_free_grid(grid):
    grid.free()


def gridff_atom_coefs(alpha, e, R, q=None):
    e = np.ascontiguousarray(e, dtype=np.float32); R = np.ascontiguousarray(R, dtype=np.float32)
    q = None if q is None else np.ascontiguousarray(q, dtype=np.float32)
    out = np.zeros((len(e), 4), np.float32)
    _check(_lib.gridff_atom_coefs(float(alpha), len(e), _hptr(e), _hptr(R), _hptr(q), _hptr(out)))
    return out


def gridff_eval(grid, d_pos, d_coef, d_E=None, d_F=None, stream=None, variant=None, want_E=True, want_F=True):
    """d_pos [n][3], d_coef [n][4] CUDA float32.  Returns (E [n], F [n][3]) CUDA tensors."""
    n = d_pos.shape[0]
    if d_E is None and want_E:
        d_E = torch.empty(n, dtype=torch.float32, device="cuda")
    if d_F is None and want_F:
        d_F = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    if variant is None:
        _check(_lib.gridff_eval(grid.handle, n, _dptr(d_pos), _dptr(d_coef), _dptr(d_E), _dptr(d_F), _stream(stream)))
    else:
        _check(_lib.gridff_eval_variant(grid.handle, n, _dptr(d_pos), _dptr(d_coef), _dptr(d_E), _dptr(d_F), int(variant), _stream(stream)))
    return d_E, d_F


def gridff_eval_binned(grid, d_pos, d_coef, d_E=None, d_F=None, d_work=None, stream=None):
    """gridff_eval for scattered points on a store beyond the L2: the points are counting-sorted by cell block on the device first.
    Returns (E [n], F [n][3]) — the same numbers as gridff_eval."""
    n = d_pos.shape[0]
    if d_E is None:
        d_E = torch.empty(n, dtype=torch.float32, device="cuda")
    if d_F is None:
        d_F = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    if d_work is None:
        d_work = _alloc(int(_lib.gridff_eval_binned_work_bytes(grid.handle, n)))
    _check(_lib.gridff_eval_binned(grid.handle, n, _dptr(d_pos), _dptr(d_coef), _dptr(d_E), _dptr(d_F), _dptr(d_work), d_work.numel(), _stream(stream)))
    return d_E, d_F


def gridff_eval_binned_noalloc_max_bytes():
    return int(_lib.gridff_eval_binned_noalloc_max_bytes())


def gridff_eval_binned_noalloc(grid, d_pos, d_coef, d_E, d_F, stream=None):
    """gridff_eval_binned with its work space in a device array built into the library (16 MiB; at most 2^18 points per call): the call
    allocates nothing, so the outputs are the caller's too.  Calls that overlap on the GPU race on the shared array.  Returns (d_E, d_F)."""
    n = d_pos.shape[0]
    _check(_lib.gridff_eval_binned_noalloc(grid.handle, n, _dptr(d_pos), _dptr(d_coef), _dptr(d_E), _dptr(d_F), _stream(stream)))
    return d_E, d_F


def gridff_eval_work_bytes(n):
    return int(_lib.gridff_eval_work_bytes(int(n)))


def gridff_eval_host(grid, h_pos, h_coef, h_E, h_F, d_work=None, stream=None):
    """host float32 arrays (numpy or pinned torch CPU tensors, contiguous); results written into h_E / h_F."""
    n = h_pos.shape[0]
    if d_work is None:
        d_work = _alloc(gridff_eval_work_bytes(n))
    p = lambda a: None if a is None else C.c_void_p(a.data_ptr() if isinstance(a, torch.Tensor) else a.ctypes.data)
    _check(_lib.gridff_eval_host(grid.handle, n, p(h_pos), p(h_coef), p(h_E), p(h_F), _dptr(d_work), d_work.numel(), _stream(stream)))
    return h_E, h_F


class Molecule:
    def __init__(self, handle, buf, n_atoms, host_arrays):
        self.handle, self.buf, self.n_atoms, self._host = handle, buf, n_atoms, host_arrays

    def free(self):
        if self.handle is not None:
            _lib.gridff_free_molecule(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def make_topology(topo, coef):
    """topology dict (see inputs.py) + channel factors [n][4] -> (Topology struct, list of arrays kept alive)."""
    n = int(topo["n_atoms"])
    f32 = lambda a, shape: np.ascontiguousarray(a, dtype=np.float32).reshape(shape)
    i32 = lambda a, shape: np.ascontiguousarray(a, dtype=np.int32).reshape(shape)
    keep = dict(mass=f32(topo["mass"], (n,)), coef=f32(coef, (n, 4)))
    for k in ("q", "lj_e", "lj_R"):
        keep[k] = f32(topo[k], (n,)) if topo.get(k) is not None else None
    keep["bond"] = i32(topo.get("bond", np.zeros((0, 2))), (-1, 2)); keep["bond_k_r0"] = f32(topo.get("bond_k_r0", np.zeros((0, 2))), (-1, 2))
    keep["angle"] = i32(topo.get("angle", np.zeros((0, 3))), (-1, 3)); keep["angle_k_t0"] = f32(topo.get("angle_k_t0", np.zeros((0, 2))), (-1, 2))
    keep["tors"] = i32(topo.get("tors", np.zeros((0, 4))), (-1, 4)); keep["tors_k_n_p0"] = f32(topo.get("tors_k_n_p0", np.zeros((0, 3))), (-1, 3))
    excl = topo.get("excl")
    keep["excl"] = None if excl is None else np.ascontiguousarray(excl, dtype=np.uint8).reshape(n, n)
    rb = topo.get("rot_bond")
    keep["rot_bond"] = i32(rb, (-1, 2)) if rb is not None and len(rb) else None
    rm = topo.get("rot_mask")
    keep["rot_mask"] = np.ascontiguousarray(rm, dtype=np.uint8).reshape(-1, n) if rm is not None and len(rm) else None
    ref = topo.get("ref_pos")
    keep["ref_pos"] = f32(ref, (n, 3)) if ref is not None else None
    t = Topology()
    t.n_atoms = n
    t.mass, t.coef, t.q, t.lj_e, t.lj_R = (_hptr(keep[k]) for k in ("mass", "coef", "q", "lj_e", "lj_R"))
    t.n_bonds, t.bond, t.bond_k_r0 = len(keep["bond"]), _hptr(keep["bond"]), _hptr(keep["bond_k_r0"])
    t.n_angles, t.angle, t.angle_k_t0 = len(keep["angle"]), _hptr(keep["angle"]), _hptr(keep["angle_k_t0"])
    t.n_tors, t.tors, t.tors_k_n_p0 = len(keep["tors"]), _hptr(keep["tors"]), _hptr(keep["tors_k_n_p0"])
    t.excl = _hptr(keep["excl"])
    t.n_rot = 0 if keep["rot_bond"] is None else len(keep["rot_bond"])
    t.rot_bond, t.rot_mask, t.ref_pos = _hptr(keep["rot_bond"]), _hptr(keep["rot_mask"]), _hptr(keep["ref_pos"])
    return t, keep


def gridff_molecule_bytes(topology):
    return int(_lib.gridff_molecule_bytes(C.byref(topology)))


def gridff_create_molecule(topo, coef, stream=None):
    t, keep = make_topology(topo, coef)
    if not torch.cuda.is_available():
        raise GridffError(ECUDA, "no CUDA device (there is no CPU fallback)")
    buf = _alloc(gridff_molecule_bytes(t))
    out = C.c_void_p(None)
    _check(_lib.gridff_create_molecule(C.byref(t), _dptr(buf), buf.numel(), _stream(stream), C.byref(out)))
    return Molecule(out, buf, int(topo["n_atoms"]), keep)


def gridff_free_molecule(mol):
    mol.free()


def make_integrator(kind, n_steps, dt, f_tol=1e-3, dt_max=0.0, f_inc=1.1, f_dec=0.5, a_start=0.1, f_a=0.99, n_min=5,
                    max_step=0.0, restart=0, seed=0, z_ref=0.0, place_z_lo=3.0, place_z_hi=6.0, place_z_min=2.0, clash=0.4, variant=0,
                    temperature=0.0, gamma=0.0, step0=0, n_scan=0, fixed=(), scan_dx=(0.0, 0.0, 0.0)):
    """kind "vv" | "fire" | "langevin"; `fixed` = indices of held atoms; n_scan / scan_dx for gridff_run_scan."""
    kind = {"vv": 0, "fire": 1, "langevin": 2}.get(kind, kind)
    mask = 0
    for i in fixed:
        mask |= 1 << int(i)
    if not dt_max:
        dt_max = 10.0 * dt
    return Integrator(int(kind), int(n_steps), dt, f_tol, dt_max, f_inc, f_dec, a_start, f_a, int(n_min), max_step, int(restart),
                      int(seed), z_ref, place_z_lo, place_z_hi, place_z_min, clash, int(variant),
                      float(temperature), float(gamma), int(step0), int(n_scan), mask, (C.c_float * 3)(*[float(c) for c in scan_dx]))


def gridff_run_replicas(grid, mol, integ, d_pos, d_vel, d_fire=None, d_energy=None, d_status=None, d_minima=None, d_n_minima=None,
                        stream=None):
    """d_pos, d_vel [n_rep][n][3] CUDA float32, updated in place.  Returns dict(energy, status) (CUDA tensors)."""
    n_rep = d_pos.shape[0]
    if d_energy is None:
        d_energy = torch.empty((n_rep, 8), dtype=torch.float32, device="cuda")
    if d_status is None:
        d_status = torch.empty((n_rep, 2), dtype=torch.int32, device="cuda")
    cap = 0 if d_minima is None else d_minima.shape[0]
    _check(_lib.gridff_run_replicas(None if grid is None else grid.handle, mol.handle, C.byref(integ), n_rep, _dptr(d_pos), _dptr(d_vel),
                                    _dptr(d_fire), _dptr(d_energy), _dptr(d_status), _dptr(d_minima), cap, _dptr(d_n_minima), _stream(stream)))
    return dict(energy=d_energy, status=d_status)


def gridff_run_scan(grid, mol, integ, d_pos, d_vel, d_energy=None, d_status=None, d_scan=None, stream=None):
    """driven scan (held atoms moved by integ.scan_dx, the rest relaxed, integ.n_scan times).  Returns dict(scan [n_rep][n_scan][4], energy, status)."""
    n_rep = d_pos.shape[0]
    if d_energy is None:
        d_energy = torch.empty((n_rep, 8), dtype=torch.float32, device="cuda")
    if d_status is None:
        d_status = torch.empty((n_rep, 2), dtype=torch.int32, device="cuda")
    if d_scan is None:
        d_scan = torch.empty((n_rep, max(int(integ.n_scan), 0), 4), dtype=torch.float32, device="cuda")
    _check(_lib.gridff_run_scan(None if grid is None else grid.handle, mol.handle, C.byref(integ), n_rep, _dptr(d_pos), _dptr(d_vel),
                                _dptr(d_energy), _dptr(d_status), _dptr(d_scan), _stream(stream)))
    return dict(scan=d_scan, energy=d_energy, status=d_status)


def make_hopping(n_cycles, md_steps, md_dt, temperature, gamma, relax_steps, relax_dt, f_tol, seed, dt_max=0.0, max_step=0.0,
                 e_tol=1e-3, rmsd_tol=0.1, cycle0=0, fixed=()):
    mask = 0
    for i in fixed:
        mask |= 1 << int(i)
    return Hopping(int(n_cycles), int(cycle0), int(md_steps), md_dt, temperature, gamma, int(relax_steps), relax_dt, f_tol, dt_max, max_step,
                   e_tol, rmsd_tol, int(seed), mask)


def gridff_hopping_work_bytes(mol, n_rep):
    return int(_lib.gridff_hopping_work_bytes(mol.handle, int(n_rep)))


def gridff_minima_hopping(grid, mol, hop, d_pos, d_library, d_n_library, d_stats=None, d_work=None, stream=None):
    """hop.n_cycles x {Langevin, FIRE, unique filter} enqueued on the stream.  d_library [cap][4+3n] float32, d_n_library int32[1]
    (both in/out), d_stats int32 [n_cycles][4].  Returns d_stats."""
    n_rep = d_pos.shape[0]
    if d_work is None:
        d_work = _alloc(gridff_hopping_work_bytes(mol, n_rep))
    if d_stats is None:
        d_stats = torch.zeros((hop.n_cycles, 4), dtype=torch.int32, device="cuda")
    _check(_lib.gridff_minima_hopping(grid.handle, mol.handle, C.byref(hop), n_rep, _dptr(d_pos), _dptr(d_library), d_library.shape[0],
                                      _dptr(d_n_library), _dptr(d_stats), _dptr(d_work), d_work.numel(), _stream(stream)))
    return d_stats


def gridff_unique_filter(grid, mol, d_pos, d_E, d_ok, d_library, d_n_library, d_steps=None, e_tol=1e-3, rmsd_tol=0.1, tag=0, stream=None):
    """the filter alone; returns int32[4] = candidates, new records, dropped (library full), library size after."""
    n_rep = d_pos.shape[0]
    stats = torch.zeros(4, dtype=torch.int32, device="cuda")
    flags = torch.empty(n_rep, dtype=torch.int32, device="cuda")
    _check(_lib.gridff_unique_filter(grid.handle, mol.handle, n_rep, _dptr(d_pos), _dptr(d_E), _dptr(d_steps), _dptr(d_ok), e_tol, rmsd_tol, int(tag),
                                     _dptr(d_library), d_library.shape[0], _dptr(d_n_library), _dptr(stats), _dptr(flags), _stream(stream)))
    return stats


def gridff_run_work_bytes(mol, n_rep):
    return int(_lib.gridff_run_work_bytes(mol.handle, int(n_rep)))


def gridff_run_replicas_host(grid, mol, integ, h_pos, h_vel, h_fire=None, h_energy=None, h_status=None, d_work=None, stream=None):
    """host float32 buffers (numpy arrays or pinned torch CPU tensors), updated in place."""
    n_rep = h_pos.shape[0]
    if d_work is None:
        d_work = _alloc(gridff_run_work_bytes(mol, n_rep))
    p = lambda a: None if a is None else C.c_void_p(a.data_ptr() if isinstance(a, torch.Tensor) else a.ctypes.data)
    _check(_lib.gridff_run_replicas_host(None if grid is None else grid.handle, mol.handle, C.byref(integ), n_rep, p(h_pos), p(h_vel), p(h_fire),
                                         p(h_energy), p(h_status), _dptr(d_work), d_work.numel(), _stream(stream)))


def gridff_probe_read(d_buf, iters=1, mode=0, stream=None):
    sink = torch.zeros(4, dtype=torch.float32, device="cuda")
    _check(_lib.gridff_probe_read(_dptr(d_buf), d_buf.numel() * d_buf.element_size(), int(iters), int(mode), _dptr(sink), _stream(stream)))
