"""ctypes wrapper around oracle/gridff_oracle.c (fp64 CPU oracle).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from
paper_2508_15522_b200 and shares no code with the CUDA path.

Argument marshalling for the C file, which holds the arithmetic of the hot path (pins listed in its header), plus — written here in
plain numpy / Python loops, fp64 — the SURVEY.md §8(f) pieces that are definitions rather than numerics:
  same_structure, unique_filter     PAPER.md:L241 criterion (R16), sequential greedy filter
                                    pinned: constructed populations collapse to the known K structures; brute-force invariants
  minima_hopping                    PAPER.md:L222 loop composed of the pinned Langevin / FIRE calls and the filter (R19)
                                    pinned: records are minima, pairwise distinct; 2 cycles == 1 + 1 cycles
  half_grid                         fp64 -> fp32 -> fp16 coefficient rounding (numpy's IEEE casts)       pinned: 2^-11 bound
  trilinear_nodes, interp_trilinear PAPER.md:L118-120 foil (R20)    pinned: scipy RegularGridInterpolator, exact at nodes
Inputs are widened to float64 exactly (the GPU path receives the same values as float32).
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gridff_oracle.c")
# GRIDFF_ORACLE_SANITIZE=1: the same source built with -fsanitize=address,undefined into its own library (run the CPU pins under
# LD_PRELOAD=$(gcc -print-file-name=libasan.so); profiles/r2_sanitizers.md)
_SAN = os.environ.get("GRIDFF_ORACLE_SANITIZE", "") == "1"
_LIB = os.path.join(_HERE, "libgridff_oracle_san.so" if _SAN else "libgridff_oracle.so")
_lib = None

KE = 14.3996454784
ACC = 9.648533212e-3
KB = 8.617333262e-5


def build(force=False):
    """Compile the oracle with gcc (-O2 -fopenmp).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if _SAN else ["-O2"]
        subprocess.check_call(["gcc"] + flags + ["-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("nch", C.c_int),
                ("Lx", C.c_double), ("Ly", C.c_double), ("hz", C.c_double), ("z0", C.c_double),
                ("periodic_xy", C.c_int), ("coef", C.c_void_p)]


class Topology(C.Structure):
    _fields_ = [("n_atoms", C.c_int),
                ("mass", C.c_void_p), ("coef", C.c_void_p), ("q", C.c_void_p), ("lj_e", C.c_void_p), ("lj_R", C.c_void_p),
                ("n_bonds", C.c_int), ("bond", C.c_void_p), ("bond_k_r0", C.c_void_p),
                ("n_angles", C.c_int), ("angle", C.c_void_p), ("angle_k_t0", C.c_void_p),
                ("n_tors", C.c_int), ("tors", C.c_void_p), ("tors_k_n_p0", C.c_void_p),
                ("excl", C.c_void_p),
                ("n_rot", C.c_int), ("rot_bond", C.c_void_p), ("rot_mask", C.c_void_p), ("ref_pos", C.c_void_p)]


class Integrator(C.Structure):
    _fields_ = [("kind", C.c_int), ("n_steps", C.c_int), ("dt", C.c_double), ("f_tol", C.c_double),
                ("dt_max", C.c_double), ("f_inc", C.c_double), ("f_dec", C.c_double), ("a_start", C.c_double),
                ("f_a", C.c_double), ("n_min", C.c_int), ("restart", C.c_int), ("seed", C.c_uint64),
                ("z_ref", C.c_double), ("place_z_lo", C.c_double), ("place_z_hi", C.c_double),
                ("place_z_min", C.c_double), ("clash", C.c_double), ("max_step", C.c_double),
                ("temperature", C.c_double), ("gamma", C.c_double), ("step0", C.c_uint32), ("n_scan", C.c_int),
                ("fixed_mask", C.c_uint64), ("scan_dx", C.c_double * 3)]


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_bspline_basis.restype = C.c_double
        _lib.orc_bspline_basis.argtypes = [C.c_double]
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads():
    return int(lib().orc_num_threads())


def bspline_basis(t):
    return float(lib().orc_bspline_basis(float(t)))


def bspline_weights(t):
    w = np.zeros(4); dw = np.zeros(4)
    lib().orc_bspline_weights(C.c_double(float(t)), _p(w), _p(dw))
    return w, dw


def image_counts(Lx, Ly, r_cut):
    """DESIGN.md R10: N = ceil(r_cut / L) image cells on each side."""
    return int(np.ceil(r_cut / Lx)), int(np.ceil(r_cut / Ly))


def morse_points(sub, alpha, Lx, Ly, r_cut, pts, grad=False):
    pts = _d(pts).reshape(-1, 3); n = len(pts)
    pos, e, R = _d(sub["pos"]), _d(sub["e"]), _d(sub["R"])
    Nx, Ny = image_counts(Lx, Ly, r_cut)
    VP = np.zeros(n); VL = np.zeros(n)
    gP = np.zeros((n, 3)) if grad else None
    gL = np.zeros((n, 3)) if grad else None
    lib().orc_morse_points(C.c_int(len(pos)), _p(pos), _p(e), _p(R), C.c_double(alpha), C.c_double(Lx), C.c_double(Ly),
                           C.c_int(Nx), C.c_int(Ny), C.c_long(n), _p(pts), _p(VP), _p(VL), _p(gP), _p(gL))
    return (VP, VL, gP, gL) if grad else (VP, VL)


def coulomb_points(sub, Lx, Ly, pts, grad=False, g_cut=37.0, z_min_above_top=None):
    pts = _d(pts).reshape(-1, 3); n = len(pts)
    pos, q = _d(sub["pos"]), _d(sub["q"])
    if z_min_above_top is None:
        z_min_above_top = float(pts[:, 2].min() - pos[:, 2].max())
    VC = np.zeros(n); g = np.zeros((n, 3)) if grad else None
    lib().orc_coulomb_points(C.c_int(len(pos)), _p(pos), _p(q), C.c_double(Lx), C.c_double(Ly), C.c_double(g_cut),
                             C.c_double(z_min_above_top), C.c_long(n), _p(pts), _p(VC), _p(g))
    return (VC, g) if grad else VC


def sample_grid(sub, alpha, Lx, Ly, r_cut, nx, ny, nz, z0, hz, kinds, g_cut=37.0):
    """samples[ix][iy][iz][c] at (ix Lx/nx, iy Ly/ny, z0 + iz hz); kinds: 0 Pauli, 1 London, 2 Coulomb, 3 zero."""
    pos, e, R, q = _d(sub["pos"]), _d(sub["e"]), _d(sub["R"]), _d(sub["q"])
    kinds = _i(kinds); Nx, Ny = image_counts(Lx, Ly, r_cut)
    out = np.zeros((nx, ny, nz, len(kinds)))
    lib().orc_sample_grid(C.c_int(len(pos)), _p(pos), _p(e), _p(R), _p(q), C.c_double(alpha), C.c_double(Lx), C.c_double(Ly),
                          C.c_int(Nx), C.c_int(Ny), C.c_double(g_cut), C.c_int(nx), C.c_int(ny), C.c_int(nz),
                          C.c_double(z0), C.c_double(hz), C.c_int(len(kinds)), _p(kinds), _p(out))
    return out


def collocation_matrix(n, periodic):
    A = np.zeros((n, n))
    lib().orc_collocation_matrix(C.c_int(n), C.c_int(int(periodic)), _p(A))
    return A


def prefilter(samples, periodic=(1, 1, 0)):
    """samples [nx][ny][nz][C] -> B-spline coefficients (new array)."""
    data = _d(samples).copy()
    if data.ndim == 3:
        data = data[..., None]
    nx, ny, nz, nch = data.shape
    per = _i(periodic)
    lib().orc_prefilter(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(nch), _p(per), _p(data))
    return data


class OracleGrid:
    """Holds fp64 coefficients [nx][ny][nz][C] and the geometry; keeps the arrays alive."""

    def __init__(self, coef, Lx, Ly, z0, hz, periodic_xy=True):
        self.coef = _d(coef)
        if self.coef.ndim == 3:
            self.coef = self.coef[..., None]
        nx, ny, nz, nch = self.coef.shape
        self.Lx, self.Ly, self.z0, self.hz = float(Lx), float(Ly), float(z0), float(hz)
        self.c = Grid(nx, ny, nz, nch, Lx, Ly, hz, z0, int(periodic_xy), self.coef.ctypes.data)

    @property
    def shape(self):
        return self.coef.shape


def interp(grid, pos, coef, channels=False):
    pos = _d(pos).reshape(-1, 3); n = len(pos)
    coef = _d(coef).reshape(n, 4)
    E = np.zeros(n); F = np.zeros((n, 3))
    Vc = np.zeros((n, grid.c.nch)) if channels else None
    dVc = np.zeros((n, grid.c.nch, 3)) if channels else None
    lib().orc_interp(C.byref(grid.c), C.c_long(n), _p(pos), _p(coef), _p(E), _p(F), _p(Vc), _p(dVc))
    return (E, F, Vc, dVc) if channels else (E, F)


def atom_coefs(e, R, q, alpha):
    e, R, q = _d(e), _d(R), _d(q)
    out = np.zeros((len(e), 4))
    lib().orc_atom_coefs(C.c_int(len(e)), _p(e), _p(R), _p(q), C.c_double(alpha), _p(out))
    return out


class OracleTopology:
    """Widen a topology dict (see paper_2508_15522_b200.inputs) to fp64 and keep it alive."""

    def __init__(self, topo, coef):
        n = int(topo["n_atoms"])
        self.n = n
        k = self.k = {}
        k["mass"] = _d(topo["mass"]); k["coef"] = _d(coef).reshape(n, 4)
        k["q"] = _d(topo["q"]); k["lj_e"] = _d(topo["lj_e"]); k["lj_R"] = _d(topo["lj_R"])
        k["bond"] = _i(topo["bond"]).reshape(-1, 2); k["bond_k_r0"] = _d(topo["bond_k_r0"]).reshape(-1, 2)
        k["angle"] = _i(topo["angle"]).reshape(-1, 3); k["angle_k_t0"] = _d(topo["angle_k_t0"]).reshape(-1, 2)
        k["tors"] = _i(topo["tors"]).reshape(-1, 4); k["tors_k_n_p0"] = _d(topo["tors_k_n_p0"]).reshape(-1, 3)
        excl = topo.get("excl")
        k["excl"] = None if excl is None else np.ascontiguousarray(excl, dtype=np.uint8).reshape(n, n)
        rot_bond = topo.get("rot_bond")
        k["rot_bond"] = _i(rot_bond).reshape(-1, 2) if rot_bond is not None else np.zeros((0, 2), np.int32)
        rot_mask = topo.get("rot_mask")
        k["rot_mask"] = (np.ascontiguousarray(rot_mask, dtype=np.uint8).reshape(-1, n)
                         if rot_mask is not None else np.zeros((0, n), np.uint8))
        ref = topo.get("ref_pos")
        k["ref_pos"] = _d(ref).reshape(n, 3) if ref is not None else np.zeros((n, 3))
        self.c = Topology(n, _p(k["mass"]), _p(k["coef"]), _p(k["q"]), _p(k["lj_e"]), _p(k["lj_R"]),
                          len(k["bond"]), _p(k["bond"]), _p(k["bond_k_r0"]),
                          len(k["angle"]), _p(k["angle"]), _p(k["angle_k_t0"]),
                          len(k["tors"]), _p(k["tors"]), _p(k["tors_k_n_p0"]),
                          _p(k["excl"]),
                          len(k["rot_bond"]), _p(k["rot_bond"]), _p(k["rot_mask"]), _p(k["ref_pos"]))


def make_integrator(kind, n_steps, dt, f_tol=1e-3, dt_max=None, f_inc=1.1, f_dec=0.5, a_start=0.1, f_a=0.99,
                    n_min=5, restart=0, seed=0, z_ref=0.0, place_z_lo=3.0, place_z_hi=6.0, place_z_min=2.0, clash=0.4, max_step=0.0,
                    temperature=0.0, gamma=0.0, step0=0, n_scan=0, fixed=(), scan_dx=(0.0, 0.0, 0.0)):
    """kind: "vv", "fire" or "langevin" (BAOAB, R18).  `fixed`: indices of held atoms; n_scan > 0 with kind "fire" = driven scan."""
    kind = {"vv": 0, "fire": 1, "langevin": 2}.get(kind, kind)
    mask = 0
    for i in fixed:
        mask |= 1 << int(i)
    if dt_max is None:
        dt_max = 10.0 * dt
    return Integrator(int(kind), int(n_steps), dt, f_tol, dt_max, f_inc, f_dec, a_start, f_a, int(n_min), int(restart),
                      int(seed), z_ref, place_z_lo, place_z_hi, place_z_min, clash, max_step,
                      float(temperature), float(gamma), int(step0), int(n_scan), mask, (C.c_double * 3)(*[float(c) for c in scan_dx]))


def langevin_normals(seed, replica, step, atom):
    """the three standard normals the Langevin O-step draws for (replica, step, atom)"""
    xi = np.zeros(3)
    lib().orc_langevin_normals(C.c_uint64(int(seed)), C.c_uint32(int(replica)), C.c_uint32(int(step)), C.c_uint32(int(atom)), _p(xi))
    return xi


def intramolecular(otopo, pos):
    pos = _d(pos).reshape(-1, 3)
    F = np.zeros_like(pos); E4 = np.zeros(4)
    lib().orc_intramolecular(C.byref(otopo.c), _p(pos), _p(F), _p(E4))
    return E4, F


def forces(grid, otopo, pos):
    pos = _d(pos).reshape(-1, 3)
    F = np.zeros_like(pos); E7 = np.zeros(7)
    lib().orc_forces(C.byref(grid.c) if grid is not None else None, C.byref(otopo.c), _p(pos), _p(F), _p(E7))
    return E7, F


def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32); key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def restart_conformation(otopo, integ, Lx, Ly, replica, restart, with_attempt=False):
    pos = np.zeros((otopo.n, 3))
    a = lib().orc_restart_conformation(C.byref(otopo.c), C.byref(integ), C.c_double(Lx), C.c_double(Ly),
                                       C.c_uint32(replica), C.c_uint32(restart), _p(pos))
    return (pos, int(a)) if with_attempt else pos


def run_replicas(grid, otopo, integ, pos, vel, fire=None, minima_cap=0, trace=False):
    """Returns dict(pos, vel, fire, energy[n_rep][8], status[n_rep][2], minima, n_minima, e_trace, scan[n_rep][n_scan][4])."""
    n = otopo.n
    pos = _d(pos).reshape(-1, n, 3).copy(); vel = _d(vel).reshape(-1, n, 3).copy()
    n_rep = len(pos)
    fire = np.zeros((n_rep, 4)) if fire is None else _d(fire).reshape(n_rep, 4).copy()
    energy = np.zeros((n_rep, 8)); status = np.zeros((n_rep, 2), np.int32)
    minima = np.zeros((max(minima_cap, 1), 4 + 3 * n)); n_minima = C.c_long(0)
    e_trace = np.zeros((n_rep, integ.n_steps + 1)) if trace else None
    scan = np.zeros((n_rep, integ.n_scan, 4)) if integ.n_scan > 0 else None
    lib().orc_run_replicas(C.byref(grid.c) if grid is not None else None, C.byref(otopo.c), C.byref(integ), C.c_int(n_rep),
                           _p(pos), _p(vel), _p(fire), _p(energy), _p(status),
                           _p(minima) if minima_cap > 0 else None, C.c_long(minima_cap), C.byref(n_minima), _p(e_trace), _p(scan))
    nm = int(n_minima.value)
    return dict(pos=pos, vel=vel, fire=fire, energy=energy, status=status,
                minima=minima[:min(nm, minima_cap)], n_minima=nm, e_trace=e_trace, scan=scan)


# ---------------------------------------------------------------------------------------------------------------
# minima hopping with the unique-structure filter
# ---------------------------------------------------------------------------------------------------------------

def same_structure(E_a, x_a, E_b, x_b, Lx, Ly, e_tol=1e-3, rmsd_tol=0.1):
    """PAPER.md:L241 criterion as read in DESIGN.md R16: |dE| < e_tol and plain RMSD < rmsd_tol (0.1 Å) after removing the whole
    cell translation nearest to the mean displacement; no rotation, no atom permutation (adsorption site and orientation count)."""
    if not abs(E_a - E_b) < e_tol:
        return False
    d = np.asarray(x_a, np.float64) - np.asarray(x_b, np.float64)
    m = d.mean(axis=0)
    d = d - np.array([round(m[0] / Lx) * Lx, round(m[1] / Ly) * Ly, 0.0])
    return bool(np.sqrt((d ** 2).sum(axis=1).mean()) < rmsd_tol)


def unique_filter(library, cand_E, cand_x, cand_ok, Lx, Ly, e_tol=1e-3, rmsd_tol=0.1, cap=None, tag=0, steps=None):
    """Sequential greedy filter, candidates in replica order: a converged candidate that matches no library entry (old or added
    earlier in this call) is appended as {replica, tag, steps, E, positions}.  `library` is a list of 1-D records [4 + 3n]; returns
    (n_candidates, n_new, n_dropped)."""
    n_cand = n_new = n_drop = 0
    for r in range(len(cand_E)):
        if not cand_ok[r]:
            continue
        n_cand += 1
        x = np.asarray(cand_x[r], np.float64)
        if any(same_structure(cand_E[r], x, rec[3], rec[4:].reshape(-1, 3), Lx, Ly, e_tol, rmsd_tol) for rec in library):
            continue
        if cap is not None and len(library) >= cap:
            n_drop += 1
            continue
        library.append(np.concatenate([[r, tag, 0 if steps is None else steps[r], cand_E[r]], x.reshape(-1)]))
        n_new += 1
    return n_cand, n_new, n_drop


def minima_hopping(grid, otopo, pos, n_cycles, md_steps, md_dt, temperature, gamma, relax_steps, relax_dt, f_tol, seed,
                   dt_max=None, max_step=0.0, e_tol=1e-3, rmsd_tol=0.1, cap=None, cycle0=0, library=None):
    """per cycle, `md_steps` of Langevin dynamics at `temperature` from the current state (noise stream step index
    continues across cycles), FIRE relaxation from rest to max |F_i| < f_tol (at most relax_steps iterations), then the unique
    filter; every replica continues from its relaxed state (R19).  Returns dict(pos, library, stats [n_cycles][3])."""
    library = [] if library is None else library
    pos = _d(pos).copy(); stats = []
    for c in range(n_cycles):
        md = make_integrator("langevin", md_steps, md_dt, temperature=temperature, gamma=gamma, seed=seed, step0=(cycle0 + c) * md_steps)
        o = run_replicas(grid, otopo, md, pos, np.zeros_like(pos))
        fi = make_integrator("fire", relax_steps, relax_dt, f_tol=f_tol, dt_max=dt_max, max_step=max_step)
        o = run_replicas(grid, otopo, fi, o["pos"], np.zeros_like(pos))
        pos = o["pos"]
        E = o["energy"][:, :7].sum(axis=1)
        stats.append(unique_filter(library, E, pos, o["status"][:, 1] == 1, grid.c.Lx, grid.c.Ly, e_tol, rmsd_tol, cap, cycle0 + c, o["status"][:, 0]))
    return dict(pos=pos, library=library, stats=np.array(stats))


# ---------------------------------------------------------------------------------------------------------------
# interpolation variants — the trilinear foil and fp16 coefficient storage
# ---------------------------------------------------------------------------------------------------------------

def half_grid(grid):
    """the same spline with every coefficient rounded fp64 -> fp32 -> fp16 (IEEE round-to-nearest-even, numpy's casts): what a
    GRIDFF_LAYOUT_HALF store holds (it is derived from the fp32 store)."""
    c = grid.coef.astype(np.float32).astype(np.float16).astype(np.float64)
    return OracleGrid(c, grid.Lx, grid.Ly, grid.z0, grid.hz)


def trilinear_nodes(grid):
    """Node tables of the foil (R20): V [nx][ny][nz][C] = the spline at the nodes, G [nx][ny][nz][C][3] = its analytic
    gradient there, for iz in [1, nz-2]; zero at iz = 0 and nz-1 (not needed: cells are clamped to [1, nz-3]).  At a node the
    cubic B-spline weights are B(-1), B(0), B(1) = 1/6, 2/3, 1/6 and B'(1), B'(0), B'(-1) = -1/2, 0, 1/2 (Eq. 6)."""
    nx, ny, nz, nch = grid.shape
    b = grid.coef
    w = (1.0 / 6.0, 2.0 / 3.0, 1.0 / 6.0); d = (-0.5, 0.0, 0.5)
    h = (grid.Lx / nx, grid.Ly / ny, grid.hz)
    V = np.zeros((nx, ny, nz, nch)); G = np.zeros((nx, ny, nz, nch, 3))
    for a in range(3):
        for bb in range(3):
            for c in range(3):
                # coefficient (i - 1 + a, j - 1 + bb, k - 1 + c): periodic in x, y; k = 1 .. nz-2 in z
                blk = np.roll(np.roll(b, 1 - a, axis=0), 1 - bb, axis=1)[:, :, c:nz - 2 + c]
                V[:, :, 1:nz - 1] += w[a] * w[bb] * w[c] * blk
                G[:, :, 1:nz - 1, :, 0] += d[a] * w[bb] * w[c] / h[0] * blk
                G[:, :, 1:nz - 1, :, 1] += w[a] * d[bb] * w[c] / h[1] * blk
                G[:, :, 1:nz - 1, :, 2] += w[a] * w[bb] * d[c] / h[2] * blk
    return V, G


def interp_trilinear(grid, nodes, pos, coef):
    """energy and the three force components stored on the grid and interpolated independently, trilinearly over the 8
    corners of the cell.  Cell and domain rules are the spline's (R5, R6): x, y periodic, i_z clamped to [1, nz-3] with
    t_z = u_z - i_z (linear continuation below), E = F = 0 for u_z >= nz - 2.  Returns (E [n], F [n][3])."""
    V, G = nodes
    nx, ny, nz, nch = grid.shape
    pos = _d(pos).reshape(-1, 3); coef = _d(coef).reshape(len(pos), 4)
    E = np.zeros(len(pos)); F = np.zeros((len(pos), 3))
    for p in range(len(pos)):
        ux = (pos[p, 0] / grid.Lx - np.floor(pos[p, 0] / grid.Lx)) * nx
        uy = (pos[p, 1] / grid.Ly - np.floor(pos[p, 1] / grid.Ly)) * ny
        uz = (pos[p, 2] - grid.z0) / grid.hz
        if uz >= nz - 2:
            continue
        ix = min(int(np.floor(ux)), nx - 1); iy = min(int(np.floor(uy)), ny - 1)
        iz = min(max(int(np.floor(uz)), 1), nz - 3)
        tx, ty, tz = ux - ix, uy - iy, uz - iz
        for a in (0, 1):
            for b in (0, 1):
                for c in (0, 1):
                    w = (tx if a else 1 - tx) * (ty if b else 1 - ty) * (tz if c else 1 - tz)
                    jx, jy, jz = (ix + a) % nx, (iy + b) % ny, iz + c
                    for ch in range(nch):
                        E[p] += coef[p, ch] * w * V[jx, jy, jz, ch]
                        F[p] -= coef[p, ch] * w * G[jx, jy, jz, ch]
    return E, F
