"""Shared builders for the parity tests: the same seeded inputs (paper_2508_15522_b200.inputs) go to the fp64 oracle and
to the CUDA library.  No method arithmetic here."""
import numpy as np

from paper_2508_15522_b200 import inputs

_ORACLE_GRIDS = {}


def oracle_grid(orc, sub, desc):
    """fp64 oracle coefficients for a grid descriptor dict (cached per process)."""
    nx, ny, nz = inputs.grid_dims(desc)
    key = (len(sub["pos"]), float(np.sum(sub["pos"])), desc["Lx"], desc["Ly"], nx, ny, nz, tuple(desc["channels"]), desc["alpha"])
    if key not in _ORACLE_GRIDS:
        z0 = desc["z_ref"] + desc["z_lo"]
        samples = orc.sample_grid(sub, desc["alpha"], desc["Lx"], desc["Ly"], desc["r_cut"], nx, ny, nz, z0, desc["spacing"], desc["channels"])
        coef = orc.prefilter(samples, (1, 1, 0))
        _ORACLE_GRIDS[key] = (orc.OracleGrid(coef, desc["Lx"], desc["Ly"], z0, desc["spacing"]), samples)
    return _ORACLE_GRIDS[key]


def gpu_desc(api, desc, layout=0, l2_persist=0, morse_window=0):
    return api.make_desc(desc["Lx"], desc["Ly"], desc["z_ref"], desc["z_lo"], desc["z_hi"], desc["spacing"], desc["alpha"],
                         desc["channels"], r_cut=desc["r_cut"], layout=layout, l2_persist=l2_persist, morse_window=morse_window)


def gpu_grid(api, sub, desc, layout=0, l2_persist=0, morse_window=0):
    d = gpu_desc(api, desc, layout, l2_persist, morse_window)
    return api.gridff_build_grid(d, sub["pos"], sub["e"], sub["R"], sub["q"])


def small_config(k, n_rep, spacing=0.1, z_hi=8.5):
    """config k on the 2x2-site slab (L = 5.64 Å for k <= 2, 8 Å for k = 3): a grid the oracle builds in about a second."""
    cfg = inputs.config(k, n_rep=n_rep, spacing=spacing, small=True)
    cfg["desc"]["z_hi"] = z_hi
    return cfg


def energy_denominator(coef, Vc):
    """sum_c |coef_c V_c| per atom — the no-cancellation denominator of the relative energy error (R14)."""
    return np.sum(np.abs(coef[:, :Vc.shape[1]] * Vc), axis=1)


def energy_scales(orc, og, topo, coef, pos, energy):
    """Per replica and energy term, the magnitude WITHOUT cancellation that a relative tolerance refers to (R14) — a tolerance
    scale only, never an expected value.  Grid channels: sum_i |coef_ic V_c(r_i)| (ch3 counted with ch2, gridff.h); bond / angle / torsion:
    sums of non-negative terms, i.e. the oracle's own value; non-bonded: the Coulomb pair sum with every charge replaced by |q| (all pair
    terms positive: the oracle evaluates sum |q_i q_j| k_e / r) plus |E_LJ| (charges set to zero); kinetic: the oracle's own value.
    `energy` = the oracle's [n_rep][8] for the same states."""
    pos = np.asarray(pos, np.float64)
    n_rep, n = pos.shape[:2]
    out = np.abs(np.asarray(energy, np.float64)).copy()
    if og is not None:
        cf = np.tile(np.asarray(coef, np.float64).reshape(n, 4), (n_rep, 1))
        _, _, Vc, _ = orc.interp(og, pos.reshape(-1, 3), cf, channels=True)
        mag = np.abs(cf[:, :Vc.shape[1]] * Vc).reshape(n_rep, n, -1).sum(axis=1)
        for c in range(mag.shape[1]):
            out[:, min(c, 2)] = mag[:, c] if c < 3 else out[:, 2] + mag[:, c]
    t_abs = orc.OracleTopology(dict(topo, q=np.abs(topo["q"]), lj_e=np.zeros_like(topo["lj_e"])), coef)
    t_lj = orc.OracleTopology(dict(topo, q=np.zeros_like(topo["q"])), coef)
    for r in range(n_rep):
        out[r, 6] = orc.intramolecular(t_abs, pos[r])[0][3] + abs(orc.intramolecular(t_lj, pos[r])[0][3])
    return out


def basin_match(Eg, xg, Eo, xo, Lx, Ly):
    """PAPER.md:L241 criterion as read in DESIGN.md R16: |dE| < 1e-3 eV and plain RMSD < 0.1 Å after removing whole lattice translations"""
    d = np.asarray(xg, np.float64) - np.asarray(xo, np.float64)
    shift = np.round(d.mean(axis=1)[:, :2] / [Lx, Ly]) * [Lx, Ly]
    d[:, :, :2] -= shift[:, None, :]
    rmsd = np.sqrt((d ** 2).sum(axis=2).mean(axis=1))
    return (np.abs(np.asarray(Eg, np.float64) - np.asarray(Eo, np.float64)) < 1e-3) & (rmsd < 0.1)


def chaos_margin(k0, n0, n):
    """Largest mismatch COUNT out of n that is consistent with the control's mismatch rate k0 / n0 (oracle vs the same oracle started 1e-6 Å
    away): the rate plus two binomial standard deviations plus one replica.  FIRE relaxation is chaotic (PAPER.md:L57, L180 bifurcations; a
    P <= 0 decision taken one step apart changes dt for the rest of the run), so WHICH minimum a far-from-minimum start reaches is only
    defined up to this floor; what is asserted is that the fp32 path adds nothing to it."""
    p = max(k0, 1) / max(n0, 1)
    return n * (k0 / max(n0, 1)) + 2.0 * np.sqrt(n * p * (1.0 - min(p, 1.0))) + 1.0
