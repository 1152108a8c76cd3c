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
