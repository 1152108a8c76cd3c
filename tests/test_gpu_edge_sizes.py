"""Edge sizes of the fused replica kernel (run on the B200 box with -m gpu): molecules of 1, 2, 3, 4, 32 (a full warp, one atom per
lane), 33 (the first size with two atoms per lane), 61 and 64 (the maximum) atoms; replica counts of 1 and one more than a whole number
of blocks; zero replicas and zero steps.  Energies at the fixed state and 40-step velocity-Verlet and Langevin trajectories against
the oracle, on the small config-1 grid."""
import numpy as np
import pytest
import torch

from paper_2508_15522_b200 import inputs
from gridff_cases import oracle_grid, gpu_grid, small_config
from test_gpu_parity import api, dev, run_gpu, check_energies, TRAJ_TOL  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_atoms,n_rep", [(1, 5), (2, 8), (3, 15), (4, 1), (32, 29), (33, 17), (61, 9), (64, 10)])
def test_molecule_sizes(api, orc, n_atoms, n_rep):
    cfg = small_config(1, n_rep=1)
    d = cfg["desc"]
    og, _ = oracle_grid(orc, cfg["sub"], d)
    g = gpu_grid(api, cfg["sub"], d)
    topo = inputs.helix_chain(n_atoms, seed=100 + n_atoms)
    ot = orc.OracleTopology(topo, orc.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], d["alpha"]))
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(d["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    pos = inputs.place_replicas(topo, n_rep, d["Lx"], d["Ly"], 0.0, 77 + n_atoms)
    vel = inputs.maxwell_boltzmann(topo, n_rep, 300.0, 78)
    r0 = run_gpu(api, g, mol, api.make_integrator("vv", 0, 0.5), pos, vel)
    o0 = orc.run_replicas(og, ot, orc.make_integrator("vv", 0, 0.5), pos, vel)
    check_energies(r0["energy"], o0["energy"], tol_rel=3e-5, tol_abs=3e-5)
    for kind, kw in (("vv", {}), ("langevin", dict(temperature=300.0, gamma=0.02, seed=5))):
        r = run_gpu(api, g, mol, api.make_integrator(kind, 40, 0.5, **kw), pos, vel)
        o = orc.run_replicas(og, ot, orc.make_integrator(kind, 40, 0.5, **kw), pos, vel)
        assert np.abs(r["pos"].astype(np.float64) - o["pos"]).max() <= TRAJ_TOL, (kind, n_atoms)
        check_energies(r["energy"], o["energy"], tol_rel=1e-4, tol_abs=2e-4)
    # every variant agrees on the forces: 40 steps bit-identical between the cached and the gather-every-step kernels
    r2 = run_gpu(api, g, mol, api.make_integrator("vv", 40, 0.5, variant=2), pos, vel)
    r3 = run_gpu(api, g, mol, api.make_integrator("vv", 40, 0.5, variant=3), pos, vel)
    if n_atoms <= 32:
        assert np.array_equal(r2["pos"], r3["pos"])
    else:
        # above 32 atoms the default kernel puts the replica on a pair of warps (one atom per lane) while variant 2 keeps two atoms per lane:
        # the same forces summed in another order
        assert np.abs(r2["pos"] - r3["pos"]).max() <= 2e-5


def test_zero_replicas_and_too_many_atoms(api):
    cfg = small_config(1, n_rep=1)
    d = cfg["desc"]
    g = gpu_grid(api, cfg["sub"], d)
    topo = inputs.helix_chain(5)
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(d["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    empty = torch.zeros((0, 5, 3), device="cuda")
    out = api.gridff_run_replicas(g, mol, api.make_integrator("vv", 10, 0.5), empty, empty.clone())
    assert out["energy"].shape == (0, 8)
    E, F = api.gridff_eval(g, torch.zeros((0, 3), device="cuda"), torch.zeros((0, 4), device="cuda"))
    assert E.shape == (0,) and F.shape == (0, 3)
    big65 = inputs.helix_chain(65)
    with pytest.raises(api.GridffError):
        api.gridff_create_molecule(big65, np.zeros((65, 4), np.float32))
    with pytest.raises(api.GridffError):
        api.gridff_run_replicas(g, mol, api.make_integrator("vv", 10, 0.5, fixed=(7,)), dev(np.zeros((2, 5, 3))), dev(np.zeros((2, 5, 3))))


def test_many_atom_kinds_above_32_atoms(api, orc):
    """33-64 atoms: the pair-of-warps kernel reads (R_i + R_j)^2 and 12 e_i e_j from a per-kind table when the molecule has at most 8
    distinct Lennard-Jones kinds, and forms them per pair otherwise.  A 40-atom chain whose atoms all differ (40 kinds) takes the second
    path; both against the oracle, and against each other on a 2-kind chain whose parameters are the same numbers."""
    cfg = small_config(1, n_rep=1)
    d = cfg["desc"]
    og, _ = oracle_grid(orc, cfg["sub"], d)
    g = gpu_grid(api, cfg["sub"], d)
    topo = inputs.helix_chain(40, seed=9)
    many = dict(topo)
    many["lj_R"] = (topo["lj_R"] * (1.0 + 1e-3 * np.arange(40))).astype(np.float32)          # 40 distinct kinds
    pos = inputs.place_replicas(topo, 11, d["Lx"], d["Ly"], 0.0, 31)
    vel = inputs.maxwell_boltzmann(topo, 11, 300.0, 32)
    for t in (topo, many):
        ot = orc.OracleTopology(t, orc.atom_coefs(t["grid_e"], t["grid_R"], t["q"], d["alpha"]))
        mol = api.gridff_create_molecule(t, api.gridff_atom_coefs(d["alpha"], t["grid_e"], t["grid_R"], t["q"]))
        r = run_gpu(api, g, mol, api.make_integrator("vv", 40, 0.5), pos, vel)
        o = orc.run_replicas(og, ot, orc.make_integrator("vv", 40, 0.5), pos, vel)
        assert np.abs(r["pos"].astype(np.float64) - o["pos"]).max() <= TRAJ_TOL
        check_energies(r["energy"], o["energy"], tol_rel=1e-4, tol_abs=2e-4)
        r0 = run_gpu(api, g, mol, api.make_integrator("vv", 0, 0.5), pos, vel)
        o0 = orc.run_replicas(og, ot, orc.make_integrator("vv", 0, 0.5), pos, vel)
        check_energies(r0["energy"], o0["energy"], tol_rel=3e-5, tol_abs=3e-5)


def test_restart_needs_the_template_conformation(api):
    """gridff_integrator.restart = 1 re-seeds from gridff_topology.ref_pos: a molecule created without it is refused (GRIDFF_EINVAL), not run
    from an all-zero template"""
    cfg = small_config(1, n_rep=4)
    d = cfg["desc"]
    g = gpu_grid(api, cfg["sub"], d)
    topo = dict(cfg["topo"]); topo["ref_pos"] = None; topo["rot_bond"] = None; topo["rot_mask"] = None
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(d["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    p, v = dev(cfg["pos"]), dev(np.zeros_like(cfg["pos"]))
    with pytest.raises(api.GridffError) as e:
        api.gridff_run_replicas(g, mol, api.make_integrator("fire", 10, 0.5, restart=1, seed=1), p, v, d_fire=torch.zeros((4, 4), device="cuda"))
    assert e.value.code == -1 and "ref_pos" in str(e.value)
    out = api.gridff_run_replicas(g, mol, api.make_integrator("fire", 10, 0.5), p, v, d_fire=torch.zeros((4, 4), device="cuda"))     # without restart: fine
    torch.cuda.synchronize()
    assert bool(torch.isfinite(p).all()) and out["status"][:, 0].max().item() == 10
