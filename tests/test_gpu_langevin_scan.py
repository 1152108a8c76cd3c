"""GPU-vs-oracle parity for SURVEY.md §8(f) rows 1-2: Langevin dynamics (BAOAB, R18), held atoms and driven scans
(PAPER.md:L178, L184, L222), through the C-ABI (gridff_run_replicas kind 2, gridff_run_scan).  Run on the B200 box with -m gpu.

Both sides draw the same noise (Philox4x32-10 counter (step, atom, 'Lang', replica), 23-bit uniforms, Box-Muller), so Langevin
trajectories are compared like the velocity-Verlet ones: 100 steps within 1e-3 Å (north_star)."""
import numpy as np
import pytest
import torch

from paper_2508_15522_b200 import inputs
from gridff_cases import oracle_grid, gpu_grid, small_config
from test_gpu_parity import api, dev, oracle_side, gpu_side, run_gpu, check_energies, TRAJ_TOL  # noqa: F401

pytestmark = pytest.mark.gpu

KB = 8.617333262e-5


@pytest.mark.parametrize("k", [1, 2])
def test_langevin_trajectory_100_steps(api, orc, k):
    n_rep = 45 if k == 1 else 19                # more than one block, ragged; k = 2 is the 60-atom molecule (two atoms per lane)
    cfg = small_config(k, n_rep=n_rep)
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    g = gpu_grid(api, cfg["sub"], cfg["desc"])
    ot, mol = oracle_side(orc, cfg, og), gpu_side(api, cfg)
    vel = inputs.maxwell_boltzmann(cfg["topo"], n_rep, 300.0, 31)
    kw = dict(temperature=300.0, gamma=0.01, seed=4242, step0=7)
    r = run_gpu(api, g, mol, api.make_integrator("langevin", 100, 0.5, **kw), cfg["pos"], vel)
    o = orc.run_replicas(og, ot, orc.make_integrator("langevin", 100, 0.5, **kw), cfg["pos"], vel)
    dmax = np.abs(r["pos"].astype(np.float64) - o["pos"]).max()
    assert dmax <= TRAJ_TOL, dmax
    assert np.abs(r["vel"].astype(np.float64) - o["vel"]).max() <= 1e-4
    assert np.all(r["status"][:, 0] == 100)
    check_energies(r["energy"], o["energy"], tol_rel=1e-4, tol_abs=2e-4)
    # the noise really acted: the same start without friction ends elsewhere
    r0 = run_gpu(api, g, mol, api.make_integrator("vv", 100, 0.5), cfg["pos"], vel)
    assert np.abs(r0["pos"] - r["pos"]).max() > 1e-2


def test_langevin_launch_split_held_atoms_and_gas_phase(api, orc):
    cfg = small_config(1, n_rep=11)
    ot, mol = oracle_side(orc, cfg, None), gpu_side(api, cfg)
    vel = np.zeros_like(cfg["pos"])
    kw = dict(temperature=300.0, gamma=0.02, seed=99, fixed=(0, 17))
    r1 = run_gpu(api, None, mol, api.make_integrator("langevin", 90, 0.5, **kw), cfg["pos"], vel)
    p, v = cfg["pos"], vel
    for b in range(3):
        r3 = run_gpu(api, None, mol, api.make_integrator("langevin", 30, 0.5, step0=30 * b, **kw), p, v)
        p, v = r3["pos"], r3["vel"]
    assert np.array_equal(r1["pos"], r3["pos"]) and np.array_equal(r1["vel"], r3["vel"])          # 1 x 90 == 3 x 30, bit for bit
    assert np.array_equal(r1["pos"][:, [0, 17]], cfg["pos"][:, [0, 17]]) and np.all(r1["vel"][:, [0, 17]] == 0)
    o = orc.run_replicas(None, ot, orc.make_integrator("langevin", 90, 0.5, **kw), cfg["pos"], vel)
    assert np.abs(r1["pos"].astype(np.float64) - o["pos"]).max() <= TRAJ_TOL
    # run-to-run determinism
    r2 = run_gpu(api, None, mol, api.make_integrator("langevin", 90, 0.5, **kw), cfg["pos"], vel)
    assert np.array_equal(r1["pos"], r2["pos"])


def test_langevin_thermalises_to_the_set_temperature(api):
    """1024 gas-phase replicas from rest, 4000 steps at 300 K, gamma = 0.02 /fs: <E_kin> = 3/2 N kT within 3 % (BAOAB's
    O(dt^2) bias at dt = 0.5 fs + sampling error 0.5 %) — a property that holds at any size, checked in the bench-sized launch shape"""
    cfg = small_config(1, n_rep=1024)
    mol = gpu_side(api, cfg)
    vel = np.zeros_like(cfg["pos"])
    r = run_gpu(api, None, mol, api.make_integrator("langevin", 4000, 0.5, temperature=300.0, gamma=0.02, seed=5), cfg["pos"], vel)
    ek = r["energy"][:, 7].astype(np.float64).mean()
    assert abs(ek / (1.5 * 30 * KB * 300.0) - 1) < 0.03, ek
    assert np.all(np.isfinite(r["pos"]))


def run_scan(api, g, mol, integ, pos):
    d_pos = dev(pos); d_vel = torch.zeros_like(d_pos)
    out = api.gridff_run_scan(g, mol, integ, d_pos, d_vel)
    torch.cuda.synchronize()
    return dict(pos=d_pos.cpu().numpy(), scan=out["scan"].cpu().numpy(), energy=out["energy"].cpu().numpy(), status=out["status"].cpu().numpy())


def test_one_atom_scan_is_the_interpolated_potential(api, orc):
    """a single held atom: E(s) must be the interpolated potential along the path (oracle interp, 1e-5 relative)"""
    cfg = small_config(1, n_rep=1)
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    g = gpu_grid(api, cfg["sub"], cfg["desc"])
    coef = np.array([[0.8, -0.3, 0.2, 0.0]], np.float32)
    topo = dict(n_atoms=1, mass=np.array([12.0]), q=np.zeros(1), lj_e=np.zeros(1), lj_R=np.ones(1),
                bond=np.zeros((0, 2)), bond_k_r0=np.zeros((0, 2)), angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
                tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((1, 1), np.uint8))
    mol = api.gridff_create_molecule(topo, coef)
    n_rep = 70
    rng = np.random.default_rng(8)
    x0 = np.zeros((n_rep, 1, 3), np.float32)
    x0[:, 0, :2] = rng.uniform(0, cfg["desc"]["Lx"], (n_rep, 2)); x0[:, 0, 2] = rng.uniform(1.7, 2.5, n_rep)
    dx = (0.03, -0.02, 0.1)
    r = run_scan(api, g, mol, api.make_integrator("fire", 20, 0.5, n_scan=40, fixed=(0,), scan_dx=dx), x0)
    # the held atom's path as the kernel walks it (repeated fp32 additions)
    path = np.zeros((n_rep, 40, 3), np.float32); p = x0[:, 0].copy()
    for s in range(40):
        p = p + np.asarray(dx, np.float32); path[:, s] = p
    assert np.array_equal(r["pos"][:, 0], path[:, -1])
    E, _, Vc, _ = orc.interp(og, path.reshape(-1, 3).astype(np.float64), np.repeat(coef, n_rep * 40, 0), channels=True)
    den = np.sum(np.abs(coef[:, :3].astype(np.float64) * Vc), axis=1)
    assert (np.abs(r["scan"][..., 0].reshape(-1) - E) / den).max() <= 1e-5
    assert np.all(r["scan"][..., 1] == 0) and np.all(r["scan"][..., 2] == 1)
    assert np.all(r["status"][:, 0] == 0) and np.all(r["status"][:, 1] == 40)


def test_lift_scan_matches_oracle(api, orc):
    """benzene lifted by one held H atom in 0.1 Å steps: per scan point the relaxed energy, convergence flag and
    final geometry against the oracle.  Relaxation paths can bifurcate, so the comparison is on tightly converged
    points, like the basin tests: |dE| < 1e-3 eV there, and at least 90 % of the points."""
    cfg = small_config(0, n_rep=24)
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    g = gpu_grid(api, cfg["sub"], cfg["desc"])
    ot, mol = oracle_side(orc, cfg, og), gpu_side(api, cfg)
    # start flat, 3.2 Å above the surface, at seeded lateral positions
    rng = np.random.default_rng(3)
    pos = np.repeat(cfg["topo"]["ref_pos"][None], 24, 0).astype(np.float32)
    pos[..., 2] += 3.2
    pos[..., :2] += rng.uniform(0, cfg["desc"]["Lx"], (24, 1, 2)).astype(np.float32)
    kw = dict(f_tol=2e-3, dt_max=10.0, max_step=0.05, fixed=(6,), scan_dx=(0.0, 0.0, 0.1), n_scan=8)
    r = run_scan(api, g, mol, api.make_integrator("fire", 4000, 1.0, **kw), pos)
    o = orc.run_replicas(og, ot, orc.make_integrator("fire", 4000, 1.0, **kw), pos, np.zeros_like(pos))
    held_path = pos[:, 6, 2].astype(np.float64) + 0.8
    assert np.abs(r["pos"][:, 6, 2] - held_path).max() < 1e-5 and np.array_equal(r["pos"][:, 6, :2], pos[:, 6, :2])
    both = (r["scan"][..., 2] == 1) & (o["scan"][..., 2] == 1)
    assert both.mean() >= 0.9, both.mean()
    dE = np.abs(r["scan"][..., 0] - o["scan"][..., 0])[both]
    print("lift scan: %d/%d points converged on both sides, max |dE| %.2e eV, median iterations GPU %d oracle %d"
          % (both.sum(), both.size, dE.max(), np.median(r["scan"][..., 1]), np.median(o["scan"][..., 1])))
    assert dE.max() < 1e-3
    assert np.all(r["scan"][..., 3][r["scan"][..., 2] == 1] < 2e-3)
    # energy rises as the molecule is pulled off (last point above the first) on both sides
    assert np.all(r["scan"][:, -1, 0] > r["scan"][:, 0, 0] - 1e-3)
    # final geometry where every point converged on both sides
    ok = both.all(axis=1)
    assert ok.sum() >= 12
    assert np.abs(r["pos"][ok].astype(np.float64) - o["pos"][ok]).max() < 0.05


def test_drag_scan_across_a_vacancy_matches_oracle(api, orc):
    """SURVEY.md §8(f) rows 2 x 4, the paper's own protocol ("removing one Na and one Cl atoms next to each other from the topmost
    atomic layer", L200-202 dragging a molecule over the defect): benzene, held by one H atom, is dragged laterally in 0.1 Å steps across the
    vacancy pair of a 4x4-site, 3-layer slab, relaxing at every point.  Per scan point: relaxed energy, convergence flag against the oracle;
    the held atom follows the prescribed path exactly; and the defect is visible — the same drag over the perfect slab gives another E(s)."""
    sub0, Lx, Ly = inputs.rocksalt_slab(4, 3, 2.82, 0.7)
    sub, removed = inputs.vacancy_pair(sub0, Lx, Ly)
    desc = inputs.grid_desc(Lx, Ly, 0.0, 1.5, 7.5, 0.2, 1.6, [inputs.PAULI, inputs.LONDON, inputs.COULOMB])
    topo = inputs.benzene()
    topo["q"] = (0.12 * np.where(np.arange(12) < 6, -1.0, 1.0)).astype(np.float32)       # C-H bond dipoles: the Coulomb channel takes part
    coef = orc.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], 1.6)
    ot = orc.OracleTopology(topo, coef)
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(1.6, topo["grid_e"], topo["grid_R"], topo["q"]))
    centre = removed[:, :2].mean(axis=0)
    n_scan, held = 30, 6
    pos = inputs.drag_starts(topo, 20, held, centre - [1.5, 0.0], 3.3, 0.6, seed=21)
    kw = dict(f_tol=2e-3, dt_max=10.0, max_step=0.05, fixed=(held,), scan_dx=(0.1, 0.0, 0.0), n_scan=n_scan)
    E = {}
    for name, s_ in (("vacancy", sub), ("perfect", sub0)):
        og, _ = oracle_grid(orc, s_, desc)
        g = gpu_grid(api, s_, desc)
        r = run_scan(api, g, mol, api.make_integrator("fire", 10000, 1.0, **kw), pos)
        o = orc.run_replicas(og, ot, orc.make_integrator("fire", 10000, 1.0, **kw), pos, np.zeros_like(pos))
        assert np.abs(r["pos"][:, held, 0] - (pos[:, held, 0].astype(np.float64) + 0.1 * n_scan)).max() < 2e-5
        assert np.array_equal(r["pos"][:, held, 1:], pos[:, held, 1:])
        both = (r["scan"][..., 2] == 1) & (o["scan"][..., 2] == 1)
        dE = np.abs(r["scan"][..., 0] - o["scan"][..., 0])[both]
        print("drag over the %s slab: %d/%d points converged on both sides; |dE| median %.2e, 99 %% %.2e, max %.2e eV; points above 1 meV: %d"
              % (name, both.sum(), both.size, np.median(dE), np.quantile(dE, 0.99), dE.max(), (dE >= 1e-3).sum()))
        # relaxed scans can bifurcate ("<0.9 meV" between the paper's two codes on such paths): all but 1 % of the points within
        # 1 meV, none beyond 5 meV
        assert both.mean() >= 0.9 and np.mean(dE < 1e-3) >= 0.99 and dE.max() < 5e-3
        assert np.all(r["scan"][..., 3][r["scan"][..., 2] == 1] < 2e-3)
        E[name] = np.where(both, o["scan"][..., 0], np.nan)
    diff = np.nanmax(np.abs(E["vacancy"] - E["perfect"]))
    print("the vacancy changes the relaxed drag profile E(s) by up to %.1f meV" % (1e3 * diff))
    assert diff > 5e-3
