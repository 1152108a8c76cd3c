"""Parity at BASELINE.json's FULL sizes, in the launch configurations bench.py times (config 1 is in test_gpu_parity.py).
Run on the B200 box with -m gpu.  Where the oracle can replay sampled units it does (configs 0, 2, 4); config 3's 24 M-node grid is
beyond what the fp64 CPU oracle builds in test time (2.6e11 pair terms), so it is checked through what holds at any size: at sampled
grid NODES the interpolant must return the un-approximated potential (the oracle's brute-force periodic sums, O4) to fp32 accuracy,
between nodes it must stay within the stated approximation error, and the kernel variants must agree bit for bit."""
import numpy as np
import pytest
import torch

from paper_2508_15522_b200 import inputs
from gridff_cases import oracle_grid, gpu_grid, energy_denominator
from test_gpu_parity import api, dev, oracle_side, gpu_side, run_gpu, check_energies, basin_match, TRAJ_TOL, E_REL_TOL, F_ABS_TOL  # noqa: F401

pytestmark = pytest.mark.gpu


def test_config0_full_size(api, orc):
    """config 0 as stated: 113 x 113 x 100 x 2-channel grid, 64 benzene replicas, 1000 FIRE steps — every replica against the oracle"""
    cfg = inputs.config(0)
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    g = gpu_grid(api, cfg["sub"], cfg["desc"], l2_persist=1)
    assert g.info()["dims"] == (113, 113, 100) and cfg["pos"].shape == (64, 12, 3)
    ot, mol = oracle_side(orc, cfg, og), gpu_side(api, cfg)
    vel = np.zeros_like(cfg["pos"])
    r60 = run_gpu(api, g, mol, api.make_integrator("fire", 30, 0.5, f_tol=1e-3), cfg["pos"], vel, fire=np.zeros((64, 4), np.float32))
    o60 = orc.run_replicas(og, ot, orc.make_integrator("fire", 30, 0.5, f_tol=1e-3), cfg["pos"], vel)
    # FIRE takes a discrete decision per step (P > 0 ?): replicas whose decision history agrees with the oracle's (same dt, a, counter at
    # the end) must track it to the trajectory tolerance; a decision taken one step apart changes dt for the rest of the run
    hist = np.all(np.isclose(r60["fire"][:, :3], o60["fire"][:, :3], rtol=1e-5), axis=1)
    assert hist.mean() >= 0.8, hist.mean()
    dev60 = np.abs(r60["pos"].astype(np.float64) - o60["pos"]).max(axis=(1, 2))
    assert np.mean(dev60[hist] <= TRAJ_TOL) >= 0.95 and dev60.max() < 0.05, (dev60[hist].max(), dev60.max())
    r = run_gpu(api, g, mol, api.make_integrator("fire", 1000, 0.5, f_tol=1e-3), cfg["pos"], vel, fire=np.zeros((64, 4), np.float32))
    o = orc.run_replicas(og, ot, orc.make_integrator("fire", 1000, 0.5, f_tol=1e-3), cfg["pos"], vel)
    Eg, Eo = r["energy"][:, :7].astype(np.float64).sum(1), o["energy"][:, :7].sum(1)
    same = basin_match(Eg, r["pos"], Eo, o["pos"], cfg["desc"]["Lx"], cfg["desc"]["Ly"])
    print("config 0 full size: %d/64 replicas end in the oracle's state after 1000 FIRE steps" % same.sum())
    # 1000 steps leave most replicas unconverged (R13), i.e. still moving along soft modes where a one-step difference in a
    # FIRE decision shifts the stopping point by more than the 0.1 Å of the basin criterion: measured 58/64; the bar is 85 %
    assert same.mean() >= 0.85


def test_config2_full_size_sampled_replicas(api, orc):
    """config 2's launch: 16,384 replicas of the 60-atom chain (two atoms per lane), FIRE with restart enabled.  60 iterations on the
    GPU; 16 sampled replicas replayed by the oracle (no replica converges that early, so no restart interferes)."""
    cfg = inputs.config(2)
    assert cfg["pos"].shape == (16384, 60, 3)
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    g = gpu_grid(api, cfg["sub"], cfg["desc"], l2_persist=1)
    ot, mol = oracle_side(orc, cfg, og), gpu_side(api, cfg)
    kw = dict(f_tol=1e-3, dt_max=20.0, max_step=0.1, restart=1, seed=1002)
    vel = np.zeros_like(cfg["pos"])
    r = run_gpu(api, g, mol, api.make_integrator("fire", 60, 0.5, **kw), cfg["pos"], vel, fire=np.zeros((16384, 4), np.float32), minima_cap=64)
    pick = np.random.default_rng(1).choice(16384, 16, replace=False); pick[:2] = [0, 16383]
    o = orc.run_replicas(og, ot, orc.make_integrator("fire", 60, 0.5, **kw), cfg["pos"][pick], vel[pick])
    assert r["n_minima"] == 0 and np.all(o["status"][:, 1] == 0)
    hist = np.all(np.isclose(r["fire"][pick, :3], o["fire"][:, :3], rtol=1e-5), axis=1)
    assert hist.sum() >= 11, hist.sum()
    dev = np.abs(r["pos"][pick].astype(np.float64) - o["pos"]).max(axis=(1, 2))
    assert np.mean(dev[hist] <= TRAJ_TOL) >= 0.9 and dev.max() < 0.05, (dev[hist].max(), dev.max())
    hist &= dev <= TRAJ_TOL
    check_energies(r["energy"][pick][hist], o["energy"][hist], tol_rel=1e-4, tol_abs=3e-4)
    assert np.all(np.isfinite(r["pos"])) and np.all(r["status"][:, 0] == 60)


def test_config4_full_size_sampled_points_and_order(api, orc):
    """config 4: 2^26 random points on the config-1 grid in one launch.  4096 sampled outputs against the oracle; the Morton-sorted
    order must give the same numbers, bit for bit, as the random order (a point's result does not depend on its neighbours)."""
    cfg = inputs.config(1, n_rep=1)
    d = cfg["desc"]
    og, _ = oracle_grid(orc, cfg["sub"], d)
    g = gpu_grid(api, cfg["sub"], d, l2_persist=1)
    n = 1 << 26
    pos, coef = inputs.c4_points(n, d["Lx"], d["Ly"], 1.6, 11.3 - 1e-3)
    d_pos, d_coef = torch.from_numpy(pos).cuda(), torch.from_numpy(coef).cuda()
    E, F = api.gridff_eval(g, d_pos, d_coef)
    pick = np.random.default_rng(2).choice(n, 4096, replace=False); pick[:2] = [0, n - 1]
    Eo, Fo, Vc, _ = orc.interp(og, pos[pick], coef[pick], channels=True)
    den = energy_denominator(coef[pick].astype(np.float64), Vc)
    tp = torch.from_numpy(pick).cuda()
    assert (np.abs(E[tp].cpu().numpy() - Eo) / den).max() <= E_REL_TOL
    assert np.abs(F[tp].cpu().numpy() - Fo).max() <= F_ABS_TOL
    assert bool(torch.isfinite(E).all()) and bool(torch.isfinite(F).all())
    perm = inputs.morton_order(d_pos, d["Lx"], d["Ly"], d["z_ref"] + d["z_lo"], 113, 113, d["spacing"], xp=torch)
    Es, Fs = api.gridff_eval(g, d_pos[perm].contiguous(), d_coef[perm].contiguous())
    assert bool(torch.equal(Es, E[perm])) and bool(torch.equal(Fs, F[perm]))
    # the spatial sort did what it says: consecutive points share a cell far more often than in random order
    cell = lambda p: (torch.floor(p[:, 0] / d["Lx"] * 113) * 113 + torch.floor(p[:, 1] / d["Ly"] * 113)).long()
    c_s = cell(d_pos[perm][: 1 << 20]); c_r = cell(d_pos[: 1 << 20])
    assert float((c_s[1:] == c_s[:-1]).float().mean()) > 0.9 and float((c_r[1:] == c_r[:-1]).float().mean()) < 0.01


def test_config3_full_size_properties(api, orc):
    """config 3: 1200-atom slab, 400 x 400 x 150 x 4-channel grid (384 MB store, beyond L2), 8192 replicas."""
    cfg = inputs.config(3, n_rep=8192)
    d, sub = cfg["desc"], cfg["sub"]
    g = gpu_grid(api, sub, d, l2_persist=1)
    info = g.info()
    assert info["dims"] == (400, 400, 150) and g.store.numel() > 380e6
    # (1) at grid nodes the interpolating spline returns the sample, i.e. the brute-force potential (oracle O4) — per channel
    rng = np.random.default_rng(4)
    m = 600
    idx = np.stack([rng.integers(0, 400, m), rng.integers(0, 400, m), rng.integers(1, 147, m)], 1)
    idx[:4] = [[0, 0, 1], [399, 399, 146], [0, 399, 70], [200, 0, 1]]
    hx = d["Lx"] / 400
    nodes = np.stack([idx[:, 0] * hx, idx[:, 1] * hx, d["z_ref"] + d["z_lo"] + idx[:, 2] * d["spacing"]], 1)
    VP, VL = orc.morse_points(sub, d["alpha"], d["Lx"], d["Ly"], d["r_cut"], nodes)
    VC = orc.coulomb_points(sub, d["Lx"], d["Ly"], nodes)
    for ch, V in enumerate((VP, VL, VC)):
        cf = np.zeros((m, 4), np.float32); cf[:, ch] = 1.0
        # fp32 positions of nodes are off the exact node by ~1e-6 Å: |dV| <= |grad V| 2e-6, inside the tolerance below
        E, _ = api.gridff_eval(g, dev(nodes), dev(cf))
        err = np.abs(E.cpu().numpy() - V)
        assert np.all(err <= 2e-5 * np.abs(V) + 1e-7 * np.abs(V).max()), (ch, (err / np.abs(V)).max())
    # (2) between nodes: within the stated approximation error of the spline at h = 0.1 Å (energy <= 1e-4 relative
    #     per channel for z >= 1.7 Å), forces against the brute-force gradient <= 2e-3 relative
    pts = np.stack([rng.uniform(0, d["Lx"], m), rng.uniform(0, d["Ly"], m), rng.uniform(1.7, 8.0, m)], 1)
    out = orc.morse_points(sub, d["alpha"], d["Lx"], d["Ly"], d["r_cut"], pts, grad=True)
    VP, VL, gP, gL = out
    for ch, (V, G) in enumerate(((VP, gP), (VL, gL))):
        cf = np.zeros((m, 4), np.float32); cf[:, ch] = 1.0
        E, F = api.gridff_eval(g, dev(pts), dev(cf))
        assert (np.abs(E.cpu().numpy() - V) / np.abs(V)).max() <= 1e-4
        assert (np.abs(F.cpu().numpy() + G).max(axis=1) / np.abs(G).max(axis=1)).max() <= 2e-3
    # (3) the replica kernel on the HBM-resident grid: cached-stencil variant == gather-every-step variant, bit for bit, all 8192 replicas
    mol = gpu_side(api, cfg)
    r3 = run_gpu(api, g, mol, api.make_integrator("vv", 200, 0.5, variant=3), cfg["pos"], cfg["vel"])
    r2 = run_gpu(api, g, mol, api.make_integrator("vv", 200, 0.5, variant=2), cfg["pos"], cfg["vel"])
    assert np.array_equal(r3["pos"], r2["pos"]) and np.array_equal(r3["energy"], r2["energy"])
    assert np.all(np.isfinite(r3["pos"])) and np.all(r3["status"][:, 0] == 200)
    # total energy is conserved over the 200 steps within the velocity-Verlet fluctuation band (as in test_vv_energy_conservation_gpu)
    r0 = run_gpu(api, g, mol, api.make_integrator("vv", 0, 0.5), cfg["pos"], cfg["vel"])
    e0, e1 = r0["energy"].astype(np.float64).sum(1), r3["energy"].astype(np.float64).sum(1)
    assert np.all(np.abs(e1 - e0) <= 0.05 * r0["energy"][:, 7] + 2e-3)


@pytest.mark.parametrize("kind", ["vv", "langevin"])
def test_config1_time_multiplexed_launch_is_bit_identical(api, kind):
    """The bench's launch shape (4096 replicas, >= 512 steps) runs the fixed-length integrators time-multiplexed: each block owns 14
    replicas and cycles them over its 8 warps in 8 chunks of steps, the state passing through the pos / vel arrays between rounds.
    It must equal, bit for bit, eight short launches (80 steps each: below the multiplexing threshold, one replica per warp) — which in
    turn are compared with the oracle in test_config1_full_grid_sampled_replicas and test_langevin_trajectory_100_steps."""
    cfg = inputs.config(1)
    g = gpu_grid(api, cfg["sub"], cfg["desc"], l2_persist=1)
    mol = gpu_side(api, cfg)
    kw = dict(temperature=300.0, gamma=0.01, seed=11) if kind == "langevin" else {}
    one = run_gpu(api, g, mol, api.make_integrator(kind, 640, 0.5, **kw), cfg["pos"], cfg["vel"])
    p, v = cfg["pos"], cfg["vel"]
    for b in range(8):
        kw_b = dict(kw, step0=80 * b) if kind == "langevin" else kw
        r = run_gpu(api, g, mol, api.make_integrator(kind, 80, 0.5, **kw_b), p, v)
        p, v = r["pos"], r["vel"]
    assert np.array_equal(one["pos"], p) and np.array_equal(one["vel"], v)
    assert np.array_equal(one["energy"], r["energy"])
    assert np.all(one["status"][:, 0] == 640) and np.all(np.isfinite(one["pos"]))
    # ragged replica counts: a last block with fewer replicas than warps, and one with more
    for n_rep in (2369, 4001):
        a = run_gpu(api, g, mol, api.make_integrator(kind, 520, 0.5, **kw), cfg["pos"][:n_rep], cfg["vel"][:n_rep])
        assert np.array_equal(a["pos"][:64], run_gpu(api, g, mol, api.make_integrator(kind, 520, 0.5, **kw), cfg["pos"][:64], cfg["vel"][:64])["pos"])
        assert np.all(np.isfinite(a["pos"])) and np.all(a["status"][:, 0] == 520)


def test_time_multiplexed_two_atoms_per_lane(api):
    """the same bit-identity for a molecule above 32 atoms (one block of 8 warps per SM): 1400 replicas of a 40-atom chain"""
    from gridff_cases import small_config
    cfg = small_config(1, n_rep=1)
    d = cfg["desc"]
    g = gpu_grid(api, cfg["sub"], d)
    topo = inputs.helix_chain(40, seed=3)
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(d["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    pos = inputs.place_replicas(topo, 1400, d["Lx"], d["Ly"], 0.0, 5)
    vel = inputs.maxwell_boltzmann(topo, 1400, 300.0, 6)
    one = run_gpu(api, g, mol, api.make_integrator("vv", 560, 0.5), pos, vel)
    p, v = pos, vel
    for _ in range(7):
        r = run_gpu(api, g, mol, api.make_integrator("vv", 80, 0.5), p, v)
        p, v = r["pos"], r["vel"]
    assert np.array_equal(one["pos"], p) and np.array_equal(one["vel"], v) and np.array_equal(one["energy"], r["energy"])
