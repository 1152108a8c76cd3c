"""Parity at BASELINE.json's FULL sizes, in the launch configurations bench.py times (config 1 is in test_gpu_parity.py).
Run on the B200 box with -m gpu.  The oracle replays sampled units of every config: replicas (configs 0, 1, 2, 3), points (configs 3, 4).
Config 3's 24 M-node, 4-channel grid is built ONCE per session by the fp64 oracle as it stands (2.6e11 pair terms: about 8 minutes on the
box's 16 cores — by far the longest item of the GPU suite) and every stored coefficient, 2^16 interpolated points and 16 sampled replicas
are compared with it; the older any-size properties (brute-force sums at nodes, variant bit-identity, energy conservation) stay."""
import time

import numpy as np
import pytest
import torch

from paper_2508_15522_b200 import inputs
from gridff_cases import oracle_grid, gpu_grid, energy_denominator
from gridff_cases import basin_match, chaos_margin
from test_gpu_parity import api, dev, oracle_side, gpu_side, run_gpu, check_energies, TRAJ_TOL, E_REL_TOL, F_ABS_TOL  # noqa: F401
from test_gpu_basins import control_run, polish

pytestmark = pytest.mark.gpu


def test_config0_full_size(api, orc):
    """config 0 as stated: 113 x 113 x 100 x 2-channel grid, 64 benzene replicas, 1000 FIRE steps — every replica against the oracle.
    First 30 iterations: trajectories; all 1000: basin assignment (polished end states, chaos control: see test_gpu_basins.py)."""
    cfg = inputs.config(0)
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    g = gpu_grid(api, cfg["sub"], cfg["desc"], l2_persist=1)
    assert g.info()["dims"] == (113, 113, 100) and cfg["pos"].shape == (64, 12, 3)
    ot, mol = oracle_side(orc, cfg, og), gpu_side(api, cfg)
    vel = np.zeros_like(cfg["pos"])
    mk = lambda n: orc.make_integrator("fire", n, 0.5, f_tol=1e-3)
    r30 = run_gpu(api, g, mol, api.make_integrator("fire", 30, 0.5, f_tol=1e-3), cfg["pos"], vel, fire=np.zeros((64, 4), np.float32))
    o30 = orc.run_replicas(og, ot, mk(30), cfg["pos"], vel)
    c30 = control_run(orc, og, ot, mk, 30, cfg["pos"], vel)
    # FIRE takes a discrete decision per step (P > 0 ?): replicas whose decision history agrees with the oracle's (same dt, a, counter at the
    # end), on the GPU and in the control, must track it to the trajectory tolerance
    same_hist = lambda a: np.all(np.isclose(a["fire"][:, :3], o30["fire"][:, :3], rtol=1e-5), axis=1)
    hist, hist_c = same_hist(r30), same_hist(c30)
    dev30 = np.abs(r30["pos"].astype(np.float64) - o30["pos"]).max(axis=(1, 2))
    print("config 0 full size, 30 FIRE steps: decision history same as the oracle's: gpu %d/64, control %d/64; max deviation %.2e Å"
          % (hist.sum(), hist_c.sum(), dev30[hist & hist_c].max()))
    assert np.all(dev30[hist & hist_c] <= TRAJ_TOL) and (~hist).sum() <= chaos_margin((~hist_c).sum(), 64, 64)
    r = run_gpu(api, g, mol, api.make_integrator("fire", 1000, 0.5, f_tol=1e-3), cfg["pos"], vel, fire=np.zeros((64, 4), np.float32))
    o = orc.run_replicas(og, ot, mk(1000), cfg["pos"], vel)
    c = control_run(orc, og, ot, mk, 1000, cfg["pos"], vel)
    (Eg, xg, cg), (Eo, xo, co), (Ec, xc, cc) = polish(orc, og, ot, r["pos"]), polish(orc, og, ot, o["pos"]), polish(orc, og, ot, c["pos"])
    Lx, Ly = cfg["desc"]["Lx"], cfg["desc"]["Ly"]
    ok = cg & co & cc
    diff, diff0 = ~basin_match(Eg, xg, Eo, xo, Lx, Ly)[ok], ~basin_match(Ec, xc, Eo, xo, Lx, Ly)[ok]
    print("config 0 full size: basin mismatch after 1000 FIRE steps: gpu-vs-oracle %d/%d, control (oracle with fp32 state) %d/%d; %d distinct basin energies"
          % (diff.sum(), ok.sum(), diff0.sum(), ok.sum(), len(np.unique(np.round(Eo[ok], 4)))))
    assert ok.sum() >= 60 and diff.sum() <= chaos_margin(diff0.sum(), ok.sum(), ok.sum())


def test_config2_full_size_sampled_replicas(api, orc):
    """config 2's launch: 16,384 replicas of the 60-atom chain (pair of warps per replica), FIRE with restart enabled.  60 iterations on the
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
    mk = lambda n: orc.make_integrator("fire", n, 0.5, **kw)
    o = orc.run_replicas(og, ot, mk(60), cfg["pos"][pick], vel[pick])
    c = control_run(orc, og, ot, mk, 60, cfg["pos"][pick], vel[pick], minima_cap=16)
    assert r["n_minima"] == 0 and np.all(o["status"][:, 1] == 0)
    same_hist = lambda f: np.all(np.isclose(f[:, :3], o["fire"][:, :3], rtol=1e-5), axis=1)
    hist, hist_c = same_hist(r["fire"][pick]), same_hist(c["fire"])
    dev = np.abs(r["pos"][pick].astype(np.float64) - o["pos"]).max(axis=(1, 2))
    must = hist & hist_c
    print("config 2 full size, 60 FIRE steps, 16 sampled replicas: decision history same as the oracle's: gpu %d, control %d; max deviation %.2e Å"
          % (hist.sum(), hist_c.sum(), dev[must].max()))
    assert must.sum() >= 6 and np.all(dev[must] <= TRAJ_TOL) and dev.max() < 0.05
    assert (~hist).sum() <= chaos_margin((~hist_c).sum(), 16, 16)
    check_energies(r["energy"][pick][must], o["energy"][must], tol_rel=1e-4, tol_abs=3e-4)
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
    # the 8-copy micro-brick store of the same grid (180 MB: beyond the L2, so the default takes the device-side choice: 5-D TMA boxes for the
    # random order, the LDG gather for the sorted one) returns the same numbers bit for bit, in the launch shape bench.py times
    gb = api.gridff_grid_derive(g, api.LAYOUT_MBRICK8)
    Eb, Fb = api.gridff_eval(gb, d_pos, d_coef)
    assert bool(torch.equal(Eb, E)) and bool(torch.equal(Fb, F))
    Eb, Fb = api.gridff_eval(gb, d_pos[perm].contiguous(), d_coef[perm].contiguous())
    assert bool(torch.equal(Eb, Es)) and bool(torch.equal(Fb, Fs))
    gb.free(); del gb, Eb, Fb
    # gridff_eval_binned (device-side counting sort of the points by cell block) over the same 2^26 points: the same numbers
    Eb, Fb = api.gridff_eval_binned(g, d_pos, d_coef)
    assert bool(torch.equal(Eb, E)) and bool(torch.equal(Fb, F))
    del Eb, Fb
    # the spatial sort did what it says: consecutive points share a cell far more often than in random order
    cell = lambda p: (torch.floor(p[:, 0] / d["Lx"] * 113) * 113 + torch.floor(p[:, 1] / d["Ly"] * 113)).long()
    c_s = cell(d_pos[perm][: 1 << 20]); c_r = cell(d_pos[: 1 << 20])
    assert float((c_s[1:] == c_s[:-1]).float().mean()) > 0.9 and float((c_r[1:] == c_r[:-1]).float().mean()) < 0.01


def test_config3_full_size_oracle_parity(api, orc):
    """config 3 (BASELINE.json configs[3]; PAPER.md:L208 20x20x3 substrate, L259-263 large supercells): 1200-atom slab, 400 x 400 x 150 x 4
    channels = 384 MB store.  Against the oracle's own fp64 grid: (1) every stored coefficient to half an fp32 ulp; (2) 2^16 random points at
    north_star's 1e-5 / 1e-4; (3) the 8192-replica launch, 100 velocity-Verlet steps, 16 sampled replicas at 1e-3 Å; (4) the launch shape
    bench.py --config 3 times (time-multiplexed blocks, >= 512 steps) equals, bit for bit, short un-multiplexed launches of the kind (3) checks."""
    cfg = inputs.config(3, n_rep=8192)
    d, sub = cfg["desc"], cfg["sub"]
    t0 = time.time()
    og, _ = oracle_grid(orc, sub, d)
    print("oracle built the config-3 grid %s in %.0f s on %d threads" % (og.shape, time.time() - t0, orc.num_threads()))
    assert og.shape == (400, 400, 150, 4)
    g = gpu_grid(api, sub, d, l2_persist=1)
    assert g.info()["dims"] == (400, 400, 150) and g.store.numel() > 380e6
    # (1)
    coef = api.gridff_grid_export(g)
    for c in range(4):
        ref = og.coef[..., c]
        got = coef[..., c].cpu().numpy()
        if c == 3:
            assert not got.any() and not ref.any()               # the ZERO channel
            continue
        scale = np.abs(ref).max()
        worst = 0.0
        for i0 in range(0, 400, 50):                              # in slabs: the fp64 difference of the whole array would be another 190 MB
            err = np.abs(got[i0:i0 + 50].astype(np.float64) - ref[i0:i0 + 50])
            assert np.all(err <= 6.0e-8 * np.abs(ref[i0:i0 + 50]) + 1e-9 * scale), (c, i0, err.max(), scale)
            worst = max(worst, float((err / (6.0e-8 * np.abs(ref[i0:i0 + 50]) + 1e-9 * scale)).max()))
        print("channel %d: all 24 M coefficients within the tolerance (half an fp32 ulp + 1e-9 of the channel's scale); worst uses %.2f of it" % (c, worst))
    del coef, got
    # (2)
    z0 = d["z_ref"] + d["z_lo"]
    pos, cf = inputs.c4_points(1 << 16, d["Lx"], d["Ly"], z0 + d["spacing"], z0 + 148 * d["spacing"] - 1e-3, seed=1003)
    E, F = api.gridff_eval(g, dev(pos), dev(cf))
    Eo, Fo, Vc, _ = orc.interp(og, pos, cf, channels=True)
    den = energy_denominator(cf.astype(np.float64), Vc)
    rel = np.abs(E.cpu().numpy() - Eo) / den
    dF = np.abs(F.cpu().numpy() - Fo).max()
    print("config 3 grid, 2^16 points: max rel energy error %.2e, max force error %.2e eV/Å" % (rel.max(), dF))
    assert rel.max() <= E_REL_TOL and dF <= F_ABS_TOL
    # (3)
    ot, mol = oracle_side(orc, cfg, og), gpu_side(api, cfg)
    r = run_gpu(api, g, mol, api.make_integrator("vv", 100, 0.5), cfg["pos"], cfg["vel"])
    pick = np.random.default_rng(3).choice(8192, 16, replace=False); pick[:2] = [0, 8191]
    o = orc.run_replicas(og, ot, orc.make_integrator("vv", 100, 0.5), cfg["pos"][pick], cfg["vel"][pick])
    dmax = np.abs(r["pos"][pick].astype(np.float64) - o["pos"]).max()
    print("config 3, 8192 replicas x 100 VV steps, 16 sampled: max deviation %.2e Å" % dmax)
    assert dmax <= TRAJ_TOL
    check_energies(r["energy"][pick], o["energy"], tol_rel=1e-4, tol_abs=2e-4)
    assert np.all(np.isfinite(r["pos"])) and np.all(r["status"][:, 0] == 100)
    # (4)
    one = run_gpu(api, g, mol, api.make_integrator("vv", 640, 0.5), cfg["pos"], cfg["vel"])
    p, v = cfg["pos"], cfg["vel"]
    for _ in range(8):
        rr = run_gpu(api, g, mol, api.make_integrator("vv", 80, 0.5), p, v)
        p, v = rr["pos"], rr["vel"]
    assert np.array_equal(one["pos"], p) and np.array_equal(one["vel"], v) and np.array_equal(one["energy"], rr["energy"])


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
