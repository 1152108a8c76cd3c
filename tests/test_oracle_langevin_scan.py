"""Pins for the oracle's SURVEY.md §8(f) rows 1-2: Langevin dynamics (BAOAB, R18), held atoms and driven scans
(PAPER.md:L178, L184, L222).  CPU only.  Each pin is something the mathematics fixes independently of the oracle's code:
the gamma = 0 limit, the exact Ornstein-Uhlenbeck decay and stationary variance, equipartition, the moments of the normal
deviates, and a one-atom scan that must reproduce the interpolated potential itself."""
import math

import numpy as np
import pytest

from paper_2508_15522_b200 import inputs

ACC = 9.648533212e-3
KB = 8.617333262e-5


def _free_atoms(orc, n, masses):
    topo = dict(n_atoms=n, mass=np.asarray(masses, float), q=np.zeros(n), lj_e=np.zeros(n), lj_R=np.ones(n),
                bond=np.zeros((0, 2)), bond_k_r0=np.zeros((0, 2)), angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
                tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((n, n), np.uint8))
    return orc.OracleTopology(topo, np.zeros((n, 4)))


def test_normal_deviates_moments_and_stream_layout(orc):
    """Box-Muller on Philox4x32-10 (itself pinned against a big-integer restatement in test_oracle_integrators): mean 0, variance 1,
    kurtosis 3, independent components; distinct (replica, step, atom) give distinct draws."""
    xs = np.array([orc.langevin_normals(99, r, s, a) for r in range(4) for s in range(500) for a in range(32)])   # 64000 x 3
    n = xs.size
    assert abs(xs.mean()) < 4 / math.sqrt(n)
    assert abs(xs.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((xs ** 4).mean() - 3) < 4 * math.sqrt(96 / n)
    c = np.corrcoef(xs.T)
    assert np.abs(c - np.eye(3)).max() < 4 / math.sqrt(len(xs))
    assert len({tuple(np.round(x, 12)) for x in xs}) == len(xs)
    # the first two components are one Box-Muller pair: x0^2 + x1^2 = -2 ln u0 is exponential with mean 2
    r2 = xs[:, 0] ** 2 + xs[:, 1] ** 2
    assert abs(r2.mean() - 2) < 4 * 2 / math.sqrt(len(xs))
    # u = ((x >> 9) + 1/2) 2^-23 bounds the radius: sqrt(-2 ln 2^-24) = 5.768
    assert np.abs(xs).max() < 5.77


def test_langevin_without_friction_is_velocity_verlet(orc):
    topo = inputs.tetracene()
    t = orc.OracleTopology(topo, np.zeros((30, 4)))
    rng = np.random.default_rng(5)
    pos = (topo["ref_pos"] + rng.normal(0, 0.03, (30, 3)))[None]
    vel = inputs.maxwell_boltzmann(topo, 1, 300.0, 4).astype(float)
    a = orc.run_replicas(None, t, orc.make_integrator("vv", 200, 0.5), pos, vel)
    b = orc.run_replicas(None, t, orc.make_integrator("langevin", 200, 0.5, temperature=300.0, gamma=0.0, seed=3), pos, vel)
    assert np.abs(a["pos"] - b["pos"]).max() < 1e-11 and np.abs(a["vel"] - b["vel"]).max() < 1e-12
    assert np.abs(a["energy"] - b["energy"]).max() < 1e-10


def test_langevin_free_particle_ou_decay_and_equilibrium(orc):
    """No forces: B and A steps leave v alone, so v_n = c1^n v_0 + noise with stationary variance kT/m per component (exact for
    any dt): <v_n> = exp(-gamma n dt) v_0 and, after many relaxation times, <v^2> = kT/m."""
    masses = [1.008, 12.011, 15.999, 35.453] * 8
    t = _free_atoms(orc, 32, masses)
    n_rep, T, gamma, dt = 600, 300.0, 0.02, 0.5
    pos = np.zeros((n_rep, 32, 3)); v0 = np.zeros((n_rep, 32, 3)); v0[..., 0] = 0.05
    o = orc.run_replicas(None, t, orc.make_integrator("langevin", 40, dt, temperature=T, gamma=gamma, seed=11), pos, v0)
    m = np.asarray(masses)
    sig = np.sqrt(KB * T / m * ACC)                                   # Å/fs
    c1n = math.exp(-gamma * dt * 40)
    mean_vx = o["vel"][..., 0].mean(0)                                 # per atom, over replicas
    se = sig * math.sqrt(1 - c1n ** 2) / math.sqrt(n_rep)
    assert np.all(np.abs(mean_vx - c1n * 0.05) < 4.5 * se)
    # 1000 steps = 10 relaxation times: stationary
    o2 = orc.run_replicas(None, t, orc.make_integrator("langevin", 1000, dt, temperature=T, gamma=gamma, seed=12), pos, v0)
    var = (o2["vel"] ** 2).mean(axis=(0, 2))                          # per atom over replicas x components
    n_s = 3 * n_rep
    assert np.all(np.abs(var / sig ** 2 - 1) < 4.5 * math.sqrt(2 / n_s))
    # kinetic energy output: <E_kin> = 3/2 N kT
    assert abs(o2["energy"][:, 7].mean() / (1.5 * 32 * KB * T) - 1) < 4.5 * math.sqrt(2 / (3 * 32 * n_rep))
    # positions: the textbook OU displacement from a fixed v_0 — mean v_0 (1 - e^{-gt})/g along x, variance per component
    # (kT/m)/g^2 [2 g t - 3 + 4 e^{-g t} - e^{-2 g t}]; discrete BAOAB differs by O(g dt) = 1 %, sampling error 3 % (600 replicas x 3)
    t_tot = 1000 * dt; gt = gamma * t_tot
    var_x = sig ** 2 / gamma ** 2 * (2 * gt - 3 + 4 * math.exp(-gt) - math.exp(-2 * gt))
    drift = 0.05 * (1 - math.exp(-gt)) / gamma
    var_pos = o2["pos"].var(axis=0).mean(-1)                         # per atom: variance over replicas, averaged over x, y, z
    assert np.all(np.abs(var_pos / var_x - 1) < 0.15)
    assert np.all(np.abs(o2["pos"][..., 0].mean(0) - drift) < 4.5 * np.sqrt(var_x / n_rep))


def test_langevin_equipartition_bonded_molecule(orc):
    """benzene in the gas phase at 300 K, dt 0.25 fs: <E_kin> = 3/2 N kT within BAOAB's O(dt^2) bias (< 2 %) + sampling error."""
    topo = inputs.benzene()
    t = orc.OracleTopology(topo, np.zeros((12, 4)))
    n_rep = 64
    pos = np.repeat(topo["ref_pos"][None], n_rep, 0)
    vel = np.zeros_like(pos)
    ek = []
    p, v = pos, vel
    for blk in range(6):
        o = orc.run_replicas(None, t, orc.make_integrator("langevin", 800, 0.25, temperature=300.0, gamma=0.02, seed=21, step0=800 * blk), p, v)
        p, v = o["pos"], o["vel"]
        if blk >= 2:
            ek.append(o["energy"][:, 7])
    ek = np.concatenate(ek)
    assert abs(ek.mean() / (1.5 * 12 * KB * 300.0) - 1) < 0.04
    assert np.all(np.isfinite(p))


def test_langevin_launch_split_and_held_atoms(orc):
    topo = inputs.tetracene()
    t = orc.OracleTopology(topo, np.zeros((30, 4)))
    pos = np.repeat(topo["ref_pos"][None], 3, 0).astype(float); vel = np.zeros_like(pos)
    kw = dict(temperature=300.0, gamma=0.01, seed=77, fixed=(0, 7))
    a = orc.run_replicas(None, t, orc.make_integrator("langevin", 120, 0.5, **kw), pos, vel)
    p, v = pos, vel
    for k in range(3):
        o = orc.run_replicas(None, t, orc.make_integrator("langevin", 40, 0.5, step0=40 * k, **kw), p, v); p, v = o["pos"], o["vel"]
    assert np.array_equal(a["pos"], p) and np.array_equal(a["vel"], v)
    assert np.array_equal(a["pos"][:, [0, 7]], pos[:, [0, 7]]) and np.all(a["vel"][:, [0, 7]] == 0)
    assert np.abs(a["pos"] - pos).max() > 1e-3                        # the others did move
    # replicas draw different noise
    assert np.abs(a["pos"][0] - a["pos"][1]).max() > 1e-4


def test_one_atom_scan_reproduces_the_potential(orc, small_grid):
    """A single held atom has nothing to relax: every scan point converges at once and E(s) is the interpolated potential at
    x0 + (s + 1) dx — compared with orc.interp (pinned elsewhere against brute-force sums and finite differences)."""
    og, _ = small_grid
    coef = np.array([[0.8, -0.3, 0.2, 0.0]])
    t_ = dict(n_atoms=1, mass=np.array([12.0]), q=np.zeros(1), lj_e=np.zeros(1), lj_R=np.ones(1),
              bond=np.zeros((0, 2)), bond_k_r0=np.zeros((0, 2)), angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
              tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((1, 1), np.uint8))
    t = orc.OracleTopology(t_, coef)
    x0 = np.array([[[1.3, 2.1, 2.0]]]); dx = (0.05, -0.02, 0.1)
    o = orc.run_replicas(og, t, orc.make_integrator("fire", 50, 0.5, n_scan=30, fixed=(0,), scan_dx=dx), x0, np.zeros_like(x0))
    pts = x0[0, 0] + np.outer(np.arange(1, 31), dx)
    E, _ = orc.interp(og, pts, np.repeat(coef, 30, 0))
    assert np.abs(o["scan"][0, :, 0] - E).max() < 1e-13
    assert np.all(o["scan"][0, :, 1] == 0) and np.all(o["scan"][0, :, 2] == 1) and np.all(o["scan"][0, :, 3] == 0)
    assert np.allclose(o["pos"][0, 0], pts[-1], atol=1e-12)


def test_lift_scan_relaxes_below_the_rigid_curve(orc, small_grid):
    """benzene lifted by one held H atom: at every scan point the relaxed energy is <= the energy of the rigidly
    translated start geometry at that point minus nothing gained... i.e. relaxation never raises E; the held atom follows the
    prescribed path exactly; converged points have max |F_i| < f_tol over the free atoms."""
    og, _ = small_grid
    topo = inputs.benzene()
    from oracle import gridff_oracle as o_
    coef = o_.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], 1.6)
    t = orc.OracleTopology(topo, coef)
    x0 = topo["ref_pos"][None].astype(float).copy()
    x0[..., 2] += 3.2; x0[..., 0] += 2.0; x0[..., 1] += 2.5
    held = 6                                                           # first H
    kw = dict(f_tol=2e-3, dt_max=10.0, max_step=0.05, fixed=(held,), scan_dx=(0.0, 0.0, 0.1))
    o = orc.run_replicas(og, t, orc.make_integrator("fire", 3000, 1.0, n_scan=6, **kw), x0, np.zeros_like(x0))
    assert np.allclose(o["pos"][0, held], x0[0, held] + [0, 0, 0.6], atol=1e-12)
    sc = o["scan"][0]
    assert np.all(sc[sc[:, 2] == 1, 3] < 2e-3)
    assert sc[:, 2].sum() >= 4
    # one scan point by hand: displace, evaluate unrelaxed, compare with the relaxed value
    x1 = x0.copy(); x1[0, held, 2] += 0.1
    E7, _ = orc.forces(og, t, x1[0])
    assert sc[0, 0] <= E7.sum() + 1e-12
    # scan = repeated single-point scans chained by hand
    p = x0
    for s in range(3):
        oo = orc.run_replicas(og, t, orc.make_integrator("fire", 3000, 1.0, n_scan=1, **kw), p, np.zeros_like(p)); p = oo["pos"]
        assert np.array_equal(oo["scan"][0, 0], sc[s])
