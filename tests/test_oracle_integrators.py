"""Pins for the oracle's integrators, RNG and restart generator (CPU only)."""
import math
import numpy as np
import pytest
from paper_2508_15522_b200 import inputs

ACC = 9.648533212e-3


def _diatomic(orc, k=25.0, r0=1.1, m1=12.011, m2=1.008):
    n = 2
    topo = dict(n_atoms=n, mass=np.array([m1, m2]), q=np.zeros(n), lj_e=np.zeros(n), lj_R=np.ones(n),
                bond=[[0, 1]], bond_k_r0=[[k, r0]], angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
                tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((n, n), np.uint8))
    return orc.OracleTopology(topo, np.zeros((n, 4))), k, m1 * m2 / (m1 + m2)


@pytest.mark.parametrize("dt", [0.5, 0.25])
def test_velocity_verlet_harmonic_closed_forms(orc, dt):
    """discrete frequency omega_eff = (2/dt) asin(omega dt/2); peak-to-peak total-energy oscillation
    (omega dt)^2/4 E0; no secular drift."""
    t, k, mu = _diatomic(orc)
    omega = math.sqrt(k / mu * ACC)
    nsteps = 4000
    integ = orc.make_integrator("vv", nsteps, dt)
    pos = np.array([[[0, 0, 0], [0, 0, 1.1 + 0.05]]], float)
    out = orc.run_replicas(None, t, integ, pos, np.zeros_like(pos), trace=True)
    e = out["e_trace"][0]
    E0 = 0.5 * k * 0.05 ** 2
    assert abs((e.max() - e.min()) / E0 - (omega * dt) ** 2 / 4) < 1e-3 * (omega * dt) ** 2 / 4
    slope = np.polyfit(np.arange(len(e)) * dt, e, 1)[0]
    assert abs(slope) * nsteps * dt < 1e-4 * E0
    # frequency from a second run sampled per step: count zero crossings of (r - r0) via short runs
    integ1 = orc.make_integrator("vv", 1, dt)
    p, v = pos.copy(), np.zeros_like(pos); xs = []
    for _ in range(600):
        o = orc.run_replicas(None, t, integ1, p, v); p, v = o["pos"], o["vel"]
        xs.append(p[0, 1, 2] - p[0, 0, 2] - 1.1)
    xs = np.array(xs); tt = dt * np.arange(1, len(xs) + 1)
    w_eff = 2 / dt * math.asin(omega * dt / 2)
    assert np.abs(xs - 0.05 * np.cos(w_eff * tt)).max() < 1e-9


def test_velocity_verlet_time_reversible(orc):
    topo = inputs.tetracene()
    t = orc.OracleTopology(topo, np.zeros((30, 4)))
    rng = np.random.default_rng(12)
    pos = (topo["ref_pos"] + rng.normal(0, 0.03, (30, 3)))[None]
    vel = inputs.maxwell_boltzmann(topo, 1, 300.0, 3).astype(float)
    integ = orc.make_integrator("vv", 300, 0.5)
    o = orc.run_replicas(None, t, integ, pos, vel)
    back = orc.run_replicas(None, t, integ, o["pos"], -o["vel"])
    assert np.abs(back["pos"] - pos).max() < 1e-10
    assert np.abs(back["vel"] + vel).max() < 1e-11
    # launch-split invariance: 1 x 300 == 3 x 100, bit for bit
    p, v = pos, vel
    integ100 = orc.make_integrator("vv", 100, 0.5)
    for _ in range(3):
        oo = orc.run_replicas(None, t, integ100, p, v); p, v = oo["pos"], oo["vel"]
    assert np.array_equal(p, o["pos"]) and np.array_equal(v, o["vel"])


def test_nve_drift_bound_on_grid(orc, small_grid):
    """north_star check 4: NVE drift at small time step.  Stated bounds: (a) over 1 ps the peak-to-peak E_total stays below
    (omega_max dt)^2/4 (E_kin + E_strain)(0), and falls to less than half when dt halves; (b) the secular slope, fitted over 10 ps so that
    the fluctuation no longer limits the fit, is below 1e-5 eV/ps per atom at dt = 0.5 fs and below 2.5e-6 at dt = 0.25 fs (measured
    5.6e-6 and 1.4e-6: the dt^2 law of a symplectic integrator on a C2 potential; SURVEY.md §8(c)'s 1e-6 is met at dt <= 0.2 fs)."""
    g, _ = small_grid
    topo = inputs.tetracene()
    coef = orc.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], 1.6)
    t = orc.OracleTopology(topo, coef)
    # nearly flat adsorbed molecules (tilt 0.1 rad) so that no atom leaves the stored z-domain of the small grid
    c, s_ = math.cos(0.1), math.sin(0.1)
    flat = topo["ref_pos"] @ np.array([[1, 0, 0], [0, c, -s_], [0, s_, c]]).T
    pos = np.stack([flat + [1.0, 2.0, 3.4], flat[:, [1, 0, 2]] + [3.3, 0.4, 3.6]]).astype(np.float32).astype(float)
    vel = inputs.maxwell_boltzmann(topo, 2, 300.0, 78).astype(float)
    pp, slopes = [], []
    for dt, ns, bound in ((0.5, 20000, 1e-5), (0.25, 40000, 2.5e-6)):
        o = orc.run_replicas(g, t, orc.make_integrator("vv", ns, dt), pos, vel, trace=True)
        assert o["pos"][:, :, 2].max() < 8.2                       # nobody left the stored domain (E = F = 0 above it)
        e = o["e_trace"]
        ekin0 = o["energy"][:, 7]          # same order of magnitude as the initial kinetic energy (equipartition)
        wmax = math.sqrt(30.0 / (12.011 * 1.008 / 13.019) * ACC)
        first_ps = e[:, :int(1000 / dt) + 1]
        assert np.all(first_ps.max(1) - first_ps.min(1) <= (wmax * dt) ** 2 / 4 * 2 * ekin0)
        slope = np.array([np.polyfit(np.arange(e.shape[1]) * dt * 1e-3, r, 1)[0] for r in e]) / 30     # eV/ps per atom over 10 ps
        assert np.all(np.abs(slope) < bound), (dt, slope)
        pp.append(first_ps.max(1) - first_ps.min(1)); slopes.append(np.abs(slope))
    assert np.all(pp[1] < 0.5 * pp[0])
    assert np.all(slopes[1] < 0.5 * slopes[0])                     # the secular slope follows the dt^2 law too


def _bowl(orc):
    """one atom on a spring to a heavy, nearly immobile anchor: quadratic bowl with known minimum."""
    n = 2
    topo = dict(n_atoms=n, mass=np.array([1e9, 12.0]), q=np.zeros(n), lj_e=np.zeros(n), lj_R=np.ones(n),
                bond=[[0, 1]], bond_k_r0=[[8.0, 1.5]], angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
                tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((n, n), np.uint8))
    return orc.OracleTopology(topo, np.zeros((n, 4)))


def test_fire_quadratic_bowl_and_split_invariance(orc):
    t = _bowl(orc)
    pos = np.array([[[0, 0, 0], [0.3, 0.4, 2.0]]], float)
    integ = orc.make_integrator("fire", 2000, 0.5, f_tol=1e-6)
    o = orc.run_replicas(None, t, integ, pos, np.zeros_like(pos))
    assert o["status"][0, 1] == 1 and o["status"][0, 0] < 500
    d = o["pos"][0, 1] - o["pos"][0, 0]
    assert abs(np.linalg.norm(d) - 1.5) < 1e-6 / 8.0 * 1.01           # |F| = k |r - r0| < f_tol
    assert np.allclose(d / np.linalg.norm(d), pos[0, 1] / np.linalg.norm(pos[0, 1]), atol=1e-6)   # radial descent
    assert o["energy"][0, 3] < 1e-13 and o["energy"][0].sum() <= 0.5 * 8 * (np.linalg.norm(pos[0, 1]) - 1.5) ** 2
    # 1 x N == k x (N/k) when the FIRE scalars are carried
    n1 = int(o["status"][0, 0])
    a = orc.run_replicas(None, t, orc.make_integrator("fire", 60, 0.5, f_tol=1e-6), pos, np.zeros_like(pos))
    p, v, f = pos, np.zeros_like(pos), None
    for _ in range(3):
        b = orc.run_replicas(None, t, orc.make_integrator("fire", 20, 0.5, f_tol=1e-6), p, v, fire=f)
        p, v, f = b["pos"], b["vel"], b["fire"]
    assert np.array_equal(a["pos"], p) and np.array_equal(a["vel"], v) and np.array_equal(a["fire"], f)
    assert n1 > 60


def test_fire_relaxes_molecule_on_grid_and_is_order_independent(orc, small_grid):
    g, _ = small_grid
    topo = inputs.benzene()
    coef = orc.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], 1.6)
    t = orc.OracleTopology(topo, coef)
    pos = inputs.place_replicas(topo, 6, g.Lx, g.Ly, 0.0, 5, z_lo=3.0, z_hi=4.0).astype(float)
    integ = orc.make_integrator("fire", 30000, 0.5, f_tol=1e-3)
    e0 = np.array([orc.forces(g, t, p)[0].sum() for p in pos])
    o = orc.run_replicas(g, t, integ, pos, np.zeros_like(pos))
    assert np.all(o["status"][:, 1] == 1)
    for r in range(6):
        E7, F = orc.forces(g, t, o["pos"][r])
        assert np.linalg.norm(F, axis=1).max() < 1e-3
        assert E7.sum() <= e0[r] and abs(E7.sum() - o["energy"][r, :7].sum()) < 1e-12
    perm = np.array([3, 0, 5, 1, 4, 2])
    o2 = orc.run_replicas(g, t, integ, pos[perm], np.zeros_like(pos))
    assert np.array_equal(o2["pos"], o["pos"][perm])


# ---------------------------------------------------------------- Philox + restart generator

def philox_bigint(ctr, key):
    """Philox4x32-10 (Salmon et al., SC'11) restated with Python integers — independent of the C code."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    c = list(ctr); k = list(key)
    for _ in range(10):
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & 0xFFFFFFFF, p1 & 0xFFFFFFFF, ((p0 >> 32) ^ c[3] ^ k[1]) & 0xFFFFFFFF, p0 & 0xFFFFFFFF]
        k = [(k[0] + W0) & 0xFFFFFFFF, (k[1] + W1) & 0xFFFFFFFF]
    return c


def test_philox_matches_bigint_restatement(orc):
    rng = np.random.default_rng(13)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2)]
    cases += [(list(map(int, rng.integers(0, 2 ** 32, 4))), list(map(int, rng.integers(0, 2 ** 32, 2)))) for _ in range(20)]
    for ctr, key in cases:
        assert list(map(int, orc.philox4x32_10(ctr, key))) == philox_bigint(ctr, key)
    # avalanche sanity: one counter bit flips about half the output bits
    a = orc.philox4x32_10([5, 0, 0, 0], [1, 2]); b = orc.philox4x32_10([4, 0, 0, 0], [1, 2])
    flips = sum(bin(int(x) ^ int(y)).count("1") for x, y in zip(a, b))
    assert 40 < flips < 88


def test_restart_conformation_invariants(orc):
    topo = inputs.chain60()
    n = 60
    t = orc.OracleTopology(topo, np.zeros((n, 4)))
    Lx = Ly = 11.28
    integ = orc.make_integrator("fire", 10, 0.5, restart=1, seed=1002)
    ref = topo["ref_pos"]
    seen = []
    for (rep, k) in ((0, 1), (0, 2), (7, 1), (4095, 3), (11, 1), (12, 1)):
        p, attempt = orc.restart_conformation(t, integ, Lx, Ly, rep, k, with_attempt=True)
        assert np.array_equal(p, orc.restart_conformation(t, integ, Lx, Ly, rep, k))        # pure function of (seed, r, k)
        # torsion moves + rigid motion keep every bond length and bond angle of the template
        for i, j in topo["bond"]:
            assert abs(np.linalg.norm(p[i] - p[j]) - np.linalg.norm(ref[i] - ref[j])) < 1e-12
        for (i, j, k3), (_, t0) in zip(topo["angle"], topo["angle_k_t0"]):
            a, b = p[i] - p[j], p[k3] - p[j]
            assert abs(math.atan2(np.linalg.norm(np.cross(a, b)), a @ b) - t0) < 1e-6
        c = p.mean(0)
        assert 0 <= c[0] < Lx and 0 <= c[1] < Ly and p[:, 2].min() >= 2.0 - 1e-12 and c[2] >= 3.0 - 1e-12
        # clash rule
        d = np.linalg.norm(p[:, None] - p[None], axis=-1)
        Rs = topo["lj_R"][:, None].astype(float) + topo["lj_R"][None]
        assert attempt == 15 or not np.any((topo["excl"] == 0) & (d < 0.4 * Rs))
        seen.append(p)
    assert np.abs(seen[0] - seen[1]).max() > 0.5 and np.abs(seen[0] - seen[2]).max() > 0.5
    # orientations are spread: the end-to-end vectors of many restarts average to ~0
    v = []
    for k in range(1, 200):
        p = orc.restart_conformation(t, integ, Lx, Ly, 3, k)
        e = p[1] - p[4]; v.append(e / np.linalg.norm(e))       # a rigid in-ring vector
    assert np.linalg.norm(np.mean(v, 0)) < 0.2


def test_fire_restart_records_minima(orc, small_grid):
    g, _ = small_grid
    topo = inputs.benzene()
    coef = orc.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], 1.6)
    t = orc.OracleTopology(topo, coef)
    pos = inputs.place_replicas(topo, 4, g.Lx, g.Ly, 0.0, 5, z_lo=3.0, z_hi=4.0).astype(float)
    integ = orc.make_integrator("fire", 40000, 0.5, f_tol=1e-3, restart=1, seed=9, clash=0.0)
    o = orc.run_replicas(g, t, integ, pos, np.zeros_like(pos), minima_cap=64)
    assert o["n_minima"] >= 4 and o["n_minima"] == o["status"][:, 1].sum()
    for m in o["minima"]:
        r, k = int(m[0]), int(m[1])
        E7, F = orc.forces(g, t, m[4:].reshape(12, 3))
        assert np.linalg.norm(F, axis=1).max() < 1e-3 and abs(E7.sum() - m[3]) < 1e-12
        if k > 0:      # any recorded restart can be replayed alone from (seed, replica, restart#)
            p0 = orc.restart_conformation(t, integ, g.Lx, g.Ly, r, k)
            solo = orc.run_replicas(g, t, orc.make_integrator("fire", 40000, 0.5, f_tol=1e-3), p0[None], np.zeros((1, 12, 3)))
            assert np.abs(solo["pos"][0] - m[4:].reshape(12, 3)).max() < 1e-12


def test_fire_schedule_on_a_constant_force(orc):
    """FIRE's time-step schedule pinned on the one case where it has a closed form: one atom on a potential that is linear in z (a
    B-spline with node values -g z reproduces it exactly), started at rest.  The force is constant, so v stays parallel to F (the mixing
    leaves it unchanged) and P = F.v > 0 from the second iteration on; the positions then depend on the schedule alone:
        x_n - x_0 = c sum_{i<=n} dt_i sum_{j<=i} dt_j ,
    with dt_i from the published rule (Bitzek et al. 2006, PAPER.md ref 72, as read in DESIGN.md R13): P <= 0 (the first iteration, v = 0)
    halves dt and zeroes v; once "the number of steps since P was negative is LARGER than N_min" dt grows by f_inc per iteration up to
    dt_max; the update of dt precedes the Euler step of the same iteration.  Ratios to the first displacement remove the unit constant c.
    An off-by-one in the N_min test, a dt update after the step, or a missing reset at P = 0 each change these ratios by percents."""
    nx = ny = 8; nz = 80; h = 0.1; z0 = 1.0; g = 0.05
    z = z0 + h * np.arange(nz)
    coef = np.broadcast_to((-g * z)[None, None, :, None], (nx, ny, nz, 1)).copy()
    og = orc.OracleGrid(coef, nx * h, ny * h, z0, h)
    topo = dict(n_atoms=1, mass=np.array([12.0]), q=np.zeros(1), lj_e=np.zeros(1), lj_R=np.ones(1),
                bond=np.zeros((0, 2)), bond_k_r0=np.zeros((0, 2)), angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
                tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((1, 1), np.uint8))
    t = orc.OracleTopology(topo, np.array([[1.0, 0.0, 0.0, 0.0]]))
    x0 = np.array([[[0.33, 0.41, 2.0]]])
    E, F = orc.forces(og, t, x0[0])[:2]
    assert np.allclose(F, [[0.0, 0.0, g]], atol=1e-12)                      # the constant force
    dt0, n_min, f_inc, f_dec, n = 0.5, 5, 1.1, 0.5, 40
    dt_max = 3.0 * dt0                                                      # reached inside the run: the cap is exercised too
    xs = []
    for k in range(1, n + 1):
        o = orc.run_replicas(og, t, orc.make_integrator("fire", k, dt0, f_tol=1e-9, dt_max=dt_max, n_min=n_min, f_inc=f_inc, f_dec=f_dec),
                             x0, np.zeros_like(x0))
        assert o["status"][0, 1] == 0 and o["status"][0, 0] == k
        assert np.allclose(o["pos"][0, 0, :2], x0[0, 0, :2], atol=1e-15)
        xs.append(o["pos"][0, 0, 2] - x0[0, 0, 2])
    # the schedule written out from the rule
    dts, dt, npos = [], dt0, 0
    for i in range(1, n + 1):
        if i == 1:                                    # v = 0: P = 0 is not > 0
            dt *= f_dec; npos = 0
        else:
            npos += 1
            if npos > n_min:
                dt = min(dt * f_inc, dt_max)
        dts.append(dt)
    dts = np.array(dts)
    assert dts[6] == dts[0] * f_inc and dts[5] == dts[0] and dts[-1] == dt_max
    expect = np.cumsum(dts * np.cumsum(dts)) / dts[0] ** 2
    got = np.array(xs) / xs[0]
    assert np.allclose(got, expect, rtol=1e-10), np.abs(got / expect - 1).max()
    # and the unit constant itself: x_1 - x_0 = dt_1^2 (g / m) * 9.648533e-3 Å/fs² per eV/(Å amu)  (CODATA: e / u * 1e-20... = 0.964853e-2)
    assert abs(xs[0] / (dts[0] ** 2 * g / 12.0) - 9.64853e-3) < 1e-7


def test_fire_mixing_order_on_a_constant_force(orc):
    """The velocity mixing pinned the same way: constant force along z, initial velocity with a component ACROSS it.  The Euler step never
    touches v_x and the mixing v <- (1 - a) v + a |v| F/|F| shrinks it by exactly (1 - a), so the lateral path depends only on the order
    of the operations and on the schedules of a and dt (Bitzek et al. 2006, PAPER.md ref 72 / DESIGN.md R13: force, P = F.v, mixing with
    the CURRENT a, then — after more than N_min steps with P > 0 — dt <- min(dt f_inc, dt_max) and a <- a f_a, then the step with the new
    dt and the mixed velocity):      x_n - x_0 = v_x0 sum_{i<=n} dt_i prod_{j<=i} (1 - a_j).
    Mixing after the step, mixing with the updated a, or stepping with the old dt each change the sum in its leading digits."""
    nx = ny = 8; nz = 120; h = 0.1; z0 = 1.0; g = 0.05
    z = z0 + h * np.arange(nz)
    coef = np.broadcast_to((-g * z)[None, None, :, None], (nx, ny, nz, 1)).copy()
    og = orc.OracleGrid(coef, nx * h, ny * h, z0, h)
    topo = dict(n_atoms=1, mass=np.array([12.0]), q=np.zeros(1), lj_e=np.zeros(1), lj_R=np.ones(1),
                bond=np.zeros((0, 2)), bond_k_r0=np.zeros((0, 2)), angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
                tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((1, 1), np.uint8))
    t = orc.OracleTopology(topo, np.array([[1.0, 0.0, 0.0, 0.0]]))
    x0 = np.array([[[0.33, 0.41, 2.0]]]); v0 = np.array([[[2.0e-3, 0.0, 1.0e-3]]])           # Å/fs; F.v > 0 from the first iteration
    dt0, n_min, f_inc, a_start, f_a, n = 0.5, 5, 1.1, 0.1, 0.99, 30
    dt_max = 2.0 * dt0
    dt, a, npos, vx, x, expect = dt0, a_start, 0, v0[0, 0, 0], 0.0, []
    for i in range(1, n + 1):
        vx *= 1.0 - a                                  # mixing with the current a
        npos += 1
        if npos > n_min:
            dt = min(dt * f_inc, dt_max); a *= f_a
        x += dt * vx                                   # the step: new dt, mixed velocity
        expect.append(x)
    for k in (1, 2, 5, 6, 7, 12, n):
        o = orc.run_replicas(og, t, orc.make_integrator("fire", k, dt0, f_tol=1e-9, dt_max=dt_max, n_min=n_min, f_inc=f_inc, a_start=a_start, f_a=f_a),
                             x0, v0)
        assert o["status"][0, 0] == k and o["status"][0, 1] == 0
        got = o["pos"][0, 0, 0] - x0[0, 0, 0]
        assert abs(got / expect[k - 1] - 1.0) < 1e-11, (k, got, expect[k - 1])
        assert o["pos"][0, 0, 1] == x0[0, 0, 1]
