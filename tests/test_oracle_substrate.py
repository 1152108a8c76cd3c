"""Pins for the oracle's substrate sums (Morse direct sums, 2D-periodic Coulomb) and for the stated
approximation error of the interpolated grid against brute force (CPU only)."""
import math
import numpy as np
import pytest
from scipy.special import erfc, erf

KE = 14.3996454784


# ---------------------------------------------------------------- Morse (Eq. 4)

def test_single_atom_closed_form(orc):
    """one substrate atom in a cell >> r_cut reduces to the analytic exponentials."""
    sub = dict(pos=np.array([[1.0, 2.0, -0.5]]), e=np.array([0.07]), R=np.array([1.8]), q=np.array([0.0]))
    L = 2000.0
    pts = np.array([[1.3, 2.9, 2.0], [4.0, 1.0, 3.5], [1.0, 2.0, 1.0]])
    VP, VL, gP, gL = orc.morse_points(sub, 1.6, L, L, 17.0, pts, grad=True)
    d = np.linalg.norm(pts - sub["pos"][0], axis=1)
    assert np.allclose(VP, 0.07 * np.exp(-3.2 * (d - 1.8)), rtol=1e-13)
    assert np.allclose(VL, 0.07 * np.exp(-1.6 * (d - 1.8)), rtol=1e-13)
    u = (pts - sub["pos"][0]) / d[:, None]
    assert np.allclose(gP, (-3.2 * VP)[:, None] * u, rtol=1e-12)
    assert np.allclose(gL, (-1.6 * VL)[:, None] * u, rtol=1e-12)


def test_morse_symmetries_and_image_convergence(orc, small_slab):
    sub, Lx, Ly = small_slab
    d = 2.82
    rng = np.random.default_rng(5)
    p = np.stack([rng.uniform(0, Lx, 40), rng.uniform(0, Ly, 40), rng.uniform(1.5, 6, 40)], 1)
    VP, VL = orc.morse_points(sub, 1.6, Lx, Ly, 17.0, p)
    # species-blind parameters -> period d; with Na != Cl the period is (d,d) diagonal and 2d
    q = p.copy(); q[:, 0] += d; q[:, 1] += d
    VP2, VL2 = orc.morse_points(sub, 1.6, Lx, Ly, 17.0, q)
    assert np.allclose(VP, VP2, rtol=1e-9) and np.allclose(VL, VL2, rtol=1e-9)
    # 4-fold rotation about the axis through the ion at the origin
    r = p.copy(); r[:, 0], r[:, 1] = -p[:, 1], p[:, 0]
    VP3, VL3 = orc.morse_points(sub, 1.6, Lx, Ly, 17.0, r)
    assert np.allclose(VP, VP3, rtol=1e-9) and np.allclose(VL, VL3, rtol=1e-9)
    # one more ring of images changes nothing (R10: neglected tail ~1e-12 relative)
    VP4, VL4 = orc.morse_points(sub, 1.6, Lx, Ly, 17.0 + Lx, p)
    assert np.abs(VP4 / VP - 1).max() < 1e-11 and np.abs(VL4 / VL - 1).max() < 1e-9
    # gradient vs central difference
    _, _, gP, gL = orc.morse_points(sub, 1.6, Lx, Ly, 17.0, p, grad=True)
    for ax in range(3):
        pp, pm = p.copy(), p.copy(); pp[:, ax] += 1e-5; pm[:, ax] -= 1e-5
        a, b = orc.morse_points(sub, 1.6, Lx, Ly, 17.0, pp), orc.morse_points(sub, 1.6, Lx, Ly, 17.0, pm)
        assert np.allclose(gP[:, ax], (a[0] - b[0]) / 2e-5, rtol=1e-6, atol=1e-9)
        assert np.allclose(gL[:, ax], (a[1] - b[1]) / 2e-5, rtol=1e-6, atol=1e-9)


# ---------------------------------------------------------------- Coulomb (Eq. 2)

def ewald2d(sub, Lx, Ly, pts, kappa, n_real=3, n_rec=12):
    """textbook 2D Ewald for a slab (erfc real-space sum + erfc-damped reciprocal sum + G=0 term),
    written with scipy.special — independent of the oracle's Fourier form."""
    A = Lx * Ly
    V = np.zeros(len(pts))
    for rj, qj in zip(sub["pos"], sub["q"]):
        dr = pts - rj
        phi = np.zeros(len(pts))
        for a in range(-n_real, n_real + 1):
            for b in range(-n_real, n_real + 1):
                d = np.linalg.norm(dr + np.array([a * Lx, b * Ly, 0.0]), axis=1)
                phi += erfc(kappa * d) / d
        dz = dr[:, 2]
        for m in range(-n_rec, n_rec + 1):
            for n in range(-n_rec, n_rec + 1):
                if m == 0 and n == 0:
                    continue
                gx, gy = 2 * math.pi * m / Lx, 2 * math.pi * n / Ly
                g = math.hypot(gx, gy)
                phi += (math.pi / A) * np.cos(gx * dr[:, 0] + gy * dr[:, 1]) / g * (
                    np.exp(g * dz) * erfc(g / (2 * kappa) + kappa * dz) + np.exp(-g * dz) * erfc(g / (2 * kappa) - kappa * dz))
        phi -= (2 * math.pi / A) * (dz * erf(kappa * dz) + np.exp(-(kappa * dz) ** 2) / (kappa * math.sqrt(math.pi)))
        V += KE * qj * phi
    return V


def test_coulomb_equals_2d_ewald_for_any_kappa(orc, small_slab):
    sub, Lx, Ly = small_slab
    rng = np.random.default_rng(6)
    p = np.stack([rng.uniform(0, Lx, 12), rng.uniform(0, Ly, 12), rng.uniform(1.5, 6, 12)], 1)
    V = orc.coulomb_points(sub, Lx, Ly, p)
    for kappa in (0.9, 1.3):
        ref = ewald2d(sub, Lx, Ly, p, kappa)
        assert np.abs(V - ref).max() < 2e-11, kappa


def test_coulomb_equals_direct_image_sum(orc, small_slab):
    """brute force: k_e sum_j Q_j sum_T 1/|r - r_j - T| over (2N+1)^2 cells of the neutral, dipole-free cell;
    the truncation error falls as N^-3, so N=40 and N=80 extrapolate to ~1e-8."""
    sub, Lx, Ly = small_slab
    p = np.array([[0.0, 0.0, 1.5], [0.7, 1.9, 2.2], [1.41, 1.41, 3.0]])
    V = orc.coulomb_points(sub, Lx, Ly, p)

    def direct(N):
        a = np.arange(-N, N + 1)
        T = np.stack(np.meshgrid(a * Lx, a * Ly, indexing="ij"), -1).reshape(-1, 2)
        out = np.zeros(len(p))
        for rj, qj in zip(sub["pos"], sub["q"]):
            for i, r in enumerate(p):
                d = r - rj
                out[i] += KE * qj * np.sum(1.0 / np.sqrt((d[0] - T[:, 0]) ** 2 + (d[1] - T[:, 1]) ** 2 + d[2] ** 2))
        return out
    v1, v2 = direct(40), direct(80)
    assert np.abs(v2 - V).max() < 2e-5 * np.abs(V).max() + 1e-7
    # successive truncations converge towards the oracle value
    assert np.all(np.abs(v2 - V) <= np.abs(v1 - V) + 1e-12)


def test_coulomb_checkerboard_decay_laplace(orc, small_slab):
    sub, Lx, Ly = small_slab
    d = 2.82
    rng = np.random.default_rng(7)
    p = np.stack([rng.uniform(0, Lx, 30), rng.uniform(0, Ly, 30), rng.uniform(1.5, 5, 30)], 1)
    V, g = orc.coulomb_points(sub, Lx, Ly, p, grad=True)
    q = p.copy(); q[:, 0] += d
    assert np.abs(orc.coulomb_points(sub, Lx, Ly, q) + V).max() < 1e-12          # V(x+d) = -V(x)
    # far-field decay over an ion: e^{-|G1| z}, |G1| = 2 pi sqrt(2) / (2 d) = 1.5755 / Å for d = 2.82
    v8, v9 = orc.coulomb_points(sub, Lx, Ly, [[0, 0, 8.0], [0, 0, 9.0]])
    assert abs(math.log(v8 / v9) - 2 * math.pi * math.sqrt(2) / (2 * d)) < 1e-5
    # harmonic above the slab: finite-difference Laplacian vanishes; gradient matches central difference
    h = 1e-3
    lap = -6 * V
    for ax in range(3):
        pp, pm = p.copy(), p.copy(); pp[:, ax] += h; pm[:, ax] -= h
        a, b = orc.coulomb_points(sub, Lx, Ly, pp, z_min_above_top=1.4), orc.coulomb_points(sub, Lx, Ly, pm, z_min_above_top=1.4)
        lap += a + b
        assert np.allclose(g[:, ax], (a - b) / (2 * h), rtol=1e-5, atol=1e-8)
    assert np.abs(lap / h ** 2).max() < 1e-4 * np.abs(V).max() / 0.1 ** 2


# ---------------------------------------------------------------- grid vs brute force (north_star check 2)

def test_sampled_nodes_are_the_pointwise_sums(orc, small_slab, small_grid):
    sub, Lx, Ly = small_slab
    g, samples = small_grid
    nx, ny, nz, _ = samples.shape
    rng = np.random.default_rng(8)
    idx = np.stack([rng.integers(0, nx, 25), rng.integers(0, ny, 25), rng.integers(0, nz, 25)], 1)
    pts = np.stack([idx[:, 0] * Lx / nx, idx[:, 1] * Ly / ny, 1.5 + 0.1 * idx[:, 2]], 1)
    VP, VL = orc.morse_points(sub, 1.6, Lx, Ly, 17.0, pts)
    VC = orc.coulomb_points(sub, Lx, Ly, pts, z_min_above_top=1.5)
    got = samples[idx[:, 0], idx[:, 1], idx[:, 2]]
    assert np.allclose(got[:, 0], VP, rtol=1e-13) and np.allclose(got[:, 1], VL, rtol=1e-13)
    assert np.allclose(got[:, 2], VC, rtol=1e-11, atol=1e-14)


def test_interpolated_grid_vs_brute_force_stated_error(orc, small_slab, small_grid):
    """Stated error at h = 0.1 Å, alpha = 1.6, z >= 1.7 Å: energy <= 1e-4 relative per channel,
    gradient <= 2e-3 relative per channel (closed-form expectation (kappa h)^4/384: 2.7e-5 Pauli, 1.7e-6 London)."""
    sub, Lx, Ly = small_slab
    g, _ = small_grid
    rng = np.random.default_rng(9)
    n = 1500
    p = np.stack([rng.uniform(0, Lx, n), rng.uniform(0, Ly, n), rng.uniform(1.7, 5.0, n)], 1)
    _, _, Vc, dVc = orc.interp(g, p, np.zeros((n, 4)), channels=True)
    VP, VL, gP, gL = orc.morse_points(sub, 1.6, Lx, Ly, 17.0, p, grad=True)
    VC, gC = orc.coulomb_points(sub, Lx, Ly, p, grad=True, z_min_above_top=1.5)
    eP, eL = np.abs(Vc[:, 0] / VP - 1).max(), np.abs(Vc[:, 1] / VL - 1).max()
    assert 5e-6 < eP < 1e-4 and 3e-7 < eL < 1e-5           # right order of magnitude, not just "small"
    assert np.abs(Vc[:, 2] - VC).max() < 1e-4 * np.abs(VC).max()
    for got, ref in ((dVc[:, 0], gP), (dVc[:, 1], gL), (dVc[:, 2], gC)):
        rel = np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1).max()
        assert rel.max() < 2e-3


def test_error_scales_as_h4(orc, small_slab):
    """halving the spacing divides the energy error by ~16 (and the gradient error by ~8)."""
    sub, Lx, Ly = small_slab
    rng = np.random.default_rng(10)
    n = 400
    p = np.stack([rng.uniform(0, Lx, n), rng.uniform(0, Ly, n), rng.uniform(2.2, 3.0, n)], 1)
    VP, VL, gP, _ = orc.morse_points(sub, 1.6, Lx, Ly, 6.0, p, grad=True)
    errs = []
    for h in (0.1, 0.05):
        nx = int(round(Lx / h)); nz = int(round(2.4 / h)) + 1
        s = orc.sample_grid(sub, 1.6, Lx, Ly, 6.0, nx, nx, nz, 1.4, h, [0, 1])
        g = orc.OracleGrid(orc.prefilter(s), Lx, Ly, 1.4, h)
        _, _, Vc, dVc = orc.interp(g, p, np.zeros((n, 4)), channels=True)
        errs.append((np.abs(Vc[:, 0] / VP - 1).max(), np.abs(dVc[:, 0] - gP).max()))
    assert 10 < errs[0][0] / errs[1][0] < 24
    assert 5 < errs[0][1] / errs[1][1] < 12


def test_atom_coefs_factorisation(orc):
    """PAPER.md:L75-90 Eqs. 3-4: P_i V^P + L_i V^L equals the pairwise Morse sum with Lorentz-Berthelot mixing."""
    sub = dict(pos=np.array([[0.0, 0.0, 0.0], [2.0, 0.5, -1.0]]), e=np.array([0.05, 0.09]), R=np.array([1.5, 1.95]), q=np.zeros(2))
    alpha = 1.6; L = 3000.0
    pt = np.array([[0.7, 0.2, 3.1]])
    ei, Ri = 0.068, 1.9
    coef = orc.atom_coefs([ei], [Ri], [0.3], alpha)[0]
    VP, VL = orc.morse_points(sub, alpha, L, L, 17.0, pt)
    d = np.linalg.norm(pt[0] - sub["pos"], axis=1)
    pair = sum(ei * ej * (math.exp(-2 * alpha * (dj - Ri - Rj)) - 2 * math.exp(-alpha * (dj - Ri - Rj)))
               for ej, Rj, dj in zip(sub["e"], sub["R"], d))
    assert abs(coef[0] * VP[0] + coef[1] * VL[0] - pair) < 1e-15 * max(1, abs(pair)) * 100
    assert coef[2] == 0.3 and coef[3] == 0.0
