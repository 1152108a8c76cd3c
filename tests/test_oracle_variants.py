"""Pins for the oracle's interpolation variants: the trilinear foil of PAPER.md:L118-120 and fp16 coefficient
storage.  CPU only.  The foil is pinned against scipy's RegularGridInterpolator (a library routine) applied to the node tables, and
by the properties that define it: exact at nodes, linear along cell edges, second-order error (the spline's is fourth-order)."""
import numpy as np
from scipy.interpolate import RegularGridInterpolator


def _points(og, n, seed, z_lo=1.75, z_hi=7.9):
    rng = np.random.default_rng(seed)
    pos = np.stack([rng.uniform(0, og.Lx, n), rng.uniform(0, og.Ly, n), rng.uniform(z_lo, z_hi, n)], axis=1)
    coef = np.zeros((n, 4)); coef[:, :3] = rng.uniform(-1, 1, (n, 3))
    return pos, coef


def test_trilinear_foil_equals_scipy_linear_interpolation(orc, small_grid):
    og, _ = small_grid
    nx, ny, nz, nch = og.shape
    V, G = orc.trilinear_nodes(og)
    pos, coef = _points(og, 300, 1)
    E, F = orc.interp_trilinear(og, (V, G), pos, coef)
    # periodic wrap by appending the first plane; scipy interpolates each table independently
    hx, hy = og.Lx / nx, og.Ly / ny
    ax = (np.arange(nx + 1) * hx, np.arange(ny + 1) * hy, og.z0 + np.arange(nz) * og.hz)
    wrap = lambda A: np.concatenate([np.concatenate([A, A[:1]], 0), np.concatenate([A, A[:1]], 0)[:, :1]], 1)
    Es = np.zeros(len(pos)); Fs = np.zeros((len(pos), 3))
    for c in range(nch):
        Es += coef[:, c] * RegularGridInterpolator(ax, wrap(V[..., c]))(pos)
        for d in range(3):
            Fs[:, d] -= coef[:, c] * RegularGridInterpolator(ax, wrap(G[..., c, d]))(pos)
    assert np.abs(E - Es).max() < 1e-12 * max(1, np.abs(Es).max()) and np.abs(F - Fs).max() < 1e-11 * max(1, np.abs(Fs).max())


def test_trilinear_foil_properties(orc, small_grid):
    og, samples = small_grid
    nx, ny, nz, nch = og.shape
    V, G = orc.trilinear_nodes(og)
    # node table = the spline at the nodes = the samples it interpolates
    assert np.abs(V[:, :, 1:nz - 1] - samples[:, :, 1:nz - 1]).max() < 1e-9 * np.abs(samples).max()
    # exact at nodes: equals the spline's E and F there
    rng = np.random.default_rng(2)
    idx = np.stack([rng.integers(0, nx, 50), rng.integers(0, ny, 50), rng.integers(2, nz - 3, 50)], 1)
    pts = np.stack([idx[:, 0] * og.Lx / nx, idx[:, 1] * og.Ly / ny, og.z0 + idx[:, 2] * og.hz], 1)
    coef = np.zeros((50, 4)); coef[:, :3] = rng.uniform(-1, 1, (50, 3))
    Et, Ft = orc.interp_trilinear(og, (V, G), pts + 1e-13, coef)
    Es, Fs = orc.interp(og, pts + 1e-13, coef)
    assert np.abs(Et - Es).max() < 1e-8 * np.abs(Es).max() and np.abs(Ft - Fs).max() < 1e-7 * np.abs(Fs).max()
    # midpoint of a z edge = mean of its two nodes
    mid = pts.copy(); mid[:, 2] += 0.5 * og.hz
    up = pts.copy(); up[:, 2] += og.hz
    Em, _ = orc.interp_trilinear(og, (V, G), mid, coef)
    Eu, _ = orc.interp_trilinear(og, (V, G), up + 1e-13, coef)
    assert np.abs(Em - 0.5 * (Et + Eu)).max() < 1e-8 * np.abs(Et).max()
    # accuracy: the foil's energy error is second order — orders of magnitude above the spline's ("several orders of
    # magnitude higher accuracy") — and periodic
    pos, cf = _points(og, 2000, 3, z_lo=1.8, z_hi=4.0)
    Et, _ = orc.interp_trilinear(og, (V, G), pos, cf)
    Es, _ = orc.interp(og, pos, cf)
    scale = np.abs(Es).max()
    assert 1e-5 < np.abs(Et - Es).max() / scale < 5e-2
    E2, _ = orc.interp_trilinear(og, (V, G), pos + [og.Lx, -2 * og.Ly, 0], cf)
    assert np.abs(E2 - Et).max() < 1e-9 * scale
    # above the domain: zero
    top = pos.copy(); top[:, 2] = og.z0 + (nz - 2) * og.hz + 0.01
    E0, F0 = orc.interp_trilinear(og, (V, G), top, cf)
    assert np.all(E0 == 0) and np.all(F0 == 0)


def test_half_grid_rounding_and_error(orc, small_grid):
    og, _ = small_grid
    hg = orc.half_grid(og)
    rel = np.abs(hg.coef - og.coef) / np.maximum(np.abs(og.coef), 1e-30)
    big = np.abs(og.coef) > 1e-4                       # normal fp16 range
    assert rel[big].max() <= 2.0 ** -11 * 1.0001       # half has an 11-bit significand: relative rounding error <= 2^-11
    assert np.all(np.abs(hg.coef[~big] - og.coef[~big]) <= 2.0 ** -25 * 1.0001 + 2.0 ** -11 * np.abs(og.coef[~big]))
    assert np.array_equal(hg.coef, hg.coef.astype(np.float16).astype(np.float64))
    pos, cf = _points(og, 2000, 4)
    Eh, Fh = orc.interp(hg, pos, cf)
    E, F, Vc, _ = orc.interp(og, pos, cf, channels=True)
    den = np.sum(np.abs(cf[:, :3] * Vc), axis=1)
    err = np.abs(Eh - E) / den
    # each coefficient moves by <= 2^-11 of itself and the weights are a partition of unity, so the error is <= 2^-11 sum w |b|: of the
    # order of 2^-11 of the channel magnitudes, larger only where a channel's V_c nearly cancels (Coulomb changes sign)
    assert 1e-6 < np.median(err) < 2.0 ** -11 and err.max() < 1e-2
