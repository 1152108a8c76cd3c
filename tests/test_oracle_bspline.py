"""Pins for the oracle's B-spline weights, prefilter and interpolation (CPU only).

Each test checks the oracle against something other than itself: PAPER.md Eq. 6 re-typed from the paper
as a basis function and evaluated at the four offsets, scipy's CubicSpline (a library routine), closed-form
polynomials, finite differences.
"""
import numpy as np
import pytest
from scipy.interpolate import CubicSpline


def paper_eq6(t):
    """PAPER.md:L133 Eq. 6, typed from the paper (golden: tests/golden/eq6_basis.txt)."""
    a = abs(t)
    if a < 1:
        return 2.0 / 3.0 - a * a + 0.5 * a ** 3
    if a < 2:
        return (2.0 - a) ** 3 / 6.0
    return 0.0


def test_basis_matches_golden_values(orc):
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "eq6_basis.txt")) if l.strip() and not l.startswith("#")]
    for t, v in rows:
        assert abs(orc.bspline_basis(float(t)) - float(v)) < 1e-15


@pytest.mark.parametrize("t", [0.0, 1e-9, 0.123, 0.5, 0.875, 1.0 - 1e-12])
def test_weights_are_eq6_at_the_four_offsets(orc, t):
    w, dw = orc.bspline_weights(t)
    # basis functions positioned at x_{i-1}, x_i, x_{i+1}, x_{i+2}  (reading R1)
    ref = [paper_eq6(t + 1), paper_eq6(t), paper_eq6(t - 1), paper_eq6(t - 2)]
    assert np.allclose(w, ref, rtol=0, atol=2e-16)
    assert abs(w.sum() - 1) < 3e-16 and abs(dw.sum()) < 3e-16
    # first moment: sum_j (j - 1 - t) w_j = 0 (linear functions are reproduced by unit coefficients b_j = j)
    assert abs(sum((j - 1 - t) * w[j] for j in range(4))) < 3e-16
    # derivative by central difference of Eq. 6
    d = 1e-6
    fd = [(paper_eq6(t + o + d) - paper_eq6(t + o - d)) / (2 * d) for o in (1, 0, -1, -2)]
    if 1e-5 < t < 1 - 1e-5:
        assert np.allclose(dw, fd, atol=1e-9)


def test_collocation_rows(orc):
    A = orc.collocation_matrix(7, True)
    assert np.allclose(A[0], [4 / 6, 1 / 6, 0, 0, 0, 0, 1 / 6]) and np.allclose(A.sum(1), 1)
    A = orc.collocation_matrix(7, False)
    assert np.allclose(A[0, :4], [8 / 6, -5 / 6, 4 / 6, -1 / 6]) and np.allclose(A[6, 3:], [-1 / 6, 4 / 6, -5 / 6, 8 / 6])
    assert np.allclose(A[3], [0, 0, 1 / 6, 4 / 6, 1 / 6, 0, 0]) and np.allclose(A.sum(1), 1)
    assert np.linalg.cond(A) < 10


def _grid_1d(orc, f, axis, n, periodic_xy):
    """data varying along one axis only, constant along the others."""
    shape = [6, 5, 8]; shape[axis] = n
    idx = [None, None, None]; idx[axis] = slice(None)
    data = np.broadcast_to(f[tuple(idx)], shape).copy()
    per = (1, 1, 0) if periodic_xy else (0, 0, 0)
    coef = orc.prefilter(data[..., None], per)
    return data, coef


def test_prefilter_node_residual_and_constants(orc):
    rng = np.random.default_rng(0)
    data = rng.normal(size=(9, 7, 11, 2))
    coef = orc.prefilter(data, (1, 1, 0))
    Ax, Ay, Az = orc.collocation_matrix(9, True), orc.collocation_matrix(7, True), orc.collocation_matrix(11, False)
    back = np.einsum("ia,jb,kc,abcd->ijkd", Ax, Ay, Az, coef)
    assert np.abs(back - data).max() < 1e-12
    const = orc.prefilter(np.full((9, 7, 11, 1), 3.25), (1, 1, 0))
    assert np.abs(const - 3.25).max() < 1e-14


def test_periodic_axis_equals_scipy_periodic_spline(orc):
    n, L = 17, 3.4
    rng = np.random.default_rng(1)
    f = rng.normal(size=n)
    _, coef = _grid_1d(orc, f, 0, n, True)
    g = orc.OracleGrid(coef, L, 2.0, 0.0, 0.25)
    xs = np.linspace(-L, 2 * L, 301)           # includes wrapped points outside the cell
    pos = np.stack([xs, np.full_like(xs, 0.3), np.full_like(xs, 0.8)], 1)
    E, F = orc.interp(g, pos, np.tile([1.0, 0, 0, 0], (len(xs), 1)))
    cs = CubicSpline(np.arange(n + 1) * L / n, np.append(f, f[0]), bc_type="periodic")
    xw = np.mod(xs, L)
    assert np.abs(E - cs(xw)).max() < 1e-13
    assert np.abs(-F[:, 0] - cs(xw, 1)).max() < 1e-12
    assert np.abs(F[:, 1:]).max() < 1e-12


def test_z_axis_equals_scipy_not_a_knot_spline(orc):
    n, hz, z0 = 13, 0.1, 1.5
    rng = np.random.default_rng(2)
    f = rng.normal(size=n)
    _, coef = _grid_1d(orc, f, 2, n, True)
    g = orc.OracleGrid(coef, 2.0, 2.0, z0, hz)
    cs = CubicSpline(z0 + hz * np.arange(n), f, bc_type="not-a-knot")
    # whole node range below the top cut (R5/R6: lowest cell's polynomial continues down to node 0)
    zs = np.linspace(z0, z0 + hz * (n - 2) - 1e-9, 257)
    pos = np.stack([np.full_like(zs, 0.7), np.full_like(zs, 1.1), zs], 1)
    E, F = orc.interp(g, pos, np.tile([1.0, 0, 0, 0], (len(zs), 1)))
    assert np.abs(E - cs(zs)).max() < 2e-13
    assert np.abs(-F[:, 2] - cs(zs, 1)).max() < 2e-11
    # above the stored domain: E = F = 0 (R6)
    E, F = orc.interp(g, [[0.1, 0.1, z0 + hz * (n - 2) + 1e-9]], [[1.0, 0, 0, 0]])
    assert E[0] == 0 and np.all(F == 0)


def test_cubic_polynomials_reproduced_in_3d(orc):
    """non-periodic mode on all axes: x^a y^b z^c, a,b,c <= 3, reproduced to round-off with gradient."""
    nx, ny, nz, h = 9, 10, 11, 0.1
    x = h * np.arange(nx)[:, None, None]; y = h * np.arange(ny)[None, :, None]; z = 1.5 + h * np.arange(nz)[None, None, :]
    rng = np.random.default_rng(3)
    c = rng.normal(size=(4, 4, 4))
    poly = lambda X, Y, Z: sum(c[a, b, k] * X ** a * Y ** b * Z ** k for a in range(4) for b in range(4) for k in range(4))
    coef = orc.prefilter(poly(x, y, z)[..., None], (0, 0, 0))
    g = orc.OracleGrid(coef, nx * h, ny * h, 1.5, h, periodic_xy=False)
    p = np.stack([rng.uniform(0, h * (nx - 1), 200), rng.uniform(0, h * (ny - 1), 200), rng.uniform(1.5, 1.5 + h * (nz - 2) - 1e-9, 200)], 1)
    E, F = orc.interp(g, p, np.tile([1.0, 0, 0, 0], (200, 1)))
    ref = poly(p[:, 0], p[:, 1], p[:, 2])
    assert np.abs(E - ref).max() < 1e-10 * max(1, np.abs(ref).max())
    d = 1e-5
    for ax in range(3):
        pp, pm = p.copy(), p.copy(); pp[:, ax] += d; pm[:, ax] -= d
        fd = (poly(pp[:, 0], pp[:, 1], pp[:, 2]) - poly(pm[:, 0], pm[:, 1], pm[:, 2])) / (2 * d)
        assert np.abs(-F[:, ax] - fd).max() < 1e-6 * max(1, np.abs(fd).max())


def test_interp_gradient_periodicity_continuity(orc, small_grid):
    g, _ = small_grid
    rng = np.random.default_rng(4)
    n = 300
    p = np.stack([rng.uniform(-3, 9, n), rng.uniform(-3, 9, n), rng.uniform(1.7, 5.0, n)], 1)
    k = np.concatenate([rng.uniform(-1, 1, (n, 3)), np.zeros((n, 1))], 1)
    E, F = orc.interp(g, p, k)
    d = 1e-4
    for ax in range(3):
        pp, pm = p.copy(), p.copy(); pp[:, ax] += d; pm[:, ax] -= d
        fd = (orc.interp(g, pp, k)[0] - orc.interp(g, pm, k)[0]) / (2 * d)
        assert np.abs(-F[:, ax] - fd).max() < 1e-6 * np.abs(F).max()
    # E(x + Lx) = E(x): identical cell + fraction after the wrap, to round-off of the wrap itself
    ps = p.copy(); ps[:, 0] += g.Lx; ps[:, 1] -= 2 * g.Ly
    E2, F2 = orc.interp(g, ps, k)
    assert np.abs(E2 - E).max() < 1e-9 * np.abs(E).max() and np.abs(F2 - F).max() < 1e-8 * np.abs(F).max()
    # C1 force continuity across a cell face in every direction
    hx = g.Lx / g.shape[0]
    for ax, h, base in ((0, hx, 3 * hx), (1, hx, 7 * hx), (2, 0.1, 1.5 + 0.1 * 9)):
        q = p[:50].copy(); q[:, ax] = base - 1e-10
        r = q.copy(); r[:, ax] = base + 1e-10
        Fa, Fb = orc.interp(g, q, k[:50])[1], orc.interp(g, r, k[:50])[1]
        assert np.abs(Fa - Fb).max() < 1e-6 * np.abs(Fa).max()
