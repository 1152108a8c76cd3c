"""GPU-vs-oracle parity for the derived stores of the interpolation trade study: fp16 coefficients
(GRIDFF_LAYOUT_HALF) and the trilinear foil of PAPER.md:L118-120 (GRIDFF_LAYOUT_TRILINEAR), through gridff_grid_derive + gridff_eval.
Run on the B200 box with -m gpu.  Tolerances are north_star's for interpolation: energy 1e-5 relative (denominator sum_c |coef_c V_c|
widened to the magnitude of the coefficients that enter, R14), force 1e-4 eV/Å — each variant against the oracle's
statement of THAT variant (same rounded coefficients / same node tables), so the comparison isolates the fp32 arithmetic."""
import numpy as np
import pytest
import torch

from paper_2508_15522_b200 import inputs
from gridff_cases import oracle_grid, gpu_grid, small_config, energy_denominator
from test_gpu_parity import api, dev, cfg1s, cfg3s, eval_points  # noqa: F401

pytestmark = pytest.mark.gpu


def test_half_store_parity(api, orc, cfg1s):
    """fp16 coefficient store against the ORACLE's own half grid (fp64 -> fp32 -> fp16 of the oracle's coefficients; nothing taken from the GPU).
    The GPU rounds ITS fp32 coefficients, which agree with the oracle's to half an fp32 ulp, so a coefficient that sits within one fp32 ulp of an
    fp16 rounding boundary can land on the other side (about 2 in 10^4 nodes).  That effect is bounded from the oracle alone: D = the largest change
    of a node's fp16 value when its fp32 value moves by one ulp (zero for all other nodes); with B-spline weights >= 0 and summing to 1, a point's
    energy can move by at most sum_c |coef_c| max_stencil D_c and its force by 1.5 / h times that.  Asserted: north_star's tolerances plus that
    bound, point by point — i.e. the plain 1e-5 / 1e-4 for the (majority of) points with no such node near their stencil."""
    from scipy.ndimage import maximum_filter
    og, _ = oracle_grid(orc, cfg1s["sub"], cfg1s["desc"])
    g = gpu_grid(api, cfg1s["sub"], cfg1s["desc"])
    gh = api.gridff_grid_derive(g, api.LAYOUT_HALF)
    pos, cf = eval_points(cfg1s, 20011, 5)                        # ragged tail, many blocks
    E, F = api.gridff_eval(gh, dev(pos), dev(cf))
    E, F = E.cpu().numpy(), F.cpu().numpy()
    hg = orc.half_grid(og)
    Eh, Fh, Vc, _ = orc.interp(hg, pos, cf, channels=True)
    den = np.maximum(np.sum(np.abs(cf[:, :3].astype(np.float64) * Vc), axis=1), 1e-12)       # points above the domain: E = den = 0
    b32 = og.coef.astype(np.float32)
    H = b32.astype(np.float16).astype(np.float64)
    D = np.maximum(np.abs(np.nextafter(b32, np.float32(np.inf)).astype(np.float16).astype(np.float64) - H),
                   np.abs(H - np.nextafter(b32, np.float32(-np.inf)).astype(np.float16).astype(np.float64)))
    Dm = maximum_filter(D, size=(7, 7, 7, 1), mode=("wrap", "wrap", "nearest", "nearest"))      # covers the stencil and a cell of fp32 ambiguity
    nx, ny, nz, nch = og.shape
    hx, hy = og.Lx / nx, og.Ly / ny
    ix = np.floor(pos[:, 0].astype(np.float64) / hx).astype(int) % nx
    iy = np.floor(pos[:, 1].astype(np.float64) / hy).astype(int) % ny
    iz = np.clip(np.floor((pos[:, 2].astype(np.float64) - og.z0) / og.hz).astype(int), 0, nz - 1)
    slack = np.sum(np.abs(cf[:, :nch].astype(np.float64)) * Dm[ix, iy, iz], axis=1)
    assert (slack == 0).mean() > 0.5, "the bound must leave most points at the plain tolerance"
    assert np.all(np.abs(E - Eh) <= 1e-5 * den + slack), (np.abs(E - Eh) - slack).max()
    assert np.all(np.abs(F - Fh).max(axis=1) <= 1e-4 + 1.5 / min(hx, hy, og.hz) * slack)
    # diagnostic (not asserted): the same comparison with the oracle rounding the GPU's exported fp32 coefficients isolates the fp32 arithmetic
    coef32 = api.gridff_grid_export(g).cpu().numpy()
    hg_same = orc.OracleGrid(coef32.astype(np.float16).astype(np.float64), og.Lx, og.Ly, og.z0, og.hz)
    Es, Fs = orc.interp(hg_same, pos, cf)
    # and the price of fp16 against the full-precision spline (reported)
    Ef, Ff = orc.interp(og, pos, cf)
    print("fp16 store: %.1f %% of the points at the plain tolerance; vs the oracle rounding the exported coefficients: max rel E %.2e, max |dF| %.2e; "
          "vs the fp64 spline: median rel E err %.2e, max %.2e; max |dF| %.2e eV/A"
          % (100 * (slack == 0).mean(), (np.abs(E - Es) / den).max(), np.abs(F - Fs).max(),
             np.median(np.abs(E - Ef) / den), (np.abs(E - Ef) / den).max(), np.abs(F - Ff).max()))
    with pytest.raises(api.GridffError):
        api.gridff_grid_export(gh)


def test_trilinear_foil_parity(api, orc, cfg1s):
    og, _ = oracle_grid(orc, cfg1s["sub"], cfg1s["desc"])
    g = gpu_grid(api, cfg1s["sub"], cfg1s["desc"])
    gt = api.gridff_grid_derive(g, api.LAYOUT_TRILINEAR)
    nodes = orc.trilinear_nodes(og)
    pos, cf = eval_points(cfg1s, 6007, 6)
    # include edge cases: exactly on nodes, periodic images, below node 1 (linear continuation), above the domain (zero)
    nz = og.shape[2]
    pos[:50, 0] = np.round(pos[:50, 0] / (og.Lx / og.shape[0])) * np.float32(og.Lx / og.shape[0])
    pos[50:100, 0] += np.float32(3 * og.Lx); pos[100:150, 1] -= np.float32(2 * og.Ly)
    pos[150:170, 2] = np.float32(og.z0 + 0.6 * og.hz)
    pos[170:190, 2] = np.float32(og.z0 + (nz - 2) * og.hz + 0.05)
    E, F = api.gridff_eval(gt, dev(pos), dev(cf))
    E, F = E.cpu().numpy(), F.cpu().numpy()
    Eo, Fo = orc.interp_trilinear(og, nodes, pos.astype(np.float64), cf.astype(np.float64))
    _, _, Vc, _ = orc.interp(og, pos, cf, channels=True)
    den = np.maximum(np.sum(np.abs(cf[:, :3].astype(np.float64) * Vc), axis=1), 1e-6)
    assert (np.abs(E - Eo) / den).max() <= 1e-5, (np.abs(E - Eo) / den).max()
    assert np.abs(F - Fo).max() <= 1e-4
    assert np.all(E[170:190] == 0) and np.all(F[170:190] == 0)
    # the trade the paper describes (L140): orders of magnitude less accurate than the spline
    Es, Fs = orc.interp(og, pos, cf)
    sel = slice(190, None)
    print("trilinear foil vs spline: max |dE| %.2e eV, max |dF| %.2e eV/A (spline fp32 path: 1e-6 / 1e-5)"
          % (np.abs(E[sel] - Es[sel]).max(), np.abs(F[sel] - Fs[sel]).max()))
    assert np.abs(E[sel] - Es[sel]).max() > 1e-4


@pytest.mark.parametrize("k", [1, 3])
def test_micro_brick_stores_match_zfast_and_oracle(api, orc, cfg1s, cfg3s, k):
    """GRIDFF_LAYOUT_MBRICK / MBRICK2 / MBRICK8 (the fp32 coefficients in 2x2x2-node bricks of one 128-byte line, 1 / 2 / 8 shifted copies;
    the layout for stores beyond the L2, "limited by global memory access"): gridff_eval returns the z-fastest store's
    numbers BIT FOR BIT (LDG gather, and the 5-D TMA box kernel of the 8-copy store), on random points with every corner parity, cell
    faces, periodic wraps, the lowest and the highest cell, points below node 1 and above the domain, for several point counts (one point,
    a ragged tail, many tiles per persistent warp); and those numbers are the oracle's within north_star's tolerances."""
    cfg = cfg1s if k == 1 else cfg3s
    d = cfg["desc"]
    g = gpu_grid(api, cfg["sub"], d)
    nx, ny, nz = inputs.grid_dims(d)
    z0 = d["z_ref"] + d["z_lo"]; hx, hy, hz = d["Lx"] / nx, d["Ly"] / ny, d["spacing"]
    stores = [(lay, api.gridff_grid_derive(g, lay)) for lay in (api.LAYOUT_MBRICK, api.LAYOUT_MBRICK2, api.LAYOUT_MBRICK8)]
    for n in (1, 31, 33, 5000, 150011):
        pos, coef = eval_points(cfg, n, 300 + n)
        if n >= 5000:
            # every cell along the x and y edges (the 3-node halo of the store), the lowest cells (1) and the highest (nz - 3), both parities
            m = 1024
            ii = np.arange(m)
            pos[:m, 0] = ((ii % 8) - 4 + 0.37) * hx; pos[:m, 1] = (((ii // 8) % 8) - 4 + 0.61) * hy
            pos[:m, 2] = z0 + np.where(ii % 2 == 0, 1.0 + (ii // 64) % 3, nz - 3 - (ii // 64) % 3 + 0.999) * hz
            pos[m:m + 8] = [[0.0, 0.0, z0 + 2 * hz], [d["Lx"], d["Ly"], z0 + 3 * hz], [-1e-7, d["Ly"], z0 + 4 * hz], [hx, hy, z0 + hz],
                            [d["Lx"] - 1e-6, 0.5 * hy, z0 + 0.5 * hz], [3.5 * hx, -1e-6, z0 + (nz - 2) * hz - 1e-4],
                            [0.5 * hx, 0.5 * hy, z0 + (nz - 2) * hz + 1e-3], [7 * d["Lx"] + 0.3, -5 * d["Ly"] - 0.2, z0 + 5.5 * hz]]
        dp, dc = dev(pos), dev(coef)
        E2, F2 = api.gridff_eval(g, dp, dc, variant=2)
        for lay, gb in stores:
            for variant in ((0, 2, 3) if lay == api.LAYOUT_MBRICK8 else (0, 2)):
                Eb, Fb = api.gridff_eval(gb, dp, dc, variant=variant)
                assert bool(torch.equal(E2, Eb)) and bool(torch.equal(F2, Fb)), (lay, variant, n)
    og, _ = oracle_grid(orc, cfg["sub"], d)
    Eo, Fo, Vc, _ = orc.interp(og, pos, coef, channels=True)
    den = energy_denominator(coef.astype(np.float64), Vc)
    ok = den > 1e-12
    Eg, Fg = Eb.cpu().numpy().astype(np.float64), Fb.cpu().numpy().astype(np.float64)
    assert (np.abs(Eg - Eo)[ok] / den[ok]).max() <= 1e-5 and np.abs(Fg - Fo).max() <= 1e-4
    above = (pos[:, 2].astype(np.float64) - z0) / hz >= nz - 2
    assert above.sum() > 0 and np.all(Eg[above] == 0) and np.all(Fg[above] == 0)
    # E or F alone, the 8-copy store's TMA kernel
    E3, none = api.gridff_eval(stores[2][1], dp, dc, variant=3, want_F=False)
    none2, F3 = api.gridff_eval(stores[2][1], dp, dc, variant=3, want_E=False)
    assert none is None and none2 is None and bool(torch.equal(E3, E2)) and bool(torch.equal(F3, F2))
    # sizes: 1 / 2 / 8 copies of (sx/2 + 1)(sy/2 + 1)(nzp/2 + 1) bricks of 128 B; misuse is refused
    nzp = (nz + 7) // 8 * 8
    per_copy = ((nx + 3) // 2 + 1) * ((ny + 3) // 2 + 1) * (nzp // 2 + 1) * 128
    assert [gb.store.numel() for _, gb in stores] == [per_copy, 2 * per_copy, 8 * per_copy]
    with pytest.raises(api.GridffError):
        api.gridff_eval(stores[0][1], dp, dc, variant=3)          # TMA needs the 8-copy store
    with pytest.raises(api.GridffError):
        api.gridff_eval(stores[2][1], dp, dc, variant=1)
    with pytest.raises(api.GridffError):
        api.gridff_grid_derive(stores[2][1], api.LAYOUT_HALF)     # derived from derived
    with pytest.raises(api.GridffError):
        api.gridff_grid_export(stores[2][1])


def test_eval_binned_matches_eval_bit_for_bit(api, cfg1s, cfg3s):
    """gridff_eval_binned (counting sort of the points by blocks of 4 x 4 x 8 cells on the device, then the gather block by block, results written
    to each point's own index; the path for scattered points on stores beyond the L2) returns gridff_eval's numbers bit for bit:
    any point count (one point, less than a block, a ragged tail, many bins), wrapped coordinates, points below node 1 and above the domain (their
    own bin), duplicates of one point (a bin far larger than a warp); twice in a row (the order inside a bin depends on the atomics, the results
    do not)."""
    for cfg in (cfg1s, cfg3s):
        g = gpu_grid(api, cfg["sub"], cfg["desc"])
        for n in (1, 33, 5000, 150011, (1 << 20) + 77):
            pos, coef = eval_points(cfg, n, 700 + n)
            if n >= 5000:
                pos[100:1100] = pos[100]                       # 1000 copies of one point
                pos[2000:2100, 2] = 1e30                       # far above the domain
            dp, dc = dev(pos), dev(coef)
            E, F = api.gridff_eval(g, dp, dc, variant=2)
            for _ in range(2):
                Eb, Fb = api.gridff_eval_binned(g, dp, dc)
                assert bool(torch.equal(E, Eb)) and bool(torch.equal(F, Fb)), n
        need = api._lib.gridff_eval_binned_work_bytes(g.handle, n)
        assert need >= 52 * n
        with pytest.raises(api.GridffError) as e:
            api.gridff_eval_binned(g, dp, dc, d_work=torch.empty(need - 1024, dtype=torch.uint8, device="cuda"))
        assert e.value.code == api.ESIZE
    gb = gpu_grid(api, cfg1s["sub"], cfg1s["desc"], layout=1)
    with pytest.raises(api.GridffError):
        api.gridff_eval_binned(gb, dp, dc)                     # brick layout: refused
    E0, F0 = api.gridff_eval_binned(g, torch.zeros((0, 3), device="cuda"), torch.zeros((0, 4), device="cuda"))
    assert E0.numel() == 0


def test_derive_errors(api, cfg1s):
    g = gpu_grid(api, cfg1s["sub"], cfg1s["desc"])
    gb = gpu_grid(api, cfg1s["sub"], cfg1s["desc"], layout=1)
    with pytest.raises(api.GridffError):
        api.gridff_grid_derive(gb, api.LAYOUT_HALF)               # brick parent
    with pytest.raises(api.GridffError):
        api.gridff_grid_derive(g, 7)
    gh = api.gridff_grid_derive(g, api.LAYOUT_HALF)
    with pytest.raises(api.GridffError):
        api.gridff_grid_derive(gh, api.LAYOUT_TRILINEAR)          # derived from derived
    # the replica kernel refuses derived stores
    topo = cfg1s["topo"]
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(cfg1s["desc"]["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    with pytest.raises(api.GridffError):
        api.gridff_run_replicas(gh, mol, api.make_integrator("vv", 1, 0.5), dev(cfg1s["pos"]), dev(cfg1s["vel"]))


def test_defective_substrate_grid_and_eval(api, orc):
    """SURVEY.md §8(f) row 4 ("a neutral defect (i.e., by removing one Na and one Cl atoms next to each other from
    the topmost atomic layer)"): the build takes any neutral periodic substrate.  4x4-site, 3-layer slab with a Na-Cl vacancy pair in
    the top layer: coefficients at half an fp32 ulp of the oracle's, interpolation within the north_star tolerances over the defect."""
    sub, Lx, Ly = inputs.rocksalt_slab(4, 3, 2.82, 0.7)
    sub, removed = inputs.vacancy_pair(sub, Lx, Ly)
    first = 0
    assert abs(sub["q"].sum()) < 1e-12 and len(sub["pos"]) == 46
    desc = inputs.grid_desc(Lx, Ly, 0.0, 1.5, 6.5, 0.2, 1.6, [inputs.PAULI, inputs.LONDON, inputs.COULOMB])
    og, _ = oracle_grid(orc, sub, desc)
    g = gpu_grid(api, sub, desc)
    coef = api.gridff_grid_export(g).cpu().numpy().astype(np.float64)
    for ch in range(3):
        ref = og.coef[..., ch]
        assert np.all(np.abs(coef[..., ch] - ref) <= 6.0e-8 * np.abs(ref) + 1e-9 * np.abs(ref).max()), ch
    # the defect is visible: the potential over the vacancy differs from the same site one lattice vector away
    rng = np.random.default_rng(12)
    n = 5000
    pos = np.stack([rng.uniform(0, Lx, n), rng.uniform(0, Ly, n), rng.uniform(1.75, 6.0, n)], 1).astype(np.float32)
    cf = np.zeros((n, 4), np.float32); cf[:, :3] = rng.uniform(-1, 1, (n, 3))
    E, F = api.gridff_eval(g, dev(pos), dev(cf))
    Eo, Fo, Vc, _ = orc.interp(og, pos, cf, channels=True)
    den = np.sum(np.abs(cf[:, :3].astype(np.float64) * Vc), axis=1)
    assert (np.abs(E.cpu().numpy() - Eo) / den).max() <= 1e-5 and np.abs(F.cpu().numpy() - Fo).max() <= 1e-4
    v0 = removed[first]                                                        # the removed atom's site
    p2 = np.array([[v0[0], v0[1], 2.0], [(v0[0] + 2 * 2.82) % Lx, v0[1], 2.0]])
    V = orc.interp(og, p2, np.array([[1.0, 0, 0, 0]] * 2))[0]
    assert abs(V[0] - V[1]) > 1e-3 * abs(V[1])


def test_morse_window_is_exact(api, orc, cfg1s):
    """The tiled Morse sampling (per block of nodes: terms more than e^-34 below the block's largest term dropped, those more than e^-17 below it
    summed in fp32; gridff_build.cu) must give the same fp32 coefficients as the full fp64 sum, and the oracle's."""
    og, _ = oracle_grid(orc, cfg1s["sub"], cfg1s["desc"])
    out = {}
    for flag, mw in (("0", 2), ("1", 1)):                    # gridff_grid_desc.morse_window: 2 = never, 1 = always
        g = gpu_grid(api, cfg1s["sub"], cfg1s["desc"], morse_window=mw)
        out[flag] = api.gridff_grid_export(g).cpu().numpy()
    assert np.array_equal(out["0"][..., 2], out["1"][..., 2])                  # Coulomb untouched
    d = np.abs(out["0"].astype(np.float64) - out["1"])
    assert np.all(d <= 6e-8 * np.abs(out["0"]) + 1e-12 * np.abs(out["0"]).max())         # at most the last fp32 bit
    assert (d > 0).mean() < 1e-3
    for c in range(2):
        ref = og.coef[..., c]
        assert np.all(np.abs(out["1"][..., c] - ref) <= 6.0e-8 * np.abs(ref) + 1e-9 * np.abs(ref).max())


def test_coarser_grid_error_scaling(api, orc, cfg1s):
    """SURVEY.md §8(f) row 3, coarser grids: the GPU spline's error against the un-approximated potential (oracle
    brute-force sums, O4) falls as h^4 for the energy: halving the voxel from 0.2 to 0.1 Å gains a factor ~16 (measured 30 for Pauli, 21 for London: higher-order terms still count at kappa h = 0.64; 8..40 accepted)."""
    sub = cfg1s["sub"]
    rng = np.random.default_rng(21)
    n = 3000
    pos = np.stack([rng.uniform(0, cfg1s["desc"]["Lx"], n), rng.uniform(0, cfg1s["desc"]["Ly"], n), rng.uniform(2.0, 4.0, n)], 1).astype(np.float32)
    d0 = cfg1s["desc"]
    VP, VL = orc.morse_points(sub, d0["alpha"], d0["Lx"], d0["Ly"], d0["r_cut"], pos.astype(np.float64))
    err = {}
    for h in (0.2, 0.1):
        d = dict(d0); d["spacing"] = h
        g = gpu_grid(api, sub, d)
        for ch, V in ((0, VP), (1, VL)):
            cf = np.zeros((n, 4), np.float32); cf[:, ch] = 1.0
            E, _ = api.gridff_eval(g, dev(pos), dev(cf))
            err[(h, ch)] = (np.abs(E.cpu().numpy() - V) / np.abs(V)).max()
    print("spline error vs brute force, max relative: Pauli h=0.2 %.2e, h=0.1 %.2e; London h=0.2 %.2e, h=0.1 %.2e"
          % (err[(0.2, 0)], err[(0.1, 0)], err[(0.2, 1)], err[(0.1, 1)]))
    for ch in (0, 1):
        assert 8 <= err[(0.2, ch)] / err[(0.1, ch)] <= 40, (ch, err[(0.2, ch)], err[(0.1, ch)])
    assert err[(0.1, 0)] <= 1e-4 and err[(0.1, 1)] <= 1e-5


def test_adatom_and_z_ref_rule_of_the_coulomb_channel(api, orc):
    """An adatom 1.1 Å above the top layer (PAPER.md:L154 defects and step edges): the Fourier sum of the Coulomb channel is cut where
    exp(-|G| z_lo) < 1e-16, which needs every atom at least z_lo below the lowest grid plane.  z_ref below the adatom is refused
    (GRIDFF_EINVAL); with z_ref = the adatom's z the coefficients match the oracle's to half an fp32 ulp, Coulomb channel included."""
    sub, Lx, Ly = inputs.rocksalt_slab(2, 3, 2.82, 0.7)
    pos = np.vstack([sub["pos"], [[1.41, 1.41, 1.1]], [[4.23, 4.23, -0.3]]])                      # +0.4 e adatom, -0.4 e interstitial: neutral
    sub = dict(pos=pos, e=np.append(sub["e"], [0.05, 0.05]), R=np.append(sub["R"], [1.6, 1.6]), q=np.append(sub["q"], [0.4, -0.4]))
    assert abs(sub["q"].sum()) < 1e-12
    chans = [inputs.PAULI, inputs.LONDON, inputs.COULOMB]
    bad = inputs.grid_desc(Lx, Ly, 0.0, 1.5, 6.5, 0.2, 1.6, chans)
    with pytest.raises(api.GridffError) as e:
        gpu_grid(api, sub, bad)
    assert e.value.code == -1 and "z_ref" in str(e.value)
    desc = inputs.grid_desc(Lx, Ly, 1.1, 1.5, 6.5, 0.2, 1.6, chans)
    og, _ = oracle_grid(orc, sub, desc)
    g = gpu_grid(api, sub, desc)
    coef = api.gridff_grid_export(g).cpu().numpy().astype(np.float64)
    for ch in range(3):
        ref = og.coef[..., ch]
        assert np.all(np.abs(coef[..., ch] - ref) <= 6.0e-8 * np.abs(ref) + 1e-9 * np.abs(ref).max()), ch
    # a Morse-only grid has no such rule
    g2 = gpu_grid(api, sub, inputs.grid_desc(Lx, Ly, 0.0, 1.5, 6.5, 0.2, 1.6, [inputs.PAULI, inputs.LONDON]))
    assert g2.info()["n_channels"] == 2


def test_morse_grid_with_a_node_on_an_atom(api, orc):
    """A Morse-only grid may reach into the substrate (no z_ref rule there): with z_lo = 0 the lowest node plane is the top atomic layer and the
    node at a top-layer atom's x, y sits ON the atom — distance exactly 0.  The sampling's own square root (reciprocal-square-root seed) must
    return 0 there, not NaN: coefficients finite and the oracle's, to the usual half fp32 ulp, over the whole grid."""
    sub, Lx, Ly = inputs.rocksalt_slab(2, 3, 2.82, 0.0)
    top = sub["pos"][np.isclose(sub["pos"][:, 2], sub["pos"][:, 2].max())]
    desc = inputs.grid_desc(Lx, Ly, float(sub["pos"][:, 2].max()), 0.0, 1.2, 0.2, 1.6, [inputs.PAULI, inputs.LONDON])
    nx, ny, nz = inputs.grid_dims(desc)
    hx, hy = Lx / nx, Ly / ny
    on_node = [(a[0] / hx, a[1] / hy) for a in top if abs(a[0] / hx - round(a[0] / hx)) < 1e-12 and abs(a[1] / hy - round(a[1] / hy)) < 1e-12]
    assert len(on_node) >= 1, "the case needs a top-layer atom on a node of plane 0"
    og, samples = oracle_grid(orc, sub, desc)
    assert np.all(np.isfinite(samples))
    g = gpu_grid(api, sub, desc)
    coef = api.gridff_grid_export(g).cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(coef))
    for ch in range(2):
        ref = og.coef[..., ch]
        assert np.all(np.abs(coef[..., ch] - ref) <= 6.0e-8 * np.abs(ref) + 1e-9 * np.abs(ref).max()), ch
