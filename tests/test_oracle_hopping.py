"""Pins for the oracle's unique-structure filter and minima-hopping loop (R16,
R19).  CPU only.  The filter is pinned by construction: a population built from K known-distinct structures plus copies that differ
by less than the tolerance and by whole cell translations must collapse to exactly K records, whatever the order; brute-force
pair checks confirm the two defining invariants of the greedy filter."""
import numpy as np

from paper_2508_15522_b200 import inputs

LX = LY = 11.28


def _population(rng, K=7, copies=5, n=12):
    base = rng.uniform(0, 8, (K, n, 3))
    base[:, :, 2] += 3.0
    E0 = -1.0 - 0.05 * np.arange(K)                      # well separated energies ...
    E0[3] = E0[2] + 2e-4                                  # ... except two structures that only geometry can tell apart
    X, E, label = [], [], []
    for k in range(K):
        for c in range(copies):
            shift = np.array([rng.integers(-2, 3) * LX, rng.integers(-2, 3) * LY, 0.0])
            X.append(base[k] + shift + rng.normal(0, 0.01, (n, 3)))      # RMSD ~ 0.017 Å << 0.1 Å
            E.append(E0[k] + rng.uniform(-2e-4, 2e-4)); label.append(k)
    order = rng.permutation(len(X))
    return np.array(X)[order], np.array(E)[order], np.array(label)[order], base, E0


def test_unique_filter_collapses_to_the_known_structures(orc):
    rng = np.random.default_rng(42)
    X, E, label, base, E0 = _population(rng)
    ok = np.ones(len(X), bool); ok[::9] = False            # some replicas did not converge: never candidates
    lib = []
    n_cand, n_new, n_drop = orc.unique_filter(lib, E, X, ok, LX, LY)
    assert n_cand == ok.sum() and n_drop == 0
    assert n_new == len(lib) == len(set(label[ok])) == 7
    # each record is the first converged member of its class, in replica order
    first = {}
    for r in range(len(X)):
        if ok[r] and label[r] not in first:
            first[label[r]] = r
    assert sorted(int(rec[0]) for rec in lib) == sorted(first.values())
    # invariants by brute force: (1) no two records are the same structure; (2) every candidate matches some record
    for i in range(len(lib)):
        for j in range(i):
            assert not orc.same_structure(lib[i][3], lib[i][4:].reshape(-1, 3), lib[j][3], lib[j][4:].reshape(-1, 3), LX, LY)
    for r in range(len(X)):
        if ok[r]:
            assert any(orc.same_structure(E[r], X[r], rec[3], rec[4:].reshape(-1, 3), LX, LY) for rec in lib)
    # a second pass with the same candidates adds nothing; a full library drops instead of growing
    assert orc.unique_filter(lib, E, X, ok, LX, LY)[1] == 0
    lib2 = []
    c2 = orc.unique_filter(lib2, E, X, ok, LX, LY, cap=4)
    assert len(lib2) == 4 and c2[1] == 4 and c2[2] > 0


def test_same_structure_criterion(orc):
    rng = np.random.default_rng(1)
    x = rng.uniform(0, 8, (12, 3))
    assert orc.same_structure(-1.0, x, -1.0, x + [3 * LX, -2 * LY, 0.0], LX, LY)
    assert not orc.same_structure(-1.0, x, -1.0, x + [0.5 * LX, 0, 0], LX, LY)            # another adsorption site
    assert not orc.same_structure(-1.0, x, -1.0, x + [0, 0, 0.11], LX, LY)                # RMSD 0.11 > 0.1
    assert orc.same_structure(-1.0, x, -1.0, x + [0, 0, 0.09], LX, LY)
    assert not orc.same_structure(-1.0, x, -1.0 + 1.1e-3, x, LX, LY)                      # energy window
    # RMSD is the root of the MEAN squared atomic displacement: one atom moved by 0.3 Å among 12 -> 0.0866 Å
    y = x.copy(); y[5, 1] += 0.3
    assert orc.same_structure(-1.0, x, -1.0, y, LX, LY)
    y[5, 1] += 0.06                                        # 0.36 / sqrt(12) = 0.104
    assert not orc.same_structure(-1.0, x, -1.0, y, LX, LY)
    # no rotation / permutation: swapping two atoms is a different structure
    z = x.copy(); z[[0, 1]] = z[[1, 0]]
    assert not orc.same_structure(-1.0, x, -1.0, z, LX, LY)


def test_minima_hopping_loop_properties(orc, small_grid):
    """benzene on the small slab, 6 replicas, 2 cycles: every record is a converged minimum (max |F_i| < f_tol when re-evaluated),
    records are pairwise distinct, every converged replica's final state matches a record, and 2 cycles in one call equal two
    calls of one cycle (noise stream and tags continue)."""
    og, _ = small_grid
    topo = inputs.benzene()
    coef = orc.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], 1.6)
    t = orc.OracleTopology(topo, coef)
    pos = inputs.place_replicas(topo, 6, og.Lx, og.Ly, 0.0, 5).astype(np.float64)
    kw = dict(md_steps=100, md_dt=0.5, temperature=300.0, gamma=0.02, relax_steps=3000, relax_dt=1.0, f_tol=5e-3, seed=9, dt_max=10.0, max_step=0.1)
    a = orc.minima_hopping(og, t, pos, 2, **kw)
    assert a["stats"][:, 0].sum() >= 6 and len(a["library"]) == a["stats"][:, 1].sum() >= 1
    for rec in a["library"]:
        _, F = orc.forces(og, t, rec[4:].reshape(-1, 3))
        assert np.sqrt((F ** 2).sum(1)).max() < 5e-3
    lib = a["library"]
    for i in range(len(lib)):
        for j in range(i):
            assert not orc.same_structure(lib[i][3], lib[i][4:].reshape(-1, 3), lib[j][3], lib[j][4:].reshape(-1, 3), og.Lx, og.Ly)
    b1 = orc.minima_hopping(og, t, pos, 1, **kw)
    b2 = orc.minima_hopping(og, t, b1["pos"], 1, cycle0=1, library=b1["library"], **kw)
    assert np.array_equal(a["pos"], b2["pos"]) and len(b2["library"]) == len(a["library"])
    assert all(np.array_equal(x, y) for x, y in zip(a["library"], b2["library"]))
