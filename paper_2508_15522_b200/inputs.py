"""Seeded synthetic inputs for the GridFF hot path — the ONLY module shared by the oracle-side and
the CUDA-side callers (tests, bench.py, smoke).  It holds none of the method's arithmetic: no B-spline,
no substrate sums, no force field, no integrator.  It builds substrates, molecules (geometry + topology +
parameters), replica placements, velocities and point sets with numpy's PCG64 (`default_rng(seed)`).

The paper's workloads (PTCDA / xylitol on NaCl, UFF tables, RESP charges) are not
available; these generators stand in for them with the same shapes, sizes and magnitudes.
The element table is synthetic, UFF-magnitude — NOT the UFF table.
"""
import math
import numpy as np

KB = 8.617333262e-5      # eV/K
ACC = 9.648533212e-3     # 1 eV/(Å amu) in Å/fs²

# element: (R / Å, eps / eV, mass / amu)      synthetic, UFF-magnitude
ELEMENTS = {
    "H": (1.40, 0.0019, 1.008),
    "C": (1.90, 0.0046, 12.011),
    "O": (1.75, 0.0026, 15.999),
    "Na": (1.50, 0.0013, 22.990),
    "Cl": (1.95, 0.0098, 35.453),
}


def _elem_arrays(elements):
    R = np.array([ELEMENTS[s][0] for s in elements])
    e = np.sqrt(np.array([ELEMENTS[s][1] for s in elements]))     # e = sqrt(eps): eps_ij = e_i e_j (R9)
    m = np.array([ELEMENTS[s][2] for s in elements])
    return R, e, m


# ----------------------------------------------------------------------------- substrates

def rocksalt_slab(n_sites, n_layers, d, q):
    """Square lattice of sites, spacing d, n_sites x n_sites per layer, layers at z = 0, -d, ...;
    species Na if (i + j + l) even else Cl; charges +q / -q.  Returns (substrate dict, Lx, Ly)."""
    pos, el, qs = [], [], []
    for l in range(n_layers):
        for i in range(n_sites):
            for j in range(n_sites):
                pos.append((i * d, j * d, -l * d))
                na = (i + j + l) % 2 == 0
                el.append("Na" if na else "Cl")
                qs.append(q if na else -q)
    R, e, _ = _elem_arrays(el)
    sub = dict(pos=np.array(pos, dtype=np.float64), e=e, R=R, q=np.array(qs, dtype=np.float64), elements=el)
    return sub, n_sites * d, n_sites * d


def vacancy_pair(sub, Lx, Ly):
    """The paper's neutral defect ("removing one Na and one Cl atoms next to each other from the topmost atomic layer"): the
    top-layer atom nearest the cell centre and its nearest oppositely charged top-layer neighbour are removed.  Returns (substrate without
    the pair, positions [2][3] of the removed atoms)."""
    pos, q = np.asarray(sub["pos"]), np.asarray(sub["q"])
    top = np.where(np.abs(pos[:, 2] - pos[:, 2].max()) < 1e-9)[0]
    first = top[np.argmin(np.linalg.norm(pos[top, :2] - [Lx / 2, Ly / 2], axis=1))]
    others = [t for t in top if t != first and q[t] == -q[first]]
    second = others[int(np.argmin([np.linalg.norm(pos[t, :2] - pos[first, :2]) for t in others]))]
    keep = np.array([i for i in range(len(pos)) if i not in (first, second)])
    out = {k: np.ascontiguousarray(np.asarray(v)[keep]) for k, v in sub.items() if k != "elements"}
    return out, pos[[first, second]].copy()


def drag_starts(topo, n_rep, held, start_xy, z_above, spread, seed):
    """replicas for a drag scan: the molecule flat (template orientation) `z_above` over z = 0, translated so that its
    held atom sits at start_xy + U(-spread, spread) in x and y; float32 [n_rep][n][3]"""
    rng = np.random.default_rng(seed)
    ref = np.asarray(topo["ref_pos"], np.float64)
    out = np.repeat(ref[None], n_rep, 0)
    out[..., 2] += z_above - ref[held, 2]
    shift = np.asarray(start_xy)[None, :] + rng.uniform(-spread, spread, (n_rep, 2)) - ref[held, :2][None, :]
    out[..., :2] += shift[:, None, :]
    return out.astype(np.float32)


# ----------------------------------------------------------------------------- topology helpers

def _neighbors(n, bonds):
    nb = [[] for _ in range(n)]
    for i, j in bonds:
        nb[i].append(j); nb[j].append(i)
    return [sorted(x) for x in nb]


def _angles_from_bonds(n, bonds):
    nb = _neighbors(n, bonds)
    out = []
    for j in range(n):
        for a in range(len(nb[j])):
            for b in range(a + 1, len(nb[j])):
                out.append((nb[j][a], j, nb[j][b]))
    return out


def _exclusions(n, bonds, depth=3):
    """excl[i][j] = 1 if i == j or j is within `depth` bonds of i (R12)."""
    nb = _neighbors(n, bonds)
    ex = np.zeros((n, n), np.uint8)
    for s in range(n):
        dist = {s: 0}; frontier = [s]
        for d in range(depth):
            nxt = []
            for u in frontier:
                for v in nb[u]:
                    if v not in dist:
                        dist[v] = d + 1; nxt.append(v)
            frontier = nxt
        for v in dist:
            ex[s, v] = 1
    return ex


def _side_mask(n, bonds, j0, j1):
    """atoms on the j1 side of bond j0-j1 (they move when the bond is twisted)."""
    nb = _neighbors(n, bonds)
    seen = {j1}; stack = [j1]
    while stack:
        u = stack.pop()
        for v in nb[u]:
            if v == j0 and u == j1:
                continue
            if v not in seen:
                seen.add(v); stack.append(v)
    assert j0 not in seen, "bond is in a ring"
    m = np.zeros(n, np.uint8); m[list(seen)] = 1
    return m


def _measure_angle(p, i, j, k):
    a, b = p[i] - p[j], p[k] - p[j]
    return math.atan2(np.linalg.norm(np.cross(a, b)), float(a @ b))


def _finish(elements, pos, bonds, bond_k, tors, rot_bonds, rng, charges, nonbonded):
    n = len(elements)
    pos = np.asarray(pos, dtype=np.float64)
    R, e, m = _elem_arrays(elements)
    bonds = [tuple(b) for b in bonds]
    bond_k_r0 = [(bond_k(elements[i], elements[j]), float(np.linalg.norm(pos[i] - pos[j]))) for i, j in bonds]
    angles = _angles_from_bonds(n, bonds)
    angle_k_t0 = [(5.0, _measure_angle(pos, *t)) for t in angles]
    q = np.zeros(n)
    if charges:
        q = rng.normal(0.0, 0.2, n); q -= q.mean()
    topo = dict(
        n_atoms=n, elements=list(elements), ref_pos=pos - pos.mean(axis=0),
        mass=m.astype(np.float32), q=q.astype(np.float32), lj_e=e.astype(np.float32), lj_R=R.astype(np.float32),
        grid_e=e.astype(np.float32), grid_R=R.astype(np.float32),
        bond=np.array(bonds, np.int32).reshape(-1, 2), bond_k_r0=np.array(bond_k_r0, np.float32).reshape(-1, 2),
        angle=np.array(angles, np.int32).reshape(-1, 3), angle_k_t0=np.array(angle_k_t0, np.float32).reshape(-1, 2),
        tors=np.array([t[:4] for t in tors], np.int32).reshape(-1, 4),
        tors_k_n_p0=np.array([t[4:] for t in tors], np.float32).reshape(-1, 3),
        excl=_exclusions(n, bonds) if nonbonded else None,
        rot_bond=np.array(rot_bonds, np.int32).reshape(-1, 2),
        rot_mask=(np.array([_side_mask(n, bonds, a, b) for a, b in rot_bonds], np.uint8).reshape(-1, n)),
    )
    if not nonbonded:
        topo["excl"] = np.ones((n, n), np.uint8)       # every pair excluded: no intramolecular non-bonded terms
    return topo


def _bond_k(a, b):
    s = {a, b}
    if "H" in s:
        return 25.0
    if "O" in s:
        return 28.0
    return 30.0


# ----------------------------------------------------------------------------- molecules

def benzene():
    """C0 molecule: 12 atoms, 12 bonds, 18 angles, no torsions, no intramolecular non-bonded terms."""
    el, pos, bonds = [], [], []
    for k in range(6):
        a = math.pi / 3 * k
        el.append("C"); pos.append((1.39 * math.cos(a), 1.39 * math.sin(a), 0.0))
    for k in range(6):
        a = math.pi / 3 * k
        el.append("H"); pos.append((2.47 * math.cos(a), 2.47 * math.sin(a), 0.0))
    for k in range(6):
        bonds.append((k, (k + 1) % 6)); bonds.append((k, 6 + k))
    return _finish(el, pos, bonds, _bond_k, [], [], None, charges=False, nonbonded=False)


def _acene(n_rings, cc=1.40, ch=1.08):
    pts = []
    w = math.sqrt(3.0) * cc
    for r in range(n_rings):
        for m in range(6):
            a = math.radians(30 + 60 * m)
            p = (r * w + cc * math.cos(a), cc * math.sin(a))
            if not any(math.hypot(p[0] - s[0], p[1] - s[1]) < 1e-6 for s in pts):
                pts.append(p)
    pts.sort(key=lambda p: (round(p[0], 6), round(p[1], 6)))
    nC = len(pts)
    bonds = [(i, j) for i in range(nC) for j in range(i + 1, nC)
             if math.hypot(pts[i][0] - pts[j][0], pts[i][1] - pts[j][1]) < cc * 1.1]
    el = ["C"] * nC; pos = [(p[0], p[1], 0.0) for p in pts]
    nb = _neighbors(nC, bonds)
    for i in range(nC):
        if len(nb[i]) == 2:
            v = np.array(pos[i]) * 2 - np.array(pos[nb[i][0]]) - np.array(pos[nb[i][1]])
            v /= np.linalg.norm(v)
            el.append("H"); pos.append(tuple(np.array(pos[i]) + ch * v)); bonds.append((i, len(pos) - 1))
    return el, pos, bonds, nb


def tetracene(seed=1001):
    """C1/C3 molecule: 18 C + 12 H planar aromatic, 33 bonds, 54 angles, 8 torsions (first 8, in sorted index
    order, of the proper torsions about the three ring-fusion bonds; n=2, phi0=pi, k=0.1 eV), charges
    N(0, 0.2 e) neutralised, LJ + Coulomb with <=3-bond exclusions."""
    rng = np.random.default_rng(seed)
    el, pos, bonds, nbC = _acene(4)
    fusion = [(i, j) for (i, j) in bonds if el[i] == "C" and el[j] == "C" and len(nbC[i]) == 3 and len(nbC[j]) == 3]
    tors = []
    for (j, k) in fusion:
        for i in nbC[j]:
            if i == k:
                continue
            for l in nbC[k]:
                if l == j:
                    continue
                tors.append((i, j, k, l, 0.1, 2.0, math.pi))
    tors.sort(key=lambda t: t[:4])
    tors = tors[:8]
    return _finish(el, pos, bonds, _bond_k, tors, [], rng, charges=True, nonbonded=True)


def _nerf(a, b, c, length, angle, dihedral):
    """place d so that |cd| = length, angle(b,c,d) = angle, dihedral(a,b,c,d) = dihedral."""
    a, b, c = map(np.asarray, (a, b, c))
    bc = c - b; bc /= np.linalg.norm(bc)
    n = np.cross(b - a, bc); n /= np.linalg.norm(n)
    m = np.cross(n, bc)
    d2 = np.array([-length * math.cos(angle), length * math.sin(angle) * math.cos(dihedral),
                   length * math.sin(angle) * math.sin(dihedral)])
    return c + d2[0] * bc + d2[1] * m + d2[2] * n


def chain60(seed=1002):
    """C2 molecule: phenyl (6 C + 5 H) - 19-atom backbone (C,C,O repeating; O at 3,6,...,18) - CH3; 60 atoms,
    20 rotatable backbone bonds, one torsion term each (n=3, phi0=0, k=0.03 eV) + 6 ring torsions
    (n=2, phi0=pi, k=0.1 eV)."""
    rng = np.random.default_rng(seed)
    el, pos, bonds = [], [], []
    for k in range(6):
        a = math.pi / 3 * k
        el.append("C"); pos.append(np.array([1.39 * math.cos(a), 1.39 * math.sin(a), 0.0]))
        bonds.append((k, (k + 1) % 6))
    for k in range(1, 6):
        a = math.pi / 3 * k
        el.append("H"); pos.append(np.array([2.47 * math.cos(a), 2.47 * math.sin(a), 0.0])); bonds.append((k, len(pos) - 1))
    tet = math.radians(111.0)
    back = []
    kinds = ["O" if (k % 3 == 0) else "C" for k in range(1, 20)] + ["C"]      # b1..b19, then CH3 carbon b20
    prev3 = [1, 0]      # ring atoms C1, C0 lead into the chain
    for k, s in enumerate(kinds):
        if k == 0:
            p = pos[0] + 1.51 * pos[0] / np.linalg.norm(pos[0]); par = 0
        else:
            chainidx = [1, 0] + back
            a, b, c = chainidx[-3], chainidx[-2], chainidx[-1]
            L = 1.43 if ("O" in (s, el[c])) else 1.53
            dih = math.radians(90.0) if k == 1 else math.pi
            p = _nerf(pos[a], pos[b], pos[c], L, tet, dih); par = c
        el.append(s); pos.append(p); back.append(len(pos) - 1); bonds.append((par, len(pos) - 1))
    full = [0] + back
    for t in range(1, len(full) - 1):          # CH2 hydrogens
        c = full[t]
        if el[c] != "C":
            continue
        u1 = pos[full[t - 1]] - pos[c]; u2 = pos[full[t + 1]] - pos[c]
        u1 /= np.linalg.norm(u1); u2 /= np.linalg.norm(u2)
        bis = -(u1 + u2); bis /= np.linalg.norm(bis)
        w = np.cross(u1, u2); w /= np.linalg.norm(w)
        beta = math.radians(54.75)
        for sgn in (1.0, -1.0):
            el.append("H"); pos.append(pos[c] + 1.09 * (math.cos(beta) * bis + sgn * math.sin(beta) * w)); bonds.append((c, len(pos) - 1))
    a, b, c = full[-3], full[-2], full[-1]     # CH3 hydrogens
    for dih in (60.0, 180.0, 300.0):
        el.append("H"); pos.append(_nerf(pos[a], pos[b], pos[c], 1.09, math.radians(109.5), math.radians(dih))); bonds.append((c, len(pos) - 1))
    assert len(el) == 60
    rot = [(full[t], full[t + 1]) for t in range(len(full) - 1)]
    nb = _neighbors(len(el), bonds)
    tors = []
    for (j, k) in rot:
        i = min(x for x in nb[j] if x != k)
        heavy = [x for x in nb[k] if x != j and el[x] != "H"]
        l = min(heavy) if heavy else min(x for x in nb[k] if x != j)
        tors.append((i, j, k, l, 0.03, 3.0, 0.0))
    for m in range(6):
        tors.append(((m - 1) % 6, m, (m + 1) % 6, (m + 2) % 6, 0.1, 2.0, math.pi))
    return _finish(el, pos, bonds, _bond_k, tors, rot, rng, charges=True, nonbonded=True)


# ----------------------------------------------------------------------------- placements

def helix_chain(n, seed=7):
    """n-atom united-atom chain (C, C, O repeating) wound as a loose helix (bond 1.5 Å, angle 112 deg, dihedral 70 deg): bonds i-(i+1),
    all angles, one n = 3 torsion per 4 consecutive atoms, partial charges, LJ + Coulomb beyond 3 bonds.  A size-parametrised molecule
    for the edge cases of the replica kernel (1, 2, 3, 32, 33, 64 atoms); not one of the BASELINE configs."""
    rng = np.random.default_rng(seed)
    el = [("C", "C", "O")[i % 3] for i in range(n)]
    pos = [np.zeros(3), np.array([1.5, 0.0, 0.0]), np.array([1.5 + 1.5 * math.cos(math.radians(68)), 1.5 * math.sin(math.radians(68)), 0.0])][:n]
    for i in range(3, n):
        pos.append(_nerf(pos[i - 3], pos[i - 2], pos[i - 1], 1.5, math.radians(112), math.radians(70)))
    bonds = [(i, i + 1) for i in range(n - 1)]
    tors = [(i, i + 1, i + 2, i + 3, 0.03, 3.0, 0.0) for i in range(n - 3)]
    return _finish(el, np.array(pos), bonds, _bond_k, tors, [], rng, True, True)


def _random_rotations(rng, n):
    q = rng.normal(size=(n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    x, y, z, w = q.T
    return np.stack([np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)], -1),
                     np.stack([2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)], -1),
                     np.stack([2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)], -1)], 1)


def _twist_grow(ref, topo, rng, n_rep, clash=0.6, tries=64, restarts=64):
    """n_rep conformers of the template, one random dihedral about every rotatable bond, free of clashes (no non-excluded pair closer than
    clash * (R_i + R_j)), by chain growth, vectorised over the replicas: the bonds are taken from the fixed core outwards (largest turning
    side first); each dihedral is drawn ~ U(-pi, pi) and re-drawn (up to `tries` times) while the atoms it puts in their final place clash
    with atoms already in theirs; a replica that finds no angle starts again from the template (up to `restarts` times).  The turning sides
    of the bonds must be nested or disjoint (a tree).  -> float64 [n_rep][n][3]"""
    n = topo["n_atoms"]
    lim2 = ((topo["lj_R"][:, None].astype(np.float64) + topo["lj_R"][None, :]) * clash) ** 2
    free = (topo["excl"] == 0) & (topo["excl"].T == 0) & ~np.eye(n, dtype=bool)
    masks = [np.asarray(m, bool) for m in topo["rot_mask"]]
    order = sorted(range(len(masks)), key=lambda b: -int(masks[b].sum()))
    # an atom's position depends on dihedral b iff it is on b's turning side and not on its axis (the far bond atom j1 turns with itself but
    # stays put); it is in its final place after the last bond, in this order, that moves it
    last = np.full(n, -1)
    for k, b in enumerate(order):
        moved = masks[b].copy(); moved[int(topo["rot_bond"][b][1])] = False
        last[moved] = k
    steps, done = [], last < 0
    for k, b in enumerate(order):
        new = last == k
        old_idx, new_idx = np.nonzero(done)[0], np.nonzero(new)[0]
        pi, pj = np.meshgrid(new_idx, old_idx, indexing="ij")
        keep = free[pi, pj]
        # pairs among the new atoms themselves are rigid with respect to this rotation: nothing to test
        steps.append((b, np.nonzero(masks[b])[0], pi[keep], pj[keep], lim2[pi, pj][keep]))
        done = done | new
    ref = np.asarray(ref, np.float64)
    out = np.broadcast_to(ref, (n_rep, n, 3)).copy()
    todo = np.arange(n_rep)
    for _ in range(restarts):
        p = np.broadcast_to(ref, (len(todo), n, 3)).copy()
        alive = np.ones(len(todo), bool)
        for b, sel, pi, pj, l2 in steps:
            j0, j1 = (int(v) for v in topo["rot_bond"][b])
            need = alive.copy()
            base = p[:, sel, :].copy()
            for _t in range(tries):
                idx = np.nonzero(need)[0]
                if len(idx) == 0:
                    break
                ang = rng.uniform(-math.pi, math.pi, len(idx))
                o = p[idx, j0, :][:, None, :]
                ax = p[idx, j1, :] - p[idx, j0, :]; ax /= np.linalg.norm(ax, axis=1, keepdims=True)
                axb = ax[:, None, :]
                v = base[idx] - o
                c, s_ = np.cos(ang)[:, None, None], np.sin(ang)[:, None, None]
                q = p[idx].copy()
                q[:, sel, :] = o + v * c + np.cross(axb, v) * s_ + axb * np.sum(v * axb, axis=2, keepdims=True) * (1 - c)
                d = q[:, pi, :] - q[:, pj, :]
                ok = np.all(np.einsum("kij,kij->ki", d, d) >= l2[None, :], axis=1) if len(pi) else np.ones(len(idx), bool)
                p[idx[ok]] = q[ok]
                need[idx[ok]] = False
            alive &= ~need
        out[todo[alive]] = p[alive]
        todo = todo[~alive]
        if len(todo) == 0:
            return out
    raise RuntimeError("chain growth found no clash-free conformer for %d replicas" % len(todo))


def place_replicas(topo, n_rep, Lx, Ly, z_ref, seed, z_lo=3.0, z_hi=6.0, z_min=2.0, twist=False):
    """centroid x,y ~ U(0,L), orientation uniform on SO(3), centroid z ~ U(z_lo, z_hi) above z_ref, lifted so the
    lowest atom is >= z_min above z_ref.  Returns float32 [n_rep][n][3].  With `twist`, EVERY replica gets its own clash-free random
    dihedrals about the rotatable bonds (config 2: "random initial dihedrals"; _twist_grow)."""
    rng = np.random.default_rng(seed)
    n = topo["n_atoms"]
    ref = np.asarray(topo["ref_pos"], dtype=np.float64)
    rots = _random_rotations(rng, n_rep)
    conf = _twist_grow(ref, topo, rng, n_rep) if twist else None
    out = np.zeros((n_rep, n, 3))
    for r in range(n_rep):
        p = conf[r] if twist else ref
        p = (p - p.mean(axis=0)) @ rots[r].T
        p = p + np.array([rng.uniform(0, Lx), rng.uniform(0, Ly), z_ref + rng.uniform(z_lo, z_hi)])
        lift = z_ref + z_min - p[:, 2].min()
        if lift > 0:
            p[:, 2] += lift
        out[r] = p
    return out.astype(np.float32)


def maxwell_boltzmann(topo, n_rep, T, seed):
    """velocities in Å/fs, sigma = sqrt(kB T / m) per component; float32 [n_rep][n][3]."""
    rng = np.random.default_rng(seed)
    m = np.asarray(topo["mass"], dtype=np.float64)
    sig = np.sqrt(KB * T / m * ACC)
    return (rng.normal(size=(n_rep, len(m), 3)) * sig[None, :, None]).astype(np.float32)


# ----------------------------------------------------------------------------- grid descriptors / configs

PAULI, LONDON, COULOMB, ZERO = 0, 1, 2, 3


def grid_desc(Lx, Ly, z_ref, z_lo, z_hi, spacing, alpha, channels, r_cut=17.0):
    return dict(Lx=Lx, Ly=Ly, z_ref=z_ref, z_lo=z_lo, z_hi=z_hi, spacing=spacing, alpha=alpha, r_cut=r_cut,
                channels=list(channels))


def grid_dims(desc):
    """DESIGN.md R7: n = round(L / spacing), h = L / n; nz = round((z_hi - z_lo) / spacing), hz = spacing."""
    nx = int(round(desc["Lx"] / desc["spacing"])); ny = int(round(desc["Ly"] / desc["spacing"]))
    nz = int(round((desc["z_hi"] - desc["z_lo"]) / desc["spacing"]))
    return nx, ny, nz


def config(k, n_rep=None, spacing=0.1, small=False):
    """The five BASELINE.json configs as concrete seeded inputs.  `small=True` shrinks the
    substrate / grid (2x2 sites, coarser spacing) for CPU-only tests of the host logic."""
    seed = 1000 + k
    if k in (0, 1, 2):
        sites = 2 if small else 4
        sub, Lx, Ly = rocksalt_slab(sites, 4, 2.82, 0.0 if k == 0 else 0.7)
        chans = [PAULI, LONDON] if k == 0 else [PAULI, LONDON, COULOMB]
        desc = grid_desc(Lx, Ly, 0.0, 1.5, 11.5, spacing, 1.6, chans)
        if k == 0:
            topo = benzene(); n_rep = n_rep or 64
            integ = dict(kind="fire", n_steps=1000, dt=0.5, f_tol=1e-3)
            vel_T = None; twist = False
        elif k == 1:
            topo = tetracene(seed); n_rep = n_rep or 4096
            integ = dict(kind="vv", n_steps=10000, dt=0.5)
            vel_T = 300.0; twist = False
        else:
            topo = chain60(seed); n_rep = n_rep or 16384
            integ = dict(kind="fire", n_steps=20000, dt=0.5, f_tol=1e-3, restart=1, seed=seed)
            vel_T = None; twist = True
    elif k == 3:
        sites = 4 if small else 20
        sub, Lx, Ly = rocksalt_slab(sites, 3, 2.0, 0.7)
        desc = grid_desc(Lx, Ly, 0.0, 1.5, 16.5, spacing, 1.6, [PAULI, LONDON, COULOMB, ZERO])
        topo = tetracene(1001); n_rep = n_rep or 8192
        integ = dict(kind="vv", n_steps=5000, dt=0.5)
        vel_T = 300.0; twist = False
    else:
        raise ValueError("config 4 is a point workload: use c4_points / c4_samples")
    pos = place_replicas(topo, n_rep, Lx, Ly, 0.0, seed + 10, twist=twist)
    vel = maxwell_boltzmann(topo, n_rep, vel_T, seed + 20) if vel_T else np.zeros_like(pos)
    return dict(k=k, seed=seed, sub=sub, desc=desc, topo=topo, n_rep=n_rep, integ=integ, pos=pos, vel=vel)


def c4_points(n, Lx, Ly, z_lo_valid, z_hi_valid, seed=1004):
    """uniform points in the valid grid volume and per-point channel factors ~ U(-1,1)^3 (4th = 0)."""
    rng = np.random.default_rng(seed)
    pos = np.empty((n, 3), np.float32)
    pos[:, 0] = rng.uniform(0, Lx, n); pos[:, 1] = rng.uniform(0, Ly, n)
    pos[:, 2] = rng.uniform(z_lo_valid, z_hi_valid, n)
    coef = np.zeros((n, 4), np.float32)
    coef[:, :3] = rng.uniform(-1, 1, (n, 3))
    return pos, coef


def c4_sample_terms(seed=1004, nch=3):
    """parameters of the synthetic sweep potential: per channel 8 terms (m, n, phase, amplitude, decay)."""
    rng = np.random.default_rng(seed + 7)
    terms = []
    for c in range(nch):
        ch = []
        for _ in range(8):
            m, n_ = rng.integers(0, 4, 2); ph = rng.uniform(0, 2 * math.pi); amp = rng.normal()
            kap = rng.uniform(0.3, 1.6)
            ch.append((int(m), int(n_), float(ph), float(amp), float(kap)))
        terms.append(ch)
    return terms


def c4_samples(nx, ny, nz, h=0.1, z_lo=1.5, seed=1004, nch=3, xp=np, device=None):
    """smooth synthetic samples [nx][ny][nz][nch]: seeded sum of 8 plane-wave x exponential terms per channel.
    (An input, like an imported density-derived grid; not a step of the method.)  `xp` = numpy (default) or torch
    (with `device`), so that the 512 x 512 x 256 sweep grid can be filled where it will live; same terms, same formula."""
    terms = c4_sample_terms(seed, nch)
    if xp is np:
        ar = lambda n: np.arange(n, dtype=np.float64)
        out = np.zeros((nx, ny, nz, nch), np.float32)
    else:
        ar = lambda n: xp.arange(n, dtype=xp.float64, device=device)
        out = xp.zeros((nx, ny, nz, nch), dtype=xp.float32, device=device)
    x = (ar(nx) / nx)[:, None, None]; y = (ar(ny) / ny)[None, :, None]
    z = (z_lo + h * ar(nz))[None, None, :]
    for c in range(nch):
        acc = None
        for (m, n_, ph, amp, kap) in terms[c]:
            t = amp * xp.cos(2 * math.pi * (m * x + n_ * y) + ph) * xp.exp(-kap * (z - z_lo))
            acc = t if acc is None else acc + t
        out[..., c] = acc
    return out


def morton_order(pos, Lx, Ly, z0, nx, ny, hz, xp=np):
    """argsort of points by the Morton code of their grid cell (spatially sorted order for config 4).  `xp` = numpy, or torch for
    points that already live on the device (2^26 of them sort in milliseconds there)."""
    if xp is np:
        i64 = lambda v: v.astype(np.int64)
        clip = np.clip
    else:
        i64 = lambda v: v.to(xp.int64)
        clip = xp.clamp
    ix = clip(i64(pos[:, 0] / Lx * nx), 0, nx - 1)
    iy = clip(i64(pos[:, 1] / Ly * ny), 0, ny - 1)
    iz = clip(i64((pos[:, 2] - z0) / hz), 0, (1 << 10) - 1)

    def spread(v):
        v = v & 0x3FF
        v = (v | (v << 16)) & 0x30000FF
        v = (v | (v << 8)) & 0x300F00F
        v = (v | (v << 4)) & 0x30C30C3
        v = (v | (v << 2)) & 0x9249249
        return v
    code = spread(iz) | (spread(iy) << 1) | (spread(ix) << 2)
    return np.argsort(code, kind="stable") if xp is np else xp.argsort(code, stable=True)
