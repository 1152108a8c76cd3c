"""GPU-vs-oracle parity for the on-device unique-structure filter and the minima-hopping loop, through the
C-ABI (gridff_unique_filter, gridff_minima_hopping).  Run on the B200 box with -m gpu.

The filter takes discrete decisions from floating-point tests; the inputs here keep every decision away from its threshold
(same-structure copies at RMSD ~ 0.02 Å, distinct ones at > 1 Å or > 5 e_tol), so fp32 and fp64 must agree record for record.
The hopping loop is chaotic over 1000 thermal steps, so it is checked by what is unique: every record is a
true minimum under the oracle's forces, records are pairwise distinct, every converged replica is represented, and the launch-split
invariance holds bit for bit."""
import numpy as np
import pytest
import torch

from paper_2508_15522_b200 import inputs
from gridff_cases import oracle_grid, gpu_grid, small_config
from test_gpu_parity import api, dev, oracle_side, gpu_side  # noqa: F401
from test_oracle_hopping import _population

pytestmark = pytest.mark.gpu


def test_unique_filter_matches_oracle_record_for_record(api, orc):
    cfg = small_config(0, n_rep=1)                         # benzene: n = 12 atoms, cell 5.64 Å
    g = gpu_grid(api, cfg["sub"], cfg["desc"])
    mol = gpu_side(api, cfg)
    Lx = cfg["desc"]["Lx"]
    rng = np.random.default_rng(7)
    import test_oracle_hopping as toh
    old = (toh.LX, toh.LY); toh.LX = toh.LY = Lx
    try:
        X, E, label, _, _ = _population(rng, K=40, copies=30)          # 1200 candidates, 40 classes: several warps and blocks, ragged
    finally:
        toh.LX, toh.LY = old
    X = X.astype(np.float32); E = E.astype(np.float32)
    ok = np.ones(len(X), np.int32); ok[::11] = 0
    lib_o = []
    st_o = orc.unique_filter(lib_o, E.astype(np.float64), X.astype(np.float64), ok.astype(bool), Lx, Lx, tag=3)
    d_lib = torch.zeros((64, 4 + 36), device="cuda"); d_n = torch.zeros(1, dtype=torch.int32, device="cuda")
    # two calls: the first half of the replicas, then all of them (old records + same-call records are both exercised)
    half = len(X) // 2
    ok1 = ok.copy(); ok1[half:] = 0
    s1 = api.gridff_unique_filter(g, mol, dev(X), dev(E), dev(ok1, torch.int32), d_lib, d_n, tag=3).cpu().numpy()
    ok2 = ok.copy(); ok2[:half] = 0
    s2 = api.gridff_unique_filter(g, mol, dev(X), dev(E), dev(ok2, torch.int32), d_lib, d_n, tag=3).cpu().numpy()
    n_lib = int(d_n.item()); lib_g = d_lib.cpu().numpy()[:n_lib]
    assert n_lib == len(lib_o) == 40 and s1[0] + s2[0] == st_o[0] and s1[1] + s2[1] == st_o[1] and s2[3] == 40
    assert np.array_equal(lib_g[:, 0].astype(int), np.array([int(r[0]) for r in lib_o]))           # same representatives, same order
    assert np.array_equal(lib_g[:, 4:], np.array([r[4:] for r in lib_o], np.float32))
    assert np.all(lib_g[:, 1] == 3)
    # a full library drops
    d_lib2 = torch.zeros((5, 40), device="cuda"); d_n2 = torch.zeros(1, dtype=torch.int32, device="cuda")
    s3 = api.gridff_unique_filter(g, mol, dev(X), dev(E), dev(ok, torch.int32), d_lib2, d_n2).cpu().numpy()
    assert int(d_n2.item()) == 5 and s3[1] == 5 and s3[2] > 0
    # nothing to do
    s4 = api.gridff_unique_filter(g, mol, dev(X), dev(E), dev(np.zeros_like(ok), torch.int32), d_lib, d_n).cpu().numpy()
    assert s4[0] == 0 and s4[1] == 0 and int(d_n.item()) == 40


def _hop(api, g, mol, pos, n_cycles, cycle0=0, lib=None, nlib=None, n_atoms=12, **kw):
    d_pos = dev(pos)
    d_lib = torch.zeros((256, 4 + 3 * n_atoms), device="cuda") if lib is None else lib
    d_n = torch.zeros(1, dtype=torch.int32, device="cuda") if nlib is None else nlib
    st = api.gridff_minima_hopping(g, mol, api.make_hopping(n_cycles, cycle0=cycle0, **kw), d_pos, d_lib, d_n)
    torch.cuda.synchronize()
    return d_pos.cpu().numpy(), d_lib, d_n, st.cpu().numpy()


def test_minima_hopping_loop(api, orc):
    cfg = small_config(0, n_rep=40)
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    g = gpu_grid(api, cfg["sub"], cfg["desc"])
    ot, mol = oracle_side(orc, cfg, og), gpu_side(api, cfg)
    kw = dict(md_steps=200, md_dt=0.5, temperature=300.0, gamma=0.02, relax_steps=6000, relax_dt=1.0, f_tol=2e-3, seed=9, dt_max=10.0, max_step=0.1)
    pos, d_lib, d_n, st = _hop(api, g, mol, cfg["pos"], 3, **kw)
    n_lib = int(d_n.item()); lib = d_lib.cpu().numpy()[:n_lib]
    print("hopping: stats per cycle (candidates, new, dropped, library size):", st.tolist())
    assert st[:, 0].min() >= 10 and st[-1, 0] >= 30 and n_lib == st[:, 1].sum() == st[-1, 3] and n_lib >= 2 and st[:, 2].sum() == 0
    Lx = cfg["desc"]["Lx"]
    # every record is a minimum under the oracle's forces and carries the oracle's energy
    for rec in lib[:24]:
        E7, F = orc.forces(og, ot, rec[4:].reshape(-1, 3).astype(np.float64))
        assert np.sqrt((F ** 2).sum(1)).max() < 2.2e-3
        assert abs(E7.sum() - rec[3]) < 1e-4
    # pairwise distinct (oracle criterion, 10 % margin on the thresholds for the fp32 decisions)
    for i in range(n_lib):
        for j in range(i):
            assert not orc.same_structure(lib[i][3], lib[i][4:].reshape(-1, 3), lib[j][3], lib[j][4:].reshape(-1, 3), Lx, Lx, 0.9e-3, 0.09)
    # the replicas' final states (cycle 3 minima) are represented
    E_fin = []
    for r in range(40):
        E7, F = orc.forces(og, ot, pos[r].astype(np.float64))
        if np.sqrt((F ** 2).sum(1)).max() < 2e-3:
            assert any(orc.same_structure(E7.sum(), pos[r], rec[3], rec[4:].reshape(-1, 3), Lx, Lx, 1.1e-3, 0.11) for rec in lib)
            E_fin.append(E7.sum())
    assert len(E_fin) >= 30
    # 3 cycles in one call == 1 + 2 cycles in two calls, bit for bit
    p1, l1, n1, _ = _hop(api, g, mol, cfg["pos"], 1, **kw)
    p2, l2, n2, _ = _hop(api, g, mol, p1, 2, cycle0=1, lib=l1, nlib=n1, **kw)
    assert np.array_equal(p2, pos) and int(n2.item()) == n_lib and np.array_equal(l2.cpu().numpy()[:n_lib], lib)
    # the first cycle against the oracle, phase by phase on the same inputs: Langevin 200 steps is chaotic beyond ~100 steps, so compare
    # the oracle's loop only statistically: same number of candidates, library sizes within a factor 2
    o = orc.minima_hopping(og, ot, cfg["pos"], 1, **kw)
    assert abs(int(o["stats"][0, 0]) - int(st[0, 0])) <= 6
    assert 0.5 * o["stats"][0, 1] <= st[0, 1] <= 2 * o["stats"][0, 1] + 1
