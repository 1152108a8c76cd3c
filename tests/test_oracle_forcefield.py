"""Pins for the oracle's intramolecular force field (R12): textbook small cases, finite differences,
zero net force and torque (CPU only)."""
import math
import numpy as np
import pytest
from paper_2508_15522_b200 import inputs

KE = 14.3996454784


def _topo(n, **kw):
    t = dict(n_atoms=n, mass=np.ones(n), q=np.zeros(n), lj_e=np.zeros(n), lj_R=np.ones(n),
             bond=np.zeros((0, 2)), bond_k_r0=np.zeros((0, 2)), angle=np.zeros((0, 3)), angle_k_t0=np.zeros((0, 2)),
             tors=np.zeros((0, 4)), tors_k_n_p0=np.zeros((0, 3)), excl=np.ones((n, n), np.uint8))
    t.update(kw)
    return t


def test_two_atom_bond(orc):
    t = orc.OracleTopology(_topo(2, bond=[[0, 1]], bond_k_r0=[[30.0, 1.4]]), np.zeros((2, 4)))
    E, F = orc.intramolecular(t, [[0, 0, 0], [0, 0, 1.5]])
    assert abs(E[0] - 0.5 * 30 * 0.01) < 1e-15
    assert np.allclose(F, [[0, 0, 3.0], [0, 0, -3.0]])          # stretched bond pulls the atoms together


def test_two_atom_lj_coulomb(orc):
    ex = np.eye(2, dtype=np.uint8)
    t = orc.OracleTopology(_topo(2, q=[0.3, -0.2], lj_e=[0.05, 0.08], lj_R=[1.9, 1.4], excl=ex), np.zeros((2, 4)))
    R = 3.3
    E, F = orc.intramolecular(t, [[0, 0, 0], [R, 0, 0]])        # at r = R_ij the LJ energy is -eps_ij, LJ force zero
    assert abs(E[3] - (-0.05 * 0.08 + KE * 0.3 * -0.2 / R)) < 1e-15
    assert abs(F[1, 0] - (KE * 0.3 * -0.2 / R ** 2)) < 1e-13   # attraction pulls atom 1 towards -x
    E, _ = orc.intramolecular(t, [[0, 0, 0], [R / 2 ** (1 / 6), 0, 0]])
    assert abs(E[3] - KE * 0.3 * -0.2 / (R / 2 ** (1 / 6))) < 1e-14     # LJ zero crossing at R / 2^(1/6)


def test_three_atom_angle(orc):
    t = orc.OracleTopology(_topo(3, angle=[[0, 1, 2]], angle_k_t0=[[5.0, math.radians(120)]]), np.zeros((3, 4)))
    th = math.radians(100)
    pos = [[1.2, 0, 0], [0, 0, 0], [1.5 * math.cos(th), 1.5 * math.sin(th), 0]]
    E, F = orc.intramolecular(t, pos)
    assert abs(E[1] - 0.5 * 5 * math.radians(20) ** 2) < 1e-14
    # |F_i| = |dE/dtheta| / |a|, perpendicular to the arm, opening the angle (theta < theta0)
    assert abs(np.linalg.norm(F[0]) - 5 * math.radians(20) / 1.2) < 1e-13
    assert abs(F[0] @ np.array(pos[0])) < 1e-13 and F[0][1] < 0
    assert np.abs(F.sum(0)).max() < 1e-14


def test_four_atom_torsion(orc):
    t = orc.OracleTopology(_topo(4, tors=[[0, 1, 2, 3]], tors_k_n_p0=[[0.1, 3.0, 0.0]]), np.zeros((4, 4)))
    for phi in (0.0, 0.4, math.pi / 3, 2.0, -1.1, math.pi - 1e-3):
        pos = [[1, 0, 0], [0, 0, 0], [0, 0, 1.5], [math.cos(phi), math.sin(phi), 1.5]]
        E, F = orc.intramolecular(t, pos)
        assert abs(E[2] - 0.1 * (1 + math.cos(3 * phi))) < 1e-14      # cis = 0, right-handed positive
        # torque about the axis on atom 3 = -dE/dphi
        tz = pos[3][0] * F[3][1] - pos[3][1] * F[3][0]
        assert abs(tz - 0.1 * 3 * math.sin(3 * phi)) < 1e-13


@pytest.mark.parametrize("mol", ["tetracene", "chain60"])
def test_molecule_fd_and_momentum(orc, mol):
    topo = getattr(inputs, mol)()
    n = topo["n_atoms"]
    t = orc.OracleTopology(topo, np.zeros((n, 4)))
    rng = np.random.default_rng(11)
    pos = topo["ref_pos"] + rng.normal(0, 0.05, (n, 3))
    E, F = orc.intramolecular(t, pos)
    assert np.abs(F.sum(0)).max() < 1e-11
    assert np.abs(np.cross(pos, F).sum(0)).max() < 1e-10
    d = 1e-5
    for i in rng.choice(n, 6, replace=False):
        for c in range(3):
            pp, pm = pos.copy(), pos.copy(); pp[i, c] += d; pm[i, c] -= d
            fd = -(orc.intramolecular(t, pp)[0].sum() - orc.intramolecular(t, pm)[0].sum()) / (2 * d)
            assert abs(F[i, c] - fd) < 1e-6 * max(1.0, np.abs(F).max())
    # the template is strain-free in bonds and angles by construction
    E0, _ = orc.intramolecular(t, topo["ref_pos"])
    assert E0[0] < 1e-10 and E0[1] < 1e-10
    if mol == "tetracene":
        assert E0[2] < 1e-12                                  # planar: ring torsions at their minimum


def test_four_channel_energy_is_the_potential_of_the_forces(orc):
    """DESIGN.md R22: with a 4-channel grid (an imported potential) the 7 reported terms sum to the potential whose gradient
    the forces are: the fourth channel is reported with the third.  Central finite differences of sum(E7) against F, and the channel
    split itself against per-channel interpolation."""
    rng = np.random.default_rng(3)
    nx = ny = 12; nz = 20; h = 0.25
    coef = rng.normal(size=(nx, ny, nz, 4))
    g = orc.OracleGrid(coef, nx * h, ny * h, 1.0, h)
    n = 3
    cf = rng.uniform(0.5, 1.5, (n, 4))
    t = orc.OracleTopology(_topo(n), cf)
    pos = np.array([[0.7, 1.9, 2.3], [2.2, 0.4, 3.1], [1.1, 2.6, 4.0]])
    E7, F = orc.forces(g, t, pos)
    _, _, Vc, _ = orc.interp(g, pos, cf, channels=True)
    per = (cf * Vc).sum(axis=0)
    assert np.allclose(E7[:3], [per[0], per[1], per[2] + per[3]], rtol=0, atol=1e-13) and abs(per[3]) > 1e-3
    eps = 1e-5
    for i in range(n):
        for c in range(3):
            p1, p2 = pos.copy(), pos.copy(); p1[i, c] += eps; p2[i, c] -= eps
            dE = (orc.forces(g, t, p1)[0].sum() - orc.forces(g, t, p2)[0].sum()) / (2 * eps)
            assert abs(dE + F[i, c]) < 1e-7 * max(1.0, abs(F[i, c]))
