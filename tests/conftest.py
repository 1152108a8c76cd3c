import os
import sys
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    from oracle import gridff_oracle
    gridff_oracle.build()
    return gridff_oracle


@pytest.fixture(scope="session")
def small_slab():
    """2x2-site, 4-layer rock-salt slab (16 atoms, L = 5.64 Å) with +-0.7 e charges."""
    from paper_2508_15522_b200 import inputs
    sub, Lx, Ly = inputs.rocksalt_slab(2, 4, 2.82, 0.7)
    return sub, Lx, Ly


@pytest.fixture(scope="session")
def small_grid(orc, small_slab):
    """oracle grid on the small slab: h ~ 0.1 Å, z0 = 1.5, 70 z-nodes (top of the stored domain at 8.3 Å), channels Pauli, London, Coulomb."""
    sub, Lx, Ly = small_slab
    nx = ny = int(round(Lx / 0.1)); nz = 70
    samples = orc.sample_grid(sub, 1.6, Lx, Ly, 17.0, nx, ny, nz, 1.5, 0.1, [0, 1, 2])
    coef = orc.prefilter(samples, (1, 1, 0))
    return orc.OracleGrid(coef, Lx, Ly, 1.5, 0.1), samples
