"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/gridff.h declares, validates
arguments on the host, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def api():
    from paper_2508_15522_b200.csrc import build
    build.build()
    from paper_2508_15522_b200 import api
    return api


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "gridff.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gridff_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(api):
    names = declared_symbols()
    assert len(names) >= 20
    lib = C.CDLL(api.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), "libgridff.so does not export %s" % n
    assert set(api.EXPORTS) == set(names), "python binding and header disagree: %s" % (set(api.EXPORTS) ^ set(names))


def test_grid_dims_follow_the_descriptor(api):
    d = api.make_desc(11.28, 11.28, 0.0, 1.5, 11.5, 0.1, 1.6, [0, 1, 2])
    dims, h, org = api.gridff_grid_dims(d)
    assert dims == (113, 113, 100)                       # BASELINE config 0/1: 113 x 113 x 100 nodes
    assert abs(h[0] - 11.28 / 113) < 1e-15 and h[2] == 0.1 and org == (0.0, 0.0, 1.5)
    store, scratch = api.gridff_grid_bytes(d, 64)
    assert store >= 116 * 116 * 104 * 16 and scratch >= 3 * 113 * 113 * 100 * 8


def test_bad_arguments_are_rejected(api):
    bad = api.make_desc(11.28, 11.28, 0.0, 1.5, 1.0, 0.1, 1.6, [0, 1])
    with pytest.raises(api.GridffError) as e:
        api.gridff_grid_dims(bad)
    assert e.value.code == api.EINVAL and "z range" in str(e.value)
    with pytest.raises(api.GridffError):
        api.gridff_grid_dims(api.make_desc(11.28, 11.28, 0.0, 1.5, 11.5, 0.1, 1.6, [0, 1], layout=7))


def test_atom_coefs_host_helper(api):
    # Eq. 4 factors in closed form for one atom: e=0.05, R=1.5, alpha=1.6
    c = api.gridff_atom_coefs(1.6, [0.05], [1.5], [0.25])
    assert np.allclose(c[0], [0.05 * np.exp(4.8), -0.1 * np.exp(2.4), 0.25, 0.0], rtol=1e-6)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback(api):
    from paper_2508_15522_b200 import inputs
    sub, Lx, Ly = inputs.rocksalt_slab(2, 2, 2.82, 0.7)
    d = api.make_desc(Lx, Ly, 0.0, 1.5, 3.5, 0.2, 1.6, [0, 1])
    with pytest.raises(api.GridffError) as e:
        api.gridff_build_grid(d, sub["pos"], sub["e"], sub["R"], sub["q"])
    assert e.value.code == api.ECUDA
