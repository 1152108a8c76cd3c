"""gridff_eval_binned_noalloc — the entry point for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid
cudaMalloc): gridff_eval_binned's passes with the work space in a 16 MiB device array built into the library (include/gridff.h).  Checked
against the existing paths (gridff_eval_binned with caller work space, gridff_eval) BIT FOR BIT — the bar tests/test_gpu_variants.py holds the
binned path to — and against the fp64 oracle at north_star's interpolation tolerances, on calls in a row that share the array.  Collected last
(the name): run on the B200 box with -m gpu, alone or after the other tests."""
import numpy as np
import pytest
import torch

from gridff_cases import oracle_grid, gpu_grid, small_config, energy_denominator

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    from paper_2508_15522_b200 import api
    return api


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float32).cuda()


def points(cfg, n, seed):
    """scattered points: wrapped coordinates, 1000 copies of one point (a bin far larger than a warp), points far above the domain (their own bin)"""
    rng = np.random.default_rng(seed)
    d = cfg["desc"]
    pos = np.stack([rng.uniform(-2 * d["Lx"], 3 * d["Lx"], n), rng.uniform(-2 * d["Ly"], 3 * d["Ly"], n), rng.uniform(1.55, 8.6, n)], 1).astype(np.float32)
    coef = np.zeros((n, 4), np.float32)
    coef[:, :3] = rng.uniform(-1, 1, (n, 3))
    if n >= 5000:
        pos[100:1100] = pos[100]
        pos[2000:2100, 2] = 1e30
    return pos, coef


def test_noalloc_entry_point_matches_the_existing_paths(api, orc):
    cfg = small_config(1, n_rep=8)
    g = gpu_grid(api, cfg["sub"], cfg["desc"])
    og, _ = oracle_grid(orc, cfg["sub"], cfg["desc"])
    assert api.gridff_eval_binned_noalloc_max_bytes() == 16 << 20
    # calls in a row over ONE shared array, with different point counts so that every call finds the previous call's ranks, records, results and
    # bin counters in it: the largest count allowed, a smaller ragged one, one point, the first again
    sets = [points(cfg, 1 << 18, 11), points(cfg, 150011, 12), points(cfg, 1, 13), points(cfg, 1 << 18, 11)]
    for k, (pos, coef) in enumerate(sets):
        n = len(pos)
        dp, dc = dev(pos), dev(coef)
        E_ref, F_ref = api.gridff_eval_binned(g, dp, dc)                       # the existing path: caller-supplied work space
        E_pl, F_pl = api.gridff_eval(g, dp, dc, variant=2)                     # and the plain gather
        E = torch.full((n,), float("nan"), device="cuda")
        F = torch.full((n, 3), float("nan"), device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]                                   # the driver's view: torch's own pool is not touched between the two readings
        api.gridff_eval_binned_noalloc(g, dp, dc, E, F)
        api.gridff_eval_binned_noalloc(g, dp, dc, E, F)                        # twice back to back on the stream: the second overwrites the first's scratch
        torch.cuda.synchronize()
        if k > 0:                                                              # (the first call of a process may load the module: not counted)
            assert torch.cuda.mem_get_info()[0] >= free0, "the no-alloc entry point took device memory"
        assert bool(torch.equal(E, E_ref)) and bool(torch.equal(F, F_ref)), "call %d (n = %d) differs from gridff_eval_binned" % (k, n)
        assert bool(torch.equal(E, E_pl)) and bool(torch.equal(F, F_pl)), "call %d (n = %d) differs from gridff_eval" % (k, n)
        # against the oracle on a sample (north_star: E 1e-5 relative to sum_c |coef_c V_c|, F 1e-4 eV/Å)
        idx = np.random.default_rng(k).choice(n, min(n, 3000), replace=False)
        Eo, Fo, Vc, _ = orc.interp(og, pos[idx], coef[idx], channels=True)
        den = np.maximum(energy_denominator(coef[idx].astype(np.float64), Vc), 1e-12)
        assert (np.abs(E.cpu().numpy()[idx] - Eo) / den).max() <= 1e-5
        assert np.abs(F.cpu().numpy()[idx] - Fo).max() <= 1e-4
    # outputs are optional as in gridff_eval
    api.gridff_eval_binned_noalloc(g, dp, dc, E, None)
    api.gridff_eval_binned_noalloc(g, dp, dc, None, F)
    torch.cuda.synchronize()
    assert bool(torch.equal(E, E_ref)) and bool(torch.equal(F, F_ref))
    # an empty batch is a no-op
    api.gridff_eval_binned_noalloc(g, torch.zeros((0, 3), device="cuda"), torch.zeros((0, 4), device="cuda"), E[:0], F[:0])


def test_noalloc_entry_point_rejects_what_does_not_fit(api):
    cfg = small_config(1, n_rep=8)
    g = gpu_grid(api, cfg["sub"], cfg["desc"])
    n = (1 << 18) + 1
    dp, dc = torch.zeros((n, 3), device="cuda"), torch.zeros((n, 4), device="cuda")
    E, F = torch.full((n,), 7.0, device="cuda"), torch.full((n, 3), 7.0, device="cuda")
    launches = api.gridff_launch_count()
    with pytest.raises(api.GridffError) as e:
        api.gridff_eval_binned_noalloc(g, dp, dc, E, F)
    assert e.value.code == api.ESIZE and "at most 262144 points" in str(e.value)
    torch.cuda.synchronize()
    assert api.gridff_launch_count() == launches and bool((E == 7.0).all()) and bool((F == 7.0).all())       # nothing ran
    gb = gpu_grid(api, cfg["sub"], cfg["desc"], layout=1)
    with pytest.raises(api.GridffError):
        api.gridff_eval_binned_noalloc(gb, dp[:100], dc[:100], E[:100], F[:100])                             # brick layout: refused like gridff_eval_binned
