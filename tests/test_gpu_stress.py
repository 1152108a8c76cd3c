"""Race stress test (run on the B200 box with -m gpu).  compute-sanitizer's racecheck / synccheck are closed on this GPU pool
(profiles/r2_sanitizers.md), so the shared-memory hand-overs of the kernels are tested by perturbing the schedule: csrc/libgridff_stress.so is
the same source built with -DGRIDFF_STRESS, which surrounds every synchronisation point (warp syncs, the named barriers of the pair-of-warps
kernel, the block barriers of the time-multiplexed rounds and of the filter, the TMA mbarrier waits) with pseudo-random per-lane delays of up
to ~1 us (gridff_internal.cuh: stress_delay).  Lanes and warps that normally run in lock-step then reach each hand-over at very different
times, so a missing or misplaced barrier, or a buffer re-used one phase too early, changes the numbers.  Asserted: the stress build returns
the product build's results BIT FOR BIT in every kernel mode exercised here.

The stress library is loaded by executing the binding's own source with the library name replaced — the product binding has no switch for it."""
import types

import numpy as np
import pytest
import torch

from paper_2508_15522_b200 import inputs
from paper_2508_15522_b200.csrc import build as cbuild
from gridff_cases import gpu_grid, small_config
from test_gpu_parity import api, dev, eval_points  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sapi(api):
    cbuild.build_stress()
    src = open(api.__file__).read()
    assert src.count('"libgridff.so"') == 1
    mod = types.ModuleType("gridff_api_stress")
    mod.__file__ = api.__file__
    exec(compile(src.replace('"libgridff.so"', '"libgridff_stress.so"'), api.__file__, "exec"), mod.__dict__)
    assert mod.LIB_PATH.endswith("libgridff_stress.so")
    return mod


def both(api, sapi, fn):
    """fn(binding) -> list of CUDA tensors / numpy arrays; run with the product and with the stress library, compare bit for bit"""
    a, b = fn(api), fn(sapi)
    torch.cuda.synchronize()
    assert len(a) == len(b)
    for k, (x, y) in enumerate(zip(a, b)):
        x = x.cpu().numpy() if isinstance(x, torch.Tensor) else np.asarray(x)
        y = y.cpu().numpy() if isinstance(y, torch.Tensor) else np.asarray(y)
        assert x.shape == y.shape and np.array_equal(x, y, equal_nan=True), "output %d differs under schedule stress" % k


def molecule(A, cfg):
    topo = cfg["topo"]
    return A.gridff_create_molecule(topo, A.gridff_atom_coefs(cfg["desc"]["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))


def test_eval_kernels_under_schedule_stress(api, sapi):
    cfg = small_config(1, n_rep=1)
    pos, coef = eval_points(cfg, 40013, 5)
    d = cfg["desc"]; nx, ny, nz = inputs.grid_dims(d)

    def run(A):
        g = gpu_grid(A, cfg["sub"], d)
        out = [A.gridff_grid_export(g)]
        dp, dc = dev(pos), dev(coef)
        order = inputs.morton_order(dp, d["Lx"], d["Ly"], d["z_ref"] + d["z_lo"], nx, ny, d["spacing"], xp=torch)
        sp, sc = dp[order].contiguous(), dc[order].contiguous()
        for v in (1, 2, 3):
            out += list(A.gridff_eval(g, dp, dc, variant=v)) + list(A.gridff_eval(g, sp, sc, variant=v))
        out += list(A.gridff_eval_binned(g, dp, dc))           # counting sort by atomics: the order inside a bin varies, the results must not
        for lay, variants in ((A.LAYOUT_HALF, (0,)), (A.LAYOUT_TRILINEAR, (0,)), (A.LAYOUT_MBRICK, (2,)), (A.LAYOUT_MBRICK2, (2,)), (A.LAYOUT_MBRICK8, (2, 3))):
            gd = A.gridff_grid_derive(g, lay)
            for v in variants:
                out += list(A.gridff_eval(gd, dp, dc, variant=v)) + list(A.gridff_eval(gd, sp, sc, variant=v))
        return out
    both(api, sapi, run)


@pytest.mark.parametrize("k", [1, 2])
def test_replica_kernels_under_schedule_stress(api, sapi, k):
    """k = 1: 30 atoms on one warp; k = 2: 60 atoms on a pair of warps (named barriers, two-word exchanges) and two atoms per lane (variant 4)"""
    cfg = small_config(k, n_rep=19)
    n = int(cfg["topo"]["n_atoms"])
    vel = inputs.maxwell_boltzmann(cfg["topo"], 19, 300.0, 23)

    def run(A):
        g = gpu_grid(A, cfg["sub"], cfg["desc"])
        mol = molecule(A, cfg)
        out = []
        for v in ((2, 3, 5) if k == 1 else (2, 3, 4)):
            p, w = dev(cfg["pos"]), dev(vel)
            r = A.gridff_run_replicas(g, mol, A.make_integrator("vv", 150, 0.5, variant=v), p, w)
            out += [p, w, r["energy"]]
        p, w = dev(cfg["pos"]), dev(vel)
        r = A.gridff_run_replicas(g, mol, A.make_integrator("langevin", 150, 0.5, temperature=300.0, gamma=0.01, seed=11, fixed=(0, n - 1)), p, w)
        out += [p, w, r["energy"]]
        # FIRE with restart: records land in the order replicas converge (an atomic counter), so compare them sorted by (replica, restart)
        p, w = dev(cfg["pos"]), torch.zeros_like(dev(vel))
        fire = torch.zeros((19, 4), device="cuda"); mn = torch.zeros((256, 4 + 3 * n), device="cuda"); nmn = torch.zeros(1, dtype=torch.int32, device="cuda")
        r = A.gridff_run_replicas(g, mol, A.make_integrator("fire", 400, 0.5, f_tol=0.3, restart=1, seed=5, dt_max=5.0, max_step=0.1), p, w,
                                  d_fire=fire, d_minima=mn, d_n_minima=nmn)
        m = mn[:min(int(nmn.item()), 256)].cpu().numpy()
        m = m[np.lexsort((m[:, 1], m[:, 0]))] if int(nmn.item()) <= 256 else np.zeros(0)
        out += [p, w, fire, r["energy"], r["status"], nmn, m]
        p, w = dev(cfg["pos"]), torch.zeros_like(dev(vel))
        r = A.gridff_run_scan(g, mol, A.make_integrator("fire", 60, 1.0, f_tol=0.05, dt_max=10.0, max_step=0.05, n_scan=3, fixed=(n - 1,), scan_dx=(0.0, 0.0, 0.1)), p, w)
        out += [p, r["scan"], r["energy"], r["status"]]
        return out
    both(api, sapi, run)


def test_time_multiplexed_blocks_and_hopping_under_schedule_stress(api, sapi):
    """more replicas than resident warp slots x 512 steps: the blocks cycle their replicas over their warps, the state passing through global
    memory across the block barrier; then two minima-hopping cycles (Langevin, FIRE, collect, library filter, sequential append)"""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    n_rep = sms * 16 + 21
    cfg = small_config(1, n_rep=n_rep)

    def run(A):
        g = gpu_grid(A, cfg["sub"], cfg["desc"])
        mol = molecule(A, cfg)
        out = []
        for kind, kw in (("vv", {}), ("langevin", dict(temperature=300.0, gamma=0.01, seed=3))):
            p, w = dev(cfg["pos"]), dev(cfg["vel"])
            r = A.gridff_run_replicas(g, mol, A.make_integrator(kind, 512, 0.5, **kw), p, w)
            out += [p, w, r["energy"]]
        hop = A.make_hopping(2, 60, 0.5, 300.0, 0.01, 300, 1.0, 0.3, seed=7, dt_max=10.0, max_step=0.1)
        p = dev(cfg["pos"][:64])
        lib = torch.zeros((256, 4 + 3 * 30), device="cuda"); nlib = torch.zeros(1, dtype=torch.int32, device="cuda")
        st = A.gridff_minima_hopping(g, mol, hop, p, lib, nlib)
        out += [p, lib, nlib, st]
        return out
    both(api, sapi, run)
