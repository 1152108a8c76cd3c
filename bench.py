#!/usr/bin/env python
"""bench.py — GridFF hot path on B200: replica MD steps/s, atom-grid evals/s and fraction of the gather roofline.

A "step" is one pass of the whole hot path over one batch of synthetic input:
    gridff_build_grid (sample Morse + Coulomb channels, prefilter, interleaved store)
    gridff_run_replicas (n_rep replicas x n_md_steps of the fused grid + intramolecular + integrator kernel).
Default workload = BASELINE.json configs[1]: NaCl(001) 4x4 slab with Coulomb, 113 x 113 x 100 x 3-channel grid, 4096 replicas of the
30-atom flexible aromatic, velocity Verlet, dt 0.5 fs, 10,000 steps.

    python bench.py --gpus 1 --steps 5 --warmup 3
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...     (replicas only: each rank runs its own batch)
    python bench.py --impl reference          (the fp64 CPU oracle on a bounded sample of the same workload)
"""
import argparse
import ctypes as C
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2508_15522_b200 import inputs  # noqa: E402

METRIC = "replica_md_steps_per_s"
UNIT = "replica-steps/s"
BYTES_PER_EVAL = 1024          # 64 nodes x 16 B stored per node: the algorithmic gather bytes of one atom-grid eval


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gridff", choices=["gridff", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--md-steps", type=int, default=0, help="override the config's MD steps per launch (0 = config value)")
    ap.add_argument("--replicas", type=int, default=0, help="override the config's replica count (0 = config value)")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="default (config 1, N = 1) run: skip the short extra measurements of configs 2, 3 and 4 reported under 'also'")
    ap.add_argument("--mode", default="run", choices=["run", "langevin", "hopping", "scan", "drag"],
                    help="SURVEY §8(f) rows on the chosen replica config: langevin = kind 2 instead of the config's integrator; hopping = "
                         "gridff_minima_hopping cycles (1000 Langevin steps at 300 K + FIRE); scan = gridff_run_scan lift of one held atom; "
                         "drag = the paper's defect protocol (L184, L200-202): a Na-Cl vacancy pair is cut into the config's substrate and every "
                         "replica drags its held atom across it in 40 steps of 0.1 A, relaxing at each (use with --config 3 for the 20x20 cell)")
    ap.add_argument("--log2-points", type=int, default=26, help="config 4: number of interpolation points = 2^k")
    ap.add_argument("--order", default="random", choices=["random", "sorted"], help="config 4: point order (sorted = Morton order of the cell)")
    ap.add_argument("--c4-grid", default="config1", help="config 4: 'config1' (the 113 x 113 x 100 NaCl grid) or NXxNYxNZ synthetic sweep grid")
    ap.add_argument("--c4-store", default="fp32", choices=["fp32", "half", "trilinear", "bricks", "bricks2", "bricks8"],
                    help="config 4: coefficient store read by gridff_eval: the fp32 spline z-fastest (default), fp16 coefficients, the paper's trilinear foil "
                         "(SURVEY §8(f)3), or the fp32 spline in 2x2x2-node bricks of 128 B, 1 / 2 / 8 shifted copies (the layouts for stores beyond the L2)")
    ap.add_argument("--binned", action="store_true", help="config 4: time gridff_eval_binned (device-side counting sort of the points by cell block, then the "
                                                          "gather) instead of gridff_eval; z-fastest fp32 store only")
    ap.add_argument("--sweep", action="store_true", help="config 4: also time the grid-size x order sweep (32^3 ... 512x512x256)")
    return ap.parse_args()


def workload(args):
    cfg = inputs.config(args.config, n_rep=args.replicas or None)
    md = args.md_steps or cfg["integ"]["n_steps"]
    nx, ny, nz = inputs.grid_dims(cfg["desc"])
    name = {0: "config0: NaCl(001) 4x4 slab, 2 channels, 64 x benzene, FIRE x 1000",
            2: "config2: config1 grid, 16384 x 60-atom flexible chain, FIRE (dt0 0.5 fs, dt_max 20 fs, displacement cap 0.1 A per step) to 1e-3 eV/A, "
               "cap 20000 iterations per launch, + Philox restart; every replica starts from its own seeded clash-free random dihedrals",
            1: "config1: NaCl(001) 4x4 slab + Coulomb, 4096 x 30-atom aromatic, VV dt 0.5 fs x 10000",
            3: "config3: 40x40 Å slab, 400x400x150x4 grid (384 MB), 8192 x 30-atom aromatic, VV x 5000"}[args.config]
    return cfg, md, (nx, ny, nz), name


# ------------------------------------------------------------------------------------------------------------------ oracle arm

def oracle_sample(cfg, md_steps, n_rep_sample=512, steps_sample=1000):
    """Times the fp64 oracle, as it stands, on a bounded sample: the whole grid build (a1-a3) + n_rep_sample replicas x
    steps_sample steps (a5-a9).  Returns (t_build, t_per_replica_step, cores)."""
    from oracle import gridff_oracle as orc
    d = cfg["desc"]; nx, ny, nz = inputs.grid_dims(d); z0 = d["z_ref"] + d["z_lo"]
    # bounded sample of the build: the direct sums cost nodes x atoms x images; above ~2e10 pair terms (config 3: 2.6e11) only the lowest
    # nz_s z-planes are built and the sampling time is scaled by nz / nz_s (it is linear in the node count)
    n_img = int(np.prod([2 * int(np.ceil(d["r_cut"] / L)) + 1 for L in (d["Lx"], d["Ly"])]))
    work = float(nx) * ny * nz * len(cfg["sub"]["pos"]) * n_img
    nz_s = nz if work <= 2e10 else max(8, int(nz * 2e10 / work))
    t0 = time.perf_counter()
    samples = orc.sample_grid(cfg["sub"], d["alpha"], d["Lx"], d["Ly"], d["r_cut"], nx, ny, nz_s, z0, d["spacing"], d["channels"])
    t_sample = time.perf_counter() - t0
    if nz_s < nz:
        # the run leg needs a grid under the molecules: prefilter (timed, full size) smooth synthetic samples of the config's dimensions —
        # interpolation cost does not depend on the values
        samples = inputs.c4_samples(nx, ny, nz, h=d["spacing"], z_lo=d["z_lo"], nch=len(d["channels"])).astype(np.float64)
    t0 = time.perf_counter()
    og = orc.OracleGrid(orc.prefilter(samples, (1, 1, 0)), d["Lx"], d["Ly"], z0, d["spacing"])
    t_build = t_sample * nz / nz_s + (time.perf_counter() - t0)
    topo = cfg["topo"]
    ot = orc.OracleTopology(topo, orc.atom_coefs(topo["grid_e"], topo["grid_R"], topo["q"], d["alpha"]))
    kind = cfg["integ"]["kind"]
    integ = orc.make_integrator(kind, steps_sample, cfg["integ"]["dt"], f_tol=1e-12)
    n = min(n_rep_sample, cfg["n_rep"])
    t0 = time.perf_counter()
    orc.run_replicas(og, ot, integ, cfg["pos"][:n], cfg["vel"][:n])
    t_run = time.perf_counter() - t0
    return t_build, t_run / (n * steps_sample), orc.num_threads(), n, steps_sample


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, md, dims, name = workload(args)
    total = cfg["n_rep"] * md
    times, extrap = [], []
    for it in range(args.warmup + args.steps):
        tb, tps, cores, n, ss = oracle_sample(cfg, md)
        if it >= args.warmup:
            times.append(tb + n * ss * tps)          # MEASURED: one step of the sample = grid build + n replicas x ss steps
            extrap.append(total / (tb + total * tps))
    t = float(np.mean(times))
    val = n * ss / t                                 # replica-steps/s of the sample as run (nothing projected)
    sample = ("one step = the whole fp64 grid build (a1-a3) + %d replicas x %d steps (a5-a9) of the %d x %d workload; value = those replica-steps / the "
              "measured time; 'extrapolated_full_workload' = the same two measured rates projected to the whole workload" % (n, ss, cfg["n_rep"], md))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "grid": list(dims), "n_replicas": cfg["n_rep"], "md_steps_per_step": md, "atoms": int(cfg["topo"]["n_atoms"])},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "extrapolated_full_workload": float(np.mean(extrap))},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------------------------ GPU arm

def ncu_facts(key):
    """what ncu measured for this config's dominant kernel at the last capture (profiles/ncu_facts.json, written from the committed
    captures): measured L2 -> L1 bytes, pipe utilisations, the binding unit.  None when no capture exists for the config."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "ncu_facts.json"))).get(key)
    except Exception:
        return None


class ClockSampler:
    Q = "index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index = index
        try:
            self.p = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill(); out, _ = self.p.communicate()
        sm, mx, pw, reasons = [], 0.0, 0.0, set()
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 8 or not f[0].isdigit() or int(f[0]) != self.index:
                continue
            try:
                sm.append(float(f[1])); mx = max(mx, float(f[2])); pw = max(pw, float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "power_w_max": pw or None,
                "samples": len(sm), "reasons": sorted(reasons)}


def run_f_rows(args):
    """--mode langevin | hopping | scan: device-timed throughput of the §8(f) entry points on the config's grid and molecule (one GPU)."""
    import torch
    from paper_2508_15522_b200 import api
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(0)
    cfg, md, dims, name = workload(args)
    d, topo, sub = cfg["desc"], cfg["topo"], cfg["sub"]
    n_rep, n_at = cfg["n_rep"], int(topo["n_atoms"])
    if args.mode == "drag":
        sub, removed = inputs.vacancy_pair(sub, d["Lx"], d["Ly"])
        cfg["pos"] = inputs.drag_starts(topo, n_rep, n_at - 1, removed[:, :2].mean(axis=0) - [2.0, 0.0], 3.3, 1.0, cfg["seed"] + 30)
    g = api.gridff_build_grid(api.make_desc(d["Lx"], d["Ly"], d["z_ref"], d["z_lo"], d["z_hi"], d["spacing"], d["alpha"], d["channels"], r_cut=d["r_cut"], l2_persist=1),
                              sub["pos"], sub["e"], sub["R"], sub["q"])
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(d["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    pos0 = torch.from_numpy(cfg["pos"]).cuda()
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    l0 = api.gridff_launch_count()
    extra = {}
    ts = []
    for it in range(max(args.warmup, 3) + args.steps):
        d_pos = pos0.clone(); d_vel = torch.zeros_like(d_pos)
        flush.fill_(1)
        a, b = ev(), ev()
        if args.mode == "langevin":
            integ = api.make_integrator("langevin", md, 0.5, temperature=300.0, gamma=0.01, seed=7)
            a.record(stream); api.gridff_run_replicas(g, mol, integ, d_pos, d_vel); b.record(stream); b.synchronize()
            units = n_rep * md
        elif args.mode == "hopping":
            cycles = 2
            hop = api.make_hopping(cycles, 1000, 0.5, 300.0, 0.01, 5000, 1.0, 1e-3, seed=7, dt_max=20.0, max_step=0.1)
            d_lib = torch.zeros((4 * n_rep, 4 + 3 * n_at), device="cuda"); d_n = torch.zeros(1, dtype=torch.int32, device="cuda")
            d_work = torch.empty(api.gridff_hopping_work_bytes(mol, n_rep), dtype=torch.uint8, device="cuda")
            a.record(stream); st = api.gridff_minima_hopping(g, mol, hop, d_pos, d_lib, d_n, d_work=d_work); b.record(stream); b.synchronize()
            st = st.cpu().numpy()
            units = n_rep * cycles                       # hops
            extra = {"cycles": cycles, "md_steps": 1000, "relax_cap": 5000, "stats_per_cycle[candidates,new,dropped,library]": st.tolist()}
        else:
            n_scan = 40 if args.mode == "drag" else 20
            sdx = (0.1, 0.0, 0.0) if args.mode == "drag" else (0.0, 0.0, 0.1)
            integ = api.make_integrator("fire", 2000, 1.0, f_tol=2e-3, dt_max=10.0, max_step=0.05, n_scan=n_scan, fixed=(n_at - 1,), scan_dx=sdx)
            a.record(stream); out = api.gridff_run_scan(g, mol, integ, d_pos, d_vel); b.record(stream); b.synchronize()
            units = int(out["status"][:, 0].sum().item())        # FIRE iterations really taken
            extra = {"n_scan": n_scan, "points_converged_frac": float(out["scan"][..., 2].mean().item()), "scan_points_per_s": None}
            if args.mode == "drag":
                e_s = out["scan"][..., 0].mean(dim=0).cpu().numpy()
                extra.update(substrate_atoms=int(len(sub["pos"])), removed_sites=removed.tolist(),
                             mean_E_along_path_eV=[round(float(v), 4) for v in e_s[::4]])
        if it >= max(args.warmup, 3):
            ts.append(a.elapsed_time(b))
    ms = float(np.mean(ts))
    if args.mode in ("scan", "drag"):
        extra["scan_points_per_s"] = n_rep * extra["n_scan"] / (ms * 1e-3)
    unit = {"langevin": "replica-steps/s", "hopping": "hops/s", "scan": "replica-steps/s", "drag": "replica-steps/s"}[args.mode]
    print(json.dumps({"metric": {"langevin": "replica_md_steps_per_s", "hopping": "minima_hops_per_s", "scan": "replica_md_steps_per_s", "drag": "replica_md_steps_per_s"}[args.mode],
                      "value": units / (ms * 1e-3), "unit": unit, "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": "%s [mode %s]" % (name, args.mode), "n_replicas_per_gpu": n_rep, "atoms": n_at, "l2_flush_between_steps": True},
                      "gpu_launches": int(api.gridff_launch_count() - l0), "details": extra}))


def run_gridff(args, emit=True):
    """one JSON line for a replica config (emit) or the same dict returned (the 'also' entries of the default run)"""
    import torch
    import torch.distributed as dist
    from paper_2508_15522_b200 import api, shard     # api raises if the CUDA library is missing: there is no fallback

    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg, md, dims, name = workload(args)
    # replicas only: every rank runs its own batch of the same size with its own seed; no data-path collective
    if world > 1:
        cfg["pos"] = inputs.place_replicas(cfg["topo"], cfg["n_rep"], cfg["desc"]["Lx"], cfg["desc"]["Ly"], 0.0, shard.rank_seed(cfg["seed"], rank, 10),
                                           twist=(args.config == 2))
    d, topo, sub = cfg["desc"], cfg["topo"], cfg["sub"]
    n_rep, n_at = cfg["n_rep"], int(topo["n_atoms"])
    desc = api.make_desc(d["Lx"], d["Ly"], d["z_ref"], d["z_lo"], d["z_hi"], d["spacing"], d["alpha"], d["channels"], r_cut=d["r_cut"], l2_persist=1)
    kind = cfg["integ"]["kind"]
    restart = int(cfg["integ"].get("restart", 0))
    ikw = dict(f_tol=cfg["integ"].get("f_tol", 1e-3), variant=args.variant)
    if restart:          # config 2: relax, record the minimum, re-seed from Philox (R13, R17); dt_max / max_step as in the parity test
        ikw.update(restart=1, seed=shard.rank_seed(cfg["integ"]["seed"], rank), dt_max=20.0, max_step=0.1)
    integ = api.make_integrator(kind, md, cfg["integ"]["dt"], **ikw)
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(d["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    sub_pos = np.ascontiguousarray(sub["pos"], np.float64); sub_e = np.ascontiguousarray(sub["e"], np.float64)
    sub_R = np.ascontiguousarray(sub["R"], np.float64); sub_q = np.ascontiguousarray(sub["q"], np.float64)
    sb, wb = api.gridff_grid_bytes(desc, len(sub_pos))
    store = torch.empty(sb, dtype=torch.uint8, device="cuda"); scratch = torch.empty(wb, dtype=torch.uint8, device="cuda")
    pos0 = torch.from_numpy(cfg["pos"]).cuda(); vel0 = torch.from_numpy(cfg["vel"]).cuda()
    d_pos, d_vel = torch.empty_like(pos0), torch.empty_like(vel0)
    d_energy = torch.empty((n_rep, 8), device="cuda"); d_status = torch.empty((n_rep, 2), dtype=torch.int32, device="cuda")
    d_fire = torch.zeros((n_rep, 4), device="cuda")
    minima_cap = 8 * n_rep if restart else 0
    d_minima = torch.zeros((minima_cap, 4 + 3 * n_at), device="cuda") if restart else None
    d_n_minima = torch.zeros(1, dtype=torch.int32, device="cuda") if restart else None
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")          # > 126 MB L2
    stream = torch.cuda.current_stream()
    sptr = C.c_void_p(stream.cuda_stream)

    def build():
        out = C.c_void_p(None)
        api._check(api._lib.gridff_build_grid(C.byref(desc), len(sub_pos), sub_pos.ctypes.data, sub_e.ctypes.data, sub_R.ctypes.data, sub_q.ctypes.data,
                                              store.data_ptr(), sb, scratch.data_ptr(), wb, sptr, C.byref(out)))
        return api.Grid(out, desc, store)

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def one_step():
        """-> (ms whole step, ms of the fused replica kernel alone)"""
        d_pos.copy_(pos0); d_vel.copy_(vel0); d_fire.zero_()
        if restart:
            d_n_minima.zero_()
        flush.fill_(1)                                    # L2 flush between timed iterations
        e0, e1, e2 = ev(), ev(), ev()
        e0.record(stream)
        g = build()
        e1.record(stream)
        api.gridff_run_replicas(g, mol, integ, d_pos, d_vel, d_fire=d_fire, d_energy=d_energy, d_status=d_status, d_minima=d_minima, d_n_minima=d_n_minima)
        e2.record(stream)
        e2.synchronize()
        return e0.elapsed_time(e2), e1.elapsed_time(e2), g

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        one_step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = api.gridff_launch_count()
    t_step, t_kern = [], []
    for _ in range(args.steps):
        a, b, grid = one_step()
        t_step.append(a); t_kern.append(b)
    barrier()
    launches = api.gridff_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    total_ms = shard.max_over_ranks(float(np.sum(t_step)), "cuda")
    ms_per_step = total_ms / args.steps
    # units one step processed on this rank: VV runs md steps per replica; FIRE counts the steps really taken (converged replicas stop)
    units = n_rep * md if kind == "vv" else int(d_status[:, 0].sum().item())
    units_all = float(shard.sum_over_ranks(np.array([float(units)]), "cuda")[0])
    value = units_all / (ms_per_step * 1e-3)
    sampling = None
    if restart:
        nm = int(d_n_minima.item())
        e_min = d_minima[:min(nm, minima_cap), 3].cpu().numpy()
        nm_all = float(shard.sum_over_ranks(np.array([float(nm)]), "cuda")[0])
        lo = float(np.floor(e_min.min() * 10) / 10) if len(e_min) else 0.0
        lo = -shard.max_over_ranks(-lo, "cuda"); hi = lo + 4.0
        hist = shard.sum_over_ranks(shard.basin_histogram(e_min, lo, hi, 0.01), "cuda")
        nzb = np.nonzero(hist)[0]
        sampling = {"relaxed_configs_per_s": nm_all / (ms_per_step * 1e-3), "minima_per_step": nm_all, "minima_cap_per_gpu": minima_cap,
                    "basin_energy_histogram": {"bin_eV": 0.01, "e_lo_eV": lo, "first_bin": int(nzb[0]) if len(nzb) else 0,
                                               "counts": hist[nzb[0]:nzb[-1] + 1].tolist() if len(nzb) else []}}
    assert bool(torch.isfinite(d_pos).all()), "non-finite positions after the timed run"

    # ---- end to end through the public host-buffer API: pinned host inputs -> device -> pinned host results, every step
    hp = torch.from_numpy(cfg["pos"]).pin_memory(); hv = torch.from_numpy(cfg["vel"]).pin_memory()
    hp_w, hv_w = torch.empty_like(hp).pin_memory(), torch.empty_like(hv).pin_memory()
    he = torch.empty((n_rep, 8)).pin_memory(); hs = torch.empty((n_rep, 2), dtype=torch.int32).pin_memory()
    d_work = torch.empty(api.gridff_run_work_bytes(mol, n_rep), dtype=torch.uint8, device="cuda")
    e2e_ms = []
    for it in range(2 + args.steps):
        hp_w.copy_(hp); hv_w.copy_(hv)
        flush.fill_(1); torch.cuda.synchronize()
        t0 = time.perf_counter()
        g = build()                                          # substrate arrays are host inputs of the C-ABI call
        api.gridff_run_replicas_host(g, mol, integ, hp_w, hv_w, h_energy=he, h_status=hs, d_work=d_work)    # synchronises
        dt_ms = (time.perf_counter() - t0) * 1e3
        if it >= 2:
            e2e_ms.append(dt_ms)
    e2e_total = shard.max_over_ranks(float(np.sum(e2e_ms)), "cuda")
    e2e_units = n_rep * md if kind == "vv" else int(hs[:, 0].sum().item())
    e2e_value = float(shard.sum_over_ranks(np.array([float(e2e_units)]), "cuda")[0]) / (e2e_total / args.steps * 1e-3)
    h2d = 2 * n_rep * n_at * 12 + sub_pos.nbytes + sub_e.nbytes + sub_R.nbytes + sub_q.nbytes
    d2h = 2 * n_rep * n_at * 12 + n_rep * 32 + n_rep * 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the fused replica kernel): algorithmic gather bytes / measured duration
    # force evaluations per launch: VV = initial + per step + final energy pass; FIRE = one per step taken + final energy pass
    evals_per_launch = float(n_rep) * n_at * (md + 2) if kind == "vv" else float(units + n_rep) * n_at
    bytes_per_launch = evals_per_launch * BYTES_PER_EVAL
    kern_ms = float(np.mean(t_kern))
    achieved = bytes_per_launch / (kern_ms * 1e-3) / 1e9
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0)); hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6.65 TB/s (B200_PROFILING.md)"
    # L2 read bandwidth measured live with the library's probe over a buffer the size of the coefficient store (stays in L2)
    probe = torch.empty(min(max(sb, 16 << 20), 96 << 20), dtype=torch.uint8, device="cuda"); probe.fill_(1)
    l2 = {}
    for mode, key in ((0, "stream"), (1, "rows64"), (2, "lines128")):
        api.gridff_probe_read(probe, iters=100, mode=mode); torch.cuda.synchronize()        # warm: clocks up, buffer in L2
        best = 0.0
        for _ in range(10):
            a, b = ev(), ev()
            a.record(stream); api.gridff_probe_read(probe, iters=100, mode=mode); b.record(stream); b.synchronize()
            best = max(best, probe.numel() * 100 / (a.elapsed_time(b) * 1e-3) / 1e9)
        l2[key] = best
    store_fits_l2 = sb < (100 << 20)
    bound = "l2" if store_fits_l2 else "hbm"
    peak = l2["stream"] if store_fits_l2 else hbm_peak
    traffic = None
    try:
        traffic = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get("config%d" % args.config)
    except Exception:
        pass
    roofline = {"bound": bound, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "kernel": "k_replicas (fused grid + intramolecular + integrator)", "kernel_ms": kern_ms, "kernel_share_of_step": kern_ms / ms_per_step,
                "bytes_per_eval": BYTES_PER_EVAL, "evals_per_launch": evals_per_launch,
                "peak_source": ("L2 read bandwidth measured in this run by gridff_probe_read (coalesced 16 B loads over a %d MB buffer)" % (probe.numel() >> 20))
                if store_fits_l2 else hbm_src,
                "l2_probe_gbs": l2, "hbm_peak_gbs": hbm_peak, "frac_of_hbm_peak": achieved / hbm_peak,
                "achieved_is": "ALGORITHMIC gather bytes (64 nodes x 16 B per atom-grid evaluation) / kernel time — north_star's gather roofline, not a "
                               "measured L2 transfer rate: the kernel keeps each atom's folded stencil in shared memory and re-gathers it only when the atom "
                               "changes cell, so the bytes that really cross L2 -> L1 are a small fraction ('ncu' below)",
                "bound_definition": "north_star's gather roofline: algorithmic stencil bytes over the measured L2 read bandwidth when the store fits "
                                    "the L2 ('l2'), over the measured HBM bandwidth otherwise ('hbm'); frac_of_hbm_peak is always given as well",
                "ncu": ncu_facts("config%d" % args.config)}

    cpu = None
    if not args.no_cpu_baseline:
        tb, tps, cores, n, ss = oracle_sample(cfg, md)
        tot = units
        cpu = {"value": n * ss / (tb + n * ss * tps), "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "MEASURED on the sample: the whole fp64 grid build (a1-a3, %.1f s) + %d replicas x %d steps (a5-a9, %.3g s per replica-step) of the "
                         "%d x %d workload; value = those replica-steps / that time" % (tb, n, ss, tps, n_rep, md),
               "extrapolated_full_workload": tot / (tb + tot * tps), "replica_steps_per_s_run_only": 1.0 / tps}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": name, "grid": list(dims), "channels": len(d["channels"]), "store_bytes": sb, "n_replicas_per_gpu": n_rep,
                   "md_steps_per_step": md, "atoms": n_at, "integrator": kind, "variant": args.variant, "parallelism": "replicas only (no collective)",
                   "l2_flush_between_steps": True, "step": "gridff_build_grid + gridff_run_replicas"},
        "atom_grid_evals_per_s": value * n_at, "kernel_only_replica_steps_per_s": units / (kern_ms * 1e-3), "sampling": sampling,
        "ms_build_grid": ms_per_step - kern_ms,
        "clocks": clocks, "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    if not emit:
        return line
    if world == 1 and args.config == 1 and not args.no_also and not args.md_steps and not args.replicas:
        torch.cuda.empty_cache()
        line["also"] = also_entries(args)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def also_entries(args):
    """The second half of BASELINE.json's metric ("atom-grid evals/s AND replica MD steps/s") and the other replica configs, measured briefly
    (2 timed steps after 3 warm-ups each, device-timed, L2 flushed) after the main timed region of the default run, so that the driver's record
    of `python bench.py` carries them: config 2 (60-atom FIRE + restart), config 3 (384 MB grid), config 4 on the config-1 grid and on the
    512 x 512 x 256 sweep grid (1.09 GB: the HBM-bound gather), random and Morton-sorted points."""
    import argparse
    out = {}
    base = dict(vars(args), steps=2, warmup=3, no_cpu_baseline=True, no_also=True, md_steps=0, replicas=0, variant=0, mode="run")
    todo = [("config2", dict(config=2)), ("config3", dict(config=3)),
            ("config4_random", dict(config=4, order="random", c4_grid="config1", log2_points=26)),
            ("config4_sorted", dict(config=4, order="sorted", c4_grid="config1", log2_points=26)),
            ("config4_hbm_512x512x256_random", dict(config=4, order="random", c4_grid="512x512x256", log2_points=25)),
            ("config4_hbm_512x512x256_sorted", dict(config=4, order="sorted", c4_grid="512x512x256", log2_points=25)),
            ("config4_hbm_512x512x256_random_bricks8", dict(config=4, order="random", c4_grid="512x512x256", log2_points=25, c4_store="bricks8")),
            ("config4_hbm_512x512x256_random_binned", dict(config=4, order="random", c4_grid="512x512x256", log2_points=25, binned=True))]
    for key, kw in todo:
        a = argparse.Namespace(**dict(dict(base, c4_store="fp32", sweep=False, binned=False), **kw))
        t0 = time.perf_counter()
        try:
            r = run_eval(a, emit=False) if a.config == 4 else run_gridff(a, emit=False)
            rf = r["roofline"]
            out[key] = {"metric": r["metric"], "value": r["value"], "unit": r["unit"], "ms_per_step": r["ms_per_step"], "kernel_ms": rf["kernel_ms"],
                        "roofline": {k: rf[k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic")}, "e2e": r["e2e"],
                        "workload": r["config"]["workload"], "gpu_launches": r["gpu_launches"], "wall_s": None}
            if r.get("sampling"):
                out[key]["relaxed_configs_per_s"] = r["sampling"]["relaxed_configs_per_s"]
            if "ms_build_grid" in r:
                out[key]["ms_build_grid"] = r["ms_build_grid"]; out[key]["kernel_only_replica_steps_per_s"] = r["kernel_only_replica_steps_per_s"]
        except Exception as e:                      # an extra must never cost the main line
            out[key] = {"error": repr(e)[:300]}
        out[key]["wall_s"] = round(time.perf_counter() - t0, 1)
    return out


# ------------------------------------------------------------------------------------------------------------------ config 4
# Bare interpolation microbenchmark (BASELINE.json configs[4]): 2^26 uniformly random points in the config-1 grid volume, 3-channel E
# and analytic gradient per point; optional sweep over grid sizes 32^3 ... 512 x 512 x 256, random vs Morton-sorted point order.

C4_METRIC, C4_UNIT = "atom_grid_evals_per_s", "evals/s"
C4_SWEEP = [(32, 32, 32), (64, 64, 64), (128, 128, 128), (256, 256, 256), (512, 512, 256)]
C4_IO_BYTES = 12 + 16 + 4 + 12            # pos + coef in, E + F out per point (streamed through HBM whatever the grid size)


def c4_grid_spec(args):
    """-> (name, dims, desc dict, substrate or None)"""
    if args.c4_grid == "config1":
        cfg = inputs.config(1, n_rep=1)
        return "config1 grid (NaCl(001) 4x4 slab, Pauli + London + Coulomb)", inputs.grid_dims(cfg["desc"]), cfg["desc"], cfg["sub"]
    nx, ny, nz = (int(v) for v in args.c4_grid.lower().split("x"))
    return "synthetic %dx%dx%d" % (nx, ny, nz), (nx, ny, nz), c4_synth_desc(nx, ny, nz), None


def c4_synth_desc(nx, ny, nz, h=0.1):
    return inputs.grid_desc(nx * h, ny * h, 0.0, 1.5, 1.5 + nz * h, h, 1.6, [inputs.PAULI, inputs.LONDON, inputs.COULOMB])


def c4_valid_z(desc, nz):
    z0 = desc["z_ref"] + desc["z_lo"]
    return z0 + desc["spacing"], z0 + (nz - 2) * desc["spacing"] - 1e-3          # DESIGN.md R5


def run_eval_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import gridff_oracle as orc
    name, dims, d, sub = c4_grid_spec(args)
    nx, ny, nz = dims; z0 = d["z_ref"] + d["z_lo"]
    if sub is not None:
        samples = orc.sample_grid(sub, d["alpha"], d["Lx"], d["Ly"], d["r_cut"], nx, ny, nz, z0, d["spacing"], d["channels"])
    else:
        samples = inputs.c4_samples(nx, ny, nz).astype(np.float64)
    og = orc.OracleGrid(orc.prefilter(samples, (1, 1, 0)), d["Lx"], d["Ly"], z0, d["spacing"])
    n_s = 1 << 22
    zl, zh = c4_valid_z(d, nz)
    pos, coef = inputs.c4_points(n_s, d["Lx"], d["Ly"], zl, zh)
    ts = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter(); orc.interp(og, pos, coef); t = time.perf_counter() - t0
        if it >= args.warmup:
            ts.append(t)
    val = n_s / float(np.mean(ts)); n = 1 << args.log2_points
    sample = "2^22 of the 2^%d points per step (grid resident, fp64 coefficients)" % args.log2_points
    print(json.dumps({
        "impl": "reference", "metric": C4_METRIC, "value": val, "unit": C4_UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": n / val * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config4: 2^%d random points, %s" % (args.log2_points, name), "grid": list(dims), "order": "random"},
        "cpu_baseline": {"value": val, "unit": C4_UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": C4_UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


def run_eval(args, emit=True):
    import torch
    import torch.distributed as dist
    from paper_2508_15522_b200 import api, shard

    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0)); hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6.65 TB/s (B200_PROFILING.md)"

    def make_grid(desc, dims, sub, store="fp32"):
        g0 = make_grid_fp32(desc, dims, sub)
        if store == "fp32":
            return g0
        gd_ = api.gridff_grid_derive(g0, {"half": api.LAYOUT_HALF, "trilinear": api.LAYOUT_TRILINEAR, "bricks": api.LAYOUT_MBRICK,
                                          "bricks2": api.LAYOUT_MBRICK2, "bricks8": api.LAYOUT_MBRICK8}[store])
        torch.cuda.synchronize()
        g0.free()
        return gd_

    def make_grid_fp32(desc, dims, sub):
        gd = api.make_desc(desc["Lx"], desc["Ly"], desc["z_ref"], desc["z_lo"], desc["z_hi"], desc["spacing"], desc["alpha"], desc["channels"],
                           r_cut=desc["r_cut"], l2_persist=1)
        if sub is not None:
            return api.gridff_build_grid(gd, sub["pos"], sub["e"], sub["R"], sub["q"])
        smp = inputs.c4_samples(*dims, xp=torch, device="cuda")
        g = api.gridff_grid_from_samples(gd, smp)
        del smp
        return g

    def make_points(desc, dims, n, seed):
        zl, zh = c4_valid_z(desc, dims[2])
        pos, coef = inputs.c4_points(n, desc["Lx"], desc["Ly"], zl, zh, seed=seed)
        return pos, coef

    def l2_probe(nbytes):
        probe = torch.empty(min(max(nbytes, 16 << 20), 96 << 20), dtype=torch.uint8, device="cuda"); probe.fill_(1)     # >= 16 MB: a smaller buffer cannot occupy every SM
        out = {}
        for mode, key in ((0, "stream"), (1, "rows64"), (2, "lines128")):
            api.gridff_probe_read(probe, iters=100, mode=mode); torch.cuda.synchronize()    # warm: clocks up, buffer in L2
            best = 0.0
            for _ in range(10):
                a, b = ev(), ev()
                a.record(stream); api.gridff_probe_read(probe, iters=100, mode=mode); b.record(stream); b.synchronize()
                best = max(best, probe.numel() * 100 / (a.elapsed_time(b) * 1e-3) / 1e9)
            out[key] = best
        return out

    binned_work = {}

    def time_eval(g, d_pos, d_coef, d_E, d_F, reps, warm):
        ts = []
        binned = getattr(args, "binned", False) and args.c4_store == "fp32"
        if binned and "w" not in binned_work:
            binned_work["w"] = torch.empty(int(api._lib.gridff_eval_binned_work_bytes(g.handle, d_pos.shape[0])), dtype=torch.uint8, device="cuda")
        for it in range(warm + reps):
            flush.fill_(1)
            a, b = ev(), ev()
            a.record(stream)
            if binned:
                api.gridff_eval_binned(g, d_pos, d_coef, d_E=d_E, d_F=d_F, d_work=binned_work["w"])
            else:
                api.gridff_eval(g, d_pos, d_coef, d_E=d_E, d_F=d_F, variant=args.variant or None)
            b.record(stream); b.synchronize()
            if it >= warm:
                ts.append(a.elapsed_time(b))
        return ts

    name, dims, desc, sub = c4_grid_spec(args)
    n = 1 << args.log2_points
    g = make_grid(desc, dims, sub, args.c4_store)
    sb = g.store.numel()
    bpe = 512 if args.c4_store in ("half", "trilinear") else BYTES_PER_EVAL          # half: 64 nodes x 8 B; trilinear foil: 8 nodes x 64 B
    pos, coef = make_points(desc, dims, n, shard.rank_seed(1004, rank))
    d_pos, d_coef = torch.from_numpy(pos).cuda(), torch.from_numpy(coef).cuda()
    z0 = desc["z_ref"] + desc["z_lo"]
    if args.order == "sorted":
        perm = inputs.morton_order(d_pos, desc["Lx"], desc["Ly"], z0, dims[0], dims[1], desc["spacing"], xp=torch)
        d_pos, d_coef = d_pos[perm].contiguous(), d_coef[perm].contiguous()
        pos, coef = d_pos.cpu().numpy(), d_coef.cpu().numpy()
        del perm
    d_E = torch.empty(n, device="cuda"); d_F = torch.empty((n, 3), device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    time_eval(g, d_pos, d_coef, d_E, d_F, 0, max(args.warmup, 3))
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = api.gridff_launch_count()
    ts = time_eval(g, d_pos, d_coef, d_E, d_F, args.steps, 0)
    barrier()
    launches = api.gridff_launch_count() - l0
    clocks = sampler.stop() if sampler else None
    total_ms = shard.max_over_ranks(float(np.sum(ts)), "cuda")
    ms_per_step = total_ms / args.steps
    value = world * n / (ms_per_step * 1e-3)
    assert bool(torch.isfinite(d_E).all()), "non-finite energies after the timed run"

    # ---- end to end: pinned host points -> device -> pinned host E, F through gridff_eval_host, every step
    hp, hc = torch.from_numpy(pos).pin_memory(), torch.from_numpy(coef).pin_memory()
    hE, hF = torch.empty(n).pin_memory(), torch.empty((n, 3)).pin_memory()
    d_work = torch.empty(api.gridff_eval_work_bytes(n), dtype=torch.uint8, device="cuda")
    e2e_ms = []
    for it in range(2 + args.steps):
        flush.fill_(1); torch.cuda.synchronize()
        t0 = time.perf_counter()
        api.gridff_eval_host(g, hp, hc, hE, hF, d_work=d_work)           # synchronises
        if it >= 2:
            e2e_ms.append((time.perf_counter() - t0) * 1e3)
    e2e_total = shard.max_over_ranks(float(np.sum(e2e_ms)), "cuda")
    e2e_value = world * n / (e2e_total / args.steps * 1e-3)
    assert float((hE - d_E.cpu()).abs().max()) == 0.0, "host path and device path disagree"
    del hp, hc, hE, hF, d_work

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    def roof(store_bytes, n_pts, ms, l2, bytes_per_eval=None):
        fits = store_bytes < (100 << 20)
        ach = n_pts * float(bytes_per_eval or bpe) / (ms * 1e-3) / 1e9
        peak = l2["stream"] if fits else hbm_peak
        return fits, ach, peak

    l2 = l2_probe(sb)
    kern_ms = float(np.mean(ts))
    tkey = "config4" if args.c4_grid == "config1" else "config4_%s" % args.c4_grid.lower()
    if args.order == "sorted":
        tkey += "_sorted"
    if args.c4_store != "fp32":
        tkey += "_" + args.c4_store
    if getattr(args, "binned", False):
        tkey += "_binned"
    fits, ach, peak = roof(sb, n, kern_ms, l2)
    traffic = None
    try:
        traffic = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(tkey)
    except Exception:
        pass
    roofline = {"bound": "l2" if fits else "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": traffic,
                "kernel": {"fp32": "k_eval_coop (warp-cooperative LDG gather)" if fits or args.variant == 2 else
                                   "k_eval_tma (one 3-D TMA box per point) for scattered points / k_eval_coop for sorted points, chosen on the device", "half": "k_eval_half (tricubic, fp16 coefficients)",
                           "trilinear": "k_eval_trilinear (8-corner foil, E and F tables)",
                           "bricks": "k_eval_bricks (warp-cooperative LDG gather over 2x2x2-node bricks)", "bricks2": "k_eval_bricks (2 shifted copies)",
                           "bricks8": "k_eval_tma<bricks> (one 5-D TMA box = 8 whole 128-byte lines per point; 8 shifted copies)"}[args.c4_store], "kernel_ms": kern_ms, "kernel_share_of_step": kern_ms / ms_per_step,
                "bytes_per_eval": bpe, "evals_per_launch": n, "io_bytes_per_eval_hbm": C4_IO_BYTES,
                "io_stream_gbs": n * float(C4_IO_BYTES) / (kern_ms * 1e-3) / 1e9,
                "peak_source": "L2 read bandwidth measured in this run by gridff_probe_read" if fits else hbm_src,
                "l2_probe_gbs": l2, "hbm_peak_gbs": hbm_peak, "frac_of_hbm_peak": ach / hbm_peak, "ncu": ncu_facts(tkey)}

    sweep = None
    if args.sweep:
        sweep = []
        del d_pos, d_coef
        specs = [("config1", dims, desc, sub)] + [("%dx%dx%d" % s_, s_, c4_synth_desc(*s_), None) for s_ in C4_SWEEP]
        for gname, gdims, gdesc, gsub in specs:
            p_, c_ = make_points(gdesc, gdims, n, 1004)
            dp0, dc0 = torch.from_numpy(p_).cuda(), torch.from_numpy(c_).cuda()
            perm = inputs.morton_order(dp0, gdesc["Lx"], gdesc["Ly"], gdesc["z_ref"] + gdesc["z_lo"], gdims[0], gdims[1], gdesc["spacing"], xp=torch)
            dp1, dc1 = dp0[perm].contiguous(), dc0[perm].contiguous()
            del perm, p_, c_
            for store in ("fp32", "half", "trilinear", "bricks", "bricks2", "bricks8"):
                gg = make_grid(gdesc, gdims, gsub, store)
                gsb = gg.store.numel()
                gl2 = l2_probe(gsb) if gsb < (100 << 20) else l2
                sbpe = 512 if store in ("half", "trilinear") else BYTES_PER_EVAL
                for order, dp, dc in (("random", dp0, dc0), ("sorted", dp1, dc1)):
                    t = float(np.mean(time_eval(gg, dp, dc, d_E, d_F, 3, 2)))
                    f_, a_, pk = roof(gsb, n, t, gl2, sbpe)
                    sweep.append({"grid": gname, "store": store, "store_MB": round(gsb / 1e6, 1), "order": order, "ms": t, "evals_per_s": n / (t * 1e-3),
                                  "bytes_per_eval": sbpe, "gather_GBs": a_, "bound": "l2" if f_ else "hbm", "peak_GBs": pk, "frac": a_ / pk})
                    sys.stderr.write("sweep %-12s %-9s %7.1f MB %-6s %8.3f ms  %.3e evals/s  %8.1f GB/s  %.3f of %s\n"
                                     % (gname, store, gsb / 1e6, order, t, n / (t * 1e-3), a_, a_ / pk, "l2" if f_ else "hbm"))
                gg.free(); del gg
            del dp0, dc0, dp1, dc1

    cpu = None
    if not args.no_cpu_baseline:
        from oracle import gridff_oracle as orc
        nx, ny, nz = dims
        if sub is not None:
            samples = orc.sample_grid(sub, desc["alpha"], desc["Lx"], desc["Ly"], desc["r_cut"], nx, ny, nz, z0, desc["spacing"], desc["channels"])
        else:
            samples = inputs.c4_samples(nx, ny, nz).astype(np.float64)
        og = orc.OracleGrid(orc.prefilter(samples, (1, 1, 0)), desc["Lx"], desc["Ly"], z0, desc["spacing"])
        n_s = min(n, 1 << 22)
        orc.interp(og, pos[:1 << 16], coef[:1 << 16])
        t0 = time.perf_counter(); orc.interp(og, pos[:n_s], coef[:n_s]); t = time.perf_counter() - t0
        cpu = {"value": n_s / t, "unit": C4_UNIT, "cores": orc.num_threads(), "kind": "oracle",
               "sample": "the first 2^%d of the 2^%d points (%.2f s), grid resident, fp64" % (int(np.log2(n_s)), args.log2_points, t)}

    line = ({
        "metric": C4_METRIC, "value": value, "unit": C4_UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "config4: 2^%d uniformly random points, %s, 3-channel E + analytic gradient" % (args.log2_points, name),
                   "grid": list(dims), "store": args.c4_store, "binned": bool(getattr(args, "binned", False)), "store_bytes": sb, "points_per_gpu": n, "order": args.order, "parallelism": "points only (no collective)",
                   "l2_flush_between_steps": True, "step": "gridff_eval over all points (grid built before the timed region)"},
        "clocks": clocks, "e2e": {"value": e2e_value, "unit": C4_UNIT, "h2d_bytes_per_step": n * 28, "d2h_bytes_per_step": n * 16},
        "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "sweep": sweep})
    if not emit:
        return line
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_eval_reference(a) if a.config == 4 else run_reference(a)
    else:
        if a.mode != "run" and a.config != 4:
            run_f_rows(a)
        else:
            run_eval(a) if a.config == 4 else run_gridff(a)
