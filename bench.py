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
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 3])
    ap.add_argument("--md-steps", type=int, default=0, help="override the config's MD steps per launch (0 = config value)")
    ap.add_argument("--replicas", type=int, default=0, help="override the config's replica count (0 = config value)")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def workload(args):
    cfg = inputs.config(args.config, n_rep=args.replicas or None)
    md = args.md_steps or cfg["integ"]["n_steps"]
    nx, ny, nz = inputs.grid_dims(cfg["desc"])
    name = {0: "config0: 64 x benzene FIRE", 1: "config1: NaCl(001) 4x4 slab + Coulomb, 4096 x 30-atom aromatic, VV dt 0.5 fs x 10000",
            3: "config3: 40x40 Å slab, 400x400x150x4 grid (384 MB), 8192 x 30-atom aromatic, VV x 5000"}[args.config]
    return cfg, md, (nx, ny, nz), name


# ------------------------------------------------------------------------------------------------------------------ oracle arm

def oracle_sample(cfg, md_steps, n_rep_sample=64, steps_sample=200):
    """Times the fp64 oracle, as it stands, on a bounded sample: the whole grid build (a1-a3) + n_rep_sample replicas x
    steps_sample steps (a5-a9).  Returns (t_build, t_per_replica_step, cores)."""
    from oracle import gridff_oracle as orc
    d = cfg["desc"]; nx, ny, nz = inputs.grid_dims(d); z0 = d["z_ref"] + d["z_lo"]
    t0 = time.perf_counter()
    samples = orc.sample_grid(cfg["sub"], d["alpha"], d["Lx"], d["Ly"], d["r_cut"], nx, ny, nz, z0, d["spacing"], d["channels"])
    og = orc.OracleGrid(orc.prefilter(samples, (1, 1, 0)), d["Lx"], d["Ly"], z0, d["spacing"])
    t_build = time.perf_counter() - t0
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
    times = []
    for it in range(args.warmup + args.steps):
        tb, tps, cores, n, ss = oracle_sample(cfg, md)
        if it >= args.warmup:
            times.append(tb + total * tps)           # whole-workload time extrapolated from the sample
    t = float(np.mean(times))
    val = total / t
    sample = "full grid build (a1-a3) + %d replicas x %d steps, extrapolated to %d x %d" % (n, ss, cfg["n_rep"], md)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "grid": list(dims), "n_replicas": cfg["n_rep"], "md_steps_per_step": md, "atoms": int(cfg["topo"]["n_atoms"])},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------------------------ GPU arm

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


def run_gridff(args):
    import torch
    import torch.distributed as dist
    from paper_2508_15522_b200 import api            # raises if the CUDA library is missing: there is no fallback

    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg, md, dims, name = workload(args)
    # replicas only: every rank runs its own batch of the same size with its own seed; no data-path collective
    if world > 1:
        cfg["pos"] = inputs.place_replicas(cfg["topo"], cfg["n_rep"], cfg["desc"]["Lx"], cfg["desc"]["Ly"], 0.0, cfg["seed"] + 10 + 1000 * rank)
    d, topo, sub = cfg["desc"], cfg["topo"], cfg["sub"]
    n_rep, n_at = cfg["n_rep"], int(topo["n_atoms"])
    desc = api.make_desc(d["Lx"], d["Ly"], d["z_ref"], d["z_lo"], d["z_hi"], d["spacing"], d["alpha"], d["channels"], r_cut=d["r_cut"], l2_persist=1)
    kind = cfg["integ"]["kind"]
    integ = api.make_integrator(kind, md, cfg["integ"]["dt"], f_tol=cfg["integ"].get("f_tol", 1e-3), variant=args.variant)
    mol = api.gridff_create_molecule(topo, api.gridff_atom_coefs(d["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))
    sub_pos = np.ascontiguousarray(sub["pos"], np.float64); sub_e = np.ascontiguousarray(sub["e"], np.float64)
    sub_R = np.ascontiguousarray(sub["R"], np.float64); sub_q = np.ascontiguousarray(sub["q"], np.float64)
    sb, wb = api.gridff_grid_bytes(desc, len(sub_pos))
    store = torch.empty(sb, dtype=torch.uint8, device="cuda"); scratch = torch.empty(wb, dtype=torch.uint8, device="cuda")
    pos0 = torch.from_numpy(cfg["pos"]).cuda(); vel0 = torch.from_numpy(cfg["vel"]).cuda()
    d_pos, d_vel = torch.empty_like(pos0), torch.empty_like(vel0)
    d_energy = torch.empty((n_rep, 8), device="cuda"); d_status = torch.empty((n_rep, 2), dtype=torch.int32, device="cuda")
    d_fire = torch.zeros((n_rep, 4), device="cuda")
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
        flush.fill_(1)                                    # L2 flush between timed iterations
        e0, e1, e2 = ev(), ev(), ev()
        e0.record(stream)
        g = build()
        e1.record(stream)
        api.gridff_run_replicas(g, mol, integ, d_pos, d_vel, d_fire=d_fire, d_energy=d_energy, d_status=d_status)
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
    total_ms = float(np.sum(t_step))
    if world > 1:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    value = world * n_rep * md / (ms_per_step * 1e-3)
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
    e2e_total = float(np.sum(e2e_ms))
    if world > 1:
        t = torch.tensor([e2e_total], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_total = float(t.item())
    e2e_value = world * n_rep * md / (e2e_total / args.steps * 1e-3)
    h2d = 2 * n_rep * n_at * 12 + sub_pos.nbytes + sub_e.nbytes + sub_R.nbytes + sub_q.nbytes
    d2h = 2 * n_rep * n_at * 12 + n_rep * 32 + n_rep * 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the fused replica kernel): algorithmic gather bytes / measured duration
    force_evals = md + 2 if kind == "vv" else md + 1                     # initial + per step + final energy pass
    bytes_per_launch = float(n_rep) * n_at * force_evals * BYTES_PER_EVAL
    kern_ms = float(np.mean(t_kern))
    achieved = bytes_per_launch / (kern_ms * 1e-3) / 1e9
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0)); hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6.65 TB/s (B200_PROFILING.md)"
    # L2 read bandwidth measured live with the library's probe over a buffer the size of the coefficient store (stays in L2)
    probe = torch.empty(min(sb, 96 << 20), dtype=torch.uint8, device="cuda"); probe.fill_(1)
    l2 = {}
    for mode, key in ((0, "stream"), (1, "rows64")):
        api.gridff_probe_read(probe, iters=20, mode=mode); torch.cuda.synchronize()
        best = 0.0
        for _ in range(5):
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
                "bytes_per_eval": BYTES_PER_EVAL, "evals_per_launch": n_rep * n_at * force_evals,
                "peak_source": ("L2 read bandwidth measured in this run by gridff_probe_read (coalesced 16 B loads over a %d MB buffer)" % (probe.numel() >> 20))
                if store_fits_l2 else hbm_src,
                "l2_probe_gbs": l2, "hbm_peak_gbs": hbm_peak, "frac_of_hbm_peak": achieved / hbm_peak}

    cpu = None
    if not args.no_cpu_baseline:
        tb, tps, cores, n, ss = oracle_sample(cfg, md)
        tot = n_rep * md
        cpu = {"value": tot / (tb + tot * tps), "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "full fp64 grid build (a1-a3, %.1f s) + %d replicas x %d steps (%.3g s per replica-step), extrapolated to %d x %d" % (tb, n, ss, tps, n_rep, md),
               "replica_steps_per_s_run_only": 1.0 / tps}

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": name, "grid": list(dims), "channels": len(d["channels"]), "store_bytes": sb, "n_replicas_per_gpu": n_rep,
                   "md_steps_per_step": md, "atoms": n_at, "integrator": kind, "variant": args.variant, "parallelism": "replicas only (no collective)",
                   "l2_flush_between_steps": True, "step": "gridff_build_grid + gridff_run_replicas"},
        "atom_grid_evals_per_s": value * n_at,
        "ms_build_grid": ms_per_step - kern_ms,
        "clocks": clocks, "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_gridff(a)
