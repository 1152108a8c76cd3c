"""One small launch of EVERY kernel and kernel mode of libgridff.so, for compute-sanitizer:

    compute-sanitizer --tool memcheck  python tests/sanitize_kernels.py
    compute-sanitizer --tool racecheck python tests/sanitize_kernels.py
    compute-sanitizer --tool synccheck python tests/sanitize_kernels.py
    compute-sanitizer --tool initcheck python tests/sanitize_kernels.py

(On this GPU pool compute-sanitizer is closed — profiles/r2_sanitizers.md — so the script serves as the plain every-mode smoke run; the race
evidence is tests/test_gpu_stress.py.)
No oracle, no assertions on values (the parity tests do that): the point is that each code path runs under the tool, at sizes that keep
the 100-1000x slow-down of racecheck within minutes.  Modes reached (printed as they run):
  grid build        Morse per-node and tiled sampling (magnitude window on / off), Coulomb, prefilters, z-fastest and 4x4x4-brick stores,
                    gridff_grid_from_samples, export; derived stores: fp16, trilinear foil, micro-bricks x 1 / 2 / 8
  gridff_eval       variants 1 (thread per point), 2 (warp-cooperative LDG), 3 (3-D TMA box), the brick kernel, fp16, trilinear,
                    micro-brick LDG gather and 5-D TMA box, gridff_eval_binned (count / scan / scatter / gather-back); the device-side kernel choice (classify + both kernels) on a store declared > L2
                    is reached through the same kernels; host-buffer pipeline
  k_replicas        <= 32 atoms on one warp: velocity Verlet variants 1, 2, 3, time-multiplexed VV and Langevin (state handed between
                    warps through global memory across __syncthreads), FIRE, FIRE + Philox restart + minima records, driven scan with a
                    held atom; 33-64 atoms: pair of warps (named barrier, two-word exchanges) VV / FIRE + restart / Langevin / scan, with the
                    per-kind pair table and without (> 8 kinds), two atoms per lane (variants 1, 2, 4)
  minima hopping    Langevin -> FIRE -> k_hop_collect -> k_filter_library -> k_filter_append (one block walks the survivors), two cycles
  probes            k_probe_stream, k_probe_rows
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2508_15522_b200 import api, inputs  # noqa: E402


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def grid(cfg, layout=0, morse_window=0, z_hi=5.5):
    d = dict(cfg["desc"]); d["z_hi"] = z_hi
    desc = api.make_desc(d["Lx"], d["Ly"], d["z_ref"], d["z_lo"], d["z_hi"], d["spacing"], d["alpha"], d["channels"], r_cut=d["r_cut"], layout=layout,
                         morse_window=morse_window)
    s = cfg["sub"]
    return api.gridff_build_grid(desc, s["pos"], s["e"], s["R"], s["q"]), d


def molecule(cfg, topo=None):
    topo = topo or cfg["topo"]
    return api.gridff_create_molecule(topo, api.gridff_atom_coefs(cfg["desc"]["alpha"], topo["grid_e"], topo["grid_R"], topo["q"]))


def say(msg):
    torch.cuda.synchronize()
    print("ok  " + msg, flush=True)


def main():
    torch.cuda.set_device(0)
    c1 = inputs.config(1, n_rep=12, small=True, spacing=0.2)
    c3 = inputs.config(3, n_rep=4, small=True, spacing=0.2)
    c2 = inputs.config(2, n_rep=6, small=True, spacing=0.2)
    c0 = inputs.config(0, n_rep=5, small=True, spacing=0.2)

    # ---- a1-a4
    g1, d1 = grid(c1)
    for mw in (1, 2):
        g3, d3 = grid(c3, morse_window=mw)
    gb, _ = grid(c1, layout=1)
    g0, d0 = grid(c0)
    api.gridff_grid_export(g1); api.gridff_grid_export(gb)
    nx, ny, nz = inputs.grid_dims(d1)
    smp = inputs.c4_samples(nx, ny, nz, xp=torch, device="cuda")
    gs = api.gridff_grid_from_samples(api.make_desc(d1["Lx"], d1["Ly"], 0.0, 1.5, d1["z_hi"], d1["spacing"], 1.6, d1["channels"]), smp)
    say("grid build: Morse (window on / off), Coulomb, prefilters, z-fastest + brick stores, from_samples, export")
    derived = {name: api.gridff_grid_derive(g1, lay) for name, lay in (("half", api.LAYOUT_HALF), ("trilinear", api.LAYOUT_TRILINEAR),
               ("bricks", api.LAYOUT_MBRICK), ("bricks2", api.LAYOUT_MBRICK2), ("bricks8", api.LAYOUT_MBRICK8))}
    say("derived stores: fp16, trilinear, micro-bricks x 1 / 2 / 8")

    # ---- a5
    z0 = d1["z_ref"] + d1["z_lo"]
    for n in (1, 777, 4500):
        pos, cf = inputs.c4_points(n, d1["Lx"], d1["Ly"], z0 - 0.05, z0 + (nz - 2) * d1["spacing"] + 0.05)
        pos[::7, 0] += np.float32(3 * d1["Lx"]); pos[::5, 1] -= np.float32(2 * d1["Ly"])
        dp, dc = dev(pos), dev(cf)
        for v in (1, 2, 3, 0):
            api.gridff_eval(g1, dp, dc, variant=v)
        api.gridff_eval(gb, dp, dc)
        api.gridff_eval(gs, dp, dc)
        api.gridff_eval_binned(g1, dp, dc)
        api.gridff_eval_binned_noalloc(g1, dp, dc, torch.empty(n, device="cuda"), torch.empty((n, 3), device="cuda"))     # the same passes over the built-in scratch
        for name, gd in derived.items():
            for v in ((0, 2, 3) if name == "bricks8" else (0, 2) if name.startswith("bricks") else (0,)):
                api.gridff_eval(gd, dp, dc, variant=v)
        order = inputs.morton_order(dp, d1["Lx"], d1["Ly"], z0, nx, ny, d1["spacing"], xp=torch)        # clustered warps: the L1 path
        for gd in (g1, derived["bricks8"], derived["bricks"]):
            api.gridff_eval(gd, dp[order].contiguous(), dc[order].contiguous(), variant=3 if gd is not derived["bricks"] else 0)
    hE, hF = torch.empty(n).pin_memory(), torch.empty((n, 3)).pin_memory()
    api.gridff_eval_host(g1, torch.from_numpy(pos).pin_memory(), torch.from_numpy(cf).pin_memory(), hE, hF)
    say("gridff_eval: variants 1, 2, 3, brick, fp16, trilinear, micro-brick LDG + TMA, sorted points, host pipeline")

    # ---- a6-a9, <= 32 atoms
    m1 = molecule(c1)
    p1, v1 = c1["pos"], c1["vel"]
    for v in (1, 2, 3):
        api.gridff_run_replicas(g1, m1, api.make_integrator("vv", 20, 0.5, variant=v), dev(p1), dev(v1))
    say("k_replicas <= 32 atoms: velocity Verlet variants 1, 2, 3")
    # time-multiplexed: needs more replicas than resident slots (2 CTAs x 8 warps per SM) and >= 512 steps
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    n_mux = sms * 2 * 8 + 37
    cm = inputs.config(1, n_rep=n_mux, small=True, spacing=0.2)
    api.gridff_run_replicas(g1, m1, api.make_integrator("vv", 512, 0.5), dev(cm["pos"]), dev(cm["vel"]))
    api.gridff_run_replicas(g1, m1, api.make_integrator("langevin", 512, 0.5, temperature=300.0, gamma=0.01, seed=3), dev(cm["pos"]), dev(cm["vel"]))
    say("k_replicas time-multiplexed VV and Langevin (%d replicas x 512 steps)" % n_mux)
    api.gridff_run_replicas(g1, m1, api.make_integrator("langevin", 30, 0.5, temperature=300.0, gamma=0.01, seed=3, fixed=(0, 29)), dev(p1), dev(v1))
    for v in (1, 2, 3):
        api.gridff_run_replicas(g0, molecule(c0), api.make_integrator("fire", 60, 0.5, variant=v), dev(c0["pos"]), dev(c0["vel"]),
                                d_fire=torch.zeros((5, 4), device="cuda"))
    mn = torch.zeros((64, 4 + 3 * 30), device="cuda"); nmn = torch.zeros(1, dtype=torch.int32, device="cuda")
    api.gridff_run_replicas(g1, m1, api.make_integrator("fire", 300, 0.5, f_tol=0.5, restart=1, seed=5, dt_max=5.0, max_step=0.1),
                            dev(p1), torch.zeros_like(dev(v1)), d_fire=torch.zeros((12, 4), device="cuda"), d_minima=mn, d_n_minima=nmn)
    api.gridff_run_scan(g1, m1, api.make_integrator("fire", 40, 1.0, f_tol=0.05, dt_max=10.0, max_step=0.05, n_scan=3, fixed=(29,), scan_dx=(0.0, 0.0, 0.1)),
                        dev(p1), torch.zeros_like(dev(v1)))
    api.gridff_run_replicas(None, m1, api.make_integrator("vv", 10, 0.5), dev(p1), dev(v1))           # gas phase: no grid
    say("k_replicas <= 32 atoms: Langevin with held atoms, FIRE variants, FIRE + restart + minima, scan, gas phase (minima %d)" % int(nmn.item()))

    # ---- 33-64 atoms
    m2 = molecule(c2)
    p2 = c2["pos"]; z2 = np.zeros_like(p2)
    api.gridff_run_replicas(g1, m2, api.make_integrator("vv", 20, 0.5), dev(p2), dev(z2))
    api.gridff_run_replicas(g1, m2, api.make_integrator("langevin", 20, 0.5, temperature=300.0, gamma=0.01, seed=9), dev(p2), dev(z2))
    mn2 = torch.zeros((64, 4 + 3 * 60), device="cuda"); nmn2 = torch.zeros(1, dtype=torch.int32, device="cuda")
    api.gridff_run_replicas(g1, m2, api.make_integrator("fire", 200, 0.5, f_tol=1.0, restart=1, seed=c2["integ"]["seed"], dt_max=20.0, max_step=0.1),
                            dev(p2), dev(z2), d_fire=torch.zeros((6, 4), device="cuda"), d_minima=mn2, d_n_minima=nmn2)
    api.gridff_run_scan(g1, m2, api.make_integrator("fire", 30, 1.0, f_tol=0.05, dt_max=10.0, max_step=0.05, n_scan=2, fixed=(59,), scan_dx=(0.1, 0.0, 0.0)),
                        dev(p2), dev(z2))
    for v in (1, 2, 4):
        api.gridff_run_replicas(g1, m2, api.make_integrator("vv", 10, 0.5, variant=v), dev(p2), dev(z2))
        api.gridff_run_replicas(g1, m2, api.make_integrator("fire", 10, 0.5, variant=v), dev(p2), dev(z2), d_fire=torch.zeros((6, 4), device="cuda"))
    # more than 8 atom kinds: the pair-of-warps kernel forms the pair parameters per pair
    tk = dict(c2["topo"]); tk["lj_R"] = (tk["lj_R"] + 0.01 * np.arange(60)).astype(np.float32)
    api.gridff_run_replicas(g1, molecule(c2, tk), api.make_integrator("vv", 10, 0.5), dev(p2), dev(z2))
    n_mux2 = sms * 2 * 4 + 5
    cm2 = inputs.config(2, n_rep=n_mux2, small=True, spacing=0.2)
    api.gridff_run_replicas(g1, m2, api.make_integrator("vv", 512, 0.5), dev(cm2["pos"]), torch.zeros_like(dev(cm2["pos"])))
    say("k_replicas 33-64 atoms: pair of warps VV / Langevin / FIRE + restart / scan / > 8 kinds / %d replicas x 512 steps, two atoms per lane (variants 1, 2, 4); minima %d"
        % (n_mux2, int(nmn2.item())))

    # ---- minima hopping
    hop = api.make_hopping(2, 40, 0.5, 300.0, 0.01, 200, 1.0, 0.5, seed=7, dt_max=10.0, max_step=0.1)
    lib = torch.zeros((64, 4 + 3 * 30), device="cuda"); nlib = torch.zeros(1, dtype=torch.int32, device="cuda")
    st = api.gridff_minima_hopping(g1, m1, hop, dev(p1), lib, nlib)
    say("minima hopping: 2 cycles, stats %s" % st.cpu().numpy().tolist())

    buf = torch.ones(1 << 20, dtype=torch.uint8, device="cuda")
    api.gridff_probe_read(buf, iters=2, mode=0); api.gridff_probe_read(buf, iters=2, mode=1)
    say("probes")
    print("launches: %d" % api.gridff_launch_count())


if __name__ == "__main__":
    main()
