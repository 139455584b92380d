"""bench.py — GRMHD zone-cycles/s of the CUDA hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n 256]

One "step" is one full RK2 cycle of the whole hot path over the whole mesh: phx_rk2_step_cfl =
2 x { x/y/z reconstruct+Riemann sweeps, flux-CT + divergence + sources + RK combine + con2prim + floors, ghost fill }
with the CFL reduction of the next time step fused into the second stage's update kernel (a8/a7 of SURVEY.md 8a).  Workload at N=1: BASELINE.json configs[3], the 256^3 periodic turbulence-like
box (WENO5-Z, HLL, flux-CT, RK2, Minkowski, Gamma=5/3) that north_star's roofline target is quoted on; inputs are
seeded synthetic fields from paper_2410_09146_b200/workloads.py (recipe in DESIGN.md section 4).

value     : interior zones x K / device time (CUDA events, max over ranks), state resident in HBM.
e2e       : same metric through phx_evolve_host (HOST buffers: H2D of the primitives and D2H of the new primitives
            and the mask inside the timed region, one call per step).
roofline  : dominant kernel class, per-launch time from CUDA events recorded by the library on the launching
            stream inside the timed region (phx_profile_*), algorithmic bytes / flops per zone from DESIGN.md 6.
cpu_baseline : the oracle (oracle/, as it stands) on a bounded sample of the same workload on the host cores.
N > 1     : the path does not shard in this build ("replicas only") - every rank runs an independent
            replica of the same workload, no data-path collective; value = N x zones x K / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "grmhd_zone_cycles_per_sec"
UNIT = "zone-cycles/s"

# Algorithmic traffic and arithmetic per interior zone and launch.
# Bytes: what the kernel's definition must move.  The sweeps read P (64 B), write the two magnetic flux components flux-CT
# needs (16 B) and accumulate the divergence of the five non-magnetic components (x: 40 B written; y, z: 40 B read + 40 B
# written).  update = that divergence (40 B) + 3 x 2 magnetic flux components (48 B) + U~0 read + U~1 read (stage 2 only:
# 32 B averaged over both stages) + 5 primitives read (sources / con2prim guess) + U~ and P written + mask.
ALGO_BYTES_PER_ZONE = {
    "sweep_x": 64.0 + 16.0 + 40.0, "sweep_y": 64.0 + 16.0 + 80.0, "sweep_z": 64.0 + 16.0 + 80.0,
    "update": 40.0 + 48.0 + 64.0 + 32.0 + 40.0 + 64.0 + 64.0 + 1.0,
    "fill_ghosts": 0.0, "cfl": 64.0, "prim_to_cons": 128.0, "c2p": 129.0, "copy": 128.0,
}
# fp64 flop per interior zone and launch for the WENO5-Z + HLL Minkowski path: dadd + dmul + 2*dfma thread-instructions of
# the committed kernels counted by ncu (profiles/r01_ncu_summary.md; con2prim iterations are data dependent, the figure
# is the one measured on this workload).  achieved = these flops / measured time, i.e. useful fp64 work only.
# update: average of the first stage (631) and the second stage, which also evaluates the signal speeds for the fused CFL
# reduction (760); the "cfl" class is the one-block final kernel of that reduction
ALGO_FLOP_PER_ZONE = {"sweep_x": 1106.0, "sweep_y": 1141.0, "sweep_z": 1141.0, "update": 695.0, "cfl": 0.0}
# fp64 peak from unit counts and clocks: 148 SM x 64 fp64 lanes x 2 flop x 1.965 GHz; a DFMA loop measured
# 33.9 TFLOP/s on this pool's B200 (16.94 T DFMA/s)
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
FP64_MEASURED_DFMA_TFLOPS = 33.9
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full capture under profiles/ (bytes)
NCU_TRAFFIC = {256: {"update": 6.126e9, "sweep_x": 2.040e9, "sweep_y": 2.797e9, "sweep_z": 2.796e9, "cfl": 0.0,
                     "fill_ghosts": 0.255e9}}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=256, help="zones per side of the config-4 box (256 = BASELINE.json)")
    ap.add_argument("--workload", default="cfg4", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "next1", "next2", "next3"],
                    help="cfg4 (default) is the bench workload; the others time BASELINE.json's other 3-D configs at full size "
                         "(reported without a roofline object: the per-zone figures of DESIGN.md 6 are config 4's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            c = [t.strip() for t in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for name, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close(); os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# --------------------------------------------------------------------------------------------- the oracle, timed
def oracle_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def make_workload(name, n):
    """(workload dict, descriptive name) of a bench workload; n only matters for cfg4 / next1 / next2."""
    from paper_2410_09146_b200 import workloads as wl
    if name == "cfg4":
        return wl.turbulence_box(n), f"cfg4_turbulence_box_{n}^3_weno5z_hll_ct_rk2_minkowski"
    if name == "next1":     # config 4 with the paper's WENO5-Z-AOAH reconstruction
        return wl.turbulence_box(n, recon=wl.RECON_WENO5Z_AOAH), f"next1_turbulence_box_{n}^3_weno5z_aoah_hll_ct_rk2_minkowski"
    if name == "next2":     # the paper's scaling workload shape, --n 128 is its size
        return wl.sedov_blast(n), f"next2_sedov_blast_{n}^3_plm_minmod_hll_rk2_minkowski"
    if name == "next3":     # config 5 carrying a passive scalar (Eq.14) with the floors rho0 r^-2, eps0 r^-1
        return _scalar_blocks(wl, (8, 8, 8)), "next3_packed_blocks_512x32^3_kerr_schild_passive_scalar_radial_floors"
    if name == "cfg1":
        return wl.shock_tube(256), "cfg1_shock_tube_256_plm_minmod_hll_rk2_minkowski"
    if name == "cfg2":
        return wl.periodic_box(64), "cfg2_periodic_box_64^3_plm_mc_llf_ct_rk2_minkowski"
    if name == "cfg3":
        return wl.kerr_schild_torus(128), "cfg3_kerr_schild_torus_128^3_plm_minmod_hll_ct_rk2"
    return wl.packed_blocks((8, 8, 8), 32), "cfg5_packed_blocks_512x32^3_kerr_schild_plm_minmod_hll_ct_rk2"


def _scalar_blocks(wl, nb):
    w = wl.packed_blocks(nb, 32)
    w = dict(w, params=dict(w["params"], floor_form=3, rho_floor=1e-2, eps_floor=1e-2, floor_alpha_rho=2.0, floor_alpha_eps=1.0))
    return wl.with_scalar(w, wl.smooth_scalar(w["params"], wl.SEED0 + 9))


def oracle_sample(name):
    """Bounded sample of a workload for the oracle's timing: (workload dict, steps, description)."""
    from paper_2410_09146_b200 import workloads as wl
    if name == "cfg4":
        return wl.turbulence_box(128), 3, "config-4 recipe at 128^3, 3 RK2 steps"
    if name == "next1":
        return wl.turbulence_box(128, recon=wl.RECON_WENO5Z_AOAH), 3, "config-4 recipe with WENO5-Z-AOAH at 128^3, 3 RK2 steps"
    if name == "next2":
        return wl.sedov_blast(128), 3, "Sedov blast at 128^3, 3 RK2 steps"
    if name == "next3":
        return _scalar_blocks(wl, (4, 4, 4)), 2, "next3 recipe on 64 blocks of 32^3 (1/8 of the mesh), 2 RK2 steps"
    if name == "cfg1":
        return wl.shock_tube(256), 247, "the whole of config 1 (256 zones, 247 RK2 steps)"
    if name == "cfg2":
        return wl.periodic_box(64), 20, "config 2 at full size (64^3), 20 of its 100 RK2 steps"
    if name == "cfg3":
        return wl.kerr_schild_torus(96), 3, "config-3 recipe at 96^3, 3 RK2 steps"
    return wl.packed_blocks((4, 4, 4), 32), 2, "config-5 recipe on 64 blocks of 32^3 (1/8 of the mesh), 2 RK2 steps"


def time_oracle(n, steps, w=None):
    """Zone-cycles/s of the CPU oracle (as it stands, OpenMP over its outer loops); default: config-4 recipe at n^3."""
    from oracle import orc
    from paper_2410_09146_b200 import workloads as wl
    if w is None:
        w = wl.turbulence_box(n)
    o = orc.Run(w["params"], w["prim"])
    per_step = []
    for _ in range(steps):
        t0 = time.perf_counter()
        dt = o.dt(w["cfl"])
        o.step(dt)
        per_step.append(time.perf_counter() - t0)
    return wl.n_zones(w["params"]), per_step


def run_reference(args):
    """--impl reference: there is no reference code (PAPER.md only); the arm is the oracle on the host cores, each
    step a bounded sample (a 64^3 box of the config-4 recipe) of the 256^3 workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = 64
    zones, per_step = time_oracle(n, args.warmup + args.steps)
    timed = per_step[args.warmup:]
    total = sum(timed)
    value = zones * len(timed) / total
    cores = oracle_cores()
    sample = f"config-4 recipe at {n}^3 (1/{(args.n // n) ** 3} of the {args.n}^3 workload), one RK2 step + CFL per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / len(timed), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"cfg4_turbulence_box_{args.n}^3_weno5z_hll_ct_rk2_minkowski", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def aggregate(ms_local, zones, steps, world, device):
    """Whole-job figure of `world` independent replicas (replicas only, no data-path collective): the device
    time is the MAX over ranks, value = world x zones x steps / that time.  Returns (ms, zone-cycles/s)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    return ms, world * zones * steps / (ms * 1e-3)


# --------------------------------------------------------------------------------------------- the CUDA path
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2410_09146_b200 import phx, workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    phx.lib()   # fails loudly if libphx.so is missing

    K, W = args.steps, max(args.warmup, 0)
    w, wname = make_workload(args.workload, args.n)
    p = w["params"]
    zones = wl.n_zones(p)
    mesh = phx.init_mesh(p)
    h_prim = torch.from_numpy(w["prim"])
    prim = h_prim.cuda()
    cons = torch.empty_like(prim); cons0 = torch.empty_like(prim)
    mask = torch.zeros((prim.shape[0],) + tuple(prim.shape[2:]), dtype=torch.uint8, device="cuda")
    d_dt = torch.zeros(1, dtype=torch.float64, device="cuda")
    field_bytes = prim.numel() * 8
    phx.prim_to_cons(mesh, prim, cons)

    phx.cfl_dt(mesh, prim, w["cfl"], d_dt)      # dt of the first step; every later dt comes out of the step itself

    def step():
        phx.rk2_step_cfl(mesh, w["cfl"], d_dt, cons0, cons, prim, mask)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        step()
    barrier()
    mesh.profile_enable(K * 12 + 8)
    l0 = mesh.launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(K):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    launches = mesh.launch_count() - l0
    prof = mesh.profile_read()
    mesh.profile_enable(0)
    bad = int(mask.to(torch.int32).bitwise_and(16 | 32).count_nonzero().item())   # no-convergence / bad-input cells
    finite = bool(torch.isfinite(cons).all().item())
    ms, value = aggregate(ms, zones, K, world, "cuda")

    # ---- the same K steps through phx_evolve_device: one C call, the step replayed from a CUDA graph (no per-kernel events)
    phx.evolve_device(mesh, 2, w["cfl"], d_dt, cons0, cons, prim, mask)      # captures the graph
    barrier()
    e0.record()
    phx.evolve_device(mesh, K, w["cfl"], d_dt, cons0, cons, prim, mask)
    e1.record()
    barrier()
    ms_graph, value_graph = aggregate(e0.elapsed_time(e1), zones, K, world, "cuda")

    # ---- end to end through the HOST-buffer C-ABI call (rank-local replica; max over ranks)
    e2e = None
    if not args.no_e2e:
        del cons0
        torch.cuda.empty_cache()
        hin = h_prim.pin_memory()
        hp = torch.empty_like(hin).pin_memory()
        hm = torch.empty(mask.shape, dtype=torch.uint8).pin_memory()
        ke = max(1, min(K, 3))
        # the step's result is the new state: the primitives (they determine U~) and the con2prim / floor mask
        phx.evolve_host(mesh, hin, 1, w["cfl"], hp, None, hm)      # warm-up (allocates the workspace)
        barrier()
        e0.record()
        for _ in range(ke):
            phx.evolve_host(mesh, hin, 1, w["cfl"], hp, None, hm)
        e1.record()
        barrier()
        _, e2e_value = aggregate(e0.elapsed_time(e1), zones, ke, world, "cuda")
        e2e = {"value": e2e_value, "unit": UNIT,
               "h2d_bytes_per_step": field_bytes, "d2h_bytes_per_step": field_bytes + hm.numel() + 16,
               "steps": ke, "call": "phx_evolve_host(nsteps=1) per step, pinned host buffers: primitives in; primitives and mask out"}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel class
    peaks, which = measured_peaks()
    nall = int(np.prod(prim.shape)) // 8
    per_launch_bytes = {k: v * zones for k, v in ALGO_BYTES_PER_ZONE.items()}
    per_launch_bytes["fill_ghosts"] = (nall - zones) * 128.0
    kern = {k: {"ms_total": v[0], "launches": v[1], "ms_per_launch": v[0] / v[1], "share": v[0] / ms}
            for k, v in prof.items() if v[1] > 0}
    top = max(kern, key=lambda k: kern[k]["ms_total"])
    dur = kern[top]["ms_per_launch"] * 1e-3
    hbm = per_launch_bytes[top] / dur / 1e9
    flops = ALGO_FLOP_PER_ZONE.get(top, 0.0) * zones / dur / 1e12
    traffic = NCU_TRAFFIC.get(args.n, {}).get(top)
    if flops / FP64_PEAK_TFLOPS >= hbm / peaks["hbm_gbs"]:
        roofline = {"kernel": top, "bound": "alu", "achieved": flops, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": flops / FP64_PEAK_TFLOPS, "traffic": traffic,
                    "peak_source": "derived: 148 SM x 64 fp64 lanes x 2 x 1.965 GHz (DFMA loop measured %.1f)" % FP64_MEASURED_DFMA_TFLOPS,
                    "hbm_gbs_achieved": hbm, "hbm_frac": hbm / peaks["hbm_gbs"]}
    else:
        roofline = {"kernel": top, "bound": "hbm", "achieved": hbm, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": hbm / peaks["hbm_gbs"], "traffic": traffic, "peak_source": which,
                    "fp64_tflops_achieved": flops, "fp64_frac": flops / FP64_PEAK_TFLOPS}
    roofline.update(ms_per_launch=kern[top]["ms_per_launch"], share_of_step=kern[top]["share"])
    # whole-step fp64 fraction: algorithmic flop of all launches of one step / step time
    step_flop = 2.0 * sum(ALGO_FLOP_PER_ZONE[k] for k in ("sweep_x", "sweep_y", "sweep_z", "update")) + ALGO_FLOP_PER_ZONE["cfl"]
    roofline["step_fp64_frac"] = step_flop * zones / (ms / K * 1e-3) / 1e12 / FP64_PEAK_TFLOPS

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wname, "zones": zones, "ng": p["ng"],
                   "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no sharding)",
                   "l2": (f"inputs larger than L2 ({field_bytes / 1e6:.0f} MB per field), no flush" if field_bytes > 126e6 else
                          f"inputs fit the 126 MB L2 ({field_bytes / 1e6:.1f} MB per field), no flush: a cache-resident small case")},
        "e2e": e2e,
        "graph_replay": {"value": value_graph, "unit": UNIT, "ms_per_step": ms_graph / K,
                         "call": "phx_evolve_device(nsteps=K): one RK2 step captured into a CUDA graph and replayed K times"},
        "gpu_launches": int(launches), "roofline": roofline, "clocks": clocks,
        "kernels": kern, "state_finite": finite, "c2p_failed_cells": bad,
    }
    if args.workload != "cfg4" or args.n != 256:
        line["roofline"] = None if args.workload != "cfg4" else roofline
    if not args.no_cpu_baseline and world >= 1:
        ws, steps, what = oracle_sample(args.workload)
        zs, per_step = time_oracle(0, steps, ws)
        line["cpu_baseline"] = {"value": zs * steps / sum(per_step), "unit": UNIT, "cores": oracle_cores(), "kind": "oracle",
                                "sample": f"{what} ({zs * steps} zone-cycles; {zones * K} timed on the GPU)"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
