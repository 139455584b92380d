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
roofline  : the dominant kernel class (the three reconstruct + Riemann sweeps, fp64-bound) against the fp64 peak measured in
            the same run (phx_debug_fp64_peak), per-launch time from CUDA events recorded by the library on the launching
            stream inside the timed region (phx_profile_*); executed fp64 work and DRAM traffic per launch from the ncu
            capture named in COUNTS_FILE, used only if it was taken from the kernel sources that run; plus the update
            kernel against the HBM copy bandwidth and the whole step as SURVEY.md 8(d) defines its roofline.
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

# Algorithmic traffic per interior zone and launch: what the kernel's definition must move.
# The sweeps read P (64 B), write the two magnetic flux components flux-CT needs (16 B) and accumulate the divergence of the
# five non-magnetic components (x: 40 B written; y, z: 40 B read + 40 B written).
# update, two byte models: "design" = everything this design makes the kernel move (the accumulated divergence 40 B + 3 x 2
# magnetic flux components 48 B + U~0 64 B + U~1 in stage 2 only, 32 B averaged + 5 primitives 40 B + U~ and P written
# 128 B + mask 1 B = 353 B); "method" = without the two intermediates the split into sweeps and update creates (265 B).
ALGO_BYTES_PER_ZONE = {
    "sweep_x": 64.0 + 16.0 + 40.0, "sweep_y": 64.0 + 16.0 + 80.0, "sweep_z": 64.0 + 16.0 + 80.0,
    "update": 40.0 + 48.0 + 64.0 + 32.0 + 40.0 + 64.0 + 64.0 + 1.0,
    "fill_ghosts": 0.0, "cfl": 64.0, "prim_to_cons": 128.0, "c2p": 129.0, "copy": 128.0,
}
UPDATE_METHOD_BYTES_PER_ZONE = 64.0 + 32.0 + 40.0 + 64.0 + 64.0 + 1.0
# Executed fp64 work per zone and DRAM traffic per launch are NOT constants of this file: they are read from the ncu
# capture named here (written by paper_2410_09146_b200/profile_counts.py), and used only if the kernel sources this run
# executes hash to what the capture was taken from.
COUNTS_FILE = os.path.join("profiles", "r02_kernel_counts.csv")
COUNTS_WORKLOAD = "cfg4_256"
SWEEPS = ("sweep_x", "sweep_y", "sweep_z")


def load_counts():
    """({class: counts}, capture id, valid) for the 256^3 bench workload; valid = the capture is of these kernel sources."""
    from paper_2410_09146_b200 import profile_counts as pc
    path = os.path.join(ROOT, COUNTS_FILE)
    if not os.path.exists(path):
        return {}, None, False
    rows, sha = pc.load(path, COUNTS_WORKLOAD)
    cap = next(iter(rows.values()))["capture"] if rows else None
    return rows, cap, bool(rows) and sha == pc.source_hash()


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


def set_oracle_threads(n):
    """Number of OpenMP threads of the oracle's loops (the OpenMP runtime liborc.so is linked against)."""
    import ctypes
    from oracle import orc
    orc.lib()
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


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
    bad = phx.count_masked(mesh, mask, phx.M_NOCONV | phx.M_BAD_INPUT)             # con2prim failures of the last stage
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

    # ---- rooflines.  The fp64 peak is measured in this run (a DFMA loop on every SM for >= 0.5 s, after the timed region).
    peaks, which = measured_peaks()
    psampler = ClockSampler(local)
    dfma_per_s, dfma_burst, peak_ms, nsm = phx.debug_fp64_peak(0.5)
    pclk = psampler.stop()
    r64 = dfma_per_s                                   # fp64 thread-instructions per second the pipe issues (any of dadd / dmul / dfma)
    fp64_peak = {"dfma_per_s": dfma_per_s, "tflops": 2.0 * dfma_per_s / 1e12, "seconds": peak_ms * 1e-3, "sms": nsm,
                 "burst_tflops": 2.0 * dfma_burst / 1e12,     # the 25 ms calibration launch: before the power cap acts
                 "which": "sustained (the step is timed inside a long loop under the power cap)",
                 "sm_mhz_during": pclk["sm_mhz"], "reasons_during": pclk["reasons"],
                 "nominal_tflops": nsm * 64 * 2 * (peaks.get("sm_max_mhz", 1965.0) * 1e6) / 1e12,
                 "how": "phx_debug_fp64_peak: 8 independent DFMA chains per thread, 64 warps per SM, CUDA events"}
    nall = int(np.prod(prim.shape)) // prim.shape[1]
    per_launch_bytes = {k: v * zones for k, v in ALGO_BYTES_PER_ZONE.items()}
    per_launch_bytes["fill_ghosts"] = (nall - zones) * 128.0
    kern = {k: {"ms_total": v[0], "launches": v[1], "ms_per_launch": v[0] / v[1], "share": v[0] / ms}
            for k, v in prof.items() if v[1] > 0}
    counts, capture, counts_ok = load_counts()
    if args.workload != "cfg4" or args.n != 256:
        counts_ok = False                               # the counts are those of the 256^3 bench workload

    def instr(k):   # executed fp64 thread-instructions / flop per zone and launch of class k (update: both stages averaged)
        if k == "update":
            return 0.5 * (counts["update"]["fp64_instr_per_zone"] + counts["update_cfl"]["fp64_instr_per_zone"]), \
                   0.5 * (counts["update"]["flop_per_zone"] + counts["update_cfl"]["flop_per_zone"])
        if k in counts:
            return counts[k]["fp64_instr_per_zone"], counts[k]["flop_per_zone"]
        return 0.0, 0.0

    def traffic(k):
        if k == "update":
            return 0.5 * sum(counts[c]["dram_read_bytes"] + counts[c]["dram_write_bytes"] for c in ("update", "update_cfl"))
        return counts[k]["dram_read_bytes"] + counts[k]["dram_write_bytes"] if k in counts else None

    roofline = None
    if all(k in kern for k in SWEEPS + ("update",)):
        # (1) the dominant kernel CLASS: the three reconstruct + Riemann sweeps (one kernel template, x and marching y / z)
        sw_ms = sum(kern[k]["ms_total"] for k in SWEEPS)
        sw_launch = sum(kern[k]["launches"] for k in SWEEPS)
        sw_dur = sw_ms / sw_launch * 1e-3
        sw_bytes = sum(per_launch_bytes[k] for k in SWEEPS) / 3.0
        roofline = {"kernel": "sweeps: k_sweep_x + k_sweep_march<y> + k_sweep_march<z> (fused reconstruct + Riemann + divergence)",
                    "bound": "alu", "unit": "TFLOP/s", "peak": fp64_peak["tflops"],
                    "peak_source": "measured in this run (DFMA loop, %.2f s, SM clock %s MHz): 2 flop x %.3e DFMA/s; nominal %d SM x 64 lanes x 2 x %.0f MHz = %.1f"
                                   % (fp64_peak["seconds"], pclk["sm_mhz"], dfma_per_s, nsm, peaks.get("sm_max_mhz", 1965.0), fp64_peak["nominal_tflops"]),
                    "ms_per_launch": sw_dur * 1e3, "share_of_step": sw_ms / ms,
                    "hbm_gbs_achieved": sw_bytes / sw_dur / 1e9, "hbm_frac": sw_bytes / sw_dur / 1e9 / peaks["hbm_gbs"],
                    "counts_from": f"{COUNTS_FILE} capture {capture}" if counts_ok else None}
        if counts_ok:
            ins = sum(instr(k)[0] for k in SWEEPS) / 3.0 * zones
            flo = sum(instr(k)[1] for k in SWEEPS) / 3.0 * zones
            roofline.update(achieved=flo / sw_dur / 1e12, frac=flo / sw_dur / 1e12 / fp64_peak["tflops"],
                            traffic=sum(traffic(k) for k in SWEEPS) / 3.0,
                            instr_rate={"achieved": ins / sw_dur, "peak": r64, "unit": "fp64 thread-instr/s", "frac": ins / sw_dur / r64})
        else:
            roofline.update(achieved=None, frac=None, traffic=None, instr_rate=None,
                            note="no ncu capture of these kernel sources under profiles/: fp64 figures withheld")
        # (2) the HBM-bound kernel: flux-CT + update + con2prim + floors
        up_dur = kern["update"]["ms_per_launch"] * 1e-3
        up = {"kernel": "k_update (flux-CT + divergence + sources + RK combine + con2prim + floors)", "bound": "hbm", "unit": "GB/s",
              "peak": peaks["hbm_gbs"], "peak_source": which,
              "achieved": UPDATE_METHOD_BYTES_PER_ZONE * zones / up_dur / 1e9,
              "frac": UPDATE_METHOD_BYTES_PER_ZONE * zones / up_dur / 1e9 / peaks["hbm_gbs"],
              "bytes_per_zone": UPDATE_METHOD_BYTES_PER_ZONE,
              "design_bytes_per_zone": ALGO_BYTES_PER_ZONE["update"],
              "design_frac": per_launch_bytes["update"] / up_dur / 1e9 / peaks["hbm_gbs"],
              "ms_per_launch": up_dur * 1e3, "share_of_step": kern["update"]["share"]}
        if counts_ok:
            up.update(traffic=traffic("update"), traffic_over_algorithmic=traffic("update") / (UPDATE_METHOD_BYTES_PER_ZONE * zones),
                      fp64_instr_rate_frac=instr("update")[0] * zones / up_dur / r64)
        else:
            up.update(traffic=None, traffic_over_algorithmic=None)
        roofline["update"] = up
        # (3) the step as SURVEY.md 8(d) defines it: T_roof = sum over launches of max(bytes / BW, fp64 instructions / R64)
        if counts_ok:
            t_roof, tot_ins, tot_flo = 0.0, 0.0, 0.0
            for k, v in kern.items():
                nl = v["launches"] / K
                by = per_launch_bytes.get(k, 0.0) if k != "update" else UPDATE_METHOD_BYTES_PER_ZONE * zones
                ik, fk = instr(k)
                t_roof += nl * max(by / (peaks["hbm_gbs"] * 1e9), ik * zones / r64)
                tot_ins += nl * ik * zones
                tot_flo += nl * fk * zones
            step_s = ms / K * 1e-3
            roofline["step"] = {"t_roof_ms": t_roof * 1e3, "ms_per_step": ms / K, "frac_of_per_kernel_rooflines": t_roof / step_s,
                                "fp64_instr_per_zone_cycle": tot_ins / zones, "instr_rate_frac": tot_ins / step_s / r64,
                                "flop_rate_frac": tot_flo / step_s / (2.0 * r64),
                                "binding": "fp64 instruction issue (the whole step is ALU-bound: %.0f fp64 instructions per zone-cycle against %.0f algorithmic bytes)"
                                           % (tot_ins / zones, 2 * (sum(ALGO_BYTES_PER_ZONE[k] for k in SWEEPS) + UPDATE_METHOD_BYTES_PER_ZONE)),
                                "claim": "north_star's >= 50 % of the binding roofline is claimed on instr_rate_frac: the fp64 pipe issues one "
                                         "thread-instruction per lane and cycle whether it is an add, a multiply or a fused multiply-add, and "
                                         "only 47 % of this path's fp64 instructions can be fused; flop_rate_frac counts the same work against "
                                         "2 flop per lane and cycle"}
    roofline_out = roofline
    if roofline_out is not None:
        if not counts_ok:
            # without a capture of these sources only the byte-counted roofline can be stated: the update kernel's
            roofline_out = dict(roofline["update"], sweeps=roofline)
            del roofline["update"]
        roofline_out["fp64_peak"] = fp64_peak

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
        "gpu_launches": int(launches), "roofline": roofline_out, "clocks": clocks,
        "kernels": kern, "state_finite": finite, "c2p_failed_cells": bad,
    }
    if not args.no_cpu_baseline and world >= 1:
        ws, steps, what = oracle_sample(args.workload)
        zs, per_step = time_oracle(0, steps, ws)
        line["cpu_baseline"] = {"value": zs * steps / sum(per_step), "unit": UNIT, "cores": oracle_cores(), "kind": "oracle",
                                "sample": f"{what} ({zs * steps} zone-cycles; {zones * K} timed on the GPU)"}
        # the same oracle on ONE host thread, on a 64^3 box of the config-4 recipe, one step
        set_oracle_threads(1)
        z1, per1 = time_oracle(64, 1)
        set_oracle_threads(oracle_cores())
        line["cpu_baseline"]["single_thread"] = {"value": z1 / sum(per1), "unit": UNIT, "cores": 1,
                                                 "sample": "config-4 recipe at 64^3, one RK2 step + CFL"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
