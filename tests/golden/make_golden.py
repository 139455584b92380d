"""Writes the stored expected values under tests/golden/ by calling ONLY the CPU oracle (oracle/) on the seeded
workloads of paper_2410_09146_b200/workloads.py (input recipes, no arithmetic of the method).

    python tests/golden/make_golden.py

The paper prints no numerical value for this path (its results are figures that are not in the container),
so these fixtures are regression anchors of the oracle, not paper values: they catch an unintended change of the oracle's
arithmetic (any deliberate change must cite the passage or DESIGN.md reading that justifies it, and regenerate them).
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import orc                                    # noqa: E402
from paper_2410_09146_b200 import workloads as wl         # noqa: E402


def shock_tube_profile():
    """Config 1 at t = 0.4 (PLM-minmod, HLL, CFL 0.4): x, rho, v^x, v^y, P, B^y at every 8th zone."""
    w = wl.shock_tube(256)
    p = w["params"]
    o = orc.Run(p, w["prim"])
    while o.t < 0.4 - 1e-14:
        o.step(min(o.dt(0.4), 0.4 - o.t))
    q = wl.from_blocks(p, o.prim)[:, 0, 0]
    W = np.sqrt(1.0 + q[1] ** 2 + q[2] ** 2 + q[3] ** 2)
    x = wl.cell_centres(p)[0]
    rows = np.stack([x, q[0], q[1] / W, q[2] / W, (p["gamma_ad"] - 1.0) * q[4], q[6]], axis=1)[::8]
    return len(o.dts), rows


def one_step_checksums():
    """Sum and sum of squares of every conserved variable after one RK2 step of small instances of configs 2-5."""
    out = []
    for name, w in (("cfg2_box_16", wl.periodic_box(16)), ("cfg3_ks_torus_16", wl.kerr_schild_torus(16)),
                    ("cfg4_turb_16", wl.turbulence_box(16)), ("cfg5_blocks_2x2x2_of_8", wl.packed_blocks((2, 2, 2), 8)),
                    ("next1_turb_16_aoah", wl.turbulence_box(16, recon=wl.RECON_WENO5Z_AOAH)),
                    ("next1b_turb_16_mp5", wl.turbulence_box(16, recon=wl.RECON_MP5)),
                    ("next2_sedov_24", wl.sedov_blast(24))):
        p = w["params"]
        o = orc.Run(p, w["prim"])
        dt = o.dt(w["cfl"])
        o.step(dt)
        c = wl.from_blocks(p, o.cons).reshape(8, -1)
        out.append((name, dt, c.sum(axis=1), (c * c).sum(axis=1)))
    return out


def next3_workloads():
    """passive scalar (Eq.14) and the floors rho0 r^-2, eps0 r^-1."""
    fl = dict(floor_form=3, rho_floor=1e-2, eps_floor=1e-2, floor_alpha_rho=2.0, floor_alpha_eps=1.0)
    def scalar(w, seed):
        return wl.with_scalar(w, wl.smooth_scalar(w["params"], seed))
    def floors(w):
        return dict(w, params=dict(w["params"], **fl))
    return (("next3_turb_16_scalar", scalar(wl.turbulence_box(16), 1)),
            ("next3_ks_torus_16_scalar_rfloor", scalar(floors(wl.kerr_schild_torus(16)), 2)),
            ("next3_blocks_2x2x2_of_8_scalar_rfloor", scalar(floors(wl.packed_blocks((2, 2, 2), 8)), 3)))


def next3_checksums():
    out = []
    for name, w in next3_workloads():
        p = w["params"]
        o = orc.Run(p, w["prim"])
        dt = o.dt(w["cfl"])
        o.step(dt)
        c = wl.from_blocks(p, o.cons).reshape(9, -1)
        m = wl.from_blocks(p, o.mask[:, None])[0]
        out.append((name, dt, c.sum(axis=1), (c * c).sum(axis=1), [int(((m & b) != 0).sum()) for b in (1, 2, 64, 128)]))
    return out


if __name__ == "__main__":
    with open(os.path.join(HERE, "one_step_checksums_next3.txt"), "w") as f:
        f.write("# oracle, one RK2 step at CFL 0.4 of small workloads with the passive scalar / radial floors; written by tests/golden/make_golden.py\n")
        f.write("# name dt  sum(U~_v) v=0..8  sum(U~_v^2) v=0..8  cells with mask bit 1, 2, 64, 128 after stage 2\n")
        for name, dt, s1, s2, bits in next3_checksums():
            f.write(name + " " + "%.15e " % dt + " ".join("%.15e" % v for v in s1) + " " + " ".join("%.15e" % v for v in s2)
                    + " " + " ".join(str(b) for b in bits) + "\n")
    nsteps, rows = shock_tube_profile()
    with open(os.path.join(HERE, "cfg1_shock_tube_t0.4.txt"), "w") as f:
        f.write("# oracle, BASELINE.json configs[0]: 256 zones, PLM-minmod, HLL, RK2, CFL 0.4, t = 0.4; %d steps\n" % nsteps)
        f.write("# written by tests/golden/make_golden.py (oracle only); columns: x rho v^x v^y P B^y, every 8th zone\n")
        for r in rows:
            f.write(" ".join("%.15e" % v for v in r) + "\n")
    with open(os.path.join(HERE, "one_step_checksums.txt"), "w") as f:
        f.write("# oracle, one RK2 step at CFL 0.4 of small instances of the workloads; written by tests/golden/make_golden.py\n")
        f.write("# name dt  sum(U~_v) v=0..7  sum(U~_v^2) v=0..7\n")
        for name, dt, s1, s2 in one_step_checksums():
            f.write(name + " " + "%.15e " % dt + " ".join("%.15e" % v for v in s1) + " " + " ".join("%.15e" % v for v in s2) + "\n")
    print("golden files written")
