"""Stored expected values (tests/golden/, written by tests/golden/make_golden.py from the oracle alone; the paper prints no
value for this path): the oracle still reproduces them (CPU), and the CUDA path reproduces them (GPU)."""
import os

import numpy as np
import pytest

from oracle import orc
from paper_2410_09146_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")

SMALL = {
    "cfg2_box_16": lambda: wl.periodic_box(16), "cfg3_ks_torus_16": lambda: wl.kerr_schild_torus(16),
    "cfg4_turb_16": lambda: wl.turbulence_box(16), "cfg5_blocks_2x2x2_of_8": lambda: wl.packed_blocks((2, 2, 2), 8),
    "next1_turb_16_aoah": lambda: wl.turbulence_box(16, recon=wl.RECON_WENO5Z_AOAH),
    "next1b_turb_16_mp5": lambda: wl.turbulence_box(16, recon=wl.RECON_MP5),
    "next2_sedov_24": lambda: wl.sedov_blast(24),
}


def read_checksums():
    out = {}
    with open(os.path.join(GOLD, "one_step_checksums.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            t = line.split()
            v = np.array([float(x) for x in t[1:]])
            out[t[0]] = (v[0], v[1:9], v[9:17])
    return out


def _next3():
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLD, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return dict(mod.next3_workloads())


def read_next3():
    out = {}
    with open(os.path.join(GOLD, "one_step_checksums_next3.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            t = line.split()
            v = np.array([float(x) for x in t[1:20]])
            out[t[0]] = (v[0], v[1:10], v[10:19], [int(x) for x in t[20:24]])
    return out


NEXT3 = ("next3_turb_16_scalar", "next3_ks_torus_16_scalar_rfloor", "next3_blocks_2x2x2_of_8_scalar_rfloor")


def read_shock_tube():
    return np.loadtxt(os.path.join(GOLD, "cfg1_shock_tube_t0.4.txt"))


def check_sums(c, s1, s2, tol):
    c = c.reshape(len(s1), -1)
    scale = np.sqrt(s2.max() * c.shape[1])                 # a sum of N terms of the largest variable's size
    assert np.abs(c.sum(axis=1) - s1).max() <= tol * scale
    assert np.abs((c * c).sum(axis=1) - s2).max() <= tol * s2.max()


@pytest.mark.parametrize("name", list(SMALL))
def test_oracle_reproduces_stored_one_step_checksums(name):
    dt, s1, s2 = read_checksums()[name]
    w = SMALL[name]()
    p = w["params"]
    o = orc.Run(p, w["prim"])
    assert abs(o.dt(w["cfl"]) - dt) <= 1e-14 * dt
    o.step(dt)
    check_sums(wl.from_blocks(p, o.cons), s1, s2, 1e-13)


@pytest.mark.parametrize("name", NEXT3)
def test_oracle_reproduces_stored_next3_checksums(name):
    dt, s1, s2, bits = read_next3()[name]
    w = _next3()[name]
    p = w["params"]
    o = orc.Run(p, w["prim"])
    assert abs(o.dt(w["cfl"]) - dt) <= 1e-14 * dt
    o.step(dt)
    check_sums(wl.from_blocks(p, o.cons), s1, s2, 1e-13)
    m = wl.from_blocks(p, o.mask[:, None])[0]
    assert [int(((m & b) != 0).sum()) for b in (1, 2, 64, 128)] == bits


def test_oracle_reproduces_stored_shock_tube_profile():
    gold = read_shock_tube()
    w = wl.shock_tube(256)
    p = w["params"]
    o = orc.Run(p, w["prim"])
    while o.t < 0.4 - 1e-14:
        o.step(min(o.dt(0.4), 0.4 - o.t))
    q = wl.from_blocks(p, o.prim)[:, 0, 0]
    W = np.sqrt(1.0 + q[1] ** 2 + q[2] ** 2 + q[3] ** 2)
    rows = np.stack([wl.cell_centres(p)[0], q[0], q[1] / W, q[2] / W, (p["gamma_ad"] - 1.0) * q[4], q[6]], axis=1)[::8]
    assert np.abs(rows - gold).max() <= 1e-12


@pytest.mark.gpu
@pytest.mark.parametrize("name", list(SMALL))
def test_gpu_reproduces_stored_one_step_checksums(name):
    from harness import GpuRun
    dt, s1, s2 = read_checksums()[name]
    w = SMALL[name]()
    p = w["params"]
    g = GpuRun(p, w["prim"])
    assert abs(g.dt(w["cfl"]) - dt) <= 1e-13 * dt
    g.step(dt)
    check_sums(wl.from_blocks(p, g.get()[0]), s1, s2, 1e-11)


@pytest.mark.gpu
@pytest.mark.parametrize("name", NEXT3)
def test_gpu_reproduces_stored_next3_checksums(name):
    from harness import GpuRun
    dt, s1, s2, bits = read_next3()[name]
    w = _next3()[name]
    p = w["params"]
    g = GpuRun(p, w["prim"])
    assert abs(g.dt(w["cfl"]) - dt) <= 1e-13 * dt
    g.step(dt)
    cons, _, _, mask = g.get()
    check_sums(wl.from_blocks(p, cons), s1, s2, 1e-11)
    m = wl.from_blocks(p, mask[:, None])[0]
    assert [int(((m & b) != 0).sum()) for b in (1, 2, 64, 128)] == bits


@pytest.mark.gpu
def test_gpu_reproduces_stored_shock_tube_profile():
    from harness import GpuRun
    gold = read_shock_tube()
    w = wl.shock_tube(256)
    p = w["params"]
    g = GpuRun(p, w["prim"])
    t = 0.0
    while t < 0.4 - 1e-14:
        dt = min(g.dt(0.4), 0.4 - t)
        g.step(dt)
        t += dt
    q = wl.from_blocks(p, g.get()[1])[:, 0, 0]
    W = np.sqrt(1.0 + q[1] ** 2 + q[2] ** 2 + q[3] ** 2)
    rows = np.stack([wl.cell_centres(p)[0], q[0], q[1] / W, q[2] / W, (p["gamma_ad"] - 1.0) * q[4], q[6]], axis=1)[::8]
    assert np.abs(rows - gold).max() <= 1e-8        # BASELINE.json's many-step tolerance (247 steps with the GPU's own dt)
