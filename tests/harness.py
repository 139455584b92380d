"""Shared helpers of the parity tests: run the same seeded workload through the CUDA path (C ABI via
paper_2410_09146_b200.phx) and through the CPU oracle (oracle.orc) and compare.

Error metric (SURVEY.md 8c / DESIGN.md 5): per conserved variable v,
    err_v = max_cells |U~_gpu - U~_orc| / max_cells |U~_orc|     over interior cells,
because point-wise relative error is ill-defined where S_j ~ 0.
"""
from __future__ import annotations

import numpy as np

from oracle import orc
from paper_2410_09146_b200 import workloads as wl

TOL_1STEP = 1e-11     # BASELINE.json north_star: max relative error per conserved variable after one RK2 step
TOL_100STEP = 1e-8    # ... after 100 steps
MARGIN_MIN = 1e-9     # no c2p decision of the oracle may sit closer than this (relative) to its threshold


def interior(p, a):
    """[nb, nvar, ...] packed blocks -> global interior [nvar, Nz, Ny, Nx]; masks ([nb, k, j, i]) too."""
    a = np.asarray(a)
    if a.ndim == 4:
        return wl.from_blocks(p, a[:, None])[0]
    return wl.from_blocks(p, a)


def var_errors(p, got, ref, scale_floor=0.0):
    """scale_floor > 0: a variable's scale is at least scale_floor x the largest scale of any variable (linear-wave
    inputs, where a momentum of 1e-6 is the difference of O(1) pressure fluxes and carries their round-off)."""
    g, r = interior(p, got), interior(p, ref)
    num = np.abs(g - r).reshape(g.shape[0], -1).max(axis=1)
    den = np.abs(r).reshape(r.shape[0], -1).max(axis=1)
    den = np.maximum(den, scale_floor * den.max())
    return num / np.where(den > 0.0, den, 1.0)


class GpuRun:
    """RK2 (Heun) driver over the C ABI with an externally supplied dt sequence."""

    def __init__(self, p, prim):
        import torch
        from paper_2410_09146_b200 import phx
        assert torch.cuda.is_available(), "GPU parity tests need a CUDA device (no CPU fallback exists)"
        self.torch, self.phx = torch, phx
        self.p = dict(p)
        self.mesh = phx.init_mesh(self.p)
        self.shape = wl.alloc_shape(self.p)
        self.prim = torch.from_numpy(np.ascontiguousarray(prim)).cuda()
        self.cons = torch.empty_like(self.prim)
        self.cons0 = torch.empty_like(self.prim)
        mshape = (self.shape[0],) + tuple(self.shape[2:])
        self.mask = torch.zeros(mshape, dtype=torch.uint8, device="cuda")
        self.mask1 = torch.zeros_like(self.mask)
        self.d_dt = torch.zeros(1, dtype=torch.float64, device="cuda")
        phx.prim_to_cons(self.mesh, self.prim, self.cons)

    def step(self, dt):
        phx = self.phx
        self.cons0.copy_(self.cons)
        phx.rk_stage(self.mesh, 1.0, 0.0, dt, self.cons0, self.cons, self.prim, self.mask1)
        phx.rk_stage(self.mesh, 0.5, 0.5, 0.5 * dt, self.cons0, self.cons, self.prim, self.mask)

    def step_device_dt(self, cfl):
        """The launch configuration bench.py times: phx_cfl_dt (device scalar) + phx_rk2_step."""
        self.phx.cfl_dt(self.mesh, self.prim, cfl, self.d_dt)
        self.phx.rk2_step(self.mesh, self.d_dt, self.cons0, self.cons, self.prim, self.mask)

    def step_fused_cfl(self, cfl, first):
        """The launch configuration bench.py times: phx_rk2_step_cfl (dt of the next step reduced inside stage 2);
        the first step of a run takes its dt from phx_cfl_dt."""
        if first:
            self.phx.cfl_dt(self.mesh, self.prim, cfl, self.d_dt)
        self.phx.rk2_step_cfl(self.mesh, cfl, self.d_dt, self.cons0, self.cons, self.prim, self.mask)

    def dt(self, cfl):
        return self.phx.cfl_dt(self.mesh, self.prim, cfl, self.d_dt, host=True)

    def get(self):
        self.torch.cuda.synchronize()
        return (self.cons.cpu().numpy(), self.prim.cpu().numpy(), self.mask1.cpu().numpy(), self.mask.cpu().numpy())


def run_both(p, prim, nsteps=None, cfl=0.4, t_end=None):
    """Advance oracle and GPU with the ORACLE's dt sequence.  Returns (oracle Run, GpuRun, per-step errors)."""
    orc.reset_c2p_margin()
    o = orc.Run(p, prim)
    g = GpuRun(p, prim)
    n = 0
    while True:
        if nsteps is not None and n >= nsteps:
            break
        if t_end is not None and o.t >= t_end - 1e-14:
            break
        dt = o.dt(cfl)
        if t_end is not None:
            dt = min(dt, t_end - o.t)
        o.step(dt)
        g.step(dt)
        n += 1
    return o, g


def compare(p, o, g, tol, check_masks=True, scale_floor=0.0):
    cons, prim, mask1, mask = g.get()
    err = var_errors(p, cons, o.cons, scale_floor)
    assert np.all(np.isfinite(cons[np.isfinite(o.cons)])), "non-finite GPU result where the oracle is finite"
    assert err.max() <= tol, f"conserved-variable errors {err} exceed {tol}"
    # full ghost frame of the primitives: same values as the oracle's ghost fill
    perr = np.abs(prim - o.prim).max() / np.abs(o.prim).max()
    assert perr <= max(tol * 100, 1e-9), f"primitive field (with ghosts) differs: {perr}"
    if check_masks:
        margin = orc.last_c2p_margin()
        assert margin > MARGIN_MIN, (f"oracle margin {margin}: a c2p decision sits on a threshold; "
                                     "bump the seed of this input (SURVEY.md C8 margin rule)")
        assert np.array_equal(interior(p, mask), interior(p, o.mask)), "stage-2 masks differ"
        assert np.array_equal(interior(p, mask1), interior(p, o.mask1)), "stage-1 masks differ"
    return err
