"""One RK2 step of the CUDA path against the oracle over the template matrix of the kernels: every metric x every
reconstruction x both Riemann solvers, with flux-CT on and off, with and without the passive scalar, with constant and
position-dependent floors, on single blocks and packed blocks, in 3-D and 2-D.  Each combination instantiates different
kernels (k_sweep_x / k_sweep_march<METRIC, RECON, D, NS>, k_update<METRIC, EXC, CFL, NS, RF>); the workloads elsewhere in
the suite cover the combinations BASELINE.json names, this file the rest.  Tolerance: BASELINE.json's 1e-11 per conserved
variable after one step, identical masks of both stages, and the fused CFL time step against the oracle's."""
import itertools

import numpy as np
import pytest

from oracle import orc
from paper_2410_09146_b200 import workloads as wl

from harness import GpuRun, TOL_1STEP, compare, run_both

pytestmark = pytest.mark.gpu

METRICS = {"minkowski": 0, "kerr_schild": 1, "boosted": 2}


def make(metric, recon, riemann, use_ct, scalar, floor_form, blocks, twod):
    """A small strongly nonlinear state on the requested mesh: the config-4 recipe for the flat metrics, the torus for Kerr-Schild."""
    ng = 3 if recon >= 3 else 2
    if metric == "kerr_schild":
        w = wl.packed_blocks((2, 2, 1), 8) if blocks else wl.kerr_schild_torus(12)
        p = dict(w["params"], recon=recon, riemann=riemann, use_ct=use_ct, ng=4)
        prim = w["prim"]
        assert not twod, "the Kerr-Schild recipes are 3-D"
    else:
        n = 12
        w = wl.turbulence_box(n, recon=recon, riemann=riemann)
        p = dict(w["params"], use_ct=use_ct)
        if metric == "boosted":
            p.update(metric=wl.MINKOWSKI_BOOSTED, shift=(0.3, -0.2, 0.1))
        q = wl.from_blocks(p, w["prim"])
        if twod:
            q = q[:, :1]                       # one k-plane: z inactive
            p.update(nz=1)
        if blocks:
            p2 = dict(p)
            p2.update(nbx=2, nby=2 if not twod else 1, nbz=1, nx=n // 2, ny=(n // 2 if not twod else n))
            p = p2
        prim = wl.finish(p, q)
    w2 = dict(name="matrix", params=p, prim=prim, cfl=0.4)
    if floor_form:
        q = wl.from_blocks(p, prim)
        fl = dict(floor_form=floor_form, floor_alpha_rho=1.0, floor_alpha_eps=0.5,
                  rho_floor=0.3 * float(q[0].min()), eps_floor=0.3 * float((q[4] / q[0]).min()))
        w2 = dict(w2, params=dict(p, **fl))
    if scalar:
        w2 = wl.with_scalar(w2, wl.smooth_scalar(w2["params"], 5))
    return w2


# a covering subset of the full product (3 x 6 x 2 x 2 x 2 x 3 x 2 x 2 = 1728): every pair (metric, recon) appears, and every
# other switch appears with every metric
def combos():
    out = []
    rng = np.random.default_rng(2410)
    for metric, recon in itertools.product(METRICS, range(6)):
        riemann = int(rng.integers(0, 2)); use_ct = int(rng.integers(0, 2)); scalar = int(rng.integers(0, 2))
        floor_form = int(rng.choice([0, 1, 3])); blocks = int(rng.integers(0, 2)); twod = int(rng.integers(0, 4) == 0)
        if metric == "kerr_schild":
            twod = 0                      # the Kerr-Schild recipes are 3-D
        out.append((metric, recon, riemann, use_ct, scalar, floor_form, blocks, twod))
    for metric in METRICS:          # the switches the draw above may have left out for a metric
        out += [(metric, 2, 0, 1, 1, 3, 1, 0), (metric, 3, 1, 0, 0, 1, 0, 0), (metric, 1, 1, 1, 1, 0, 1, int(metric != "kerr_schild"))]
    return out


@pytest.mark.parametrize("metric,recon,riemann,use_ct,scalar,floor_form,blocks,twod", combos())
def test_one_step_over_the_kernel_template_matrix(metric, recon, riemann, use_ct, scalar, floor_form, blocks, twod):
    w = make(metric, recon, riemann, use_ct, scalar, floor_form, blocks, twod)
    p = w["params"]
    o, g = run_both(p, w["prim"], nsteps=1, cfl=0.4)
    err = compare(p, o, g, TOL_1STEP)
    assert abs(g.dt(0.4) - o.dt(0.4)) <= 1e-12 * o.dt(0.4)
    # the same step in the launch configuration bench.py times (fused CFL reduction, dt on the device): same bits as the stages
    g2 = GpuRun(p, w["prim"])
    g2.step_fused_cfl(0.4, first=True)
    c1 = g.get()[0]; c2 = g2.get()[0]
    assert np.abs(c1 - c2).max() <= 1e-13 * np.abs(c1).max()     # the oracle's dt and the device's differ in the last bits
    g.mesh.free(); g2.mesh.free()
