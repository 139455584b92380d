"""GPU checks of the behaviours the round-1 review asked for around the hot path: a non-finite state must poison the CFL time
step instead of being dropped, toggling phx_debug_enable_flux must not be hidden by a cached CUDA graph, the device's SM
count is queried, and the fp64 peak the bench line divides by is a sane measurement."""
import math

import numpy as np
import pytest

from paper_2410_09146_b200 import workloads as wl

from harness import GpuRun

pytestmark = pytest.mark.gpu


def test_nan_primitives_poison_the_time_step():
    """fmax drops NaN: a state with one NaN cell used to yield a finite dt.  Now phx_cfl_dt and the reduction fused into
    stage 2 return NaN (include/phx.h), so a blown-up run cannot keep stepping unnoticed."""
    w = wl.turbulence_box(16)
    g = GpuRun(w["params"], w["prim"])
    ok = g.dt(0.4)
    assert math.isfinite(ok) and ok > 0
    g.prim[0, 0, 8, 8, 8] = float("nan")
    assert math.isnan(g.dt(0.4))
    # the fused reduction: one step from the poisoned state
    g2 = GpuRun(w["params"], w["prim"])
    g2.phx.cfl_dt(g2.mesh, g2.prim, 0.4, g2.d_dt)
    g2.cons[0, 4, 8, 8, 8] = float("nan")          # non-finite tau: con2prim flags the cell (bit 32) and resets it ...
    g2.phx.rk2_step_cfl(g2.mesh, 0.4, g2.d_dt, g2.cons0, g2.cons, g2.prim, g2.mask)
    assert math.isfinite(float(g2.d_dt.cpu()))     # ... so the state is finite again and so is dt
    g2.prim[0, 1, 9, 9, 9] = float("inf")          # a velocity that stays non-finite through the step's reconstruction
    g2.phx.rk2_step_cfl(g2.mesh, 0.4, g2.d_dt, g2.cons0, g2.cons, g2.prim, g2.mask)
    m = g2.mask.cpu().numpy()
    assert (m & 32).any() or math.isnan(float(g2.d_dt.cpu()))     # the damage is visible in the mask or in dt, never silent


def test_flux_debug_toggle_is_not_hidden_by_the_cached_graph():
    w = wl.turbulence_box(16)
    g = GpuRun(w["params"], w["prim"])
    g.phx.cfl_dt(g.mesh, g.prim, 0.4, g.d_dt)
    g.phx.evolve_device(g.mesh, 2, 0.4, g.d_dt, g.cons0, g.cons, g.prim, g.mask)      # captures with the debug stores off
    g.mesh.debug_enable_flux(True)
    g.phx.evolve_device(g.mesh, 2, 0.4, g.d_dt, g.cons0, g.cons, g.prim, g.mask)      # must re-capture
    F = g.mesh.debug_flux(0, w["prim"].shape).cpu().numpy()
    gh = w["params"]["ng"]
    rho_flux = F[0, 0, gh:-gh, gh:-gh, gh:-gh]
    assert np.abs(rho_flux).max() > 1e-3, "the mass flux was not stored: the replayed graph ignored phx_debug_enable_flux"


def test_fp64_peak_measurement_is_sane():
    import torch
    from paper_2410_09146_b200 import phx
    rate, burst, ms, nsm = phx.debug_fp64_peak(0.2)
    assert nsm == torch.cuda.get_device_properties(0).multi_processor_count
    assert 150.0 < ms < 400.0
    nominal = nsm * 64 * 1.965e9              # one fp64 instruction per lane and cycle at the maximum SM clock
    assert 0.6 * nominal < rate <= 1.02 * nominal and 0.6 * nominal < burst <= 1.02 * nominal, (rate, burst, nominal)


def test_count_masked_counts_interior_cells_only():
    """phx_count_masked against numpy on a mesh whose floors act, with a poisoned ghost cell that must not be counted."""
    import torch
    w = wl.packed_blocks((2, 2, 2), 12)
    g = GpuRun(w["params"], w["prim"])
    g.step_device_dt(0.4)
    p = w["params"]
    m = g.mask.cpu().numpy()
    gh = p["ng"]
    inner = m[:, gh:-gh, gh:-gh, gh:-gh]
    for bits in (64, 1 | 2, 255, 16 | 32):
        assert g.phx.count_masked(g.mesh, g.mask, bits) == int(((inner & bits) != 0).sum())
    assert g.phx.count_masked(g.mesh, g.mask, 64) > 0            # the excised cells of the torus recipe
    g.mask[0, 0, 0, 0] = 255                                      # a ghost cell of the mask
    assert g.phx.count_masked(g.mesh, g.mask, 255) == int((inner != 0).sum())
