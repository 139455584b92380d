"""phx_evolve_device: `nsteps` RK2 steps replayed from a CUDA graph - or, on a small 1-D mesh, run inside one launch of one
thread block - must give the bits of `nsteps` phx_rk2_step_cfl calls, on the default stream and on a side stream, with the
graph cached and re-captured when the arguments change."""
import numpy as np
import pytest

from paper_2410_09146_b200 import workloads as wl

from harness import GpuRun

pytestmark = pytest.mark.gpu


def _reference(w, nsteps):
    g = GpuRun(w["params"], w["prim"])
    t = 0.0
    g.phx.cfl_dt(g.mesh, g.prim, w["cfl"], g.d_dt)
    for _ in range(nsteps):
        t += float(g.d_dt.cpu())
        g.phx.rk2_step_cfl(g.mesh, w["cfl"], g.d_dt, g.cons0, g.cons, g.prim, g.mask)
    return g.get(), float(g.d_dt.cpu()), t


@pytest.mark.parametrize("name", ["shock_tube", "turbulence", "blocks", "scalar_blocks"])
def test_graph_replay_equals_step_calls(name):
    import torch
    w = {"shock_tube": lambda: wl.shock_tube(256), "turbulence": lambda: wl.turbulence_box(20),
         "blocks": lambda: wl.packed_blocks((2, 1, 2), 8),
         "scalar_blocks": lambda: wl.with_scalar(wl.packed_blocks((2, 1, 2), 8), np.full((16, 8, 16), 0.25))}[name]()
    n = 7
    (cr, pr, _, mr), dt_r, t_r = _reference(w, n)
    for use_side_stream in (False, True):
        g = GpuRun(w["params"], w["prim"])
        d_t = torch.zeros(1, dtype=torch.float64, device="cuda")
        st = torch.cuda.Stream() if use_side_stream else torch.cuda.current_stream()
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            g.phx.cfl_dt(g.mesh, g.prim, w["cfl"], g.d_dt, stream=st)
            l0 = g.mesh.launch_count()
            g.phx.evolve_device(g.mesh, 3, w["cfl"], g.d_dt, g.cons0, g.cons, g.prim, g.mask, d_t=d_t, stream=st)   # captures
            l1 = g.mesh.launch_count()
            g.phx.evolve_device(g.mesh, n - 3, w["cfl"], g.d_dt, g.cons0, g.cons, g.prim, g.mask, d_t=d_t, stream=st)  # cached graph
            l2 = g.mesh.launch_count()
        st.synchronize()
        c, p, _, m = g.get()
        assert np.array_equal(c, cr) and np.array_equal(p, pr) and np.array_equal(m, mr)
        assert float(g.d_dt.cpu()) == dt_r
        assert abs(float(d_t.cpu()) - t_r) <= 1e-15 * t_r
        if name == "shock_tube":      # a small 1-D mesh: all steps of a call run in one launch of one thread block (k_evolve_1d)
            assert l1 - l0 == 1 and l2 - l1 == 1
        else:
            assert (l1 - l0) * (n - 3) == (l2 - l1) * 3 and l1 > l0        # replays are counted as the launches they stand for


def test_graph_is_recaptured_when_the_arguments_change():
    import torch
    w = wl.turbulence_box(16)
    (cr, pr, _, mr), dt_r, _ = _reference(w, 4)
    g = GpuRun(w["params"], w["prim"])
    other = torch.empty_like(g.cons0)
    g.phx.cfl_dt(g.mesh, g.prim, w["cfl"], g.d_dt)
    g.phx.evolve_device(g.mesh, 2, w["cfl"], g.d_dt, g.cons0, g.cons, g.prim, g.mask)
    g.phx.evolve_device(g.mesh, 2, w["cfl"], g.d_dt, other, g.cons, g.prim, g.mask)       # another scratch field: new capture
    c, p, _, m = g.get()
    assert np.array_equal(c, cr) and np.array_equal(p, pr) and np.array_equal(m, mr) and float(g.d_dt.cpu()) == dt_r
    with pytest.raises(g.phx.PhxError):
        g.phx.evolve_device(g.mesh, 2, w["cfl"], g.d_dt, g.cons, g.cons, g.prim, g.mask)  # aliased scratch


@pytest.mark.parametrize("case", ["shock_tube_plm_256", "shock_tube_weno_200", "shock_tube_aoah_97", "shock_tube_mp5_510", "shock_tube_const_33",
                                  "periodic_fast_wave_mc_64", "periodic_alfven_wave_weno_129", "llf_shock_tube_300"])
def test_one_block_path_of_small_1d_meshes_equals_step_calls(case):
    """k_evolve_1d (one thread block owns the mesh and loops over the steps on the device) against the general multi-kernel
    path, bit for bit: every reconstruction, outflow and periodic ghosts, LLF and HLL, sizes that are no multiple of the
    warp size and the largest one the path takes."""
    import torch
    w = {"shock_tube_plm_256": lambda: wl.shock_tube(256),
         "shock_tube_weno_200": lambda: wl.shock_tube(200, recon=wl.RECON_WENO5Z, ng=3),
         "shock_tube_aoah_97": lambda: wl.shock_tube(97, recon=wl.RECON_WENO5Z_AOAH, ng=4),
         "shock_tube_mp5_510": lambda: wl.shock_tube(510, recon=wl.RECON_MP5, ng=3),
         "shock_tube_const_33": lambda: wl.shock_tube(33, recon=wl.RECON_CONST, ng=2),
         "periodic_fast_wave_mc_64": lambda: wl.linear_wave_1d(64, "fast", A=1e-2),
         "periodic_alfven_wave_weno_129": lambda: wl.linear_wave_1d(129, "alfven", A=1e-2, recon=wl.RECON_WENO5Z),
         "llf_shock_tube_300": lambda: wl.shock_tube(300)}[case]()
    if case.startswith("llf"):
        w = dict(w, params=dict(w["params"], riemann=wl.RIEMANN_LLF))
    n = 40
    (cr, pr, _, mr), dt_r, t_r = _reference(w, n)
    g = GpuRun(w["params"], w["prim"])
    d_t = torch.zeros(1, dtype=torch.float64, device="cuda")
    g.phx.cfl_dt(g.mesh, g.prim, w["cfl"], g.d_dt)
    l0 = g.mesh.launch_count()
    g.phx.evolve_device(g.mesh, n, w["cfl"], g.d_dt, g.cons0, g.cons, g.prim, g.mask, d_t=d_t)
    assert g.mesh.launch_count() - l0 == 1, "the one-block path was not taken"
    c, p, _, m = g.get()
    assert np.array_equal(c, cr) and np.array_equal(p, pr) and np.array_equal(m, mr)
    assert float(g.d_dt.cpu()) == dt_r and abs(float(d_t.cpu()) - t_r) <= 1e-15 * t_r


def test_meshes_the_one_block_path_does_not_take_still_replay_the_graph():
    """Too long for one block, more than one block, or carrying a passive scalar: the graph path, same bits."""
    for w in (wl.shock_tube(511), wl.with_scalar(wl.shock_tube(64), np.linspace(0.1, 0.9, 64)[None, None, :])):
        n = 6
        (cr, pr, _, mr), dt_r, _ = _reference(w, n)
        g = GpuRun(w["params"], w["prim"])
        g.phx.cfl_dt(g.mesh, g.prim, w["cfl"], g.d_dt)
        l0 = g.mesh.launch_count()
        g.phx.evolve_device(g.mesh, n, w["cfl"], g.d_dt, g.cons0, g.cons, g.prim, g.mask)
        assert g.mesh.launch_count() - l0 > n
        c, p, _, m = g.get()
        assert np.array_equal(c, cr) and np.array_equal(p, pr) and np.array_equal(m, mr)
