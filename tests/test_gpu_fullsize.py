"""Full-size GPU parity: BASELINE.json's configs at their full sizes, in the launch configuration bench.py times
(phx_cfl_dt once, then phx_rk2_step_cfl with the time step kept on the device), checked

  (i)  on sampled outputs the oracle can compute one by one: the update of a cell depends on the primitives within
       HALO = 8 cells (two stages x (3 cells of WENO5 stencil to a face + 1 transverse cell of flux-CT)), so the oracle
       run on a (16+2*HALO)^3 sub-box cut around a sample point reproduces the central 16^3 cells of the full run
       exactly (sub-box faces that coincide with an outflow domain face carry the true boundary condition and are
       valid up to the face); and
  (ii) via properties that hold at any size: corner-centred div(sqrt(gamma) B) unchanged, totals conserved on the
       periodic box, state finite, no con2prim failure bits.

Tolerance: BASELINE.json's 1e-11 relative per conserved variable after one RK2 step, scale = max |U~_v| over the whole
mesh (SURVEY.md 8c error metric), identical masks on the sampled cells.
"""
import numpy as np
import pytest

from oracle import orc
from paper_2410_09146_b200 import workloads as wl

from harness import GpuRun, TOL_1STEP

pytestmark = pytest.mark.gpu

HALO = 8
CORE = 16


def sub_box(p, q_glob, origin):
    """Cut a (CORE+2*HALO)^3 box with lower corner `origin` (global interior indices, x y z) out of the global interior
    array q_glob [8, Nz, Ny, Nx]; periodic axes wrap, outflow axes must stay inside the domain.  Returns (p_sub, prim)."""
    s = CORE + 2 * HALO
    N = (q_glob.shape[3], q_glob.shape[2], q_glob.shape[1])
    idx = []
    for d in range(3):
        i = np.arange(origin[d], origin[d] + s)
        if p["bc"][d][0] == wl.BC_PERIODIC:
            i = i % N[d]
        assert i.min() >= 0 and i.max() < N[d]
        idx.append(i)
    q = q_glob[:, idx[2]][:, :, idx[1]][:, :, :, idx[0]]
    ps = dict(p)
    dx = [(p["xmax"][d] - p["xmin"][d]) / N[d] for d in range(3)]
    ps.update(nbx=1, nby=1, nbz=1, nx=s, ny=s, nz=s,
              xmin=tuple(p["xmin"][d] + origin[d] * dx[d] for d in range(3)),
              xmax=tuple(p["xmin"][d] + (origin[d] + s) * dx[d] for d in range(3)))
    return ps, wl.finish(ps, np.ascontiguousarray(q))


def valid_range(p, origin, N):
    """Per axis: slice of sub-box interior cells whose full-mesh update the sub-box reproduces."""
    s = CORE + 2 * HALO
    out = []
    for d in range(3):
        lo, hi = HALO, s - HALO
        if p["bc"][d][0] == wl.BC_OUTFLOW:
            if origin[d] == 0:
                lo = 0
            if origin[d] + s == N[d]:
                hi = s
        out.append(slice(lo, hi))
    return out


def corner_div(Bt, rdx):
    """Corner-centred divergence of a densitised field, numpy [3, Nz, Ny, Nx] -> [Nz-1, Ny-1, Nx-1]."""
    def mu(a, ax):
        n = a.shape[ax]
        return 0.5 * (np.take(a, range(0, n - 1), axis=ax) + np.take(a, range(1, n), axis=ax))

    def de(a, ax):
        n = a.shape[ax]
        return np.take(a, range(1, n), axis=ax) - np.take(a, range(0, n - 1), axis=ax)
    X, Y, Z = 2, 1, 0
    return (de(mu(mu(Bt[0], Y), Z), X) * rdx[0] + de(mu(mu(Bt[1], X), Z), Y) * rdx[1] + de(mu(mu(Bt[2], X), Y), Z) * rdx[2])


def run_full(w, origins, check_conservation):
    import torch
    p = w["params"]
    q_glob = wl.from_blocks(p, w["prim"])
    N = (q_glob.shape[3], q_glob.shape[2], q_glob.shape[1])
    g = GpuRun(p, w["prim"])
    gx, gy, gz = wl.ghosts(p)
    rdx = [N[d] / (p["xmax"][d] - p["xmin"][d]) for d in range(3)]
    c0 = wl.from_blocks(p, g.cons.cpu().numpy())
    div0 = corner_div(c0[5:8], rdx)
    dt_ref = orc.cfl_dt(p, w["prim"], w["cfl"])
    g.phx.cfl_dt(g.mesh, g.prim, w["cfl"], g.d_dt)
    dt_gpu = float(g.d_dt.cpu())
    assert abs(dt_gpu - dt_ref) <= 1e-13 * dt_ref
    g.step_fused_cfl(w["cfl"], first=False)          # phx_rk2_step_cfl with the device dt: what bench.py times
    dt_next = float(g.d_dt.cpu())
    assert dt_next == g.dt(w["cfl"])                 # fused reduction = phx_cfl_dt on the new state, bit for bit
    cons, prim, _, mask = g.get()
    assert np.isfinite(cons[:, :, gz:gz + p["nz"], gy:gy + p["ny"], gx:gx + p["nx"]]).all()
    assert not (mask & (16 | 32)).any(), "con2prim failure bits at full size"
    cg = wl.from_blocks(p, cons)
    mg = wl.from_blocks(p, mask[:, None])[0]
    nv = cg.shape[0]
    scale = np.abs(cg).reshape(nv, -1).max(axis=1)
    scale = np.where(scale > 0.0, scale, 1.0)          # B = 0 workloads
    ddiv = np.abs(corner_div(cg[5:8], rdx) - div0).max()
    bscale = np.abs(c0[5:8]).max() * max(rdx)
    assert ddiv <= 1e-13 * bscale, f"corner div B changed by {ddiv} (scale {bscale})"
    if check_conservation:
        rel = np.abs(np.sum(cg - c0, axis=(1, 2, 3), dtype=np.longdouble)) / np.sum(np.abs(c0), axis=(1, 2, 3))
        assert rel.max() <= 1e-13, f"totals drifted by {rel}"
    del c0, div0
    worst = np.zeros(nv)
    for origin in origins:
        ps, sprim = sub_box(p, q_glob, origin)
        orc.reset_c2p_margin()
        o = orc.Run(ps, sprim)
        o.step(dt_ref)
        assert orc.last_c2p_margin() > 1e-9
        oc = wl.from_blocks(ps, o.cons); om = wl.from_blocks(ps, o.mask[:, None])[0]
        vr = valid_range(p, origin, N)
        sl_sub = (slice(None), vr[2], vr[1], vr[0])
        gi = [np.arange(origin[d] + vr[d].start, origin[d] + vr[d].stop) % N[d] for d in range(3)]
        got = cg[:, gi[2]][:, :, gi[1]][:, :, :, gi[0]]
        gm = mg[gi[2]][:, gi[1]][:, :, gi[0]]
        err = np.abs(got - oc[sl_sub]).reshape(nv, -1).max(axis=1) / scale
        worst = np.maximum(worst, err)
        assert err.max() <= TOL_1STEP, f"sub-box at {origin}: errors {err}"
        assert np.array_equal(gm, om[sl_sub[1:]]), f"sub-box at {origin}: masks differ"
    print(w["name"], "full size, worst sampled error per variable", worst)
    g.mesh.free()
    del g
    torch.cuda.empty_cache()


def test_cfg4_turbulence_256_sampled():
    """BASELINE.json configs[3], the bench workload: 256^3 periodic, WENO5-Z + HLL + flux-CT."""
    w = wl.turbulence_box(256)
    n, s = 256, CORE + 2 * HALO
    origins = [(0, 0, 0), (n - HALO - 3, 100, n - 20), (117, n - s // 2, 5), (64, 200, 131), (201, 37, 88)]
    run_full(w, origins, check_conservation=True)


def test_cfg2_periodic_box_64_sampled():
    """BASELINE.json configs[1]: 64^3 periodic, PLM-MC + LLF + flux-CT."""
    w = wl.periodic_box(64)
    run_full(w, [(0, 0, 0), (50, 20, 40), (30, 60, 7)], check_conservation=True)


def test_cfg3_kerr_schild_128_sampled():
    """BASELINE.json configs[2]: 128^3 Kerr-Schild torus with excision (sub-boxes: a domain corner with its outflow
    faces, the excised region at the centre, the torus body)."""
    w = wl.kerr_schild_torus(128)
    n, s = 128, CORE + 2 * HALO
    run_full(w, [(0, 0, 0), (n - s, n - s, n - s), (48, 48, 48), (80, 50, 52), (20, 60, 56)], check_conservation=False)


def test_cfg5_packed_blocks_512x32_sampled():
    """BASELINE.json configs[4]: 512 blocks of 32^3 in one batched launch per kernel; sub-boxes straddle block faces,
    edges and corners (the oracle runs them as one block: block invariance is pin P11)."""
    w = wl.packed_blocks((8, 8, 8), 32)
    n, s = 256, CORE + 2 * HALO
    run_full(w, [(0, 0, 0), (n - s, n - s, n - s), (112, 112, 112), (16, 48, 80), (150, 100, 120), (176, 16, 208)],
             check_conservation=False)


def test_next1_turbulence_256_aoah_sampled():
    """SURVEY.md 8(f) rank 1 at the bench size: config 4's box with WENO5-Z-AOAH (App.B B16-B18)."""
    w = wl.turbulence_box(256, recon=wl.RECON_WENO5Z_AOAH)
    n = 256
    run_full(w, [(0, 0, 0), (n - HALO - 5, 31, 140), (90, 180, n - 12)], check_conservation=True)


def test_next2_sedov_128_sampled():
    """SURVEY.md 8(f) rank 2 at the paper's size (3-D Sedov, 128^3): the deposit region, the domain
    corner with its outflow faces, and the quiescent ambient medium."""
    w = wl.sedov_blast(128)
    n, s = 128, CORE + 2 * HALO
    run_full(w, [(48, 48, 48), (0, 0, 0), (n - s, 40, 60), (56, 60, 44)], check_conservation=False)


def test_next3_packed_blocks_scalar_radial_floors_sampled():
    """SURVEY.md 8(f) rank 3 at config 5's size: 512 blocks of 32^3 carrying the passive scalar of Eq.14 with the floors
    rho0 r^-2, eps0 r^-1; nine variables and the masks (floor bits near the hole, excision) on sub-boxes
    around the hole, at a domain corner and across block corners."""
    w = wl.packed_blocks((8, 8, 8), 32)
    w = dict(w, params=dict(w["params"], floor_form=3, rho_floor=1e-2, eps_floor=1e-2, floor_alpha_rho=2.0, floor_alpha_eps=1.0))
    w = wl.with_scalar(w, wl.smooth_scalar(w["params"], wl.SEED0 + 9))
    n, s = 256, CORE + 2 * HALO
    run_full(w, [(112, 112, 112), (0, 0, 0), (n - s, n - s, n - s), (100, 120, 90), (176, 16, 208)], check_conservation=False)


def test_largest_mesh_indexing_beyond_2_to_31_elements():
    """Maximum size: one 1024 x 1024 x 256 block (2.25e9 doubles per field, 18 GB; the whole state with flux scratch is
    108 GB of the 180 GB) so that element offsets exceed 2^31 in every kernel.  Inputs are analytic smooth periodic fields
    written on the device (workloads.smooth_periodic_prims); one RK2 step with a fixed dt; the oracle reproduces sampled
    16^3 cores from (16+2*HALO)^3 sub-boxes cut out of the initial state, including cells of the last variables at high k
    whose offsets lie beyond 2^31."""
    import torch
    from paper_2410_09146_b200 import phx
    free, total = torch.cuda.mem_get_info()
    if free < 125e9:
        pytest.skip("needs ~110 GB of free device memory")
    n = (1024, 1024, 256)
    p = wl.default_params(nx=n[0], ny=n[1], nz=n[2], ng=4, recon=wl.RECON_PLM_MC, riemann=wl.RIEMANN_HLL, gamma_ad=5.0 / 3.0,
                          xmax=(4.0, 4.0, 1.0))
    prim = wl.smooth_periodic_prims(p, "cuda")
    assert prim.numel() > 2 ** 31
    mesh = phx.init_mesh(p)
    cons = torch.empty_like(prim); cons0 = torch.empty_like(prim)
    mask = torch.zeros((1,) + tuple(prim.shape[2:]), dtype=torch.uint8, device="cuda")
    d_dt = torch.zeros(1, dtype=torch.float64, device="cuda")
    s = CORE + 2 * HALO
    g = p["ng"]
    origins = [(0, 0, 0), (n[0] - s + 5, n[1] - s + 3, n[2] - s + 7), (500, 1000, 236), (1010, 17, 200), (333, 777, 120)]
    subs = []
    for o in origins:       # sub-boxes of the initial state (periodic wrap), pulled to the host before the step
        idx = [(torch.arange(o[d], o[d] + s, device="cuda") % n[d]) + g for d in range(3)]
        q = prim[0][:, idx[2]][:, :, idx[1]][:, :, :, idx[0]].cpu().numpy()
        dx = [(p["xmax"][d] - p["xmin"][d]) / n[d] for d in range(3)]
        ps = dict(p, nx=s, ny=s, nz=s, xmin=tuple(p["xmin"][d] + o[d] * dx[d] for d in range(3)),
                  xmax=tuple(p["xmin"][d] + (o[d] + s) * dx[d] for d in range(3)))
        subs.append((ps, wl.finish(ps, np.ascontiguousarray(q))))
    dt = 0.2 * (p["xmax"][0] - p["xmin"][0]) / n[0]          # all signal speeds are below 1
    phx.prim_to_cons(mesh, prim, cons)
    d_dt.fill_(dt)
    phx.rk2_step(mesh, d_dt, cons0, cons, prim, mask)
    torch.cuda.synchronize()
    assert not bool(mask.bitwise_and(16 | 32).any())
    scale = cons[0].abs().amax(dim=(1, 2, 3)).cpu().numpy()
    for o, (ps, sprim) in zip(origins, subs):
        orc.reset_c2p_margin()
        r = orc.Run(ps, sprim)
        r.step(dt)
        assert orc.last_c2p_margin() > 1e-9
        oc = wl.from_blocks(ps, r.cons)[:, HALO:HALO + CORE, HALO:HALO + CORE, HALO:HALO + CORE]
        om = wl.from_blocks(ps, r.mask[:, None])[0][HALO:HALO + CORE, HALO:HALO + CORE, HALO:HALO + CORE]
        idx = [(torch.arange(o[d] + HALO, o[d] + HALO + CORE, device="cuda") % n[d]) + g for d in range(3)]
        got = cons[0][:, idx[2]][:, :, idx[1]][:, :, :, idx[0]].cpu().numpy()
        gm = mask[0][idx[2]][:, idx[1]][:, :, idx[0]].cpu().numpy()
        err = np.abs(got - oc).reshape(8, -1).max(axis=1) / scale
        assert err.max() <= TOL_1STEP, f"sub-box at {o}: errors {err}"
        assert np.array_equal(gm, om)
    # the last cell of the last variable sits beyond 2^31 elements and was written
    flat_last = ((7 * prim.shape[2] + (n[2] + g - 1)) * prim.shape[3] + (n[1] + g - 1)) * prim.shape[4] + (n[0] + g - 1)
    assert flat_last > 2 ** 31
    mesh.free()
    del prim, cons, cons0, mask
    torch.cuda.empty_cache()


@pytest.mark.parametrize("cfg", ["cfg2", "cfg3", "cfg4", "cfg5"])
def test_baseline_configs_run_their_full_step_counts(cfg):
    """BASELINE.json configs[1..4] at full size for their full step counts (100, 50, 20, 20) through phx_evolve_device (the
    graph-replayed step loop), checked by properties that hold at any size: corner-centred div(sqrt(gamma) B) stays at its
    initial value, totals are conserved on the periodic boxes, the state stays finite with no con2prim failure, excised
    cells stay frozen bit for bit."""
    import torch
    w = {"cfg2": lambda: wl.periodic_box(64), "cfg3": lambda: wl.kerr_schild_torus(128), "cfg4": lambda: wl.turbulence_box(256),
         "cfg5": lambda: wl.packed_blocks((8, 8, 8), 32)}[cfg]()
    p = w["params"]
    g = GpuRun(p, w["prim"])
    N = (p["nbx"] * p["nx"], p["nby"] * p["ny"], p["nbz"] * p["nz"])
    rdx = [N[d] / (p["xmax"][d] - p["xmin"][d]) for d in range(3)]
    c0 = wl.from_blocks(p, g.cons.cpu().numpy())
    div0 = corner_div(c0[5:8], rdx)
    d_t = torch.zeros(1, dtype=torch.float64, device="cuda")
    g.phx.cfl_dt(g.mesh, g.prim, w["cfl"], g.d_dt)
    g.phx.evolve_device(g.mesh, w["steps"], w["cfl"], g.d_dt, g.cons0, g.cons, g.prim, g.mask, d_t=d_t)
    cons, prim, _, mask = g.get()
    c1 = wl.from_blocks(p, cons)
    m = wl.from_blocks(p, mask[:, None])[0]
    assert float(d_t.cpu()) > 0.0 and np.isfinite(c1).all()
    assert not (m & (16 | 32)).any(), "con2prim failure bits"
    bscale = np.abs(c0[5:8]).max() * max(rdx)
    ddiv = np.abs(corner_div(c1[5:8], rdx) - div0).max()
    assert ddiv <= 1e-12 * bscale, f"corner div B drifted by {ddiv} (scale {bscale}) over {w['steps']} steps"
    assert np.abs(c1 - c0).max() > 1e-8, "nothing happened"
    if p["bc"][0][0] == wl.BC_PERIODIC:
        rel = np.abs(np.sum(c1 - c0, axis=(1, 2, 3), dtype=np.longdouble)) / np.sum(np.abs(c0), axis=(1, 2, 3))
        assert rel.max() <= 1e-12, f"totals drifted by {rel}"
        assert not m.any()
    else:
        ex = (m & 64) != 0
        assert ex.any() and np.array_equal(c1[:, ex], c0[:, ex]), "excised cells must stay frozen"
    print(cfg, w["steps"], "steps to t =", float(d_t.cpu()), "div B drift", ddiv / bscale, "mask bits", int(np.bitwise_or.reduce(m.ravel())))
    g.mesh.free()
    del g
    torch.cuda.empty_cache()
