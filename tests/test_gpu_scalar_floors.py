"""GPU parity for SURVEY.md 8(f) rank 3: the passive scalar of Eq.14 carried as variable 8, and the
radial floor forms of PAPER.md:288-290.  Same bar as test_gpu_parity.py: <= 1e-11 relative per conserved variable
(now nine of them) after one RK2 step, <= 1e-8 after many, identical masks including the scalar-clipped bit 128.
"""
import numpy as np
import pytest

from oracle import orc
from paper_2410_09146_b200 import workloads as wl

from harness import GpuRun, MARGIN_MIN, TOL_100STEP, TOL_1STEP, compare, interior, run_both

pytestmark = pytest.mark.gpu

FLOORS_R2 = dict(floor_form=3, rho_floor=1e-2, eps_floor=1e-2, floor_alpha_rho=2.0, floor_alpha_eps=1.0)


def _gpu():
    import torch
    from paper_2410_09146_b200 import phx
    assert torch.cuda.is_available(), "these tests must run on the GPU box"
    return torch, phx


def _with_params(w, **kw):
    return dict(w, params=dict(w["params"], **kw))


def _scales(a):
    """Per-variable magnitude over the cells; the three components of a vector share the largest of theirs (the torus
    data have u~^z = 0 exactly, where a component-wise scale would be zero)."""
    sc = np.abs(a).max(axis=(1, 2, 3))
    for g in ((1, 2, 3), (5, 6, 7)):
        sc[list(g)] = sc[list(g)].max()
    return sc[:, None, None, None]


def scalar_workloads():
    out = {}
    w = wl.turbulence_box(24)
    out["turb_24_weno_scalar"] = wl.with_scalar(w, wl.smooth_scalar(w["params"], 1))
    w = wl.periodic_box(20)
    out["box_20_mc_llf_scalar"] = wl.with_scalar(w, wl.smooth_scalar(w["params"], 2))
    w = wl.turbulence_box(20, recon=wl.RECON_WENO5Z_AOAH)
    out["turb_20_aoah_scalar"] = wl.with_scalar(w, wl.smooth_scalar(w["params"], 3))
    w = wl.turbulence_box(16, recon=wl.RECON_MP5)
    out["turb_16_mp5_scalar"] = wl.with_scalar(w, wl.smooth_scalar(w["params"], 4))
    # shock tube with the scalar jumping at the membrane: it must follow the contact discontinuity
    w = wl.shock_tube(256)
    x = wl.cell_centres(w["params"])[0]
    out["shock_tube_256_scalar"] = wl.with_scalar(w, np.where(x < 0.5, 0.45, 0.1)[None, None, :])
    # Kerr-Schild: torus with the scalar and the radial floors (the density floor acts inside r ~ 10, the energy floor inside r ~ 7), single block and packed blocks
    w = _with_params(wl.kerr_schild_torus(24), **FLOORS_R2)
    out["ks_torus_24_scalar_rfloor"] = wl.with_scalar(w, wl.smooth_scalar(w["params"], 5))
    w = _with_params(wl.packed_blocks((2, 2, 2), 12), **FLOORS_R2)
    out["blocks_2x2x2_of_12_scalar_rfloor"] = wl.with_scalar(w, wl.smooth_scalar(w["params"], 6))
    # floors alone: exponential form on the torus, power law with WENO5-Z (position-dependent positivity fallback)
    out["ks_torus_20_expfloor"] = _with_params(wl.kerr_schild_torus(20), floor_form=1, rho_floor=1e-2, eps_floor=1e-2,
                                               floor_alpha_rho=0.5, floor_alpha_eps=0.25)
    out["ks_torus_20_weno_rfloor"] = _with_params(wl.kerr_schild_torus(20, recon=wl.RECON_WENO5Z), **FLOORS_R2)
    return out


WORKLOADS = scalar_workloads()


@pytest.mark.parametrize("name", list(WORKLOADS))
def test_one_rk2_step_matches_oracle(name):
    w = WORKLOADS[name]
    o, g = run_both(w["params"], w["prim"], nsteps=1, cfl=w["cfl"])
    err = compare(w["params"], o, g, TOL_1STEP)
    if "rfloor" in name or "expfloor" in name:
        m = interior(w["params"], o.mask)
        assert (m & 1).any() and not (m & 1).all(), "the radial floor should act in part of the domain only"
    print(name, "err", err)


@pytest.mark.parametrize("name,nsteps", [("turb_24_weno_scalar", 20), ("shock_tube_256_scalar", 100),
                                         ("blocks_2x2x2_of_12_scalar_rfloor", 20), ("ks_torus_20_weno_rfloor", 20)])
def test_many_steps_match_oracle(name, nsteps):
    w = WORKLOADS[name]
    o, g = run_both(w["params"], w["prim"], nsteps=nsteps, cfl=w["cfl"])
    err = compare(w["params"], o, g, TOL_100STEP)
    print(name, nsteps, "steps err", err)


def test_scalar_does_not_change_the_other_variables_on_gpu():
    """The eight GRMHD variables of a run with the scalar equal those of the run without it bit for bit."""
    w9 = WORKLOADS["turb_24_weno_scalar"]
    w8 = wl.turbulence_box(24)
    a, b = GpuRun(w9["params"], w9["prim"]), GpuRun(w8["params"], w8["prim"])
    for first in (True, False):
        a.step_fused_cfl(0.4, first); b.step_fused_cfl(0.4, first)
    ca, pa, _, ma = a.get(); cb, pb, _, mb = b.get()
    assert np.array_equal(ca[:, :8], cb) and np.array_equal(pa[:, :8], pb) and np.array_equal(ma, mb)
    assert float(a.d_dt.cpu()) == float(b.d_dt.cpu())


def test_constant_scalar_stays_constant_on_gpu():
    w0 = wl.turbulence_box(24)
    w = wl.with_scalar(w0, np.full((24, 24, 24), 0.3))
    g = GpuRun(w["params"], w["prim"])
    for s in range(5):
        g.step_fused_cfl(0.4, s == 0)
    _, prim, _, mask = g.get()
    X = interior(w["params"], prim)[8]
    assert np.abs(X - 0.3).max() < 1e-13 and not (mask & 128).any()


def test_point_ops_with_scalar_match_oracle():
    torch, phx = _gpu()
    w = WORKLOADS["blocks_2x2x2_of_12_scalar_rfloor"]
    p = w["params"]
    mesh = phx.init_mesh(p)
    assert mesh.field_elems == w["prim"].size and w["prim"].shape[1] == 9
    # prim -> cons
    ref = orc.prim_to_cons(p, w["prim"])
    prim = torch.from_numpy(w["prim"]).cuda()
    cons = torch.empty_like(prim)
    phx.prim_to_cons(mesh, prim, cons)
    got = cons.cpu().numpy()
    assert (np.abs(got - ref).max(axis=(0, 2, 3, 4)) / np.abs(ref).max(axis=(0, 2, 3, 4))).max() < 1e-13
    # ghost fill, nine variables, bit exact
    rng = np.random.default_rng(9)
    f = rng.standard_normal(w["prim"].shape)
    fr = orc.fill_ghosts(p, f.copy())
    t = torch.from_numpy(f).cuda()
    phx.fill_ghosts(mesh, t)
    assert np.array_equal(t.cpu().numpy(), fr)
    # cons -> prim with scalars pushed outside their bounds and densities below the radial floor
    for attempt in range(5):
        cons_in = ref.copy()
        sel = rng.uniform(size=cons_in[:, 8].shape)
        cons_in[:, 8] = np.where(sel < 0.1, 1.3 * cons_in[:, 0], np.where(sel > 0.9, -0.2 * cons_in[:, 0], cons_in[:, 8]))
        orc.reset_c2p_margin()
        cons_ref = cons_in.copy()
        prim_ref, mask_ref = orc.cons_to_prim(p, cons_ref)
        if orc.last_c2p_margin() > MARGIN_MIN:
            break
    else:
        pytest.fail("no seed with a safe margin found")
    mr = interior(p, mask_ref)
    assert (mr & 128).any() and (mr & 1).any() and (mr & 64).any()
    c = torch.from_numpy(cons_in).cuda()
    pg = torch.zeros_like(c)
    mk = torch.zeros(mask_ref.shape, dtype=torch.uint8, device="cuda")
    phx.cons_to_prim(mesh, c, pg, mk)
    assert np.array_equal(interior(p, mk.cpu().numpy()), mr)
    live = (mr & 64) == 0
    gp, rp = interior(p, pg.cpu().numpy()), interior(p, prim_ref)
    assert (np.abs(gp - rp) / np.maximum(np.abs(rp), 1e-3 * _scales(rp)))[:, live].max() < 1e-11
    gc, rc = interior(p, c.cpu().numpy()), interior(p, cons_ref)
    assert (np.abs(gc - rc) / np.maximum(np.abs(rc), 1e-3 * _scales(rc)))[:, live].max() < 1e-11
    clipped = (mr & 128) != 0
    assert np.all((gp[8][clipped] == p["scalar_min"]) | (gp[8][clipped] == p["scalar_max"]))


def test_evolve_host_with_scalar_matches_device_path():
    torch, phx = _gpu()
    w = WORKLOADS["turb_24_weno_scalar"]
    p = w["params"]
    b = GpuRun(p, w["prim"])
    for s in range(2):
        b.step_fused_cfl(0.4, s == 0)
    cb, pb, _, mb = b.get()
    mesh = phx.init_mesh(p)
    hin = torch.from_numpy(w["prim"]).pin_memory()
    hp = torch.empty_like(hin).pin_memory(); hc = torch.empty_like(hin).pin_memory()
    hm = torch.empty(mb.shape, dtype=torch.uint8).pin_memory()
    phx.evolve_host(mesh, hin, 2, 0.4, hp, hc, hm)
    assert np.array_equal(hp.numpy(), pb) and np.array_equal(hc.numpy(), cb) and np.array_equal(hm.numpy(), mb)


def test_bad_scalar_and_floor_parameters_are_rejected():
    torch, phx = _gpu()
    for kw in (dict(nscalar=2), dict(nscalar=1, scalar_min=0.5, scalar_max=0.5), dict(floor_form=4),
               dict(floor_form=3, floor_alpha_rho=-1.0)):
        with pytest.raises(phx.PhxError):
            phx.init_mesh(wl.default_params(nx=8, ny=8, nz=8, **kw))
