"""Pins P16 (passive scalar, Eq.14) and P17 (floor forms) for the CPU oracle.
As in test_oracle_pins.py the oracle is checked against what the paper and the mathematics fix, never against
itself: exact solutions of the advection equation Eq.14 reduces to, conservation, closed-form special cases of the
Kerr-Schild radius.  No GPU needed.
"""
import math

import numpy as np
import pytest

from oracle import orc
from paper_2410_09146_b200 import workloads as wl

M_SCALAR_CLIPPED = 128


def _run(w, nsteps=None, t_end=None, cfl=0.4):
    r = orc.Run(w["params"], w["prim"])
    n = 0
    while (nsteps is None or n < nsteps) and (t_end is None or r.t < t_end * (1 - 1e-12)):
        dt = r.dt(cfl)
        if t_end is not None:
            dt = min(dt, t_end - r.t)
        r.step(dt)
        n += 1
    return r


# ----------------------------------------------------------------------------- P16a
@pytest.mark.parametrize("kind", ["turbulence", "kerr_schild"])
def test_p16a_constant_scalar_stays_constant(kind):
    """Eq.14 with S = 0 and X = const is the continuity equation times a constant: X must stay constant whatever the
    flow does.  Fails if the scalar flux is not F~_D X (a missing lapse, shift or sqrt(gamma), a different upwinding)."""
    if kind == "turbulence":
        w0 = wl.turbulence_box(12, recon=wl.RECON_PLM_MC)
    else:
        w0 = wl.kerr_schild_torus(16)
    p0 = w0["params"]
    shape = (p0["nbz"] * p0["nz"], p0["nby"] * p0["ny"], p0["nbx"] * p0["nx"])
    w = wl.with_scalar(w0, np.full(shape, 0.3))
    r = _run(w, nsteps=5)
    X = wl.from_blocks(w["params"], r.prim)[8]
    rho0 = wl.from_blocks(p0, w0["prim"])[0]
    rho1 = wl.from_blocks(w["params"], r.prim)[0]
    assert np.abs(rho1 - rho0).max() > 1e-6 * np.abs(rho0).max()      # the flow did move mass around
    assert np.abs(X - 0.3).max() < 1e-13
    assert not (r.mask & M_SCALAR_CLIPPED).any()
    # the other eight variables do not know about the scalar
    r8 = _run(w0, nsteps=5)
    assert np.array_equal(r8.cons, r.cons[:, :8])


# ----------------------------------------------------------------------------- P16b
def test_p16b_scalar_is_conserved_on_a_periodic_box():
    w0 = wl.turbulence_box(12, recon=wl.RECON_WENO5Z)
    w = wl.with_scalar(w0, wl.smooth_scalar(w0["params"], 7))
    p = w["params"]
    r = orc.Run(p, w["prim"])
    c0 = wl.from_blocks(p, r.cons)[8].copy()
    for _ in range(5):
        r.step(r.dt(0.4))
    c1 = wl.from_blocks(p, r.cons)[8]
    s0, s1 = math.fsum(c0.ravel()), math.fsum(c1.ravel())
    assert abs(s1 - s0) <= 5e-15 * math.fsum(np.abs(c0).ravel())
    assert np.abs(c1 - c0).max() > 1e-6


# ----------------------------------------------------------------------------- P16c
def _advection_error(n, boosted, t_frac=1.0, recon=wl.RECON_PLM_MC):
    """1-D uniform flow carrying a smooth X profile: Eq.14 reduces to d_t X + V d_x X = 0 with the coordinate velocity
    V = alpha v - beta (Eq.6): V = v in Minkowski, V = -shift for a fluid at rest in the boosted flat metric."""
    v = 0.5
    if boosted:
        p = wl.default_params(nx=n, ng=4, recon=recon, metric=wl.MINKOWSKI_BOOSTED, shift=(v, 0.0, 0.0))
        V, ux = -v, 0.0
    else:
        p = wl.default_params(nx=n, ng=4, recon=recon)
        V, ux = v, v / math.sqrt(1 - v * v)
    x = wl.cell_centres(p)[0]
    prof = lambda s: 0.3 + 0.1 * np.sin(2 * np.pi * s) + 0.05 * np.cos(4 * np.pi * s)
    q = np.zeros((9, 1, 1, n))
    q[0], q[1], q[4], q[5] = 1.0, ux, 1.5, 0.3
    q[8, 0, 0] = prof(x)
    p = dict(p, nscalar=1, scalar_min=0.0, scalar_max=1.0)
    r = orc.Run(p, wl.finish(p, q))
    T = t_frac / v
    while r.t < T * (1 - 1e-12):
        r.step(min(r.dt(0.4), T - r.t))
    X = wl.from_blocks(p, r.prim)[8, 0, 0]
    assert np.abs(wl.from_blocks(p, r.prim)[0] - 1.0).max() < 1e-13     # the uniform flow stays uniform
    return np.abs(X - prof(x - V * T)).sum() / n


@pytest.mark.parametrize("boosted", [False, True])
def test_p16c_scalar_advection_converges_to_the_exact_solution(boosted):
    # a quarter period: the profile sits a quarter wavelength downstream (wrong sign of V fails here)
    assert _advection_error(64, boosted, t_frac=0.25) < 2e-3
    # one full period.  WENO5-Z does not clip the smooth extrema, so the second-order time integration shows cleanly;
    # MC-limited PLM clips them and sits at the ~5/3 of TVD schemes in L1
    errs = [_advection_error(n, boosted, recon=wl.RECON_WENO5Z) for n in (32, 64, 128)]
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert errs[-1] < 1e-4 and slopes[0] > 1.9 and slopes[1] > 1.9, (errs, slopes)
    errs = [_advection_error(n, boosted) for n in (32, 64, 128)]
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert errs[-1] < 1e-3 and slopes[0] > 1.6 and slopes[1] > 1.6, (errs, slopes)


# ----------------------------------------------------------------------------- P16d
def test_p16d_scalar_riemann_flux_consistency_and_upwinding():
    rng = np.random.default_rng(16)
    for riemann in (0, 1):
        p = wl.default_params(riemann=riemann, nscalar=1)
        for _ in range(20):
            g4 = np.diag([-1.0, 1.0, 1.0, 1.0])
            q = np.zeros(9)
            q[0] = 10 ** rng.uniform(-2, 1); q[1:4] = rng.uniform(-1, 1, 3); q[4] = q[0] * 10 ** rng.uniform(-2, 1)
            q[5:8] = rng.uniform(-1, 1, 3); q[8] = rng.uniform(0, 1)
            for d in range(3):
                F = orc.point_riemann_scalar(p, g4, d, q, q)
                F8 = orc.point_riemann(p, g4, d, q[:8], q[:8])
                assert np.array_equal(F[:8], F8)
                assert abs(F[8] - F8[0] * q[8]) <= 4e-16 * abs(F8[0] * q[8])        # consistency: F_X(q,q) = F_D X
    # HLL with every wave moving to the right takes the left state's flux F_D,L X_L
    p = wl.default_params(riemann=1, nscalar=1)
    qL = np.array([1.0, 5.0, 0.0, 0.0, 0.01, 0.0, 0.0, 0.0, 0.2])
    qR = np.array([0.5, 5.0, 0.0, 0.0, 0.005, 0.0, 0.0, 0.0, 0.7])
    g4 = np.diag([-1.0, 1.0, 1.0, 1.0])
    F = orc.point_riemann_scalar(p, g4, 0, qL, qR)
    W = math.sqrt(1 + 25.0)
    assert abs(F[8] - 1.0 * W * (5.0 / W) * 0.2) < 1e-14                  # D v X of the left state
    F = orc.point_riemann_scalar(p, g4, 0, qR * np.array([1, -1, 1, 1, 1, 1, 1, 1, 1]), qL * np.array([1, -1, 1, 1, 1, 1, 1, 1, 1]))
    assert abs(F[8] + 1.0 * 5.0 * 0.2) < 1e-14                            # mirrored: everything moves left, right state wins


# ----------------------------------------------------------------------------- P16e
def test_p16e_scalar_bounds_and_floors():
    n = 4
    p = wl.default_params(nx=n, ny=n, nz=n, ng=2, nscalar=1, scalar_min=0.05, scalar_max=0.55, rho_floor=1e-6, eps_floor=1e-6)
    q = np.zeros((9, n, n, n))
    q[0], q[4], q[5] = 1.0, 1.0, 0.1
    q[8] = 0.3
    prim = wl.finish(p, q)
    cons = orc.prim_to_cons(p, prim)
    g = p["ng"]
    D = cons[0, 0, g, g, g]
    assert cons[0, 8, g, g, g] == D * 0.3                                 # sqrt(gamma) D X with sqrt(gamma) = 1, W = 1
    cons[0, 8, g, g, g] = D * 0.9                                         # above the upper bound
    cons[0, 8, g, g, g + 1] = -D * 0.1                                    # below the lower bound
    cons[0, 8, g, g + 1, g] = np.nan                                      # not a number
    cons[0, 0, g + 1, g, g] = 1e-9; cons[0, 8, g + 1, g, g] = 1e-9 * 0.4  # density below its floor, X = 0.4 legal
    cons[0, 0, g + 1, g + 1, g] = -1.0                                    # bad input
    prim2, mask = orc.cons_to_prim(p, cons)
    assert mask[0, g, g, g] == M_SCALAR_CLIPPED and prim2[0, 8, g, g, g] == 0.55 and cons[0, 8, g, g, g] == D * 0.55
    assert mask[0, g, g, g + 1] == M_SCALAR_CLIPPED and prim2[0, 8, g, g, g + 1] == 0.05
    assert mask[0, g, g + 1, g] == M_SCALAR_CLIPPED and prim2[0, 8, g, g + 1, g] == 0.05
    assert mask[0, g + 1, g, g] & 1 and not mask[0, g + 1, g, g] & M_SCALAR_CLIPPED
    assert abs(prim2[0, 8, g + 1, g, g] - 0.4) < 1e-15 and prim2[0, 0, g + 1, g, g] == 1e-6
    assert cons[0, 8, g + 1, g, g] == cons[0, 0, g + 1, g, g] * prim2[0, 8, g + 1, g, g]   # rewritten with the floored D
    assert mask[0, g + 1, g + 1, g] == 32 | M_SCALAR_CLIPPED and prim2[0, 8, g + 1, g + 1, g] == 0.05
    untouched = mask == 0
    assert untouched.sum() >= n ** 3 - 5 and np.all(prim2[0, 8][untouched[0]][: 1] == 0.3)


# ----------------------------------------------------------------------------- P17
def test_p17_floor_forms_follow_the_radius():
    """rho0, rho0 exp(-alpha x1), rho0 x1^-alpha, rho0 r^-alpha with x1 read as r (Cartesian coordinates).
    The Kerr-Schild radius has closed forms on the spin axis (r = |z|), in the equatorial plane (r^2 = R^2 - a^2) and for
    a = 0 (r = R); on the flat metrics r is the Euclidean distance."""
    a = 0.9
    base = dict(rho_floor=1e-5, eps_floor=1e-3, floor_alpha_rho=2.0, floor_alpha_eps=1.0)
    ks = wl.default_params(metric=wl.KERR_SCHILD, bh_spin=a, **base)
    pts = [((0.0, 0.0, 3.0), 3.0), ((0.0, 0.0, -7.5), 7.5), ((3.0, 4.0, 0.0), math.sqrt(25.0 - a * a)),
           ((-6.0, 2.5, 0.0), math.sqrt(42.25 - a * a))]
    for form in (2, 3):
        for x, r in pts:
            rf, ef = orc.point_floors(dict(ks, floor_form=form), x)
            assert abs(rf - 1e-5 / r ** 2) < 1e-15 * rf and abs(ef - 1e-3 / r) < 1e-15 * ef
    for x, r in pts:
        rf, ef = orc.point_floors(dict(ks, floor_form=1, floor_alpha_rho=0.5, floor_alpha_eps=0.25), x)
        assert abs(rf - 1e-5 * math.exp(-0.5 * r)) < 1e-15 * rf and abs(ef - 1e-3 * math.exp(-0.25 * r)) < 1e-15 * ef
        assert orc.point_floors(dict(ks, floor_form=0), x) == (1e-5, 1e-3)
    # general point: r solves the defining quartic r^4 - (R^2 - a^2) r^2 - a^2 z^2 = 0
    x = (2.0, -1.0, 1.5)
    rf, _ = orc.point_floors(dict(ks, floor_form=3), x)
    r = math.sqrt(1e-5 / rf)
    R2 = sum(t * t for t in x)
    assert abs(r ** 4 - (R2 - a * a) * r ** 2 - a * a * x[2] ** 2) < 1e-12
    # a = 0 and the flat metrics: Euclidean distance
    for par in (dict(ks, bh_spin=0.0), wl.default_params(**base), wl.default_params(metric=wl.MINKOWSKI_BOOSTED, shift=(0.1, 0, 0), **base)):
        rf, ef = orc.point_floors(dict(par, floor_form=3), x)
        assert abs(rf - 1e-5 / R2) < 1e-15 * rf and abs(ef - 1e-3 / math.sqrt(R2)) < 1e-15 * ef


def test_p17b_radial_floor_acts_in_con2prim():
    """A near-vacuum state on a Kerr-Schild (a = 0) grid is floored to rho0 r^-2 and eps0 r^-1, r the distance of the
    cell centre from the origin; the mask says so; with floor_form = 0 the same input gives the constants."""
    n = 6
    p = wl.default_params(metric=wl.KERR_SCHILD, bh_spin=0.0, nx=n, ny=n, nz=n, ng=2, xmin=(2.0, 2.0, 2.0), xmax=(8.0, 8.0, 8.0),
                          bc=((1, 1),) * 3, rho_floor=1e-4, eps_floor=1e-2, floor_form=3, floor_alpha_rho=2.0, floor_alpha_eps=1.0)
    q = np.zeros((8, n, n, n))
    q[0], q[4] = 1e-9, 1e-14
    prim = wl.finish(p, q)
    cons = orc.prim_to_cons(p, prim)
    prim2, mask = orc.cons_to_prim(p, cons.copy())
    x, y, z = wl.cell_centres(p)
    r = np.sqrt(x[None, None, :] ** 2 + y[None, :, None] ** 2 + z[:, None, None] ** 2)
    rho = wl.from_blocks(p, prim2)[0]
    eps = wl.from_blocks(p, prim2)[4] / rho
    assert np.all(wl.from_blocks(p, mask[:, None])[0] == 3)
    assert np.abs(rho * r ** 2 / 1e-4 - 1).max() < 1e-14 and np.abs(eps * r / 1e-2 - 1).max() < 1e-14
    prim3, mask3 = orc.cons_to_prim(dict(p, floor_form=0), cons.copy())
    assert np.all(wl.from_blocks(p, prim3)[0] == 1e-4)
