"""Pin P18 of the CPU oracle: the positivity fallback of the fifth-order reconstructions (reading C5.1;
oracle/orc.cpp block_fluxes).  The paper's App. B never discusses positivity of the reconstructed face
values; the reading taken is: if the reconstructed rho or u at EITHER face of a cell is below its floor (rho_flr, and
rho_flr * eps_flr for u, both evaluated at the centre of the cell, both lowered by one part in 1e12), that cell falls
back to piecewise constant in that direction for ALL variables; piecewise-linear reconstructions never take the branch.
The 1e-12 keeps the decision away from the value the floors themselves produce: con2prim holds whole regions exactly at
the floor, every reconstruction returns the floor there up to rounding, and a threshold at the floor itself would be decided
by the last bit of whoever does the arithmetic (the CUDA path evaluates WENO5-Z in a different but equivalent form).

What is checked here is the branch logic, on hand-built stencils whose WENO5-Z face values are worked out by hand:
which cells fall back, in which direction, for which variables, at which threshold.  The reconstruction itself
(orc.recon_line) is pinned by P12 / P12b / P12d and the Riemann solver (orc.point_riemann) by P8b; the density flux of
the states at rest is also checked against the closed form F_D = -c/2 (rho_R - rho_L) of HLL between two states at rest.
All of these run without a GPU.
"""
import math

import numpy as np
import pytest

from oracle import orc
from paper_2410_09146_b200 import workloads as wl

ETA = np.diag([-1.0, 1.0, 1.0, 1.0])
FIFTH = [wl.RECON_WENO5Z, wl.RECON_WENO5Z_AOAH, wl.RECON_MP5]

# Two hand-built density / energy profiles (cell values along the sweep direction, outflow ghosts):
#   V : 1 1 1 1 1 1 0.5 1 1 1 1 1 1      a one-cell dip at c = 6
#   K : 2 2 2 2 2 2 1.0 0.2 0.2 0.2 ...  a kink at c = 6, steep side above it
V = np.array([1.0] * 6 + [0.5] + [1.0] * 6)
K = np.array([2.0] * 6 + [1.0] + [0.2] * 6)
C = 6


def line_params(n, recon, x0=1.0, **kw):
    """1-D mesh along x starting at x0 whose cell centres have y = z = 0, so that the flat-metric floor radius is |x|."""
    base = dict(nx=n, ng=3 if recon >= 3 else 2, recon=recon, riemann=wl.RIEMANN_HLL, use_ct=0,
                bc=((wl.BC_OUTFLOW, wl.BC_OUTFLOW),) * 3, xmin=(x0, -0.5, -0.5), xmax=(x0 + 0.125 * n, 0.5, 0.5),
                rho_floor=1e-10, eps_floor=1e-10)
    base.update(kw)
    return wl.default_params(**base)


def line_prims(p, rho, u, extra=False):
    n = len(rho)
    q = np.zeros((8, 1, 1, n))
    q[0, 0, 0], q[4, 0, 0] = rho, u
    if extra:   # every other variable varies too, so that "all eight variables fall back" is visible in the fluxes
        i = np.arange(n)
        q[1, 0, 0] = 0.10 * np.sin(0.9 * i); q[2, 0, 0] = 0.05 * np.cos(0.7 * i); q[3, 0, 0] = -0.07 * np.sin(0.5 * i + 1.0)
        q[5, 0, 0] = 0.3
        q[6, 0, 0] = 0.2 + 0.1 * np.sin(1.1 * i); q[7, 0, 0] = -0.1 + 0.05 * np.cos(0.8 * i)
    return wl.finish(p, q)


def face_states(p, prim):
    """(qm, qp)[var, i] of every allocated cell of the line, from the pinned reconstruction of each variable alone."""
    line = prim[0, :, 0, 0, :]
    qm = np.empty_like(line); qp = np.empty_like(line)
    for v in range(8):
        qm[v], qp[v] = orc.recon_line(p["recon"], line[v])
    return line, qm, qp


def expected_fluxes(p, prim, fallback_cells):
    """F at face (i-1/2) for i = g .. g+n: HLL of (upper-face state of cell i-1, lower-face state of cell i), with the
    cells in `fallback_cells` (allocated indices) replaced by their cell-centre values."""
    line, qm, qp = face_states(p, prim)
    qm, qp = qm.copy(), qp.copy()
    for c in fallback_cells:
        qm[:, c] = line[:, c]; qp[:, c] = line[:, c]
    g, n = p["ng"], p["nx"]
    out = {}
    for i in range(g, g + n + 1):
        out[i] = orc.point_riemann(p, ETA, 0, qp[:, i - 1], qm[:, i])
    return out


def flagged(p, prim, rfl, ufl):
    """The reading itself, written once more on the pinned face values: allocated indices of the cells that fall back."""
    line, qm, qp = face_states(p, prim)
    g, n = p["ng"], p["nx"]
    tr, tu = rfl * (1.0 - 1e-12), ufl * (1.0 - 1e-12)
    return [i for i in range(g - 1, g + n + 1)
            if qm[0, i] < tr or qp[0, i] < tr or qm[4, i] < tu or qp[4, i] < tu]


def check_line(p, prim, expect_cells):
    g, n = p["ng"], p["nx"]
    F = orc.stage_fluxes(p, prim)[0][0, :, 0, 0, :]
    want = expected_fluxes(p, prim, expect_cells)
    other = expected_fluxes(p, prim, [])
    for i in range(g, g + n + 1):
        assert np.array_equal(F[:, i], want[i]), (i, F[:, i], want[i])
    return F, want, other


def test_hand_worked_weno5z_face_values_of_the_two_profiles():
    """The stencils are chosen so that the face values can be worked out by hand (B12-B15, cell-average coefficients).
    V at c: tau_Z = 0, weights = (1/10, 6/10, 3/10), candidates (1/12, 7/12, 10/12) -> 73/120 at both faces; the cells next to
    the dip select their flat stencil and return 1.  K at c, upper face: candidates (1/6, 17/30, 7/15), beta = (10/3, 64/75,
    32/15), tau_Z = 6/5 -> 0.52979..."""
    qm, qp = orc.recon_line(wl.RECON_WENO5Z, V)
    assert abs(qp[C] - 73.0 / 120.0) < 1e-15 and abs(qm[C] - 73.0 / 120.0) < 1e-15
    assert np.abs(qp[[2, 3, 4, 5, 7, 8, 9, 10]] - 1.0).max() < 1e-15 and np.abs(qm[[2, 3, 4, 5, 7, 8, 9, 10]] - 1.0).max() < 1e-15
    qm, qp = orc.recon_line(wl.RECON_WENO5Z, K)
    b = np.array([10.0 / 3.0, 64.0 / 75.0, 32.0 / 15.0]); tau = 6.0 / 5.0
    w = np.array([0.1, 0.6, 0.3]) * (1.0 + (tau / b) ** 2)
    val = (w * np.array([1.0 / 6.0, 17.0 / 30.0, 7.0 / 15.0])).sum() / w.sum()
    assert abs(qp[C] - val) < 1e-15 and 0.52 < val < 0.54
    assert qm[C] > 1.0 and qp[C - 1] > 1.9 and qm[C - 1] > 1.9


@pytest.mark.parametrize("recon", FIFTH)
def test_p18_dip_in_density_falls_back_in_that_cell_only_and_for_all_variables(recon):
    p = line_params(len(V), recon, rho_floor=0.7, eps_floor=1e-3)
    prim = line_prims(p, V, np.full_like(V, 3.0), extra=True)
    c = C + p["ng"]
    assert flagged(p, prim, 0.7, 0.7e-3) == [c]          # the profile does what it was built for, for this scheme
    F, want, other = check_line(p, prim, [c])
    # the branch changes the two faces of the cell and nothing else, in every variable that has a flux there
    for i in want:
        changed = np.abs(want[i] - other[i]) > 1e-6
        if i in (c, c + 1):
            assert changed[[0, 1, 2, 3, 4, 6, 7]].all(), (i, want[i], other[i])     # F[B^x] = 0 identically
        else:
            assert not changed.any()


@pytest.mark.parametrize("recon", FIFTH)
def test_p18_density_flux_of_states_at_rest_is_the_closed_form(recon):
    """No oracle routine in the expected value: between two states at rest without field HLL gives
    F_D = s+ s- (rho_R - rho_L)/(s+ - s-) = -c/2 (rho_R - rho_L), c = max sound speed, c_s^2 = Gamma P/(rho + u + P).
    With the fallback the two faces of the dip see the cell-centre density 0.5 against the neighbours' face value 1."""
    p = line_params(len(V), recon, rho_floor=0.7, eps_floor=1e-3)
    prim = line_prims(p, V, np.full_like(V, 3.0))
    c = C + p["ng"]
    F = orc.stage_fluxes(p, prim)[0][0, :, 0, 0, :]
    gam = p["gamma_ad"]
    cs = lambda rho: math.sqrt(gam * (gam - 1.0) * 3.0 / (rho + 3.0 + (gam - 1.0) * 3.0))
    cmax = max(cs(0.5), cs(1.0))
    assert abs(F[0, c] - (-0.5 * cmax * (0.5 - 1.0))) < 1e-15       # face c-1/2: (1 | 0.5)
    assert abs(F[0, c + 1] - (-0.5 * cmax * (1.0 - 0.5))) < 1e-15   # face c+1/2: (0.5 | 1)
    # without the branch the cell would have shown its reconstructed face value instead of 0.5
    p2 = dict(p, rho_floor=1e-10)
    F2 = orc.stage_fluxes(p2, prim)[0][0, :, 0, 0, :]
    qm, qp = orc.recon_line(recon, prim[0, 0, 0, 0, :])
    cm = max(cs(qm[c]), cs(1.0))
    assert abs(F2[0, c] - (-0.5 * cm * (qm[c] - 1.0))) < 1e-15
    if recon != wl.RECON_MP5:       # MP5 limits the value at an extremum to the cell value itself: nothing to see in rho there
        assert abs(F2[0, c] - F[0, c]) > 1e-3


def test_p18_threshold_sits_just_below_the_floor_and_u_is_measured_against_rho_floor_times_eps_floor():
    recon = wl.RECON_WENO5Z
    rho = np.full_like(V, 2.0)
    base = line_params(len(V), recon)
    face = 73.0 / 120.0                                   # hand-worked face value of the dip in u
    c = C + base["ng"]
    prim = line_prims(base, rho, V, extra=True)
    qm, qp = orc.recon_line(recon, prim[0, 4, 0, 0, :])
    assert qm[c] == qp[c] and abs(qp[c] - face) < 1e-15
    # u floor = rho_flr * eps_flr = 0.7: taken (0.6083 <= 0.7) although u is above eps_flr = 0.5 and below rho_flr = 1.4
    p = dict(base, rho_floor=1.4, eps_floor=0.5)
    check_line(p, prim, [c])
    # u floor 0.56 < 0.6083: not taken, although u < rho_flr
    p = dict(base, rho_floor=1.4, eps_floor=0.4)
    check_line(p, prim, [])
    # a value AT the floor (or within rounding of it) does not count, one that is 2e-12 below it does
    # (eps_flr = 1 keeps the product exact)
    for fl, cells in ((float(qp[c]), []), (float(qp[c]) * (1.0 + 1e-15), []), (float(qp[c]) * (1.0 + 5e-13), []),
                      (float(qp[c]) * (1.0 + 2e-12), [c])):
        check_line(dict(base, rho_floor=fl, eps_floor=1.0), prim, cells)
    # the same for the density: dip in rho, u far above rho_flr * eps_flr
    prim = line_prims(base, V, np.full_like(V, 3.0), extra=True)
    qm, qp = orc.recon_line(recon, prim[0, 0, 0, 0, :])
    for fl, cells in ((float(qp[c]), []), (float(qp[c]) * (1.0 + 5e-13), []), (float(qp[c]) * (1.0 + 2e-12), [c])):
        check_line(dict(base, rho_floor=fl, eps_floor=1e-3), prim, cells)


def test_p18_a_region_held_at_the_floor_keeps_its_reconstruction():
    """What the 1e-12 is for: cells that con2prim floored carry rho = rho_flr exactly; in a run of such cells WENO5-Z returns
    rho_flr (1 +- a few 1e-16).  None of them may fall back, whichever way the last bit went."""
    recon = wl.RECON_WENO5Z
    fl = 0.3
    rho = np.array([1.0, 0.9, 0.7, fl, fl, fl, fl, fl, fl, 0.8, 1.1, 1.0, 1.0])
    p = line_params(len(rho), recon, rho_floor=fl, eps_floor=1e-3)
    prim = line_prims(p, rho, np.full_like(rho, 3.0), extra=True)
    line, qm, qp = face_states(p, prim)
    g = p["ng"]
    inner = slice(g + 5, g + 7)                           # cells whose whole stencil is at the floor
    assert np.abs(qm[0, inner] / fl - 1.0).max() < 1e-15 and np.abs(qp[0, inner] / fl - 1.0).max() < 1e-15
    check_line(p, prim, flagged(p, prim, fl, fl * 1e-3))
    assert not set(range(g + 3, g + 9)) & set(flagged(p, prim, fl, fl * 1e-3))


@pytest.mark.parametrize("recon", FIFTH)
def test_p18_one_low_face_is_enough_and_the_neighbour_above_the_floor_keeps_its_reconstruction(recon):
    """Kink profile: the cell's centre value (1.0) and lower face are above the floor, only its upper face is below."""
    p = line_params(len(K), recon, rho_floor=0.6, eps_floor=1e-3)
    prim = line_prims(p, K, np.full_like(K, 3.0), extra=True)
    c = C + p["ng"]
    line, qm, qp = face_states(p, prim)
    assert qp[0, c] <= 0.6 < qm[0, c] and line[0, c] == 1.0
    fl = flagged(p, prim, 0.6, 0.6e-3)
    assert fl[0] == c and c - 1 not in fl                 # the cells beyond the kink (0.2 < floor) are flagged too
    F, want, other = check_line(p, prim, fl)
    assert np.abs(want[c] - other[c]).max() > 1e-3        # face c-1/2 changed although the state there was admissible


@pytest.mark.parametrize("recon", [wl.RECON_CONST, wl.RECON_PLM_MINMOD, wl.RECON_PLM_MC])
def test_p18_piecewise_linear_never_takes_the_branch(recon):
    """A floor above every value in the mesh: a piecewise-linear scheme that fell back would lose its slopes."""
    p = line_params(len(K), recon, rho_floor=5.0, eps_floor=2.0)
    prim = line_prims(p, K + 0.1 * np.arange(len(K)), 3.0 + 0.2 * np.arange(len(K)), extra=True)
    F, want, other = check_line(p, prim, [])
    if recon != wl.RECON_CONST:
        const = expected_fluxes(p, prim, list(range(p["ng"] - 1, p["ng"] + p["nx"] + 1)))
        assert max(np.abs(const[i] - want[i]).max() for i in want) > 1e-3


def test_p18_position_dependent_floor_is_taken_at_the_centre_of_the_cell():
    """floor_form 3 (rho0 r^-alpha), flat metric: r = |x| on this line, which starts at x = 10; alpha = 12 makes
    the floor steep enough to tell the centre of a cell from its face.  rho0 is chosen so that the floor is 0.55 at the centre
    of the kink cell: above its upper face value 0.5298 (taken), while the floor at that face's own position,
    0.55 (x_c/(x_c + dx/2))^12 = 0.513, is below it (a threshold taken at the face would not fall back)."""
    recon = wl.RECON_WENO5Z
    al = 12.0
    p = line_params(len(K), recon, x0=10.0, floor_form=3, floor_alpha_rho=al, floor_alpha_eps=0.0, eps_floor=1e-3)
    xc = wl.cell_centres(p)[0][C]
    dx = 0.125
    p["rho_floor"] = 0.55 * xc ** al
    prim = line_prims(p, K, np.full_like(K, 3.0), extra=True)
    c = C + p["ng"]
    line, qm, qp = face_states(p, prim)
    x_all = p["xmin"][0] + (np.arange(-p["ng"], p["nx"] + p["ng"]) + 0.5) * dx
    fl_centre = p["rho_floor"] / x_all ** al
    assert abs(fl_centre[c] - 0.55) < 1e-14 and qp[0, c] < fl_centre[c] * (1 - 1e-12)
    assert qp[0, c] > p["rho_floor"] / (xc + 0.5 * dx) ** al
    want_cells = [i for i in range(p["ng"] - 1, p["ng"] + p["nx"] + 1)
                  if min(qm[0, i], qp[0, i]) < fl_centre[i] * (1 - 1e-12) or min(qm[4, i], qp[4, i]) < fl_centre[i] * 1e-3 * (1 - 1e-12)]
    assert want_cells[0] == c
    check_line(p, prim, want_cells)
    # one cell further from the origin the same face value would be above the (smaller) floor: the constant form differs
    pc = dict(p, floor_form=0, rho_floor=0.52)
    check_line(pc, prim, [i for i in want_cells if i != c])


def test_p18_fallback_is_per_direction():
    """2-D: the kink along x at column c makes that cell fall back in the x sweep; its y stencil is smooth and stays above
    the floor, so the y sweep keeps the fifth-order states of that cell."""
    recon = wl.RECON_WENO5Z
    n = len(K)
    p = wl.default_params(nx=n, ny=n, nz=1, ng=3, recon=recon, riemann=wl.RIEMANN_HLL, use_ct=0,
                          bc=((wl.BC_OUTFLOW, wl.BC_OUTFLOW),) * 3, rho_floor=0.6, eps_floor=1e-3)
    yy = 1.0 + 0.1 * np.sin(2.0 * np.pi * (np.arange(n) + 0.5) / n)
    q = np.zeros((8, 1, n, n))
    q[0, 0] = yy[:, None] * K[None, :]
    q[4, 0] = 3.0
    q[2, 0] = 0.05 * yy[:, None]
    prim = wl.finish(p, q)
    F = orc.stage_fluxes(p, prim)
    g = p["ng"]
    j = g + 4; c = g + C
    assert q[0, 0, 4, C] > 0.9
    # x sweep along row j: cell c (and the cells beyond the kink) constant
    row = prim[0, :, 0, j, :]
    qm = np.empty_like(row); qp = np.empty_like(row)
    for v in range(8):
        qm[v], qp[v] = orc.recon_line(recon, row[v])
    assert qp[0, c] <= 0.6 < qm[0, c]
    Fx = orc.point_riemann(p, ETA, 0, qp[:, c - 1], row[:, c])
    assert np.array_equal(F[0][0, :, 0, j, c], Fx)
    # y sweep along column c: fifth-order states on both faces of (j, c)
    col = prim[0, :, 0, :, c]
    qm = np.empty_like(col); qp = np.empty_like(col)
    for v in range(8):
        qm[v], qp[v] = orc.recon_line(recon, col[v])
    assert min(qm[0, j - 1:j + 2].min(), qp[0, j - 1:j + 2].min()) > 0.6
    assert abs(qm[0, j] - col[0, j]) > 1e-4               # not the cell-centre value
    assert np.array_equal(F[1][0, :, 0, j, c], orc.point_riemann(p, ETA, 1, qp[:, j - 1], qm[:, j]))
    assert np.array_equal(F[1][0, :, 0, j + 1, c], orc.point_riemann(p, ETA, 1, qp[:, j], qm[:, j + 1]))
