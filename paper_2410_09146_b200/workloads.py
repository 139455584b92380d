"""Seeded synthetic workloads shaped like the paper's tests (BASELINE.json configs 1-5).

This module is the ONLY thing the CUDA path and the CPU oracle share.  It holds the input
recipes (initial primitives on packed blocks with ghosts already filled, parameter
dictionaries) and none of the method's arithmetic: no fluxes, no reconstruction, no
con2prim, no wave speeds.  The two geometric formulas it needs to *shape* the Kerr-Schild
inputs (the Kerr-Schild radius r and sqrt(gamma)=sqrt(1+2H), used to place the excised
region and to turn the divergence-free densitised field into the primitive B) are part of
the recipe stated in DESIGN.md section 4.

Layout of every field: [block][var][k][j][i], i fastest, fp64, var order
(rho, u~1, u~2, u~3, u=rho*eps, B1, B2, B3)  (Eq.13), plus the passive scalar X
(Eq.14) as variable 8 when params["nscalar"] = 1.
Block id = (bz*nby + by)*nbx + bx.  A dimension with one zone in total is inactive and has
no ghost zones.
"""
from __future__ import annotations

import numpy as np

NV = 8
SEED0 = 241009146

MINKOWSKI, KERR_SCHILD, MINKOWSKI_BOOSTED = 0, 1, 2
RECON_CONST, RECON_PLM_MINMOD, RECON_PLM_MC, RECON_WENO5Z, RECON_WENO5Z_AOAH, RECON_MP5 = 0, 1, 2, 3, 4, 5
RIEMANN_LLF, RIEMANN_HLL = 0, 1
BC_PERIODIC, BC_OUTFLOW = 0, 1


def default_params(**kw):
    p = dict(
        metric=MINKOWSKI, bh_mass=1.0, bh_spin=0.0, r_excise=0.0,
        nbx=1, nby=1, nbz=1, nx=1, ny=1, nz=1, ng=4,
        xmin=(0.0, 0.0, 0.0), xmax=(1.0, 1.0, 1.0),
        bc=((BC_PERIODIC, BC_PERIODIC),) * 3,
        gamma_ad=5.0 / 3.0, recon=RECON_PLM_MINMOD, riemann=RIEMANN_HLL, use_ct=1,
        rho_floor=1e-10, eps_floor=1e-10, w_max=50.0, c2p_tol=1e-15, c2p_maxit=64,
        shift=(0.0, 0.0, 0.0),
    )
    p.update(kw)
    return p


# --------------------------------------------------------------------------- layout helpers
def ghosts(p):
    """Ghost depth per dimension (0 in an inactive dimension)."""
    tot = (p["nbx"] * p["nx"], p["nby"] * p["ny"], p["nbz"] * p["nz"])
    return tuple(p["ng"] if t > 1 else 0 for t in tot)


def alloc_shape(p):
    gx, gy, gz = ghosts(p)
    nb = p["nbx"] * p["nby"] * p["nbz"]
    return (nb, NV + (1 if p.get("nscalar", 0) else 0), p["nz"] + 2 * gz, p["ny"] + 2 * gy, p["nx"] + 2 * gx)


def n_zones(p):
    return p["nbx"] * p["nx"] * p["nby"] * p["ny"] * p["nbz"] * p["nz"]


def cell_centres(p):
    """Global interior cell-centre coordinates (x[i], y[j], z[k])."""
    out = []
    for d, (nb, n) in enumerate(((p["nbx"], p["nx"]), (p["nby"], p["ny"]), (p["nbz"], p["nz"]))):
        N = nb * n
        dx = (p["xmax"][d] - p["xmin"][d]) / N
        out.append(p["xmin"][d] + (np.arange(N) + 0.5) * dx)
    return out


def node_coords(p):
    out = []
    for d, (nb, n) in enumerate(((p["nbx"], p["nx"]), (p["nby"], p["ny"]), (p["nbz"], p["nz"]))):
        N = nb * n
        dx = (p["xmax"][d] - p["xmin"][d]) / N
        out.append(p["xmin"][d] + np.arange(N + 1) * dx)
    return out


def pad_global(p, q):
    """q: [NV, Nz, Ny, Nx] global interior -> global array with ghosts, filled x then y then z
    (periodic: wrap; outflow: copy of the nearest interior cell)."""
    gx, gy, gz = ghosts(p)
    for axis, g, d in ((3, gx, 0), (2, gy, 1), (1, gz, 2)):
        if g == 0:
            continue
        lo, hi = p["bc"][d]
        if lo != hi:
            raise ValueError("mixed boundary conditions on one axis are not used by any workload")
        w = [(0, 0)] * 4
        w[axis] = (g, g)
        q = np.pad(q, w, mode="wrap" if lo == BC_PERIODIC else "edge")
    return q


def to_blocks(p, qpad):
    """Cut a global padded array [NV, Nz+2gz, Ny+2gy, Nx+2gx] into packed blocks with ghosts."""
    gx, gy, gz = ghosts(p)
    nx, ny, nz = p["nx"], p["ny"], p["nz"]
    out = np.empty(alloc_shape(p), dtype=np.float64)
    for bz in range(p["nbz"]):
        for by in range(p["nby"]):
            for bx in range(p["nbx"]):
                b = (bz * p["nby"] + by) * p["nbx"] + bx
                out[b] = qpad[:, bz * nz: bz * nz + nz + 2 * gz,
                              by * ny: by * ny + ny + 2 * gy,
                              bx * nx: bx * nx + nx + 2 * gx]
    return out


def from_blocks(p, qb):
    """Packed blocks -> global interior array [nvar, Nz, Ny, Nx] (ghosts dropped)."""
    gx, gy, gz = ghosts(p)
    nx, ny, nz = p["nx"], p["ny"], p["nz"]
    qb = np.asarray(qb)
    nvar = qb.shape[1]
    out = np.empty((nvar, p["nbz"] * nz, p["nby"] * ny, p["nbx"] * nx), dtype=qb.dtype)
    for bz in range(p["nbz"]):
        for by in range(p["nby"]):
            for bx in range(p["nbx"]):
                b = (bz * p["nby"] + by) * p["nbx"] + bx
                out[:, bz * nz:(bz + 1) * nz, by * ny:(by + 1) * ny, bx * nx:(bx + 1) * nx] = \
                    qb[b][:, gz: gz + nz, gy: gy + ny, gx: gx + nx]
    return out


def finish(p, q):
    """Global interior primitives -> packed blocks with ghosts."""
    return np.ascontiguousarray(to_blocks(p, pad_global(p, np.ascontiguousarray(q))))


# --------------------------------------------------------------------------- recipe helpers
def node_curl(Ax, Ay, Az, dx, dy, dz):
    """Cell-centred densitised field from nodal vector potential, arrays [Nz+1, Ny+1, Nx+1]:
    B~x = d_y(avg_xz Az) - d_z(avg_xy Ay) etc.  Difference and average operators commute, so
    the corner-centred divergence of the result vanishes to round-off."""
    def mu(a, ax):
        s0 = [slice(None)] * 3; s1 = [slice(None)] * 3
        s0[ax] = slice(0, -1); s1[ax] = slice(1, None)
        return 0.5 * (a[tuple(s0)] + a[tuple(s1)])

    def de(a, ax, h):
        s0 = [slice(None)] * 3; s1 = [slice(None)] * 3
        s0[ax] = slice(0, -1); s1[ax] = slice(1, None)
        return (a[tuple(s1)] - a[tuple(s0)]) / h
    X, Y, Z = 2, 1, 0  # array axes of x, y, z
    Bx = de(mu(mu(Az, X), Z), Y, dy) - de(mu(mu(Ay, X), Y), Z, dz)
    By = de(mu(mu(Ax, X), Y), Z, dz) - de(mu(mu(Az, Y), Z), X, dx)
    Bz = de(mu(mu(Ay, Y), Z), X, dx) - de(mu(mu(Ax, X), Z), Y, dy)
    return Bx, By, Bz


def ks_radius(x, y, z, a):
    R2 = x * x + y * y + z * z
    t = R2 - a * a
    return np.sqrt(0.5 * (t + np.sqrt(t * t + 4.0 * a * a * z * z)))


def ks_sqrt_gamma(x, y, z, M, a):
    r = ks_radius(x, y, z, a)
    H = M * r ** 3 / (r ** 4 + a * a * z * z)
    return np.sqrt(1.0 + 2.0 * H)


def band_field(rng, n, kmin=1, kmax=8, slope=-2.0):
    """Real periodic Gaussian field on an n^3 lattice: integer wavevectors kmin<=|k|<=kmax,
    amplitude ~ |k|^slope, random phases, normalised to unit variance."""
    kx = np.fft.fftfreq(n, 1.0 / n)
    kz = np.fft.rfftfreq(n, 1.0 / n)
    K2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2
    K = np.sqrt(K2)
    sel = (K >= kmin) & (K <= kmax)
    amp = np.zeros_like(K)
    amp[sel] = K[sel] ** slope
    ph = rng.uniform(0.0, 2.0 * np.pi, size=K.shape)
    g = rng.standard_normal(K.shape)
    f = np.fft.irfftn(amp * g * np.exp(1j * ph), s=(n, n, n), axes=(0, 1, 2))
    f -= f.mean()
    f /= f.std()
    return f


def solenoidal_from_potential(a0, a1, a2, n):
    """curl of a periodic vector field (spectral), arrays indexed [z][y][x]."""
    k = 2.0 * np.pi * np.fft.fftfreq(n, 1.0 / n)
    kr = 2.0 * np.pi * np.fft.rfftfreq(n, 1.0 / n)
    KZ, KY, KX = k[:, None, None], k[None, :, None], kr[None, None, :]
    fx, fy, fz = (np.fft.rfftn(a) for a in (a0, a1, a2))
    cx = 1j * (KY * fz - KZ * fy)
    cy = 1j * (KZ * fx - KX * fz)
    cz = 1j * (KX * fy - KY * fx)
    return tuple(np.fft.irfftn(c, s=(n, n, n), axes=(0, 1, 2)) for c in (cx, cy, cz))


# --------------------------------------------------------------------------- the five configs
def shock_tube(n=256, recon=RECON_PLM_MINMOD, ng=2):
    """Config 1: 1-D relativistic MHD shock tube (PAPER.md:443-445 shape; states from BASELINE.json)."""
    p = default_params(nx=n, ng=ng, gamma_ad=2.0, recon=recon, riemann=RIEMANN_HLL,
                       bc=((BC_OUTFLOW, BC_OUTFLOW),) * 3, xmin=(0.0, 0.0, 0.0), xmax=(1.0, 1.0, 1.0))
    x = cell_centres(p)[0]
    left = x < 0.5
    q = np.zeros((NV, 1, 1, n))
    q[0, 0, 0] = np.where(left, 1.0, 0.125)
    q[4, 0, 0] = np.where(left, 1.0, 0.1) / (p["gamma_ad"] - 1.0)
    q[5, 0, 0] = 0.5
    q[6, 0, 0] = np.where(left, 1.0, -1.0)
    return dict(name="cfg1_shock_tube", params=p, prim=finish(p, q), cfl=0.4, t_end=0.4, steps=None)


def periodic_box(n=64, seed=SEED0 + 2, recon=RECON_PLM_MC, riemann=RIEMANN_LLF):
    """Config 2: 3-D periodic box with small seeded perturbations."""
    p = default_params(nx=n, ny=n, nz=n, ng=4, gamma_ad=5.0 / 3.0, recon=recon, riemann=riemann)
    rng = np.random.default_rng(seed)
    q = np.zeros((NV, n, n, n))
    q[0] = 1.0 + 1e-3 * rng.uniform(-1, 1, (n, n, n))
    P = 1.0 + 1e-3 * rng.uniform(-1, 1, (n, n, n))
    v = (0.1 / np.sqrt(3.0)) * rng.uniform(-1, 1, (3, n, n, n))
    W = 1.0 / np.sqrt(1.0 - (v ** 2).sum(0))
    q[1:4] = W * v
    q[4] = P / (p["gamma_ad"] - 1.0)
    q[5], q[6], q[7] = 1.0, 0.5, 0.25
    return dict(name="cfg2_periodic_box", params=p, prim=finish(p, q), cfl=0.4, steps=100)


def _torus_prims(p, seed):
    M, a, gam = p["bh_mass"], p["bh_spin"], p["gamma_ad"]
    x, y, z = cell_centres(p)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    rng = np.random.default_rng(seed)
    shape = X.shape
    wcyl = np.sqrt(X * X + Y * Y)
    rho = np.maximum(1e-4, np.exp(-((wcyl - 10.0) ** 2 + Z * Z) / 8.0))
    P = 0.01 * rho ** gam * (1.0 + 0.02 * rng.uniform(-1, 1, shape))
    # Keplerian-like azimuthal motion given directly as the primitive u~ (any u~ is subluminal)
    uK = np.where(rho > 1e-4, np.minimum(0.5, 1.0 / np.sqrt(np.maximum(wcyl, 1e-30))), 0.0)
    q = np.zeros((NV,) + shape)
    q[0] = rho
    q[1] = -uK * Y / np.maximum(wcyl, 1e-30)
    q[2] = uK * X / np.maximum(wcyl, 1e-30)
    q[4] = P / (gam - 1.0)
    # B from nodal A_phi = max(rho - 0.2, 0)
    xn, yn, zn = node_coords(p)
    Zn, Yn, Xn = np.meshgrid(zn, yn, xn, indexing="ij")
    wn2 = np.maximum(Xn * Xn + Yn * Yn, 1e-30)
    rhon = np.maximum(1e-4, np.exp(-((np.sqrt(wn2) - 10.0) ** 2 + Zn * Zn) / 8.0))
    Aphi = np.maximum(rhon - 0.2, 0.0)
    Ax, Ay, Az = -Yn * Aphi / wn2, Xn * Aphi / wn2, np.zeros_like(Aphi)
    dx = [(p["xmax"][d] - p["xmin"][d]) / N for d, N in enumerate((len(x), len(y), len(z)))]
    Bx, By, Bz = node_curl(Ax, Ay, Az, *dx)
    sg = ks_sqrt_gamma(X, Y, Z, M, a)
    q[5], q[6], q[7] = Bx / sg, By / sg, Bz / sg
    return q


def kerr_schild_torus(n=128, seed=SEED0 + 3, spin=0.9375, half=20.0, recon=RECON_PLM_MINMOD):
    """Config 3: single 3-D block in Cartesian Kerr-Schild coordinates, torus-like data."""
    p = default_params(metric=KERR_SCHILD, bh_mass=1.0, bh_spin=spin, r_excise=2.0,
                       nx=n, ny=n, nz=n, ng=4, xmin=(-half,) * 3, xmax=(half,) * 3,
                       bc=((BC_OUTFLOW, BC_OUTFLOW),) * 3, gamma_ad=4.0 / 3.0,
                       recon=recon, riemann=RIEMANN_HLL,
                       rho_floor=1e-6, eps_floor=1e-6, w_max=10.0)
    q = _torus_prims(p, seed)
    return dict(name="cfg3_kerr_schild_torus", params=p, prim=finish(p, q), cfl=0.4, steps=50)


def turbulence_box(n=256, seed=SEED0 + 4, recon=RECON_WENO5Z, riemann=RIEMANN_HLL):
    """Config 4: periodic turbulence-like box (the roofline-target workload at n=256)."""
    p = default_params(nx=n, ny=n, nz=n, ng=4, gamma_ad=5.0 / 3.0, recon=recon, riemann=riemann)
    rng = np.random.default_rng(seed)
    kmax = min(8, n // 4)
    q = np.zeros((NV, n, n, n))
    q[0] = np.exp(0.5 * band_field(rng, n, 1, kmax))
    P = np.exp(0.5 * band_field(rng, n, 1, kmax))
    q[4] = P / (p["gamma_ad"] - 1.0)
    ux, uy, uz = solenoidal_from_potential(*(band_field(rng, n, 1, kmax) for _ in range(3)), n)
    rms = np.sqrt(np.mean(ux ** 2 + uy ** 2 + uz ** 2))
    q[1], q[2], q[3] = (0.3 / rms) * ux, (0.3 / rms) * uy, (0.3 / rms) * uz
    # nodal vector potential on the periodic node lattice (same lattice shifted by half a cell)
    A = [np.pad(band_field(rng, n, 1, kmax), ((0, 1),) * 3, mode="wrap") for _ in range(3)]
    Bx, By, Bz = node_curl(A[0], A[1], A[2], 1.0 / n, 1.0 / n, 1.0 / n)
    s = np.sqrt(2.0 * P.sum() / (10.0 * (Bx ** 2 + By ** 2 + Bz ** 2).sum()))   # beta = 2P/B^2 = 10
    q[5], q[6], q[7] = s * Bx, s * By, s * Bz
    return dict(name="cfg4_turbulence_box", params=p, prim=finish(p, q), cfl=0.4, steps=20)


def packed_blocks(nb=(8, 8, 8), n=32, seed=SEED0 + 5, spin=0.5, half=20.0):
    """Config 5: many small blocks tiling a Kerr-Schild domain (512 x 32^3 at full size)."""
    half = (half, half, half * nb[2] / nb[0])
    p = default_params(metric=KERR_SCHILD, bh_mass=1.0, bh_spin=spin, r_excise=2.0,
                       nbx=nb[0], nby=nb[1], nbz=nb[2], nx=n, ny=n, nz=n, ng=4,
                       xmin=tuple(-h for h in half), xmax=half,
                       bc=((BC_OUTFLOW, BC_OUTFLOW),) * 3, gamma_ad=4.0 / 3.0,
                       recon=RECON_PLM_MINMOD, riemann=RIEMANN_HLL,
                       rho_floor=1e-6, eps_floor=1e-6, w_max=10.0)
    q = _torus_prims(p, seed)
    return dict(name="cfg5_packed_blocks", params=p, prim=finish(p, q), cfl=0.4, steps=20)


def sedov_blast(n=128, E=1e-5, r_init=0.1, recon=RECON_PLM_MINMOD):
    """the paper's Sedov-Taylor blast (E = 1e-5 deposited in all cells with
    r < r_init = 0.1, rho = 1, p = 1e-7, domain [-1,1]^d) as a uniform 3-D block with B = 0 and Gamma = 5/3 -- the
    shape of the paper's weak-scaling workload (3-D Sedov, 128^3 per start).  The energy is spread evenly
    over the cells whose centres lie inside r_init, so that the deposited total is exactly E.  No RNG."""
    p = default_params(nx=n, ny=n, nz=n, ng=4, gamma_ad=5.0 / 3.0, recon=recon, riemann=RIEMANN_HLL,
                       bc=((BC_OUTFLOW, BC_OUTFLOW),) * 3, xmin=(-1.0,) * 3, xmax=(1.0,) * 3)
    x, y, z = cell_centres(p)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    inside = X * X + Y * Y + Z * Z < r_init * r_init
    dV = (2.0 / n) ** 3
    q = np.zeros((NV, n, n, n))
    q[0] = 1.0
    q[4] = 1e-7 / (p["gamma_ad"] - 1.0)
    if not inside.any():
        raise ValueError("sedov_blast: no cell centre inside r_init at this resolution")
    q[4][inside] += E / (inside.sum() * dV)
    return dict(name="next2_sedov_blast", params=p, prim=finish(p, q), cfl=0.4, steps=20)


def linear_mode(kind, rho0, P0, gam, Bpar, Bperp, direction=1):
    """Closed-form linear eigenmode of ideal relativistic MHD about a fluid at rest (the exact solution the linear-wave
    inputs sample; PAPER.md:430-441 names the four families).  Wave normal n, background field B = Bpar n + Bperp t with t a
    unit vector orthogonal to n, third direction z = n x t.  Linearising Eq.1-3 about v = 0 with a = rho h, E = a + B^2:
      drho = rho v_n / lam,  dP = a c_s^2 v_n / lam,  dB_t = (Bperp v_n - Bpar v_t)/lam,  dB_z = -Bpar v_z / lam,
      [lam^2 (a + Bperp^2) - a c_s^2 - Bperp^2] v_n - Bpar Bperp (lam^2 - 1) v_t = 0,
      Bpar Bperp (lam^2 - 1) v_n - [lam^2 (a + Bpar^2) - Bpar^2] v_t = 0,       E lam^2 v_z = Bpar^2 v_z,
    so lam^2 solves  E s^2 - (B^2 + a c_s^2 + c_s^2 Bpar^2) s + c_s^2 Bpar^2 = 0  (fast: larger root, slow: smaller root),
    lam_Alfven^2 = Bpar^2 / E, and with Bperp = 0 the roots are c_s^2 (sound) and the Alfven speed.
    Returns the perturbation per unit amplitude (normalised to drho = rho0 for the compressive modes, dv_z = 1 for Alfven)
    of a wave travelling along direction * n: dict(lam, drho, dP, dvn, dvt, dvz, dBt, dBz)."""
    a = rho0 + P0 / (gam - 1.0) + P0
    cs2 = gam * P0 / a
    B2 = Bpar * Bpar + Bperp * Bperp
    E = a + B2
    out = dict(drho=0.0, dP=0.0, dvn=0.0, dvt=0.0, dvz=0.0, dBt=0.0, dBz=0.0)
    if kind == "alfven":
        lam = direction * abs(Bpar) / np.sqrt(E)
        out.update(lam=lam, dvz=1.0, dBz=-Bpar / lam)
        return out
    if kind == "sound":
        if Bperp != 0.0:
            raise ValueError("a pure sound wave needs the field along the wave normal (or none)")
        s = cs2
    else:
        b = B2 + a * cs2 + cs2 * Bpar * Bpar
        disc = np.sqrt(b * b - 4.0 * E * cs2 * Bpar * Bpar)
        if kind == "fast":
            s = (b + disc) / (2.0 * E)
        elif kind == "slow":
            s = 2.0 * cs2 * Bpar * Bpar / (b + disc)      # the smaller root, without cancellation
        else:
            raise ValueError(kind)
    lam = direction * np.sqrt(s)
    vn = lam                                              # drho = rho0
    vt = Bpar * Bperp * (s - 1.0) * vn / (s * (a + Bpar * Bpar) - Bpar * Bpar) if Bperp != 0.0 else 0.0
    out.update(lam=lam, drho=rho0, dP=a * cs2, dvn=vn, dvt=vt, dBt=(Bperp * vn - Bpar * vt) / lam)
    return out


WAVE_KINDS = ("sound", "alfven", "fast", "slow")
WAVE_BPAR, WAVE_BPERP = 1.0, 1.5                          # background field of the magnetosonic waves (the paper gives none)


def _wave_background(kind):
    """(Bpar, Bperp) of the background of each family: none for sound, along n for Alfven, oblique for fast / slow."""
    return {"sound": (0.0, 0.0), "alfven": (1.0, 0.0)}.get(kind, (WAVE_BPAR, WAVE_BPERP))


def linear_wave_1d(n=64, kind="sound", A=1e-6, recon=RECON_PLM_MC, riemann=RIEMANN_HLL):
    """SURVEY.md 8(c) pin P9: 1-D linear wave on the periodic unit interval, Minkowski, Gamma = 5/3, rho = P = 1 at rest,
    one wavelength, travelling towards +x: the eigenmode of `linear_mode` with n = x, t = y.  Returns the workload plus
    the period and the variable the L1 norm of Eq.61 is taken of.  No RNG."""
    gam = 5.0 / 3.0
    p = default_params(nx=n, ng=2 if recon in (1, 2) else 3, gamma_ad=gam, recon=recon, riemann=riemann)
    x = cell_centres(p)[0]
    s = np.sin(2.0 * np.pi * x)
    Bpar, Bperp = _wave_background(kind)
    m = linear_mode(kind, 1.0, 1.0, gam, Bpar, Bperp, +1)
    q = np.zeros((NV, 1, 1, n))
    q[0, 0, 0] = 1.0 + A * m["drho"] * s
    q[4, 0, 0] = (1.0 + A * m["dP"] * s) / (gam - 1.0)
    v = A * np.array([m["dvn"], m["dvt"], m["dvz"]])[:, None] * s[None, :]
    W = 1.0 / np.sqrt(1.0 - (v * v).sum(0))
    q[1:4, 0, 0] = W * v
    q[5, 0, 0] = Bpar
    q[6, 0, 0] = Bperp + A * m["dBt"] * s
    q[7, 0, 0] = A * m["dBz"] * s
    var = 7 if kind == "alfven" else 0
    return dict(name=f"p9_{kind}_wave", params=p, prim=finish(p, q), cfl=0.4, steps=None, period=1.0 / abs(m["lam"]), var=var,
                amplitude=A * (abs(m["dBz"]) if kind == "alfven" else 1.0), mode=m)


def boosted_linear_wave(n=64, kind="sound", boost=0.617213, A=1e-6, recon=RECON_PLM_MC):
    """the paper's linear-wave set-up: 2-D, Gamma = 5/3, flat metric with
    coordinate boosts v_x = v_y = 0.617213, periodic unit square, the four families sound, Alfven, fast and slow magnetosonic
    (PAPER.md:441).  Background rho = P = 1 at rest in the unboosted frame; a plane wave of amplitude A with phase
    2 pi (x + y), wave normal n = (1,1)/sqrt 2, travelling against the boost (so that one period of the pattern in the boosted
    coordinates is short); t = (-1,1)/sqrt 2.  Sound: no field; Alfven: B_0 = 1 along n; fast / slow: B_0 = 1 n + 1.5 t (the
    paper prints no background).  The perturbation is the closed-form eigenmode of `linear_mode`.
    Returns the workload plus the period T of the pattern and the index of the variable the L1 norm of Eq.61 is taken
    of.  No RNG."""
    gam = 5.0 / 3.0
    p = default_params(metric=MINKOWSKI_BOOSTED, shift=(boost, boost, 0.0), nx=n, ny=n, nz=1, ng=2 if recon in (1, 2) else 3,
                       gamma_ad=gam, recon=recon, riemann=RIEMANN_HLL)
    x, y, _ = cell_centres(p)
    Y, X = np.meshgrid(y, x, indexing="ij")
    s = np.sin(2.0 * np.pi * (X + Y))[None]           # [1, Ny, Nx]
    Bpar, Bperp = _wave_background(kind)
    m = linear_mode(kind, 1.0, 1.0, gam, Bpar, Bperp, -1)
    r2 = np.sqrt(0.5)
    nx_, ny_, tx_, ty_ = r2, r2, -r2, r2
    q = np.zeros((NV, 1, n, n))
    q[0] = 1.0 + A * m["drho"] * s
    q[4] = (1.0 + A * m["dP"] * s) / (gam - 1.0)
    vn, vt, vz = A * m["dvn"] * s, A * m["dvt"] * s, A * m["dvz"] * s
    W = 1.0 / np.sqrt(1.0 - (vn * vn + vt * vt + vz * vz))
    q[1] = W * (vn * nx_ + vt * tx_)
    q[2] = W * (vn * ny_ + vt * ty_)
    q[3] = W * vz
    Bt = Bperp + A * m["dBt"] * s
    q[5] = Bpar * nx_ + Bt * tx_
    q[6] = Bpar * ny_ + Bt * ty_
    q[7] = A * m["dBz"] * s
    var = 7 if kind == "alfven" else 0
    T = 1.0 / (np.sqrt(2.0) * abs(m["lam"]) + 2.0 * boost)
    return dict(name=f"next4_boosted_{kind}_wave", params=p, prim=finish(p, q), cfl=0.4, steps=None, period=T, var=var,
                amplitude=A * (abs(m["dBz"]) if kind == "alfven" else 1.0), mode=m)


def with_scalar(w, X, scalar_min=0.0, scalar_max=1.0):
    """Workload `w` with a passive scalar (Eq.14; the paper's use is the electron fraction Y_e)
    appended as variable 8.  X: global interior array [Nz, Ny, Nx] of the advected quantity."""
    p0 = w["params"]
    q = np.concatenate([from_blocks(p0, w["prim"]), np.asarray(X, dtype=np.float64)[None]], axis=0)
    p = dict(p0, nscalar=1, scalar_min=float(scalar_min), scalar_max=float(scalar_max))
    return dict(w, name=w["name"] + "_scalar", params=p, prim=finish(p, q))


def smooth_scalar(p, seed, lo=0.1, hi=0.5):
    """A seeded smooth field in [lo, hi] on the global interior grid: a few low random Fourier modes (Y_e-like values)."""
    rng = np.random.default_rng(seed)
    x, y, z = cell_centres(p)
    L = [p["xmax"][d] - p["xmin"][d] for d in range(3)]
    X = np.zeros((len(z), len(y), len(x)))
    for _ in range(4):
        k = rng.integers(0, 3, size=3)
        ph = rng.uniform(0.0, 2.0 * np.pi, size=3)
        X += (np.cos(2 * np.pi * k[0] * (x - p["xmin"][0]) / L[0] + ph[0])[None, None, :]
              * np.cos(2 * np.pi * k[1] * (y - p["xmin"][1]) / L[1] + ph[1])[None, :, None]
              * np.cos(2 * np.pi * k[2] * (z - p["xmin"][2]) / L[2] + ph[2])[:, None, None])
    X = (X - X.min()) / max(X.max() - X.min(), 1e-300)
    return lo + (hi - lo) * X


def smooth_periodic_prims(p, device="cpu"):
    """Analytic smooth periodic primitives for a single-block periodic Minkowski mesh, written with torch on `device`
    straight into the allocated layout [1, 8, nz+2g, ny+2g, nx+2g] (the functions are periodic, so the ghost zones are
    consistent by construction).  For meshes too large to build on the host (the > 2^31-element indexing test)."""
    import math
    import torch
    assert p["nbx"] == p["nby"] == p["nbz"] == 1
    gx, gy, gz = ghosts(p)
    co = []
    for d, (n, g) in enumerate(((p["nx"], gx), (p["ny"], gy), (p["nz"], gz))):
        i = torch.arange(-g, n + g, dtype=torch.float64, device=device)
        co.append(2.0 * math.pi * (i + 0.5) / n)                # phase 2 pi (x - xmin)/L at the cell centres
    x = co[0][None, None, :]; y = co[1][None, :, None]; z = co[2][:, None, None]
    q = torch.empty((1, NV, len(co[2]), len(co[1]), len(co[0])), dtype=torch.float64, device=device)
    q[0, 0] = 1.0 + 0.2 * torch.sin(x) * torch.cos(y) + 0.1 * torch.sin(2.0 * z)
    q[0, 1] = 0.2 * torch.sin(y) * torch.cos(z)
    q[0, 2] = 0.15 * torch.sin(z + 0.3) * torch.cos(x)
    q[0, 3] = -0.1 * torch.sin(x + y)
    q[0, 4] = 1.5 + 0.3 * torch.cos(x) * torch.sin(z) + 0.1 * torch.cos(2.0 * y)
    q[0, 5] = 0.5 + 0.1 * torch.sin(y) + 0.0 * x + 0.0 * z
    q[0, 6] = 0.3 + 0.1 * torch.sin(z) + 0.0 * x + 0.0 * y
    q[0, 7] = 0.2 + 0.1 * torch.sin(x) + 0.0 * y + 0.0 * z
    return q


def reblock(p, prim_blocks, nb):
    """Same global data on a different block decomposition (for the block-invariance pin)."""
    tot = (p["nbx"] * p["nx"], p["nby"] * p["ny"], p["nbz"] * p["nz"])
    p2 = dict(p)
    p2.update(nbx=nb[0], nby=nb[1], nbz=nb[2], nx=tot[0] // nb[0], ny=tot[1] // nb[1], nz=tot[2] // nb[2])
    return p2, finish(p2, from_blocks(p, prim_blocks))
