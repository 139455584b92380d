// oracle/orc.cpp — CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow, double-precision restatement of the ideal-GRMHD finite-volume update of
// PHOEBUS (arXiv:2410.09146; /root/reference/PAPER.md) in the Valencia formulation, written
// from the paper's equations (Eq.1-13; Appendix B) and,
// where the paper is silent, from the readings C1-C10 of SURVEY.md section 8(c) which DESIGN.md
// section 3 lists one by one.  It shares no code with the CUDA path under
// paper_2410_09146_b200/csrc and neither includes the other.  Only tests/, bench.py's
// cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load it.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC   (strict IEEE, no FMA contraction).
// OpenMP is used only over independent cells/faces; every cell's arithmetic is sequential and
// written in the order of the formulas it cites.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 uniform state bitwise, P2 conservation,
// P3 corner div B, P4 round trip, P5 algebraic identities against T^{mu nu} of Eq.9, P6
// Kerr-Schild identities and derivatives, P7 sources against the printed Eq.4 forms, P8 wave
// speeds against the covariant dispersion relation, P9 linear-wave convergence, P10 shock-tube
// structure, P11 block invariance, P12 WENO5-Z order, P12b/c WENO5-Z-AOAH, P12d MP5, P13 Bondi
// inflow stationary in Kerr-Schild (a = 0), P14 Sedov-Taylor shock radius, P15 boosted linear waves.
// Parity-unpinned parts: the absolute accuracy of the synthetic configs 3-5 for spin a != 0 (no
// printed values exist in the paper for this path, no closed-form solution is used there).
//
// P16 passive scalar (Eq.14): constant X stays constant, sum of sqrt(gamma) D X conserved, smooth profile advected at
// second order, bounds; P17 floor forms of PAPER.md:288 against the closed-form Kerr-Schild radius on the axis, in the
// equatorial plane and for a = 0.  P18 (tests/test_oracle_pins_positivity.py): the positivity fallback of the fifth-order
// reconstructions in block_fluxes (which cell, which direction, all variables, threshold just below the floors at the cell centre,
// never for piecewise-linear schemes) on hand-worked stencils.  P9 / P15 cover the four linear-wave families of PAPER.md:441
// (tests/test_oracle_pins_waves.py: eigenmodes against a numerical flux Jacobian of Eq.2-3 written in the test); P19: a
// finite-amplitude entropy wave, an exact nonlinear solution, is carried at alpha v - beta at second order; con2prim against a
// 50-digit inversion (tests/test_c2p_accuracy.py).
//
// Layout of every field: [block][var][k][j][i], i fastest; var order of primitives
// P=(rho, W v^1, W v^2, W v^3, rho*eps, B^1, B^2, B^3) (Eq.13) and conserved, stored densitised,
// sqrt(gamma)*(D, S_1, S_2, S_3, tau, B^1, B^2, B^3) (Eq.1-2).
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>

extern "C" {
typedef struct {
  int metric;  double bh_mass, bh_spin, r_excise;
  int nbx, nby, nbz;
  int nx, ny, nz;
  int ng;
  double xmin[3], xmax[3];
  int bc[3][2];
  double gamma_ad;  int recon, riemann, use_ct;
  double rho_floor, eps_floor, w_max;
  double c2p_tol;  int c2p_maxit;
  double shift[3];   /* metric 2: flat metric in coordinates boosted by x' = x - shift*t */
  int nscalar;       /* 0 or 1 passive scalar X carried as variable 8 of every field (Eq.14) */
  double scalar_min, scalar_max;   /* X is kept inside these bounds */
  int floor_form;    /* 0 rho0; 1 rho0 exp(-alpha x1); 2 rho0 x1^-alpha; 3 rho0 r^-alpha (x1 = r here) */
  double floor_alpha_rho, floor_alpha_eps;
} orc_params;
}

namespace {

enum { NV = 8, RHO = 0, UX = 1, UY = 2, UZ = 3, UU = 4, BX = 5, BY = 6, BZ = 7 };
enum { CD = 0, CS1 = 1, CS2 = 2, CS3 = 3, CTAU = 4 };
enum { M_RHO_FLOOR = 1, M_EPS_FLOOR = 2, M_EPS_CLIPPED = 4, M_W_CEIL = 8, M_NOCONV = 16, M_BAD_INPUT = 32,
       M_EXCISED = 64, M_SCALAR_CLIPPED = 128 };
enum { XS = 8, NVMAX = 9 };   // index of the passive scalar (primitive X, conserved sqrt(gamma) D X) when nscalar = 1

double g_last_margin = 1e300;   // smallest relative distance of any c2p decision to its threshold

// ------------------------------------------------------------------------------------------ C1
struct Grid {
  orc_params p;
  int nb[3], n[3], g[3], na[3], N[3];
  bool act[3];
  double dx[3];
  long ncell;   // allocated cells per block
  int nblk;
  int nv;       // variables per field: 8 + nscalar
  explicit Grid(const orc_params& q) : p(q) {
    nv = NV + (q.nscalar > 0 ? 1 : 0);
    nb[0] = q.nbx; nb[1] = q.nby; nb[2] = q.nbz;
    n[0] = q.nx; n[1] = q.ny; n[2] = q.nz;
    for (int d = 0; d < 3; ++d) {
      N[d] = nb[d] * n[d];
      act[d] = N[d] > 1;
      g[d] = act[d] ? q.ng : 0;
      na[d] = n[d] + 2 * g[d];
      dx[d] = (q.xmax[d] - q.xmin[d]) / N[d];
    }
    ncell = (long)na[0] * na[1] * na[2];
    nblk = nb[0] * nb[1] * nb[2];
  }
  long idx(int b, int v, int k, int j, int i) const {
    return (((long)b * nv + v) * na[2] + k) * (long)na[1] * na[0] + (long)j * na[0] + i;
  }
  long cidx(int b, int k, int j, int i) const {   // one-variable arrays (mask)
    return ((long)b * na[2] + k) * (long)na[1] * na[0] + (long)j * na[0] + i;
  }
  void bcoord(int b, int bc[3]) const { bc[0] = b % nb[0]; bc[1] = (b / nb[0]) % nb[1]; bc[2] = b / (nb[0] * nb[1]); }
  // coordinate of the centre of local cell index il along d in block b
  double xc(int d, int b, int il) const {
    int c[3]; bcoord(b, c);
    long gi = (long)c[d] * n[d] + (il - g[d]);
    return p.xmin[d] + ((double)gi + 0.5) * dx[d];
  }
  // coordinate of the lower face of that cell
  double xf(int d, int b, int il) const {
    int c[3]; bcoord(b, c);
    long gi = (long)c[d] * n[d] + (il - g[d]);
    return p.xmin[d] + (double)gi * dx[d];
  }
};

// ------------------------------------------------------------------------------------------ C2
// Covariant 4-metric g_{mu nu}(x).  Minkowski: eta.  Kerr-Schild (Cartesian, ingoing):
// g = eta + 2 H l l, r^4 - (R^2-a^2) r^2 - a^2 z^2 = 0, H = M r^3/(r^4+a^2 z^2),
// l = (1, (r x + a y)/(r^2+a^2), (r y - a x)/(r^2+a^2), z/r).
void ks_scalars(const orc_params& p, const double x[3], double& r, double& H, double l[4]) {
  const double a = p.bh_spin, M = p.bh_mass;
  const double R2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
  const double t = R2 - a * a;
  r = std::sqrt(0.5 * (t + std::sqrt(t * t + 4.0 * a * a * x[2] * x[2])));
  H = M * r * r * r / (r * r * r * r + a * a * x[2] * x[2]);
  l[0] = 1.0;
  l[1] = (r * x[0] + a * x[1]) / (r * r + a * a);
  l[2] = (r * x[1] - a * x[0]) / (r * r + a * a);
  l[3] = x[2] / r;
}

void metric4(const orc_params& p, const double x[3], double g[4][4]) {
  for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) g[m][n] = 0.0;
  g[0][0] = -1.0; g[1][1] = g[2][2] = g[3][3] = 1.0;
  if (p.metric == 1) {
    double r, H, l[4];
    ks_scalars(p, x, r, H, l);
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) g[m][n] += 2.0 * H * l[m] * l[n];
  }
  if (p.metric == 2) {
    // "flat metric with coordinate boosts" (reading C2b): x = x' + v t turns
    // ds^2 = -dt^2 + dx^2 into -(1 - v^2) dt^2 + 2 v_i dx'^i dt + dx'^2, i.e. alpha = 1, beta^i = v^i, gamma_ij = delta_ij
    double v2 = 0.0;
    for (int i = 0; i < 3; ++i) { g[0][i + 1] = g[i + 1][0] = p.shift[i]; v2 += p.shift[i] * p.shift[i]; }
    g[0][0] = -1.0 + v2;
  }
}

// d_k g_{mu nu}, analytic (d_t = 0).  dg[k][mu][nu], k = 0,1,2 for x,y,z.
void metric4_derivs(const orc_params& p, const double x[3], double dg[3][4][4]) {
  for (int k = 0; k < 3; ++k) for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) dg[k][m][n] = 0.0;
  if (p.metric != 1) return;
  const double a = p.bh_spin, M = p.bh_mass;
  double r, H, l[4];
  ks_scalars(p, x, r, H, l);
  const double R2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
  const double z = x[2];
  const double r2 = r * r, r3 = r2 * r, r4 = r2 * r2;
  const double den = r4 + a * a * z * z;
  const double ra = r2 + a * a;
  for (int k = 0; k < 3; ++k) {
    const double dkz = (k == 2) ? 1.0 : 0.0, dkx = (k == 0) ? 1.0 : 0.0, dky = (k == 1) ? 1.0 : 0.0;
    const double rk = (x[k] * r + a * a * z * dkz / r) / (2.0 * r2 - R2 + a * a);
    const double Hk = M * (3.0 * r2 * rk * den - r3 * (4.0 * r3 * rk + 2.0 * a * a * z * dkz)) / (den * den);
    double lk[4];
    lk[0] = 0.0;
    lk[1] = ((rk * x[0] + r * dkx + a * dky) * ra - (r * x[0] + a * x[1]) * 2.0 * r * rk) / (ra * ra);
    lk[2] = ((rk * x[1] + r * dky - a * dkx) * ra - (r * x[1] - a * x[0]) * 2.0 * r * rk) / (ra * ra);
    lk[3] = dkz / r - z * rk / r2;
    for (int m = 0; m < 4; ++m)
      for (int n = 0; n < 4; ++n)
        dg[k][m][n] = 2.0 * Hk * l[m] * l[n] + 2.0 * H * (lk[m] * l[n] + l[m] * lk[n]);
  }
}

// 3+1 split of a 4-metric: gamma_ij = g_ij, beta_i = g_0i, beta^i = gamma^ij beta_j,
// alpha^2 = beta^i beta_i - g_00, sqrt(gamma) = sqrt(det gamma_ij).
struct Geo {
  double alpha, bu[3], bl[3], gl[3][3], gu[3][3], sg;
};

Geo split31(const double g[4][4]) {
  Geo G;
  for (int i = 0; i < 3; ++i) { G.bl[i] = g[0][i + 1]; for (int j = 0; j < 3; ++j) G.gl[i][j] = g[i + 1][j + 1]; }
  const double (*a)[3] = G.gl;
  const double det = a[0][0] * (a[1][1] * a[2][2] - a[1][2] * a[2][1]) - a[0][1] * (a[1][0] * a[2][2] - a[1][2] * a[2][0]) +
                     a[0][2] * (a[1][0] * a[2][1] - a[1][1] * a[2][0]);
  G.gu[0][0] = (a[1][1] * a[2][2] - a[1][2] * a[2][1]) / det;
  G.gu[0][1] = (a[0][2] * a[2][1] - a[0][1] * a[2][2]) / det;
  G.gu[0][2] = (a[0][1] * a[1][2] - a[0][2] * a[1][1]) / det;
  G.gu[1][0] = G.gu[0][1];
  G.gu[1][1] = (a[0][0] * a[2][2] - a[0][2] * a[2][0]) / det;
  G.gu[1][2] = (a[0][2] * a[1][0] - a[0][0] * a[1][2]) / det;
  G.gu[2][0] = G.gu[0][2];
  G.gu[2][1] = G.gu[1][2];
  G.gu[2][2] = (a[0][0] * a[1][1] - a[0][1] * a[1][0]) / det;
  double b2 = 0.0;
  for (int i = 0; i < 3; ++i) {
    G.bu[i] = 0.0;
    for (int j = 0; j < 3; ++j) G.bu[i] += G.gu[i][j] * G.bl[j];
    b2 += G.bu[i] * G.bl[i];
  }
  G.alpha = std::sqrt(b2 - g[0][0]);
  G.sg = std::sqrt(det);
  return G;
}

Geo geo_at(const orc_params& p, const double x[3]) {
  double g[4][4];
  metric4(p, x, g);
  return split31(g);
}

// ------------------------------------------------------------------------------------------ C3
// Everything Eq.2, 3, 5-7, 10-12 need at one point.
struct Fluid {
  double W, v[3], vl[3], Bu[3], Bl[3], Bv, B2, ab0, b2, bl[3], P, rhoh, vt[3], rho;
};

Fluid fluid_at(const double q[NV], const Geo& G, double gam) {
  Fluid f;
  double uu = 0.0;
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) uu += G.gl[i][j] * q[UX + i] * q[UX + j];
  f.W = std::sqrt(1.0 + uu);                                  // W^2 = 1 + gamma_ij u~^i u~^j
  for (int i = 0; i < 3; ++i) { f.v[i] = q[UX + i] / f.W; f.Bu[i] = q[BX + i]; }
  for (int i = 0; i < 3; ++i) {
    f.vl[i] = 0.0; f.Bl[i] = 0.0;
    for (int j = 0; j < 3; ++j) { f.vl[i] += G.gl[i][j] * f.v[j]; f.Bl[i] += G.gl[i][j] * f.Bu[j]; }
  }
  f.Bv = 0.0; f.B2 = 0.0;
  for (int i = 0; i < 3; ++i) { f.Bv += f.Bu[i] * f.vl[i]; f.B2 += f.Bu[i] * f.Bl[i]; }
  f.ab0 = f.W * f.Bv;                                         // alpha b^0, Eq.10
  f.b2 = f.B2 / (f.W * f.W) + f.Bv * f.Bv;                    // Eq.12 with alpha b^0 = W (B.v)
  for (int i = 0; i < 3; ++i) f.bl[i] = f.Bl[i] / f.W + f.ab0 * f.vl[i];   // Eq.11 lowered
  f.rho = q[RHO];
  f.P = (gam - 1.0) * q[UU];                                  // ideal gas
  f.rhoh = q[RHO] + q[UU] + f.P;
  for (int i = 0; i < 3; ++i) f.vt[i] = G.alpha * f.v[i] - G.bu[i];        // Eq.6
  return f;
}

// Eq.2 (not densitised)
void cons_at(const double q[NV], const Geo& G, double gam, double U[NV]) {
  const Fluid f = fluid_at(q, G, gam);
  const double w = (f.rhoh + f.b2) * f.W * f.W;
  U[CD] = f.rho * f.W;
  for (int j = 0; j < 3; ++j) U[CS1 + j] = w * f.vl[j] - f.ab0 * f.bl[j];
  U[CTAU] = w - (f.P + 0.5 * f.b2) - f.ab0 * f.ab0 - U[CD];
  for (int k = 0; k < 3; ++k) U[BX + k] = f.Bu[k];
}

// Eq.3, direction d (not densitised)
void flux_at(const double q[NV], const Geo& G, double gam, int d, double F[NV]) {
  const Fluid f = fluid_at(q, G, gam);
  double U[NV];
  cons_at(q, G, gam, U);
  const double pt = f.P + 0.5 * f.b2;
  F[CD] = U[CD] * f.vt[d] / G.alpha;
  for (int j = 0; j < 3; ++j)
    F[CS1 + j] = U[CS1 + j] * f.vt[d] / G.alpha + pt * (j == d ? 1.0 : 0.0) - f.bl[j] * f.Bu[d] / f.W;
  F[CTAU] = U[CTAU] * f.vt[d] / G.alpha + pt * f.v[d] - f.ab0 * f.Bu[d] / f.W;
  for (int k = 0; k < 3; ++k) F[BX + k] = (f.Bu[k] * f.vt[d] - f.Bu[d] * f.vt[k]) / G.alpha;
  F[BX + d] = 0.0;
}

// ------------------------------------------------------------------------------------------ C4
// Upper-bound magnetosonic coordinate speeds along d (Gammie et al. 2003 style).
void speeds_at(const double q[NV], const Geo& G, double gam, int d, double& lm, double& lp) {
  const Fluid f = fluid_at(q, G, gam);
  const double cs2 = gam * f.P / f.rhoh;
  const double va2 = f.b2 / (f.rhoh + f.b2);
  const double c2 = cs2 + va2 - cs2 * va2;
  double v2 = 0.0;
  for (int i = 0; i < 3; ++i) v2 += f.v[i] * f.vl[i];
  const double vd = f.v[d];
  double rad = c2 * (1.0 - v2) * (G.gu[d][d] * (1.0 - v2 * c2) - vd * vd * (1.0 - c2));
  if (rad < 0.0) rad = 0.0;
  const double s = std::sqrt(rad);
  lp = G.alpha * (vd * (1.0 - c2) + s) / (1.0 - v2 * c2) - G.bu[d];
  lm = G.alpha * (vd * (1.0 - c2) - s) / (1.0 - v2 * c2) - G.bu[d];
}

// ------------------------------------------------------------------------------------------ C5.1
double minmod2(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  return std::fabs(a) < std::fabs(b) ? a : b;
}
double minmod3(double a, double b, double c) {
  if (a > 0.0 && b > 0.0 && c > 0.0) return std::fmin(a, std::fmin(b, c));
  if (a < 0.0 && b < 0.0 && c < 0.0) return std::fmax(a, std::fmax(b, c));
  return 0.0;
}

// WENO5-Z value at the +1/2 face of the centre cell of the stencil f[0..4] (centre f[2]).
// B12-B15 with the cell-average coefficient set, tau_Z = |beta_2 - beta_0|,
// eps = 1e-40, p = 2.
double weno5z_plus(const double f[5]) {
  const double p0 = (2.0 * f[0] - 7.0 * f[1] + 11.0 * f[2]) / 6.0;
  const double p1 = (-f[1] + 5.0 * f[2] + 2.0 * f[3]) / 6.0;
  const double p2 = (2.0 * f[2] + 5.0 * f[3] - f[4]) / 6.0;
  const double a0 = f[0] - 2.0 * f[1] + f[2], c0 = f[0] - 4.0 * f[1] + 3.0 * f[2];
  const double a1 = f[1] - 2.0 * f[2] + f[3], c1 = f[1] - f[3];
  const double a2 = f[2] - 2.0 * f[3] + f[4], c2 = 3.0 * f[2] - 4.0 * f[3] + f[4];
  const double b0 = 13.0 / 12.0 * a0 * a0 + 0.25 * c0 * c0;
  const double b1 = 13.0 / 12.0 * a1 * a1 + 0.25 * c1 * c1;
  const double b2 = 13.0 / 12.0 * a2 * a2 + 0.25 * c2 * c2;
  const double tau = std::fabs(b2 - b0);
  const double eps = 1e-40;
  const double t0 = tau / (b0 + eps), t1 = tau / (b1 + eps), t2 = tau / (b2 + eps);
  const double w0 = 0.1 * (1.0 + t0 * t0), w1 = 0.6 * (1.0 + t1 * t1), w2 = 0.3 * (1.0 + t2 * t2);
  return (w0 * p0 + w1 * p1 + w2 * p2) / (w0 + w1 + w2);
}

// WENO5-Z-AOAH (B16-B18).  Nonlinear weights of B14 normalised to sum 1 and the fifth-order value
// of B12 with those weights, for the +1/2 face of the centre cell of the stencil f[0..4].
void weno5z_weights(const double f[5], double w[3], double& P5) {
  const double p0 = (2.0 * f[0] - 7.0 * f[1] + 11.0 * f[2]) / 6.0;
  const double p1 = (-f[1] + 5.0 * f[2] + 2.0 * f[3]) / 6.0;
  const double p2 = (2.0 * f[2] + 5.0 * f[3] - f[4]) / 6.0;
  const double a0 = f[0] - 2.0 * f[1] + f[2], c0 = f[0] - 4.0 * f[1] + 3.0 * f[2];
  const double a1 = f[1] - 2.0 * f[2] + f[3], c1 = f[1] - f[3];
  const double a2 = f[2] - 2.0 * f[3] + f[4], c2 = 3.0 * f[2] - 4.0 * f[3] + f[4];
  const double b0 = 13.0 / 12.0 * a0 * a0 + 0.25 * c0 * c0;
  const double b1 = 13.0 / 12.0 * a1 * a1 + 0.25 * c1 * c1;
  const double b2 = 13.0 / 12.0 * a2 * a2 + 0.25 * c2 * c2;
  const double tau = std::fabs(b2 - b0);
  const double eps = 1e-40;
  const double t0 = tau / (b0 + eps), t1 = tau / (b1 + eps), t2 = tau / (b2 + eps);
  const double u0 = 0.1 * (1.0 + t0 * t0), u1 = 0.6 * (1.0 + t1 * t1), u2 = 0.3 * (1.0 + t2 * t2);
  const double sum = u0 + u1 + u2;
  w[0] = u0 / sum; w[1] = u1 / sum; w[2] = u2 / sum;
  P5 = w[0] * p0 + w[1] * p1 + w[2] * p2;
}
// B17: "nonlinearity" of the weights of one face, 1 when w = gamma.
double aoah_sigma_face(const double w[3]) {
  const double g0 = 0.1, g1 = 0.6, g2 = 0.3;
  return 3.0 * w[0] * w[1] * w[2] / (g2 * w[0] * w[1] + g1 * w[0] * w[2] + g0 * w[1] * w[2]);
}
// One cell: sigma of B18 from both faces, clamped to [0,1] (B17 can exceed 1, reading C5.1b), then the mix
// B16 of the WENO5-Z value with the MC-limited piecewise linear value at each face.
void weno5z_aoah_cell(const double f[5], double& qm, double& qp) {
  double r[5];
  for (int m = 0; m < 5; ++m) r[4 - m] = f[m];          // mirror x -> -x
  double wp[3], wm[3], P5p, P5m;
  weno5z_weights(f, wp, P5p);
  weno5z_weights(r, wm, P5m);
  const double sp = aoah_sigma_face(wp), sm = aoah_sigma_face(wm);
  double sigma = 2.0 * sp * sm / (sp + sm);
  if (!(sigma > 0.0)) sigma = 0.0;                        // also catches 0/0 when both faces have a vanishing weight
  if (sigma > 1.0) sigma = 1.0;
  const double dl = f[2] - f[1], dr = f[3] - f[2];
  const double sl = minmod3(2.0 * dl, 0.5 * (f[3] - f[1]), 2.0 * dr);
  const double plm_p = f[2] + 0.5 * sl, plm_m = f[2] - 0.5 * sl;
  qp = sigma * P5p + (1.0 - sigma) * plm_p;
  qm = sigma * P5m + (1.0 - sigma) * plm_m;
}

// MP5 (Suresh & Huynh 1997; named at PAPER.md:275, no parameters given -> alpha = 4, eps = 1e-10 of the original paper).
// Value at the +1/2 face of the centre cell of f[0..4]: the fifth-order linear value, kept if it lies between f_j and
// the monotonicity-preserving bound, else limited to the interval [vmin, vmax] built from the curvature measures d.
double minmod4(double a, double b, double c, double d) {
  if (a > 0.0 && b > 0.0 && c > 0.0 && d > 0.0) return std::fmin(std::fmin(a, b), std::fmin(c, d));
  if (a < 0.0 && b < 0.0 && c < 0.0 && d < 0.0) return std::fmax(std::fmax(a, b), std::fmax(c, d));
  return 0.0;
}
double mp5_plus(const double f[5]) {
  const double alpha = 4.0, eps = 1e-10;
  const double vor = (2.0 * f[0] - 13.0 * f[1] + 47.0 * f[2] + 27.0 * f[3] - 3.0 * f[4]) / 60.0;
  const double vmp = f[2] + minmod2(f[3] - f[2], alpha * (f[2] - f[1]));
  if ((vor - f[2]) * (vor - vmp) <= eps) return vor;
  const double djm1 = f[0] - 2.0 * f[1] + f[2];
  const double dj = f[1] - 2.0 * f[2] + f[3];
  const double djp1 = f[2] - 2.0 * f[3] + f[4];
  const double dm4jph = minmod4(4.0 * dj - djp1, 4.0 * djp1 - dj, dj, djp1);
  const double dm4jmh = minmod4(4.0 * dj - djm1, 4.0 * djm1 - dj, dj, djm1);
  const double vul = f[2] + alpha * (f[2] - f[1]);
  const double vav = 0.5 * (f[2] + f[3]);
  const double vmd = vav - 0.5 * dm4jph;
  const double vlc = f[2] + 0.5 * (f[2] - f[1]) + 4.0 / 3.0 * dm4jmh;
  const double vmin = std::fmax(std::fmin(std::fmin(f[2], f[3]), vmd), std::fmin(std::fmin(f[2], vul), vlc));
  const double vmax = std::fmin(std::fmax(std::fmax(f[2], f[3]), vmd), std::fmax(std::fmax(f[2], vul), vlc));
  return vor + minmod2(vmin - vor, vmax - vor);
}

// Face values of one variable in one cell from its stencil s[-2..2] (s points at the centre).
// qm = value at the lower face (x_{j-1/2}, the "R" state of that face), qp = value at the upper
// face (x_{j+1/2}, the "L" state of that face).
void recon_cell(int recon, const double* s, long stride, double& qm, double& qp) {
  const double q0 = s[0];
  if (recon == 0) { qm = q0; qp = q0; return; }
  if (recon == 1 || recon == 2) {
    const double dl = q0 - s[-stride], dr = s[stride] - q0;
    double sl;
    if (recon == 1) sl = minmod2(dl, dr);
    else sl = minmod3(2.0 * dl, 0.5 * (s[stride] - s[-stride]), 2.0 * dr);
    qp = q0 + 0.5 * sl;
    qm = q0 - 0.5 * sl;
    return;
  }
  double f[5], r[5];
  for (int m = 0; m < 5; ++m) { f[m] = s[(m - 2) * stride]; r[4 - m] = f[m]; }
  if (recon == 4) { weno5z_aoah_cell(f, qm, qp); return; }
  if (recon == 5) { qp = mp5_plus(f); qm = mp5_plus(r); return; }
  qp = weno5z_plus(f);
  qm = weno5z_plus(r);   // mirror x -> -x
}

int stencil_halfwidth(int recon) { return recon == 0 ? 0 : (recon >= 3 ? 2 : 1); }

// ------------------------------------------------------------------------------------------ C5.2
// ns = 1: qL, qR, F carry the passive scalar at index XS.  Eq.14, (X rho u^mu)_{;mu} = 0, in conservation form is
// d_t (sqrt(gamma) D X) + d_i (sqrt(gamma) D X (alpha v^i - beta^i)) = 0, i.e. for one state U~_X = U~_D X and
// F~_X = F~_D X; the two states are combined by the same HLL / LLF formula and speeds as every other variable.
void riemann_face(const orc_params& p, const Geo& G, int d, const double* qL, const double* qR, double* F, int ns = 0) {
  double UL[NVMAX], UR[NVMAX], FL[NVMAX], FR[NVMAX], lmL, lpL, lmR, lpR;
  cons_at(qL, G, p.gamma_ad, UL); cons_at(qR, G, p.gamma_ad, UR);
  flux_at(qL, G, p.gamma_ad, d, FL); flux_at(qR, G, p.gamma_ad, d, FR);
  speeds_at(qL, G, p.gamma_ad, d, lmL, lpL); speeds_at(qR, G, p.gamma_ad, d, lmR, lpR);
  for (int v = 0; v < NV; ++v) {   // densitise: U~ = sqrt(gamma) U, F~ = alpha sqrt(gamma) F (Eq.1)
    UL[v] *= G.sg; UR[v] *= G.sg; FL[v] *= G.alpha * G.sg; FR[v] *= G.alpha * G.sg;
  }
  const int nv = NV + (ns ? 1 : 0);
  if (ns) {
    UL[XS] = UL[CD] * qL[XS]; UR[XS] = UR[CD] * qR[XS];
    FL[XS] = FL[CD] * qL[XS]; FR[XS] = FR[CD] * qR[XS];
  }
  if (p.riemann == 1) {   // HLL
    const double sp = std::fmax(0.0, std::fmax(lpL, lpR));
    const double sm = std::fmin(0.0, std::fmin(lmL, lmR));
    for (int v = 0; v < nv; ++v) F[v] = (sp * FL[v] - sm * FR[v] + sp * sm * (UR[v] - UL[v])) / (sp - sm);
  } else {                // LLF
    const double c = std::fmax(std::fmax(std::fabs(lmL), std::fabs(lpL)), std::fmax(std::fabs(lmR), std::fabs(lpR)));
    for (int v = 0; v < nv; ++v) F[v] = 0.5 * (FL[v] + FR[v]) - 0.5 * c * (UR[v] - UL[v]);
  }
  F[BX + d] = 0.0;
}

// ------------------------------------------------------------------------------------------ C5.4
// alpha sqrt(gamma) S of Eq.4 with G_nu = 0, from primitives at a cell centre.
// momentum: 1/2 T^{mu nu} d_j g_{mu nu};  energy: T^{i0} d_i alpha - alpha T^{mu nu} Gamma^0_{mu nu}.
void inverse4(const Geo& G, double gi[4][4]) {
  const double a2 = G.alpha * G.alpha;
  gi[0][0] = -1.0 / a2;
  for (int i = 0; i < 3; ++i) {
    gi[0][i + 1] = gi[i + 1][0] = G.bu[i] / a2;
    for (int j = 0; j < 3; ++j) gi[i + 1][j + 1] = G.gu[i][j] - G.bu[i] * G.bu[j] / a2;
  }
}

void stress_energy(const double q[NV], const Geo& G, double gam, double T[4][4]) {
  const Fluid f = fluid_at(q, G, gam);
  double u[4], b[4], gi[4][4];
  inverse4(G, gi);
  u[0] = f.W / G.alpha;
  for (int i = 0; i < 3; ++i) u[i + 1] = q[UX + i] - f.W * G.bu[i] / G.alpha;     // Eq.5 solved for u^i
  b[0] = f.ab0 / G.alpha;                                                         // Eq.10
  for (int i = 0; i < 3; ++i) b[i + 1] = (f.Bu[i] + f.ab0 * u[i + 1]) / f.W;      // Eq.11
  for (int m = 0; m < 4; ++m)
    for (int n = 0; n < 4; ++n)
      T[m][n] = (f.rhoh + f.b2) * u[m] * u[n] + (f.P + 0.5 * f.b2) * gi[m][n] - b[m] * b[n];   // Eq.9
}

void source_at(const double q[NV], const double g4[4][4], const double dg[3][4][4], double gam, double S[NV]) {
  const Geo G = split31(g4);
  double T[4][4], gi[4][4];
  stress_energy(q, G, gam, T);
  inverse4(G, gi);
  for (int v = 0; v < NV; ++v) S[v] = 0.0;
  for (int j = 0; j < 3; ++j) {
    double s = 0.0;
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) s += T[m][n] * dg[j][m][n];
    S[CS1 + j] = 0.5 * s;
  }
  // d_i alpha from g^{00} = -1/alpha^2:  d_i alpha = -(alpha^3/2) g^{0 mu} g^{0 nu} d_i g_{mu nu}
  double dalpha[3];
  for (int i = 0; i < 3; ++i) {
    double s = 0.0;
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) s += gi[0][m] * gi[0][n] * dg[i][m][n];
    dalpha[i] = -0.5 * G.alpha * G.alpha * G.alpha * s;
  }
  // Gamma^0_{mu nu} = 1/2 g^{0 lam} (d_mu g_{lam nu} + d_nu g_{lam mu} - d_lam g_{mu nu}), d_0 = 0
  auto D = [&](int der, int m, int n) -> double { return der == 0 ? 0.0 : dg[der - 1][m][n]; };
  double TG = 0.0;
  for (int m = 0; m < 4; ++m)
    for (int n = 0; n < 4; ++n) {
      double gam0 = 0.0;
      for (int l = 0; l < 4; ++l) gam0 += 0.5 * gi[0][l] * (D(m, l, n) + D(n, l, m) - D(l, m, n));
      TG += T[m][n] * gam0;
    }
  double Ta = 0.0;
  for (int i = 0; i < 3; ++i) Ta += T[i + 1][0] * dalpha[i];
  S[CTAU] = Ta - G.alpha * TG;
  for (int v = 0; v < NV; ++v) S[v] *= G.alpha * G.sg;
}

// ------------------------------------------------------------------------------------------ C7, C8
// Kastaun, Kalinani & Ciolfi (2021) master function (cited PAPER.md:277), ideal gas, h0 = 1.
struct C2P {
  double q, r2, b2, rb, rperp2, v02, gam;
  void aux(double mu, double& x, double& rbar2, double& qbar) const {
    x = 1.0 / (1.0 + mu * b2);
    rbar2 = r2 * x * x + mu * x * (1.0 + x) * rb * rb;
    qbar = q - 0.5 * b2 - 0.5 * mu * mu * x * x * b2 * rperp2;
  }
  double fa(double mu) const {
    double x, rbar2, qbar; aux(mu, x, rbar2, qbar);
    return mu * std::sqrt(1.0 + rbar2) - 1.0;
  }
  // returns f(mu); W and unclipped eps through references
  double f(double mu, double& What, double& epsraw) const {
    double x, rbar2, qbar; aux(mu, x, rbar2, qbar);
    const double vhat2 = std::fmin(mu * mu * rbar2, v02);
    What = 1.0 / std::sqrt(1.0 - vhat2);
    epsraw = What * (qbar - mu * rbar2) + vhat2 * What * What / (1.0 + What);
    const double eps = std::fmax(epsraw, 0.0);
    const double ahat = (gam - 1.0) * eps / (1.0 + eps);
    const double nuA = (1.0 + ahat) * (1.0 + eps) / What;
    const double nuB = (1.0 + ahat) * (1.0 + qbar - mu * rbar2);
    return mu - 1.0 / (std::fmax(nuA, nuB) + rbar2 * mu);
  }
};

void note_margin(double& margin, double value, double threshold) {
  const double m = std::fabs(value / threshold - 1.0);
  if (m < margin) margin = m;
}

// U: densitised conserved at one cell (rewritten when floored), q: primitives out.
// rho_flr, eps_flr: the floors at this cell (floors_at).
unsigned char c2p_cell(const orc_params& p, const Geo& G, double rho_flr, double eps_flr, double Ut[NV], double q[NV],
                       double& margin) {
  unsigned char mask = 0;
  double U[NV];
  for (int v = 0; v < NV; ++v) U[v] = Ut[v] / G.sg;
  bool bad = !(U[CD] > 0.0);
  for (int v = 0; v < NV; ++v) if (!std::isfinite(U[v])) bad = true;
  double rho, eps, ut[3];
  const double Bu[3] = {U[BX], U[BX + 1], U[BX + 2]};
  if (bad) {
    mask |= M_BAD_INPUT;
    rho = rho_flr; eps = eps_flr; ut[0] = ut[1] = ut[2] = 0.0;
  } else {
    const double D = U[CD];
    C2P c;
    c.gam = p.gamma_ad;
    c.q = U[CTAU] / D;
    double rl[3], ru[3], bu[3];
    for (int i = 0; i < 3; ++i) { rl[i] = U[CS1 + i] / D; bu[i] = Bu[i] / std::sqrt(D); }
    c.r2 = 0.0; c.b2 = 0.0; c.rb = 0.0;
    for (int i = 0; i < 3; ++i) {
      ru[i] = 0.0;
      for (int j = 0; j < 3; ++j) { ru[i] += G.gu[i][j] * rl[j]; c.b2 += G.gl[i][j] * bu[i] * bu[j]; }
      c.r2 += ru[i] * rl[i];
      c.rb += rl[i] * bu[i];
    }
    c.rperp2 = (c.b2 > 0.0) ? std::fmax(c.r2 - c.rb * c.rb / c.b2, 0.0) : c.r2;
    c.v02 = c.r2 / (1.0 + c.r2);
    // bracket: mu_+ = 1/h0 if r < h0, else the root of f_a in (0, 1/h0]
    double mup = 1.0;
    if (c.r2 >= 1.0) {
      double lo = 0.0, hi = 1.0;
      for (int it = 0; it < 200; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (mid <= lo || mid >= hi) break;
        if (c.fa(mid) > 0.0) hi = mid; else lo = mid;
      }
      mup = hi;
    }
    // root of f in (0, mu_+] by bisection until the bracket stops shrinking
    double lo = 0.0, hi = mup, W, er;
    if (c.f(hi, W, er) <= 0.0) lo = hi;   // root at (or numerically beyond) the upper end
    for (int it = 0; it < 200; ++it) {
      const double mid = 0.5 * (lo + hi);
      if (mid <= lo || mid >= hi) break;
      if (c.f(mid, W, er) > 0.0) hi = mid; else lo = mid;
    }
    const double mu = 0.5 * (lo + hi);
    c.f(mu, W, er);
    double x, rbar2, qbar; c.aux(mu, x, rbar2, qbar);
    rho = D / W;
    eps = er;
    note_margin(margin, eps + eps_flr, eps_flr);   // distance of eps from 0 in units of the floor
    if (eps < 0.0) { mask |= M_EPS_CLIPPED; eps = 0.0; }
    for (int i = 0; i < 3; ++i) ut[i] = W * mu * x * (ru[i] + mu * c.rb * bu[i]);
  }
  // floors
  if (!bad) note_margin(margin, rho, rho_flr);
  if (rho < rho_flr) { rho = rho_flr; mask |= M_RHO_FLOOR; }
  if (!bad && !(mask & M_EPS_CLIPPED)) note_margin(margin, eps, eps_flr);
  if (eps < eps_flr) { eps = eps_flr; mask |= M_EPS_FLOOR; }
  double uu = 0.0;
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) uu += G.gl[i][j] * ut[i] * ut[j];
  const double W = std::sqrt(1.0 + uu);
  if (!bad) note_margin(margin, W, p.w_max);
  if (W > p.w_max) {
    const double s = std::sqrt((p.w_max * p.w_max - 1.0) / (W * W - 1.0));
    for (int i = 0; i < 3; ++i) ut[i] *= s;
    mask |= M_W_CEIL;
  }
  q[RHO] = rho; q[UX] = ut[0]; q[UY] = ut[1]; q[UZ] = ut[2]; q[UU] = rho * eps;
  q[BX] = Bu[0]; q[BY] = Bu[1]; q[BZ] = Bu[2];
  if (mask & (M_RHO_FLOOR | M_EPS_FLOOR | M_W_CEIL | M_BAD_INPUT)) {
    double Un[NV];
    cons_at(q, G, p.gamma_ad, Un);
    for (int v = 0; v <= CTAU; ++v) Ut[v] = G.sg * Un[v];   // B~ untouched
  }
  return mask;
}

// Floor forms of PAPER.md:288: rho_flr = rho0, rho0 exp(-alpha x^1), rho0 (x^1)^-alpha, rho0 r^-alpha, "the specific
// internal energy is set similarly" with its own exponent.  The coordinates here are Cartesian, so the
// "radial coordinate x^1" is read as r (reading C8b): the Kerr-Schild radius for metric 1, the Euclidean
// distance from the origin for the flat metrics; forms 2 and 3 therefore coincide.
void floors_at(const orc_params& p, const double x[3], double& rho_flr, double& eps_flr) {
  rho_flr = p.rho_floor; eps_flr = p.eps_floor;
  if (p.floor_form == 0) return;
  double r;
  if (p.metric == 1) { double H, l[4]; ks_scalars(p, x, r, H, l); }
  else r = std::sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
  if (p.floor_form == 1) {
    rho_flr = p.rho_floor * std::exp(-p.floor_alpha_rho * r);
    eps_flr = p.eps_floor * std::exp(-p.floor_alpha_eps * r);
  } else {
    rho_flr = p.rho_floor * std::pow(r, -p.floor_alpha_rho);
    eps_flr = p.eps_floor * std::pow(r, -p.floor_alpha_eps);
  }
}

// Passive scalar of one cell after con2prim (Eq.14; bounds PAPER.md:290 "we simply require that it stay within the
// bounds").  Dt_in: sqrt(gamma) D the update produced (before any floor), Dt_out: after the floors.
// X = (sqrt(gamma) D X) / (sqrt(gamma) D), clipped to [scalar_min, scalar_max] (bit 128; a non-finite X or a bad cell goes
// to scalar_min); where a floor, the ceiling or the clip acted, the conserved scalar is recomputed as Dt_out * X.
void scalar_recover(const orc_params& p, double Dt_in, double Dt_out, unsigned char& mask, double& UX, double& X,
                    double& margin) {
  if (mask & M_BAD_INPUT) {
    X = p.scalar_min;
    mask |= M_SCALAR_CLIPPED;
  } else {
    X = UX / Dt_in;
    const double range = p.scalar_max - p.scalar_min;
    if (std::isfinite(X)) {
      const double m = std::fmin(std::fabs(X - p.scalar_min), std::fabs(X - p.scalar_max)) / range;
      if (m < margin) margin = m;
    }
    if (!(X >= p.scalar_min)) { X = p.scalar_min; mask |= M_SCALAR_CLIPPED; }
    else if (X > p.scalar_max) { X = p.scalar_max; mask |= M_SCALAR_CLIPPED; }
  }
  if (mask & (M_RHO_FLOOR | M_EPS_FLOOR | M_W_CEIL | M_BAD_INPUT | M_SCALAR_CLIPPED)) UX = Dt_out * X;
}

// ------------------------------------------------------------------------------------------ C9
// Ghost fill through the global array: gather block interiors, fill x then y then z (periodic wrap
// or zero-gradient copy, including already-filled ghosts), scatter every block's ghost frame.
void fill_ghosts(const Grid& G, double* prim) {
  const int* g = G.g;
  const long NA[3] = {G.N[0] + 2 * g[0], G.N[1] + 2 * g[1], G.N[2] + 2 * g[2]};
  const int NVg = G.nv;
  std::vector<double> glob((size_t)NVg * NA[0] * NA[1] * NA[2]);
  auto gid = [&](int v, long k, long j, long i) { return ((v * NA[2] + k) * NA[1] + j) * NA[0] + i; };
  for (int b = 0; b < G.nblk; ++b) {
    int c[3]; G.bcoord(b, c);
    for (int v = 0; v < NVg; ++v)
      for (int k = 0; k < G.n[2]; ++k) for (int j = 0; j < G.n[1]; ++j) for (int i = 0; i < G.n[0]; ++i)
        glob[gid(v, c[2] * G.n[2] + k + g[2], c[1] * G.n[1] + j + g[1], c[0] * G.n[0] + i + g[0])] =
            prim[G.idx(b, v, k + g[2], j + g[1], i + g[0])];
  }
  for (int d = 0; d < 3; ++d) {
    if (g[d] == 0) continue;
    for (int v = 0; v < NVg; ++v)
      for (long k = 0; k < NA[2]; ++k) for (long j = 0; j < NA[1]; ++j) for (long i = 0; i < NA[0]; ++i) {
        long c[3] = {i, j, k};
        // only cells whose later-dimension indices are interior or whose earlier dims are anything
        bool skip = false;
        for (int e = d + 1; e < 3; ++e) if (g[e] && (c[e] < g[e] || c[e] >= g[e] + G.N[e])) skip = true;
        if (skip) continue;
        long s[3] = {i, j, k};
        if (c[d] < g[d]) {
          s[d] = (G.p.bc[d][0] == 0) ? c[d] + G.N[d] : g[d];
        } else if (c[d] >= g[d] + G.N[d]) {
          s[d] = (G.p.bc[d][1] == 0) ? c[d] - G.N[d] : g[d] + G.N[d] - 1;
        } else continue;
        glob[gid(v, c[2], c[1], c[0])] = glob[gid(v, s[2], s[1], s[0])];
      }
  }
  for (int b = 0; b < G.nblk; ++b) {
    int c[3]; G.bcoord(b, c);
    for (int v = 0; v < NVg; ++v)
      for (int k = 0; k < G.na[2]; ++k) for (int j = 0; j < G.na[1]; ++j) for (int i = 0; i < G.na[0]; ++i) {
        const bool interior = k >= g[2] && k < g[2] + G.n[2] && j >= g[1] && j < g[1] + G.n[1] && i >= g[0] && i < g[0] + G.n[0];
        if (interior) continue;
        prim[G.idx(b, v, k, j, i)] = glob[gid(v, c[2] * G.n[2] + k, c[1] * G.n[1] + j, c[0] * G.n[0] + i)];
      }
  }
}

bool excised(const Grid& G, int b, int k, int j, int i) {
  if (G.p.metric != 1 || !(G.p.r_excise > 0.0)) return false;
  const double x[3] = {G.xc(0, b, i), G.xc(1, b, j), G.xc(2, b, k)};
  double r, H, l[4];
  ks_scalars(G.p, x, r, H, l);
  return r < G.p.r_excise;
}

// ------------------------------------------------------------------------------------------ C5
// Face fluxes of one block after flux-CT.  F[d] has the layout of one block's 8-variable field;
// face (i-1/2) along d is stored at cell i.
void block_fluxes(const Grid& G, int b, const double* prim, std::vector<double> F[3]) {
  const orc_params& p = G.p;
  const int* g = G.g; const int* na = G.na; const int* n = G.n;
  const long str[3] = {1, na[0], (long)na[0] * na[1]};
  const long vstr = G.ncell;
  const double* P = prim + G.idx(b, 0, 0, 0, 0);
  auto cid = [&](int k, int j, int i) { return (long)k * str[2] + (long)j * str[1] + i; };
  const bool par = (long)n[1] * n[2] > 1;
  const int nv = G.nv, ns = G.nv - NV;
  for (int d = 0; d < 3; ++d) {
    F[d].assign((size_t)nv * vstr, 0.0);
    if (!G.act[d]) continue;
    // 1. reconstruct every cell that borders a needed face (the passive scalar like any other primitive)
    std::vector<double> qm((size_t)nv * vstr, 0.0), qp((size_t)nv * vstr, 0.0);
    int lo[3], hi[3];   // cell ranges (inclusive)
    for (int e = 0; e < 3; ++e) {
      lo[e] = G.act[e] ? g[e] - 1 : 0;
      hi[e] = G.act[e] ? g[e] + n[e] : 0;
    }
#pragma omp parallel for collapse(2) schedule(static) if (par)
    for (int k = lo[2]; k <= hi[2]; ++k)
      for (int j = lo[1]; j <= hi[1]; ++j)
        for (int i = lo[0]; i <= hi[0]; ++i) {
          const long c = cid(k, j, i);
          double m[NVMAX], pl[NVMAX];
          for (int v = 0; v < nv; ++v) recon_cell(p.recon, P + v * vstr + c, str[d], m[v], pl[v]);
          if (p.recon >= 3) {
            // positivity fallback: piecewise constant in this direction for all variables; the thresholds are the
            // floors at the centre of the cell, lowered by one part in 1e12 (reading C5.1): con2prim holds
            // whole regions exactly AT the floor, where every reconstruction returns the floor up to rounding; a
            // threshold at the floor itself would leave the decision there to the last bit of the arithmetic
            const double xc[3] = {G.xc(0, b, i), G.xc(1, b, j), G.xc(2, b, k)};
            double rfl, efl;
            floors_at(p, xc, rfl, efl);
            const double thr_rho = rfl * (1.0 - 1e-12), thr_u = rfl * efl * (1.0 - 1e-12);
            if (m[RHO] < thr_rho || pl[RHO] < thr_rho || m[UU] < thr_u || pl[UU] < thr_u)
              for (int v = 0; v < nv; ++v) m[v] = pl[v] = P[v * vstr + c];
          }
          for (int v = 0; v < nv; ++v) { qm[v * vstr + c] = m[v]; qp[v * vstr + c] = pl[v]; }
        }
    // 2. Riemann problem at every face (i-1/2) along d, i in [g, g+n]
    int flo[3], fhi[3];
    for (int e = 0; e < 3; ++e) { flo[e] = lo[e]; fhi[e] = hi[e]; }
    flo[d] = g[d]; fhi[d] = g[d] + n[d];
#pragma omp parallel for collapse(2) schedule(static) if (par)
    for (int k = flo[2]; k <= fhi[2]; ++k)
      for (int j = flo[1]; j <= fhi[1]; ++j)
        for (int i = flo[0]; i <= fhi[0]; ++i) {
          const long c = cid(k, j, i);
          double x[3] = {G.xc(0, b, i), G.xc(1, b, j), G.xc(2, b, k)};
          const int il[3] = {i, j, k};
          x[d] = G.xf(d, b, il[d]);
          const Geo geo = geo_at(p, x);
          double qL[NVMAX], qR[NVMAX], Ff[NVMAX];
          for (int v = 0; v < nv; ++v) { qL[v] = qp[v * vstr + c - str[d]]; qR[v] = qm[v * vstr + c]; }
          riemann_face(p, geo, d, qL, qR, Ff, ns);
          for (int v = 0; v < nv; ++v) F[d][v * vstr + c] = Ff[v];
        }
  }
  // 3. flux-CT (Toth 2000, cell-centred field)
  if (!p.use_ct) return;
  auto ex = [&](int k, int j, int i) { return excised(G, b, k, j, i); };
  // pairs of active directions (a, c) with third direction e: E_e at the (a-1/2, c-1/2) edge
  for (int e = 0; e < 3; ++e) {
    const int a = (e + 1) % 3, c = (e + 2) % 3;   // e=2: (x,y) -> E3; e=0: (y,z) -> E1; e=1: (z,x) -> E2
    if (!G.act[a] || !G.act[c]) continue;
    // E_e(a-1/2, c-1/2) = 1/4 [ Fa[Bc](.,.) + Fa[Bc](c-1) - Fc[Ba](.,.) - Fc[Ba](a-1) ]
    std::vector<double> E((size_t)vstr, 0.0);
    int lo[3], hi[3];
    for (int dd = 0; dd < 3; ++dd) { lo[dd] = g[dd]; hi[dd] = g[dd] + n[dd] - 1; }
    hi[a] = g[a] + n[a]; hi[c] = g[c] + n[c];
    const double* FaBc = F[a].data() + (BX + c) * vstr;
    const double* FcBa = F[c].data() + (BX + a) * vstr;
    for (int k = lo[2]; k <= hi[2]; ++k)
      for (int j = lo[1]; j <= hi[1]; ++j)
        for (int i = lo[0]; i <= hi[0]; ++i) {
          const long id = cid(k, j, i);
          double val = 0.25 * (FaBc[id] + FaBc[id - str[c]] - FcBa[id] - FcBa[id - str[a]]);
          // excision: an edge touching a masked cell carries no EMF
          int c0[3] = {i, j, k};
          bool touch = false;
          for (int sa = 0; sa < 2; ++sa) for (int sc = 0; sc < 2; ++sc) {
            int cc[3] = {c0[0], c0[1], c0[2]};
            cc[a] -= sa; cc[c] -= sc;
            if (ex(cc[2], cc[1], cc[0])) touch = true;
          }
          E[id] = touch ? 0.0 : val;
        }
    // Fa[Bc] = 1/2 [E(c) + E(c+1)],  Fc[Ba] = -1/2 [E(a) + E(a+1)]
    double* FaBc_w = F[a].data() + (BX + c) * vstr;
    double* FcBa_w = F[c].data() + (BX + a) * vstr;
    {
      int l2[3], h2[3];
      for (int dd = 0; dd < 3; ++dd) { l2[dd] = g[dd]; h2[dd] = g[dd] + n[dd] - 1; }
      h2[a] = g[a] + n[a];
      for (int k = l2[2]; k <= h2[2]; ++k) for (int j = l2[1]; j <= h2[1]; ++j) for (int i = l2[0]; i <= h2[0]; ++i) {
        const long id = cid(k, j, i);
        FaBc_w[id] = 0.5 * (E[id] + E[id + str[c]]);
      }
      for (int dd = 0; dd < 3; ++dd) { l2[dd] = g[dd]; h2[dd] = g[dd] + n[dd] - 1; }
      h2[c] = g[c] + n[c];
      for (int k = l2[2]; k <= h2[2]; ++k) for (int j = l2[1]; j <= h2[1]; ++j) for (int i = l2[0]; i <= h2[0]; ++i) {
        const long id = cid(k, j, i);
        FcBa_w[id] = -0.5 * (E[id] + E[id + str[a]]);
      }
    }
  }
}

void rk_stage(const Grid& G, double g0, double g1, double bdt, const double* cons0, double* cons, double* prim,
              unsigned char* mask) {
  const orc_params& p = G.p;
  const int* g = G.g; const int* n = G.n; const int* na = G.na;
  const long str[3] = {1, na[0], (long)na[0] * na[1]};
  const long vstr = G.ncell;
  for (int b = 0; b < G.nblk; ++b) {
    std::vector<double> F[3];
    block_fluxes(G, b, prim, F);
    double marg = 1e300;
#pragma omp parallel for collapse(2) schedule(static) reduction(min : marg) if ((long)n[1] * n[2] > 1)
    for (int k = g[2]; k < g[2] + n[2]; ++k)
      for (int j = g[1]; j < g[1] + n[1]; ++j)
        for (int i = g[0]; i < g[0] + n[0]; ++i) {
          const long c = (long)k * str[2] + (long)j * str[1] + i;
          if (excised(G, b, k, j, i)) { mask[G.cidx(b, k, j, i)] = M_EXCISED; continue; }
          const double x[3] = {G.xc(0, b, i), G.xc(1, b, j), G.xc(2, b, k)};
          const int nv = G.nv;
          double R[NVMAX];
          for (int v = 0; v < nv; ++v) R[v] = 0.0;
          for (int d = 0; d < 3; ++d) {
            if (!G.act[d]) continue;
            for (int v = 0; v < nv; ++v) R[v] -= (F[d][v * vstr + c + str[d]] - F[d][v * vstr + c]) / G.dx[d];
          }
          if (p.metric != 0) {
            double g4[4][4], dg[3][4][4], q[NV], S[NV];
            metric4(p, x, g4);
            metric4_derivs(p, x, dg);
            for (int v = 0; v < NV; ++v) q[v] = prim[G.idx(b, v, k, j, i)];
            source_at(q, g4, dg, p.gamma_ad, S);
            for (int v = 0; v < NV; ++v) R[v] += S[v];
          }
          double U[NVMAX], q[NVMAX];
          for (int v = 0; v < nv; ++v) {   // the scalar has no source (S = 0 in Eq.14: no neutrino exchange on this path)
            const long id = G.idx(b, v, k, j, i);
            U[v] = g0 * cons0[id] + g1 * cons[id] + bdt * R[v];
          }
          const Geo geo = geo_at(p, x);
          double rfl, efl;
          floors_at(p, x, rfl, efl);
          const double Dt_in = U[CD];
          unsigned char m = c2p_cell(p, geo, rfl, efl, U, q, marg);   // 6. con2prim + floors
          if (nv > NV) scalar_recover(p, Dt_in, U[CD], m, U[XS], q[XS], marg);
          // this block's fluxes are complete and every block reads ghosts from its own storage,
          // so the interior primitives may be overwritten now
          for (int v = 0; v < nv; ++v) { cons[G.idx(b, v, k, j, i)] = U[v]; prim[G.idx(b, v, k, j, i)] = q[v]; }
          mask[G.cidx(b, k, j, i)] = m;
        }
    if (marg < g_last_margin) g_last_margin = marg;
  }
  fill_ghosts(G, prim);   // 7.
}

}  // namespace

// ============================================================================================
extern "C" {

size_t orc_field_elems(const orc_params* p) { Grid G(*p); return (size_t)G.nblk * G.nv * G.ncell; }
double orc_last_c2p_margin(void) { return g_last_margin; }
void orc_reset_c2p_margin(void) { g_last_margin = 1e300; }

// C10: densitised conserved variables from primitives, every allocated cell.
int orc_prim_to_cons(const orc_params* p, const double* prim, double* cons) {
  Grid G(*p);
  for (int b = 0; b < G.nblk; ++b)
#pragma omp parallel for collapse(2) schedule(static) if ((long)G.n[1] * G.n[2] > 1)
    for (int k = 0; k < G.na[2]; ++k) for (int j = 0; j < G.na[1]; ++j) for (int i = 0; i < G.na[0]; ++i) {
      const double x[3] = {G.xc(0, b, i), G.xc(1, b, j), G.xc(2, b, k)};
      const Geo geo = geo_at(*p, x);
      double q[NV], U[NV];
      for (int v = 0; v < NV; ++v) q[v] = prim[G.idx(b, v, k, j, i)];
      cons_at(q, geo, p->gamma_ad, U);
      for (int v = 0; v < NV; ++v) cons[G.idx(b, v, k, j, i)] = geo.sg * U[v];
      if (G.nv > NV) cons[G.idx(b, XS, k, j, i)] = geo.sg * U[CD] * prim[G.idx(b, XS, k, j, i)];   // sqrt(gamma) D X (Eq.14)
    }
  return 0;
}

// C7+C8 on interior cells; ghosts of prim are then filled (C9).
int orc_cons_to_prim(const orc_params* p, double* cons, double* prim, unsigned char* mask) {
  Grid G(*p);
  double marg = 1e300;
  for (int b = 0; b < G.nblk; ++b)
#pragma omp parallel for collapse(2) schedule(static) reduction(min : marg) if ((long)G.n[1] * G.n[2] > 1)
    for (int k = G.g[2]; k < G.g[2] + G.n[2]; ++k)
      for (int j = G.g[1]; j < G.g[1] + G.n[1]; ++j)
        for (int i = G.g[0]; i < G.g[0] + G.n[0]; ++i) {
          if (excised(G, b, k, j, i)) { mask[G.cidx(b, k, j, i)] = M_EXCISED; continue; }
          const double x[3] = {G.xc(0, b, i), G.xc(1, b, j), G.xc(2, b, k)};
          const Geo geo = geo_at(*p, x);
          double U[NVMAX], q[NVMAX];
          for (int v = 0; v < G.nv; ++v) U[v] = cons[G.idx(b, v, k, j, i)];
          double rfl, efl;
          floors_at(*p, x, rfl, efl);
          const double Dt_in = U[CD];
          unsigned char m = c2p_cell(*p, geo, rfl, efl, U, q, marg);
          if (G.nv > NV) scalar_recover(*p, Dt_in, U[CD], m, U[XS], q[XS], marg);
          mask[G.cidx(b, k, j, i)] = m;
          for (int v = 0; v < G.nv; ++v) { cons[G.idx(b, v, k, j, i)] = U[v]; prim[G.idx(b, v, k, j, i)] = q[v]; }
        }
  if (marg < g_last_margin) g_last_margin = marg;
  fill_ghosts(G, prim);
  return 0;
}

int orc_fill_ghosts(const orc_params* p, double* prim) { Grid G(*p); fill_ghosts(G, prim); return 0; }

int orc_rk_stage(const orc_params* p, double g0, double g1, double beta_dt, const double* cons0, double* cons,
                 double* prim, unsigned char* mask) {
  Grid G(*p);
  rk_stage(G, g0, g1, beta_dt, cons0, cons, prim, mask);
  return 0;
}

// C6: dt = cfl * min over interior cells of 1 / sum_d max(|lam+|,|lam-|)/dx_d
int orc_cfl_dt(const orc_params* p, const double* prim, double cfl, double* dt) {
  Grid G(*p);
  double best = std::numeric_limits<double>::infinity();
  for (int b = 0; b < G.nblk; ++b)
#pragma omp parallel for collapse(2) schedule(static) reduction(min : best) if ((long)G.n[1] * G.n[2] > 1)
    for (int k = G.g[2]; k < G.g[2] + G.n[2]; ++k)
      for (int j = G.g[1]; j < G.g[1] + G.n[1]; ++j)
        for (int i = G.g[0]; i < G.g[0] + G.n[0]; ++i) {
          if (excised(G, b, k, j, i)) continue;
          const double x[3] = {G.xc(0, b, i), G.xc(1, b, j), G.xc(2, b, k)};
          const Geo geo = geo_at(*p, x);
          double q[NV];
          for (int v = 0; v < NV; ++v) q[v] = prim[G.idx(b, v, k, j, i)];
          double s = 0.0;
          for (int d = 0; d < 3; ++d) {
            if (!G.act[d]) continue;
            double lm, lp;
            speeds_at(q, geo, p->gamma_ad, d, lm, lp);
            s += std::fmax(std::fabs(lm), std::fabs(lp)) / G.dx[d];
          }
          const double t = 1.0 / s;
          if (t < best) best = t;
        }
  *dt = cfl * best;
  return 0;
}

// Face fluxes after CT of every block (debug / pin hook): F1,F2,F3 each of orc_field_elems.
int orc_stage_fluxes(const orc_params* p, const double* prim, double* F1, double* F2, double* F3) {
  Grid G(*p);
  double* out[3] = {F1, F2, F3};
  for (int b = 0; b < G.nblk; ++b) {
    std::vector<double> F[3];
    block_fluxes(G, b, prim, F);
    for (int d = 0; d < 3; ++d) std::memcpy(out[d] + G.idx(b, 0, 0, 0, 0), F[d].data(), sizeof(double) * G.nv * G.ncell);
  }
  return 0;
}

// ---- point-wise hooks used by the pins -----------------------------------------------------
void orc_metric(const orc_params* p, const double* x, double* g16) {
  double g[4][4]; metric4(*p, x, g); std::memcpy(g16, g, sizeof g);
}
void orc_metric_derivs(const orc_params* p, const double* x, double* dg48) {
  double dg[3][4][4]; metric4_derivs(*p, x, dg); std::memcpy(dg48, dg, sizeof dg);
}
// out: alpha, beta^i(3), beta_i(3), gamma_ij(9), gamma^ij(9), sqrt(gamma)  = 26 doubles
void orc_split31(const double* g16, double* out) {
  double g[4][4]; std::memcpy(g, g16, sizeof g);
  const Geo G = split31(g);
  out[0] = G.alpha;
  for (int i = 0; i < 3; ++i) { out[1 + i] = G.bu[i]; out[4 + i] = G.bl[i]; }
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { out[7 + 3 * i + j] = G.gl[i][j]; out[16 + 3 * i + j] = G.gu[i][j]; }
  out[25] = G.sg;
}
void orc_point_cons(const double* g16, double gam, const double* q, double* U) {
  double g[4][4]; std::memcpy(g, g16, sizeof g);
  cons_at(q, split31(g), gam, U);
}
void orc_point_flux(const double* g16, double gam, const double* q, int d, double* F) {
  double g[4][4]; std::memcpy(g, g16, sizeof g);
  flux_at(q, split31(g), gam, d, F);
}
void orc_point_speeds(const double* g16, double gam, const double* q, int d, double* lm, double* lp) {
  double g[4][4]; std::memcpy(g, g16, sizeof g);
  speeds_at(q, split31(g), gam, d, *lm, *lp);
}
void orc_point_source(const double* g16, const double* dg48, double gam, const double* q, double* S) {
  double g[4][4], dg[3][4][4]; std::memcpy(g, g16, sizeof g); std::memcpy(dg, dg48, sizeof dg);
  source_at(q, g, dg, gam, S);
}
void orc_point_stress_energy(const double* g16, double gam, const double* q, double* T16) {
  double g[4][4], T[4][4]; std::memcpy(g, g16, sizeof g);
  stress_energy(q, split31(g), gam, T); std::memcpy(T16, T, sizeof T);
}
// U: densitised conserved (in/out), q: primitives out; returns the mask
int orc_point_c2p(const orc_params* p, const double* g16, double* U, double* q) {
  double g[4][4]; std::memcpy(g, g16, sizeof g);
  double marg = 1e300;
  const int m = c2p_cell(*p, split31(g), p->rho_floor, p->eps_floor, U, q, marg);   // constant-form floors
  if (marg < g_last_margin) g_last_margin = marg;
  return m;
}
void orc_point_riemann(const orc_params* p, const double* g16, int d, const double* qL, const double* qR, double* F) {
  double g[4][4]; std::memcpy(g, g16, sizeof g);
  riemann_face(*p, split31(g), d, qL, qR, F);
}
// floors at a point (PAPER.md:288 forms)
void orc_point_floors(const orc_params* p, const double* x, double* rho_flr, double* eps_flr) { floors_at(*p, x, *rho_flr, *eps_flr); }
// Riemann flux of the 8 variables plus the passive scalar (qL, qR, F: 9 entries)
void orc_point_riemann_scalar(const orc_params* p, const double* g16, int d, const double* qL, const double* qR, double* F) {
  double g[4][4]; std::memcpy(g, g16, sizeof g);
  riemann_face(*p, split31(g), d, qL, qR, F, 1);
}
// reconstruct a line f[0..n-1]: qm[i], qp[i] for cells with a full stencil (others untouched)
void orc_recon_line(int recon, int n, const double* f, double* qm, double* qp) {
  const int hw = stencil_halfwidth(recon);
  for (int i = hw; i < n - hw; ++i) recon_cell(recon, f + i, 1, qm[i], qp[i]);
}

}  // extern "C"
