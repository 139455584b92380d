/* phx.h — C ABI of the B200-native ideal-GRMHD finite-volume hot path (after PHOEBUS, arXiv:2410.09146).
 *
 * Every entry point runs hand-written sm_100a CUDA kernels; there is no CPU fallback.  All `d_*`
 * pointers are DEVICE pointers owned by the caller (16-byte aligned), all `h_*` pointers are HOST
 * pointers.  `stream` is a cudaStream_t passed as void* (NULL = default stream); every call is
 * asynchronous on it unless stated otherwise.  Every function returns PHX_OK or an error code and
 * never throws or aborts; phx_last_error() returns a thread-local message for the last failure.
 * Numerical trouble is never an error code: it is reported per cell in the mask.
 *
 * Field layout (all fp64): [block][var][k][j][i], i fastest, 8 + nscalar variables, ghosts included.
 *   primitives  P  = (rho, W v^1, W v^2, W v^3, rho*eps, B^1, B^2, B^3 [, X])      PAPER.md:111-113 (Eq.13)
 *   conserved   U~ = sqrt(gamma) * (D, S_1, S_2, S_3, tau, B^1, B^2, B^3 [, D X])   PAPER.md:59-63 (Eq.1-2)
 * X is the passive scalar of Eq.14 (the paper's use is the electron fraction), present as
 * variable 8 of every field when params.nscalar = 1: (X rho u^mu)_{;mu} = 0, i.e. sqrt(gamma) D X is advected with
 * the mass flux, F~_X = F~_D X per state, combined by the same LLF / HLL formula as every other variable.
 * Block id = (bz*nby + by)*nbx + bx.  A dimension with one zone in the whole domain is inactive:
 * it has no ghost zones and no sweep.  Ghosts of U~ are never read or written.
 * Mask layout: [block][k][j][i] (uint8, same cell indexing as one variable).
 */
#ifndef PHX_H
#define PHX_H
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct phx_mesh phx_mesh; /* opaque; owns flux scratch, excision flags and reduction scratch on the device */

enum { PHX_OK = 0, PHX_EINVAL = 1, PHX_ECUDA = 2, PHX_ENOMEM = 3, PHX_EUNSUPPORTED = 4 };
enum { PHX_MINKOWSKI = 0, PHX_KERR_SCHILD = 1,   /* Cartesian Kerr-Schild, ingoing (analytic metrics) */
       PHX_MINKOWSKI_BOOSTED = 2 };              /* flat metric in coordinates x' = x - shift*t: alpha = 1, beta^i = shift^i,
                                                    gamma_ij = delta_ij ("flat metric with coordinate boosts") */
enum { PHX_RECON_CONST = 0, PHX_RECON_PLM_MINMOD = 1, PHX_RECON_PLM_MC = 2, PHX_RECON_WENO5Z = 3,    /* PAPER.md:275, App.B B12-B15 */
       PHX_RECON_WENO5Z_AOAH = 4,    /* the paper's WENO5-Z mixed with PLM-MC by the weight sigma, App.B B16-B18 */
       PHX_RECON_MP5 = 5 };          /* Suresh & Huynh (1997) monotonicity-preserving fifth order, alpha = 4 */
enum { PHX_RIEMANN_LLF = 0, PHX_RIEMANN_HLL = 1 };
enum { PHX_BC_PERIODIC = 0, PHX_BC_OUTFLOW = 1 };
/* con2prim / floor mask bits */
enum {
  PHX_M_RHO_FLOOR = 1, PHX_M_EPS_FLOOR = 2, PHX_M_EPS_CLIPPED = 4, PHX_M_W_CEIL = 8,
  PHX_M_NOCONV = 16, PHX_M_BAD_INPUT = 32, PHX_M_EXCISED = 64,
  PHX_M_SCALAR_CLIPPED = 128   /* the passive scalar left [scalar_min, scalar_max] and was put back */
};
/* floor forms of PAPER.md:288: rho_flr = rho0 | rho0 exp(-alpha x^1) | rho0 (x^1)^-alpha | rho0 r^-alpha, and "the specific
 * internal energy is set similarly".  The coordinates of this library are Cartesian, so the radial coordinate
 * x^1 is read as r: the Kerr-Schild radius for PHX_KERR_SCHILD, the Euclidean distance from the origin for the flat
 * metrics (forms 2 and 3 coincide).  rho0 = rho_floor, eps0 = eps_floor. */
enum { PHX_FLOOR_CONST = 0, PHX_FLOOR_EXP_X1 = 1, PHX_FLOOR_POW_X1 = 2, PHX_FLOOR_POW_R = 3 };

typedef struct {
  int metric;
  double bh_mass, bh_spin, r_excise; /* Kerr-Schild only; r_excise <= 0: no excision */
  int nbx, nby, nbz;                 /* block grid */
  int nx, ny, nz;                    /* interior zones per block */
  int ng;                            /* ghosts per side in active dimensions: >=2 for PLM, >=3 for WENO5-Z(-AOAH) and MP5 */
  double xmin[3], xmax[3];           /* global domain, uniform spacing */
  int bc[3][2];                      /* [dimension][lower, upper] */
  double gamma_ad;                   /* ideal gas P = (Gamma-1) rho eps */
  int recon, riemann, use_ct;
  double rho_floor, eps_floor, w_max; /* constant-form floors (first case) */
  double c2p_tol;                     /* relative tolerance on the con2prim root mu */
  int c2p_maxit;
  double shift[3];                    /* PHX_MINKOWSKI_BOOSTED only: the constant shift vector, |shift| < 1 */
  int nscalar;                        /* 0 or 1 passive scalar (Eq.14) carried as variable 8 of every field */
  double scalar_min, scalar_max;      /* after recovery X = U~_X / U~_D is clipped to these bounds (mask bit 128); where a
                                         floor, the ceiling or the clip acted U~_X is rewritten as U~_D X */
  int floor_form;                     /* PHX_FLOOR_*; 0 keeps rho_floor and eps_floor constant */
  double floor_alpha_rho, floor_alpha_eps; /* exponents alpha of the density and specific-energy floors (paper: 2.0) */
} phx_params;

/* Build a mesh object: validates the parameters, allocates flux scratch (3 x one field) and the divergence accumulator
 * (5 + nscalar variables of one field: the sweeps add -(F_{+1/2} - F_{-1/2})/dx of D, S_j, tau and the scalar to it),
 * the excision flag array and reduction scratch, and runs the geometry-flag kernel on `stream`.
 * Errors: PHX_EINVAL (bad sizes, ng too small for recon, inactive dimension split over blocks),
 * PHX_ENOMEM, PHX_ECUDA.  The mesh is freed with phx_free_mesh. */
int phx_init_mesh(const phx_params* params, void* stream, phx_mesh** out);
int phx_free_mesh(phx_mesh* mesh);

/* Number of doubles in one field: nblocks*(8+nscalar)*(nz+2gz)*(ny+2gy)*(nx+2gx). */
size_t phx_field_elems(const phx_mesh* mesh);
/* Number of bytes in one mask: nblocks*(nz+2gz)*(ny+2gy)*(nx+2gx). */
size_t phx_mask_elems(const phx_mesh* mesh);

/* U~ = sqrt(gamma) U(P) (Eq.2) at every allocated cell (ghosts included). */
int phx_prim_to_cons(const phx_mesh* mesh, const double* d_prim, double* d_cons, void* stream);

/* Primitive recovery after Kastaun et al. 2021 plus floors on every
 * interior cell, then ghost fill of d_prim.  d_cons is rewritten only where a floor or ceiling acted
 * (D, S_j, tau recomputed from the floored primitives; B~ untouched).  d_mask receives the per-cell bits. */
int phx_cons_to_prim(const phx_mesh* mesh, double* d_cons, double* d_prim, unsigned char* d_mask, void* stream);

/* Ghost zones of a primitive field: periodic wrap / zero-gradient outflow at domain faces, copies from the
 * owning neighbour block elsewhere (faces, edges and corners). */
int phx_fill_ghosts(const phx_mesh* mesh, double* d_prim, void* stream);

/* One Runge-Kutta stage of Eq.1:  U~ <- g0*U~0 + g1*U~ + beta_dt * [ -div F~ + alpha sqrt(gamma) S ],
 * with F~ from reconstruction + LLF/HLL + flux-CT, then con2prim, floors and
 * ghost fill.  RK2 (Heun): (1, 0, dt) then (1/2, 1/2, dt/2).
 *   in : d_prim = primitives of d_cons with ghosts filled;  d_cons0 = U~ at the start of the step
 *   out: d_cons updated (interior), d_prim = new primitives with ghosts filled, d_mask = this stage's mask.
 * d_cons0 may alias d_cons (stage 1). */
int phx_rk_stage(phx_mesh* mesh, double g0, double g1, double beta_dt, const double* d_cons0, double* d_cons,
                 double* d_prim, unsigned char* d_mask, void* stream);

/* dt = cfl * min over interior, non-excised cells of 1 / sum_d max(|lambda+^d|, |lambda-^d|)/dx_d.
 * d_dt (device, required) receives the result; if h_dt is non-NULL the value is also copied to the host
 * and the stream is synchronised.  A cell whose speeds are not finite (NaN primitives) makes the result NaN rather than
 * being skipped; a mesh without any evolving cell gives +inf.  The fused reductions of phx_rk2_step_cfl behave the same. */
int phx_cfl_dt(const phx_mesh* mesh, const double* d_prim, double cfl, double* d_dt, double* h_dt, void* stream);

/* One full RK2 step with the time step read from the device scalar d_dt (no host round trip); the result equals two
 * phx_rk_stage calls bit for bit.  d_cons0 is scratch (same size as d_cons, must not alias it): stage 1 writes its
 * state U~1 there, stage 2 combines U~0 = d_cons and U~1 into d_cons; on return d_cons0 holds U~1.  Between the two stages only
 * the ghost layers stage 2 reads are filled (stencil half-width + 1 in y and z); on return the whole ghost frame of d_prim is. */
int phx_rk2_step(phx_mesh* mesh, const double* d_dt, double* d_cons0, double* d_cons, double* d_prim,
                 unsigned char* d_mask, void* stream);

/* phx_rk2_step followed by phx_cfl_dt on the new primitives, with the reduction fused into the second stage's update
 * kernel: on entry *d_dt (device) is the time step of this step, on return it is cfl * min 1/sum_d max|lambda^d|/dx_d of the
 * state the step produced -- the same bits phx_cfl_dt would write.  Start a run with one phx_cfl_dt call. */
int phx_rk2_step_cfl(phx_mesh* mesh, double cfl, double* d_dt, double* d_cons0, double* d_cons, double* d_prim,
                     unsigned char* d_mask, void* stream);

/* `nsteps` RK2 steps with the time step kept on the device: the same bits as `nsteps` calls of phx_rk2_step_cfl (*d_dt on
 * entry = the time step of the first step, e.g. from phx_cfl_dt; on return = the CFL time step of the final state).
 * d_t (DEVICE, nullable): the dt of every step is added to it before the step is taken (elapsed coordinate time).
 * For nsteps >= 2 and no per-kernel timing active, the launches of one step are captured once into a CUDA graph (cached in
 * the mesh for this set of arguments) and replayed on a mesh-owned stream fenced by events against `stream`, which removes
 * the launch gaps that dominate small meshes (64^3: 11 launches of 10-25 microseconds per step).  A small one-dimensional
 * mesh (one block, x the only active direction, nx <= 510, flat metric without shift, no passive scalar, constant floors, no
 * excision) instead runs all `nsteps` steps inside ONE launch of one thread block that owns the mesh (k_evolve_1d: shared-
 * memory exchange between the phases of a stage, the time step reduced block-wide): 256 zones take 0.010 ms per step
 * instead of 0.022 from the graph; the bits are those of the general path.  Asynchronous. */
int phx_evolve_device(phx_mesh* mesh, int nsteps, double cfl, double* d_dt, double* d_t, double* d_cons0, double* d_cons,
                      double* d_prim, unsigned char* d_mask, void* stream);

/* HOST-buffer path (the end-to-end call): copies h_prim_in (HOST, phx_field_elems doubles, ghosts filled) to
 * mesh-owned device fields, computes U~ (phx_prim_to_cons), then runs phx_cfl_dt once and phx_evolve_device for `nsteps` steps
 * (the time step kept on the device), and copies the primitives (required), the conserved variables and the
 * last stage's mask (both nullable) back to HOST buffers.  *h_t (nullable) receives the elapsed coordinate time.
 * Synchronises `stream` before returning.  The device workspace (3 fields + mask) is allocated on first use and
 * freed with the mesh.  Pinned host buffers make the copies asynchronous-capable but are not required. */
int phx_evolve_host(phx_mesh* mesh, const double* h_prim_in, int nsteps, double cfl, double* h_prim_out,
                    double* h_cons_out, unsigned char* h_mask_out, double* h_t, void* stream);

/* The sweeps store only what the update needs from other cells: the magnetic components of F~^d (flux-CT); the divergence
 * of D, S_j, tau (and the passive scalar) is accumulated on the fly.  phx_debug_enable_flux(mesh, 1) makes every later
 * stage store all components of F~^d as well, for phx_debug_flux. */
int phx_debug_enable_flux(phx_mesh* mesh, int on);

/* Raw Riemann face fluxes F~^d (before flux-CT) of the last stage (after phx_debug_enable_flux(mesh, 1)), for debugging and
 * tests: copies the mesh-owned scratch of direction d (0,1,2) into d_out (DEVICE, phx_field_elems doubles, layout of one field,
 * the face (i-1/2) stored at cell i), asynchronously on `stream`.  PHX_EINVAL for an inactive direction. */
int phx_debug_flux(const phx_mesh* mesh, int d, double* d_out, void* stream);

/* Failure detection ("guaranteed to always converge", 279-290 floors): the number of INTERIOR cells whose mask
 * (as written by phx_cons_to_prim / phx_rk_stage / phx_rk2_step*) carries any of `bits` (PHX_M_*; e.g. PHX_M_NOCONV |
 * PHX_M_BAD_INPUT for con2prim failures, PHX_M_RHO_FLOOR | PHX_M_EPS_FLOOR for the floors).  d_count (DEVICE, required) receives
 * the count; h_count (HOST, nullable) also, with a stream synchronisation.  Excised cells carry PHX_M_EXCISED only. */
int phx_count_masked(const phx_mesh* mesh, const unsigned char* d_mask, unsigned bits, unsigned long long* d_count,
                     unsigned long long* h_count, void* stream);

/* Count of this library's kernel launches since the mesh was created (for bench.py's gpu_launches). */
unsigned long long phx_launch_count(const phx_mesh* mesh);

/* Per-kernel-class timing with CUDA events recorded on the launching stream around every launch (bench.py's
 * roofline figures).  phx_profile_enable(mesh, n) allocates n event pairs (n = 0 switches timing off); launches beyond
 * n are not recorded.  phx_profile_read synchronises the recorded events, writes the summed milliseconds and the
 * number of records per class into HOST arrays of PHX_K_COUNT entries, and resets the record list.
 * PHX_K_CFL covers both reduction kernels of one phx_cfl_dt call; PHX_K_COPY is unused (phx_rk2_step makes no copy). */
enum { PHX_K_SWEEP_X = 0, PHX_K_SWEEP_Y = 1, PHX_K_SWEEP_Z = 2, PHX_K_UPDATE = 3, PHX_K_FILL_GHOSTS = 4, PHX_K_CFL = 5,
       PHX_K_PRIM_TO_CONS = 6, PHX_K_C2P = 7, PHX_K_COPY = 8, PHX_K_COUNT = 9 };
int phx_profile_enable(phx_mesh* mesh, int max_records);
int phx_profile_read(phx_mesh* mesh, double* h_ms, unsigned long long* h_count);

/* Peak of the fp64 pipe, measured: a loop of independent fused multiply-adds (8 chains per thread, 64 warps per SM) on every
 * SM for at least `min_seconds` (0 < min_seconds <= 10) after a calibration launch, timed with CUDA events on `stream`.
 * *h_dfma_per_s (HOST, required) receives DFMA thread-instructions per second (x 2 = flop/s) of that sustained launch;
 * *h_dfma_per_s_burst (HOST, nullable) the rate of the short calibration launch before it (min_seconds / 20: the burst figure,
 * before a power cap acts); *h_ms (HOST, nullable) the duration of the timed launch; *h_nsm (HOST, nullable) the SM count of
 * the current device.  Synchronises `stream`.
 * The denominator of bench.py's ALU roofline (R64 is to be measured, not assumed). */
int phx_debug_fp64_peak(double min_seconds, double* h_dfma_per_s, double* h_dfma_per_s_burst, double* h_ms, int* h_nsm, void* stream);

const char* phx_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
