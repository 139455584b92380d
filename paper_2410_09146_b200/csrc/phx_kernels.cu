// phx_kernels.cu — sm_100a kernels and the C ABI of include/phx.h.
//
// Kernels per Runge-Kutta stage (all launched on the caller's stream, no host synchronisation):
//   k_sweep_x      fused reconstruct + Riemann flux along x: one thread per cell, upper-face states and face fluxes exchanged
//                  through shared memory, flat tiling over (row, i) so that warps stay full for any row length
//   k_sweep_march  fused reconstruct + Riemann flux along y or z: lanes along x (coalesced), each thread marches along the
//                  sweep direction; the 2*HW+1 stencil rows of its column sit in a shared-memory ring that cp.async fills
//                  one row ahead, so every primitive is read from HBM once
//                  (all three sweeps store the magnetic flux components and accumulate the divergence of the others)
//   k_update       flux-CT + accumulated divergence + geometric sources + RK combine + con2prim + floors, one thread per cell
//   k_fill_ghosts  periodic / outflow / block-to-block ghost copies in one gather pass over the ghost cells
// and k_cfl_partial / k_cfl_final (warp-shuffle min reduction), k_cfl_final_slots (fused into stage 2), k_prim_to_cons,
// k_c2p, k_excision_flags, k_count_masked (failure detection), k_fp64_peak (the measured denominator of the ALU roofline);
// phx_evolve_device replays one captured
// step as a CUDA graph, or runs a small 1-D mesh entirely inside one thread block (k_evolve_1d).
#include "phx_device.cuh"
#include "../../include/phx.h"

#include <new>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

using namespace phx;

// ================================================================================================ kernels
// launch shapes (tuned on B200 with ncu, profiles/): threads per block and minimum resident blocks per SM; the x sweep is
// bound to 6 blocks/SM for WENO5-Z-AOAH, to 5 for PLM (96 registers, no spills: 0.90 -> 0.83 ms on 512 Kerr-Schild blocks
// of 32^3) and to 4 for WENO5-Z / MP5 (121 registers; more blocks per SM measured slower there)
#ifndef PHX_XS_BLOCK
#define PHX_XS_BLOCK 128
#endif
#ifndef PHX_XS_MINB
#define PHX_XS_MINB 4
#endif
#ifndef PHX_MS_BLOCK
#define PHX_MS_BLOCK 64
#endif
#ifndef PHX_MS_MINB
#define PHX_MS_MINB 6
#endif
#ifndef PHX_UP_BLOCK
#define PHX_UP_BLOCK 128
#endif
#ifndef PHX_UP_MINB
#define PHX_UP_MINB 7      // Minkowski update: HBM-bound, wants resident warps (80 registers); Kerr-Schild keeps its registers
#endif
#ifndef PHX_UP_MINB_KS
#define PHX_UP_MINB_KS 4
#endif
constexpr int XS_BLOCK = PHX_XS_BLOCK;   // threads per block of the x sweep (XS_BLOCK-1 faces per block)
constexpr int MS_BLOCK = PHX_MS_BLOCK;   // threads per block of the marching sweeps
constexpr int UP_BLOCK = PHX_UP_BLOCK;
#ifndef PHX_UP_STAGE_KS
#define PHX_UP_STAGE_KS 1  // Kerr-Schild update: U~0, U~_in and the stage-input primitives go through cp.async (2.42 -> 2.38 ms on
#endif                     // 512 blocks of 32^3); the flat-metric update loses L1 capacity to it (1.51 -> 1.61 ms at 256^3): off there


// (x, y, z): centre of the cell, used only when the floors depend on the position (floor_form != 0)
template <int METRIC, int RECON, int NS>
__device__ __forceinline__ void positivity_fallback(const MeshDev& m, double x, double y, double z, const double* centre, double* qm,
                                                    double* qp) {
  if constexpr (RECON >= 3) {
    double rfl, efl;
    floors_at<METRIC>(m, x, y, z, rfl, efl);
    // thresholds one part in 1e12 below the floors: regions that con2prim holds exactly at the floor reconstruct to the
    // floor up to rounding and must not sit on the threshold (reading C5.1)
    const double trho = rfl * (1.0 - 1e-12), tu = rfl * efl * (1.0 - 1e-12);
    if (qm[RHO] < trho || qp[RHO] < trho || qm[UU] < tu || qp[UU] < tu) {
#pragma unroll
      for (int v = 0; v < NV + NS; ++v) { qm[v] = centre[v]; qp[v] = centre[v]; }
    }
  }
}

// NS = 1: qL, qR, F carry the passive scalar at index XS; per state U~_X = U~_D X and F~_X = F~_D X (Eq.14)
template <int METRIC, int D, int NS>
__device__ __forceinline__ void face_flux(const MeshDev& m, const Geo<METRIC>& G, const double* qL, const double* qR, double* F) {
  double UL[NV + NS], UR[NV + NS], FL[NV + NS], FR[NV + NS], lmL, lpL, lmR, lpR;
  state_flux<METRIC, D>(qL, G, m.gam, UL, FL, lmL, lpL);
  state_flux<METRIC, D>(qR, G, m.gam, UR, FR, lmR, lpR);
  if constexpr (NS == 1) {
    UL[XS] = UL[CD] * qL[XS]; UR[XS] = UR[CD] * qR[XS];
    FL[XS] = FL[CD] * qL[XS]; FR[XS] = FR[CD] * qR[XS];
  }
  riemann_combine<NS>(m.riemann, UL, UR, FL, FR, lmL, lpL, lmR, lpR, F);
  F[BX + D] = 0.0;
}

// ---- x sweep ------------------------------------------------------------------------------------
// position p = row*rowlen + ii, cell i = g0-1+ii of row (b, k0+kk, j0+jj); thread t>=1 with ii>=1 owns face (i-1/2).
// The flux divergence of the non-magnetic components is accumulated by the sweeps themselves into racc (layout
// [block][NH][k][j][i], NH = 5 + NS: D, S_j, tau and the passive scalar): R <- R - (F_{+1/2} - F_{-1/2})/dx, the first active
// direction starting from zero.  Only the magnetic components of the fluxes, which flux-CT needs at neighbouring cells, are
// stored (all components when `store_all` is set: phx_debug_flux).  The sweeps are fp64-bound with HBM to spare, the update
// is HBM-bound: this moves 80 bytes per zone of flux reads out of the update.
template <int NS>
__device__ __forceinline__ int hydro_var(int h) { return h < 5 ? h : XS; }   // h-th accumulated component -> variable index

template <int METRIC, int RECON, int NS>
__global__ void __launch_bounds__(XS_BLOCK, (RECON == 4 ? 6 : (RECON <= 2 ? 5 : PHX_XS_MINB))) k_sweep_x(MeshDev m, const double* __restrict__ prim, double* __restrict__ flux,
                                                      double* __restrict__ racc, int store_all, int nplane, int rowlen, int j0, int k0) {
  // blockIdx.z = block, blockIdx.y = kk selects one k-plane; positions inside the plane are tiled flat over (jj, ii);
  // consecutive thread blocks overlap by two positions: thread 0 only supplies the left state of thread 1's face, the last
  // thread only the upper face of the cell before it
  constexpr int HW = ReconTraits<RECON>::HW;
  constexpr int NQ = NV + NS;
  constexpr int NH = 5 + NS;
  __shared__ double sh[NQ][XS_BLOCK];
  __shared__ double shF[NH][XS_BLOCK];
  const int t = threadIdx.x;
  const int p = blockIdx.x * (XS_BLOCK - 2) + t;
  const bool valid = p < nplane;
  double qm[NQ], qp[NQ];
  long long base = 0;
  int ii = 0, i = 0, j = 0, k = 0;
  const int b = blockIdx.z;
  if (valid) {
    const int kk = blockIdx.y;
    const int jj = p / rowlen;
    ii = p - jj * rowlen;
    i = m.g[0] - 1 + ii; j = j0 + jj; k = k0 + kk;
    base = (long long)b * m.nvar * m.ncell + (long long)k * m.sk + (long long)j * m.sj + i;
    double centre[NQ];
#pragma unroll
    for (int v = 0; v < NQ; ++v) {
      double f[2 * HW + 1];
#pragma unroll
      for (int s = 0; s <= 2 * HW; ++s) f[s] = prim[base + v * m.ncell + (s - HW)];
      centre[v] = f[HW];
      recon1<RECON>(f, qm[v], qp[v]);
    }
    {
      int cbc[3];
      double xc = 0.0, yc = 0.0, zc = 0.0;
      if (RECON >= 3 && m.floor_form != 0) {
        block_coords(m, b, cbc);
        xc = xcen(m, 0, cbc[0], i); yc = xcen(m, 1, cbc[1], j); zc = xcen(m, 2, cbc[2], k);
      }
      positivity_fallback<METRIC, RECON, NS>(m, xc, yc, zc, centre, qm, qp);
    }
#pragma unroll
    for (int v = 0; v < NQ; ++v) sh[v][t] = qp[v];
  }
  __syncthreads();
  const bool face = valid && t > 0 && ii > 0;          // this thread owns the face (i-1/2)
  double F[NQ];
  if (face) {
    double qL[NQ];
#pragma unroll
    for (int v = 0; v < NQ; ++v) qL[v] = sh[v][t - 1];
    int cb[3];
    block_coords(m, b, cb);
    Geo<METRIC> G;
    G.at(m, xface(m, 0, cb[0], i), xcen(m, 1, cb[1], j), xcen(m, 2, cb[2], k));
    face_flux<METRIC, 0, NS>(m, G, qL, qm, F);
#pragma unroll
    for (int h = 0; h < NH; ++h) shF[h][t] = F[hydro_var<NS>(h)];
  }
  __syncthreads();
  if (!face || t > XS_BLOCK - 2) return;               // the last thread's face belongs to the next block's thread 1
  if (store_all) {
#pragma unroll
    for (int v = 0; v < NQ; ++v) flux[base + v * m.ncell] = F[v];
  } else {
    flux[base + BY * m.ncell] = F[BY];
    flux[base + BZ * m.ncell] = F[BZ];
  }
  // cell (i, j, k): interior along x (ii <= n) and in the transverse directions
  if (ii <= m.n[0] && j >= m.g[1] && j < m.g[1] + m.n[1] && k >= m.g[2] && k < m.g[2] + m.n[2]) {
    const long long rb = (long long)b * NH * m.ncell + (long long)k * m.sk + (long long)j * m.sj + i;
#pragma unroll
    for (int h = 0; h < NH; ++h) racc[rb + h * m.ncell] = 0.0 - (shF[h][t + 1] - F[hydro_var<NS>(h)]) * m.rdx[0];
  }
}

// ---- y / z sweep ---------------------------------------------------------------------------------
// Lanes along x (coalesced); every thread marches along the sweep direction over one segment of cells c0..c1: it computes
// the faces c0..c1+1 (the last one again belongs to the next segment, which stores it), keeps the previous face's flux
// and accumulates the divergence of the non-magnetic components of the cells in between into racc.  The (2*HW+1)-row
// stencil window of its column lives in shared memory as a ring of rows that cp.async fills one row ahead of the
// arithmetic (each primitive is read from HBM once per segment, no register window, no long-scoreboard stall); a thread
// reads only its own column of the ring, so no block barrier is needed, only cp.async.wait_group.
// transverse position p -> (t1, t0) with t0 along x (fastest); blockIdx.y = segment, blockIdx.z = block.
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int METRIC, int RECON, int D, int NS>
__global__ void __launch_bounds__(MS_BLOCK, PHX_MS_MINB) k_sweep_march(MeshDev m, const double* __restrict__ prim, double* __restrict__ flux,
                                                                       double* __restrict__ racc, int store_all, int first,
                                                                       int ntr, int n0, int lo0, int lo1, int L) {
  constexpr int HW = ReconTraits<RECON>::HW;
  constexpr int NW = 2 * HW + 1;   // stencil rows
  constexpr int NR = NW + 1;       // ring: the stencil plus one row in flight
  constexpr int NQ = NV + NS;
  constexpr int NH = 5 + NS;
  constexpr int O = (D == 1) ? 2 : 1;   // the other transverse direction
  __shared__ double win[NR][NQ][MS_BLOCK];
  const int tid = threadIdx.x;
  const int p = blockIdx.x * MS_BLOCK + tid;
  if (p >= ntr) return;
  const int b = blockIdx.z;
  const int seg = blockIdx.y;
  const int t1 = p / n0, t0 = p - t1 * n0;
  const int i = lo0 + t0;             // x index
  const int o = lo1 + t1;             // the other transverse index (k for D=1, j for D=2)
  const long long sd = (D == 1) ? m.sj : m.sk;
  const long long so = (D == 1) ? m.sk : m.sj;
  const int clast = m.g[D] + m.n[D] - 1;          // last interior cell along D
  const int f0 = m.g[D] + seg * L;                // first cell (and first face) of this segment
  const int c1 = min(f0 + L - 1, clast);          // last cell
  if (f0 > c1) return;
  const int f1 = c1 + 1;                          // last face computed here
  const long long col = (long long)b * m.nvar * m.ncell + (long long)o * so + i;
  const long long rcol = (long long)b * NH * m.ncell + (long long)o * so + i;
  const bool inner = i >= m.g[0] && i < m.g[0] + m.n[0] && o >= m.g[O] && o < m.g[O] + m.n[O];   // interior column
  int cb[3];
  block_coords(m, b, cb);
  const double xx = xcen(m, 0, cb[0], i);
  const double xo = (D == 1) ? xcen(m, 2, cb[2], o) : xcen(m, 1, cb[1], o);

  const int rlast = f1 + HW;                      // last row any cell of this segment needs
  const double* src = prim + col + (long long)(f0 - 1 - HW) * sd;   // row f0-1-HW of this column
  // prologue: rows of the first cell's stencil, one commit group per row
#pragma unroll
  for (int r = 0; r < NW; ++r) {
#pragma unroll
    for (int v = 0; v < NQ; ++v) cp_async8(&win[r][v][tid], src + v * m.ncell);
    cp_async_commit();
    src += sd;
  }
  int s0 = 0;                                     // ring slot of row c-HW
  int snew = NW;                                  // ring slot the next prefetched row goes to
  // rst: divergence accumulated so far in the cell below the current face, fetched at the top of the iteration; fst: the
  // previous face's flux.  Kerr-Schild keeps both in shared memory (own column only, cp.async) to spare registers
  // (0.86 -> 0.78 ms on 512 blocks of 32^3); the flat metrics keep them in registers (PLM 0.55 vs 0.57 ms at 256^3).
  constexpr bool RSM = (METRIC == 1);
  __shared__ double rst[RSM ? NH : 1][MS_BLOCK];
  __shared__ double fst[RSM ? NH : 1][MS_BLOCK];
  double Rreg[NH], Freg[NH];
#pragma unroll
  for (int h = 0; h < NH; ++h) { Rreg[h] = 0.0; Freg[h] = 0.0; }
  double qpPrev[NQ];
#pragma unroll
  for (int v = 0; v < NQ; ++v) qpPrev[v] = 0.0;
  for (int c = f0 - 1; c <= f1; ++c) {
    const bool cell = inner && c >= f0 + 1;
    if (cell && !first) {
#pragma unroll
      for (int h = 0; h < NH; ++h) {
        if constexpr (RSM) cp_async8(&rst[h][tid], racc + rcol + h * m.ncell + (long long)(c - 1) * sd);
        else Rreg[h] = racc[rcol + h * m.ncell + (long long)(c - 1) * sd];
      }
    }
    if (c + HW + 1 <= rlast) {
#pragma unroll
      for (int v = 0; v < NQ; ++v) cp_async8(&win[snew][v][tid], src + v * m.ncell);
      src += sd;
    }
    cp_async_commit();
    cp_async_wait<1>();                           // everything but the row just issued has landed
    const double* wrow[NW];
#pragma unroll
    for (int r = 0; r < NW; ++r) {
      int sl = s0 + r;
      sl = (sl >= NR) ? sl - NR : sl;
      wrow[r] = &win[sl][0][tid];
    }
    double qm[NQ], qp[NQ], centre[NQ];
#pragma unroll
    for (int v = 0; v < NQ; ++v) {
      double f[NW];
#pragma unroll
      for (int r = 0; r < NW; ++r) f[r] = wrow[r][v * MS_BLOCK];
      centre[v] = f[HW];
      recon1<RECON>(f, qm[v], qp[v]);
    }
    {
      double xc = 0.0;
      if (RECON >= 3 && m.floor_form != 0) xc = xcen(m, D, cb[D], c);
      if (D == 1) positivity_fallback<METRIC, RECON, NS>(m, xx, xc, xo, centre, qm, qp);
      else positivity_fallback<METRIC, RECON, NS>(m, xx, xo, xc, centre, qm, qp);
    }
    if (c >= f0) {
      Geo<METRIC> G;
      const double xf = xface(m, D, cb[D], c);
      if (D == 1) G.at(m, xx, xf, xo); else G.at(m, xx, xo, xf);
      double F[NQ];
      face_flux<METRIC, D, NS>(m, G, qpPrev, qm, F);
      if (c <= c1 || c == clast + 1) {            // the face c1+1 is stored by the next segment unless it is the last face
        if (store_all) {
#pragma unroll
          for (int v = 0; v < NQ; ++v) flux[col + v * m.ncell + (long long)c * sd] = F[v];
        } else {
          flux[col + BX * m.ncell + (long long)c * sd] = F[BX];
          flux[col + (D == 1 ? BZ : BY) * m.ncell + (long long)c * sd] = F[D == 1 ? BZ : BY];
        }
      }
      if (cell) {
        if constexpr (RSM) cp_async_wait<0>();    // rst (and the row in flight) have landed long ago
#pragma unroll
        for (int h = 0; h < NH; ++h) {
          const double Rold = first ? 0.0 : (RSM ? rst[h][tid] : Rreg[h]);
          const double Fp = RSM ? fst[h][tid] : Freg[h];
          racc[rcol + h * m.ncell + (long long)(c - 1) * sd] = Rold - (F[hydro_var<NS>(h)] - Fp) * m.rdx[D];
        }
      }
#pragma unroll
      for (int h = 0; h < NH; ++h) {
        if constexpr (RSM) fst[h][tid] = F[hydro_var<NS>(h)];
        else Freg[h] = F[hydro_var<NS>(h)];
      }
    }
#pragma unroll
    for (int v = 0; v < NQ; ++v) qpPrev[v] = qp[v];
    s0 = (s0 + 1 == NR) ? 0 : s0 + 1;
    snew = (snew + 1 == NR) ? 0 : snew + 1;
  }
  cp_async_wait<0>();
}

// ---- update: flux-CT + divergence + sources + RK combine + con2prim + floors ----------------------
struct FluxPtrs { const double* f[3]; const double* racc; };

// A cell whose sum_d max|lambda^d|/dx_d is NaN (non-finite primitives) must not be dropped by fmax: it enters the reduction
// as +inf, and the final kernels turn an infinite maximum into dt = NaN, which no later step can hide.  A mesh without any
// evolving cell (maximum 0) gets dt = +inf: nothing constrains the step.
__device__ __forceinline__ double cfl_guard(double s) { return (s >= 0.0) ? s : __longlong_as_double(0x7ff0000000000000LL); }
__device__ __forceinline__ double cfl_dt_of(double cfl, double vmax) {
  return isinf(vmax) ? __longlong_as_double(0x7ff8000000000000LL) : cfl * (1.0 / vmax);
}


// contribution of the edge-EMF pair (A, C) (third direction E) to d/dt of B~^C and B~^A, reading C5.3
template <int A, int C, bool EXC>
__device__ __forceinline__ void ct_pair(const MeshDev& m, const FluxPtrs& fl, const unsigned char* __restrict__ xfl, long long vb,
                                        long long fb, long long c, const long long* str, unsigned xbit, double* dB) {
  const double* FaBc = fl.f[A] + vb + (long long)(BX + C) * m.ncell;
  const double* FcBa = fl.f[C] + vb + (long long)(BX + A) * m.ncell;
  auto E = [&](long long id) {
    double e = 0.25 * (FaBc[id] + FaBc[id - str[C]] - FcBa[id] - FcBa[id - str[A]]);
    if (EXC) { if (xfl[fb + id] & xbit) e = 0.0; }
    return e;
  };
  const double e00 = E(c), e10 = E(c + str[A]), e01 = E(c + str[C]), e11 = E(c + str[A] + str[C]);
  dB[C] -= (0.5 * (e10 + e11) - 0.5 * (e00 + e01)) * m.rdx[A];
  dB[A] -= (-0.5 * (e01 + e11) + 0.5 * (e00 + e10)) * m.rdx[C];
}

// One cell of the update.  Returns sum_d max|lambda^d|/dx_d of the new primitives when CFL is set (0 for a thread without
// a cell or with an excised one), so that the kernel can reduce the next time step on the fly.
// RF: the floors depend on the position (floor_form != 0); a template flag so that the constant-floor kernels carry none of it
template <int METRIC, bool EXC, bool CFL, int NS, bool RF>
__device__ __forceinline__ double update_cell(const MeshDev& m, const FluxPtrs& fl, const unsigned char* __restrict__ xfl, double g0, double g1,
                                              double bdt_host, const double* __restrict__ d_dt, double beta,
                                              const double* cons0, const double* cons_in, double* cons_out,
                                              double* __restrict__ prim, unsigned char* __restrict__ mask) {
  // U~_out = g0 U~0 + g1 U~_in + bdt R.  cons_out may alias cons_in or cons0 (every thread touches only its own cell of
  // the conserved fields); cons_in is not read when g1 == 0 (first stage).
  // blockIdx.z = block, blockIdx.y = kk selects one interior k-plane; the plane is tiled flat over (jj, ii)
  const int p = blockIdx.x * UP_BLOCK + threadIdx.x;
  if (p >= m.n[0] * m.n[1]) return 0.0;
  const int jj = p / m.n[0];
  const int ii = p - jj * m.n[0];
  const int b = blockIdx.z;
  const int kk = blockIdx.y;
  const int i = ii + m.g[0], j = jj + m.g[1], k = kk + m.g[2];
  const long long c = (long long)k * m.sk + (long long)j * m.sj + i;
  constexpr int NQ = NV + NS;
  const long long vb = (long long)b * m.nvar * m.ncell;  // block offset in a field of nvar variables
  const long long fb = (long long)b * m.ncell;          // block offset in a one-variable field
  if (EXC) {
    if (xfl[fb + c] & XF_CELL) {   // frozen cell: the RK combination of two equal states is exact
#pragma unroll
      for (int v = 0; v < NQ; ++v) {
        const long long id = vb + v * m.ncell + c;
        cons_out[id] = (g1 != 0.0) ? g0 * cons0[id] + g1 * cons_in[id] : cons0[id];
      }
      mask[fb + c] = M_EXCISED;
      return 0.0;
    }
  }
  // Kerr-Schild only (see PHX_UP_STAGE_KS): the cell's own streaming operands (U~0, U~_in, stage-input primitives) are fetched
  // by cp.async into shared memory before the flux phase: they are in flight while the flux / CT loads go out and cost no
  // registers until they are used.
  // Every thread reads back only what it copied itself, so cp.async.wait_group is all the synchronisation needed.
  constexpr int STG = (METRIC == 1) ? PHX_UP_STAGE_KS : 0;
  constexpr int NPQ = (METRIC == 1) ? NV : 5;
  __shared__ double stg[STG ? (2 * NQ + (STG == 1 ? NPQ : 0)) : 1][UP_BLOCK];
  const int tid = threadIdx.x;
  if constexpr (STG != 0) {
#pragma unroll
    for (int v = 0; v < NQ; ++v) cp_async8(&stg[v][tid], cons0 + vb + v * m.ncell + c);
    if (g1 != 0.0) {
#pragma unroll
      for (int v = 0; v < NQ; ++v) cp_async8(&stg[NQ + v][tid], cons_in + vb + v * m.ncell + c);
    }
    if constexpr (STG == 1) {
#pragma unroll
      for (int v = 0; v < NPQ; ++v) cp_async8(&stg[2 * NQ + v][tid], prim + vb + v * m.ncell + c);
    }
    cp_async_commit();
  }
  const double bdt = d_dt ? beta * (*d_dt) : bdt_host;
  const long long str[3] = {1, m.sj, m.sk};
  double R[NQ];
#pragma unroll
  for (int v = 0; v < NQ; ++v) R[v] = 0.0;
  // D, S_j, tau (and the passive scalar, which has no source: S = 0 in Eq.14): the divergence the sweeps accumulated
  if (m.act[0] || m.act[1] || m.act[2]) {
    constexpr int NH = 5 + NS;
    const double* A = fl.racc + (long long)b * NH * m.ncell + c;
#pragma unroll
    for (int h = 0; h < NH; ++h) R[hydro_var<NS>(h)] = A[h * m.ncell];
  }
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (!m.act[d]) continue;
    const double* F = fl.f[d] + vb + c;
    // magnetic components that flux-CT does not replace (inactive partner direction, or CT switched off)
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
      if (cc == d) continue;
      if (m.use_ct && m.act[cc]) continue;
      R[BX + cc] -= (F[(BX + cc) * m.ncell + str[d]] - F[(BX + cc) * m.ncell]) * m.rdx[d];
    }
  }
  if (m.use_ct) {
    double dB[3] = {0.0, 0.0, 0.0};
    if (m.act[0] && m.act[1]) ct_pair<0, 1, EXC>(m, fl, xfl, vb, fb, c, str, XF_E3, dB);
    if (m.act[1] && m.act[2]) ct_pair<1, 2, EXC>(m, fl, xfl, vb, fb, c, str, XF_E1, dB);
    if (m.act[2] && m.act[0]) ct_pair<2, 0, EXC>(m, fl, xfl, vb, fb, c, str, XF_E2, dB);
    R[BX] += dB[0]; R[BY] += dB[1]; R[BZ] += dB[2];
  }
  int cb[3];
  block_coords(m, b, cb);
  const double x = xcen(m, 0, cb[0], i), y = xcen(m, 1, cb[1], j), z = xcen(m, 2, cb[2], k);
  double U[NQ], q[NQ];
  // stage-input primitives of this cell: sources, and the initial guess of the con2prim root
  if constexpr (STG != 0) cp_async_wait<0>();
  if constexpr (STG == 1) {
#pragma unroll
    for (int v = 0; v < NPQ; ++v) q[v] = stg[2 * NQ + v][tid];
  } else {
    q[RHO] = prim[vb + RHO * m.ncell + c];
    q[UX] = prim[vb + UX * m.ncell + c]; q[UY] = prim[vb + UY * m.ncell + c]; q[UZ] = prim[vb + UZ * m.ncell + c];
    q[UU] = prim[vb + UU * m.ncell + c];
    if constexpr (METRIC == 1) { q[BX] = prim[vb + BX * m.ncell + c]; q[BY] = prim[vb + BY * m.ncell + c]; q[BZ] = prim[vb + BZ * m.ncell + c]; }
  }
  if constexpr (METRIC == 1) {
    double S[4];
    ks_sources(m, x, y, z, q, S);
    R[CS1] += S[0]; R[CS2] += S[1]; R[CS3] += S[2]; R[CTAU] += S[3];
  }
#pragma unroll
  for (int v = 0; v < NQ; ++v) {
    const long long id = vb + v * m.ncell + c;
    if constexpr (STG != 0) U[v] = (g1 != 0.0) ? g0 * stg[v][tid] + g1 * stg[NQ + v][tid] + bdt * R[v] : g0 * stg[v][tid] + bdt * R[v];
    else U[v] = (g1 != 0.0) ? g0 * cons0[id] + g1 * cons_in[id] + bdt * R[v] : g0 * cons0[id] + bdt * R[v];
  }
  Geo<METRIC> G;
  G.at(m, x, y, z);
  const double mu_guess = c2p_guess<METRIC>(G, q, m.gam);
  double rfl = m.rho_floor, efl = m.eps_floor;
  if constexpr (RF) floors_at<METRIC>(m, x, y, z, rfl, efl);
  const double Dt_in = U[CD];
  unsigned mk = c2p_cell<METRIC>(m, G, rfl, efl, U, q, mu_guess);
  if constexpr (NS == 1) scalar_recover(m, Dt_in, U[CD], mk, U[XS], q[XS]);
#pragma unroll
  for (int v = 0; v < NQ; ++v) {
    const long long id = vb + v * m.ncell + c;
    cons_out[id] = U[v];
    prim[id] = q[v];
  }
  mask[fb + c] = (unsigned char)mk;
  if constexpr (CFL) {
    double lam[3];
    max_speeds<METRIC>(q, G, m.gam, lam);
    double sum = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) if (m.act[d]) sum += lam[d] * m.rdx[d];
    return cfl_guard(sum);
  }
  return 0.0;
}

// smax: PHX_NSLOT accumulators of the largest sum_d max|lambda^d|/dx_d seen (bit pattern of a non-negative double, which
// orders like the unsigned integer), one atomicMax per thread block; k_cfl_final_slots turns them into the time step.
constexpr int PHX_NSLOT = 1024;
template <int METRIC, bool EXC, bool CFL, int NS, bool RF>
__global__ void __launch_bounds__(UP_BLOCK, (METRIC == 1 ? PHX_UP_MINB_KS : PHX_UP_MINB)) k_update(MeshDev m, FluxPtrs fl, const unsigned char* __restrict__ xfl, double g0, double g1,
                                                     double bdt_host, const double* __restrict__ d_dt, double beta,
                                                     const double* cons0, const double* cons_in, double* cons_out,
                                                     double* __restrict__ prim, unsigned char* __restrict__ mask,
                                                     unsigned long long* __restrict__ smax) {
  double sum = update_cell<METRIC, EXC, CFL, NS, RF>(m, fl, xfl, g0, g1, bdt_host, d_dt, beta, cons0, cons_in, cons_out, prim, mask);
  if constexpr (CFL) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum = fmax(sum, __shfl_xor_sync(0xffffffffu, sum, o));
    __shared__ double sh[UP_BLOCK / 32];
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
      double v = sh[0];
#pragma unroll
      for (int w = 1; w < UP_BLOCK / 32; ++w) v = fmax(v, sh[w]);
      const unsigned slot = (blockIdx.x + blockIdx.y * gridDim.x + blockIdx.z * gridDim.x * gridDim.y) % PHX_NSLOT;
      atomicMax(&smax[slot], (unsigned long long)__double_as_longlong(v));
    }
  }
}

// dt = cfl / max over the slots; the slots are reset for the next accumulation
__global__ void __launch_bounds__(256) k_cfl_final_slots(unsigned long long* __restrict__ smax, double cfl, double* __restrict__ dt) {
  double best = 0.0;
  for (int p = threadIdx.x; p < PHX_NSLOT; p += 256) { best = fmax(best, __longlong_as_double((long long)smax[p])); smax[p] = 0ull; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ double sh[8];
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    double v = sh[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) v = fmax(v, sh[w]);
    *dt = cfl_dt_of(cfl, v);
  }
}

// ---- stand-alone con2prim, prim->cons ---------------------------------------------------------------
template <int METRIC, bool EXC, int NS, bool RF>
__global__ void __launch_bounds__(UP_BLOCK) k_c2p(MeshDev m, const unsigned char* __restrict__ xfl, double* __restrict__ cons,
                                                  double* __restrict__ prim, unsigned char* __restrict__ mask, long long ninterior) {
  const long long p = (long long)blockIdx.x * UP_BLOCK + threadIdx.x;
  if (p >= ninterior) return;
  const int ii = (int)(p % m.n[0]);
  long long r = p / m.n[0];
  const int jj = (int)(r % m.n[1]); r /= m.n[1];
  const int kk = (int)(r % m.n[2]);
  const int b = (int)(r / m.n[2]);
  const int i = ii + m.g[0], j = jj + m.g[1], k = kk + m.g[2];
  const long long c = (long long)k * m.sk + (long long)j * m.sj + i;
  constexpr int NQ = NV + NS;
  const long long vb = (long long)b * m.nvar * m.ncell, fb = (long long)b * m.ncell;
  if (EXC) {
    if (xfl[fb + c] & XF_CELL) { mask[fb + c] = M_EXCISED; return; }
  }
  int cb[3];
  block_coords(m, b, cb);
  Geo<METRIC> G;
  const double x = xcen(m, 0, cb[0], i), y = xcen(m, 1, cb[1], j), z = xcen(m, 2, cb[2], k);
  G.at(m, x, y, z);
  double U[NQ], q[NQ];
#pragma unroll
  for (int v = 0; v < NQ; ++v) U[v] = cons[vb + v * m.ncell + c];
  double rfl = m.rho_floor, efl = m.eps_floor;
  if constexpr (RF) floors_at<METRIC>(m, x, y, z, rfl, efl);
  const double Dt_in = U[CD];
  unsigned mk = c2p_cell<METRIC>(m, G, rfl, efl, U, q);
  if constexpr (NS == 1) scalar_recover(m, Dt_in, U[CD], mk, U[XS], q[XS]);
#pragma unroll
  for (int v = 0; v < NQ; ++v) {
    if (mk & (M_RHO_FLOOR | M_EPS_FLOOR | M_W_CEIL | M_BAD_INPUT | M_SCALAR_CLIPPED)) cons[vb + v * m.ncell + c] = U[v];
    prim[vb + v * m.ncell + c] = q[v];
  }
  mask[fb + c] = (unsigned char)mk;
}

template <int METRIC>
__global__ void __launch_bounds__(256) k_prim_to_cons(MeshDev m, const double* __restrict__ prim, double* __restrict__ cons, long long nall) {
  const long long p = (long long)blockIdx.x * 256 + threadIdx.x;
  if (p >= nall) return;
  const int i = (int)(p % m.na[0]);
  long long r = p / m.na[0];
  const int j = (int)(r % m.na[1]); r /= m.na[1];
  const int k = (int)(r % m.na[2]);
  const int b = (int)(r / m.na[2]);
  const long long id = (long long)b * m.nvar * m.ncell + (long long)k * m.sk + (long long)j * m.sj + i;
  int cb[3];
  block_coords(m, b, cb);
  Geo<METRIC> G;
  G.at(m, xcen(m, 0, cb[0], i), xcen(m, 1, cb[1], j), xcen(m, 2, cb[2], k));
  double q[NV], U[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) q[v] = prim[id + v * m.ncell];
  prim_to_cons_pt<METRIC>(q, G, m.gam, U);
#pragma unroll
  for (int v = 0; v < NV; ++v) cons[id + v * m.ncell] = U[v];
  if (m.nvar > NV) cons[id + XS * m.ncell] = U[CD] * prim[id + XS * m.ncell];   // sqrt(gamma) D X (Eq.14)
}

// ---- ghost fill: one gather pass -------------------------------------------------------------------
// blockIdx.z = block; the threads enumerate the ghost cells of the block only: first the k-planes below and above the
// interior, then the rows below and above the interior rows of every interior k-plane, then the end cells of every interior
// row (nA, nB: sizes of the first two groups, ntot: all ghost cells enumerated).
// GhostShell: the ghost cells within dep[d] <= g[d] layers of the interior (the whole frame: dep = g).  The first stage of a
// fused two-stage step fills only the layers its second stage reads: stencil half-width + 1 along a sweep, 1 across it.
struct GhostShell { int dep[3]; int nA, nB, ntot; };

// source of the ghost cell l (allocated indices) of the block at coordinates cb: element index of its variable 0
__device__ __forceinline__ long long ghost_source(const MeshDev& m, const int* cb, const int* l) {
  int sb[3], sl[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    // source cell in block-local terms: inside this block, in the neighbour block, wrapped or clamped at a domain face
    int li = l[d] - m.g[d];            // -g .. n+g-1
    int nbk = cb[d];
    if (li < 0) {
      if (nbk > 0) { nbk -= 1; li += m.n[d]; }
      else if (m.bc[d][0] == 0) { nbk = m.nb[d] - 1; li += m.n[d]; }
      else li = 0;
    } else if (li >= m.n[d]) {
      if (nbk < m.nb[d] - 1) { nbk += 1; li -= m.n[d]; }
      else if (m.bc[d][1] == 0) { nbk = 0; li -= m.n[d]; }
      else li = m.n[d] - 1;
    }
    sb[d] = nbk;
    sl[d] = li + m.g[d];
  }
  const int bs = (sb[2] * m.nb[1] + sb[1]) * m.nb[0] + sb[0];
  return (long long)bs * m.nvar * m.ncell + (long long)sl[2] * m.sk + (long long)sl[1] * m.sj + sl[0];
}

// VEC = 2: one thread copies two x-adjacent ghost cells (n_x, g_x and the x depth of the shell even: every run of ghost cells
// along x then starts at an even, 16-byte aligned index) with one 16-byte load and store per variable where the two sources
// are adjacent too (everywhere but at an outflow face, whose ghosts all copy the same cell).
template <int VEC>
__global__ void __launch_bounds__(256) k_fill_ghosts(MeshDev m, double* __restrict__ prim, GhostShell gs) {
  int t = blockIdx.x * 256 + threadIdx.x;
  if (t >= gs.ntot) return;
  int l[3];
  const int w0 = (m.n[0] + 2 * gs.dep[0]) / VEC, w1 = m.n[1] + 2 * gs.dep[1];     // extent of the shell's bounding box (x in units of VEC cells)
  const int o0 = m.g[0] - gs.dep[0], o1 = m.g[1] - gs.dep[1], o2 = m.g[2] - gs.dep[2];
  if (t < gs.nA) {                      // the k-planes below and above the interior
    const int plane = w0 * w1;
    const int kz = t / plane;
    t -= kz * plane;
    l[2] = kz < gs.dep[2] ? o2 + kz : m.g[2] + m.n[2] + (kz - gs.dep[2]);
    const int jy = t / w0;
    l[1] = o1 + jy;
    l[0] = o0 + VEC * (t - jy * w0);
  } else if (t < gs.nA + gs.nB) {       // the rows below and above the interior rows of every interior k-plane
    t -= gs.nA;
    const int per = 2 * gs.dep[1] * w0;
    const int kk = t / per;
    t -= kk * per;
    const int jy = t / w0;
    l[2] = m.g[2] + kk;
    l[1] = jy < gs.dep[1] ? o1 + jy : m.g[1] + m.n[1] + (jy - gs.dep[1]);
    l[0] = o0 + VEC * (t - jy * w0);
  } else {                              // the end cells of every interior row
    t -= gs.nA + gs.nB;
    const int w = 2 * gs.dep[0] / VEC;
    const int row = t / w;
    const int ix = VEC * (t - row * w);
    const int kk = row / m.n[1];
    l[2] = m.g[2] + kk;
    l[1] = m.g[1] + (row - kk * m.n[1]);
    l[0] = ix < gs.dep[0] ? o0 + ix : m.g[0] + m.n[0] + (ix - gs.dep[0]);
  }
  const int b = blockIdx.z;
  int cb[3];
  block_coords(m, b, cb);
  const long long src = ghost_source(m, cb, l);
  const long long dst = (long long)b * m.nvar * m.ncell + (long long)l[2] * m.sk + (long long)l[1] * m.sj + l[0];
  if constexpr (VEC == 1) {
    double v[NV + 1];
#pragma unroll
    for (int q = 0; q < NV; ++q) v[q] = prim[src + q * m.ncell];
    if (m.nvar > NV) v[XS] = prim[src + XS * m.ncell];
#pragma unroll
    for (int q = 0; q < NV; ++q) prim[dst + q * m.ncell] = v[q];
    if (m.nvar > NV) prim[dst + XS * m.ncell] = v[XS];
  } else {
    int l1[3] = {l[0] + 1, l[1], l[2]};
    const long long src1 = ghost_source(m, cb, l1);
    double2 v[NV + 1];
    if (src1 == src + 1 && (src & 1) == 0) {
#pragma unroll
      for (int q = 0; q < NV; ++q) v[q] = *reinterpret_cast<const double2*>(prim + src + q * m.ncell);
      if (m.nvar > NV) v[XS] = *reinterpret_cast<const double2*>(prim + src + XS * m.ncell);
    } else {
#pragma unroll
      for (int q = 0; q < NV; ++q) { v[q].x = prim[src + q * m.ncell]; v[q].y = prim[src1 + q * m.ncell]; }
      if (m.nvar > NV) { v[XS].x = prim[src + XS * m.ncell]; v[XS].y = prim[src1 + XS * m.ncell]; }
    }
#pragma unroll
    for (int q = 0; q < NV; ++q) *reinterpret_cast<double2*>(prim + dst + q * m.ncell) = v[q];
    if (m.nvar > NV) *reinterpret_cast<double2*>(prim + dst + XS * m.ncell) = v[XS];
  }
}

// ---- CFL: warp-shuffle min reduction ------------------------------------------------------------------
template <int METRIC, bool EXC>
__global__ void __launch_bounds__(256) k_cfl_partial(MeshDev m, const unsigned char* __restrict__ xfl, const double* __restrict__ prim,
                                                     double* __restrict__ partial, long long ninterior) {
  // max of sum_d max|lambda^d|/dx_d; the final kernel takes cfl * (1/max), which equals cfl * min(1/sum) bit for bit
  // because IEEE division is monotone
  double best = 0.0;
  for (long long p = (long long)blockIdx.x * 256 + threadIdx.x; p < ninterior; p += (long long)gridDim.x * 256) {
    const int ii = (int)(p % m.n[0]);
    long long r = p / m.n[0];
    const int jj = (int)(r % m.n[1]); r /= m.n[1];
    const int kk = (int)(r % m.n[2]);
    const int b = (int)(r / m.n[2]);
    const int i = ii + m.g[0], j = jj + m.g[1], k = kk + m.g[2];
    const long long c = (long long)k * m.sk + (long long)j * m.sj + i;
    if (EXC) { if (xfl[(long long)b * m.ncell + c] & XF_CELL) continue; }
    int cb[3];
    block_coords(m, b, cb);
    Geo<METRIC> G;
    G.at(m, xcen(m, 0, cb[0], i), xcen(m, 1, cb[1], j), xcen(m, 2, cb[2], k));
    double q[NV], lam[3];
#pragma unroll
    for (int v = 0; v < NV; ++v) q[v] = prim[(long long)b * m.nvar * m.ncell + v * m.ncell + c];
    max_speeds<METRIC>(q, G, m.gam, lam);
    double s = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) if (m.act[d]) s += lam[d] * m.rdx[d];
    best = fmax(best, cfl_guard(s));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ double sh[8];
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x < 32) {
    double v = (threadIdx.x < 8) ? sh[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (threadIdx.x == 0) partial[blockIdx.x] = v;
  }
}

__global__ void __launch_bounds__(256) k_cfl_final(const double* __restrict__ partial, int n, double cfl, double* __restrict__ dt) {
  double best = 0.0;
  for (int p = threadIdx.x; p < n; p += 256) best = fmax(best, partial[p]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ double sh[8];
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x < 32) {
    double v = (threadIdx.x < 8) ? sh[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (threadIdx.x == 0) *dt = cfl_dt_of(cfl, v);
  }
}

// ---- excision flags (init only) ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_excision_flags(MeshDev m, unsigned char* __restrict__ xfl, long long nall) {
  const long long p = (long long)blockIdx.x * 256 + threadIdx.x;
  if (p >= nall) return;
  int l[3];
  l[0] = (int)(p % m.na[0]);
  long long r = p / m.na[0];
  l[1] = (int)(r % m.na[1]); r /= m.na[1];
  l[2] = (int)(r % m.na[2]);
  const int b = (int)(r / m.na[2]);
  int cb[3];
  block_coords(m, b, cb);
  auto ex = [&](int di, int dj, int dk) {
    double rr, H, lv[3];
    ks_scalars(m, xcen(m, 0, cb[0], l[0] - di), xcen(m, 1, cb[1], l[1] - dj), xcen(m, 2, cb[2], l[2] - dk), rr, H, lv);
    return rr < m.r_exc;
  };
  unsigned f = 0;
  if (ex(0, 0, 0)) f |= XF_CELL;
  if (ex(0, 0, 0) || ex(0, 1, 0) || ex(0, 0, 1) || ex(0, 1, 1)) f |= XF_E1;   // edge (j-1/2, k-1/2)
  if (ex(0, 0, 0) || ex(1, 0, 0) || ex(0, 0, 1) || ex(1, 0, 1)) f |= XF_E2;   // edge (i-1/2, k-1/2)
  if (ex(0, 0, 0) || ex(1, 0, 0) || ex(0, 1, 0) || ex(1, 1, 0)) f |= XF_E3;   // edge (i-1/2, j-1/2)
  xfl[p] = (unsigned char)f;
}

// ================================================================================================ host side
struct phx_mesh {
  MeshDev m;
  phx_params par;
  double* flux[3];
  double* racc;               // divergence of the non-magnetic flux components accumulated by the sweeps: [block][5+nscalar][cells]
  int store_all_fluxes;       // phx_debug_enable_flux: the sweeps also store the non-magnetic flux components
  int small_1d;               // phx_evolve_device may take the one-block path for small 1-D meshes (PHX_SMALL_1D=0 switches it off)
  unsigned char* xfl;
  double* partial;
  int npartial;
  unsigned long long* smax;   // PHX_NSLOT accumulators of the fused CFL reduction (zero between steps)
  int nsm;                    // SMs of the device the mesh lives on (launch sizing)
  // bookkeeping that calls on a const mesh update (launch counter, event records): not part of the mesh's logical state
  mutable unsigned long long launches;
  long long nall, ninterior;
  // workspace of the host-buffer path (phx_evolve_host), allocated on first use
  double* ws_field[3];
  unsigned char* ws_mask;
  double* ws_scal;   // [0] dt, [1] t
  // per-kernel-class CUDA-event timing (phx_profile_enable / phx_profile_read)
  mutable cudaEvent_t* ev;   // 2 events per recorded launch
  mutable int* evcls;
  mutable int evcap, evn;
  // CUDA graph of one RK2 step (phx_evolve_device): captured once per argument set on a mesh-owned stream and replayed
  cudaStream_t gstream;
  cudaEvent_t gev_in, gev_out;
  cudaGraphExec_t gexec;
  unsigned long long glaunches;        // kernel launches one replay stands for
  struct { double cfl; double *dt, *t, *cons0, *cons, *prim; unsigned char* mask; } gkey;
};

// RAII pair of events around one launch (or one group of launches) of class `cls`, recorded on the launching stream
struct ProfScope {
  const phx_mesh* M; cudaStream_t st; int slot;
  ProfScope(const phx_mesh* M_, int cls, cudaStream_t st_) : M(M_), st(st_), slot(-1) {
    if (M->ev && M->evn < M->evcap) { slot = M->evn++; M->evcls[slot] = cls; cudaEventRecord(M->ev[2 * slot], st); }
  }
  ~ProfScope() { if (slot >= 0) cudaEventRecord(M->ev[2 * slot + 1], st); }
};

static thread_local char g_err[512] = "";
static int fail(int code, const char* msg) {
  snprintf(g_err, sizeof g_err, "%s", msg);
  return code;
}
static int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_err, sizeof g_err, "%s: %s", where, cudaGetErrorString(e));
  return PHX_ECUDA;
}
#define CUDA_TRY(x, where) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)
#define LAUNCH_CHECK(mesh, where) do { (mesh)->launches++; cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

static bool aligned16(const void* p) { return p && (((uintptr_t)p) & 15u) == 0; }

extern "C" const char* phx_last_error(void) { return g_err; }

extern "C" int phx_init_mesh(const phx_params* p, void* stream, phx_mesh** out) {
  if (!p || !out) return fail(PHX_EINVAL, "phx_init_mesh: null argument");
  *out = nullptr;
  if (p->nx < 1 || p->ny < 1 || p->nz < 1 || p->nbx < 1 || p->nby < 1 || p->nbz < 1) return fail(PHX_EINVAL, "phx_init_mesh: sizes must be >= 1");
  if (p->metric != PHX_MINKOWSKI && p->metric != PHX_KERR_SCHILD && p->metric != PHX_MINKOWSKI_BOOSTED) return fail(PHX_EINVAL, "phx_init_mesh: unknown metric");
  if (p->metric == PHX_MINKOWSKI_BOOSTED && !(p->shift[0] * p->shift[0] + p->shift[1] * p->shift[1] + p->shift[2] * p->shift[2] < 1.0))
    return fail(PHX_EINVAL, "phx_init_mesh: |shift| must be below 1");
  if (p->recon < 0 || p->recon > 5) return fail(PHX_EUNSUPPORTED, "phx_init_mesh: unknown reconstruction");
  if (p->riemann < 0 || p->riemann > 1) return fail(PHX_EUNSUPPORTED, "phx_init_mesh: unknown Riemann solver");
  const int need = (p->recon >= 3) ? 3 : 2;
  if (p->ng < need) return fail(PHX_EINVAL, "phx_init_mesh: ng too small for the reconstruction stencil (>=2 PLM, >=3 WENO5-Z)");
  if (!(p->gamma_ad > 1.0)) return fail(PHX_EINVAL, "phx_init_mesh: gamma_ad must exceed 1");
  if (!(p->rho_floor > 0.0) || !(p->eps_floor > 0.0) || !(p->w_max > 1.0)) return fail(PHX_EINVAL, "phx_init_mesh: floors must be positive, w_max > 1");
  if (!(p->c2p_tol > 0.0) || p->c2p_maxit < 1) return fail(PHX_EINVAL, "phx_init_mesh: c2p_tol > 0 and c2p_maxit >= 1 required");
  if (p->metric == PHX_KERR_SCHILD && !(p->bh_mass > 0.0)) return fail(PHX_EINVAL, "phx_init_mesh: bh_mass must be positive");
  if (p->nscalar < 0 || p->nscalar > 1) return fail(PHX_EUNSUPPORTED, "phx_init_mesh: nscalar must be 0 or 1");
  if (p->nscalar == 1 && !(p->scalar_max > p->scalar_min)) return fail(PHX_EINVAL, "phx_init_mesh: scalar_max must exceed scalar_min");
  if (p->floor_form < PHX_FLOOR_CONST || p->floor_form > PHX_FLOOR_POW_R) return fail(PHX_EUNSUPPORTED, "phx_init_mesh: unknown floor form");
  if (p->floor_form != PHX_FLOOR_CONST && (!(p->floor_alpha_rho >= 0.0) || !(p->floor_alpha_eps >= 0.0)))
    return fail(PHX_EINVAL, "phx_init_mesh: floor exponents must be non-negative");
  phx_mesh* M = new (std::nothrow) phx_mesh();
  if (!M) return fail(PHX_ENOMEM, "phx_init_mesh: host allocation failed");
  memset(M, 0, sizeof *M);
  M->par = *p;
  MeshDev& m = M->m;
  m.metric = p->metric; m.M = p->bh_mass; m.a = p->bh_spin; m.r_exc = p->r_excise;
  m.nb[0] = p->nbx; m.nb[1] = p->nby; m.nb[2] = p->nbz;
  m.n[0] = p->nx; m.n[1] = p->ny; m.n[2] = p->nz;
  for (int d = 0; d < 3; ++d) {
    m.N[d] = m.nb[d] * m.n[d];
    m.act[d] = m.N[d] > 1;
    if (!m.act[d]) { /* nothing */ }
    if (m.act[d] && m.n[d] < p->ng) { delete M; return fail(PHX_EINVAL, "phx_init_mesh: an active dimension needs at least ng zones per block"); }
    m.g[d] = m.act[d] ? p->ng : 0;
    m.na[d] = m.n[d] + 2 * m.g[d];
    if (!(p->xmax[d] > p->xmin[d])) { delete M; return fail(PHX_EINVAL, "phx_init_mesh: xmax must exceed xmin"); }
    m.xmin[d] = p->xmin[d];
    m.dx[d] = (p->xmax[d] - p->xmin[d]) / m.N[d];
    m.rdx[d] = 1.0 / m.dx[d];
    for (int s = 0; s < 2; ++s) {
      if (p->bc[d][s] != PHX_BC_PERIODIC && p->bc[d][s] != PHX_BC_OUTFLOW) { delete M; return fail(PHX_EINVAL, "phx_init_mesh: unknown boundary condition"); }
      m.bc[d][s] = p->bc[d][s];
    }
  }
  m.nblk = m.nb[0] * m.nb[1] * m.nb[2];
  m.sj = m.na[0];
  m.sk = (long long)m.na[0] * m.na[1];
  m.ncell = m.sk * m.na[2];
  m.gam = p->gamma_ad; m.recon = p->recon; m.riemann = p->riemann; m.use_ct = p->use_ct ? 1 : 0;
  m.rho_floor = p->rho_floor; m.eps_floor = p->eps_floor; m.w_max = p->w_max; m.c2p_tol = p->c2p_tol; m.c2p_maxit = p->c2p_maxit;
  m.excise = (p->metric == PHX_KERR_SCHILD && p->r_excise > 0.0) ? 1 : 0;
  for (int d = 0; d < 3; ++d) m.shift[d] = (p->metric == PHX_MINKOWSKI_BOOSTED) ? p->shift[d] : 0.0;
  m.nvar = NV + p->nscalar;
  m.xs_min = p->scalar_min; m.xs_max = p->scalar_max;
  m.floor_form = p->floor_form; m.fl_arho = p->floor_alpha_rho; m.fl_aeps = p->floor_alpha_eps;
  { const char* e = getenv("PHX_SMALL_1D"); M->small_1d = e ? atoi(e) != 0 : 1; }
  M->nall = (long long)m.nblk * m.ncell;
  M->ninterior = (long long)m.nblk * m.n[0] * m.n[1] * m.n[2];
  if (M->nall * m.nvar >= (1LL << 40)) { delete M; return fail(PHX_EINVAL, "phx_init_mesh: field too large"); }
  // launch geometry: blocks ride on gridDim.z, k-planes or sweep segments on gridDim.y (both limited to 65535)
  if (m.nblk > 65535 || m.na[2] > 65535 ||
      (long long)m.na[0] * m.na[1] >= (1LL << 31) || m.ncell >= (1LL << 31)) {
    delete M; return fail(PHX_EUNSUPPORTED, "phx_init_mesh: more than 65535 blocks or k-planes, or a k-plane of 2^31 cells");
  }
  const size_t fbytes = (size_t)M->nall * m.nvar * sizeof(double);
  cudaStream_t st = (cudaStream_t)stream;
  for (int d = 0; d < 3; ++d) {
    if (!m.act[d]) continue;
    cudaError_t e = cudaMalloc((void**)&M->flux[d], fbytes);
    if (e != cudaSuccess) { phx_free_mesh(M); return (e == cudaErrorMemoryAllocation) ? fail(PHX_ENOMEM, "phx_init_mesh: out of device memory (flux scratch)") : cuda_fail(e, "cudaMalloc"); }
    e = cudaMemsetAsync(M->flux[d], 0, fbytes, st);
    if (e != cudaSuccess) { phx_free_mesh(M); return cuda_fail(e, "cudaMemsetAsync"); }
  }
  {
    const size_t rbytes = (size_t)M->nall * (5 + p->nscalar) * sizeof(double);
    cudaError_t e = cudaMalloc((void**)&M->racc, rbytes);
    if (e != cudaSuccess) { phx_free_mesh(M); return (e == cudaErrorMemoryAllocation) ? fail(PHX_ENOMEM, "phx_init_mesh: out of device memory (divergence scratch)") : cuda_fail(e, "cudaMalloc"); }
    e = cudaMemsetAsync(M->racc, 0, rbytes, st);
    if (e != cudaSuccess) { phx_free_mesh(M); return cuda_fail(e, "cudaMemsetAsync"); }
  }
  {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) {
      cudaGetLastError(); phx_free_mesh(M); return fail(PHX_ECUDA, "phx_init_mesh: cannot query the SM count of the device");
    }
    M->nsm = nsm;
  }
  M->npartial = M->nsm * 8;
  if (cudaMalloc((void**)&M->partial, sizeof(double) * M->npartial) != cudaSuccess) { phx_free_mesh(M); return fail(PHX_ENOMEM, "phx_init_mesh: out of device memory"); }
  if (cudaMalloc((void**)&M->smax, sizeof(unsigned long long) * PHX_NSLOT) != cudaSuccess) { phx_free_mesh(M); return fail(PHX_ENOMEM, "phx_init_mesh: out of device memory"); }
  if (cudaMemsetAsync(M->smax, 0, sizeof(unsigned long long) * PHX_NSLOT, st) != cudaSuccess) { phx_free_mesh(M); return fail(PHX_ECUDA, "phx_init_mesh: cudaMemsetAsync failed"); }
  if (m.excise) {
    if (cudaMalloc((void**)&M->xfl, (size_t)M->nall) != cudaSuccess) { phx_free_mesh(M); return fail(PHX_ENOMEM, "phx_init_mesh: out of device memory"); }
    k_excision_flags<<<(unsigned)((M->nall + 255) / 256), 256, 0, st>>>(m, M->xfl, M->nall);
    M->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { phx_free_mesh(M); return cuda_fail(e, "k_excision_flags"); }
  }
  *out = M;
  return PHX_OK;
}

extern "C" int phx_free_mesh(phx_mesh* M) {
  if (!M) return PHX_OK;
  for (int d = 0; d < 3; ++d) if (M->flux[d]) cudaFree(M->flux[d]);
  if (M->racc) cudaFree(M->racc);
  if (M->xfl) cudaFree(M->xfl);
  if (M->partial) cudaFree(M->partial);
  if (M->smax) cudaFree(M->smax);
  for (int d = 0; d < 3; ++d) if (M->ws_field[d]) cudaFree(M->ws_field[d]);
  if (M->ws_mask) cudaFree(M->ws_mask);
  if (M->ws_scal) cudaFree(M->ws_scal);
  if (M->ev) { for (int i = 0; i < 2 * M->evcap; ++i) cudaEventDestroy(M->ev[i]); delete[] M->ev; delete[] M->evcls; }
  if (M->gexec) cudaGraphExecDestroy(M->gexec);
  if (M->gev_in) cudaEventDestroy(M->gev_in);
  if (M->gev_out) cudaEventDestroy(M->gev_out);
  if (M->gstream) cudaStreamDestroy(M->gstream);
  delete M;
  return PHX_OK;
}

extern "C" size_t phx_field_elems(const phx_mesh* M) { return M ? (size_t)M->nall * M->m.nvar : 0; }
extern "C" size_t phx_mask_elems(const phx_mesh* M) { return M ? (size_t)M->nall : 0; }
extern "C" unsigned long long phx_launch_count(const phx_mesh* M) { return M ? M->launches : 0; }
extern "C" int phx_debug_enable_flux(phx_mesh* M, int on) {
  if (!M) return fail(PHX_EINVAL, "phx_debug_enable_flux: null mesh");
  const int v = on ? 1 : 0;
  if (v != M->store_all_fluxes && M->gexec) { cudaGraphExecDestroy(M->gexec); M->gexec = nullptr; }   // the flag is baked into the captured launches
  M->store_all_fluxes = v;
  return PHX_OK;
}

extern "C" int phx_debug_flux(const phx_mesh* M, int d, double* d_out, void* stream) {
  if (!M || d < 0 || d > 2 || !M->flux[d] || !aligned16(d_out)) return fail(PHX_EINVAL, "phx_debug_flux: null argument or inactive direction");
  CUDA_TRY(cudaMemcpyAsync(d_out, M->flux[d], (size_t)M->nall * M->m.nvar * sizeof(double), cudaMemcpyDeviceToDevice, (cudaStream_t)stream), "cudaMemcpyAsync");
  return PHX_OK;
}

// PHX_BUILD_SUBSET (development only): instantiate the flat-metric WENO5-Z / PLM and the Kerr-Schild PLM kernels alone, for quick A/B builds
#ifdef PHX_BUILD_SUBSET
#define DISPATCH_METRIC(mesh, CALL) do { if ((mesh)->m.metric == 1) { CALL(1); } else { CALL(0); } } while (0)
#else
#define DISPATCH_METRIC(mesh, CALL)                 \
  do {                                              \
    if ((mesh)->m.metric == 0) { CALL(0); }         \
    else if ((mesh)->m.metric == 1) { CALL(1); }    \
    else { CALL(2); }                               \
  } while (0)
#endif

extern "C" int phx_prim_to_cons(const phx_mesh* M, const double* d_prim, double* d_cons, void* stream) {
  if (!M || !aligned16(d_prim) || !aligned16(d_cons)) return fail(PHX_EINVAL, "phx_prim_to_cons: null or misaligned argument");
  cudaStream_t st = (cudaStream_t)stream;
  const unsigned nb = (unsigned)((M->nall + 255) / 256);
  {
  ProfScope ps(M, PHX_K_PRIM_TO_CONS, st);
#define CALL(MET) k_prim_to_cons<MET><<<nb, 256, 0, st>>>(M->m, d_prim, d_cons, M->nall)
  DISPATCH_METRIC(M, CALL);
#undef CALL
  }
  LAUNCH_CHECK(M, "k_prim_to_cons");
  return PHX_OK;
}

// depth < 0: the whole frame; otherwise the layers a stage of this mesh's reconstruction reads (half-width + 1, at most g)
static int fill_ghosts_impl(const phx_mesh* M, double* d_prim, int depth, cudaStream_t st) {
  if (M->nall == M->ninterior) return PHX_OK;
  { ProfScope ps(M, PHX_K_FILL_GHOSTS, st);
    const MeshDev& m = M->m;
    GhostShell gs;
    for (int d = 0; d < 3; ++d) gs.dep[d] = (depth < 0 || depth > m.g[d]) ? m.g[d] : depth;
    gs.dep[0] = m.g[0];      // along x always the whole depth: a thinner shell would write partial 32-byte sectors (measured: no gain)
    // two cells per thread where every run of ghost cells along x is even and 16-byte aligned (field strides: ncell, sk, sj even)
    const int vec = (m.act[0] && m.n[0] % 2 == 0 && m.g[0] % 2 == 0 && gs.dep[0] % 2 == 0) ? 2 : 1;
    const long long w0 = (m.n[0] + 2 * gs.dep[0]) / vec, w1 = m.n[1] + 2 * gs.dep[1];
    const long long nA = 2LL * gs.dep[2] * w1 * w0, nB = 2LL * m.n[2] * gs.dep[1] * w0, nC = 2LL * m.n[2] * m.n[1] * gs.dep[0] / vec;
    gs.nA = (int)nA; gs.nB = (int)nB; gs.ntot = (int)(nA + nB + nC);
    const dim3 grid((unsigned)((nA + nB + nC + 255) / 256), 1, m.nblk);
    if (vec == 2) k_fill_ghosts<2><<<grid, 256, 0, st>>>(m, d_prim, gs);
    else k_fill_ghosts<1><<<grid, 256, 0, st>>>(m, d_prim, gs); }
  LAUNCH_CHECK(M, "k_fill_ghosts");
  return PHX_OK;
}

extern "C" int phx_fill_ghosts(const phx_mesh* M, double* d_prim, void* stream) {
  if (!M || !aligned16(d_prim)) return fail(PHX_EINVAL, "phx_fill_ghosts: null or misaligned argument");
  return fill_ghosts_impl(M, d_prim, -1, (cudaStream_t)stream);
}

extern "C" int phx_cons_to_prim(const phx_mesh* M, double* d_cons, double* d_prim, unsigned char* d_mask, void* stream) {
  if (!M || !aligned16(d_cons) || !aligned16(d_prim) || !d_mask) return fail(PHX_EINVAL, "phx_cons_to_prim: null or misaligned argument");
  cudaStream_t st = (cudaStream_t)stream;
  const unsigned nb = (unsigned)((M->ninterior + UP_BLOCK - 1) / UP_BLOCK);
  {
  ProfScope ps(M, PHX_K_C2P, st);
#define C2P(MET, EXC, NSC, RFL) k_c2p<MET, EXC, NSC, RFL><<<nb, UP_BLOCK, 0, st>>>(M->m, M->xfl, d_cons, d_prim, d_mask, M->ninterior)
#define CALL(MET)                                                      \
  if (M->m.nvar == NV) {                                               \
    if (M->m.floor_form == 0) { if (M->m.excise) C2P(MET, true, 0, false); else C2P(MET, false, 0, false); } \
    else { if (M->m.excise) C2P(MET, true, 0, true); else C2P(MET, false, 0, true); }                        \
  } else {                                                             \
    if (M->m.floor_form == 0) { if (M->m.excise) C2P(MET, true, 1, false); else C2P(MET, false, 1, false); } \
    else { if (M->m.excise) C2P(MET, true, 1, true); else C2P(MET, false, 1, true); }                        \
  }
  DISPATCH_METRIC(M, CALL);
#undef CALL
#undef C2P
  }
  LAUNCH_CHECK(M, "k_c2p");
  return phx_fill_ghosts(M, d_prim, stream);
}

// ---- sweeps -------------------------------------------------------------------------------------------------
template <int METRIC, int RECON, int NS>
static void launch_sweeps_t(phx_mesh* M, const double* prim, cudaStream_t st) {
  const MeshDev& m = M->m;
  int lo[3], cnt[3];
  for (int d = 0; d < 3; ++d) {
    lo[d] = m.act[d] ? m.g[d] - 1 : 0;
    cnt[d] = m.act[d] ? m.n[d] + 2 : 1;
  }
  if (m.act[0]) {
    const int rowlen = m.n[0] + 2;
    const int nplane = cnt[1] * rowlen;
    dim3 grid((nplane - 1 + (XS_BLOCK - 3)) / (XS_BLOCK - 2), cnt[2], m.nblk);   // every position >= 1 is some block's thread 1..XS_BLOCK-2
    ProfScope ps(M, PHX_K_SWEEP_X, st);
    k_sweep_x<METRIC, RECON, NS><<<grid, XS_BLOCK, 0, st>>>(m, prim, M->flux[0], M->racc, M->store_all_fluxes, nplane, rowlen, lo[1], lo[2]);
    M->launches++;
  }
  // Segments of at most 33 faces along the sweep direction; a small mesh gets more, shorter segments (at least 4 faces)
  // until the launch has about four waves of thread blocks, so that the marching sweeps do not starve for parallelism
  // (64^3: 2 segments = 0.9 blocks per SM -> 17 segments).  The fluxes do not depend on the segmentation.
  auto segments = [&](int ncells, int ntr) {
    const int nfaces = ncells;
    int nseg = (nfaces + 32) / 33;
    const long long per_seg = (long long)((ntr + MS_BLOCK - 1) / MS_BLOCK) * m.nblk;
    const long long want = (long long)M->nsm * PHX_MS_MINB * 4;
    const int need = (int)((want + per_seg - 1) / per_seg);
    const int cap = (nfaces + 3) / 4;
    if (need > nseg) nseg = need < cap ? need : cap;
    return nseg < 1 ? 1 : nseg;
  };
  if (m.act[1]) {
    const int ncells = m.n[1];
    const int ntr = cnt[0] * cnt[2];
    const int nseg = segments(ncells, ntr);
    const int L = (ncells + nseg - 1) / nseg;
    dim3 grid((ntr + MS_BLOCK - 1) / MS_BLOCK, nseg, m.nblk);
    ProfScope ps(M, PHX_K_SWEEP_Y, st);
    k_sweep_march<METRIC, RECON, 1, NS><<<grid, MS_BLOCK, 0, st>>>(m, prim, M->flux[1], M->racc, M->store_all_fluxes, m.act[0] ? 0 : 1, ntr, cnt[0], lo[0], lo[2], L);
    M->launches++;
  }
  if (m.act[2]) {
    const int ncells = m.n[2];
    const int ntr = cnt[0] * cnt[1];
    const int nseg = segments(ncells, ntr);
    const int L = (ncells + nseg - 1) / nseg;
    dim3 grid((ntr + MS_BLOCK - 1) / MS_BLOCK, nseg, m.nblk);
    ProfScope ps(M, PHX_K_SWEEP_Z, st);
    k_sweep_march<METRIC, RECON, 2, NS><<<grid, MS_BLOCK, 0, st>>>(m, prim, M->flux[2], M->racc, M->store_all_fluxes, (m.act[0] || m.act[1]) ? 0 : 1, ntr, cnt[0], lo[0], lo[1], L);
    M->launches++;
  }
}

static void launch_sweeps(phx_mesh* M, const double* prim, cudaStream_t st) {
  const int key = M->m.metric * 6 + M->m.recon;
  switch (key) {
#define PHX_CASE(MET, REC) case MET * 6 + REC: if (M->m.nvar == NV) launch_sweeps_t<MET, REC, 0>(M, prim, st); else launch_sweeps_t<MET, REC, 1>(M, prim, st); break;
#ifdef PHX_BUILD_SUBSET
    PHX_CASE(0, 1) PHX_CASE(0, 3) PHX_CASE(1, 1)
#else
    PHX_CASE(0, 0) PHX_CASE(0, 1) PHX_CASE(0, 2) PHX_CASE(0, 3) PHX_CASE(0, 4) PHX_CASE(0, 5)
    PHX_CASE(1, 0) PHX_CASE(1, 1) PHX_CASE(1, 2) PHX_CASE(1, 3) PHX_CASE(1, 4) PHX_CASE(1, 5)
    PHX_CASE(2, 0) PHX_CASE(2, 1) PHX_CASE(2, 2) PHX_CASE(2, 3) PHX_CASE(2, 4) PHX_CASE(2, 5)
#endif
#undef PHX_CASE
    default: break;
  }
}

static int stage_impl(phx_mesh* M, double g0, double g1, double bdt_host, const double* d_dt, double beta, const double* d_cons0,
                      const double* d_cons_in, double* d_cons_out, double* d_prim, unsigned char* d_mask, cudaStream_t st,
                      bool reduce_cfl = false, bool inner_stage = false) {
  launch_sweeps(M, d_prim, st);
  { cudaError_t e = cudaGetLastError(); if (e != cudaSuccess) return cuda_fail(e, "flux sweep"); }
  FluxPtrs fl;
  for (int d = 0; d < 3; ++d) fl.f[d] = M->flux[d];
  fl.racc = M->racc;
  const dim3 nb((M->m.n[0] * M->m.n[1] + UP_BLOCK - 1) / UP_BLOCK, M->m.n[2], M->m.nblk);
  {
  ProfScope ps(M, PHX_K_UPDATE, st);
#define UPD(MET, EXC, CFLR, NSC, RFL) k_update<MET, EXC, CFLR, NSC, RFL><<<nb, UP_BLOCK, 0, st>>>(M->m, fl, M->xfl, g0, g1, bdt_host, d_dt, beta, d_cons0, d_cons_in, d_cons_out, d_prim, d_mask, M->smax)
#define UPD2(MET, NSC, RFL)                                                                                  \
  if (M->m.excise) { if (reduce_cfl) UPD(MET, true, true, NSC, RFL); else UPD(MET, true, false, NSC, RFL); } \
  else { if (reduce_cfl) UPD(MET, false, true, NSC, RFL); else UPD(MET, false, false, NSC, RFL); }
#define CALL(MET)                                                                    \
  if (M->m.nvar == NV) { if (M->m.floor_form == 0) { UPD2(MET, 0, false) } else { UPD2(MET, 0, true) } } \
  else { if (M->m.floor_form == 0) { UPD2(MET, 1, false) } else { UPD2(MET, 1, true) } }
  DISPATCH_METRIC(M, CALL);
#undef CALL
#undef UPD2
#undef UPD
  }
  LAUNCH_CHECK(M, "k_update");
  // a stage whose primitives only the next stage of the same call reads fills the ghost layers that stage's sweeps touch
  // (stencil half-width + 1); the last stage of a call leaves the whole frame filled, as the header promises
  const int hw = (M->m.recon == 0) ? 0 : (M->m.recon >= 3 ? 2 : 1);
  return fill_ghosts_impl(M, d_prim, inner_stage ? hw + 1 : -1, st);
}

extern "C" int phx_rk_stage(phx_mesh* M, double g0, double g1, double beta_dt, const double* d_cons0, double* d_cons, double* d_prim,
                            unsigned char* d_mask, void* stream) {
  if (!M || !aligned16(d_cons0) || !aligned16(d_cons) || !aligned16(d_prim) || !d_mask)
    return fail(PHX_EINVAL, "phx_rk_stage: null or misaligned argument");
  return stage_impl(M, g0, g1, beta_dt, nullptr, 0.0, d_cons0, d_cons, d_cons, d_prim, d_mask, (cudaStream_t)stream);
}

extern "C" int phx_rk2_step(phx_mesh* M, const double* d_dt, double* d_cons0, double* d_cons, double* d_prim, unsigned char* d_mask,
                            void* stream) {
  if (!M || !d_dt || !aligned16(d_cons0) || !aligned16(d_cons) || !aligned16(d_prim) || !d_mask || d_cons0 == d_cons)
    return fail(PHX_EINVAL, "phx_rk2_step: null, misaligned or aliased argument");
  cudaStream_t st = (cudaStream_t)stream;
  // no copy of U~0: stage 1 reads U~0 = d_cons and writes U~1 into the scratch field; stage 2 combines both into d_cons
  int rc = stage_impl(M, 1.0, 0.0, 0.0, d_dt, 1.0, d_cons, d_cons, d_cons0, d_prim, d_mask, st, false, true);
  if (rc != PHX_OK) return rc;
  return stage_impl(M, 0.5, 0.5, 0.0, d_dt, 0.5, d_cons, d_cons0, d_cons, d_prim, d_mask, st);
}

extern "C" int phx_rk2_step_cfl(phx_mesh* M, double cfl, double* d_dt, double* d_cons0, double* d_cons, double* d_prim,
                                unsigned char* d_mask, void* stream) {
  if (!M || !d_dt || !(cfl > 0.0) || !aligned16(d_cons0) || !aligned16(d_cons) || !aligned16(d_prim) || !d_mask || d_cons0 == d_cons)
    return fail(PHX_EINVAL, "phx_rk2_step_cfl: null, misaligned or aliased argument, or cfl <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  int rc = stage_impl(M, 1.0, 0.0, 0.0, d_dt, 1.0, d_cons, d_cons, d_cons0, d_prim, d_mask, st, false, true);
  if (rc != PHX_OK) return rc;
  // stage 2 also reduces max sum_d |lambda^d|/dx_d of the new primitives; the final kernel overwrites *d_dt after every
  // block of stage 2 has read it (stream order)
  rc = stage_impl(M, 0.5, 0.5, 0.0, d_dt, 0.5, d_cons, d_cons0, d_cons, d_prim, d_mask, st, true);
  if (rc != PHX_OK) return rc;
  { ProfScope ps(M, PHX_K_CFL, st);
    k_cfl_final_slots<<<1, 256, 0, st>>>(M->smax, cfl, d_dt); }
  LAUNCH_CHECK(M, "k_cfl_final_slots");
  return PHX_OK;
}

extern "C" int phx_cfl_dt(const phx_mesh* M, const double* d_prim, double cfl, double* d_dt, double* h_dt, void* stream) {
  if (!M || !aligned16(d_prim) || !d_dt || !(cfl > 0.0)) return fail(PHX_EINVAL, "phx_cfl_dt: null or misaligned argument, or cfl <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  long long want = (M->ninterior + 255) / 256;
  const int nb = (int)(want < M->npartial ? want : M->npartial);
  {
  ProfScope ps(M, PHX_K_CFL, st);
#define CALL(MET)                                                                                          \
  if (M->m.excise) k_cfl_partial<MET, true><<<nb, 256, 0, st>>>(M->m, M->xfl, d_prim, M->partial, M->ninterior); \
  else k_cfl_partial<MET, false><<<nb, 256, 0, st>>>(M->m, M->xfl, d_prim, M->partial, M->ninterior)
  DISPATCH_METRIC(M, CALL);
#undef CALL
  LAUNCH_CHECK(M, "k_cfl_partial");
  k_cfl_final<<<1, 256, 0, st>>>(M->partial, nb, cfl, d_dt);
  LAUNCH_CHECK(M, "k_cfl_final");
  }
  if (h_dt) {
    CUDA_TRY(cudaMemcpyAsync(h_dt, d_dt, sizeof(double), cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync");
    CUDA_TRY(cudaStreamSynchronize(st), "cudaStreamSynchronize");
  }
  return PHX_OK;
}

// ---- failure detection: how many interior cells carry any of the given mask bits ------------------------------------------
__global__ void __launch_bounds__(256) k_count_masked(MeshDev m, const unsigned char* __restrict__ mask, unsigned bits,
                                                      unsigned long long* __restrict__ count, long long ninterior) {
  unsigned n = 0;
  for (long long p = (long long)blockIdx.x * 256 + threadIdx.x; p < ninterior; p += (long long)gridDim.x * 256) {
    const int ii = (int)(p % m.n[0]);
    long long r = p / m.n[0];
    const int jj = (int)(r % m.n[1]); r /= m.n[1];
    const int kk = (int)(r % m.n[2]);
    const int b = (int)(r / m.n[2]);
    const long long c = (long long)b * m.ncell + (long long)(kk + m.g[2]) * m.sk + (long long)(jj + m.g[1]) * m.sj + (ii + m.g[0]);
    n += (mask[c] & bits) != 0;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
  if ((threadIdx.x & 31) == 0 && n) atomicAdd(count, (unsigned long long)n);
}

extern "C" int phx_count_masked(const phx_mesh* M, const unsigned char* d_mask, unsigned bits, unsigned long long* d_count,
                                unsigned long long* h_count, void* stream) {
  if (!M || !d_mask || !d_count) return fail(PHX_EINVAL, "phx_count_masked: null argument");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), st), "cudaMemsetAsync");
  long long want = (M->ninterior + 255) / 256;
  const int nb = (int)(want < (long long)M->nsm * 8 ? want : (long long)M->nsm * 8);
  k_count_masked<<<nb, 256, 0, st>>>(M->m, d_mask, bits, d_count, M->ninterior);
  LAUNCH_CHECK(M, "k_count_masked");
  if (h_count) {
    CUDA_TRY(cudaMemcpyAsync(h_count, d_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync");
    CUDA_TRY(cudaStreamSynchronize(st), "cudaStreamSynchronize");
  }
  return PHX_OK;
}

// ---- per-kernel-class event timing ------------------------------------------------------------------------------
extern "C" int phx_profile_enable(phx_mesh* M, int max_records) {
  if (!M || max_records < 0) return fail(PHX_EINVAL, "phx_profile_enable: null mesh or negative capacity");
  if (M->ev) { for (int i = 0; i < 2 * M->evcap; ++i) cudaEventDestroy(M->ev[i]); delete[] M->ev; delete[] M->evcls; M->ev = nullptr; M->evcls = nullptr; }
  M->evcap = M->evn = 0;
  if (max_records == 0) return PHX_OK;
  M->ev = new (std::nothrow) cudaEvent_t[2 * (size_t)max_records];
  M->evcls = new (std::nothrow) int[max_records];
  if (!M->ev || !M->evcls) { delete[] M->ev; delete[] M->evcls; M->ev = nullptr; M->evcls = nullptr; return fail(PHX_ENOMEM, "phx_profile_enable: host allocation failed"); }
  for (int i = 0; i < 2 * max_records; ++i) CUDA_TRY(cudaEventCreate(&M->ev[i]), "cudaEventCreate");
  M->evcap = max_records;
  return PHX_OK;
}

extern "C" int phx_profile_read(phx_mesh* M, double* h_ms, unsigned long long* h_count) {
  if (!M || !h_ms || !h_count) return fail(PHX_EINVAL, "phx_profile_read: null argument");
  for (int c = 0; c < PHX_K_COUNT; ++c) { h_ms[c] = 0.0; h_count[c] = 0; }
  for (int i = 0; i < M->evn; ++i) {
    CUDA_TRY(cudaEventSynchronize(M->ev[2 * i + 1]), "cudaEventSynchronize");
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, M->ev[2 * i], M->ev[2 * i + 1]), "cudaEventElapsedTime");
    h_ms[M->evcls[i]] += ms;
    h_count[M->evcls[i]]++;
  }
  M->evn = 0;
  return PHX_OK;
}

// ---- fp64 pipe peak: a DFMA loop on every SM (bench.py's ALU roofline denominator, measured in the same run) ---------------
// 8 independent fused multiply-add chains per thread, 64 warps per SM: nothing but the fp64 pipe limits it.
__global__ void __launch_bounds__(256) k_fp64_peak(double* __restrict__ sink, long long iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = 1.0 + 1e-3 * k + 1e-9 * threadIdx.x;
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fma(x[k], a, b);
    }
  }
  double t = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) t += x[k];
  if (t == 123456.789) sink[0] = t;      // never true: keeps the chains alive
}

extern "C" int phx_debug_fp64_peak(double min_seconds, double* h_dfma_per_s, double* h_dfma_per_s_burst, double* h_ms, int* h_nsm, void* stream) {
  if (!(min_seconds > 0.0) || min_seconds > 10.0 || !h_dfma_per_s) return fail(PHX_EINVAL, "phx_debug_fp64_peak: min_seconds in (0, 10] and a result pointer required");
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, nsm = 0;
  CUDA_TRY(cudaGetDevice(&dev), "cudaGetDevice");
  CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute");
  double* sink = nullptr;
  CUDA_TRY(cudaMalloc((void**)&sink, sizeof(double)), "cudaMalloc");
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int nblk = nsm * 8;
  const double per_iter = (double)nblk * 256.0 * 32.0;          // DFMA thread-instructions per loop iteration
  long long iters = 1 << 14;
  float ms = 0.f;
  cudaError_t e = cudaSuccess;
  for (int pass = 0; pass < 3 && e == cudaSuccess; ++pass) {    // warm-up / calibration, then the timed launch
    cudaEventRecord(e0, st);
    k_fp64_peak<<<nblk, 256, 0, st>>>(sink, iters, 0.999999, 1e-6);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (pass == 2 || e != cudaSuccess) break;
    const double rate = per_iter * (double)iters / (ms * 1e-3);
    if (pass == 1 && h_dfma_per_s_burst) *h_dfma_per_s_burst = rate;   // the short second launch: before any power cap acts
    iters = (long long)(min_seconds * rate / per_iter * (pass == 0 ? 0.05 : 1.0)) + 1;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
  if (e != cudaSuccess) return cuda_fail(e, "k_fp64_peak");
  *h_dfma_per_s = per_iter * (double)iters / (ms * 1e-3);
  if (h_ms) *h_ms = ms;
  if (h_nsm) *h_nsm = nsm;
  return PHX_OK;
}

// ---- small one-dimensional meshes: the whole run in ONE thread block ---------------------------------------------------
// A 1-D mesh of a few hundred zones (BASELINE.json config 1: 256 zones) is pure launch latency on the general path: 8 kernels
// of 2-3 us per step.  Here one thread block owns the mesh (one thread per cell, the two ghost-adjacent cells included) and
// loops over `nsteps` RK2 steps on the device: per stage reconstruct + Riemann flux with the face states and fluxes exchanged
// through shared memory, divergence, RK combination, con2prim + floors, ghost cells, and after the second stage the block-wide
// maximum of the signal speeds gives the next time step.  Barriers are __syncthreads; nothing leaves the SM between stages
// but the few KB of state in L1 / L2.  Same device functions and the same expressions as k_sweep_x / update_cell (flat
// metric, no passive scalar, constant floors, no excision): the results are the bits of the general path.
constexpr int SM1_MAXT = 512;
template <int RECON>
__global__ void __launch_bounds__(SM1_MAXT, 1) k_evolve_1d(MeshDev m, int nsteps, double cfl, double* __restrict__ d_dt, double* __restrict__ d_t,
                                                          double* __restrict__ cons0, double* __restrict__ cons, double* __restrict__ prim,
                                                          unsigned char* __restrict__ mask) {
  constexpr int HW = ReconTraits<RECON>::HW;
  extern __shared__ double smem1[];
  const int T = blockDim.x;
  double (*sh)[SM1_MAXT] = reinterpret_cast<double (*)[SM1_MAXT]>(smem1);                  // upper-face states, NV rows
  double (*shF)[SM1_MAXT] = reinterpret_cast<double (*)[SM1_MAXT]>(smem1 + NV * SM1_MAXT);   // face fluxes, NV rows
  __shared__ double red[SM1_MAXT / 32];
  __shared__ double dt_sh;
  const int t = threadIdx.x;
  const int n = m.n[0], g = m.g[0];
  const bool valid = t < n + 2;                    // cell i = g - 1 + t
  const int i = g - 1 + t;
  const bool interior = t >= 1 && t <= n;
  (void)T;
  for (int step = 0; step < nsteps; ++step) {
    if (t == 0) { dt_sh = *d_dt; if (d_t) *d_t += dt_sh; }
    __syncthreads();
    const double dt = dt_sh;
    double speed = 0.0;
    for (int stage = 0; stage < 2; ++stage) {
      // stage 1: U~1 = U~0 + dt R -> cons0 (scratch); stage 2: U~ = (U~0 + U~1)/2 + dt/2 R -> cons   (phx_rk2_step)
      const double g0 = stage == 0 ? 1.0 : 0.5, g1 = stage == 0 ? 0.0 : 0.5;
      const double bdt = (stage == 0 ? 1.0 : 0.5) * dt;
      const double* c0 = cons;
      const double* cin = stage == 0 ? cons : cons0;
      double* cout = stage == 0 ? cons0 : cons;
      double qm[NV], qp[NV], F[NV];
      if (valid) {
        double centre[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          double f[2 * HW + 1];
#pragma unroll
          for (int s = 0; s <= 2 * HW; ++s) f[s] = prim[v * m.ncell + i + (s - HW)];
          centre[v] = f[HW];
          recon1<RECON>(f, qm[v], qp[v]);
        }
        positivity_fallback<0, RECON, 0>(m, 0.0, 0.0, 0.0, centre, qm, qp);
#pragma unroll
        for (int v = 0; v < NV; ++v) sh[v][t] = qp[v];
      }
      __syncthreads();
      const bool face = valid && t > 0;            // face (i - 1/2)
      if (face) {
        double qL[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) qL[v] = sh[v][t - 1];
        Geo<0> G;
        face_flux<0, 0, 0>(m, G, qL, qm, F);
#pragma unroll
        for (int v = 0; v < NV; ++v) shF[v][t] = F[v];
      }
      __syncthreads();
      if (interior) {
        double R[NV], U[NV], q[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) R[v] = 0.0 - (shF[v][t + 1] - F[v]) * m.rdx[0];
        R[BX] = 0.0;                               // F~^x[B^x] = 0: the update leaves B^x alone in 1-D
        q[RHO] = prim[RHO * m.ncell + i];
        q[UX] = prim[UX * m.ncell + i]; q[UY] = prim[UY * m.ncell + i]; q[UZ] = prim[UZ * m.ncell + i];
        q[UU] = prim[UU * m.ncell + i];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const long long id = v * m.ncell + i;
          U[v] = (g1 != 0.0) ? g0 * c0[id] + g1 * cin[id] + bdt * R[v] : g0 * c0[id] + bdt * R[v];
        }
        Geo<0> G;
        const double mu_guess = c2p_guess<0>(G, q, m.gam);
        unsigned mk = c2p_cell<0>(m, G, m.rho_floor, m.eps_floor, U, q, mu_guess);
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const long long id = v * m.ncell + i;
          cout[id] = U[v];
          prim[id] = q[v];
        }
        mask[i] = (unsigned char)mk;
        if (stage == 1) {
          double lam[3];
          max_speeds<0>(q, G, m.gam, lam);
          speed = cfl_guard(lam[0] * m.rdx[0]);
        }
      }
      __syncthreads();
      // ghost cells: periodic wrap or zero-gradient copy (k_fill_ghosts in one dimension)
      if (t < 2 * g) {
        const int l = t < g ? t : t + n;           // allocated index of the ghost cell
        int li = l - g;
        if (li < 0) li = (m.bc[0][0] == 0) ? li + n : 0;
        else li = (m.bc[0][1] == 0) ? li - n : n - 1;
#pragma unroll
        for (int v = 0; v < NV; ++v) prim[v * m.ncell + l] = prim[v * m.ncell + li + g];
      }
      __syncthreads();
    }
    // next time step: cfl / max over the cells of |lambda|/dx
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
    if ((t & 31) == 0) red[t >> 5] = speed;
    __syncthreads();
    if (t == 0) {
      double v = red[0];
      for (int w = 1; w < (blockDim.x + 31) / 32; ++w) v = fmax(v, red[w]);
      *d_dt = cfl_dt_of(cfl, v);
    }
    __syncthreads();
  }
}

// the single-block path applies to: one block, x the only active direction, flat metric without shift, no passive scalar,
// constant floors, a mesh that fits one thread block
static bool small_1d_eligible(const phx_mesh* M) {
  const MeshDev& m = M->m;
  return m.nblk == 1 && m.act[0] && !m.act[1] && !m.act[2] && m.metric == 0 && m.nvar == NV && m.floor_form == 0 && !m.excise &&
         m.n[0] + 2 <= SM1_MAXT && 2 * m.g[0] <= ((m.n[0] + 2 + 31) / 32) * 32 &&   // one thread per cell, and per ghost cell in the fill
         !M->store_all_fluxes && M->small_1d;
}

static int launch_evolve_1d(phx_mesh* M, int nsteps, double cfl, double* d_dt, double* d_t, double* d_cons0, double* d_cons, double* d_prim,
                            unsigned char* d_mask, cudaStream_t st) {
  const MeshDev& m = M->m;
  const int threads = ((m.n[0] + 2 + 31) / 32) * 32;
  const size_t smem = 2 * NV * SM1_MAXT * sizeof(double);
  // 128 KB of dynamic shared memory need the opt-in of the kernel attribute (per device and context: set on every call)
#define EV1(REC) case REC: \
    CUDA_TRY(cudaFuncSetAttribute(k_evolve_1d<REC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "cudaFuncSetAttribute"); \
    k_evolve_1d<REC><<<1, threads, smem, st>>>(m, nsteps, cfl, d_dt, d_t, d_cons0, d_cons, d_prim, d_mask); break;
  switch (m.recon) {
    EV1(0) EV1(1) EV1(2) EV1(3) EV1(4) EV1(5)
    default: return fail(PHX_EUNSUPPORTED, "k_evolve_1d: unknown reconstruction");
  }
#undef EV1
  LAUNCH_CHECK(M, "k_evolve_1d");
  return PHX_OK;
}

// ---- host-buffer path ------------------------------------------------------------------------------------------
__global__ void k_accumulate_time(double* __restrict__ t, const double* __restrict__ dt) { *t += *dt; }

// One step of phx_evolve_device: t += dt (before the step replaces dt), then phx_rk2_step_cfl.
static int evolve_one(phx_mesh* M, double cfl, double* d_dt, double* d_t, double* d_cons0, double* d_cons, double* d_prim,
                      unsigned char* d_mask, cudaStream_t st) {
  if (d_t) {
    k_accumulate_time<<<1, 1, 0, st>>>(d_t, d_dt);
    LAUNCH_CHECK(M, "k_accumulate_time");
  }
  return phx_rk2_step_cfl(M, cfl, d_dt, d_cons0, d_cons, d_prim, d_mask, st);
}

extern "C" int phx_evolve_device(phx_mesh* M, int nsteps, double cfl, double* d_dt, double* d_t, double* d_cons0, double* d_cons,
                                 double* d_prim, unsigned char* d_mask, void* stream) {
  if (!M || nsteps < 0 || !d_dt || !(cfl > 0.0) || !aligned16(d_cons0) || !aligned16(d_cons) || !aligned16(d_prim) || !d_mask || d_cons0 == d_cons)
    return fail(PHX_EINVAL, "phx_evolve_device: null, misaligned or aliased argument, nsteps < 0 or cfl <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  if (nsteps == 0) return PHX_OK;
  // a small 1-D mesh runs all its steps in one launch of one thread block (no per-kernel timing there: one kernel)
  if (!M->ev && small_1d_eligible(M)) return launch_evolve_1d(M, nsteps, cfl, d_dt, d_t, d_cons0, d_cons, d_prim, d_mask, st);
  // per-kernel timing records events around every launch, which a replayed graph cannot serve: launch directly then
  if (M->ev || nsteps < 2) {
    for (int s = 0; s < nsteps; ++s) {
      const int rc = evolve_one(M, cfl, d_dt, d_t, d_cons0, d_cons, d_prim, d_mask, st);
      if (rc != PHX_OK) return rc;
    }
    return PHX_OK;
  }
  if (!M->gstream) {
    CUDA_TRY(cudaStreamCreateWithFlags(&M->gstream, cudaStreamNonBlocking), "cudaStreamCreateWithFlags");
    CUDA_TRY(cudaEventCreateWithFlags(&M->gev_in, cudaEventDisableTiming), "cudaEventCreateWithFlags");
    CUDA_TRY(cudaEventCreateWithFlags(&M->gev_out, cudaEventDisableTiming), "cudaEventCreateWithFlags");
  }
  const bool same = M->gexec && M->gkey.cfl == cfl && M->gkey.dt == d_dt && M->gkey.t == d_t && M->gkey.cons0 == d_cons0 &&
                    M->gkey.cons == d_cons && M->gkey.prim == d_prim && M->gkey.mask == d_mask;
  if (!same) {
    if (M->gexec) { cudaGraphExecDestroy(M->gexec); M->gexec = nullptr; }
    // capture on the mesh-owned stream (the caller's may be the legacy default stream, which cannot be captured)
    const unsigned long long before = M->launches;
    CUDA_TRY(cudaStreamBeginCapture(M->gstream, cudaStreamCaptureModeThreadLocal), "cudaStreamBeginCapture");
    const int rc = evolve_one(M, cfl, d_dt, d_t, d_cons0, d_cons, d_prim, d_mask, M->gstream);
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(M->gstream, &graph);
    M->glaunches = M->launches - before;
    M->launches = before;                              // nothing ran during the capture
    if (rc != PHX_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
    const cudaError_t ei = cudaGraphInstantiate(&M->gexec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess) { M->gexec = nullptr; return cuda_fail(ei, "cudaGraphInstantiate"); }
    M->gkey.cfl = cfl; M->gkey.dt = d_dt; M->gkey.t = d_t; M->gkey.cons0 = d_cons0; M->gkey.cons = d_cons; M->gkey.prim = d_prim;
    M->gkey.mask = d_mask;
  }
  // fence the mesh-owned stream behind the caller's stream, replay, fence the caller's stream behind the replays
  CUDA_TRY(cudaEventRecord(M->gev_in, st), "cudaEventRecord");
  CUDA_TRY(cudaStreamWaitEvent(M->gstream, M->gev_in, 0), "cudaStreamWaitEvent");
  for (int s = 0; s < nsteps; ++s) CUDA_TRY(cudaGraphLaunch(M->gexec, M->gstream), "cudaGraphLaunch");
  M->launches += M->glaunches * (unsigned long long)nsteps;
  CUDA_TRY(cudaEventRecord(M->gev_out, M->gstream), "cudaEventRecord");
  CUDA_TRY(cudaStreamWaitEvent(st, M->gev_out, 0), "cudaStreamWaitEvent");
  return PHX_OK;
}

extern "C" int phx_evolve_host(phx_mesh* M, const double* h_prim_in, int nsteps, double cfl, double* h_prim_out, double* h_cons_out,
                               unsigned char* h_mask_out, double* h_t, void* stream) {
  if (!M || !h_prim_in || !h_prim_out || nsteps < 0 || !(cfl > 0.0)) return fail(PHX_EINVAL, "phx_evolve_host: null argument, nsteps < 0 or cfl <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t fbytes = (size_t)M->nall * M->m.nvar * sizeof(double);
  // each buffer is allocated once; a failure part-way leaves the ones already there for the next call (freed with the mesh)
  for (int d = 0; d < 3; ++d)
    if (!M->ws_field[d] && cudaMalloc((void**)&M->ws_field[d], fbytes) != cudaSuccess) { M->ws_field[d] = nullptr; cudaGetLastError(); return fail(PHX_ENOMEM, "phx_evolve_host: out of device memory"); }
  if (!M->ws_mask && cudaMalloc((void**)&M->ws_mask, (size_t)M->nall) != cudaSuccess) { M->ws_mask = nullptr; cudaGetLastError(); return fail(PHX_ENOMEM, "phx_evolve_host: out of device memory"); }
  if (!M->ws_scal && cudaMalloc((void**)&M->ws_scal, 2 * sizeof(double)) != cudaSuccess) { M->ws_scal = nullptr; cudaGetLastError(); return fail(PHX_ENOMEM, "phx_evolve_host: out of device memory"); }
  double* prim = M->ws_field[0];
  double* cons = M->ws_field[1];
  double* cons0 = M->ws_field[2];
  CUDA_TRY(cudaMemcpyAsync(prim, h_prim_in, fbytes, cudaMemcpyHostToDevice, st), "cudaMemcpyAsync H2D");
  CUDA_TRY(cudaMemsetAsync(M->ws_scal, 0, 2 * sizeof(double), st), "cudaMemsetAsync");
  CUDA_TRY(cudaMemsetAsync(M->ws_mask, 0, (size_t)M->nall, st), "cudaMemsetAsync");
  int rc = phx_prim_to_cons(M, prim, cons, st);
  if (rc != PHX_OK) return rc;
  if (nsteps > 0) {
    rc = phx_cfl_dt(M, prim, cfl, M->ws_scal, nullptr, st);
    if (rc != PHX_OK) return rc;
  }
  rc = phx_evolve_device(M, nsteps, cfl, M->ws_scal, M->ws_scal + 1, cons0, cons, prim, M->ws_mask, st);   // t += dt, step; graph replay
  if (rc != PHX_OK) return rc;
  CUDA_TRY(cudaMemcpyAsync(h_prim_out, prim, fbytes, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync D2H");
  if (h_cons_out) CUDA_TRY(cudaMemcpyAsync(h_cons_out, cons, fbytes, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync D2H");
  if (h_mask_out) CUDA_TRY(cudaMemcpyAsync(h_mask_out, M->ws_mask, (size_t)M->nall, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync D2H");
  double scal[2] = {0.0, 0.0};
  CUDA_TRY(cudaMemcpyAsync(scal, M->ws_scal, sizeof scal, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync D2H");
  CUDA_TRY(cudaStreamSynchronize(st), "cudaStreamSynchronize");
  if (h_t) *h_t = scal[1];
  return PHX_OK;
}
