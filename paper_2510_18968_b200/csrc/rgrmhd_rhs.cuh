// rgrmhd_rhs.cuh -- device pieces shared by the flux-divergence kernels: one HLLE face flux from
// global-memory stencils (a2+a3) and the flux-divergence part of the IMEX stage combine (a5).
#pragma once
#include "rgrmhd_common.cuh"

namespace rg {

// a2+a3. HLLE flux at the LOWER face, in direction K, of the cell with padded index cR.
// Reconstruction stencil: cells cR-3s .. cR+2s of the 14 primitives and of jc^K (reading R3/R4).
template <int K, int RECON, int CHARGE>
__device__ __forceinline__ void face_flux(const GridView& G, long long cR, double Fh[NCONS]) {
  const long long s = G.stride[K];
  const long long cL = cR - s;
  Met mf;
  load_met_face(G, cL, cR, mf);
  double PL[NPRIM], PR[NPRIM], jL = 0.0, jR = 0.0;
#pragma unroll
  for (int v = 0; v < NPRIM; ++v) {
    const double* __restrict__ f = G.P[v];
    if (RECON == RECON_WENO5) {
      const double u0 = f[cR - 3 * s], u1 = f[cR - 2 * s], u2 = f[cL], u3 = f[cR], u4 = f[cR + s], u5 = f[cR + 2 * s];
      PL[v] = recon_hi<RECON>(G.weno_eps, u0, u1, u2, u3, u4);
      PR[v] = recon_lo<RECON>(G.weno_eps, u1, u2, u3, u4, u5);
    } else {
      const double u1 = f[cR - 2 * s], u2 = f[cL], u3 = f[cR], u4 = f[cR + s];
      PL[v] = recon_hi<RECON>(0.0, 0.0, u1, u2, u3, 0.0);
      PR[v] = recon_lo<RECON>(0.0, 0.0, u2, u3, u4, 0.0);
    }
  }
  if (CHARGE == CHARGE_CELL_CURRENT) {
    const double* __restrict__ f = G.jc[K];
    if (RECON == RECON_WENO5) {
      const double u0 = f[cR - 3 * s], u1 = f[cR - 2 * s], u2 = f[cL], u3 = f[cR], u4 = f[cR + s], u5 = f[cR + 2 * s];
      jL = recon_hi<RECON>(G.weno_eps, u0, u1, u2, u3, u4);
      jR = recon_lo<RECON>(G.weno_eps, u1, u2, u3, u4, u5);
    } else {
      const double u1 = f[cR - 2 * s], u2 = f[cL], u3 = f[cR], u4 = f[cR + s];
      jL = recon_hi<RECON>(0.0, 0.0, u1, u2, u3, 0.0);
      jR = recon_lo<RECON>(0.0, 0.0, u2, u3, u4, 0.0);
    }
  }
  // reading R4: unphysical face values fall back to the cell value
  if (!(PL[RHO] > 0.0)) PL[RHO] = G.P[RHO][cL];
  if (!(PL[PRS] > 0.0)) PL[PRS] = G.P[PRS][cL];
  if (!(PR[RHO] > 0.0)) PR[RHO] = G.P[RHO][cR];
  if (!(PR[PRS] > 0.0)) PR[PRS] = G.P[PRS][cR];
  double sigL = 0.0, sigR = 0.0;
  if (CHARGE == CHARGE_FACE_OHM) {   // reading R6: piecewise-constant sigma from the adjacent cells
    Met mc;
    double vU[3], vD[3];
    load_met_cell(G, cL, mc);
    vU[0] = G.P[VX][cL]; vU[1] = G.P[VY][cL]; vU[2] = G.P[VZ][cL];
    lower(mc, vU, vD);
    sigL = sigma_of(G, G.P[RHO][cL] * (1.0 / sqrt(1.0 - dot3(vU, vD))), cL);
    load_met_cell(G, cR, mc);
    vU[0] = G.P[VX][cR]; vU[1] = G.P[VY][cR]; vU[2] = G.P[VZ][cR];
    lower(mc, vU, vD);
    sigR = sigma_of(G, G.P[RHO][cR] * (1.0 / sqrt(1.0 - dot3(vU, vD))), cR);
  }
  hlle<K, CHARGE>(mf, G.Gamma, PL, PR, sigL, sigR, jL, jR, G.wave_mode, G.wave_rho_switch, Fh);
}

// a5 (flux-divergence part; the point-wise part is stage_precombine in rgrmhd_sources.cuh).  dU = -div F of the
// cell.  The flux kernels only WRITE the increment w dt dU (w = 1 in stage 1, 1/2 in stage 2) to G.dU; the
// recovery kernel that follows adds it to the bracket of its stage vector (U*2 or U^{n+1}) as it loads it.  No
// load sits in the stencil kernel's critical path and no registers are held for a read-modify-write.
template <int STAGE>
__device__ __forceinline__ void divergence_update(const GridView& G, long long c, double dt, const double dU[NCONS]) {
  const double w = (STAGE == 1) ? dt : 0.5 * dt;
#pragma unroll
  for (int v = 0; v < NCONS; ++v) G.dU[v][c] = w * dU[v];
}

}  // namespace rg
