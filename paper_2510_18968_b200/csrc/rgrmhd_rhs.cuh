// rgrmhd_rhs.cuh -- device pieces shared by the RHS kernels: one HLLE face flux from global-memory
// stencils (a2+a3), the explicit geometric sources (a4), and the IMEX stage combine (a5).
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
  hlle<K, CHARGE>(mf, G.Gamma, PL, PR, sigL, sigR, jL, jR, Fh);
}

// 4th-order centred difference (reading R2)
__device__ __forceinline__ double d4(const double* __restrict__ f, long long c, long long s, double inv_12dx) {
  return (-__ldg(f + c + 2 * s) + 8.0 * __ldg(f + c + s) - 8.0 * __ldg(f + c - s) + __ldg(f + c - 2 * s)) * inv_12dx;
}

// a4 (second half). explicit sources at a cell centre (Eq. 27 S; Eq. 39-40;
// reading R1 / SURVEY.md O6).  P = the cell's primitives; ADDS the sources to S[].
__device__ __forceinline__ void add_sources(const GridView& G, long long c, const double P[NPRIM], double S[NCONS]) {
  Met m;
  load_met_cell(G, c, m);
  double KDD[6];
#pragma unroll
  for (int q = 0; q < 6; ++q) KDD[q] = __ldg(G.met[MKXX + q] + c);
  double dalpha[3], dbeta[3][3], dg[3][6];   // dalpha[k] = d_k alpha; dbeta[k][i] = d_k beta^i; dg[k][q] = d_k gamma_q
#pragma unroll
  for (int kk = 0; kk < 3; ++kk) {
    if (G.n[kk] > 1) {
      const long long s = G.stride[kk];
      const double w = G.inv_12dx[kk];
      dalpha[kk] = d4(G.met[MALP], c, s, w);
#pragma unroll
      for (int a = 0; a < 3; ++a) dbeta[kk][a] = d4(G.met[MBX + a], c, s, w);
#pragma unroll
      for (int q = 0; q < 6; ++q) dg[kk][q] = d4(G.met[MGXX + q], c, s, w);
    } else {
      dalpha[kk] = 0.0;
#pragma unroll
      for (int a = 0; a < 3; ++a) dbeta[kk][a] = 0.0;
#pragma unroll
      for (int q = 0; q < 6; ++q) dg[kk][q] = 0.0;
    }
  }
  double U[NCONS];
  prim2cons(m, G.Gamma, P, U);
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  const double v2 = dot3(vU, vD), W2 = 1.0 / (1.0 - v2);
  const double h = rho + G.Gamma / (G.Gamma - 1.0) * p;
  const double pem = 0.5 * (dot3(EU, ED) + dot3(BU, BD)), hW2 = h * W2;
  // T^ab = h W^2 v^a v^b + g^ab (p + (E^2+B^2)/2) - E^a E^b - B^a B^b   (symmetric storage)
  double T[6];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b)
      T[sym(a, b)] = hW2 * vU[a] * vU[b] + m.gi[sym(a, b)] * (p + pem) - EU[a] * EU[b] - BU[a] * BU[b];
  const double al = m.alpha, sg = m.sg;
  const double SD[3] = {U[CSX], U[CSY], U[CSZ]};
  double SU[3];
  raise(m, SD, SU);
  // symmetric contraction X^ab Y_ab = sum_q w_q X_q Y_q, w = (1,2,2,1,2,1)
  const double wq[6] = {1.0, 2.0, 2.0, 1.0, 2.0, 1.0};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double t1 = 0.0, t2 = 0.0;
#pragma unroll
    for (int q = 0; q < 6; ++q) t1 += wq[q] * T[q] * dg[a][q];
#pragma unroll
    for (int b = 0; b < 3; ++b) t2 += SD[b] * dbeta[a][b];
    S[CSX + a] += 0.5 * al * sg * t1 + t2 - (U[CTAU] + U[CD]) * dalpha[a];
  }
  {
    double t1 = 0.0, trK = 0.0;
#pragma unroll
    for (int q = 0; q < 6; ++q) { t1 += wq[q] * T[q] * KDD[q]; trK += wq[q] * m.gi[q] * KDD[q]; }
    S[CTAU] += al * sg * t1 - dot3(SU, dalpha);
    // G^i = gamma^ij d_j alpha - alpha gamma^il gamma^jk (d_j gamma_lk - 1/2 d_l gamma_jk)
    double Cl[3];
#pragma unroll
    for (int l = 0; l < 3; ++l) {
      double t = 0.0;
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int k2 = 0; k2 < 3; ++k2)
          t += m.gi[sym(j, k2)] * (dg[j][sym(l, k2)] - 0.5 * dg[l][sym(j, k2)]);
      Cl[l] = t;
    }
    double Gi[3], gda[3];
    raise(m, Cl, Gi);
    raise(m, dalpha, gda);
#pragma unroll
    for (int a = 0; a < 3; ++a) Gi[a] = gda[a] - al * Gi[a];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double tB = 0.0, tE = 0.0;
#pragma unroll
      for (int kk = 0; kk < 3; ++kk) { tB += U[CBX + kk] * dbeta[kk][a]; tE += U[CEX + kk] * dbeta[kk][a]; }
      S[CBX + a] += -tB + U[CPHI] * Gi[a];
      S[CEX + a] += -tE + U[CPSI] * Gi[a] - al * U[CQ] * vU[a];
    }
    double BdA = 0.0, EdA = 0.0;
#pragma unroll
    for (int kk = 0; kk < 3; ++kk) { BdA += U[CBX + kk] * dalpha[kk]; EdA += U[CEX + kk] * dalpha[kk]; }
    S[CPHI] += -al * U[CPHI] * trK + BdA - al * G.kappa * U[CPHI];
    S[CPSI] += -al * U[CPSI] * trK + EdA + al * U[CQ] - al * G.kappa * U[CPSI];
  }
}

// a5. IMEX-SSP2(2,2,2) stage combine (Eq. 35-37; gamma = 1 - 1/sqrt(2); readings R11, R12)
// for one cell, given F = F[U^(stage)] (flux divergence + sources) and sgE = sqrt(gamma) E^(stage) of the cell.
//   STAGE 1:  U*2 = U^n + dt F1;  X*2 += dt (1-2g) R1,  R1 = (X1 - X^n)/(g dt)                       -> G.Us
//   STAGE 2:  U^{n+1} = U^n + dt/2 (F1 + F2) + dt/2 (R1 + R2) on X, with dt F1 recovered from U*2:
//             Y^{n+1} = (Y^n + Y*2)/2 + dt/2 F2_Y
//             X^{n+1} = (X^n + X*2)/2 + dt/2 F2_X + (X1 - X^n) + (X2 - X*2)/(2g)                      -> G.Un
template <int STAGE>
__device__ __forceinline__ void stage_combine(const GridView& G, long long c, double dt, const double F[NCONS],
                                              const double sgE[3]) {
  const double gam = 1.0 - 0.70710678118654752440;   // 1 - 1/sqrt(2)
  if (STAGE == 1) {
#pragma unroll
    for (int v = 0; v < NCONS; ++v) {
      const double un = G.Un[v][c];
      double us = un + dt * F[v];
      if (v >= CEX && v <= CEZ) {
        const double R1 = (sgE[v - CEX] - un) / (gam * dt);
        us += dt * (1.0 - 2.0 * gam) * R1;
      }
      G.Us[v][c] = us;
    }
  } else {
#pragma unroll
    for (int v = 0; v < NCONS; ++v) {
      const double un = G.Un[v][c], us = G.Us[v][c];
      double u = 0.5 * (un + us) + 0.5 * dt * F[v];
      if (v >= CEX && v <= CEZ) {
        const double x1 = G.X1[v - CEX][c];
        u += (x1 - un) + (sgE[v - CEX] - us) / (2.0 * gam);
      }
      G.Un[v][c] = u;
    }
  }
}

}  // namespace rg
