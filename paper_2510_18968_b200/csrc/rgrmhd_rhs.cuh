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
//   S(S_i)  = 1/2 alpha sg T^jk d_i gamma_jk + S_j d_i beta^j - (tau + D) d_i alpha
//   S(tau)  = alpha sg T^ij K_ij - S^j d_j alpha
//   S(calB^i) = -calB^k d_k beta^i + Phi G^i ;  S(calE^i) = -calE^k d_k beta^i + Psi G^i - alpha calQ v^i
//   S(Phi)  = -alpha Phi K + calB^k d_k alpha - alpha kappa Phi ;  S(Psi) likewise + alpha calQ
//   G^i = gamma^ij d_j alpha - alpha gamma^il gamma^jk (d_j gamma_lk - 1/2 d_l gamma_jk)
// The metric derivatives (4th-order centred, reading R2) are consumed direction by direction so that
// only one direction's ten derivatives are live at a time.
__device__ __forceinline__ void add_sources(const GridView& G, long long c, const double P[NPRIM], double S[NCONS]) {
  Met m;
  load_met_cell(G, c, m);
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3], ExB[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  cross_raw(EU, BU, ExB);
  const double v2 = dot3(vU, vD), W2 = rcp_fast(1.0 - v2);
  const double h = rho + G.Gamma / (G.Gamma - 1.0) * p;
  const double pem = 0.5 * (dot3(EU, ED) + dot3(BU, BD)), hW2 = h * W2;
  const double al = m.alpha, sg = m.sg;
  // T^ab = h W^2 v^a v^b + g^ab (p + (E^2+B^2)/2) - E^a E^b - B^a B^b, stored with the symmetric-contraction
  // weights (1,2,2,1,2,1) folded in:  X^ab Y_ab = sum_q Tw_q Y_q
  double Tw[6];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b) {
      const double t = hW2 * vU[a] * vU[b] + m.gi[sym(a, b)] * (p + pem) - EU[a] * EU[b] - BU[a] * BU[b];
      Tw[sym(a, b)] = (a == b) ? t : 2.0 * t;
    }
  double SD[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) SD[a] = sg * (hW2 * vD[a] + sg * ExB[a]);            // Eq. 24
  double SU[3];
  raise(m, SD, SU);
  const double tauD = sg * (hW2 - p + pem);                                         // tau + D (Eq. 22-23)
  const double cE[3] = {sg * EU[0], sg * EU[1], sg * EU[2]}, cB[3] = {sg * BU[0], sg * BU[1], sg * BU[2]};
  const double cPsi = sg * P[PSI], cPhi = sg * P[PHI], cQ = sg * P[QCH];
  const double asg = al * sg;
  double trK = 0.0;
  {
    double t1 = 0.0;
#pragma unroll
    for (int q = 0; q < 6; ++q) {
      const double Kq = __ldg(G.met[MKXX + q] + c);
      t1 += Tw[q] * Kq;
      trK += ((q == 0 || q == 3 || q == 5) ? 1.0 : 2.0) * m.gi[q] * Kq;
    }
    S[CTAU] += asg * t1;
  }
  double Cl[3] = {0.0, 0.0, 0.0}, da[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (G.n[d] > 1) {
      const long long s = G.stride[d];
      const double w = G.inv_12dx[d];
      const double dal = d4(G.met[MALP], c, s, w);
      double db[3], dg[6];
#pragma unroll
      for (int a = 0; a < 3; ++a) db[a] = d4(G.met[MBX + a], c, s, w);
#pragma unroll
      for (int q = 0; q < 6; ++q) dg[q] = d4(G.met[MGXX + q], c, s, w);
      da[d] = dal;
      double tg = 0.0, gdg = 0.0;
#pragma unroll
      for (int q = 0; q < 6; ++q) {
        tg += Tw[q] * dg[q];
        gdg += ((q == 0 || q == 3 || q == 5) ? 1.0 : 2.0) * m.gi[q] * dg[q];
      }
      S[CSX + d] += 0.5 * asg * tg + (SD[0] * db[0] + SD[1] * db[1] + SD[2] * db[2]) - tauD * dal;
      S[CTAU] -= SU[d] * dal;
#pragma unroll
      for (int l = 0; l < 3; ++l)
        Cl[l] += m.gi[sym(d, 0)] * dg[sym(l, 0)] + m.gi[sym(d, 1)] * dg[sym(l, 1)] + m.gi[sym(d, 2)] * dg[sym(l, 2)];
      Cl[d] -= 0.5 * gdg;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        S[CBX + a] -= cB[d] * db[a];
        S[CEX + a] -= cE[d] * db[a];
      }
      S[CPHI] += cB[d] * dal;
      S[CPSI] += cE[d] * dal;
    }
  }
  double Gi[3], gda[3];
  raise(m, Cl, Gi);
  raise(m, da, gda);
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double Ga = gda[a] - al * Gi[a];
    S[CBX + a] += cPhi * Ga;
    S[CEX + a] += cPsi * Ga - al * cQ * vU[a];
  }
  S[CPHI] -= al * cPhi * (trK + G.kappa);
  S[CPSI] += al * (cQ - cPsi * (trK + G.kappa));
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
