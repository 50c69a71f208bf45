// rgrmhd_sources.cuh -- the point-wise half of the right-hand side: explicit geometric sources (a4) and the
// point-wise part of the IMEX stage combine (a5).  Both depend on the cell's own primitives and on the
// (time-independent) metric only, so they run in the recovery kernel that has just produced those
// primitives (rgrmhd_c2p.cu) and the stencil kernel is left with the flux divergence alone.
#pragma once
#include "rgrmhd_common.cuh"

namespace rg {

// 4th-order centred difference (reading R2)
__device__ __forceinline__ double d4(const double* __restrict__ f, long long c, long long s, double inv_12dx) {
  return (-__ldg(f + c + 2 * s) + 8.0 * __ldg(f + c + s) - 8.0 * __ldg(f + c - s) + __ldg(f + c - 2 * s)) * inv_12dx;
}

// Static source coefficients.  The metric is fixed in time (north_star), so everything in the sources that
// depends on the metric alone is computed ONCE per set_metric (k_metric_coeffs) and stored as NSRC fields:
//   SRC_DAL + d          d_d alpha                       (3)
//   SRC_DB  + 3 d + a    d_d beta^a                      (9)
//   SRC_DG  + 6 d + q    d_d gamma_q, q = xx..zz         (18)
//   SRC_GA  + a          G^a = gamma^ab d_b alpha - alpha gamma^al gamma^jk (d_j gamma_lk - 1/2 d_l gamma_jk)   (3)
//   SRC_TRK              K = gamma^ij K_ij               (1)
// with the 4th-order centred differences of reading R2 (inactive direction -> 0).
enum { SRC_DAL = 0, SRC_DB = 3, SRC_DG = 12, SRC_GA = 30, SRC_TRK = 33 };
static_assert(SRC_TRK + 1 == NSRC, "source coefficient count");

__device__ __forceinline__ void metric_coeffs_cell(const GridView& G, long long c, double out[NSRC]) {
  Met m;
  load_met_cell(G, c, m);
  double trK = 0.0;
#pragma unroll
  for (int q = 0; q < 6; ++q)
    trK += ((q == 0 || q == 3 || q == 5) ? 1.0 : 2.0) * m.gi[q] * __ldg(G.met[MKXX + q] + c);
  out[SRC_TRK] = trK;
  double Cl[3] = {0.0, 0.0, 0.0}, da[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double dal = 0.0, db[3] = {0.0, 0.0, 0.0}, dg[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (G.n[d] > 1) {
      const long long s = G.stride[d];
      const double w = G.inv_12dx[d];
      dal = d4(G.met[MALP], c, s, w);
#pragma unroll
      for (int a = 0; a < 3; ++a) db[a] = d4(G.met[MBX + a], c, s, w);
#pragma unroll
      for (int q = 0; q < 6; ++q) dg[q] = d4(G.met[MGXX + q], c, s, w);
    }
    da[d] = dal;
    double gdg = 0.0;
#pragma unroll
    for (int q = 0; q < 6; ++q) gdg += ((q == 0 || q == 3 || q == 5) ? 1.0 : 2.0) * m.gi[q] * dg[q];
#pragma unroll
    for (int l = 0; l < 3; ++l)
      Cl[l] += m.gi[sym(d, 0)] * dg[sym(l, 0)] + m.gi[sym(d, 1)] * dg[sym(l, 1)] + m.gi[sym(d, 2)] * dg[sym(l, 2)];
    Cl[d] -= 0.5 * gdg;
    out[SRC_DAL + d] = dal;
#pragma unroll
    for (int a = 0; a < 3; ++a) out[SRC_DB + 3 * d + a] = db[a];
#pragma unroll
    for (int q = 0; q < 6; ++q) out[SRC_DG + 6 * d + q] = dg[q];
  }
  double Gi[3], gda[3];
  raise(m, Cl, Gi);
  raise(m, da, gda);
#pragma unroll
  for (int a = 0; a < 3; ++a) out[SRC_GA + a] = gda[a] - m.alpha * Gi[a];
}

// a4 (second half). explicit sources at a cell centre (Eq. 27 S; Eq. 39-40;
// reading R1 / SURVEY.md O6).  P = the cell's primitives, m = the cell's metric; ADDS the sources to S[].
//   S(S_i)  = 1/2 alpha sg T^jk d_i gamma_jk + S_j d_i beta^j - (tau + D) d_i alpha
//   S(tau)  = alpha sg T^ij K_ij - S^j d_j alpha
//   S(calB^i) = -calB^k d_k beta^i + Phi G^i ;  S(calE^i) = -calE^k d_k beta^i + Psi G^i - alpha calQ v^i
//   S(Phi)  = -alpha Phi K + calB^k d_k alpha - alpha kappa Phi ;  S(Psi) likewise + alpha calQ
// All metric derivatives, G^i and K come from the static coefficient fields (G.src): 40 coalesced loads,
// no stencil.
// src[NSRC], Kq[6]: the cell's static coefficients and K_ij (the caller stages them, rgrmhd_c2p.cu).
__device__ __forceinline__ void add_sources(const GridView& G, const Met& m, const double src[NSRC], const double Kq[6],
                                            const double P[NPRIM], double S[NCONS]) {
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3], ExB[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  cross_raw(EU, BU, ExB);
  const double v2 = dot3(vU, vD), W2 = rcp_fast(1.0 - v2);
  const double h = rho + G.gog1 * p;
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
  // charge mode DIV_E: the stage's charge is computed from its electric field AFTER this kernel
  // (k_charge_div_e), which also applies the two source terms that carry it
  const double cPsi = sg * P[PSI], cPhi = sg * P[PHI], cQ = (G.charge_mode == CHARGE_DIV_E) ? 0.0 : sg * P[QCH];
  const double asg = al * sg;
  {
    double t1 = 0.0;
#pragma unroll
    for (int q = 0; q < 6; ++q) t1 += Tw[q] * Kq[q];
    S[CTAU] += asg * t1;
  }
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const double dal = src[SRC_DAL + d];
    const double* db = &src[SRC_DB + 3 * d];
    const double* dg = &src[SRC_DG + 6 * d];
    double tg = 0.0;
#pragma unroll
    for (int q = 0; q < 6; ++q) tg += Tw[q] * dg[q];
    S[CSX + d] += 0.5 * asg * tg + (SD[0] * db[0] + SD[1] * db[1] + SD[2] * db[2]) - tauD * dal;
    S[CTAU] -= SU[d] * dal;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      S[CBX + a] -= cB[d] * db[a];
      S[CEX + a] -= cE[d] * db[a];
    }
    S[CPHI] += cB[d] * dal;
    S[CPSI] += cE[d] * dal;
  }
  const double trK = src[SRC_TRK];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double Ga = src[SRC_GA + a];
    S[CBX + a] += cPhi * Ga;
    S[CEX + a] += cPsi * Ga - al * cQ * vU[a];
  }
  S[CPHI] -= al * cPhi * (trK + G.kappa);
  S[CPSI] += al * (cQ - cPsi * (trK + G.kappa));
}

// a5. IMEX-SSP2(2,2,2) stage combine (Eq. 35-37; gamma = 1 - 1/sqrt(2); readings R11, R12),
// split into a point-wise part (here) and the flux-divergence part (rgrmhd_rhs.cuh, divergence_update).
// With F = -div F + S the explicit operator, X = calE, R^(i) = (X^(i) - X*^(i))/(gamma dt):
//   STAGE 1:  U*2     = [U^n + dt S1 + (1-2 gamma)/gamma (X1 - X^n)|_X]                        - dt div F1
//   STAGE 2:  U^{n+1} = [(U^n + U*2)/2 + dt/2 S2 + ((X1 - X^n) + (X2 - X*2)/(2 gamma))|_X]   - dt/2 div F2
// (dt F1 is carried by U*2).  This function writes the bracket: stage 1 into G.Us, stage 2 into G.Un (in place).
// S = explicit sources of the cell, sgE = sqrt(gamma) E^(stage), un / us = the cell's U^n / U*2 (us: stage 2), x1 = its calE^(1) (stage 2).
template <int STAGE>
__device__ __forceinline__ void stage_precombine(const GridView& G, long long c, double dt, const double S[NCONS],
                                                 const double sgE[3], const double un[NCONS], const double us[NCONS],
                                                 const double x1[3]) {
  const double gam = 1.0 - 0.70710678118654752440;   // 1 - 1/sqrt(2)
  const double c1 = (1.0 - 2.0 * gam) / gam, c2 = 1.0 / (2.0 * gam);   // compile-time constants
  if (STAGE == 1) {
#pragma unroll
    for (int v = 0; v < NCONS; ++v) {
      double u = un[v] + dt * S[v];
      if (v >= CEX && v <= CEZ) u += c1 * (sgE[v - CEX] - un[v]);       // dt (1 - 2 gamma) R1, R1 = (X1 - X^n)/(gamma dt)
      G.Us[v][c] = u;
    }
  } else {
#pragma unroll
    for (int v = 0; v < NCONS; ++v) {
      double u = 0.5 * (un[v] + us[v]) + 0.5 * dt * S[v];
      if (v >= CEX && v <= CEZ) u += (x1[v - CEX] - un[v]) + c2 * (sgE[v - CEX] - us[v]);
      G.Un[v][c] = u;
    }
  }
}

}  // namespace rg
