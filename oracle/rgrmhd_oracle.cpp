// rgrmhd_oracle.cpp -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
//
// A plain, slow, obviously-correct FP64 implementation of one IMEX-SSP2(2,2,2) step of the
// resistive GRMHD system of arxiv/paper_2510_18968 on a uniform Cartesian block with a fixed
// 3+1 metric.  It follows the paper's equations in the paper's order and notation; every
// function cites the passage (PAPER.md:line, equation) it restates, and every reading of a
// silent / garbled passage is the one listed in DESIGN.md ("Readings", R1..R12).
//
// Rules this file obeys (task prompt, section 3):
//   * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
//     may load it; the product (paper_2510_18968_b200/) never does;
//   * it shares no code, header, table or helper with the CUDA path;
//   * no blocking, fusion or reordering beyond what the equations state; one cell at a time;
//   * built with  g++ -O2 -ffp-contract=off  (no FMA contraction); `#pragma omp` lines are
//     active only in the separately built OpenMP variant used for the large parity samples
//     (cell updates are independent and max is exact, so results do not depend on threads).
//
// Pinned by tests/test_oracle_*.py (-m "not gpu").  UNPINNED conventions (fixed by DESIGN.md
// only, "parity unpinned" against the paper): charge-flux evaluation (charge_mode), WENO
// epsilon, face-metric averaging, metric-derivative order, floor threshold, sigma-at-face
// rule, choice of reconstructed variables.
//
// Notation: hats = undensitised conserved variables X^ = X/sqrt(gamma).  Index placement is
// spelled out in names: vU = v^i, vD = v_i.  h = rho(1+eps)+p is the enthalpy DENSITY
// (PAPER.md:131).  Z = h W^2.

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

// Instrumented build (oracle/count_flops.py): every `double` below becomes a counting scalar that
// tallies add/mul/div/sqrt per region of the step.  Same arithmetic, same results; never used by tests or timing.
#ifdef ORACLE_COUNT_FLOPS
#include "flopcount.h"
namespace flopcount { long long counts[R_COUNT][OP_COUNT]; long long calls[R_COUNT]; int region = R_OTHER; }
#define double cdouble
#define FLOP_REGION(r) flopcount::Scope flop_scope__(flopcount::r)
#else
#define FLOP_REGION(r)
#endif

namespace {

enum { NPRIM = 14, NCONS = 14, NMET = 16 };
// primitive indices
enum { RHO = 0, PRS, VX, VY, VZ, EX, EY, EZ, BX, BY, BZ, PSI, PHI, QCH };
// conserved indices
enum { CD = 0, CSX, CSY, CSZ, CTAU, CEX, CEY, CEZ, CBX, CBY, CBZ, CPSI, CPHI, CQ };
// metric field indices
enum { MALP = 0, MBX, MBY, MBZ, MGXX, MGXY, MGXZ, MGYY, MGYZ, MGZZ, MKXX, MKXY, MKXZ, MKYY, MKYZ, MKZZ };
enum { BC_PERIODIC = 0, BC_OUTFLOW = 1 };
enum { SIGMA_UNIFORM = 0, SIGMA_ARRAY = 1, SIGMA_POWER_D = 2, SIGMA_ATMO = 3 };
enum { CHARGE_FACE_OHM = 0, CHARGE_CELL_CURRENT = 1, CHARGE_DIV_E = 2 };
enum { RECON_MINMOD = 0, RECON_MC = 1, RECON_WENO5 = 2 };
enum { WAVE_LIGHT = 0, WAVE_MHD_INSIDE = 1 };

// permutation symbol [ijk]
inline double perm(int i, int j, int k) { return 0.5 * (i - j) * (j - k) * (k - i); }

// ---------------------------------------------------------------------------------------------
// O1. metric algebra at one point (Eq. 1-5; PAPER.md:119 for K)
// ---------------------------------------------------------------------------------------------
struct Metric {
  double alpha;
  double betaU[3];
  double gDD[3][3];   // gamma_ij
  double gUU[3][3];   // gamma^ij, algebraic inverse (adjugate / det)
  double sqrtg;       // sqrt(det gamma_ij)
  double KDD[3][3];   // K_ij (cell centres only)
};

void metric_finish(Metric& m) {
  const double (*g)[3] = m.gDD;
  double det = g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[2][1])
             - g[0][1] * (g[1][0] * g[2][2] - g[1][2] * g[2][0])
             + g[0][2] * (g[1][0] * g[2][1] - g[1][1] * g[2][0]);
  m.sqrtg = std::sqrt(det);
  m.gUU[0][0] = (g[1][1] * g[2][2] - g[1][2] * g[2][1]) / det;
  m.gUU[0][1] = (g[0][2] * g[2][1] - g[0][1] * g[2][2]) / det;
  m.gUU[0][2] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det;
  m.gUU[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[2][0]) / det;
  m.gUU[1][2] = (g[0][2] * g[1][0] - g[0][0] * g[1][2]) / det;
  m.gUU[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[1][0]) / det;
  m.gUU[1][0] = m.gUU[0][1];
  m.gUU[2][0] = m.gUU[0][2];
  m.gUU[2][1] = m.gUU[1][2];
}

inline void lower(const Metric& m, const double aU[3], double aD[3]) {
  for (int i = 0; i < 3; ++i) { aD[i] = 0; for (int j = 0; j < 3; ++j) aD[i] += m.gDD[i][j] * aU[j]; }
}
inline void raise(const Metric& m, const double aD[3], double aU[3]) {
  for (int i = 0; i < 3; ++i) { aU[i] = 0; for (int j = 0; j < 3; ++j) aU[i] += m.gUU[i][j] * aD[j]; }
}
inline double dotUD(const double aU[3], const double bD[3]) { return aU[0] * bD[0] + aU[1] * bD[1] + aU[2] * bD[2]; }
// (a x b)^i = [ijk] a_j b_k / sqrt(gamma)      (SURVEY.md Sec. 8 notation; eps^{ijk} = [ijk]/sqrt(gamma))
inline void crossU(const Metric& m, const double aD[3], const double bD[3], double cU[3]) {
  cU[0] = (aD[1] * bD[2] - aD[2] * bD[1]) / m.sqrtg;
  cU[1] = (aD[2] * bD[0] - aD[0] * bD[2]) / m.sqrtg;
  cU[2] = (aD[0] * bD[1] - aD[1] * bD[0]) / m.sqrtg;
}
// (a x b)_i = sqrt(gamma) [ijk] a^j b^k        (eps_{ijk} = sqrt(gamma) [ijk])
inline void crossD(const Metric& m, const double aU[3], const double bU[3], double cD[3]) {
  cD[0] = m.sqrtg * (aU[1] * bU[2] - aU[2] * bU[1]);
  cD[1] = m.sqrtg * (aU[2] * bU[0] - aU[0] * bU[2]);
  cD[2] = m.sqrtg * (aU[0] * bU[1] - aU[1] * bU[0]);
}

// ---------------------------------------------------------------------------------------------
// a0. primitive -> conserved at one point (Eq. 22-24; Eq. 28;
//     EOS PAPER.md:267 Eq. 49)
// ---------------------------------------------------------------------------------------------
void prim2cons_point(const Metric& m, double Gamma, const double P[NPRIM], double U[NCONS]) {
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3], ExB_D[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  const double v2 = dotUD(vU, vD);
  const double W = 1.0 / std::sqrt(1.0 - v2);                 // Eq. 45 / PAPER.md:71
  const double eps = p / ((Gamma - 1.0) * rho);               // Eq. 49
  const double h = rho * (1.0 + eps) + p;
  const double E2 = dotUD(EU, ED), B2 = dotUD(BU, BD);
  crossD(m, EU, BU, ExB_D);                                   // eps_ijk E^j B^k
  const double sg = m.sqrtg;
  U[CD] = sg * rho * W;                                       // Eq. 22
  for (int i = 0; i < 3; ++i) U[CSX + i] = sg * (h * W * W * vD[i] + ExB_D[i]);   // Eq. 24
  U[CTAU] = sg * (h * W * W - p + 0.5 * (E2 + B2)) - U[CD];   // Eq. 23
  for (int i = 0; i < 3; ++i) { U[CEX + i] = sg * EU[i]; U[CBX + i] = sg * BU[i]; }   // Eq. 28
  U[CPSI] = sg * P[PSI]; U[CPHI] = sg * P[PHI]; U[CQ] = sg * P[QCH];
}

// ---------------------------------------------------------------------------------------------
// a3 (first half). conserved vector U and flux F^k of one state at one face
//   Eq. 27 as re-derived in DESIGN.md reading R1 (the printed F is garbled):
//   T^k_j = h W^2 v^k v_j + delta^k_j p - E^k E_j - B^k B_j + delta^k_j (E^2+B^2)/2
//   F(D)=(alpha v^k - beta^k) D ; F(S_j)=alpha sqrt(g) T^k_j - beta^k S_j ;
//   F(tau)=alpha(S^k - v^k D) - beta^k tau ;
//   F(calB^i)= alpha([ikj] E_j + g^ik Phi) - beta^k calB^i ;
//   F(calE^i)=-alpha([ikj] B_j - g^ik Psi) - beta^k calE^i ;
//   F(Phi)=alpha calB^k - beta^k Phi ; F(Psi)=alpha calE^k - beta^k Psi ;
//   F(calQ)=alpha J^k - beta^k calQ, J^k = calQ v^k + Jc^k  (Eq. 29)
//   Jc^k: charge_mode FACE_OHM : W sigma [calE^k + sqrt(g)(v x B)^k - (v.E) sqrt(g) v^k]
//         charge_mode CELL_CURRENT : sqrt(g) * jck, jck = reconstructed undensitised cell current
//         charge_mode DIV_E : as CELL_CURRENT; the evolved calQ is discarded (charge_from_div_E replaces it)
// ---------------------------------------------------------------------------------------------
void state_flux(const Metric& m, double Gamma, int k, const double P[NPRIM], int charge_mode,
                double sigma, double jck, double U[NCONS], double F[NCONS]) {
  prim2cons_point(m, Gamma, P, U);
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  const double v2 = dotUD(vU, vD);
  const double W = 1.0 / std::sqrt(1.0 - v2);
  const double eps = p / ((Gamma - 1.0) * rho);
  const double h = rho * (1.0 + eps) + p;
  const double E2 = dotUD(EU, ED), B2 = dotUD(BU, BD);
  const double a = m.alpha, bk = m.betaU[k], sg = m.sqrtg;
  F[CD] = (a * vU[k] - bk) * U[CD];
  for (int j = 0; j < 3; ++j) {
    const double dkj = (j == k) ? 1.0 : 0.0;
    const double Tkj = h * W * W * vU[k] * vD[j] + dkj * p - EU[k] * ED[j] - BU[k] * BD[j] + 0.5 * dkj * (E2 + B2);
    F[CSX + j] = a * sg * Tkj - bk * U[CSX + j];
  }
  double SD[3] = {U[CSX], U[CSY], U[CSZ]}, SU[3];
  raise(m, SD, SU);
  F[CTAU] = a * (SU[k] - vU[k] * U[CD]) - bk * U[CTAU];
  for (int i = 0; i < 3; ++i) {
    double curlE = 0, curlB = 0;
    for (int j = 0; j < 3; ++j) { curlE += perm(i, k, j) * ED[j]; curlB += perm(i, k, j) * BD[j]; }
    F[CBX + i] = a * (curlE + m.gUU[i][k] * U[CPHI]) - bk * U[CBX + i];
    F[CEX + i] = -a * (curlB - m.gUU[i][k] * U[CPSI]) - bk * U[CEX + i];
  }
  F[CPHI] = a * U[CBX + k] - bk * U[CPHI];
  F[CPSI] = a * U[CEX + k] - bk * U[CPSI];
  double Jck;
  if (charge_mode == CHARGE_FACE_OHM) {
    double vxB_U[3];
    crossU(m, vD, BD, vxB_U);
    const double vE = dotUD(EU, vD);
    Jck = W * sigma * (U[CEX + k] + sg * vxB_U[k] - vE * sg * vU[k]);     // Eq. 29, densitised
  } else {
    Jck = sg * jck;
  }
  F[CQ] = a * (U[CQ] * vU[k] + Jck) - bk * U[CQ];
}

// ---------------------------------------------------------------------------------------------
// a2. reconstruction of one variable from the 5-cell stencil centred on a cell (R4;
//     named only in PAPER.md:169, 287 (minmod), 359 (MC2), 390 (WENO5)).
//     Returns the cell's values at its lower face (i-1/2: the RIGHT state of that face) and at its
//     upper face (i+1/2: the LEFT state of that face).
// ---------------------------------------------------------------------------------------------
inline double minmod2(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  return (a > 0.0 ? 1.0 : -1.0) * std::min(std::fabs(a), std::fabs(b));
}
inline double minmod3(double a, double b, double c) {
  if (a > 0.0 && b > 0.0 && c > 0.0) return std::min(a, std::min(b, c));
  if (a < 0.0 && b < 0.0 && c < 0.0) return std::max(a, std::max(b, c));
  return 0.0;
}
// classic Jiang-Shu WENO5 value at the +1/2 face of the centre cell u2 from cells u0..u4
double weno5_plus(double u0, double u1, double u2, double u3, double u4, double eps_w) {
  const double q0 = (2.0 * u0 - 7.0 * u1 + 11.0 * u2) / 6.0;
  const double q1 = (-u1 + 5.0 * u2 + 2.0 * u3) / 6.0;
  const double q2 = (2.0 * u2 + 5.0 * u3 - u4) / 6.0;
  const double b0 = 13.0 / 12.0 * (u0 - 2.0 * u1 + u2) * (u0 - 2.0 * u1 + u2) + 0.25 * (u0 - 4.0 * u1 + 3.0 * u2) * (u0 - 4.0 * u1 + 3.0 * u2);
  const double b1 = 13.0 / 12.0 * (u1 - 2.0 * u2 + u3) * (u1 - 2.0 * u2 + u3) + 0.25 * (u1 - u3) * (u1 - u3);
  const double b2 = 13.0 / 12.0 * (u2 - 2.0 * u3 + u4) * (u2 - 2.0 * u3 + u4) + 0.25 * (3.0 * u2 - 4.0 * u3 + u4) * (3.0 * u2 - 4.0 * u3 + u4);
  const double a0 = 0.1 / ((eps_w + b0) * (eps_w + b0));
  const double a1 = 0.6 / ((eps_w + b1) * (eps_w + b1));
  const double a2 = 0.3 / ((eps_w + b2) * (eps_w + b2));
  return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
}
void recon_cell(int scheme, double eps_w, double um2, double um1, double u0, double up1, double up2,
                double* at_minus_half, double* at_plus_half) {
  FLOP_REGION(R_RECON);
  if (scheme == RECON_WENO5) {
    *at_plus_half = weno5_plus(um2, um1, u0, up1, up2, eps_w);
    *at_minus_half = weno5_plus(up2, up1, u0, um1, um2, eps_w);   // mirror image
  } else {
    const double a = u0 - um1, b = up1 - u0;
    const double slope = (scheme == RECON_MINMOD) ? minmod2(a, b) : minmod3(2.0 * a, 2.0 * b, 0.5 * (a + b));
    *at_plus_half = u0 + 0.5 * slope;
    *at_minus_half = u0 - 0.5 * slope;
  }
}

// ---------------------------------------------------------------------------------------------
// A18. conductivity models (Eq. 52; Eq. 61); Dhat = D/sqrt(gamma)
// ---------------------------------------------------------------------------------------------
struct Params {
  int n[3]; double dx[3]; int ng; int bc[3];
  double Gamma; int sigma_model; double sigma0, sigma_exp, sigma_dref;
  double kappa, rho_floor, k_atmo, c2p_tol; int c2p_max_iter; int charge_mode; double weno_eps;
  int wave_speed_mode; double wave_rho_switch;
};

double sigma_of(const Params& p, double Dhat, double sigma_cell) {
  switch (p.sigma_model) {
    case SIGMA_UNIFORM: return p.sigma0;
    case SIGMA_ARRAY: return sigma_cell;
    case SIGMA_POWER_D: {
      const int e = (int)std::lround(p.sigma_exp);
      double x = Dhat / p.sigma_dref, r = 1.0;
      for (int i = 0; i < e; ++i) r *= x;                 // integer exponent by multiplication
      return p.sigma0 * r;
    }
    case SIGMA_ATMO: {
      const double x = std::max(1.0 - p.sigma_dref / Dhat, 0.0);
      return p.sigma0 * x * x;
    }
  }
  return 0.0;
}

// ---------------------------------------------------------------------------------------------
// A14. implicit E at fixed v: closed form of the linear system Eq. 42 (G4: the
//      printed "alpha_ii" is the Butcher diagonal a_ii) -- DESIGN.md reading R7.
//      (1+s) E - s (v.E) v + s v x B = Estar,  s = a_ii dt alpha sigma W
//      => kE = v.E = (v.Estar)/(1 + s/W^2);  E = (Estar - s v x B + s kE v)/(1+s)
// ---------------------------------------------------------------------------------------------
void implicit_E_closed(const Metric& m, const double vU[3], double W, double s, const double EstarU[3],
                       const double BD[3], double EU[3]) {
  double vD[3], EstarD[3], vxB_U[3];
  lower(m, vU, vD); lower(m, EstarU, EstarD);
  crossU(m, vD, BD, vxB_U);
  const double kE = dotUD(vU, EstarD) / (1.0 + s / (W * W));
  for (int i = 0; i < 3; ++i) EU[i] = (EstarU[i] - s * vxB_U[i] + s * kE * vU[i]) / (1.0 + s);
}

// The paper's own route (Eq. 42-43): Newton-Raphson on the 3-vector f(E) with its
// 3x3 Jacobian df^i/dE^j = (1+s) delta^i_j - s v^i v_j, solved by Cramer's rule.  f is linear in E,
// so one iteration from any start lands on the root; `iters` iterations are taken anyway.
void implicit_E_newton(const Metric& m, const double vU[3], double W, double s, const double EstarU[3],
                       const double BD[3], const double E0U[3], int iters, double EU[3]) {
  (void)W;
  double vD[3], vxB_U[3];
  lower(m, vU, vD);
  crossU(m, vD, BD, vxB_U);
  double E[3] = {E0U[0], E0U[1], E0U[2]};
  for (int it = 0; it < iters; ++it) {
    double ED[3]; lower(m, E, ED);
    const double vE = dotUD(vU, ED);                     // v_k E^k
    double f[3], J[3][3];
    for (int i = 0; i < 3; ++i) {
      f[i] = E[i] - EstarU[i] + s * (E[i] + vxB_U[i] - vE * vU[i]);
      for (int j = 0; j < 3; ++j) J[i][j] = ((i == j) ? (1.0 + s) : 0.0) - s * vU[i] * vD[j];
    }
    const double det = J[0][0] * (J[1][1] * J[2][2] - J[1][2] * J[2][1]) - J[0][1] * (J[1][0] * J[2][2] - J[1][2] * J[2][0])
                     + J[0][2] * (J[1][0] * J[2][1] - J[1][1] * J[2][0]);
    double dE[3];
    for (int c = 0; c < 3; ++c) {
      double A[3][3];
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) A[i][j] = (j == c) ? f[i] : J[i][j];
      dE[c] = (A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1]) - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0])
             + A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0])) / det;
    }
    for (int i = 0; i < 3; ++i) E[i] -= dE[i];
  }
  for (int i = 0; i < 3; ++i) EU[i] = E[i];
}

// ---------------------------------------------------------------------------------------------
// a6. implicit Ohm update fused with the 1D recovery.
// ---------------------------------------------------------------------------------------------
struct C2PResult { int evals; int failed; };

// (literal) PAPER.md:246-271, steps (i)-(v): loop { E from Eq. 42 with the current v (closed form);
// Eq. 44-47 with the current p (G2: Eq. 44's numerator carries eps_ijk calE^j calB^k / sqrt(gamma));
// ONE Newton step on p with f' = v^2 cs^2 - 1 (Eq. 48; G3: cs^2 = Gamma(Gamma-1)eps/(1+Gamma eps)) }
// until max(|dv^i|, |dp|/p) < tol.   Cross-check only: it diverges for strongly magnetised
// states ("when the magnetic pressure remains moderate").
C2PResult c2p_literal(const Metric& m, double Gamma, const double U[NCONS], double adt, double sigma,
                      double tol, int maxit, double P[NPRIM] /* in: guess (p, v); out: primitives */) {
  const double sg = m.sqrtg;
  const double Dh = U[CD] / sg, tauh = U[CTAU] / sg;
  const double ShD[3] = {U[CSX] / sg, U[CSY] / sg, U[CSZ] / sg};
  const double EstarU[3] = {U[CEX] / sg, U[CEY] / sg, U[CEZ] / sg};
  const double BU[3] = {U[CBX] / sg, U[CBY] / sg, U[CBZ] / sg};
  double BD[3]; lower(m, BU, BD);
  const double B2 = dotUD(BU, BD);
  double p = P[PRS];
  double vU[3] = {P[VX], P[VY], P[VZ]};
  double EU[3] = {EstarU[0], EstarU[1], EstarU[2]};
  double rho = P[RHO];
  C2PResult res = {0, 1};
  for (int it = 0; it < maxit; ++it) {
    res.evals = it + 1;
    double vD[3]; lower(m, vU, vD);
    double v2 = dotUD(vU, vD);
    if (!(v2 < 1.0)) return res;
    double W = 1.0 / std::sqrt(1.0 - v2);
    // (ii) E at the current v
    const double s = adt * m.alpha * sigma * W;
    implicit_E_closed(m, vU, W, s, EstarU, BD, EU);
    // (iii) Eq. 44-47 at the current p
    double ED[3], ExB_D[3]; lower(m, EU, ED);
    const double E2 = dotUD(EU, ED);
    crossD(m, EU, BU, ExB_D);
    const double Z = tauh + Dh + p - 0.5 * (E2 + B2);
    double vnewD[3], vnewU[3];
    for (int i = 0; i < 3; ++i) vnewD[i] = (ShD[i] - ExB_D[i]) / Z;           // Eq. 44
    raise(m, vnewD, vnewU);
    v2 = dotUD(vnewU, vnewD);
    if (!(v2 < 1.0)) return res;
    W = 1.0 / std::sqrt(1.0 - v2);                                             // Eq. 45
    rho = Dh / W;                                                              // Eq. 46
    const double eps = (tauh - Dh * (W - 1.0) - p * (W * W - 1.0) - 0.5 * (E2 + B2)) / (Dh * W);   // Eq. 47
    // (iv) one Newton step on p (Eq. 48-50)
    const double f = (Gamma - 1.0) * rho * eps - p;
    const double cs2 = Gamma * (Gamma - 1.0) * eps / (1.0 + Gamma * eps);
    const double fp = v2 * cs2 - 1.0;
    const double pnew = p - f / fp;
    double dv = 0;
    for (int i = 0; i < 3; ++i) dv = std::max(dv, std::fabs(vnewU[i] - vU[i]));
    const double dp = std::fabs(pnew - p) / std::fabs(pnew);
    for (int i = 0; i < 3; ++i) vU[i] = vnewU[i];
    p = pnew;
    if (!(p > 0.0) || !std::isfinite(p)) return res;
    if (dv < tol && dp < tol) { res.failed = 0; break; }
  }
  P[RHO] = rho; P[PRS] = p;
  for (int i = 0; i < 3; ++i) { P[VX + i] = vU[i]; P[EX + i] = EU[i]; P[BX + i] = BU[i]; }
  P[PSI] = U[CPSI] / sg; P[PHI] = U[CPHI] / sg; P[QCH] = U[CQ] / sg;
  return res;
}

// (robust; reading R8 = SURVEY.md Sec. 8(c) O8) The result is DEFINED as the root (E, v, p) of
//   (1+s) E - s (v.E) v + s v x B = Estar^,  s = adt alpha sigma W           [Eq. 42]
//   Z v_i = S^_i - (E x B)_i,  Z = tau^ + D^ + p - (E^2+B^2)/2                [Eq. 44]
//   rho = D^/W, p = (Gamma-1)/Gamma (Z/W^2 - rho)                             [Eq. 45-49]
// found by eliminating E from the momentum relation: for frozen scalars (s, kE = v.E), with
// r = s/(1+s), N = S^ - (Estar^ x B)/(1+s), A = Z + r B^2, c = r kE:
//   v_par = N_par / Z (component along B),  v_perp = (A N_perp + c B x N_perp)/(A^2 + c^2 B^2)
// then W(v), E(v) by the closed form, and the scalar residual
//   g(Z) = Z - [tau^ + D^ + p - (E^2+B^2)/2]
// is driven to zero by a bracketed secant/bisection on Z in [D^, Gamma (tau^ + D^ - B^2/2)]
// (both bounds rigorous; v^2 >= 1 counts as g < 0).  An outer fixed point updates (s, kE) from the
// new v until |dW|/W and |d kE| are below tol.  With adt = 0: s = 0, one inner solve.
struct C2PWork {
  const Metric* m; double Gamma, Dh, tauh, B2, s, kE, r;
  double EstarU[3], BU[3], BD[3];
  double NparU[3], NperpU[3], BxNperpU[3];
  // last evaluation
  double vU[3], EU[3], W, rho, p;
};
// residual g(Z) for frozen (s, kE); returns false when v^2 >= 1 (treated as g = -infinity)
bool c2p_residual(C2PWork& w, double Z, double* g) {
  FLOP_REGION(R_C2P_EVAL);
  const Metric& m = *w.m;
  const double A = Z + w.r * w.B2, c = w.r * w.kE;
  const double den = A * A + c * c * w.B2;
  for (int i = 0; i < 3; ++i) w.vU[i] = w.NparU[i] / Z + (A * w.NperpU[i] + c * w.BxNperpU[i]) / den;
  double vD[3]; lower(m, w.vU, vD);
  const double v2 = dotUD(w.vU, vD);
  if (!(v2 < 1.0)) return false;
  w.W = 1.0 / std::sqrt(1.0 - v2);
  double vxB_U[3]; crossU(m, vD, w.BD, vxB_U);
  for (int i = 0; i < 3; ++i) w.EU[i] = (w.EstarU[i] - w.s * vxB_U[i] + w.s * w.kE * w.vU[i]) / (1.0 + w.s);
  double ED[3]; lower(m, w.EU, ED);
  const double E2 = dotUD(w.EU, ED);
  w.rho = w.Dh / w.W;
  w.p = (w.Gamma - 1.0) / w.Gamma * (Z / (w.W * w.W) - w.rho);
  *g = Z - (w.tauh + w.Dh + w.p - 0.5 * (E2 + w.B2));
  return true;
}

C2PResult c2p_robust(const Metric& m, double Gamma, const double U[NCONS], double adt, double sigma,
                     double tol, int maxit, double P[NPRIM] /* in: guess (rho, p, v); out: primitives */) {
  FLOP_REGION(R_C2P_SETUP);
  C2PWork w;
  w.m = &m; w.Gamma = Gamma;
  const double sg = m.sqrtg;
  w.Dh = U[CD] / sg; w.tauh = U[CTAU] / sg;
  const double ShD[3] = {U[CSX] / sg, U[CSY] / sg, U[CSZ] / sg};
  double ShU[3]; raise(m, ShD, ShU);
  double EstarD[3];
  for (int i = 0; i < 3; ++i) { w.EstarU[i] = U[CEX + i] / sg; w.BU[i] = U[CBX + i] / sg; }
  lower(m, w.BU, w.BD); lower(m, w.EstarU, EstarD);
  w.B2 = dotUD(w.BU, w.BD);
  double EsxB_U[3]; crossU(m, EstarD, w.BD, EsxB_U);
  const double s0 = adt * m.alpha * sigma;
  const double escale = std::sqrt(dotUD(w.EstarU, EstarD) + w.B2);
  C2PResult res = {0, 1};
  // EM fields that do not depend on the solve
  for (int i = 0; i < 3; ++i) P[BX + i] = w.BU[i];
  P[PSI] = U[CPSI] / sg; P[PHI] = U[CPHI] / sg; P[QCH] = U[CQ] / sg;
  const double Zlo = w.Dh, Zhi = Gamma * (w.tauh + w.Dh - 0.5 * w.B2);
  // guess
  double vgU[3] = {P[VX], P[VY], P[VZ]}, vgD[3];
  lower(m, vgU, vgD);
  double v2g = dotUD(vgU, vgD);
  if (!(v2g < 1.0)) { vgU[0] = vgU[1] = vgU[2] = 0; vgD[0] = vgD[1] = vgD[2] = 0; v2g = 0; }
  double W = 1.0 / std::sqrt(1.0 - v2g);
  double kE = dotUD(vgU, EstarD) / (1.0 + s0 * W / (W * W));
  if (!(w.Dh > 0.0) || !(Zhi > Zlo)) {            // no physical bracket: keep the guess, E from the guess v
    implicit_E_closed(m, vgU, W, s0 * W, w.EstarU, w.BD, &P[EX]);
    return res;
  }
  double Z = (P[RHO] + Gamma / (Gamma - 1.0) * P[PRS]) * W * W;
  bool converged = false, state_ok = false;
  const int max_outer = 50;
  double fW_prev = 0, fk_prev = 0, GW_prev = 0, Gk_prev = 0, slope = 1.0, step_prev = 0.0;
  for (int outer = 0; outer < max_outer && res.evals < maxit; ++outer) {
    w.s = s0 * W; w.r = w.s / (1.0 + w.s); w.kE = kE;
    double NU[3], ND[3];
    for (int i = 0; i < 3; ++i) NU[i] = ShU[i] - EsxB_U[i] / (1.0 + w.s);
    lower(m, NU, ND);
    const double NdotB = dotUD(NU, w.BD);
    for (int i = 0; i < 3; ++i) {
      w.NparU[i] = (w.B2 > 0.0) ? NdotB / w.B2 * w.BU[i] : 0.0;
      w.NperpU[i] = NU[i] - w.NparU[i];
    }
    double NperpD[3]; lower(m, w.NperpU, NperpD);
    crossU(m, w.BD, NperpD, w.BxNperpU);
    // ---- inner: bracketed secant / bisection on Z; invariant g(a) < 0 < g(b) -------------------
    // `slope` (the running secant estimate of dg/dZ, 1 at the start) is kept across outer passes.
    double a = Zlo, b = Zhi;
    double x = std::min(std::max(Z, a), b), f = 0, xp = 0, fp = 0;
    bool ok = c2p_residual(w, x, &f), okp = false, inner_conv = false;
    ++res.evals;
    for (;;) {                                       // w holds the state evaluated at x
      if (ok && f == 0.0) { inner_conv = true; break; }
      if (!ok || f < 0.0) a = x; else b = x;
      if (ok && okp && f != fp && x != xp) slope = (f - fp) / (x - xp);
      const double delta = ok ? f / slope : 0.0;     // predicted distance to the root
      if (ok && std::fabs(delta) <= tol * std::fabs(x)) { inner_conv = true; break; }
      if (ok && (b - a) <= tol * std::fabs(x)) { inner_conv = true; break; }
      if (res.evals >= maxit) break;
      double xn = ok ? x - delta : 0.5 * (a + b);
      if (!(xn > a && xn < b)) xn = 0.5 * (a + b);   // bisection safeguard
      xp = x; fp = f; okp = ok;
      x = xn; ok = c2p_residual(w, x, &f); ++res.evals;
    }
    Z = x; state_ok = ok;
    if (!inner_conv || !ok) break;
    // ---- outer: update (s, kE) from the new v ----------------------------------------------------
    const double Wnew = w.W;
    const double kEnew = dotUD(w.vU, EstarD) / (1.0 + s0 * Wnew / (Wnew * Wnew));
    const bool same = std::fabs(Wnew - W) <= tol * Wnew && std::fabs(kEnew - kE) <= tol * escale;
    if (s0 == 0.0 || same) { W = Wnew; kE = kEnew; converged = true; break; }
    // round-off stagnation (same rule as c2p_plain): the fixed-point residual has stopped shrinking below 1000 tol
    const double step = std::max(std::fabs(Wnew - W) / Wnew, escale > 0.0 ? std::fabs(kEnew - kE) / escale : 0.0);
    if (outer >= 2 && step >= step_prev && step <= 1000.0 * tol) { W = Wnew; kE = kEnew; converged = true; break; }
    step_prev = step;
    // Anderson(1) acceleration of the fixed point x -> G(x), x = (W, kE/escale): with the residuals
    // f_n = G(x_n) - x_n,  x_{n+1} = G(x_n) - theta (G(x_n) - G(x_{n-1})),
    // theta = f_n.(f_n - f_{n-1}) / |f_n - f_{n-1}|^2   (the secant method when one component dominates).
    const double es = escale > 0.0 ? escale : 1.0;
    const double fW = Wnew - W, fk = (kEnew - kE) / es;
    double Wnext = Wnew, knext = kEnew;
    if (outer > 0) {
      const double dW = fW - fW_prev, dk = fk - fk_prev, den = dW * dW + dk * dk;
      if (den > 0.0) {
        const double theta = (fW * dW + fk * dk) / den;
        const double Wa = Wnew - theta * (Wnew - GW_prev), ka = kEnew - theta * (kEnew - Gk_prev);
        if (std::isfinite(Wa) && std::isfinite(ka) && Wa >= 1.0 && std::fabs(theta) < 10.0) { Wnext = Wa; knext = ka; }
      }
    }
    fW_prev = fW; fk_prev = fk; GW_prev = Wnew; Gk_prev = kEnew;
    W = Wnext; kE = knext;
  }
  res.failed = converged ? 0 : 1;
  if (state_ok) {
    P[RHO] = w.rho; P[PRS] = w.p;
    for (int i = 0; i < 3; ++i) { P[VX + i] = w.vU[i]; P[EX + i] = w.EU[i]; }
  } else {
    implicit_E_closed(m, vgU, 1.0 / std::sqrt(1.0 - v2g), s0 / std::sqrt(1.0 - v2g), w.EstarU, w.BD, &P[EX]);
  }
  return res;
}

// (plain; the solver the parity runs use)  The SAME defining system as above -- Eq. 42,
// Eq. 44-49, readings R7/R8 -- solved the dull way, so that it can be checked by eye
// and shares no iteration logic with the CUDA kernel:
//   outer: plain fixed point on (W, kE): freeze s = adt alpha sigma W and kE = v.E, solve the inner
//          problem, replace (W, kE) by the values of the new v; no acceleration.  Stop when
//          |dW| <= tol W and |d kE| <= tol |(E*^, B)|, or when the steps have stopped shrinking below
//          1000 tol (round-off stagnation), or after `max_outer` passes (failure).
//   inner: plain bisection of g(Z) (c2p_residual) on the rigorous bracket [D^, Gamma(tau^ + D^ - B^2/2)]
//          (g increasing; v^2 >= 1 counts as g < 0), started from the full bracket in EVERY pass, until
//          the bracket is <= 4 ulp wide; the midpoint of the last bracket is the root.
// No secant, no kept slope, no safeguard logic, no Anderson mixing.  With adt = 0 or sigma = 0 the outer
// loop is one pass.  No physical bracket (D^ <= 0 or Zhi <= Zlo): failure; rho, p, v keep the guess and
// E is the closed form of Eq. 42 at the guess velocity.
C2PResult c2p_plain(const Metric& m, double Gamma, const double U[NCONS], double adt, double sigma,
                    double tol, int max_outer, double P[NPRIM] /* in: guess (v); out: primitives */) {
  FLOP_REGION(R_C2P_SETUP);
  C2PWork w;
  w.m = &m; w.Gamma = Gamma;
  const double sg = m.sqrtg;
  w.Dh = U[CD] / sg; w.tauh = U[CTAU] / sg;
  const double ShD[3] = {U[CSX] / sg, U[CSY] / sg, U[CSZ] / sg};
  double ShU[3]; raise(m, ShD, ShU);
  double EstarD[3];
  for (int i = 0; i < 3; ++i) { w.EstarU[i] = U[CEX + i] / sg; w.BU[i] = U[CBX + i] / sg; }
  lower(m, w.BU, w.BD); lower(m, w.EstarU, EstarD);
  w.B2 = dotUD(w.BU, w.BD);
  double EsxB_U[3]; crossU(m, EstarD, w.BD, EsxB_U);
  const double s0 = adt * m.alpha * sigma;
  const double escale = std::sqrt(dotUD(w.EstarU, EstarD) + w.B2);
  C2PResult res = {0, 1};
  for (int i = 0; i < 3; ++i) P[BX + i] = w.BU[i];
  P[PSI] = U[CPSI] / sg; P[PHI] = U[CPHI] / sg; P[QCH] = U[CQ] / sg;
  const double Zlo = w.Dh, Zhi = Gamma * (w.tauh + w.Dh - 0.5 * w.B2);
  // (W, kE) of the guess velocity
  double vgU[3] = {P[VX], P[VY], P[VZ]}, vgD[3];
  lower(m, vgU, vgD);
  double v2g = dotUD(vgU, vgD);
  if (!(v2g < 1.0)) { vgU[0] = vgU[1] = vgU[2] = 0; vgD[0] = vgD[1] = vgD[2] = 0; v2g = 0; }
  double W = 1.0 / std::sqrt(1.0 - v2g);
  double kE = dotUD(vgU, EstarD) / (1.0 + s0 * W / (W * W));
  if (!(w.Dh > 0.0) || !(Zhi > Zlo)) {
    implicit_E_closed(m, vgU, W, s0 * W, w.EstarU, w.BD, &P[EX]);
    return res;
  }
  bool converged = false, ok = false;
  double step_prev = 0.0;
  for (int outer = 0; outer < max_outer; ++outer) {
    w.s = s0 * W; w.r = w.s / (1.0 + w.s); w.kE = kE;
    double NU[3], ND[3];
    for (int i = 0; i < 3; ++i) NU[i] = ShU[i] - EsxB_U[i] / (1.0 + w.s);
    lower(m, NU, ND);
    const double NdotB = dotUD(NU, w.BD);
    for (int i = 0; i < 3; ++i) {
      w.NparU[i] = (w.B2 > 0.0) ? NdotB / w.B2 * w.BU[i] : 0.0;
      w.NperpU[i] = NU[i] - w.NparU[i];
    }
    double NperpD[3]; lower(m, w.NperpU, NperpD);
    crossU(m, w.BD, NperpD, w.BxNperpU);
    // inner: bisection, invariant g(a) < 0 < g(b)
    double a = Zlo, b = Zhi, g = 0;
    for (;;) {
      const double mid = 0.5 * (a + b);
      if (!(mid > a && mid < b)) break;
      if (b - a <= 4.0 * std::numeric_limits<double>::epsilon() * std::fabs(mid)) break;
      const bool okm = c2p_residual(w, mid, &g); ++res.evals;
      if (okm && g == 0.0) { a = b = mid; break; }
      if (!okm || g < 0.0) a = mid; else b = mid;
    }
    ok = c2p_residual(w, 0.5 * (a + b), &g); ++res.evals;    // w now holds the state at the root
    if (!ok) break;
    const double Wnew = w.W;
    const double kEnew = dotUD(w.vU, EstarD) / (1.0 + s0 * Wnew / (Wnew * Wnew));
    // size of this pass's step, in units of the scales the tolerance refers to
    const double step = std::max(std::fabs(Wnew - W) / Wnew, escale > 0.0 ? std::fabs(kEnew - kE) / escale : 0.0);
    W = Wnew; kE = kEnew;
    if (s0 == 0.0 || step <= tol) { converged = true; break; }
    // round-off stagnation: a contraction's steps shrink until the 4-ulp noise of the inner bisection
    // (amplified by the conditioning of strongly magnetised states) takes over; once a step is no smaller
    // than the one before AND below 1000 tol, the fixed point has been reached as well as FP64 defines it
    if (outer >= 2 && step >= step_prev && step <= 1000.0 * tol) { converged = true; break; }
    step_prev = step;
  }
  res.failed = converged ? 0 : 1;
  if (ok) {
    P[RHO] = w.rho; P[PRS] = w.p;
    for (int i = 0; i < 3; ++i) { P[VX + i] = w.vU[i]; P[EX + i] = w.EU[i]; }
  } else {
    implicit_E_closed(m, vgU, 1.0 / std::sqrt(1.0 - v2g), s0 / std::sqrt(1.0 - v2g), w.EstarU, w.BD, &P[EX]);
  }
  return res;
}

// ---------------------------------------------------------------------------------------------
// grid container
// ---------------------------------------------------------------------------------------------
enum { SOLVER_PLAIN = 0, SOLVER_ROBUST = 1 };
enum { PLAIN_MAX_OUTER = 2000 };   // passes of the un-accelerated outer fixed point before a solve counts as failed
struct Grid {
  Params par;
  int solver = SOLVER_PLAIN;   // which root finder solve_all uses (oracle_set_solver)
  int np[3], g[3];           // padded sizes, ghost offsets
  long ntot;
  bool have_metric = false, have_prims = false, have_sigma = false;
  std::vector<double> met[NMET], sigma;
  std::vector<double> P[NPRIM], jc[3], jc1[3];       // primitives; conduction current of the current stage / of stage 1
  std::vector<double> Un[NCONS], Us[NCONS];          // U^n ; stage vector U*
  std::vector<double> F1[NCONS], F2[NCONS];          // F[U^(1)], F[U^(2)]
  std::vector<double> X1[3], X2[3];                  // stage electric fields calE^(1), calE^(2)
  std::vector<double> Xs2[3];                        // calE*^(2)
  // stats
  long long solves = 0, evals = 0, failures = 0, floors = 0, face_fixups = 0; int max_evals = 0;

  long idx(int i, int j, int k) const { return (long)(i + g[0]) + (long)np[0] * ((long)(j + g[1]) + (long)np[1] * (long)(k + g[2])); }
  bool active(int d) const { return par.n[d] > 1; }
};

void metric_at(const Grid& G, long c, Metric& m) {
  m.alpha = G.met[MALP][c];
  for (int i = 0; i < 3; ++i) m.betaU[i] = G.met[MBX + i][c];
  m.gDD[0][0] = G.met[MGXX][c]; m.gDD[0][1] = m.gDD[1][0] = G.met[MGXY][c]; m.gDD[0][2] = m.gDD[2][0] = G.met[MGXZ][c];
  m.gDD[1][1] = G.met[MGYY][c]; m.gDD[1][2] = m.gDD[2][1] = G.met[MGYZ][c]; m.gDD[2][2] = G.met[MGZZ][c];
  m.KDD[0][0] = G.met[MKXX][c]; m.KDD[0][1] = m.KDD[1][0] = G.met[MKXY][c]; m.KDD[0][2] = m.KDD[2][0] = G.met[MKXZ][c];
  m.KDD[1][1] = G.met[MKYY][c]; m.KDD[1][2] = m.KDD[2][1] = G.met[MKYZ][c]; m.KDD[2][2] = G.met[MKZZ][c];
  metric_finish(m);
}
// O1 (reading R2): face metric = arithmetic mean of alpha, beta^i, gamma_ij of the two adjacent cell
// centres; sqrt(gamma) and gamma^ij from the averaged gamma_ij.
void metric_face(const Grid& G, long cL, long cR, Metric& m) {
  m.alpha = 0.5 * (G.met[MALP][cL] + G.met[MALP][cR]);
  for (int i = 0; i < 3; ++i) m.betaU[i] = 0.5 * (G.met[MBX + i][cL] + G.met[MBX + i][cR]);
  double g6[6];
  for (int q = 0; q < 6; ++q) g6[q] = 0.5 * (G.met[MGXX + q][cL] + G.met[MGXX + q][cR]);
  m.gDD[0][0] = g6[0]; m.gDD[0][1] = m.gDD[1][0] = g6[1]; m.gDD[0][2] = m.gDD[2][0] = g6[2];
  m.gDD[1][1] = g6[3]; m.gDD[1][2] = m.gDD[2][1] = g6[4]; m.gDD[2][2] = g6[5];
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) m.KDD[i][j] = 0.0;
  metric_finish(m);
}

// ---------------------------------------------------------------------------------------------
// A9. characteristic speeds "used in ideal GRMHD" (reading R16).  The ideal-GRMHD HLLE solvers
// bound the fast magnetosonic speed in the fluid frame by
//   a^2 = cs^2 + vA^2 - cs^2 vA^2,   cs^2 = Gamma p / h (Eq. 50 in reading G3),   vA^2 = b^2/(h + b^2),
//   b^2 = B^2/W^2 + (B.v)^2  (comoving field of ideal MHD; h = enthalpy density)
// and boost it to the Eulerian coordinate frame along direction k:
//   lambda+- = alpha [ v^k (1 - a^2) +- sqrt( a^2 (1 - v^2) [ gamma^kk (1 - v^2 a^2) - v^k v^k (1 - a^2) ] ) ] / (1 - v^2 a^2) - beta^k.
// With a = 1 this is Eq. 30's light cone, +-alpha sqrt(gamma^kk) - beta^k.
// ---------------------------------------------------------------------------------------------
void mhd_wave_speeds(const Metric& m, double Gamma, int k, const double P[NPRIM], double* lam_minus, double* lam_plus) {
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], BD[3];
  lower(m, vU, vD); lower(m, BU, BD);
  const double v2 = dotUD(vU, vD), B2 = dotUD(BU, BD), Bv = dotUD(BU, vD);
  const double h = rho * (1.0 + p / ((Gamma - 1.0) * rho)) + p;
  const double b2 = B2 * (1.0 - v2) + Bv * Bv;
  const double cs2 = Gamma * p / h, vA2 = b2 / (h + b2);
  const double a2 = cs2 + vA2 - cs2 * vA2;
  const double den = 1.0 - v2 * a2;
  const double disc = a2 * (1.0 - v2) * (m.gUU[k][k] * den - vU[k] * vU[k] * (1.0 - a2));
  const double root = std::sqrt(std::max(disc, 0.0));
  *lam_plus = m.alpha * (vU[k] * (1.0 - a2) + root) / den - m.betaU[k];
  *lam_minus = m.alpha * (vU[k] * (1.0 - a2) - root) / den - m.betaU[k];
}

// ---------------------------------------------------------------------------------------------
// a1. ghost fill ("copied from the nearest interior point"; PAPER.md:359 periodic);
//     x, then y, then z, each over the full padded extent of the other directions (reading R10).
// ---------------------------------------------------------------------------------------------
void ghost_fill_field(const Grid& G, std::vector<double>& f) {
  for (int d = 0; d < 3; ++d) {
    if (!G.active(d)) continue;
    const int n = G.par.n[d], ng = G.par.ng;
    // ranges of the other two directions: full padded extent
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) { lo[e] = -G.g[e]; hi[e] = G.par.n[e] + G.g[e]; }
    for (int gi = 1; gi <= ng; ++gi) {
      for (int side = 0; side < 2; ++side) {
        const int dst = side == 0 ? -gi : n - 1 + gi;
        int src;
        if (G.par.bc[d] == BC_PERIODIC) src = side == 0 ? n - gi : gi - 1;
        else src = side == 0 ? 0 : n - 1;
        int a[3];
        for (a[2] = (d == 2 ? 0 : lo[2]); a[2] < (d == 2 ? 1 : hi[2]); ++a[2])
          for (a[1] = (d == 1 ? 0 : lo[1]); a[1] < (d == 1 ? 1 : hi[1]); ++a[1])
            for (a[0] = (d == 0 ? 0 : lo[0]); a[0] < (d == 0 ? 1 : hi[0]); ++a[0]) {
              int s[3] = {a[0], a[1], a[2]}, t[3] = {a[0], a[1], a[2]};
              s[d] = src; t[d] = dst;
              f[G.idx(t[0], t[1], t[2])] = f[G.idx(s[0], s[1], s[2])];
            }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// a2+a3. HLLE flux at the lower face (index -1/2 in direction d) of cell (i,j,k)
//   PAPER.md:171-173, Eq. 30 (reading R6: lambda+- = +-alpha sqrt(gamma^kk) - beta^k, clipped)
// ---------------------------------------------------------------------------------------------
void face_state(const Grid& G, int scheme, int d, int i, int j, int k, int which /*0: at -1/2, 1: at +1/2*/,
                double Pf[NPRIM], double* jck, int* fixups) {
  int o[3] = {0, 0, 0}; o[d] = 1;
  long c[5];
  for (int q = -2; q <= 2; ++q) c[q + 2] = G.idx(i + q * o[0], j + q * o[1], k + q * o[2]);
  for (int v = 0; v <= NPRIM; ++v) {
    const std::vector<double>& f = (v < NPRIM) ? G.P[v] : G.jc[d];
    double lo_face, hi_face;
    recon_cell(scheme, G.par.weno_eps, f[c[0]], f[c[1]], f[c[2]], f[c[3]], f[c[4]], &lo_face, &hi_face);
    const double val = which ? hi_face : lo_face;
    if (v < NPRIM) Pf[v] = val; else *jck = val;
  }
  // reading R4: unphysical face values fall back to the cell value
  if (!(Pf[RHO] > 0.0)) { Pf[RHO] = G.P[RHO][c[2]]; ++*fixups; }
  if (!(Pf[PRS] > 0.0)) { Pf[PRS] = G.P[PRS][c[2]]; ++*fixups; }
}

// the two states of the Riemann problem at the lower face (index -1/2 in direction d) of cell (i,j,k), after the
// fix-ups of reading R4 (rho, p fallback above; |v| limited with the FACE metric mf); returns the number of fix-ups
int face_states(const Grid& G, int scheme, int d, int i, int j, int k, const Metric& mf, double PL[NPRIM],
                double PR[NPRIM], double* jL, double* jR) {
  int o[3] = {0, 0, 0}; o[d] = 1;
  int fixups = 0;
  face_state(G, scheme, d, i - o[0], j - o[1], k - o[2], 1, PL, jL, &fixups);      // left cell's value at its +1/2 face
  face_state(G, scheme, d, i, j, k, 0, PR, jR, &fixups);                          // right cell's value at its -1/2 face
  double* Ps[2] = {PL, PR};
  for (int sd = 0; sd < 2; ++sd) {
    double vU[3] = {Ps[sd][VX], Ps[sd][VY], Ps[sd][VZ]}, vD[3];
    lower(mf, vU, vD);
    const double v2 = dotUD(vU, vD), v2max = 1.0 - 1e-10;
    if (v2 >= v2max) { const double f = std::sqrt(v2max / v2); for (int q = 0; q < 3; ++q) Ps[sd][VX + q] *= f; ++fixups; }
  }
  return fixups;
}

int hlle_face(const Grid& G, int scheme, int d, int i, int j, int k, double Fh[NCONS]) {
  FLOP_REGION(R_RIEMANN);
  int o[3] = {0, 0, 0}; o[d] = 1;
  const int il = i - o[0], jl = j - o[1], kl = k - o[2];
  const long cL = G.idx(il, jl, kl), cR = G.idx(i, j, k);
  Metric mf; metric_face(G, cL, cR, mf);
  double PL[NPRIM], PR[NPRIM], jL, jR;
  const int fixups = face_states(G, scheme, d, i, j, k, mf, PL, PR, &jL, &jR);
  double sigL = 0, sigR = 0;
  if (G.par.charge_mode == CHARGE_FACE_OHM) {            // reading R6b: piecewise-constant sigma
    Metric mL, mR; metric_at(G, cL, mL); metric_at(G, cR, mR);
    double vD[3], vU[3];
    for (int q = 0; q < 3; ++q) vU[q] = G.P[VX + q][cL];
    lower(mL, vU, vD);
    double W = 1.0 / std::sqrt(1.0 - dotUD(vU, vD));
    sigL = sigma_of(G.par, G.P[RHO][cL] * W, G.have_sigma ? G.sigma[cL] : 0.0);
    for (int q = 0; q < 3; ++q) vU[q] = G.P[VX + q][cR];
    lower(mR, vU, vD);
    W = 1.0 / std::sqrt(1.0 - dotUD(vU, vD));
    sigR = sigma_of(G.par, G.P[RHO][cR] * W, G.have_sigma ? G.sigma[cR] : 0.0);
  }
  double UL[NCONS], FL[NCONS], UR[NCONS], FR[NCONS];
  state_flux(mf, G.par.Gamma, d, PL, G.par.charge_mode, sigL, jL, UL, FL);
  state_flux(mf, G.par.Gamma, d, PR, G.par.charge_mode, sigR, jR, UR, FR);
  double lp, lm;
  if (G.par.wave_speed_mode == WAVE_MHD_INSIDE && PL[RHO] > G.par.wave_rho_switch && PR[RHO] > G.par.wave_rho_switch) {
    // reading R16: "inside the star" = both face states denser than wave_rho_switch; the ideal-GRMHD bound of
    // both states, HLLE's usual envelope
    double lmL, lpL, lmR, lpR;
    mhd_wave_speeds(mf, G.par.Gamma, d, PL, &lmL, &lpL);
    mhd_wave_speeds(mf, G.par.Gamma, d, PR, &lmR, &lpR);
    lp = std::max(0.0, std::max(lpL, lpR));
    lm = std::min(0.0, std::min(lmL, lmR));
  } else {
    const double c = mf.alpha * std::sqrt(mf.gUU[d][d]);
    lp = std::max(0.0, c - mf.betaU[d]);
    lm = std::min(0.0, -c - mf.betaU[d]);
  }
  for (int v = 0; v < NCONS; ++v) Fh[v] = (lp * FL[v] - lm * FR[v] + lp * lm * (UR[v] - UL[v])) / (lp - lm);
  return fixups;
}

// ---------------------------------------------------------------------------------------------
// a4 (second half). explicit sources at a cell centre (Eq. 27 S; PAPER.md:222-224
//   Eq. 39-40) in the reading R1/R9; metric derivatives 4th-order centred (R2).
// ---------------------------------------------------------------------------------------------
inline double d4(const std::vector<double>& f, long c, long stride, double dx) {
  return (-f[c + 2 * stride] + 8.0 * f[c + stride] - 8.0 * f[c - stride] + f[c - 2 * stride]) / (12.0 * dx);
}
void sources_cell(const Grid& G, int i, int j, int k, double S[NCONS]) {
  FLOP_REGION(R_SOURCES);
  const long c = G.idx(i, j, k);
  const long stride[3] = {1, (long)G.np[0], (long)G.np[0] * G.np[1]};
  Metric m; metric_at(G, c, m);
  double dalpha[3], dbeta[3][3], dg[3][3][3];   // dalpha[k]=d_k alpha; dbeta[k][i]=d_k beta^i; dg[k][i][j]=d_k gamma_ij
  static const int sym[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};
  for (int kk = 0; kk < 3; ++kk) {
    if (!G.active(kk)) {
      dalpha[kk] = 0;
      for (int a = 0; a < 3; ++a) { dbeta[kk][a] = 0; for (int b = 0; b < 3; ++b) dg[kk][a][b] = 0; }
      continue;
    }
    dalpha[kk] = d4(G.met[MALP], c, stride[kk], G.par.dx[kk]);
    for (int a = 0; a < 3; ++a) dbeta[kk][a] = d4(G.met[MBX + a], c, stride[kk], G.par.dx[kk]);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) dg[kk][a][b] = d4(G.met[MGXX + sym[a][b]], c, stride[kk], G.par.dx[kk]);
  }
  double P[NPRIM], U[NCONS];
  for (int v = 0; v < NPRIM; ++v) P[v] = G.P[v][c];
  prim2cons_point(m, G.par.Gamma, P, U);
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  const double v2 = dotUD(vU, vD), W = 1.0 / std::sqrt(1.0 - v2);
  const double h = rho * (1.0 + p / ((G.par.Gamma - 1.0) * rho)) + p;
  const double E2 = dotUD(EU, ED), B2 = dotUD(BU, BD);
  double TUU[3][3];
  for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
    TUU[a][b] = h * W * W * vU[a] * vU[b] + m.gUU[a][b] * p - EU[a] * EU[b] - BU[a] * BU[b] + 0.5 * m.gUU[a][b] * (E2 + B2);
  const double al = m.alpha, sg = m.sqrtg;
  const double SD[3] = {U[CSX], U[CSY], U[CSZ]};
  double SU[3]; raise(m, SD, SU);
  S[CD] = 0.0; S[CQ] = 0.0;
  for (int a = 0; a < 3; ++a) {
    double t1 = 0, t2 = 0;
    for (int b = 0; b < 3; ++b) { t2 += SD[b] * dbeta[a][b]; for (int cc = 0; cc < 3; ++cc) t1 += TUU[b][cc] * dg[a][b][cc]; }
    S[CSX + a] = 0.5 * al * sg * t1 + t2 - (U[CTAU] + U[CD]) * dalpha[a];
  }
  {
    double t1 = 0, t2 = 0;
    for (int a = 0; a < 3; ++a) { t2 += SU[a] * dalpha[a]; for (int b = 0; b < 3; ++b) t1 += TUU[a][b] * m.KDD[a][b]; }
    S[CTAU] = al * sg * t1 - t2;
  }
  // G^i = gamma^ij d_j alpha - alpha gamma^jk Gamma^i_jk,  gamma^jk Gamma^i_jk = gamma^il gamma^jk (d_j gamma_lk - 1/2 d_l gamma_jk)
  double Gi[3];
  for (int a = 0; a < 3; ++a) {
    double t1 = 0, t2 = 0;
    for (int b = 0; b < 3; ++b) t1 += m.gUU[a][b] * dalpha[b];
    for (int l = 0; l < 3; ++l) for (int b = 0; b < 3; ++b) for (int cc = 0; cc < 3; ++cc)
      t2 += m.gUU[a][l] * m.gUU[b][cc] * (dg[b][l][cc] - 0.5 * dg[l][b][cc]);
    Gi[a] = t1 - al * t2;
  }
  double trK = 0;
  for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) trK += m.gUU[a][b] * m.KDD[a][b];
  for (int a = 0; a < 3; ++a) {
    double tB = 0, tE = 0;
    for (int kk = 0; kk < 3; ++kk) { tB += U[CBX + kk] * dbeta[kk][a]; tE += U[CEX + kk] * dbeta[kk][a]; }
    S[CBX + a] = -tB + U[CPHI] * Gi[a];
    S[CEX + a] = -tE + U[CPSI] * Gi[a] - al * U[CQ] * vU[a];
  }
  double BdA = 0, EdA = 0;
  for (int kk = 0; kk < 3; ++kk) { BdA += U[CBX + kk] * dalpha[kk]; EdA += U[CEX + kk] * dalpha[kk]; }
  S[CPHI] = -al * U[CPHI] * trK + BdA - al * G.par.kappa * U[CPHI];
  S[CPSI] = -al * U[CPSI] * trK + EdA + al * U[CQ] - al * G.par.kappa * U[CPSI];
}

// F[U] of Eq. 31/39-40 for every interior cell: -sum_k (F^k_{+1/2} - F^k_{-1/2})/dx^k + S
void rhs_all(Grid& G, int scheme, std::vector<double> Fout[NCONS]) {
  FLOP_REGION(R_DIVERGENCE);
  const int nx = G.par.n[0], ny = G.par.n[1], nz = G.par.n[2];
  for (int v = 0; v < NCONS; ++v) std::fill(Fout[v].begin(), Fout[v].end(), 0.0);
  std::vector<double> Fh[NCONS];
  for (int v = 0; v < NCONS; ++v) Fh[v].assign(G.ntot, 0.0);
  long long fixups = 0;
  for (int d = 0; d < 3; ++d) {
    if (!G.active(d)) continue;
    int o[3] = {0, 0, 0}; o[d] = 1;
    // faces at the lower side of cells 0..n (inclusive) in direction d
#pragma omp parallel for collapse(3) schedule(static) reduction(+ : fixups)
    for (int k = 0; k < nz + o[2]; ++k)
      for (int j = 0; j < ny + o[1]; ++j)
        for (int i = 0; i < nx + o[0]; ++i) {
          double f[NCONS];
          fixups += hlle_face(G, scheme, d, i, j, k, f);
          const long c = G.idx(i, j, k);
          for (int v = 0; v < NCONS; ++v) Fh[v][c] = f[v];
        }
#pragma omp parallel for collapse(3) schedule(static)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const long c = G.idx(i, j, k), cp = G.idx(i + o[0], j + o[1], k + o[2]);
          for (int v = 0; v < NCONS; ++v) Fout[v][c] -= (Fh[v][cp] - Fh[v][c]) / G.par.dx[d];
        }
  }
#pragma omp parallel for collapse(3) schedule(static)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        double S[NCONS];
        sources_cell(G, i, j, k, S);
        const long c = G.idx(i, j, k);
        for (int v = 0; v < NCONS; ++v) Fout[v][c] += S[v];
      }
  G.face_fixups += fixups;
}

// ---------------------------------------------------------------------------------------------
// a6 over the grid: solve every interior cell of the stage vector Ust (its calE entries are X*),
// guess = current G.P; writes G.P, the stage calE = sqrt(gamma) E into Xout, and the undensitised
// conduction current jc^i = (E*^ - E)/(adt alpha) (reading R3, charge_mode CELL_CURRENT) into G.jc.
// Floor rule: reading R9.
// ---------------------------------------------------------------------------------------------
void solve_all(Grid& G, std::vector<double> Ust[NCONS], double adt, std::vector<double>* Xout, bool write_back_floor) {
  FLOP_REGION(R_C2P_SETUP);
  const int nx = G.par.n[0], ny = G.par.n[1], nz = G.par.n[2];
  long long evals = 0, failures = 0, floors = 0; int max_evals = 0;
#pragma omp parallel for collapse(3) schedule(static) reduction(+ : evals, failures, floors) reduction(max : max_evals)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const long c = G.idx(i, j, k);
        Metric m; metric_at(G, c, m);
        double U[NCONS], P[NPRIM];
        for (int v = 0; v < NCONS; ++v) U[v] = Ust[v][c];
        for (int v = 0; v < NPRIM; ++v) P[v] = G.P[v][c];
        const double Dh = U[CD] / m.sqrtg;
        const double sigma = (adt > 0.0) ? sigma_of(G.par, Dh, G.have_sigma ? G.sigma[c] : 0.0) : 0.0;
        C2PResult r = (G.solver == SOLVER_PLAIN)
                          ? c2p_plain(m, G.par.Gamma, U, adt, sigma, G.par.c2p_tol, PLAIN_MAX_OUTER, P)
                          : c2p_robust(m, G.par.Gamma, U, adt, sigma, G.par.c2p_tol, G.par.c2p_max_iter, P);
        evals += r.evals; failures += r.failed; max_evals = std::max(max_evals, r.evals);
        if (G.par.rho_floor > 0.0 && (r.failed || !(P[RHO] > G.par.rho_floor * (1.0 + 1e-3)))) {
          // reading R9: atmosphere reset -- rho = rho_floor, v = 0, p = K rho^Gamma; E from the
          // closed form at v = 0 (E = E*^/(1 + adt alpha sigma)); other EM fields kept
          ++floors;
          P[RHO] = G.par.rho_floor; P[VX] = P[VY] = P[VZ] = 0.0;
          P[PRS] = G.par.k_atmo * std::pow(G.par.rho_floor, G.par.Gamma);
          const double s = adt * m.alpha * sigma;
          for (int q = 0; q < 3; ++q) P[EX + q] = (U[CEX + q] / m.sqrtg) / (1.0 + s);
          if (write_back_floor) {
            double Unew[NCONS];
            prim2cons_point(m, G.par.Gamma, P, Unew);
            Ust[CD][c] = Unew[CD]; Ust[CTAU][c] = Unew[CTAU];
            for (int q = 0; q < 3; ++q) Ust[CSX + q][c] = Unew[CSX + q];
          }
        }
        for (int v = 0; v < NPRIM; ++v) G.P[v][c] = P[v];
        for (int q = 0; q < 3; ++q) {
          const double Xq = m.sqrtg * P[EX + q];
          if (Xout) Xout[q][c] = Xq;
          G.jc[q][c] = (adt > 0.0) ? (U[CEX + q] / m.sqrtg - P[EX + q]) / (adt * m.alpha) : 0.0;
        }
      }
  G.solves += (long long)nx * ny * nz; G.evals += evals; G.failures += failures; G.floors += floors;
  G.max_evals = std::max(G.max_evals, max_evals);
}

// ---------------------------------------------------------------------------------------------
// A22. charge_mode DIV_E: the charge density is not evolved but computed from the electric
// field of the stage, q = nabla_i E^i = d_i(sqrt(gamma) E^i)/sqrt(gamma).  Reading R15 (the paper names no
// stencil): second-order centred differences of calE^i = sqrt(gamma) E^i, inactive directions dropped.  Needs
// the ghost zones of E^i filled.  Writes q into P (interior) and, if asked, calQ = sqrt(gamma) q into Un.
// ---------------------------------------------------------------------------------------------
void charge_from_div_E(Grid& G, bool write_cons) {
  const int nx = G.par.n[0], ny = G.par.n[1], nz = G.par.n[2];
  const long stride[3] = {1, (long)G.np[0], (long)G.np[0] * G.np[1]};
#pragma omp parallel for collapse(3) schedule(static)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const long c = G.idx(i, j, k);
        Metric m; metric_at(G, c, m);
        double div = 0.0;
        for (int d = 0; d < 3; ++d) {
          if (!G.active(d)) continue;
          Metric mp, mm; metric_at(G, c + stride[d], mp); metric_at(G, c - stride[d], mm);
          div += (mp.sqrtg * G.P[EX + d][c + stride[d]] - mm.sqrtg * G.P[EX + d][c - stride[d]]) / (2.0 * G.par.dx[d]);
        }
        G.P[QCH][c] = div / m.sqrtg;
        if (write_cons) G.Un[CQ][c] = div;
      }
}

// ---------------------------------------------------------------------------------------------
// O2. one IMEX-SSP2(2,2,2) step (Eq. 35-37; gamma = 1 - 1/sqrt(2)).
//   Table I's body is missing from the text; Eq. 35-37 fix it: explicit A~=[[0,0],[1,0]], w~=(1/2,1/2);
//   implicit A=[[g,0],[1-2g,g]], w=(1/2,1/2).   X = calE^i (stiff), Y = the other 11.
//   R[U^(i)] is evaluated as the difference quotient (X^(i) - X*^(i))/(g dt) (reading R11).
// ---------------------------------------------------------------------------------------------
// after a stage's solve: ghost zones of the stage primitives and of the conduction current; in charge mode DIV_E
// the stage's charge density from its electric field (A22), ghost-filled in turn
void stage_ghosts_and_charge(Grid& G) {
  for (int v = 0; v < NPRIM; ++v) ghost_fill_field(G, G.P[v]);
  for (int q = 0; q < 3; ++q) ghost_fill_field(G, G.jc[q]);
  if (G.par.charge_mode == CHARGE_DIV_E) { charge_from_div_E(G, false); ghost_fill_field(G, G.P[QCH]); }
}
// charge mode DIV_E: the new state's q and calQ from its electric field
void final_charge(Grid& G) {
  if (G.par.charge_mode != CHARGE_DIV_E) return;
  for (int q = 0; q < 3; ++q) ghost_fill_field(G, G.P[EX + q]);
  charge_from_div_E(G, true);
}

void step(Grid& G, double dt, int scheme) {
  FLOP_REGION(R_COMBINE);
  const double gam = 1.0 - 1.0 / std::sqrt(2.0);
  const int nx = G.par.n[0], ny = G.par.n[1], nz = G.par.n[2];
  // stage 1 (Eq. 35): X*1 = X^n, Y1 = Y^n
  solve_all(G, G.Un, gam * dt, G.X1, false);
  for (int q = 0; q < 3; ++q) G.jc1[q] = G.jc[q];
  stage_ghosts_and_charge(G);
  rhs_all(G, scheme, G.F1);
  // stage 2 (Eq. 36)
#pragma omp parallel for collapse(3) schedule(static)
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    const long c = G.idx(i, j, k);
    for (int v = 0; v < NCONS; ++v) G.Us[v][c] = G.Un[v][c] + dt * G.F1[v][c];
    for (int q = 0; q < 3; ++q) {
      const double R1 = (G.X1[q][c] - G.Un[CEX + q][c]) / (gam * dt);
      G.Us[CEX + q][c] += dt * (1.0 - 2.0 * gam) * R1;
      G.Xs2[q][c] = G.Us[CEX + q][c];
    }
  }
  solve_all(G, G.Us, gam * dt, G.X2, false);
  stage_ghosts_and_charge(G);
  rhs_all(G, scheme, G.F2);
  // final combination (Eq. 37)
#pragma omp parallel for collapse(3) schedule(static)
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    const long c = G.idx(i, j, k);
    double Unew[NCONS];
    for (int v = 0; v < NCONS; ++v) Unew[v] = G.Un[v][c] + 0.5 * dt * (G.F1[v][c] + G.F2[v][c]);
    for (int q = 0; q < 3; ++q) {
      const double R1 = (G.X1[q][c] - G.Un[CEX + q][c]) / (gam * dt);
      const double R2 = (G.X2[q][c] - G.Xs2[q][c]) / (gam * dt);
      Unew[CEX + q] += 0.5 * dt * (R1 + R2);
    }
    for (int v = 0; v < NCONS; ++v) G.Un[v][c] = Unew[v];
  }
  // recovery of the new state at fixed calE (reading R12), guess = P^(2)
  solve_all(G, G.Un, 0.0, nullptr, true);
  final_charge(G);
}

// ---------------------------------------------------------------------------------------------
// A12. the other IMEX-RK SSP schemes the paper incorporates: SSP2(3,3,2), SSP3(3,3,2), SSP3(4,3,3),
// through the GENERAL form Eq. 32 with a double Butcher tableau (Eq. 33-34).  PAPER.md does not
// print these tableaux (refs [19], [31]); the coefficients below are the published Pareschi-Russo ones, PINNED by
// the order conditions they must satisfy (tests/test_oracle_imex_tableaux.py), not by trust.
//   U^(i)   = U^n + dt sum_{j<i} at_ij F[U^(j)] + dt sum_{j<=i} a_ij R[U^(j)]
//   U^{n+1} = U^n + dt sum_i wt_i F[U^(i)] + dt sum_i w_i R[U^(i)]
// with the split of PAPER.md:216 (R acts on X = calE only) and R^(i) = (X^(i) - X*^(i))/(a_ii dt) (reading R11),
// X*^(i) = the explicit part of the stage vector; the recovery of U^{n+1} at fixed calE (reading R12).
// A stage whose F is used by nobody (zero column in At and zero weight) is not evaluated.
// ---------------------------------------------------------------------------------------------
struct Tableau { int s; double At[4][4], wt[4], A[4][4], w[4]; };
enum { TIME_SSP2_222 = 0, TIME_SSP2_332 = 1, TIME_SSP3_332 = 2, TIME_SSP3_433 = 3, TIME_SSP2_222_GENERAL = 4 };

bool tableau_of(int time_scheme, Tableau& T) {
  std::memset(&T, 0, sizeof(T));
  const double g = 1.0 - 1.0 / std::sqrt(2.0);
  switch (time_scheme) {
    case TIME_SSP2_222: case TIME_SSP2_222_GENERAL:          // Eq. 35-37 / Table I
      T.s = 2;
      T.At[1][0] = 1.0; T.wt[0] = T.wt[1] = 0.5;
      T.A[0][0] = g; T.A[1][0] = 1.0 - 2.0 * g; T.A[1][1] = g; T.w[0] = T.w[1] = 0.5;
      return true;
    case TIME_SSP2_332:                                      // stiffly accurate, second order
      T.s = 3;
      T.At[1][0] = 0.5; T.At[2][0] = 0.5; T.At[2][1] = 0.5; T.wt[0] = T.wt[1] = T.wt[2] = 1.0 / 3.0;
      T.A[0][0] = 0.25; T.A[1][1] = 0.25; T.A[2][0] = T.A[2][1] = T.A[2][2] = 1.0 / 3.0;
      T.w[0] = T.w[1] = T.w[2] = 1.0 / 3.0;
      return true;
    case TIME_SSP3_332:                                      // third-order SSP explicit part, second order overall
      T.s = 3;
      T.At[1][0] = 1.0; T.At[2][0] = 0.25; T.At[2][1] = 0.25; T.wt[0] = T.wt[1] = 1.0 / 6.0; T.wt[2] = 2.0 / 3.0;
      T.A[0][0] = g; T.A[1][0] = 1.0 - 2.0 * g; T.A[1][1] = g; T.A[2][0] = 0.5 - g; T.A[2][2] = g;
      T.w[0] = T.w[1] = 1.0 / 6.0; T.w[2] = 2.0 / 3.0;
      return true;
    case TIME_SSP3_433: {                                    // third order
      const double al = 0.24169426078821, be = 0.06042356519705, et = 0.12915286960590;
      T.s = 4;
      T.At[2][1] = 1.0; T.At[3][1] = 0.25; T.At[3][2] = 0.25; T.wt[1] = T.wt[2] = 1.0 / 6.0; T.wt[3] = 2.0 / 3.0;
      T.A[0][0] = al; T.A[1][0] = -al; T.A[1][1] = al; T.A[2][1] = 1.0 - al; T.A[2][2] = al;
      T.A[3][0] = be; T.A[3][1] = et; T.A[3][2] = 0.5 - be - et - al; T.A[3][3] = al;
      T.w[1] = T.w[2] = 1.0 / 6.0; T.w[3] = 2.0 / 3.0;
      return true;
    }
  }
  return false;
}

void step_tableau(Grid& G, double dt, int scheme, const Tableau& T) {
  FLOP_REGION(R_COMBINE);
  const int nx = G.par.n[0], ny = G.par.n[1], nz = G.par.n[2], s = T.s;
  std::vector<double> F[4][NCONS], R[4][3], Xst[3], Xi[3];
  for (int q = 0; q < 3; ++q) { Xst[q].assign(G.ntot, 0.0); Xi[q].assign(G.ntot, 0.0); }
  for (int i = 0; i < s; ++i) {
    for (int q = 0; q < 3; ++q) R[i][q].assign(G.ntot, 0.0);
    // stage vector: explicit part (its calE entries are X*^(i)) ...
#pragma omp parallel for collapse(3) schedule(static)
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int ii = 0; ii < nx; ++ii) {
      const long c = G.idx(ii, j, k);
      for (int v = 0; v < NCONS; ++v) {
        double u = G.Un[v][c];
        for (int jj = 0; jj < i; ++jj) if (T.At[i][jj] != 0.0) u += dt * T.At[i][jj] * F[jj][v][c];
        G.Us[v][c] = u;
      }
      for (int q = 0; q < 3; ++q) {
        double x = G.Us[CEX + q][c];
        for (int jj = 0; jj < i; ++jj) if (T.A[i][jj] != 0.0) x += dt * T.A[i][jj] * R[jj][q][c];
        G.Us[CEX + q][c] = x;
        Xst[q][c] = x;
      }
    }
    // ... and its implicit part: solve for (calE^(i), P^(i)) with a = a_ii dt
    solve_all(G, G.Us, T.A[i][i] * dt, Xi, false);
#pragma omp parallel for collapse(3) schedule(static)
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int ii = 0; ii < nx; ++ii) {
      const long c = G.idx(ii, j, k);
      for (int q = 0; q < 3; ++q) R[i][q][c] = (Xi[q][c] - Xst[q][c]) / (T.A[i][i] * dt);
    }
    bool used = T.wt[i] != 0.0;
    for (int jj = i + 1; jj < s; ++jj) used = used || T.At[jj][i] != 0.0;
    if (!used) continue;
    stage_ghosts_and_charge(G);
    for (int v = 0; v < NCONS; ++v) F[i][v].assign(G.ntot, 0.0);
    rhs_all(G, scheme, F[i]);
  }
#pragma omp parallel for collapse(3) schedule(static)
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int ii = 0; ii < nx; ++ii) {
    const long c = G.idx(ii, j, k);
    for (int v = 0; v < NCONS; ++v) {
      double u = G.Un[v][c];
      for (int i = 0; i < s; ++i) if (T.wt[i] != 0.0) u += dt * T.wt[i] * F[i][v][c];
      if (v >= CEX && v <= CEZ) for (int i = 0; i < s; ++i) if (T.w[i] != 0.0) u += dt * T.w[i] * R[i][v - CEX][c];
      G.Un[v][c] = u;
    }
  }
  solve_all(G, G.Un, 0.0, nullptr, true);
  final_charge(G);
}

// a7. max over interior cells and active directions of (alpha sqrt(gamma^kk) + |beta^k|)/dx^k (Eq. 30); with
// wave_speed_mode MHD_INSIDE (A9) the cell's own max(|lambda-|, |lambda+|)/dx^k where rho > wave_rho_switch
double max_speed(const Grid& G) {
  double mx = 0.0;
  for (int k = 0; k < G.par.n[2]; ++k) for (int j = 0; j < G.par.n[1]; ++j) for (int i = 0; i < G.par.n[0]; ++i) {
    const long c = G.idx(i, j, k);
    Metric m; metric_at(G, c, m);
    const bool mhd = G.par.wave_speed_mode == WAVE_MHD_INSIDE && G.have_prims && G.P[RHO][c] > G.par.wave_rho_switch;
    double P[NPRIM];
    if (mhd) for (int v = 0; v < NPRIM; ++v) P[v] = G.P[v][c];
    for (int d = 0; d < 3; ++d) if (G.active(d)) {
      if (mhd) {       // A9: the cell's own ideal-GRMHD speeds where it counts as "inside the star"
        double lm, lp;
        mhd_wave_speeds(m, G.par.Gamma, d, P, &lm, &lp);
        mx = std::max(mx, std::max(std::fabs(lm), std::fabs(lp)) / G.par.dx[d]);
      } else {
        mx = std::max(mx, (m.alpha * std::sqrt(m.gUU[d][d]) + std::fabs(m.betaU[d])) / G.par.dx[d]);
      }
    }
  }
  return mx;
}

void cons_from_prims_all(Grid& G) {
  FLOP_REGION(R_P2C);
  for (long c = 0; c < G.ntot; ++c) {
    Metric m; metric_at(G, c, m);
    double P[NPRIM], U[NCONS];
    for (int v = 0; v < NPRIM; ++v) P[v] = G.P[v][c];
    prim2cons_point(m, G.par.Gamma, P, U);
    for (int v = 0; v < NCONS; ++v) G.Un[v][c] = U[v];
  }
}

Metric metric_from_arrays(double alpha, const double* beta3, const double* g6) {
  Metric m;
  m.alpha = alpha;
  for (int i = 0; i < 3; ++i) m.betaU[i] = beta3 ? beta3[i] : 0.0;
  m.gDD[0][0] = g6[0]; m.gDD[0][1] = m.gDD[1][0] = g6[1]; m.gDD[0][2] = m.gDD[2][0] = g6[2];
  m.gDD[1][1] = g6[3]; m.gDD[1][2] = m.gDD[2][1] = g6[4]; m.gDD[2][2] = g6[5];
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) m.KDD[i][j] = 0;
  metric_finish(m);
  return m;
}

}  // namespace

// =================================================================================================
// C ABI (host pointers everywhere).  Mirrors include/rgrmhd.h with an oracle_ prefix, plus
// point-wise entry points used by the pins.
// =================================================================================================
extern "C" {

struct oracle_params {
  int n[3]; double dx[3]; int ng; int bc[3]; double gamma_eos; int sigma_model;
  double sigma0, sigma_exp, sigma_dref, kappa, rho_floor, k_atmo, c2p_tol; int c2p_max_iter;
  int charge_mode; double weno_eps; int device;
  int wave_speed_mode; double wave_rho_switch;
};
struct oracle_stats { long long c2p_solves, c2p_evals, c2p_failures, floor_resets; int c2p_max_evals, reserved; };

int oracle_create(void** out, const oracle_params* p) {
  if (!out || !p) return -1;
  if (p->ng != 3 || !(p->gamma_eos > 1.0)) return -1;
  for (int d = 0; d < 3; ++d) if (p->n[d] < 1 || (p->n[d] > 1 && !(p->dx[d] > 0.0)) || p->bc[d] < 0 || p->bc[d] > 1) return -1;
  if (p->sigma_model < 0 || p->sigma_model > 3 || p->charge_mode < 0 || p->charge_mode > 2) return -1;
  if (p->wave_speed_mode < 0 || p->wave_speed_mode > 1) return -1;
  Grid* G = new Grid();
  Params& q = G->par;
  for (int d = 0; d < 3; ++d) { q.n[d] = p->n[d]; q.dx[d] = p->dx[d]; q.bc[d] = p->bc[d]; }
  q.ng = 3; q.Gamma = p->gamma_eos; q.sigma_model = p->sigma_model; q.sigma0 = p->sigma0; q.sigma_exp = p->sigma_exp;
  q.sigma_dref = p->sigma_dref; q.kappa = p->kappa; q.rho_floor = p->rho_floor; q.k_atmo = p->k_atmo;
  q.c2p_tol = p->c2p_tol > 0 ? p->c2p_tol : 8.0 * std::ldexp(1.0, -52);
  q.c2p_max_iter = p->c2p_max_iter > 0 ? p->c2p_max_iter : 100;
  q.charge_mode = p->charge_mode; q.weno_eps = p->weno_eps > 0 ? p->weno_eps : 1e-26;
  q.wave_speed_mode = p->wave_speed_mode; q.wave_rho_switch = p->wave_rho_switch;
  G->ntot = 1;
  for (int d = 0; d < 3; ++d) { G->g[d] = q.n[d] > 1 ? 3 : 0; G->np[d] = q.n[d] + 2 * G->g[d]; G->ntot *= G->np[d]; }
  for (int v = 0; v < NMET; ++v) G->met[v].assign(G->ntot, 0.0);
  for (int v = 0; v < NPRIM; ++v) G->P[v].assign(G->ntot, 0.0);
  for (int v = 0; v < NCONS; ++v) { G->Un[v].assign(G->ntot, 0.0); G->Us[v].assign(G->ntot, 0.0); G->F1[v].assign(G->ntot, 0.0); G->F2[v].assign(G->ntot, 0.0); }
  for (int q3 = 0; q3 < 3; ++q3) { G->jc[q3].assign(G->ntot, 0.0); G->jc1[q3].assign(G->ntot, 0.0); G->X1[q3].assign(G->ntot, 0.0); G->X2[q3].assign(G->ntot, 0.0); G->Xs2[q3].assign(G->ntot, 0.0); }
  *out = G;
  return 0;
}
int oracle_destroy(void* h) { delete (Grid*)h; return 0; }

int oracle_set_metric(void* h, const double* alpha, const double* const beta[3], const double* const gam[6], const double* const K[6]) {
  Grid* G = (Grid*)h;
  if (!G || !alpha || !beta || !gam || !K) return -1;
  std::copy(alpha, alpha + G->ntot, G->met[MALP].begin());
  for (int i = 0; i < 3; ++i) std::copy(beta[i], beta[i] + G->ntot, G->met[MBX + i].begin());
  for (int i = 0; i < 6; ++i) { std::copy(gam[i], gam[i] + G->ntot, G->met[MGXX + i].begin()); std::copy(K[i], K[i] + G->ntot, G->met[MKXX + i].begin()); }
  G->have_metric = true;
  return 0;
}
int oracle_set_sigma(void* h, const double* sigma) {
  Grid* G = (Grid*)h;
  if (!G || !sigma) return -1;
  if (G->par.sigma_model != SIGMA_ARRAY) return -2;
  G->sigma.assign(sigma, sigma + G->ntot); G->have_sigma = true;
  return 0;
}
int oracle_set_prims(void* h, const double* const prims[14]) {
  Grid* G = (Grid*)h;
  if (!G || !prims) return -1;
  if (!G->have_metric) return -2;
  for (int v = 0; v < NPRIM; ++v) std::copy(prims[v], prims[v] + G->ntot, G->P[v].begin());
  cons_from_prims_all(*G);
  G->have_prims = true;
  return 0;
}
int oracle_step(void* h, double dt, int scheme) {
  Grid* G = (Grid*)h;
  if (!G || !(dt > 0.0)) return -1;
  if (!G->have_metric || !G->have_prims || (G->par.sigma_model == SIGMA_ARRAY && !G->have_sigma)) return -2;
  const int recon = scheme & 0xff, time_scheme = (scheme >> 8) & 0xff;
  Tableau T;
  if (recon < 0 || recon > 2 || (scheme & ~0xffff) != 0 || !tableau_of(time_scheme, T)) return -1;
  if (time_scheme == TIME_SSP2_222) step(*G, dt, recon);      // Eq. 35-37 written out
  else step_tableau(*G, dt, recon, T);                        // Eq. 32 with the scheme's tableau
  return 0;
}
int oracle_max_speed(void* h, double* out) {
  Grid* G = (Grid*)h;
  if (!G || !out) return -1;
  if (!G->have_metric) return -2;
  *out = max_speed(*G);
  return 0;
}
int oracle_get_prims(void* h, double* const prims[14]) {
  Grid* G = (Grid*)h;
  if (!G || !prims) return -1;
  if (!G->have_prims) return -2;
  for (int v = 0; v < NPRIM; ++v) { ghost_fill_field(*G, G->P[v]); std::copy(G->P[v].begin(), G->P[v].end(), prims[v]); }
  return 0;
}
int oracle_get_cons(void* h, double* const cons[14]) {
  Grid* G = (Grid*)h;
  if (!G || !cons) return -1;
  if (!G->have_prims) return -2;
  for (int v = 0; v < NCONS; ++v) std::copy(G->Un[v].begin(), G->Un[v].end(), cons[v]);
  return 0;
}
int oracle_get_stats(void* h, oracle_stats* s) {
  Grid* G = (Grid*)h;
  if (!G || !s) return -1;
  s->c2p_solves = G->solves; s->c2p_evals = G->evals; s->c2p_failures = G->failures; s->floor_resets = G->floors;
  s->c2p_max_evals = G->max_evals; s->reserved = (int)std::min<long long>(G->face_fixups, 2147483647LL);
  return 0;
}
int oracle_reset_stats(void* h) {
  Grid* G = (Grid*)h;
  if (!G) return -1;
  G->solves = G->evals = G->failures = G->floors = G->face_fixups = 0; G->max_evals = 0;
  return 0;
}

// Which root finder the grid solves use: 0 = c2p_plain (default; bisection inside an un-accelerated fixed
// point), 1 = c2p_robust (bracketed secant + Anderson; ~100x fewer residual evaluations; a cross-check, and
// the only one that makes the largest multi-step parity runs finish).  Both find the root of the same system.
int oracle_set_solver(void* h, int which) {
  Grid* G = (Grid*)h;
  if (!G || which < 0 || which > 1) return -1;
  G->solver = which;
  return 0;
}

// ---- stage-level entry points (for pins that look inside a step) ---------------------------------
// F[U] (flux divergence + explicit sources) of the CURRENT primitives (ghosts are filled first; the
// conduction current jc is whatever the last solve left, zero after set_prims).
int oracle_rhs(void* h, int scheme, double* const out[14]) {
  Grid* G = (Grid*)h;
  if (!G || !out) return -1;
  for (int v = 0; v < NPRIM; ++v) ghost_fill_field(*G, G->P[v]);
  for (int q = 0; q < 3; ++q) ghost_fill_field(*G, G->jc[q]);
  rhs_all(*G, scheme & 0xff, G->F1);
  for (int v = 0; v < NCONS; ++v) std::copy(G->F1[v].begin(), G->F1[v].end(), out[v]);
  return 0;
}
// explicit sources S (a4, second half) of the CURRENT primitives alone, no flux divergence
int oracle_sources(void* h, double* const out[14]) {
  Grid* G = (Grid*)h;
  if (!G || !out) return -1;
  for (int k = 0; k < G->par.n[2]; ++k) for (int j = 0; j < G->par.n[1]; ++j) for (int i = 0; i < G->par.n[0]; ++i) {
    double S[NCONS];
    sources_cell(*G, i, j, k, S);
    for (int v = 0; v < NCONS; ++v) out[v][G->idx(i, j, k)] = S[v];
  }
  return 0;
}
// the two reconstructed states (after the fix-ups of reading R4) at the lower face, in direction d, of cell (i,j,k)
// of the CURRENT primitives (ghosts must be filled: call oracle_get_prims or oracle_rhs first); returns the fix-up count
int oracle_face_states(void* h, int scheme, int d, int i, int j, int k, double* PL, double* PR) {
  Grid* G = (Grid*)h;
  if (!G || !PL || !PR || d < 0 || d > 2) return -1;
  int o[3] = {0, 0, 0}; o[d] = 1;
  Metric mf; metric_face(*G, G->idx(i - o[0], j - o[1], k - o[2]), G->idx(i, j, k), mf);
  double jL, jR;
  return face_states(*G, scheme & 0xff, d, i, j, k, mf, PL, PR, &jL, &jR);
}
int oracle_ghost_fill(void* h, double* field) {
  Grid* G = (Grid*)h;
  if (!G || !field) return -1;
  std::vector<double> f(field, field + G->ntot);
  ghost_fill_field(*G, f);
  std::copy(f.begin(), f.end(), field);
  return 0;
}

// ---- point-wise entry points -----------------------------------------------------------------------
// metric arguments: alpha, beta[3] (may be null -> 0), gamma6 = xx,xy,xz,yy,yz,zz
int oracle_prim2cons_point(double Gamma, double alpha, const double* beta3, const double* g6, const double* P, double* U) {
  Metric m = metric_from_arrays(alpha, beta3, g6);
  prim2cons_point(m, Gamma, P, U);
  return 0;
}
// robust solve; P holds the guess on entry and the primitives on return.  returns evals, or -(evals + 1) if failed
int oracle_c2p_point(double Gamma, double alpha, const double* g6, const double* U, double adt, double sigma,
                     double tol, int maxit, double* P) {
  Metric m = metric_from_arrays(alpha, nullptr, g6);
  C2PResult r = c2p_robust(m, Gamma, U, adt, sigma, tol > 0 ? tol : 8.0 * std::ldexp(1.0, -52), maxit > 0 ? maxit : 100, P);
  return r.failed ? -(r.evals + 1) : r.evals;
}
int oracle_c2p_plain_point(double Gamma, double alpha, const double* g6, const double* U, double adt, double sigma,
                           double tol, int max_outer, double* P) {
  Metric m = metric_from_arrays(alpha, nullptr, g6);
  C2PResult r = c2p_plain(m, Gamma, U, adt, sigma, tol > 0 ? tol : 8.0 * std::ldexp(1.0, -52),
                          max_outer > 0 ? max_outer : PLAIN_MAX_OUTER, P);
  return r.failed ? -(r.evals + 1) : r.evals;
}
// A9: lambda-, lambda+ of one state at one point in direction k
int oracle_wave_speeds_point(double Gamma, double alpha, const double* beta3, const double* g6, int k, const double* P,
                             double* lam_minus, double* lam_plus) {
  Metric m = metric_from_arrays(alpha, beta3, g6);
  mhd_wave_speeds(m, Gamma, k, P, lam_minus, lam_plus);
  return 0;
}
// the double Butcher tableau of a time scheme: s, then At, wt, A, w as 4x4 / 4 arrays (row major); returns s or -1
int oracle_tableau(int time_scheme, double* At, double* wt, double* A, double* w) {
  Tableau T;
  if (!tableau_of(time_scheme, T)) return -1;
  for (int i = 0; i < 4; ++i) { wt[i] = T.wt[i]; w[i] = T.w[i]; for (int j = 0; j < 4; ++j) { At[4 * i + j] = T.At[i][j]; A[4 * i + j] = T.A[i][j]; } }
  return T.s;
}
// conductivity models at one point (A18)
double oracle_sigma_point(int model, double sigma0, double sigma_exp, double sigma_dref, double Dhat, double sigma_cell) {
  Params p{};
  p.sigma_model = model; p.sigma0 = sigma0; p.sigma_exp = sigma_exp; p.sigma_dref = sigma_dref;
  return sigma_of(p, Dhat, sigma_cell);
}
int oracle_c2p_literal_point(double Gamma, double alpha, const double* g6, const double* U, double adt, double sigma,
                             double tol, int maxit, double* P) {
  Metric m = metric_from_arrays(alpha, nullptr, g6);
  C2PResult r = c2p_literal(m, Gamma, U, adt, sigma, tol, maxit, P);
  return r.failed ? -(r.evals + 1) : r.evals;
}
// implicit E at fixed v: closed form (mode 0) or `iters` Newton iterations of Eq. 43 from E0 (mode 1)
int oracle_implicit_E_point(double alpha, const double* g6, const double* vU, double s, const double* EstarU,
                            const double* BU, int mode, const double* E0U, int iters, double* EU) {
  Metric m = metric_from_arrays(alpha, nullptr, g6);
  double vD[3], BD[3];
  lower(m, vU, vD); lower(m, BU, BD);
  const double W = 1.0 / std::sqrt(1.0 - dotUD(vU, vD));
  if (mode == 0) implicit_E_closed(m, vU, W, s, EstarU, BD, EU);
  else implicit_E_newton(m, vU, W, s, EstarU, BD, E0U, iters, EU);
  return 0;
}
// U and F^k of one state at one point (mode CELL_CURRENT uses jck, FACE_OHM uses sigma)
int oracle_state_flux_point(double Gamma, double alpha, const double* beta3, const double* g6, int k, const double* P,
                            int charge_mode, double sigma, double jck, double* U, double* F) {
  Metric m = metric_from_arrays(alpha, beta3, g6);
  state_flux(m, Gamma, k, P, charge_mode, sigma, jck, U, F);
  return 0;
}
// reconstruction of a 1D array u[0..n): at_minus[i], at_plus[i] for 2 <= i < n-2
int oracle_recon_1d(int scheme, double eps_w, int n, const double* u, double* at_minus, double* at_plus) {
  for (int i = 2; i < n - 2; ++i) recon_cell(scheme, eps_w > 0 ? eps_w : 1e-26, u[i - 2], u[i - 1], u[i], u[i + 1], u[i + 2], &at_minus[i], &at_plus[i]);
  return 0;
}
// number of OpenMP threads of the -fopenmp build (no effect on results: cells are independent, max is exact)
int oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n;
  return 1;
#endif
}
#ifdef ORACLE_COUNT_FLOPS
// counters of the instrumented build: out[region][op] (add, mul, div, sqrt), calls[region]
int oracle_flops_get(long long* out, long long* calls) {
  for (int r = 0; r < flopcount::R_COUNT; ++r) {
    calls[r] = flopcount::calls[r];
    for (int o = 0; o < flopcount::OP_COUNT; ++o) out[r * flopcount::OP_COUNT + o] = flopcount::counts[r][o];
  }
  return flopcount::R_COUNT;
}
int oracle_flops_reset(void) {
  std::memset(flopcount::counts, 0, sizeof(flopcount::counts));
  std::memset(flopcount::calls, 0, sizeof(flopcount::calls));
  return 0;
}
#endif
int oracle_omp_enabled(void) {
#ifdef _OPENMP
  return 1;
#else
  return 0;
#endif
}

}  // extern "C"
