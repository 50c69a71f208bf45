// rgrmhd_common.cuh -- device-side data model and point-wise physics of the B200-native resistive
// GRMHD step (product code; shares nothing with oracle/).
//
// Every function cites the passage of the paper (PAPER.md:line, equation) or the DESIGN.md reading
// (R1..R14) it implements.  All arithmetic is FP64; nvcc may contract a*b+c into DFMA, which is the
// only divergence from the oracle that DESIGN.md Sec. 3 allows.  No rsqrt, no pow.
//
// Notation: hats = undensitised conserved variables X^ = X/sqrt(gamma); vU = v^i, vD = v_i;
// h = rho(1+eps)+p is the enthalpy density; Z = h W^2.  Symmetric tensors are stored
// xx,xy,xz,yy,yz,zz.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace rg {

enum { NPRIM = 14, NCONS = 14, NMET = 16, NSRC = 34 };
// primitive indices
enum { RHO = 0, PRS, VX, VY, VZ, EX, EY, EZ, BX, BY, BZ, PSI, PHI, QCH };
// conserved indices
enum { CD = 0, CSX, CSY, CSZ, CTAU, CEX, CEY, CEZ, CBX, CBY, CBZ, CPSI, CPHI, CQ };
enum { MALP = 0, MBX, MBY, MBZ, MGXX, MGXY, MGXZ, MGYY, MGYZ, MGZZ, MKXX, MKXY, MKXZ, MKYY, MKYZ, MKZZ };
enum { BC_PERIODIC = 0, BC_OUTFLOW = 1, BC_EXTERNAL = 2 };
enum { SIGMA_UNIFORM = 0, SIGMA_ARRAY = 1, SIGMA_POWER_D = 2, SIGMA_ATMO = 3 };
enum { CHARGE_FACE_OHM = 0, CHARGE_CELL_CURRENT = 1, CHARGE_DIV_E = 2 };
enum { RECON_MINMOD = 0, RECON_MC = 1, RECON_WENO5 = 2 };
enum { WAVE_LIGHT = 0, WAVE_MHD_INSIDE = 1 };

// Device view of one block: geometry, model constants and the SoA field pointers (all DEVICE memory,
// padded layout of include/rgrmhd.h).  Passed to kernels by value as a __grid_constant__ parameter.
struct GridView {
  int n[3];        // interior cells
  int np[3];       // padded cells
  int g[3];        // ghost offset (3 for active directions, 0 for inactive)
  int bc[3];
  long long stride[3];
  long long ntot;
  double dx[3], inv_dx[3], inv_12dx[3];
  double Gamma, sigma0, sigma_dref, kappa, rho_floor, p_atmo, tol, weno_eps;
  double gog1, gm1og;    // Gamma/(Gamma-1), (Gamma-1)/Gamma (host-computed: no division in the kernels)
  int sigma_model, sigma_exp, maxit, charge_mode;
  int wave_mode;             // WAVE_LIGHT | WAVE_MHD_INSIDE (reading R16)
  double wave_rho_switch;    // MHD_INSIDE: both face states (or the cell) denser than this count as inside the star
  const double* met[NMET];
  const double* sigma;   // SIGMA_ARRAY only, else nullptr
  double* P[NPRIM];      // primitives of the current stage (ghosts filled by k_ghost_fill)
  double* jc[3];         // undensitised conduction current of the current stage (reading R3)
  double* Un[NCONS];     // U^n, overwritten with U^{n+1} by the stage-2 combine
  double* Us[NCONS];     // stage vector U*^(2)
  double* X1[3];         // calE^(1) (needed again by the final combine, Eq. 37)
  double* dU[NCONS];     // w dt (-div F) of the last flux launch (w = 1 stage 1, 1/2 stage 2); the next recovery adds it
  double* src[NSRC];     // static source coefficients (metric derivatives, G^i, tr K; rgrmhd_sources.cuh)
  unsigned long long* maxspeed_word;    // bit pattern of the running max of the CFL reduction (a7)
  const unsigned long long* src_mask;   // device word: bit q set <=> src[q] (q < NSRC) / K_ij[q - NSRC] is not identically 0
};

struct StatsDev {
  unsigned long long evals, failures, floors;
  int max_evals, pad;
};

// ------------------------------------------------------------------------------------------------
// metric algebra at one point (Eq. 1-5)
// ------------------------------------------------------------------------------------------------
struct Met {
  double alpha, b[3];   // lapse, shift beta^i
  double g[6];          // gamma_ij
  double gi[6];         // gamma^ij
  double sg;            // sqrt(det gamma_ij)
};

__device__ __forceinline__ constexpr int sym(int i, int j) {
  return (i == 0) ? j : (j == 0) ? i : (i == 1) ? ((j == 1) ? 3 : 4) : ((j == 1) ? 4 : 5);
}

// ------------------------------------------------------------------------------------------------
// Branch-free FP64 reciprocal / square root: hardware seed (MUFU.RCP64H / MUFU.RSQ64H; measured on B200:
// relative error e <= 1.0e-6 for both) + the series of the correction factor to second order in e, so that the
// truncation error is O(e^3) ~ 1e-18, below 2^-53:
//   1/x       = r / (1 - e),       e = 1 - x r    ->  r (1 + e + e^2)              3 dependent DFMA
//   1/sqrt(x) = r / sqrt(1 - e),   e = 1 - x r^2  ->  r (1 + e/2 + 3 e^2 / 8)      DMUL, DFMA, DFMA, DMUL, DFMA
// Measured over 4 x 2^28 arguments (ln x uniform in [-600, 600], [-1, 1], [-40, 0], [0, 40]): max relative error
// 1.12e-16 (reciprocal; equal to IEEE 1/x except for 0.03 % of the arguments, which are one ulp off), 1.40e-16
// (inverse square root), 1.67e-16 (square root).  Two Newton steps, the round-1 version, cost one (reciprocal) and
// five (coupled square roots) more dependent instructions for 1.11e-16 / 2.2e-16 / 1.11e-16.
// For normal, positive-finite arguments (every use below: determinants, 1 - v^2, WENO weight sums); no
// special-case path, so the surrounding code stays one basic block and independent chains interleave.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  return fma(r, fma(e, e, e), r);
}
// g = sqrt(x), rs = 1/sqrt(x): both from the same correction factor
__device__ __forceinline__ void sqrt_rsqrt_fast(double x, double& g, double& rs) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double g0 = x * r;
  const double e = fma(-g0, r, 1.0);
  const double t = fma(0.375, e, 0.5) * e;
  rs = fma(r, t, r);
  g = fma(g0, t, g0);
}
__device__ __forceinline__ double sqrt_fast(double x) { double g, rs; sqrt_rsqrt_fast(x, g, rs); return g; }
__device__ __forceinline__ double rsqrt_fast(double x) { double g, rs; sqrt_rsqrt_fast(x, g, rs); return rs; }

// sqrt(gamma) and gamma^ij = adjugate/det from gamma_ij
__device__ __forceinline__ void met_finish(Met& m) {
  const double gxx = m.g[0], gxy = m.g[1], gxz = m.g[2], gyy = m.g[3], gyz = m.g[4], gzz = m.g[5];
  const double cxx = gyy * gzz - gyz * gyz;
  const double cxy = gxz * gyz - gxy * gzz;
  const double cxz = gxy * gyz - gxz * gyy;
  const double det = gxx * cxx + gxy * cxy + gxz * cxz;
  const double idet = rcp_fast(det);
  m.sg = sqrt_fast(det);
  m.gi[0] = cxx * idet;
  m.gi[1] = cxy * idet;
  m.gi[2] = cxz * idet;
  m.gi[3] = (gxx * gzz - gxz * gxz) * idet;
  m.gi[4] = (gxy * gxz - gxx * gyz) * idet;
  m.gi[5] = (gxx * gyy - gxy * gxy) * idet;
}

__device__ __forceinline__ void lower(const Met& m, const double aU[3], double aD[3]) {
  aD[0] = m.g[0] * aU[0] + m.g[1] * aU[1] + m.g[2] * aU[2];
  aD[1] = m.g[1] * aU[0] + m.g[3] * aU[1] + m.g[4] * aU[2];
  aD[2] = m.g[2] * aU[0] + m.g[4] * aU[1] + m.g[5] * aU[2];
}
__device__ __forceinline__ void raise(const Met& m, const double aD[3], double aU[3]) {
  aU[0] = m.gi[0] * aD[0] + m.gi[1] * aD[1] + m.gi[2] * aD[2];
  aU[1] = m.gi[1] * aD[0] + m.gi[3] * aD[1] + m.gi[4] * aD[2];
  aU[2] = m.gi[2] * aD[0] + m.gi[4] * aD[1] + m.gi[5] * aD[2];
}
__device__ __forceinline__ double dot3(const double a[3], const double b[3]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}
// [ijk] a_j b_k (no metric factor)
__device__ __forceinline__ void cross_raw(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

__device__ __forceinline__ void load_met_cell(const GridView& G, long long c, Met& m) {
  m.alpha = __ldg(G.met[MALP] + c);
#pragma unroll
  for (int i = 0; i < 3; ++i) m.b[i] = __ldg(G.met[MBX + i] + c);
#pragma unroll
  for (int q = 0; q < 6; ++q) m.g[q] = __ldg(G.met[MGXX + q] + c);
  met_finish(m);
}
// reading R2: face metric = arithmetic mean of alpha, beta^i, gamma_ij of the two adjacent centres;
// sqrt(gamma), gamma^ij from the averaged gamma_ij
__device__ __forceinline__ void load_met_face(const GridView& G, long long cL, long long cR, Met& m) {
  m.alpha = 0.5 * (__ldg(G.met[MALP] + cL) + __ldg(G.met[MALP] + cR));
#pragma unroll
  for (int i = 0; i < 3; ++i) m.b[i] = 0.5 * (__ldg(G.met[MBX + i] + cL) + __ldg(G.met[MBX + i] + cR));
#pragma unroll
  for (int q = 0; q < 6; ++q) m.g[q] = 0.5 * (__ldg(G.met[MGXX + q] + cL) + __ldg(G.met[MGXX + q] + cR));
  met_finish(m);
}

// ------------------------------------------------------------------------------------------------
// A18. conductivity models (Eq. 52; Eq. 61; reading R13), Dhat = D/sqrt(gamma)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double sigma_of(const GridView& G, double Dhat, long long c) {
  switch (G.sigma_model) {
    case SIGMA_UNIFORM: return G.sigma0;
    case SIGMA_ARRAY: return __ldg(G.sigma + c);
    case SIGMA_POWER_D: {
      const double x = Dhat / G.sigma_dref;
      double r = 1.0;
      for (int i = 0; i < G.sigma_exp; ++i) r *= x;   // integer exponent by multiplication, no pow
      return G.sigma0 * r;
    }
    case SIGMA_ATMO: {
      const double x = fmax(1.0 - G.sigma_dref / Dhat, 0.0);
      return G.sigma0 * x * x;
    }
  }
  return 0.0;
}

// ------------------------------------------------------------------------------------------------
// a0. primitive -> conserved at one point (Eq. 22-24; Eq. 28; EOS Eq. 49)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void prim2cons(const Met& m, double Gamma, const double P[NPRIM], double U[NCONS]) {
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3], ExB[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  const double v2 = dot3(vU, vD);
  const double W = 1.0 / sqrt(1.0 - v2);
  const double h = rho + Gamma / (Gamma - 1.0) * p;            // rho(1+eps)+p with Eq. 49
  const double E2 = dot3(EU, ED), B2 = dot3(BU, BD);
  cross_raw(EU, BU, ExB);                                      // eps_ijk E^j B^k = sg [ijk] E^j B^k
  const double sg = m.sg, hW2 = h * W * W;
  U[CD] = sg * rho * W;                                        // Eq. 22
#pragma unroll
  for (int i = 0; i < 3; ++i) U[CSX + i] = sg * (hW2 * vD[i] + sg * ExB[i]);   // Eq. 24
  U[CTAU] = sg * (hW2 - p + 0.5 * (E2 + B2)) - U[CD];          // Eq. 23
#pragma unroll
  for (int i = 0; i < 3; ++i) { U[CEX + i] = sg * EU[i]; U[CBX + i] = sg * BU[i]; }   // Eq. 28
  U[CPSI] = sg * P[PSI]; U[CPHI] = sg * P[PHI]; U[CQ] = sg * P[QCH];
}

// ------------------------------------------------------------------------------------------------
// a3 (first half). U and F^k of one state at one face: Eq. 27 in reading R1
//   T^k_j = h W^2 v^k v_j + delta^k_j p - E^k E_j - B^k B_j + delta^k_j (E^2+B^2)/2
//   F(D)=(alpha v^k - beta^k) D ; F(S_j)=alpha sg T^k_j - beta^k S_j ; F(tau)=alpha(S^k - v^k D) - beta^k tau
//   F(calB^i)= alpha([ikj] E_j + g^ik Phi) - beta^k calB^i ; F(calE^i)=-alpha([ikj] B_j - g^ik Psi) - beta^k calE^i
//   F(Phi)=alpha calB^k - beta^k Phi ; F(Psi)=alpha calE^k - beta^k Psi
//   F(calQ)=alpha J^k - beta^k calQ, J^k = calQ v^k + Jc^k (Eq. 29; reading R3)
// ------------------------------------------------------------------------------------------------
template <int K, int CHARGE>
__device__ __forceinline__ void state_flux(const Met& m, double Gamma, const double P[NPRIM], double sigma,
                                           double jck, double U[NCONS], double F[NCONS]) {
  const double rho = P[RHO], p = P[PRS];
  const double vU[3] = {P[VX], P[VY], P[VZ]}, EU[3] = {P[EX], P[EY], P[EZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], ED[3], BD[3], ExB[3];
  lower(m, vU, vD); lower(m, EU, ED); lower(m, BU, BD);
  const double v2 = dot3(vU, vD);
  const double W = 1.0 / sqrt(1.0 - v2);
  const double h = rho + Gamma / (Gamma - 1.0) * p;
  const double E2 = dot3(EU, ED), B2 = dot3(BU, BD);
  cross_raw(EU, BU, ExB);
  const double sg = m.sg, hW2 = h * W * W, a = m.alpha, bk = m.b[K];
  const double pem = 0.5 * (E2 + B2);
  U[CD] = sg * rho * W;
#pragma unroll
  for (int i = 0; i < 3; ++i) U[CSX + i] = sg * (hW2 * vD[i] + sg * ExB[i]);
  U[CTAU] = sg * (hW2 - p + pem) - U[CD];
#pragma unroll
  for (int i = 0; i < 3; ++i) { U[CEX + i] = sg * EU[i]; U[CBX + i] = sg * BU[i]; }
  U[CPSI] = sg * P[PSI]; U[CPHI] = sg * P[PHI]; U[CQ] = sg * P[QCH];

  F[CD] = (a * vU[K] - bk) * U[CD];
  const double asg = a * sg;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    double Tkj = hW2 * vU[K] * vD[j] - EU[K] * ED[j] - BU[K] * BD[j];
    if (j == K) Tkj += p + pem;
    F[CSX + j] = asg * Tkj - bk * U[CSX + j];
  }
  const double SUk = m.gi[sym(K, 0)] * U[CSX] + m.gi[sym(K, 1)] * U[CSY] + m.gi[sym(K, 2)] * U[CSZ];
  F[CTAU] = a * (SUk - vU[K] * U[CD]) - bk * U[CTAU];
  // [ikj] X_j: for i = K zero; i = K+1: [K+1,K,K+2] = -1 -> -X_{K+2}; i = K+2: [K+2,K,K+1] = +1 -> +X_{K+1}
  constexpr int K1 = (K + 1) % 3, K2 = (K + 2) % 3;
  double curlE[3], curlB[3];
  curlE[K] = 0.0;      curlB[K] = 0.0;
  curlE[K1] = -ED[K2]; curlB[K1] = -BD[K2];
  curlE[K2] = ED[K1];  curlB[K2] = BD[K1];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    F[CBX + i] = a * (curlE[i] + m.gi[sym(i, K)] * U[CPHI]) - bk * U[CBX + i];
    F[CEX + i] = -a * (curlB[i] - m.gi[sym(i, K)] * U[CPSI]) - bk * U[CEX + i];
  }
  F[CPHI] = a * U[CBX + K] - bk * U[CPHI];
  F[CPSI] = a * U[CEX + K] - bk * U[CPSI];
  double Jck;
  if (CHARGE == CHARGE_FACE_OHM) {
    double vxB[3];
    cross_raw(vD, BD, vxB);                                 // (v x B)^i = [ijk] v_j B_k / sg
    const double vE = dot3(EU, vD);
    Jck = W * sigma * (U[CEX + K] + vxB[K] - vE * sg * vU[K]);   // Eq. 29 densitised: sg (v x B)^k = [kij] v_i B_j
  } else {
    Jck = sg * jck;
  }
  F[CQ] = a * (U[CQ] * vU[K] + Jck) - bk * U[CQ];
}

// ------------------------------------------------------------------------------------------------
// a2. reconstruction of one variable from the 5-cell stencil centred on a cell (reading R4).
//     lo = value at the cell's lower face (right state of face i-1/2), hi = at its upper face.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double minmod2(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  return copysign(fmin(fabs(a), fabs(b)), a);
}
__device__ __forceinline__ double minmod3(double a, double b, double c) {
  if (a > 0.0 && b > 0.0 && c > 0.0) return fmin(a, fmin(b, c));
  if (a < 0.0 && b < 0.0 && c < 0.0) return fmax(a, fmax(b, c));
  return 0.0;
}
// Jiang-Shu smoothness indicators of the stencil u0..u4 (shared by both faces of the centre cell)
__device__ __forceinline__ void weno5_beta(double u0, double u1, double u2, double u3, double u4, double eps_w,
                                           double& b0, double& b1, double& b2) {
  const double d0 = u0 - 2.0 * u1 + u2, e0 = u0 - 4.0 * u1 + 3.0 * u2;
  const double d1 = u1 - 2.0 * u2 + u3, e1 = u1 - u3;
  const double d2 = u2 - 2.0 * u3 + u4, e2 = 3.0 * u2 - 4.0 * u3 + u4;
  b0 = eps_w + (13.0 / 12.0 * d0 * d0 + 0.25 * e0 * e0);
  b1 = eps_w + (13.0 / 12.0 * d1 * d1 + 0.25 * e1 * e1);
  b2 = eps_w + (13.0 / 12.0 * d2 * d2 + 0.25 * e2 * e2);
}
// value at the +1/2 face of the centre cell u2; b0,b1,b2 = eps_w + beta_k of the stencils
// {u0,u1,u2},{u1,u2,u3},{u2,u3,u4}.  Weights d_k/b_k^2 with d = (0.1,0.6,0.3), normalised; written in
// product form (one division): w_k ~ d_k (b_l b_m)^2.
__device__ __forceinline__ double weno5_eval(double u0, double u1, double u2, double u3, double u4,
                                             double b0, double b1, double b2) {
  const double q0 = 2.0 * u0 - 7.0 * u1 + 11.0 * u2;
  const double q1 = -u1 + 5.0 * u2 + 2.0 * u3;
  const double q2 = 2.0 * u2 + 5.0 * u3 - u4;
  const double p12 = b1 * b2, p02 = b0 * b2, p01 = b0 * b1;
  const double a0 = 0.1 * (p12 * p12), a1 = 0.6 * (p02 * p02), a2 = 0.3 * (p01 * p01);
  return (a0 * q0 + a1 * q1 + a2 * q2) * rcp_fast(6.0 * (a0 + a1 + a2));
}
// Both face values of the centre cell u2 from one set of smoothness indicators.  Same scheme as
// weno5_eval (Jiang-Shu indicators, weights d_k / (eps + beta_k)^2 with d = (0.1, 0.6, 0.3) seen from the
// face, in product form: one reciprocal per face value), written in the first differences
// D_i = u_{i+1} - u_i: the second differences and the candidate values minus u2 are linear in them,
//   beta_0: d = D1 - D0, e = 3 D1 - D0;  beta_1: d = D2 - D1, e = D1 + D2;  beta_2: d = D3 - D2, e = D3 - 3 D2
//   q0 - u2 = (5 D1 - 2 D0)/6,  q1 - u2 = (2 D2 + D1)/6,  q2 - u2 = (4 D2 - D3)/6    (upper face; lower = mirror)
// with the linear weights folded into the candidate coefficients and the indicators scaled by 4 (a common factor of
// the three drops out of the weights): 58 FP64 instructions for both faces.
__device__ __forceinline__ void weno5_pair(double u0, double u1, double u2, double u3, double u4, double eps_w,
                                           double& lo, double& hi) {
  const double D0 = u1 - u0, D1 = u2 - u1, D2 = u3 - u2, D3 = u4 - u3;
  const double d0 = D1 - D0, e0 = fma(3.0, D1, -D0);
  const double d1 = D2 - D1, e1 = D1 + D2;
  const double d2 = D3 - D2, e2 = fma(-3.0, D2, D3);
  // 4 (eps + beta_k): the weights are ratios of products of all three, so a common factor drops out
  const double e4 = 4.0 * eps_w;
  const double b0 = fma((13.0 / 3.0) * d0, d0, fma(e0, e0, e4));
  const double b1 = fma((13.0 / 3.0) * d1, d1, fma(e1, e1, e4));
  const double b2 = fma((13.0 / 3.0) * d2, d2, fma(e2, e2, e4));
  const double p12 = b1 * b2, p02 = b0 * b2, p01 = b0 * b1;
  const double s12 = p12 * p12, s02 = p02 * p02, s01 = p01 * p01;
  // upper face: stencils {u0,u1,u2}, {u1,u2,u3}, {u2,u3,u4} weighted 0.1 s12, 0.6 s02, 0.3 s01
  const double hA = fma(0.1 * 5.0 / 6.0, D1, (-0.1 * 2.0 / 6.0) * D0);
  const double hB = fma(0.6 * 2.0 / 6.0, D2, (0.6 / 6.0) * D1);
  const double hC = fma(0.3 * 4.0 / 6.0, D2, (-0.3 / 6.0) * D3);
  const double hn = fma(s12, hA, fma(s02, hB, s01 * hC));
  const double mid = 0.6 * s02;
  const double hd = fma(0.1, s12, fma(0.3, s01, mid));
  // lower face: the mirror image (u0 <-> u4, u1 <-> u3: D_i -> -D_{3-i}, beta_0 <-> beta_2)
  const double lA = fma(-0.1 * 5.0 / 6.0, D2, (0.1 * 2.0 / 6.0) * D3);
  const double lB = fma(-0.6 * 2.0 / 6.0, D1, (-0.6 / 6.0) * D2);
  const double lC = fma(-0.3 * 4.0 / 6.0, D1, (0.3 / 6.0) * D0);
  const double ln = fma(s01, lA, fma(s02, lB, s12 * lC));
  const double ld = fma(0.1, s01, fma(0.3, s12, mid));
  hi = fma(hn, rcp_fast(hd), u2);
  lo = fma(ln, rcp_fast(ld), u2);
}
// N independent cells at once, statement by statement across the cells, so that the instruction stream
// interleaves N dependency chains (the reciprocal tails are serial: seed + 3 dependent DFMA).
template <int N>
__device__ __forceinline__ void weno5_pair_n(const double (&u)[N][5], double eps_w, double (&lo)[N], double (&hi)[N]) {
  double D0[N], D1[N], D2[N], D3[N], b0[N], b1[N], b2[N], s12[N], s02[N], s01[N], hn[N], hd[N], ln[N], ld[N];
#pragma unroll
  for (int j = 0; j < N; ++j) { D0[j] = u[j][1] - u[j][0]; D1[j] = u[j][2] - u[j][1]; D2[j] = u[j][3] - u[j][2]; D3[j] = u[j][4] - u[j][3]; }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double d0 = D1[j] - D0[j], e0 = fma(3.0, D1[j], -D0[j]);
    const double d1 = D2[j] - D1[j], e1 = D1[j] + D2[j];
    const double d2 = D3[j] - D2[j], e2 = fma(-3.0, D2[j], D3[j]);
    const double e4 = 4.0 * eps_w;
    b0[j] = fma((13.0 / 3.0) * d0, d0, fma(e0, e0, e4));
    b1[j] = fma((13.0 / 3.0) * d1, d1, fma(e1, e1, e4));
    b2[j] = fma((13.0 / 3.0) * d2, d2, fma(e2, e2, e4));
  }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double p12 = b1[j] * b2[j], p02 = b0[j] * b2[j], p01 = b0[j] * b1[j];
    s12[j] = p12 * p12; s02[j] = p02 * p02; s01[j] = p01 * p01;
  }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double hA = fma(0.1 * 5.0 / 6.0, D1[j], (-0.1 * 2.0 / 6.0) * D0[j]);
    const double hB = fma(0.6 * 2.0 / 6.0, D2[j], (0.6 / 6.0) * D1[j]);
    const double hC = fma(0.3 * 4.0 / 6.0, D2[j], (-0.3 / 6.0) * D3[j]);
    hn[j] = fma(s12[j], hA, fma(s02[j], hB, s01[j] * hC));
    const double mid = 0.6 * s02[j];
    hd[j] = fma(0.1, s12[j], fma(0.3, s01[j], mid));
    const double lA = fma(-0.1 * 5.0 / 6.0, D2[j], (0.1 * 2.0 / 6.0) * D3[j]);
    const double lB = fma(-0.6 * 2.0 / 6.0, D1[j], (-0.6 / 6.0) * D2[j]);
    const double lC = fma(-0.3 * 4.0 / 6.0, D1[j], (0.3 / 6.0) * D0[j]);
    ln[j] = fma(s01[j], lA, fma(s02[j], lB, s12[j] * lC));
    ld[j] = fma(0.1, s01[j], fma(0.3, s12[j], mid));
  }
  // 2N reciprocals (rcp_fast written out), interleaved
  double r[2 * N], e[2 * N], x[2 * N];
#pragma unroll
  for (int j = 0; j < N; ++j) { x[2 * j] = hd[j]; x[2 * j + 1] = ld[j]; }
#pragma unroll
  for (int q = 0; q < 2 * N; ++q) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r[q]) : "d"(x[q]));
#pragma unroll
  for (int q = 0; q < 2 * N; ++q) e[q] = fma(-x[q], r[q], 1.0);
#pragma unroll
  for (int q = 0; q < 2 * N; ++q) e[q] = fma(e[q], e[q], e[q]);
#pragma unroll
  for (int q = 0; q < 2 * N; ++q) r[q] = fma(r[q], e[q], r[q]);
#pragma unroll
  for (int j = 0; j < N; ++j) { hi[j] = fma(hn[j], r[2 * j], u[j][2]); lo[j] = fma(ln[j], r[2 * j + 1], u[j][2]); }
}

// reconstruction of N cells at once (lo/hi = values at each cell's lower/upper face)
template <int RECON, int N>
__device__ __forceinline__ void recon_cells(double eps_w, const double (&u)[N][5], double (&lo)[N], double (&hi)[N]) {
  if (RECON == RECON_WENO5) {
    weno5_pair_n<N>(u, eps_w, lo, hi);
  } else {
#pragma unroll
    for (int j = 0; j < N; ++j) {
      const double a = u[j][2] - u[j][1], b = u[j][3] - u[j][2];
      const double slope = (RECON == RECON_MINMOD) ? minmod2(a, b) : minmod3(2.0 * a, 2.0 * b, 0.5 * (a + b));
      hi[j] = u[j][2] + 0.5 * slope;
      lo[j] = u[j][2] - 0.5 * slope;
    }
  }
}

// Upper-face value only (the halo cells of a tile need one face): the same expressions as the upper face of
// weno5_pair, so the result is bit-identical; the lower-face value of a cell is this function of the mirrored stencil
// (u4 .. u0), also bit for bit (the differences change sign and order, the indicators swap, every product keeps its
// magnitude).
template <int RECON>
__device__ __forceinline__ double recon_hi(double eps_w, const double (&u)[5]) {
  if (RECON == RECON_WENO5) {
    const double D0 = u[1] - u[0], D1 = u[2] - u[1], D2 = u[3] - u[2], D3 = u[4] - u[3];
    const double d0 = D1 - D0, e0 = fma(3.0, D1, -D0);
    const double d1 = D2 - D1, e1 = D1 + D2;
    const double d2 = D3 - D2, e2 = fma(-3.0, D2, D3);
    const double e4 = 4.0 * eps_w;
    const double b0 = fma((13.0 / 3.0) * d0, d0, fma(e0, e0, e4));
    const double b1 = fma((13.0 / 3.0) * d1, d1, fma(e1, e1, e4));
    const double b2 = fma((13.0 / 3.0) * d2, d2, fma(e2, e2, e4));
    const double p12 = b1 * b2, p02 = b0 * b2, p01 = b0 * b1;
    const double s12 = p12 * p12, s02 = p02 * p02, s01 = p01 * p01;
    const double hA = fma(0.1 * 5.0 / 6.0, D1, (-0.1 * 2.0 / 6.0) * D0);
    const double hB = fma(0.6 * 2.0 / 6.0, D2, (0.6 / 6.0) * D1);
    const double hC = fma(0.3 * 4.0 / 6.0, D2, (-0.3 / 6.0) * D3);
    const double hn = fma(s12, hA, fma(s02, hB, s01 * hC));
    const double mid = 0.6 * s02;
    const double hd = fma(0.1, s12, fma(0.3, s01, mid));
    return fma(hn, rcp_fast(hd), u[2]);
  } else {
    const double a = u[2] - u[1], b = u[3] - u[2];
    const double slope = (RECON == RECON_MINMOD) ? minmod2(a, b) : minmod3(2.0 * a, 2.0 * b, 0.5 * (a + b));
    return u[2] + 0.5 * slope;
  }
}

template <int RECON>
__device__ __forceinline__ void recon_cell(double eps_w, double um2, double um1, double u0, double up1, double up2,
                                           double& lo, double& hi) {
  if (RECON == RECON_WENO5) {
    weno5_pair(um2, um1, u0, up1, up2, eps_w, lo, hi);
  } else {
    const double a = u0 - um1, b = up1 - u0;
    const double slope = (RECON == RECON_MINMOD) ? minmod2(a, b) : minmod3(2.0 * a, 2.0 * b, 0.5 * (a + b));
    hi = u0 + 0.5 * slope;
    lo = u0 - 0.5 * slope;
  }
}
// one-sided versions (a face needs `hi` of its left cell and `lo` of its right cell)
template <int RECON>
__device__ __forceinline__ double recon_hi(double eps_w, double um2, double um1, double u0, double up1, double up2) {
  if (RECON == RECON_WENO5) {
    double b0, b1, b2;
    weno5_beta(um2, um1, u0, up1, up2, eps_w, b0, b1, b2);
    return weno5_eval(um2, um1, u0, up1, up2, b0, b1, b2);
  } else {
    const double a = u0 - um1, b = up1 - u0;
    const double slope = (RECON == RECON_MINMOD) ? minmod2(a, b) : minmod3(2.0 * a, 2.0 * b, 0.5 * (a + b));
    return u0 + 0.5 * slope;
  }
}
template <int RECON>
__device__ __forceinline__ double recon_lo(double eps_w, double um2, double um1, double u0, double up1, double up2) {
  if (RECON == RECON_WENO5) {
    double b0, b1, b2;
    weno5_beta(um2, um1, u0, up1, up2, eps_w, b0, b1, b2);
    return weno5_eval(up2, up1, u0, um1, um2, b2, b1, b0);
  } else {
    const double a = u0 - um1, b = up1 - u0;
    const double slope = (RECON == RECON_MINMOD) ? minmod2(a, b) : minmod3(2.0 * a, 2.0 * b, 0.5 * (a + b));
    return u0 - 0.5 * slope;
  }
}

// reading R4: limit |v| of a face state with the face metric
__device__ __forceinline__ void limit_velocity(const Met& m, double P[NPRIM]) {
  const double vU[3] = {P[VX], P[VY], P[VZ]};
  double vD[3];
  lower(m, vU, vD);
  const double v2 = dot3(vU, vD), v2max = 1.0 - 1e-10;
  if (v2 >= v2max) {
    const double f = sqrt(v2max / v2);
    P[VX] *= f; P[VY] *= f; P[VZ] *= f;
  }
}

// A9. characteristic speeds "used in ideal GRMHD" (reading R16) of one state along direction K:
// the fluid-frame bound of the fast speed a^2 = cs^2 + vA^2 - cs^2 vA^2 (cs^2 = Gamma p/h, vA^2 = b^2/(h + b^2),
// b^2 = B^2/W^2 + (B.v)^2) boosted to the coordinate frame,
//   lambda+- = alpha [v^K (1-a^2) +- sqrt(a^2 (1-v^2) [gamma^KK (1 - v^2 a^2) - v^K v^K (1-a^2)])]/(1 - v^2 a^2) - beta^K.
// Arguments: the scalars v^2, B^2, B.v (taken with the face/cell metric), v^K, gamma^KK.
__device__ __forceinline__ void mhd_speeds(double alpha, double betaK, double giKK, double Gamma, double gog1, double rho,
                                           double p, double v2, double B2, double Bv, double vK, double& lm, double& lp) {
  const double h = rho + gog1 * p;
  const double b2 = B2 * (1.0 - v2) + Bv * Bv;
  const double cs2 = Gamma * p / h, vA2 = b2 / (h + b2);
  const double a2 = cs2 + vA2 - cs2 * vA2;
  const double den = 1.0 - v2 * a2, om = 1.0 - a2;
  const double root = sqrt(fmax(a2 * (1.0 - v2) * (giKK * den - vK * vK * om), 0.0));
  const double iden = 1.0 / den;
  lp = alpha * (vK * om + root) * iden - betaK;
  lm = alpha * (vK * om - root) * iden - betaK;
}
// natural-frame wrapper: P = primitives (after the fix-ups of reading R4), m = face or cell metric
template <int K>
__device__ __forceinline__ void mhd_speeds_nat(const Met& m, double Gamma, const double P[NPRIM], double& lm, double& lp) {
  const double vU[3] = {P[VX], P[VY], P[VZ]}, BU[3] = {P[BX], P[BY], P[BZ]};
  double vD[3], BD[3];
  lower(m, vU, vD); lower(m, BU, BD);
  mhd_speeds(m.alpha, m.b[K], m.gi[sym(K, K)], Gamma, Gamma / (Gamma - 1.0), P[RHO], P[PRS], dot3(vU, vD), dot3(BU, BD),
             dot3(BU, vD), vU[K], lm, lp);
}

// a7, one cell: max over the active directions of the CFL speed / dx -- Eq. 30, (alpha sqrt(gamma^kk) + |beta^k|)/dx^k,
// or with wave mode MHD_INSIDE (reading R16) the cell's own max(|lambda-|, |lambda+|)/dx^k where rho > wave_rho_switch.
// NOT inlined on purpose: the stand-alone reduction (k_max_speed) and the one fused into the final recovery call the
// same compiled function, so the two give the same bits.
static __device__ __noinline__ double cell_cfl_speed(const Met& m, double Gamma, const double P[NPRIM], bool mhd, double idx0,
                                              double idx1, double idx2, bool a0, bool a1, bool a2) {
  double s0, s1, s2;
  if (mhd) {
    double lm, lp;
    mhd_speeds_nat<0>(m, Gamma, P, lm, lp); s0 = fmax(fabs(lm), fabs(lp));
    mhd_speeds_nat<1>(m, Gamma, P, lm, lp); s1 = fmax(fabs(lm), fabs(lp));
    mhd_speeds_nat<2>(m, Gamma, P, lm, lp); s2 = fmax(fabs(lm), fabs(lp));
  } else {
    s0 = m.alpha * sqrt(m.gi[0]) + fabs(m.b[0]);
    s1 = m.alpha * sqrt(m.gi[3]) + fabs(m.b[1]);
    s2 = m.alpha * sqrt(m.gi[5]) + fabs(m.b[2]);
  }
  double mx = 0.0;
  if (a0) mx = fmax(mx, s0 * idx0);
  if (a1) mx = fmax(mx, s1 * idx1);
  if (a2) mx = fmax(mx, s2 * idx2);
  return mx;
}

// a3 (second half). HLLE combination (Eq. 30; reading R6; wave speeds: reading R16)
template <int K, int CHARGE>
__device__ __forceinline__ void hlle(const Met& mf, double Gamma, double PL[NPRIM], double PR[NPRIM],
                                     double sigL, double sigR, double jL, double jR, int wave_mode, double rho_switch,
                                     double Fh[NCONS]) {
  // F = (lp FL - lm FR + lp lm (UR - UL))/(lp - lm), accumulated state by state so that only one
  // state's (U, F) pair is live at a time
  limit_velocity(mf, PL);
  limit_velocity(mf, PR);
  double lp, lm;
  if (wave_mode == WAVE_MHD_INSIDE && PL[RHO] > rho_switch && PR[RHO] > rho_switch) {
    double lmL, lpL, lmR, lpR;
    mhd_speeds_nat<K>(mf, Gamma, PL, lmL, lpL);
    mhd_speeds_nat<K>(mf, Gamma, PR, lmR, lpR);
    lp = fmax(0.0, fmax(lpL, lpR));
    lm = fmin(0.0, fmin(lmL, lmR));
  } else {
    const double c = mf.alpha * sqrt(mf.gi[sym(K, K)]);
    lp = fmax(0.0, c - mf.b[K]);
    lm = fmin(0.0, -c - mf.b[K]);
  }
  const double inv = 1.0 / (lp - lm);
  const double cL = lp * inv, cR = -lm * inv, cU = lp * lm * inv;
  double U[NCONS], F[NCONS];
  state_flux<K, CHARGE>(mf, Gamma, PL, sigL, jL, U, F);
#pragma unroll
  for (int v = 0; v < NCONS; ++v) Fh[v] = cL * F[v] - cU * U[v];
  state_flux<K, CHARGE>(mf, Gamma, PR, sigR, jR, U, F);
#pragma unroll
  for (int v = 0; v < NCONS; ++v) Fh[v] += cR * F[v] + cU * U[v];
}

__device__ __forceinline__ long long cell_index(const GridView& G, int i, int j, int k) {
  return (long long)(i + G.g[0]) + G.stride[1] * (long long)(j + G.g[1]) + G.stride[2] * (long long)(k + G.g[2]);
}

}  // namespace rg
