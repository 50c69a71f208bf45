// rgrmhd_flux_rot.cuh -- the direction-rotated Riemann machinery shared by the tiled flux-divergence
// kernels (rgrmhd_rhs_pencil.cu, rgrmhd_rhs_tma.cu).  The three directions run through ONE copy of the
// reconstruction and Riemann code: direction K is a run-time cyclic rotation of the vector/tensor
// components (cyclic permutations keep the Levi-Civita sign, so Eq. 27 is form invariant), realised as
// index arithmetic on pointer / field-index tables.
#pragma once
#include "rgrmhd_rhs.cuh"

namespace rg {
namespace {

constexpr int NVR = 15;   // 14 primitives + the normal component of the conduction current (reading R3)

struct PencilTabs {
  const double* P[3][NVR];   // rotated order: rho, p, v^K v^K1 v^K2, E.., B.., psi, phi, q, jc^K
  const double* M[3][8];     // alpha, beta^K, gamma rotated: 00 01 02 11 12 22 (0 = K, 1 = K+1, 2 = K+2)
  int nat[3][NCONS];         // rotated conserved index -> natural conserved index
  int fld[3][NVR];           // field index of P[K][v] relative to G.P[0] (fields are equally spaced in the slab)
};

struct FaceMet {
  double alpha, b0, g[6], gi0[3], sg;
};

// reading R2: face metric = arithmetic mean of the two adjacent centres; sqrt(gamma) and the K-row of
// gamma^ij from the averaged gamma_ij (rotated components).  Split into the raw loads (which a kernel
// can issue long before it needs the values) and the arithmetic.
struct FaceRaw {
  double l[8], r[8];   // alpha, beta^K, gamma (rotated 00 01 02 11 12 22) of the left / right cell
};
__device__ __forceinline__ void load_face_raw(const PencilTabs& T, int K, long long cl, long long cr, FaceRaw& w) {
#pragma unroll
  for (int q = 0; q < 8; ++q) { w.l[q] = __ldg(T.M[K][q] + cl); w.r[q] = __ldg(T.M[K][q] + cr); }
}
__device__ __forceinline__ void finish_face_met(const FaceRaw& w, FaceMet& m) {
  m.alpha = 0.5 * (w.l[0] + w.r[0]);
  m.b0 = 0.5 * (w.l[1] + w.r[1]);
#pragma unroll
  for (int q = 0; q < 6; ++q) m.g[q] = 0.5 * (w.l[2 + q] + w.r[2 + q]);
  const double c00 = m.g[3] * m.g[5] - m.g[4] * m.g[4];
  const double c01 = m.g[2] * m.g[4] - m.g[1] * m.g[5];
  const double c02 = m.g[1] * m.g[4] - m.g[2] * m.g[3];
  const double det = m.g[0] * c00 + m.g[1] * c01 + m.g[2] * c02;
  double rs;
  sqrt_rsqrt_fast(det, m.sg, rs);
  const double idet = rs * rs;
  m.gi0[0] = c00 * idet; m.gi0[1] = c01 * idet; m.gi0[2] = c02 * idet;
}
__device__ __forceinline__ void load_face_met(const PencilTabs& T, int K, long long cl, long long cr, FaceMet& m) {
  FaceRaw w;
  load_face_raw(T, K, cl, cr, w);
  finish_face_met(w, m);
}

// a3, one state.  X = (rho, p, v[3], E[3], B[3], psi, phi, q, jc^0) in the rotated frame (0 = face normal).
// Adds wa*G + wu*U to Fh, where F = alpha G - beta^0 U is Eq. 27 (reading R1), i.e. the
// state's share w F + sd U of the HLLE flux with wa = w alpha, wu = sd - w beta^0.
template <int CHARGE, bool FIRST>
__device__ __forceinline__ void half_flux(const FaceMet& m, double gog1, const double X[NVR], double sigma,
                                          double wa, double wu, double Fh[NCONS]) {
  const double rho = X[0], p = X[1];
  double v[3] = {X[2], X[3], X[4]};
  const double E[3] = {X[5], X[6], X[7]}, B[3] = {X[8], X[9], X[10]};
  double vD[3];
  vD[0] = m.g[0] * v[0] + m.g[1] * v[1] + m.g[2] * v[2];
  vD[1] = m.g[1] * v[0] + m.g[3] * v[1] + m.g[4] * v[2];
  vD[2] = m.g[2] * v[0] + m.g[4] * v[1] + m.g[5] * v[2];
  double vsq = v[0] * vD[0] + v[1] * vD[1] + v[2] * vD[2];
  const double v2max = 1.0 - 1e-10;
  if (vsq >= v2max) {   // reading R4: limit |v| of a face state with the face metric
    const double f = sqrt_fast(v2max * rcp_fast(vsq));
#pragma unroll
    for (int a = 0; a < 3; ++a) { v[a] *= f; vD[a] *= f; }
    vsq = v[0] * vD[0] + v[1] * vD[1] + v[2] * vD[2];
  }
  const double ED[3] = {m.g[0] * E[0] + m.g[1] * E[1] + m.g[2] * E[2], m.g[1] * E[0] + m.g[3] * E[1] + m.g[4] * E[2],
                        m.g[2] * E[0] + m.g[4] * E[1] + m.g[5] * E[2]};
  const double BD[3] = {m.g[0] * B[0] + m.g[1] * B[1] + m.g[2] * B[2], m.g[1] * B[0] + m.g[3] * B[1] + m.g[4] * B[2],
                        m.g[2] * B[0] + m.g[4] * B[1] + m.g[5] * B[2]};
  const double W = rsqrt_fast(1.0 - vsq);
  const double h = rho + gog1 * p;                               // rho(1+eps)+p with Eq. 49, gog1 = Gamma/(Gamma-1)
  const double hW2 = h * W * W;
  const double pem = 0.5 * ((E[0] * ED[0] + E[1] * ED[1] + E[2] * ED[2]) + (B[0] * BD[0] + B[1] * BD[1] + B[2] * BD[2]));
  const double sg = m.sg;
  const double ExB[3] = {E[1] * B[2] - E[2] * B[1], E[2] * B[0] - E[0] * B[2], E[0] * B[1] - E[1] * B[0]};
  double U[NCONS], Gf[NCONS];
  U[CD] = sg * rho * W;                                          // Eq. 22
#pragma unroll
  for (int a = 0; a < 3; ++a) U[CSX + a] = sg * (hW2 * vD[a] + sg * ExB[a]);   // Eq. 24
  U[CTAU] = sg * (hW2 - p + pem) - U[CD];                        // Eq. 23
#pragma unroll
  for (int a = 0; a < 3; ++a) { U[CEX + a] = sg * E[a]; U[CBX + a] = sg * B[a]; }   // Eq. 28
  U[CPSI] = sg * X[11]; U[CPHI] = sg * X[12]; U[CQ] = sg * X[13];
  Gf[CD] = v[0] * U[CD];
  const double hv = hW2 * v[0];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double t = hv * vD[a] - E[0] * ED[a] - B[0] * BD[a];
    if (a == 0) t += p + pem;
    Gf[CSX + a] = sg * t;
  }
  Gf[CTAU] = (m.gi0[0] * U[CSX] + m.gi0[1] * U[CSX + 1] + m.gi0[2] * U[CSX + 2]) - v[0] * U[CD];
  Gf[CBX] = m.gi0[0] * U[CPHI];
  Gf[CBX + 1] = m.gi0[1] * U[CPHI] - ED[2];
  Gf[CBX + 2] = m.gi0[2] * U[CPHI] + ED[1];
  Gf[CEX] = m.gi0[0] * U[CPSI];
  Gf[CEX + 1] = m.gi0[1] * U[CPSI] + BD[2];
  Gf[CEX + 2] = m.gi0[2] * U[CPSI] - BD[1];
  Gf[CPHI] = U[CBX];
  Gf[CPSI] = U[CEX];
  double Jc;
  if (CHARGE == CHARGE_FACE_OHM) {   // Eq. 29 densitised: sg (v x B)^0 = v_1 B_2 - v_2 B_1
    const double vE = E[0] * vD[0] + E[1] * vD[1] + E[2] * vD[2];
    Jc = W * sigma * (U[CEX] + (vD[1] * BD[2] - vD[2] * BD[1]) - vE * sg * v[0]);
  } else {
    Jc = sg * X[14];
  }
  Gf[CQ] = U[CQ] * v[0] + Jc;
#pragma unroll
  for (int c = 0; c < NCONS; ++c) {
    Fh[c] = FIRST ? fma(wa, Gf[c], wu * U[c]) : fma(wa, Gf[c], fma(wu, U[c], Fh[c]));
  }
}

// A9 (reading R16) in the rotated frame: lambda-+ of the state whose rho, p, v[3], B[3] sit at xp[q * xs], q = 0, 1, 2-4,
// 8-10; the |v| limiter of reading R4 is applied first, as half_flux does.  Returns the state's rho.
__device__ __forceinline__ double mhd_speeds_rot(const FaceMet& m, double Gamma, const double* __restrict__ xp, int xs,
                                                 double& lm, double& lp) {
  const double rho = xp[0], p = xp[xs];
  double v[3] = {xp[2 * xs], xp[3 * xs], xp[4 * xs]};
  const double B[3] = {xp[8 * xs], xp[9 * xs], xp[10 * xs]};
  double vD[3];
  vD[0] = m.g[0] * v[0] + m.g[1] * v[1] + m.g[2] * v[2];
  vD[1] = m.g[1] * v[0] + m.g[3] * v[1] + m.g[4] * v[2];
  vD[2] = m.g[2] * v[0] + m.g[4] * v[1] + m.g[5] * v[2];
  double vsq = v[0] * vD[0] + v[1] * vD[1] + v[2] * vD[2];
  const double v2max = 1.0 - 1e-10;
  if (vsq >= v2max) {
    const double f = sqrt_fast(v2max * rcp_fast(vsq));
#pragma unroll
    for (int a = 0; a < 3; ++a) { v[a] *= f; vD[a] *= f; }
    vsq = v[0] * vD[0] + v[1] * vD[1] + v[2] * vD[2];
  }
  const double BD[3] = {m.g[0] * B[0] + m.g[1] * B[1] + m.g[2] * B[2], m.g[1] * B[0] + m.g[3] * B[1] + m.g[4] * B[2],
                        m.g[2] * B[0] + m.g[4] * B[1] + m.g[5] * B[2]};
  mhd_speeds(m.alpha, m.b0, m.gi0[0], Gamma, Gamma / (Gamma - 1.0), rho, p, vsq, B[0] * BD[0] + B[1] * BD[1] + B[2] * BD[2],
             B[0] * vD[0] + B[1] * vD[1] + B[2] * vD[2], v[0], lm, lp);
  return rho;
}
// HLLE bounds lambda-, lambda+ of a face (Eq. 30, reading R6; WAVE: PAPER.md:424, 437, reading R16)
template <int WAVE>
__device__ __forceinline__ void face_bounds(const GridView& G, const FaceMet& m, const double* __restrict__ plp, int pl_stride,
                                            const double* __restrict__ prp, int pr_stride, double& lm, double& lp) {
  if (WAVE == WAVE_MHD_INSIDE) {
    double lmL, lpL, lmR, lpR;
    const double rhoL = mhd_speeds_rot(m, G.Gamma, plp, pl_stride, lmL, lpL);
    const double rhoR = mhd_speeds_rot(m, G.Gamma, prp, pr_stride, lmR, lpR);
    if (rhoL > G.wave_rho_switch && rhoR > G.wave_rho_switch) {
      lp = fmax(0.0, fmax(lpL, lpR));
      lm = fmin(0.0, fmin(lmL, lmR));
      return;
    }
  }
  const double c = m.alpha * sqrt_fast(m.gi0[0]);
  lp = fmax(0.0, c - m.b0);
  lm = fmin(0.0, -c - m.b0);
}

// FACE_OHM only (reading R6): conductivity of a CELL from its primitives and metric
__device__ __forceinline__ double sigma_cell(const GridView& G, long long c) {
  if (G.sigma_model == SIGMA_UNIFORM) return G.sigma0;
  if (G.sigma_model == SIGMA_ARRAY) return __ldg(G.sigma + c);
  Met mc;
  load_met_cell(G, c, mc);
  double vU[3] = {G.P[VX][c], G.P[VY][c], G.P[VZ][c]}, vD[3];
  lower(mc, vU, vD);
  return sigma_of(G, G.P[RHO][c] * (1.0 / sqrt(1.0 - dot3(vU, vD))), c);
}

// a3 for one face with metric m: right state PR (registers), left state read from plp (strided); F in the
// rotated order
template <int CHARGE, int NV, int WAVE>
__device__ __forceinline__ void riemann_m(const GridView& G, const FaceMet& m, long long cl, long long cr,
                                          const double* __restrict__ plp, int pl_stride, double PR[NVR], double Fh[NCONS]) {
  // HLLE weights (Eq. 30; reading R6)
  double lp, lm;
  face_bounds<WAVE>(G, m, plp, pl_stride, PR, 1, lm, lp);
  const double inv = rcp_fast(lp - lm);
  const double wL = lp * inv, wR = -lm * inv, sd = lp * lm * inv;
  double sigL = 0.0, sigR = 0.0;
  if (CHARGE == CHARGE_FACE_OHM) { sigL = sigma_cell(G, cl); sigR = sigma_cell(G, cr); }
  if (NV < NVR) PR[NVR - 1] = 0.0;
  // Gamma/(Gamma-1) is grid-uniform; written as the division on purpose: ptxas hoists it, and with the
  // host-computed G.gog1 in its place the same kernel scheduled 4 % slower (measured, 256^3)
  half_flux<CHARGE, true>(m, G.Gamma / (G.Gamma - 1.0), PR, sigR, wR * m.alpha, sd - wR * m.b0, Fh);
  double PL[NVR];
#pragma unroll
  for (int vr = 0; vr < NV; ++vr) PL[vr] = plp[vr * pl_stride];
  if (NV < NVR) PL[NVR - 1] = 0.0;
  half_flux<CHARGE, false>(m, G.Gamma / (G.Gamma - 1.0), PL, sigL, wL * m.alpha, -sd - wL * m.b0, Fh);
}
// the same with both states in (shared) memory: right state at prp, left state at plp, each read just before
// its half of the flux, so that only one state is live at a time
template <int CHARGE, int NV, int WAVE>
__device__ __forceinline__ void riemann_mm(const GridView& G, const FaceMet& m, long long cl, long long cr,
                                           const double* __restrict__ plp, int pl_stride, const double* __restrict__ prp,
                                           int pr_stride, double Fh[NCONS]) {
  double lp, lm;
  face_bounds<WAVE>(G, m, plp, pl_stride, prp, pr_stride, lm, lp);
  const double inv = rcp_fast(lp - lm);
  const double wL = lp * inv, wR = -lm * inv, sd = lp * lm * inv;
  double sigL = 0.0, sigR = 0.0;
  if (CHARGE == CHARGE_FACE_OHM) { sigL = sigma_cell(G, cl); sigR = sigma_cell(G, cr); }
  {
    double PR[NVR];
#pragma unroll
    for (int vr = 0; vr < NV; ++vr) PR[vr] = prp[vr * pr_stride];
    if (NV < NVR) PR[NVR - 1] = 0.0;
    half_flux<CHARGE, true>(m, G.Gamma / (G.Gamma - 1.0), PR, sigR, wR * m.alpha, sd - wR * m.b0, Fh);
  }
  {
    double PL[NVR];
#pragma unroll
    for (int vr = 0; vr < NV; ++vr) PL[vr] = plp[vr * pl_stride];
    if (NV < NVR) PL[NVR - 1] = 0.0;
    half_flux<CHARGE, false>(m, G.Gamma / (G.Gamma - 1.0), PL, sigL, wL * m.alpha, -sd - wL * m.b0, Fh);
  }
}
template <int CHARGE, int NV>
__device__ __forceinline__ void riemann(const GridView& G, const PencilTabs& T, int K, long long cl, long long cr,
                                        const double* __restrict__ plp, int pl_stride, double PR[NVR], double Fh[NCONS]) {
  FaceMet m;
  load_face_met(T, K, cl, cr, m);
  if (G.wave_mode == WAVE_MHD_INSIDE) riemann_m<CHARGE, NV, WAVE_MHD_INSIDE>(G, m, cl, cr, plp, pl_stride, PR, Fh);
  else riemann_m<CHARGE, NV, WAVE_LIGHT>(G, m, cl, cr, plp, pl_stride, PR, Fh);
}
inline PencilTabs make_tabs(const GridView& G) {
  PencilTabs T;
  for (int K = 0; K < 3; ++K) {
    const int r[3] = {K, (K + 1) % 3, (K + 2) % 3};
    T.P[K][0] = G.P[RHO]; T.P[K][1] = G.P[PRS];
    for (int a = 0; a < 3; ++a) {
      T.P[K][2 + a] = G.P[VX + r[a]];
      T.P[K][5 + a] = G.P[EX + r[a]];
      T.P[K][8 + a] = G.P[BX + r[a]];
    }
    T.P[K][11] = G.P[PSI]; T.P[K][12] = G.P[PHI]; T.P[K][13] = G.P[QCH];
    T.P[K][14] = G.jc[K];
    const long long fs = G.P[1] - G.P[0];
    for (int v = 0; v < NVR; ++v) T.fld[K][v] = (int)((T.P[K][v] - G.P[0]) / fs);
    T.M[K][0] = G.met[MALP];
    T.M[K][1] = G.met[MBX + K];
    static const int symtab[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};   // xx xy xz yy yz zz
    int q = 0;
    for (int a = 0; a < 3; ++a)
      for (int b = a; b < 3; ++b) T.M[K][2 + q++] = G.met[MGXX + symtab[r[a]][r[b]]];
    for (int v = 0; v < NCONS; ++v) T.nat[K][v] = v;
    for (int a = 0; a < 3; ++a) {
      T.nat[K][CSX + a] = CSX + r[a];
      T.nat[K][CEX + a] = CEX + r[a];
      T.nat[K][CBX + a] = CBX + r[a];
    }
  }
  return T;
}

}  // namespace
}  // namespace rg
