// rgrmhd_rhs_pencil.cu -- flux-divergence kernel (a2, a3, divergence of a4, divergence part of a5):
// reconstruct + HLLE + flux divergence + update of the stage target in ONE launch.  Face states and fluxes
// never leave the SM.  (The point-wise sources and the rest of the stage combine run in the recovery kernel.)
//
// Decomposition ("pencil-tiled"): a CTA owns a TX x TY (x, y) tile of z-pencils and marches CZ planes
// along z; one thread = one cell of the current plane.  Per plane, for each direction K (x, y, z):
//   a2  every thread reconstructs ITS OWN CELL along K for all 15 variables: the smoothness
//       indicators are computed once and give both the value at the cell's lower face (kept in
//       registers: the right state of that face) and at its upper face (the left state of the next
//       face).  The upper-face values are handed to the neighbouring thread through shared memory
//       (x, y) or kept in a thread-private shared-memory slot for the next plane (z).
//   a3  every thread solves the HLLE problem at its cell's lower face (x, y) / upper face (z); the
//       flux goes to shared memory (aliasing the exchange buffer) and each cell differences its own
//       and its neighbour's flux.  No face is solved twice except the TX + TY faces on the tile's
//       upper x / y edge, which one warp each handles in an extra pass (their reconstruction halo:
//       two more partial warps).
//   a5  U*2 += dt dU or U^{n+1} += dt/2 dU (one read-modify-write of the stage target).
// The three directions run through ONE copy of the reconstruction and Riemann code: direction K is a
// run-time cyclic rotation of the vector/tensor components (cyclic permutations keep the Levi-Civita
// sign, so Eq. 27 is form invariant), realised for free as index arithmetic on pointer tables and
// shared-memory planes.  This keeps the kernel ~4x smaller than the fully templated version, whose
// instruction-cache misses dominated its stall profile (profiles/r01_rhs_tiled_ncu.md).
// Stencils are read straight from global memory (x: coalesced rows, L1; y: L1; z: L2).
#include "rgrmhd_rhs.cuh"

namespace rg {

namespace {
constexpr int TX = 32, TY = 8, NT = TX * TY;
constexpr int EXW = TX + 1, EXH = TY + 1, EXP = EXW * EXH;
constexpr int NVR = 15;   // 14 primitives + the normal component of the conduction current (reading R3)

struct PencilTabs {
  const double* P[3][NVR];   // rotated order: rho, p, v^K v^K1 v^K2, E.., B.., psi, phi, q, jc^K
  const double* M[3][8];     // alpha, beta^K, gamma rotated: 00 01 02 11 12 22 (0 = K, 1 = K+1, 2 = K+2)
  int nat[3][NCONS];         // rotated conserved index -> natural conserved index
};

struct Smem {
  double ex[NVR][EXP];       // upper-face states of the tile's cells (+ lower halo); later the face fluxes
  double exlo[NVR][TX];      // lower-face states of the upper-halo cells
  double exhi[NVR][TX];      // upper-face states of the last interior row/column (left states of the edge faces)
  double chi[NVR][NT];       // z carry: upper-face states of the current plane (left states of its upper z faces)
  double du[NCONS][NT];      // flux divergence being accumulated for the current plane (thread-private slots)
};

struct FaceMet {
  double alpha, b0, g[6], gi0[3], sg;
};

// reading R2: face metric = arithmetic mean of the two adjacent centres; sqrt(gamma) and the K-row of
// gamma^ij from the averaged gamma_ij (rotated components)
__device__ __forceinline__ void load_face_met(const PencilTabs& T, int K, long long cl, long long cr, FaceMet& m) {
  m.alpha = 0.5 * (__ldg(T.M[K][0] + cl) + __ldg(T.M[K][0] + cr));
  m.b0 = 0.5 * (__ldg(T.M[K][1] + cl) + __ldg(T.M[K][1] + cr));
#pragma unroll
  for (int q = 0; q < 6; ++q) m.g[q] = 0.5 * (__ldg(T.M[K][2 + q] + cl) + __ldg(T.M[K][2 + q] + cr));
  const double c00 = m.g[3] * m.g[5] - m.g[4] * m.g[4];
  const double c01 = m.g[2] * m.g[4] - m.g[1] * m.g[5];
  const double c02 = m.g[1] * m.g[4] - m.g[2] * m.g[3];
  const double det = m.g[0] * c00 + m.g[1] * c01 + m.g[2] * c02;
  const double idet = rcp_fast(det);
  m.sg = sqrt_fast(det);
  m.gi0[0] = c00 * idet; m.gi0[1] = c01 * idet; m.gi0[2] = c02 * idet;
}

// a3, one state.  X = (rho, p, v[3], E[3], B[3], psi, phi, q, jc^0) in the rotated frame (0 = face normal).
// Adds wa*G + wu*U to Fh, where F = alpha G - beta^0 U is Eq. 27 (reading R1), i.e. the
// state's share w F + sd U of the HLLE flux with wa = w alpha, wu = sd - w beta^0.
template <int CHARGE, bool FIRST>
__device__ __forceinline__ void half_flux(const FaceMet& m, double Gamma, const double X[NVR], double sigma,
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
  const double h = rho + Gamma / (Gamma - 1.0) * p;              // rho(1+eps)+p with Eq. 49
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
    const double t = wa * Gf[c] + wu * U[c];
    Fh[c] = FIRST ? t : Fh[c] + t;
  }
}

// stencil of one variable along one direction (TVD uses the inner three values only)
template <int RECON>
__device__ __forceinline__ void load_stencil(const double* __restrict__ f, long long s, double u[5]) {
  if (RECON == RECON_WENO5) { u[0] = f[-2 * s]; u[4] = f[2 * s]; } else { u[0] = 0.0; u[4] = 0.0; }
  u[1] = f[-s]; u[2] = f[0]; u[3] = f[s];
}

// a2 for the thread's own cell along direction K, all variables: lower-face values stay in lo[]
// (registers), upper-face values go to hi_dst (strided) and, for the last cell of a row / column, also
// to hi2_dst.  The loads run PF variables ahead of the arithmetic (software pipeline in registers).
template <int RECON, int NV>
__device__ __forceinline__ void recon_own(const PencilTabs& T, int K, long long ct, long long s, double eps_w,
                                          double lo[NVR], double* __restrict__ hi_dst, int hi_stride,
                                          double* __restrict__ hi2_dst, bool st_hi2) {
  constexpr int PF = 2;
  double buf[PF + 1][5];
#pragma unroll
  for (int vr = 0; vr < PF && vr < NV; ++vr) load_stencil<RECON>(T.P[K][vr] + ct, s, buf[vr]);
#pragma unroll
  for (int vr = 0; vr < NV; ++vr) {
    if (vr + PF < NV) load_stencil<RECON>(T.P[K][vr + PF] + ct, s, buf[(vr + PF) % (PF + 1)]);
    const double* u = buf[vr % (PF + 1)];
    double l, h;
    recon_cell<RECON>(eps_w, u[0], u[1], u[2], u[3], u[4], l, h);
    if (vr < 2) {   // reading R4: unphysical face values fall back to the cell value
      if (!(l > 0.0)) l = u[2];
      if (!(h > 0.0)) h = u[2];
    }
    lo[vr] = l;
    hi_dst[vr * hi_stride] = h;
    if (st_hi2) hi2_dst[vr * TX] = h;
  }
}

// a2 for the halo cells of the tile (x, y only): the cell below the tile's first row / column gives the
// left state of the tile's first faces (its upper-face value -> ex halo slot); the cell above the last
// row / column gives the right state of the tile's edge faces (its lower-face value -> exlo).  Work
// unit = (variable, lower | upper) x one lane per row (x: 2*TY lanes) or per column (y: TX lanes);
// the units are dealt round-robin to the TY warps so that every warp carries the same extra load.
template <int RECON, int NV>
__device__ __forceinline__ void recon_halo(const PencilTabs& T, int K, Smem& S, long long c, long long s, long long sy,
                                           double eps_w, int tx, int ty, int txn, int tyn) {
  const int nunits = (K == 0) ? NV : 2 * NV;
  bool upper, valid;
  int r;
  long long cell;
  if (K == 0) {
    r = tx % TY; upper = (tx / TY) == 1; valid = tx < 2 * TY && r < tyn;
    cell = c + (long long)((upper ? txn : -1) - tx) + sy * (long long)(r - ty);
  } else {
    r = tx; upper = false; valid = tx < txn;
    cell = 0;
  }
  double cur[5], nxt[5];
  auto unit_ptr = [&](int u, bool& up_u) -> const double* {
    if (K == 0) { up_u = upper; return T.P[K][u] + cell; }
    up_u = (u & 1) != 0;
    return T.P[K][u >> 1] + (c + sy * (long long)((up_u ? tyn : -1) - ty));
  };
  bool up_c = false, up_n = false;
  int u = ty;
  if (valid && u < nunits) load_stencil<RECON>(unit_ptr(u, up_c), s, cur);
#pragma unroll 1
  while (u < nunits) {
    const int un = u + TY;
    if (valid && un < nunits) load_stencil<RECON>(unit_ptr(un, up_n), s, nxt);
    if (valid) {
      const int vr = (K == 0) ? u : (u >> 1);
      double l, h;
      recon_cell<RECON>(eps_w, cur[0], cur[1], cur[2], cur[3], cur[4], l, h);
      if (vr < 2) {
        if (!(l > 0.0)) l = cur[2];
        if (!(h > 0.0)) h = cur[2];
      }
      if (up_c) S.exlo[vr][r] = l;
      else S.ex[vr][(K == 0) ? r * EXW : r] = h;
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) cur[q] = nxt[q];
    up_c = up_n;
    u = un;
  }
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

// a3 for one face: right state PR (registers), left state read from plp (strided); F in the rotated order
template <int CHARGE, int NV>
__device__ __forceinline__ void riemann(const GridView& G, const PencilTabs& T, int K, long long cl, long long cr,
                                        const double* __restrict__ plp, int pl_stride, double PR[NVR], double Fh[NCONS]) {
  FaceMet m;
  load_face_met(T, K, cl, cr, m);
  // HLLE weights (Eq. 30; reading R6)
  const double c = m.alpha * sqrt_fast(m.gi0[0]);
  const double lp = fmax(0.0, c - m.b0), lm = fmin(0.0, -c - m.b0);
  const double inv = rcp_fast(lp - lm);
  const double wL = lp * inv, wR = -lm * inv, sd = lp * lm * inv;
  double sigL = 0.0, sigR = 0.0;
  if (CHARGE == CHARGE_FACE_OHM) { sigL = sigma_cell(G, cl); sigR = sigma_cell(G, cr); }
  if (NV < NVR) PR[NVR - 1] = 0.0;
  half_flux<CHARGE, true>(m, G.Gamma, PR, sigR, wR * m.alpha, sd - wR * m.b0, Fh);
  double PL[NVR];
#pragma unroll
  for (int vr = 0; vr < NV; ++vr) PL[vr] = plp[vr * pl_stride];
  if (NV < NVR) PL[NVR - 1] = 0.0;
  half_flux<CHARGE, false>(m, G.Gamma, PL, sigL, wL * m.alpha, -sd - wL * m.b0, Fh);
}
}  // namespace

template <int RECON, int CHARGE, int STAGE>
__global__ void __launch_bounds__(NT, 2)
k_rhs_pencil(const __grid_constant__ GridView G, const __grid_constant__ PencilTabs T, double dt, int CZ) {
  constexpr int NV = (CHARGE == CHARGE_CELL_CURRENT) ? NVR : NVR - 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& S = *reinterpret_cast<Smem*>(smem_raw);
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int txn = min(TX, G.n[0] - i0), tyn = min(TY, G.n[1] - j0);   // valid extent of this tile
  const bool in = tx < txn && ty < tyn;
  const int k0 = blockIdx.z * CZ, k1 = min(k0 + CZ, G.n[2]);
  const long long sy = G.stride[1], sz = G.stride[2];
  const int base = ty * EXW + tx;                                     // own flux slot = slot of the left state
  long long c = cell_index(G, i0 + tx, j0 + ty, k0 - 2);
  // k = k0-2: upper-face z states of plane k0-1; k = k0-1: z flux through the lower face of plane k0
  for (int k = k0 - 2; k < k1; ++k, c += sz) {
    const bool lead = k < k0;
#pragma unroll 1
    for (int K = lead ? 2 : 0; K < 3; ++K) {
      const long long s = G.stride[K];
      const int up = (K == 0) ? 1 : (K == 1) ? EXW : 0;                // own upper-face slot relative to base
      const long long cm = (K == 2) ? c + sz : c;                      // the cell this thread reconstructs
      double lo[NVR];
      // ---- a2: reconstruction (halo cells of the tile: all warps share them; then the own cell)
      if (K < 2) recon_halo<RECON, NV>(T, K, S, c, s, sy, G.weno_eps, tx, ty, txn, tyn);
      if (in) {
        const bool edge = (K == 0) ? (tx == txn - 1) : (K == 1) ? (ty == tyn - 1) : false;
        recon_own<RECON, NV>(T, K, cm, s, G.weno_eps, lo, &S.ex[0][base + up], EXP, &S.exhi[0][(K == 0) ? ty : tx], edge);
      }
      if (K < 2) __syncthreads();                                      // A: upper-face states visible
      // ---- a3: Riemann passes (p = 0: own lower face (x, y) / upper face (z); p = 1: faces on the tile's upper edge)
      {
        bool e_valid = false;
        int e_r = 0;
        if (K == 0 && ty == TY - 1 && tx < tyn) { e_valid = true; e_r = tx; }
        if (K == 1 && ty == TY - 1 && tx < txn) { e_valid = true; e_r = tx; }
#pragma unroll 1
        for (int p = 0; p < 2; ++p) {
          bool valid;
          long long cr;
          const double* plp;
          int pls, dst;
          if (p == 0) {
            valid = in && k >= k0 - 1; cr = cm; dst = base;
            plp = (K == 2) ? &S.chi[0][tid] : &S.ex[0][base];
            pls = (K == 2) ? NT : EXP;
          } else {
            valid = e_valid; plp = &S.exhi[0][e_r]; pls = TX;
            if (K == 0) { cr = c + (long long)(txn - tx) + sy * (long long)(e_r - ty); dst = e_r * EXW + txn; }
            else        { cr = c + sy * (long long)(tyn - ty); dst = tyn * EXW + e_r; }
            if (valid) {
#pragma unroll
              for (int vr = 0; vr < NV; ++vr) lo[vr] = S.exlo[vr][e_r];
            }
          }
          double F[NCONS];
          if (valid) riemann<CHARGE, NV>(G, T, K, cr - s, cr, plp, pls, lo, F);
          if (p == 0) {
            if (K < 2) __syncthreads();                                // B: every left state has been read
            else if (in) {                                             // z: the new upper-face states become the carry
#pragma unroll
              for (int vr = 0; vr < NV; ++vr) S.chi[vr][tid] = S.ex[vr][base];
            }
          }
          if (valid) {
#pragma unroll
            for (int v = 0; v < NCONS; ++v) S.ex[T.nat[K][v]][dst] = F[v];
          }
        }
      }
      if (K < 2) {
        __syncthreads();                                               // C: fluxes visible
        if (in) {
          const double idx = G.inv_dx[K];
#pragma unroll
          for (int v = 0; v < NCONS; ++v) S.du[v][tid] -= (S.ex[v][base + up] - S.ex[v][base]) * idx;
        }
      }
    }
    if (in && k >= k0 - 1) {
      double dU[NCONS];
#pragma unroll
      for (int v = 0; v < NCONS; ++v) {
        const double Fz = S.ex[v][base] * G.inv_dx[2];
        dU[v] = S.du[v][tid] - Fz;
        S.du[v][tid] = Fz;                                             // lower z face of the next plane
      }
      if (k >= k0) divergence_update<STAGE>(G, c, dt, dU);             // a5 (divergence part)
    }
    __syncthreads();                                                   // D: exchange buffer free for the next plane
  }
}

bool rhs_pencil_supported(const GridView& G) {
  return G.n[0] > 1 && G.n[1] > 1 && G.n[2] > 1;
}

static int choose_cz(const GridView& G) {
  // several waves of 148 SMs x 2 CTAs, but long enough pencils to amortise the two lead-in planes
  const long long tiles = (long long)((G.n[0] + TX - 1) / TX) * ((G.n[1] + TY - 1) / TY);
  int cz = 64;
  while (cz > 8 && tiles * ((G.n[2] + cz - 1) / cz) < 148LL * 2 * 4) cz /= 2;
  return cz;
}

static PencilTabs make_tabs(const GridView& G) {
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

template <int RECON, int CHARGE, int STAGE>
static cudaError_t launch_one(const GridView& G, double dt, cudaStream_t st) {
  const int cz = choose_cz(G);
  const PencilTabs T = make_tabs(G);
  dim3 block(TX, TY, 1);
  dim3 grid((G.n[0] + TX - 1) / TX, (G.n[1] + TY - 1) / TY, (G.n[2] + cz - 1) / cz);
  const size_t smem = sizeof(Smem);
  cudaError_t e = cudaFuncSetAttribute(k_rhs_pencil<RECON, CHARGE, STAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_rhs_pencil<RECON, CHARGE, STAGE><<<grid, block, smem, st>>>(G, T, dt, cz);
  return cudaGetLastError();
}

template <int RECON, int CHARGE>
static cudaError_t launch_rc(const GridView& G, double dt, int stage, cudaStream_t st) {
  return stage == 1 ? launch_one<RECON, CHARGE, 1>(G, dt, st) : launch_one<RECON, CHARGE, 2>(G, dt, st);
}

cudaError_t launch_rhs_pencil(const GridView& G, double dt, int stage, int recon, cudaStream_t st) {
  const bool ohm = G.charge_mode == CHARGE_FACE_OHM;
  switch (recon) {
    case RECON_MINMOD:
      return ohm ? launch_rc<RECON_MINMOD, CHARGE_FACE_OHM>(G, dt, stage, st)
                 : launch_rc<RECON_MINMOD, CHARGE_CELL_CURRENT>(G, dt, stage, st);
    case RECON_MC:
      return ohm ? launch_rc<RECON_MC, CHARGE_FACE_OHM>(G, dt, stage, st)
                 : launch_rc<RECON_MC, CHARGE_CELL_CURRENT>(G, dt, stage, st);
    default:
      return ohm ? launch_rc<RECON_WENO5, CHARGE_FACE_OHM>(G, dt, stage, st)
                 : launch_rc<RECON_WENO5, CHARGE_CELL_CURRENT>(G, dt, stage, st);
  }
}

}  // namespace rg
