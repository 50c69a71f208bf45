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
//   a5  the increment dt dU or dt/2 dU is written once per cell (G.dU, write only); the next recovery kernel adds it.
// The three directions run through ONE copy of the reconstruction and Riemann code: direction K is a
// run-time cyclic rotation of the vector/tensor components (cyclic permutations keep the Levi-Civita
// sign, so Eq. 27 is form invariant), realised for free as index arithmetic on pointer tables and
// shared-memory planes.  This keeps the kernel ~4x smaller than the fully templated version, whose
// instruction-cache misses dominated its stall profile.
// Stencils are read straight from global memory (x: coalesced rows, L1; y: L1; z: L2).
#include "rgrmhd_flux_rot.cuh"

namespace rg {

namespace {
constexpr int TX = 32, TY = 8, NT = TX * TY;
constexpr int EXW = TX + 1, EXH = TY + 1, EXP = EXW * EXH;
struct Smem {
  double ex[NVR][EXP];       // upper-face states of the tile's cells (+ lower halo); later the face fluxes
  double exlo[NVR][TX];      // lower-face states of the upper-halo cells
  double exhi[NVR][TX];      // upper-face states of the last interior row/column (left states of the edge faces)
  double chi[NVR][NT];       // z carry: upper-face states of the current plane (left states of its upper z faces)
  double du[NCONS][NT];      // flux divergence being accumulated for the current plane (thread-private slots)
};

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

static int choose_cz(const GridView& G, int sm_count) {
  // several waves of (SM count) x 2 CTAs, but long enough pencils to amortise the two lead-in planes
  const long long tiles = (long long)((G.n[0] + TX - 1) / TX) * ((G.n[1] + TY - 1) / TY);
  int cz = 64;
  while (cz > 8 && tiles * ((G.n[2] + cz - 1) / cz) < (long long)sm_count * 2 * 4) cz /= 2;
  return cz;
}

template <int RECON, int CHARGE, int STAGE>
static cudaError_t launch_one(const GridView& G, double dt, int sm_count, cudaStream_t st) {
  const int cz = choose_cz(G, sm_count);
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
static cudaError_t launch_rc(const GridView& G, double dt, int stage, int sm_count, cudaStream_t st) {
  return stage == 1 ? launch_one<RECON, CHARGE, 1>(G, dt, sm_count, st) : launch_one<RECON, CHARGE, 2>(G, dt, sm_count, st);
}

cudaError_t launch_rhs_pencil(const GridView& G, double dt, int stage, int recon, int sm_count, cudaStream_t st) {
  const bool ohm = G.charge_mode == CHARGE_FACE_OHM;
  switch (recon) {
    case RECON_MINMOD:
      return ohm ? launch_rc<RECON_MINMOD, CHARGE_FACE_OHM>(G, dt, stage, sm_count, st)
                 : launch_rc<RECON_MINMOD, CHARGE_CELL_CURRENT>(G, dt, stage, sm_count, st);
    case RECON_MC:
      return ohm ? launch_rc<RECON_MC, CHARGE_FACE_OHM>(G, dt, stage, sm_count, st)
                 : launch_rc<RECON_MC, CHARGE_CELL_CURRENT>(G, dt, stage, sm_count, st);
    default:
      return ohm ? launch_rc<RECON_WENO5, CHARGE_FACE_OHM>(G, dt, stage, sm_count, st)
                 : launch_rc<RECON_WENO5, CHARGE_CELL_CURRENT>(G, dt, stage, sm_count, st);
  }
}

}  // namespace rg
