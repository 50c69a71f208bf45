// rgrmhd_rhs_tiled.cu -- the production RHS kernel (a2-a5): reconstruct + HLLE + flux divergence +
// explicit sources + IMEX stage combine in ONE launch, every face computed exactly once, face states
// and fluxes never leaving the SM.
//
// Decomposition ("pencil-tiled"): a CTA owns a TX x TY (x, y) tile of z-pencils and marches CZ planes
// along z.  Per plane and thread (= one cell):
//   z   the flux through the cell's upper z-face is computed and differenced against the flux kept
//       from the previous plane (shared memory, thread-private slot) -> no z-face is computed twice;
//   x,y the flux through the cell's lower x- and y-face goes to shared memory; the TY + TX faces on the
//       tile's upper x / y boundary are computed by two warps in an extra pass; after one barrier every
//       cell differences its own and its neighbour's flux;
//   the divergence accumulates in registers, then the geometric sources (a4) and the stage combine (a5)
//   are applied and U*2 / U^{n+1} is written once.
// Reconstruction stencils are read straight from global memory: along x they are coalesced and hit L1,
// along y they hit L1 (the tile's rows + 6 halo rows), along z they hit L2 (6 planes of the tile).
// Grid: (ceil(nx/TX), ceil(ny/TY), ceil(nz/CZ)); CZ is chosen so that the grid has several waves of
// 148 SMs x 2 resident CTAs.
#include "rgrmhd_rhs.cuh"

namespace rg {

namespace {
constexpr int TX = 32, TY = 8, NT = TX * TY;

struct TileSmem {
  double Fx[NCONS][TY][TX + 1];
  double Fy[NCONS][TY + 1][TX];
  double Fz[NCONS][NT];
};
}  // namespace

template <int RECON, int CHARGE, int STAGE>
__global__ void __launch_bounds__(NT, 2)
k_rhs_tiled(const __grid_constant__ GridView G, double dt, int CZ) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileSmem& S = *reinterpret_cast<TileSmem*>(smem_raw);
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int txn = min(TX, G.n[0] - i0), tyn = min(TY, G.n[1] - j0);   // valid extent of this tile
  const int i = i0 + tx, j = j0 + ty;
  const bool in = tx < txn && ty < tyn;
  const int k0 = blockIdx.z * CZ, k1 = min(k0 + CZ, G.n[2]);
  const long long sz = G.stride[2];
  long long c = cell_index(G, i, j, k0);
  double F[NCONS];
  if (in) {
    face_flux<2, RECON, CHARGE>(G, c, F);
#pragma unroll
    for (int v = 0; v < NCONS; ++v) S.Fz[v][tid] = F[v];
  }
  for (int k = k0; k < k1; ++k, c += sz) {
    double dU[NCONS];
    if (in) {
      face_flux<2, RECON, CHARGE>(G, c + sz, F);
#pragma unroll
      for (int v = 0; v < NCONS; ++v) {
        dU[v] = -(F[v] - S.Fz[v][tid]) * G.inv_dx[2];
        S.Fz[v][tid] = F[v];
      }
      face_flux<0, RECON, CHARGE>(G, c, F);
#pragma unroll
      for (int v = 0; v < NCONS; ++v) S.Fx[v][ty][tx] = F[v];
      face_flux<1, RECON, CHARGE>(G, c, F);
#pragma unroll
      for (int v = 0; v < NCONS; ++v) S.Fy[v][ty][tx] = F[v];
    }
    // extra pass: faces on the tile's upper y boundary (warp 0) and upper x boundary (warp 1)
    if (ty == 0 && tx < txn) {
      face_flux<1, RECON, CHARGE>(G, cell_index(G, i0 + tx, j0 + tyn, k), F);
#pragma unroll
      for (int v = 0; v < NCONS; ++v) S.Fy[v][tyn][tx] = F[v];
    } else if (ty == 1 && tx < tyn) {
      face_flux<0, RECON, CHARGE>(G, cell_index(G, i0 + txn, j0 + tx, k), F);
#pragma unroll
      for (int v = 0; v < NCONS; ++v) S.Fx[v][tx][txn] = F[v];
    }
    __syncthreads();
    if (in) {
#pragma unroll
      for (int v = 0; v < NCONS; ++v) {
        dU[v] -= (S.Fx[v][ty][tx + 1] - S.Fx[v][ty][tx]) * G.inv_dx[0];
        dU[v] -= (S.Fy[v][ty + 1][tx] - S.Fy[v][ty][tx]) * G.inv_dx[1];
      }
      double P[NPRIM];
#pragma unroll
      for (int v = 0; v < NPRIM; ++v) P[v] = G.P[v][c];
      add_sources(G, c, P, dU);
      Met m;
#pragma unroll
      for (int q = 0; q < 6; ++q) m.g[q] = __ldg(G.met[MGXX + q] + c);
      met_finish(m);
      const double sgE[3] = {m.sg * P[EX], m.sg * P[EY], m.sg * P[EZ]};
      stage_combine<STAGE>(G, c, dt, dU, sgE);
    }
    __syncthreads();
  }
}

bool rhs_tiled_supported(const GridView& G) {
  return G.n[0] > 1 && G.n[1] > 1 && G.n[2] > 1;
}

static int choose_cz(const GridView& G) {
  // several waves of 148 SMs x 2 CTAs, but long enough pencils to amortise the first z-face
  const long long tiles = (long long)((G.n[0] + TX - 1) / TX) * ((G.n[1] + TY - 1) / TY);
  int cz = 32;
  while (cz > 8 && tiles * ((G.n[2] + cz - 1) / cz) < 148LL * 2 * 6) cz /= 2;
  return cz;
}

template <int RECON, int CHARGE>
static cudaError_t launch_rhs_tiled_rc(const GridView& G, double dt, int stage, cudaStream_t st) {
  const int cz = choose_cz(G);
  dim3 block(TX, TY, 1);
  dim3 grid((G.n[0] + TX - 1) / TX, (G.n[1] + TY - 1) / TY, (G.n[2] + cz - 1) / cz);
  const size_t smem = sizeof(TileSmem);
  cudaError_t e;
  if (stage == 1) {
    e = cudaFuncSetAttribute(k_rhs_tiled<RECON, CHARGE, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_rhs_tiled<RECON, CHARGE, 1><<<grid, block, smem, st>>>(G, dt, cz);
  } else {
    e = cudaFuncSetAttribute(k_rhs_tiled<RECON, CHARGE, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_rhs_tiled<RECON, CHARGE, 2><<<grid, block, smem, st>>>(G, dt, cz);
  }
  return cudaGetLastError();
}

cudaError_t launch_rhs_tiled(const GridView& G, double dt, int stage, int recon, cudaStream_t st) {
  const int ch = G.charge_mode;
  switch (recon) {
    case RECON_MINMOD:
      return ch == CHARGE_FACE_OHM ? launch_rhs_tiled_rc<RECON_MINMOD, CHARGE_FACE_OHM>(G, dt, stage, st)
                                   : launch_rhs_tiled_rc<RECON_MINMOD, CHARGE_CELL_CURRENT>(G, dt, stage, st);
    case RECON_MC:
      return ch == CHARGE_FACE_OHM ? launch_rhs_tiled_rc<RECON_MC, CHARGE_FACE_OHM>(G, dt, stage, st)
                                   : launch_rhs_tiled_rc<RECON_MC, CHARGE_CELL_CURRENT>(G, dt, stage, st);
    default:
      return ch == CHARGE_FACE_OHM ? launch_rhs_tiled_rc<RECON_WENO5, CHARGE_FACE_OHM>(G, dt, stage, st)
                                   : launch_rhs_tiled_rc<RECON_WENO5, CHARGE_CELL_CURRENT>(G, dt, stage, st);
  }
}

}  // namespace rg
