// rgrmhd_rhs_simple.cu -- reference-quality flux-divergence kernel (a2, a3, divergence): one thread per
// interior cell, each thread evaluates the HLLE flux at all of its (up to six) faces straight from global
// memory.  Every face is therefore computed twice; this kernel exists as the simplest correct CUDA
// statement of the flux divergence (rgrmhd_set_rhs_variant(1), and block shapes with an inactive
// direction) and as the in-library cross-check of the tiled kernels.  Also here: a1 ghost fill and a7
// max-speed reduction.
#include "rgrmhd_rhs.cuh"

namespace rg {

template <int RECON, int CHARGE, int STAGE>
__global__ void __launch_bounds__(128)
k_rhs_simple(const __grid_constant__ GridView G, double dt) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nint) return;
  const int i = (int)(t % nx);
  const long long r = t / nx;
  const int j = (int)(r % ny), k = (int)(r / ny);
  const long long c = cell_index(G, i, j, k);
  double F[NCONS];
#pragma unroll
  for (int v = 0; v < NCONS; ++v) F[v] = 0.0;
  double Fm[NCONS], Fp[NCONS];
  if (G.n[0] > 1) {
    face_flux<0, RECON, CHARGE>(G, c, Fm);
    face_flux<0, RECON, CHARGE>(G, c + G.stride[0], Fp);
#pragma unroll
    for (int v = 0; v < NCONS; ++v) F[v] -= (Fp[v] - Fm[v]) * G.inv_dx[0];
  }
  if (G.n[1] > 1) {
    face_flux<1, RECON, CHARGE>(G, c, Fm);
    face_flux<1, RECON, CHARGE>(G, c + G.stride[1], Fp);
#pragma unroll
    for (int v = 0; v < NCONS; ++v) F[v] -= (Fp[v] - Fm[v]) * G.inv_dx[1];
  }
  if (G.n[2] > 1) {
    face_flux<2, RECON, CHARGE>(G, c, Fm);
    face_flux<2, RECON, CHARGE>(G, c + G.stride[2], Fp);
#pragma unroll
    for (int v = 0; v < NCONS; ++v) F[v] -= (Fp[v] - Fm[v]) * G.inv_dx[2];
  }
  divergence_update<STAGE>(G, c, dt, F);
}

template <int RECON, int CHARGE>
static cudaError_t launch_rhs_simple_rc(const GridView& G, double dt, int stage, cudaStream_t st) {
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  const int threads = 128;
  const unsigned blocks = (unsigned)((nint + threads - 1) / threads);
  if (stage == 1) k_rhs_simple<RECON, CHARGE, 1><<<blocks, threads, 0, st>>>(G, dt);
  else k_rhs_simple<RECON, CHARGE, 2><<<blocks, threads, 0, st>>>(G, dt);
  return cudaGetLastError();
}

cudaError_t launch_rhs_simple(const GridView& G, double dt, int stage, int recon, cudaStream_t st) {
  const int ch = G.charge_mode;
  switch (recon) {
    case RECON_MINMOD:
      return ch == CHARGE_FACE_OHM ? launch_rhs_simple_rc<RECON_MINMOD, CHARGE_FACE_OHM>(G, dt, stage, st)
                                   : launch_rhs_simple_rc<RECON_MINMOD, CHARGE_CELL_CURRENT>(G, dt, stage, st);
    case RECON_MC:
      return ch == CHARGE_FACE_OHM ? launch_rhs_simple_rc<RECON_MC, CHARGE_FACE_OHM>(G, dt, stage, st)
                                   : launch_rhs_simple_rc<RECON_MC, CHARGE_CELL_CURRENT>(G, dt, stage, st);
    default:
      return ch == CHARGE_FACE_OHM ? launch_rhs_simple_rc<RECON_WENO5, CHARGE_FACE_OHM>(G, dt, stage, st)
                                   : launch_rhs_simple_rc<RECON_WENO5, CHARGE_CELL_CURRENT>(G, dt, stage, st);
  }
}

// ------------------------------------------------------------------------------------------------
// a1. ghost fill ("copied from the nearest interior point"; PAPER.md:359 periodic;
// reading R10).  Filling x, then y, then z over the full padded extent is the same as mapping every
// coordinate of a ghost cell independently into the interior (wrap or clamp), so one launch does all
// three directions.  One thread per (ghost cell, field group); NF fields share the index arithmetic.
// ------------------------------------------------------------------------------------------------
struct GhostArgs {
  double* f[NPRIM + 3];
  int nf;
};

__device__ __forceinline__ int ghost_src(int a, int n, int bc) {
  // a = interior-relative coordinate in [-3, n+3)
  if (a >= 0 && a < n) return a;
  if (bc == BC_EXTERNAL) return a;                 // ghost layers owned by the caller (halo exchange): identity
  if (bc == BC_PERIODIC) return a < 0 ? a + n : a - n;
  return a < 0 ? 0 : n - 1;
}

__global__ void __launch_bounds__(256)
k_ghost_fill(const __grid_constant__ GridView G, const __grid_constant__ GhostArgs A, long long nghost_x,
             long long nghost_y, long long nghost_z) {
  // Ghost cells are enumerated as three slab families:
  //  X: i in ghosts (2*3 values), all padded j, k              -> 6 * nyp * nzp cells
  //  Y: i interior, j in ghosts, all padded k                  -> nx * 6 * nzp
  //  Z: i, j interior, k in ghosts                             -> nx * ny * 6
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int pi, pj, pk;   // padded coordinates
  if (t < nghost_x) {
    const int gi = (int)(t % 6);
    const long long r = t / 6;
    pj = (int)(r % G.np[1]); pk = (int)(r / G.np[1]);
    pi = gi < 3 ? gi : G.n[0] + gi;                 // 0,1,2, n+3, n+4, n+5
  } else if ((t -= nghost_x) < nghost_y) {
    const int ii = (int)(t % G.n[0]);
    const long long r = t / G.n[0];
    const int gj = (int)(r % 6);
    pk = (int)(r / 6);
    pi = ii + G.g[0];
    pj = gj < 3 ? gj : G.n[1] + gj;
  } else if ((t -= nghost_y) < nghost_z) {
    const int ii = (int)(t % G.n[0]);
    const long long r = t / G.n[0];
    const int jj = (int)(r % G.n[1]);
    const int gk = (int)(r / G.n[1]);
    pi = ii + G.g[0]; pj = jj + G.g[1];
    pk = gk < 3 ? gk : G.n[2] + gk;
  } else {
    return;
  }
  const int si = ghost_src(pi - G.g[0], G.n[0], G.bc[0]) + G.g[0];
  const int sj = ghost_src(pj - G.g[1], G.n[1], G.bc[1]) + G.g[1];
  const int sk = ghost_src(pk - G.g[2], G.n[2], G.bc[2]) + G.g[2];
  const long long dst = pi + G.stride[1] * pj + G.stride[2] * pk;
  const long long src = si + G.stride[1] * sj + G.stride[2] * sk;
  if (dst == src) return;                          // every ghost coordinate of this cell is the caller's
  for (int v = 0; v < A.nf; ++v) A.f[v][dst] = A.f[v][src];
}

cudaError_t launch_ghost_fill(const GridView& G, double* const* fields, int nf, cudaStream_t st) {
  GhostArgs A;
  A.nf = nf;
  for (int v = 0; v < nf; ++v) A.f[v] = fields[v];
  const long long gx = G.n[0] > 1 ? 6LL * G.np[1] * G.np[2] : 0;
  const long long gy = G.n[1] > 1 ? 6LL * G.n[0] * G.np[2] : 0;
  const long long gz = G.n[2] > 1 ? 6LL * G.n[0] * G.n[1] : 0;
  const long long tot = gx + gy + gz;
  if (tot == 0) return cudaSuccess;
  const int threads = 256;
  k_ghost_fill<<<(unsigned)((tot + threads - 1) / threads), threads, 0, st>>>(G, A, gx, gy, gz);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Halo layers for a caller that owns the ghost zones of a direction (bc = BC_EXTERNAL): pack =
// the three interior layers next to `side` of direction `dir`, over the FULL padded extent of the other two directions
// (so that a neighbour receives the ghost columns this block has just filled in those directions: the result equals
// the single-block fill x, then y, then z), into buf[field][layer][plane]; unpack = buf into the three ghost layers.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_halo_copy(const __grid_constant__ GridView G, const __grid_constant__ GhostArgs A, int dir, int side, double* __restrict__ buf,
            int pack, long long plane) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 3 * plane) return;
  const int layer = (int)(t / plane);
  const long long r = t % plane;
  const int d1 = (dir == 0) ? 1 : 0, d2 = (dir == 2) ? 1 : 2;          // the other two directions, d1 faster
  int p[3];
  p[d1] = (int)(r % G.np[d1]);
  p[d2] = (int)(r / G.np[d1]);
  // padded coordinate of the layer: interior layers [g, g+3) or [g+n-3, g+n) for pack; ghost layers [0, 3) or [g+n, g+n+3) for unpack
  const int g = G.g[dir], n = G.n[dir];
  p[dir] = pack ? (side == 0 ? g + layer : g + n - 3 + layer) : (side == 0 ? layer : g + n + layer);
  const long long c = p[0] + G.stride[1] * p[1] + G.stride[2] * p[2];
  for (int v = 0; v < A.nf; ++v) {
    double* b = buf + ((long long)v * 3 + layer) * plane + r;
    if (pack) *b = A.f[v][c]; else A.f[v][c] = *b;
  }
}

cudaError_t launch_halo_copy(const GridView& G, double* const* fields, int nf, int dir, int side, double* buf, bool pack,
                             cudaStream_t st) {
  GhostArgs A;
  A.nf = nf;
  for (int v = 0; v < nf; ++v) A.f[v] = fields[v];
  long long plane = 1;
  for (int d = 0; d < 3; ++d) if (d != dir) plane *= G.np[d];
  k_halo_copy<<<(unsigned)((3 * plane + 255) / 256), 256, 0, st>>>(G, A, dir, side, buf, pack ? 1 : 0, plane);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// A22. charge mode DIV_E (reading R15): q = nabla_i E^i = d_i(sqrt(gamma) E^i)/sqrt(gamma) of the
// stage, second-order centred differences (inactive directions dropped), from the ghost-filled stage primitives.
// Writes q into P and applies the two explicit source terms that carry the charge,
//   S(calE^i) -= alpha calQ v^i,   S(Psi) += alpha calQ            (Eq. 27 / reading R1),
// to the bracket of the next stage vector (STAGE 1: U*2 += dt ...; STAGE 2: U^{n+1} += dt/2 ...);
// STAGE 3 (new state, on output): q and calQ = sqrt(gamma) q only; STAGE 0 (general tableau driver): q only.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double sqrtg_cell(const GridView& G, long long c) {
  const double gxx = __ldg(G.met[MGXX] + c), gxy = __ldg(G.met[MGXY] + c), gxz = __ldg(G.met[MGXZ] + c);
  const double gyy = __ldg(G.met[MGYY] + c), gyz = __ldg(G.met[MGYZ] + c), gzz = __ldg(G.met[MGZZ] + c);
  return sqrt(gxx * (gyy * gzz - gyz * gyz) + gxy * (gxz * gyz - gxy * gzz) + gxz * (gxy * gyz - gxz * gyy));
}

template <int STAGE>
__global__ void __launch_bounds__(128)
k_charge_div_e(const __grid_constant__ GridView G, double dt) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nint) return;
  const int i = (int)(t % nx);
  const long long r = t / nx;
  const long long c = cell_index(G, i, (int)(r % ny), (int)(r / ny));
  double div = 0.0;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (G.n[d] > 1) {
      const long long s = G.stride[d];
      div += (sqrtg_cell(G, c + s) * G.P[EX + d][c + s] - sqrtg_cell(G, c - s) * G.P[EX + d][c - s]) * (0.5 * G.inv_dx[d]);
    }
  }
  G.P[QCH][c] = div / sqrtg_cell(G, c);
  if (STAGE == 0) {
    // general tableau driver: q only; k_charge_sources_gen distributes the source terms
  } else if (STAGE == 3) {
    G.Un[CQ][c] = div;
  } else {
    const double w = (STAGE == 1) ? dt : 0.5 * dt, aq = __ldg(G.met[MALP] + c) * div;
    double* const* T = (STAGE == 1) ? G.Us : G.Un;
#pragma unroll
    for (int a = 0; a < 3; ++a) T[CEX + a][c] -= w * aq * G.P[VX + a][c];
    T[CPSI][c] += w * aq;
  }
}

cudaError_t launch_charge_div_e(const GridView& G, int stage, double dt, cudaStream_t st) {
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  const int threads = 128;
  const unsigned blocks = (unsigned)((nint + threads - 1) / threads);
  if (stage == 0) k_charge_div_e<0><<<blocks, threads, 0, st>>>(G, dt);
  else if (stage == 1) k_charge_div_e<1><<<blocks, threads, 0, st>>>(G, dt);
  else if (stage == 2) k_charge_div_e<2><<<blocks, threads, 0, st>>>(G, dt);
  else k_charge_div_e<3><<<blocks, threads, 0, st>>>(G, dt);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a7. max over interior cells and active directions of (alpha sqrt(gamma^kk) + |beta^k|)/dx^k
// (Eq. 30; reading R14): warp shuffle -> block -> one atomicMax on the bit pattern
// (non-negative doubles order like unsigned integers).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_max_speed(const __grid_constant__ GridView G, unsigned long long* __restrict__ out, bool mhd_mode) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  double mx = 0.0;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < nint; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % nx);
    const long long r = t / nx;
    const int j = (int)(r % ny), k = (int)(r / ny);
    Met m;
    const long long c = cell_index(G, i, j, k);
    load_met_cell(G, c, m);
    const bool mhd = mhd_mode && G.P[RHO][c] > G.wave_rho_switch;   // A9: the cell's own ideal-GRMHD speeds (reading R16)
    double P[NPRIM];
#pragma unroll
    for (int v = 0; v < NPRIM; ++v) P[v] = (mhd && (v <= VZ || (v >= BX && v <= BZ))) ? G.P[v][c] : 0.0;
    mx = fmax(mx, cell_cfl_speed(m, G.Gamma, P, mhd, G.inv_dx[0], G.inv_dx[1], G.inv_dx[2], G.n[0] > 1, G.n[1] > 1, G.n[2] > 1));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  __shared__ double smx[8];
  if ((threadIdx.x & 31) == 0) smx[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) mx = fmax(mx, smx[w]);
    atomicMax(out, (unsigned long long)__double_as_longlong(mx));
  }
}

cudaError_t launch_max_speed(const GridView& G, unsigned long long* out, bool have_prims, int sm_count, cudaStream_t st) {
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  const int threads = 256;
  long long blocks = (nint + threads - 1) / threads;
  if (blocks > (long long)sm_count * 8) blocks = (long long)sm_count * 8;   // 8 resident 256-thread CTAs per SM
  k_max_speed<<<(unsigned)blocks, threads, 0, st>>>(G, out, G.wave_mode == WAVE_MHD_INSIDE && have_prims);
  return cudaGetLastError();
}

}  // namespace rg
