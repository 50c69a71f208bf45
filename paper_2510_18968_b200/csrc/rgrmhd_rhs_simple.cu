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
// a7. max over interior cells and active directions of (alpha sqrt(gamma^kk) + |beta^k|)/dx^k
// (Eq. 30; reading R14): warp shuffle -> block -> one atomicMax on the bit pattern
// (non-negative doubles order like unsigned integers).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_max_speed(const __grid_constant__ GridView G, unsigned long long* __restrict__ out) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  double mx = 0.0;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < nint; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % nx);
    const long long r = t / nx;
    const int j = (int)(r % ny), k = (int)(r / ny);
    Met m;
    load_met_cell(G, cell_index(G, i, j, k), m);
#pragma unroll
    for (int d = 0; d < 3; ++d)
      if (G.n[d] > 1) mx = fmax(mx, (m.alpha * sqrt(m.gi[sym(d, d)]) + fabs(m.b[d])) * G.inv_dx[d]);
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

cudaError_t launch_max_speed(const GridView& G, unsigned long long* out, int sm_count, cudaStream_t st) {
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  const int threads = 256;
  long long blocks = (nint + threads - 1) / threads;
  if (blocks > (long long)sm_count * 8) blocks = (long long)sm_count * 8;   // 8 resident 256-thread CTAs per SM
  k_max_speed<<<(unsigned)blocks, threads, 0, st>>>(G, out);
  return cudaGetLastError();
}

}  // namespace rg
