// rgrmhd_c2p.cu -- a6: implicit Ohm's-law update of the electric field fused with the 1D
// conservative-to-primitive recovery (Eq. 42-50), one thread per cell, all
// iterations in registers; followed, in the same thread, by the point-wise half of the right-hand side
// of that stage: explicit sources (a4) and the point-wise part of the stage combine (a5), which need
// nothing but the primitives just recovered.  Also here: a0 (prim -> cons at set_prims).
// The per-cell solver is c2p_solve (rgrmhd_c2p_solve.cuh).
#include "rgrmhd_c2p_solve.cuh"

namespace rg {

// a6 (+ a4, a5 point-wise) over the grid.
//   STAGE 1: stage vector U^n (X*1 = X^n),  a = gamma dt; writes P, jc, X1 and the bracket of U*2 into G.Us
//   STAGE 2: stage vector U*2 (G.Us),       a = gamma dt; writes P, jc and the bracket of U^{n+1} into G.Un
//   STAGE 3: recovery of U^{n+1} (G.Un) at fixed calE (a = 0, reading R12); writes P; floor write-back (R9)
//   STAGE 4: STAGE 3 of the previous step followed by STAGE 1 of this one in the same thread (rgrmhd_step defers the
//            final recovery until the state is asked for or the next step starts): P^{n+1} and U^{n+1} go from the
//            first solve to the second in registers, same arithmetic as the two launches
// The guess is the current G.P.  jc = undensitised conduction current of the stage (reading R3).
constexpr int C2P_TX = 32, C2P_TY = 1;
// staging slots of the point-wise right-hand side (doubles per thread)
enum { PF_SRC = 0, PF_K = NSRC, PF_UN = NSRC + 6, PF_X1 = NSRC + 6 + NCONS, PF_US = NSRC + 6 + NCONS + 3,
       PF_COUNT1 = PF_X1, PF_COUNT2 = PF_US + NCONS };
__device__ __forceinline__ void cp_async8(double* dst_smem, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src)
               : "memory");
}
#ifndef C2P_MINB
#define C2P_MINB 12
#endif

template <int STAGE>
__global__ void __launch_bounds__(C2P_TX * C2P_TY, C2P_MINB)
k_c2p(const __grid_constant__ GridView G, double dt, StatsDev* __restrict__ stats) {
  const int i = blockIdx.x * C2P_TX + (threadIdx.x & (C2P_TX - 1));
  const int j = blockIdx.y * C2P_TY + (threadIdx.x / C2P_TX);
  const int k = blockIdx.z;
  const double gam = 1.0 - 0.70710678118654752440;   // 1 - 1/sqrt(2) (Eq. 35-37)
  const double adt = (STAGE == 3) ? 0.0 : gam * dt;
  double* const* Ust = (STAGE == 2) ? G.Us : G.Un;
  int evals = 0, evmax = 0, failed = 0, floored = 0;
  double cfl = 0.0;
  const bool in_range = i < G.n[0] && j < G.n[1];
  if (in_range) {
    const long long c = cell_index(G, i, j, k);
    double g6[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) g6[q] = __ldg(G.met[MGXX + q] + c);
    const double alpha = __ldg(G.met[MALP] + c);
    // loads that depend on nothing but the cell index go out with the first batch: left inside sigma_of / behind the
    // first solve they each cost a DRAM round trip of their own (measured: -2 % of this kernel on config 4)
    const double sig_arr = (STAGE != 3 && G.sigma_model == SIGMA_ARRAY) ? __ldg(G.sigma + c) : 0.0;
    const unsigned long long nz = (STAGE != 3) ? __ldg(G.src_mask) : 0ull;
    Triad t;
    triad_make(g6, t);
    const double sg = t.l11 * t.l22 * t.l33;
    double U[NCONS], P[NPRIM];
#pragma unroll
    for (int v = 0; v < NCONS; ++v) U[v] = Ust[v][c];
    if (STAGE != 1) {   // stage vector = bracket written by the previous recovery + increment of the flux kernel
      double inc[NCONS];
#pragma unroll
      for (int v = 0; v < NCONS; ++v) inc[v] = G.dU[v][c];
#pragma unroll
      for (int v = 0; v < NCONS; ++v) U[v] += inc[v];
      if (STAGE >= 3) {   // U^{n+1} complete: the next step and get_cons read it from G.Un
#pragma unroll
        for (int v = 0; v < NCONS; ++v) Ust[v][c] = U[v];
      }
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) P[v] = G.P[v][c];
    const double isg = rcp_fast(sg);
    if (STAGE == 4) {
      // deferred final recovery of the previous step (a = 0): its primitives are the guess of the stage-1 solve
      C2POut r0 = c2p_solve(t, isg, alpha, G.Gamma, G.gog1, G.gm1og, U, 0.0, 0.0, G.tol, G.maxit, P);
      evals = evmax = r0.evals; failed = r0.failed;
      if (G.rho_floor > 0.0 && (r0.failed || !(P[RHO] > G.rho_floor * (1.0 + 1e-3)))) {
        // reading R9: atmosphere reset with write-back, as in STAGE 3
        floored = 1;
        P[RHO] = G.rho_floor; P[VX] = P[VY] = P[VZ] = 0.0;
        P[PRS] = G.p_atmo;
#pragma unroll
        for (int q = 0; q < 3; ++q) P[EX + q] = (U[CEX + q] * isg) / (1.0 + 0.0);
        Met m;
        load_met_cell(G, c, m);
        double Unew[NCONS];
        prim2cons(m, G.Gamma, P, Unew);
        U[CD] = Unew[CD]; U[CTAU] = Unew[CTAU];
        Ust[CD][c] = U[CD]; Ust[CTAU][c] = U[CTAU];
#pragma unroll
        for (int q = 0; q < 3; ++q) { U[CSX + q] = Unew[CSX + q]; Ust[CSX + q][c] = U[CSX + q]; }
      }
    }
    const double sigma = (STAGE == 3) ? 0.0 : (G.sigma_model == SIGMA_ARRAY) ? sig_arr : sigma_of(G, U[CD] * isg, c);
    // The point-wise right-hand side after the solve reads ~57 more fields of this cell.  Start those loads
    // now as asynchronous copies into a thread-private shared-memory column: no registers are held and
    // the solve below hides their DRAM latency.
    extern __shared__ double pf_smem[];
    double* const pf = pf_smem + threadIdx.x;              // pf[q * NTH]: conflict-free, private to this thread
    constexpr int NTH = C2P_TX * C2P_TY;
    if (STAGE != 3) {
      // fields that are identically zero on this grid (zero shift, K_ij = 0, diagonal metric, ...) are not read
#pragma unroll
      for (int q = 0; q < NSRC; ++q) {
        if ((nz >> q) & 1ull) cp_async8(pf + (PF_SRC + q) * NTH, G.src[q] + c);
        else pf[(PF_SRC + q) * NTH] = 0.0;
      }
#pragma unroll
      for (int q = 0; q < 6; ++q) {
        if ((nz >> (NSRC + q)) & 1ull) cp_async8(pf + (PF_K + q) * NTH, G.met[MKXX + q] + c);
        else pf[(PF_K + q) * NTH] = 0.0;
      }
#pragma unroll
      for (int v = 0; v < NCONS; ++v) {
        if (STAGE == 4) pf[(PF_UN + v) * NTH] = U[v];            // U^n of this step: in registers already
        else cp_async8(pf + (PF_UN + v) * NTH, G.Un[v] + c);
      }
      if (STAGE == 2) {
#pragma unroll
        for (int q = 0; q < 3; ++q) cp_async8(pf + (PF_X1 + q) * NTH, G.X1[q] + c);
#pragma unroll
        for (int v = 0; v < NCONS; ++v) pf[(PF_US + v) * NTH] = U[v];   // U*2 = bracket + increment (needed again below)
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    }
    C2POut r2 = c2p_solve(t, isg, alpha, G.Gamma, G.gog1, G.gm1og, U, adt, sigma, G.tol, G.maxit, P);
    evals += r2.evals; failed += r2.failed;
    evmax = max(evmax, r2.evals);
    if (G.rho_floor > 0.0 && (r2.failed || !(P[RHO] > G.rho_floor * (1.0 + 1e-3)))) {
      // reading R9: atmosphere reset
      floored += 1;
      P[RHO] = G.rho_floor; P[VX] = P[VY] = P[VZ] = 0.0;
      P[PRS] = G.p_atmo;
      const double s = adt * alpha * sigma;
#pragma unroll
      for (int q = 0; q < 3; ++q) P[EX + q] = (U[CEX + q] * isg) / (1.0 + s);
      if (STAGE == 3) {
        Met m;
        load_met_cell(G, c, m);
        double Unew[NCONS];
        prim2cons(m, G.Gamma, P, Unew);
        Ust[CD][c] = Unew[CD]; Ust[CTAU][c] = Unew[CTAU];
#pragma unroll
        for (int q = 0; q < 3; ++q) Ust[CSX + q][c] = Unew[CSX + q];
      }
    }
#pragma unroll
    for (int v = 0; v < NPRIM; ++v) G.P[v][c] = P[v];
    if (STAGE == 3 && G.wave_mode == WAVE_MHD_INSIDE) {
      // a7 fused into the final recovery (f1): with state-dependent wave speeds the CFL reduction is a per-step one,
      // and the new primitives are in registers here
      Met m;
      load_met_cell(G, c, m);
      const bool mhd = P[RHO] > G.wave_rho_switch;
      double Pq[NPRIM];
#pragma unroll
      for (int v = 0; v < NPRIM; ++v) Pq[v] = (mhd && (v <= VZ || (v >= BX && v <= BZ))) ? P[v] : 0.0;
      cfl = cell_cfl_speed(m, G.Gamma, Pq, mhd, G.inv_dx[0], G.inv_dx[1], G.inv_dx[2], G.n[0] > 1, G.n[1] > 1, G.n[2] > 1);
    }
    double sgE[3];
    const double iada = (STAGE == 3) ? 0.0 : rcp_fast(adt * alpha);
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      sgE[q] = sg * P[EX + q];
      if (STAGE == 1 || STAGE == 4) G.X1[q][c] = sgE[q];
      G.jc[q][c] = (STAGE == 3) ? 0.0 : (U[CEX + q] * isg - P[EX + q]) * iada;
    }
    if (STAGE != 3) {
      // ---- a4 + a5 (point-wise part)
      double S[NCONS];
#pragma unroll
      for (int v = 0; v < NCONS; ++v) S[v] = 0.0;
      Met m;
      load_met_cell(G, c, m);
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      double src[NSRC], Kq[6], un[NCONS], us[NCONS], x1[3] = {0.0, 0.0, 0.0};
#pragma unroll
      for (int q = 0; q < NSRC; ++q) src[q] = pf[(PF_SRC + q) * NTH];
#pragma unroll
      for (int q = 0; q < 6; ++q) Kq[q] = pf[(PF_K + q) * NTH];
      add_sources(G, m, src, Kq, P, S);
#pragma unroll
      for (int v = 0; v < NCONS; ++v) un[v] = pf[(PF_UN + v) * NTH];
      if (STAGE == 2) {
#pragma unroll
        for (int q = 0; q < 3; ++q) x1[q] = pf[(PF_X1 + q) * NTH];
#pragma unroll
        for (int v = 0; v < NCONS; ++v) us[v] = pf[(PF_US + v) * NTH];
      }
      stage_precombine<(STAGE == 4) ? 1 : STAGE>(G, c, dt, S, sgE, un, us, x1);
    }
  }
  if (STAGE == 3 && G.wave_mode == WAVE_MHD_INSIDE) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cfl = fmax(cfl, __shfl_xor_sync(0xffffffffu, cfl, o));
    if ((threadIdx.x & 31) == 0) atomicMax(G.maxspeed_word, (unsigned long long)__double_as_longlong(cfl));
  }
  // stats: warp reduce, one atomic per warp
  int fl = failed, fo = floored, mx = evmax;
  long long ev = evals;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ev += __shfl_xor_sync(0xffffffffu, ev, o);
    fl += __shfl_xor_sync(0xffffffffu, fl, o);
    fo += __shfl_xor_sync(0xffffffffu, fo, o);
    mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&stats->evals, (unsigned long long)ev);
    if (fl) atomicAdd(&stats->failures, (unsigned long long)fl);
    if (fo) atomicAdd(&stats->floors, (unsigned long long)fo);
    atomicMax(&stats->max_evals, mx);
  }
}

// a0 over every padded cell (ghosts included, like set_prims of the C-ABI states)
__global__ void __launch_bounds__(256)
k_prim2cons(const __grid_constant__ GridView G) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= G.ntot) return;
  Met m;
  load_met_cell(G, c, m);
  double P[NPRIM], U[NCONS];
#pragma unroll
  for (int v = 0; v < NPRIM; ++v) P[v] = G.P[v][c];
  prim2cons(m, G.Gamma, P, U);
#pragma unroll
  for (int v = 0; v < NCONS; ++v) G.Un[v][c] = U[v];
}

// Static source coefficients of every interior cell (once per set_metric), in two passes: STORE = false only records
// which of the NSRC coefficient fields (and which K_ij) are not identically zero on this grid (bit mask); the host then
// allocates exactly those fields, and STORE = true fills them (G.src[q] is null for an all-zero field: never read,
// never written -- zero shift, K_ij = 0 and a diagonal metric leave 15 of 40 fields in BASELINE configs 4 and 5).
template <bool STORE>
__global__ void __launch_bounds__(128)
k_metric_coeffs(const __grid_constant__ GridView G, unsigned long long* __restrict__ mask) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long nz = 0;
  if (t < nint) {
    const int i = (int)(t % nx);
    const long long r = t / nx;
    const long long c = cell_index(G, i, (int)(r % ny), (int)(r / ny));
    double out[NSRC];
    metric_coeffs_cell(G, c, out);
    if (STORE) {
#pragma unroll
      for (int q = 0; q < NSRC; ++q)
        if (G.src[q]) G.src[q][c] = out[q];
    } else {
#pragma unroll
      for (int q = 0; q < NSRC; ++q)
        if (out[q] != 0.0) nz |= 1ull << q;
#pragma unroll
      for (int q = 0; q < 6; ++q)
        if (__ldg(G.met[MKXX + q] + c) != 0.0) nz |= 1ull << (NSRC + q);
    }
  }
  if (!STORE) {   // which fields are not identically zero: warp OR, one atomic per warp
    unsigned lo = (unsigned)nz, hi = (unsigned)(nz >> 32);
    lo = __reduce_or_sync(0xffffffffu, lo);
    hi = __reduce_or_sync(0xffffffffu, hi);
    if ((threadIdx.x & 31) == 0 && (lo | hi)) atomicOr(mask, ((unsigned long long)hi << 32) | lo);
  }
}

cudaError_t launch_metric_coeffs(const GridView& G, bool store, cudaStream_t st) {
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  unsigned long long* mask = const_cast<unsigned long long*>(G.src_mask);
  const unsigned blocks = (unsigned)((nint + 127) / 128);
  if (store) {
    k_metric_coeffs<true><<<blocks, 128, 0, st>>>(G, mask);
  } else {
    cudaError_t e = cudaMemsetAsync(mask, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    k_metric_coeffs<false><<<blocks, 128, 0, st>>>(G, mask);
  }
  return cudaGetLastError();
}

// ---- launchers -----------------------------------------------------------------------------------
cudaError_t launch_c2p(const GridView& G, int stage, double dt, StatsDev* stats, cudaStream_t st) {
  const dim3 block(C2P_TX * C2P_TY, 1, 1);
  const dim3 grid((G.n[0] + C2P_TX - 1) / C2P_TX, (G.n[1] + C2P_TY - 1) / C2P_TY, G.n[2]);
  if (grid.y > 65535u || grid.z > 65535u) return cudaErrorInvalidConfiguration;
  size_t smem = (size_t)PF_COUNT1 * C2P_TX * C2P_TY * sizeof(double);
  cudaError_t e;
  if (stage == 1) {
    if ((e = cudaFuncSetAttribute(k_c2p<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    k_c2p<1><<<grid, block, smem, st>>>(G, dt, stats);
  } else if (stage == 2) {
    smem = (size_t)PF_COUNT2 * C2P_TX * C2P_TY * sizeof(double);
    if ((e = cudaFuncSetAttribute(k_c2p<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    k_c2p<2><<<grid, block, smem, st>>>(G, dt, stats);
  } else if (stage == 4) {
    if ((e = cudaFuncSetAttribute(k_c2p<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    k_c2p<4><<<grid, block, smem, st>>>(G, dt, stats);
  } else {
    k_c2p<3><<<grid, block, 0, st>>>(G, dt, stats);
  }
  return cudaGetLastError();
}

cudaError_t launch_prim2cons(const GridView& G, cudaStream_t st) {
  const int threads = 256;
  const unsigned blocks = (unsigned)((G.ntot + threads - 1) / threads);
  k_prim2cons<<<blocks, threads, 0, st>>>(G);
  return cudaGetLastError();
}

}  // namespace rg
