// rgrmhd_imex_gen.cu -- the point-wise kernel of the GENERAL IMEX-RK driver (PAPER.md:44:
// SSP2(3,3,2), SSP3(3,3,2), SSP3(4,3,3) next to SSP2(2,2,2)), for any s-stage double Butcher tableau of the form
// Eq. 32-34:
//   U^(i)   = U^n + dt sum_{j<i} at_ij F[U^(j)] + dt sum_{j<=i} a_ij R[U^(j)],
//   U^{n+1} = U^n + dt sum_i wt_i F[U^(i)] + dt sum_i w_i R[U^(i)],
// F = -div(flux) + S the explicit operator, R the stiff Ohm term acting on X = calE only, evaluated
// as the difference quotient R^(i) = (X^(i) - X*^(i))/(a_ii dt) (reading R11), final recovery at fixed calE (R12).
//
// Low-storage organisation: one ACCUMULATOR per pending stage vector and one for U^{n+1} (which is G.Un, in place).
// The kernel of stage i
//   1. reads the flux increment D = dt (-div F^(i-1)) the flux kernel has just written (G.dU) and adds
//      at_{k,i-1} D to the accumulator of every stage k >= i and wt_{i-1} D to the final one,
//   2. takes its own, now complete, accumulator as the stage vector (its calE entries are X*^(i)), solves the
//      implicit stage with a = a_ii dt (c2p_solve), stores P^(i) and the conduction current,
//   3. evaluates the explicit sources S^(i) from P^(i) and adds dt at_{k,i} S^(i) + (a_{k,i}/a_ii) (X^(i) - X*^(i))
//      to the accumulators of the later stages k > i (and wt_i, w_i to the final one);
// stage 0 initialises the accumulators from U^n instead of updating them; the final kernel adds wt_{s-1} D, stores
// U^{n+1}, recovers it with a = 0 and applies the atmosphere rule with write-back (reading R9).
// The SSP2(2,2,2) production path (rgrmhd_c2p.cu) is this scheme with the algebra specialised by hand; the two are
// compared in the tests.
#include "rgrmhd_c2p_solve.cuh"

namespace rg {

struct AccTab { double* f[NCONS]; };

struct StageGen {
  int stage, nstages;      // 0-based stage index; stage == nstages marks the final kernel
  int use_dprev;           // G.dU holds dt (-div F) of the previous stage and somebody needs it
  int init;                // first kernel of the step: accumulators are initialised from U^n
  double aii;              // a_ii of this stage
  // weights for the targets: slot k < nstages = accumulator of stage k, slot 4 = U^{n+1}
  double w_dprev[5];       // at_{k,stage-1} (wt_{stage-1} for slot 4): weight of D
  double w_src[5];         // at_{k,stage}   (wt_stage): weight of dt S^(stage)
  double w_stiff[5];       // a_{k,stage}/a_ii (w_stage/a_ii): weight of X^(stage) - X*^(stage)
  AccTab acc[5];           // field tables of the targets (slot 4 = G.Un)
};

template <bool FINAL>
__global__ void __launch_bounds__(32, 12)
k_stage_gen(const __grid_constant__ GridView G, const __grid_constant__ StageGen W, double dt, StatsDev* __restrict__ stats) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  int evals = 0, failed = 0, floored = 0;
  const bool in_range = i < G.n[0];
  if (in_range) {
    const long long c = cell_index(G, i, j, k);
    const int me = FINAL ? 4 : W.stage;
    double D[NCONS], U[NCONS];
#pragma unroll
    for (int v = 0; v < NCONS; ++v) D[v] = W.use_dprev ? G.dU[v][c] : 0.0;
    // the stage vector: own accumulator (stage 0: U^n) + the share of the flux increment that was still missing
#pragma unroll
    for (int v = 0; v < NCONS; ++v) U[v] = (W.init ? G.Un[v][c] : W.acc[me].f[v][c]) + W.w_dprev[me] * D[v];
    double g6[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) g6[q] = __ldg(G.met[MGXX + q] + c);
    const double alpha = __ldg(G.met[MALP] + c);
    Triad t;
    triad_make(g6, t);
    const double sg = t.l11 * t.l22 * t.l33, isg = rcp_fast(sg);
    double P[NPRIM];
#pragma unroll
    for (int v = 0; v < 5; ++v) P[v] = G.P[v][c];
    const double adt = FINAL ? 0.0 : W.aii * dt;
    const double sigma = FINAL ? 0.0 : sigma_of(G, U[CD] * isg, c);
    C2POut r = c2p_solve(t, isg, alpha, G.Gamma, G.gog1, G.gm1og, U, adt, sigma, G.tol, G.maxit, P);
    evals = r.evals; failed = r.failed;
    if (G.rho_floor > 0.0 && (r.failed || !(P[RHO] > G.rho_floor * (1.0 + 1e-3)))) {   // reading R9
      floored = 1;
      P[RHO] = G.rho_floor; P[VX] = P[VY] = P[VZ] = 0.0;
      P[PRS] = G.p_atmo;
      const double s = adt * alpha * sigma;
#pragma unroll
      for (int q = 0; q < 3; ++q) P[EX + q] = (U[CEX + q] * isg) / (1.0 + s);
      if (FINAL) {
        Met m;
        load_met_cell(G, c, m);
        double Unew[NCONS];
        prim2cons(m, G.Gamma, P, Unew);
        U[CD] = Unew[CD]; U[CTAU] = Unew[CTAU];
#pragma unroll
        for (int q = 0; q < 3; ++q) U[CSX + q] = Unew[CSX + q];
      }
    }
#pragma unroll
    for (int v = 0; v < NPRIM; ++v) G.P[v][c] = P[v];
    if (FINAL) {
#pragma unroll
      for (int v = 0; v < NCONS; ++v) G.Un[v][c] = U[v];
#pragma unroll
      for (int q = 0; q < 3; ++q) G.jc[q][c] = 0.0;
    } else {
      double dX[3];
      const double iada = rcp_fast(adt * alpha);
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        dX[q] = sg * P[EX + q] - U[CEX + q];                                 // X^(i) - X*^(i) = a_ii dt R^(i)
        G.jc[q][c] = (U[CEX + q] * isg - P[EX + q]) * iada;                  // reading R3
      }
      // a4: explicit sources of this stage
      double S[NCONS];
#pragma unroll
      for (int v = 0; v < NCONS; ++v) S[v] = 0.0;
      Met m;
      load_met_cell(G, c, m);
      const unsigned long long nz = __ldg(G.src_mask);
      double src[NSRC], Kq[6];
#pragma unroll
      for (int q = 0; q < NSRC; ++q) src[q] = ((nz >> q) & 1ull) ? __ldg(G.src[q] + c) : 0.0;
#pragma unroll
      for (int q = 0; q < 6; ++q) Kq[q] = ((nz >> (NSRC + q)) & 1ull) ? __ldg(G.met[MKXX + q] + c) : 0.0;
      add_sources(G, m, src, Kq, P, S);
      // a5: feed the accumulators of the later stages and of U^{n+1}
      double Un0[NCONS];
      if (W.init) {
#pragma unroll
        for (int v = 0; v < NCONS; ++v) Un0[v] = U[v];                        // stage 0: U = U^n
      }
#pragma unroll 1
      for (int tgt = W.stage + 1; tgt <= W.nstages; ++tgt) {
        const int slot = (tgt == W.nstages) ? 4 : tgt;
        const double wd = W.w_dprev[slot], ws = W.w_src[slot] * dt, wx = W.w_stiff[slot];
#pragma unroll
        for (int v = 0; v < NCONS; ++v) {
          double a = W.init ? Un0[v] : W.acc[slot].f[v][c];
          a += wd * D[v] + ws * S[v];
          if (v >= CEX && v <= CEZ) a += wx * dX[v - CEX];
          W.acc[slot].f[v][c] = a;
        }
      }
    }
  }
  int fl = failed, fo = floored, mx = evals;
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

cudaError_t launch_stage_gen(const GridView& G, const StageGen& W, double dt, StatsDev* stats, cudaStream_t st) {
  const dim3 block(32, 1, 1), grid((G.n[0] + 31) / 32, G.n[1], G.n[2]);
  if (grid.y > 65535u || grid.z > 65535u) return cudaErrorInvalidConfiguration;
  if (W.stage == W.nstages) k_stage_gen<true><<<grid, block, 0, st>>>(G, W, dt, stats);
  else k_stage_gen<false><<<grid, block, 0, st>>>(G, W, dt, stats);
  return cudaGetLastError();
}

// charge mode DIV_E with a general tableau: the two source terms that carry the stage's charge, -alpha calQ v^i in
// S(calE^i) and +alpha calQ in S(Psi), go to the later targets with the weights of S^(stage)
__global__ void __launch_bounds__(128)
k_charge_sources_gen(const __grid_constant__ GridView G, const __grid_constant__ StageGen W, double dt) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nint) return;
  const int i = (int)(t % nx);
  const long long r = t / nx;
  const long long c = cell_index(G, i, (int)(r % ny), (int)(r / ny));
  Met m;
  load_met_cell(G, c, m);
  const double aq = m.alpha * m.sg * G.P[QCH][c];          // alpha calQ, q = div E written by k_charge_div_e<3>
  for (int tgt = W.stage + 1; tgt <= W.nstages; ++tgt) {
    const int slot = (tgt == W.nstages) ? 4 : tgt;
    const double w = W.w_src[slot] * dt;
    if (w == 0.0) continue;
#pragma unroll
    for (int a = 0; a < 3; ++a) W.acc[slot].f[CEX + a][c] -= w * aq * G.P[VX + a][c];
    W.acc[slot].f[CPSI][c] += w * aq;
  }
}

cudaError_t launch_charge_sources_gen(const GridView& G, const StageGen& W, double dt, cudaStream_t st) {
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  k_charge_sources_gen<<<(unsigned)((nint + 127) / 128), 128, 0, st>>>(G, W, dt);
  return cudaGetLastError();
}

}  // namespace rg
