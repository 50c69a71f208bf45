// rgrmhd_c2p.cu -- a6: implicit Ohm's-law update of the electric field fused with the 1D
// conservative-to-primitive recovery (Eq. 42-50), one thread per cell, all
// iterations in registers; plus a0 (prim -> cons at set_prims).
//
// The result is DEFINED (reading R8) as the root (E, v, p) of
//   (1+s) E - s (v.E) v + s v x B = Estar^,  s = a_ii dt alpha sigma W            [Eq. 42, R7]
//   Z v_i = S^_i - (E x B)_i,  Z = tau^ + D^ + p - (E^2+B^2)/2                    [Eq. 44, G2]
//   rho = D^/W,  p = (Gamma-1)/Gamma (Z/W^2 - rho)                                [Eq. 45-49]
// found by eliminating E from the momentum relation for frozen scalars (s, kE = v.E) and driving the
// scalar residual g(Z) to zero with a bracketed secant; an outer Anderson(1) fixed point updates
// (W, kE).  The solver is written as ONE loop whose body holds exactly one residual evaluation, so
// lanes that are in different inner/outer phases still execute the expensive part convergently;
// the loop ends for a warp when every lane is done (warp vote).
#include "rgrmhd_common.cuh"

namespace rg {

struct C2POut {
  int evals;
  int failed;
};

// Work in the cell's coordinate basis with explicit index placement.
struct C2PState {
  // constants of the cell
  double Dh, tauh, B2, s0, gm1og;
  double EstarU[3], BU[3], BD[3];
  // frozen per outer pass
  double s, kE, r;
  double NparU[3], NperpU[3], BxNperpU[3];
  // last evaluation
  double vU[3], EU[3], W, rho, p;
};

// residual g(Z) for frozen (s, kE); false when v^2 >= 1 (treated as g = -infinity)
__device__ __forceinline__ bool c2p_residual(const Met& m, C2PState& w, double Z, double& g) {
  const double A = Z + w.r * w.B2, c = w.r * w.kE;
  const double iden = 1.0 / (A * A + c * c * w.B2), iZ = 1.0 / Z;
#pragma unroll
  for (int i = 0; i < 3; ++i) w.vU[i] = w.NparU[i] * iZ + (A * w.NperpU[i] + c * w.BxNperpU[i]) * iden;
  double vD[3];
  lower(m, w.vU, vD);
  const double v2 = dot3(w.vU, vD);
  if (!(v2 < 1.0)) return false;
  const double W2 = 1.0 / (1.0 - v2);
  w.W = sqrt(W2);
  double vxB[3];
  cross_raw(vD, w.BD, vxB);                               // (v x B)^i = [ijk] v_j B_k / sg
  const double isg = 1.0 / m.sg, i1s = 1.0 / (1.0 + w.s), skE = w.s * w.kE;
#pragma unroll
  for (int i = 0; i < 3; ++i) w.EU[i] = (w.EstarU[i] - w.s * (vxB[i] * isg) + skE * w.vU[i]) * i1s;
  double ED[3];
  lower(m, w.EU, ED);
  const double E2 = dot3(w.EU, ED);
  w.rho = w.Dh / w.W;
  w.p = w.gm1og * (Z * (1.0 - v2) - w.rho);
  g = Z - (w.tauh + w.Dh + w.p - 0.5 * (E2 + w.B2));
  return true;
}

// closed form of Eq. 42 at fixed v (reading R7)
__device__ __forceinline__ void implicit_E_closed(const Met& m, const double vU[3], double W, double s,
                                                  const double EstarU[3], const double BD[3], double EU[3]) {
  double vD[3], EstarD[3], vxB[3];
  lower(m, vU, vD); lower(m, EstarU, EstarD);
  cross_raw(vD, BD, vxB);
  const double kE = dot3(vU, EstarD) / (1.0 + s / (W * W));
#pragma unroll
  for (int i = 0; i < 3; ++i) EU[i] = (EstarU[i] - s * (vxB[i] / m.sg) + s * kE * vU[i]) / (1.0 + s);
}

// P holds the guess (rho, p, v) on entry and all 14 primitives on return.
__device__ C2POut c2p_solve(const Met& m, double Gamma, const double U[NCONS], double adt, double sigma,
                            double tol, int maxit, double P[NPRIM]) {
  C2PState w;
  const double isg = 1.0 / m.sg;
  w.gm1og = (Gamma - 1.0) / Gamma;
  w.Dh = U[CD] * isg; w.tauh = U[CTAU] * isg;
  const double ShD[3] = {U[CSX] * isg, U[CSY] * isg, U[CSZ] * isg};
  double ShU[3], EstarD[3], EsxB[3];
  raise(m, ShD, ShU);
#pragma unroll
  for (int i = 0; i < 3; ++i) { w.EstarU[i] = U[CEX + i] * isg; w.BU[i] = U[CBX + i] * isg; }
  lower(m, w.BU, w.BD); lower(m, w.EstarU, EstarD);
  w.B2 = dot3(w.BU, w.BD);
  cross_raw(EstarD, w.BD, EsxB);
#pragma unroll
  for (int i = 0; i < 3; ++i) EsxB[i] *= isg;              // (E* x B)^i
  w.s0 = adt * m.alpha * sigma;
  const double s0 = w.s0;
  const double escale = sqrt(dot3(w.EstarU, EstarD) + w.B2);
  C2POut res = {0, 1};
  // EM fields that do not depend on the solve
#pragma unroll
  for (int i = 0; i < 3; ++i) P[BX + i] = w.BU[i];
  P[PSI] = U[CPSI] * isg; P[PHI] = U[CPHI] * isg; P[QCH] = U[CQ] * isg;
  const double Zlo = w.Dh, Zhi = Gamma * (w.tauh + w.Dh - 0.5 * w.B2);
  // guess
  double vgU[3] = {P[VX], P[VY], P[VZ]}, vgD[3];
  lower(m, vgU, vgD);
  double v2g = dot3(vgU, vgD);
  if (!(v2g < 1.0)) { vgU[0] = vgU[1] = vgU[2] = 0.0; v2g = 0.0; }
  const double Wg = 1.0 / sqrt(1.0 - v2g);
  double W = Wg;
  double kE = dot3(vgU, EstarD) / (1.0 + s0 / W);
  if (!(w.Dh > 0.0) || !(Zhi > Zlo)) {   // no physical bracket: keep the guess, E from the guess v
    double EU[3];
    implicit_E_closed(m, vgU, W, s0 * W, w.EstarU, w.BD, EU);
    P[EX] = EU[0]; P[EY] = EU[1]; P[EZ] = EU[2];
    return res;
  }
  double Z = (P[RHO] + Gamma / (Gamma - 1.0) * P[PRS]) * W * W;
  bool converged = false, state_ok = false;
  const int max_outer = 50;
  double fW_prev = 0, fk_prev = 0, GW_prev = 0, Gk_prev = 0, slope = 1.0;
  // inner-loop state
  double a = Zlo, b = Zhi, x = Z, f = 0, xp = 0, fp = 0;
  bool ok = false, okp = false;
  int outer = 0;
  bool need_setup = true, done = false;
  // ONE loop, one residual evaluation per trip.
  while (true) {
    if (!done) {
      if (need_setup) {
        // ---- outer pass set-up: freeze (s, kE), decompose N along/across B ---------------------
        w.s = s0 * W; w.r = w.s / (1.0 + w.s); w.kE = kE;
        double NU[3], ND[3], NperpD[3];
        const double i1s = 1.0 / (1.0 + w.s);
#pragma unroll
        for (int i = 0; i < 3; ++i) NU[i] = ShU[i] - EsxB[i] * i1s;
        lower(m, NU, ND);
        const double NdotB = dot3(NU, w.BD);
        const double fpar = (w.B2 > 0.0) ? NdotB / w.B2 : 0.0;
#pragma unroll
        for (int i = 0; i < 3; ++i) { w.NparU[i] = fpar * w.BU[i]; w.NperpU[i] = NU[i] - w.NparU[i]; }
        lower(m, w.NperpU, NperpD);
        cross_raw(w.BD, NperpD, w.BxNperpU);
#pragma unroll
        for (int i = 0; i < 3; ++i) w.BxNperpU[i] *= isg;
        a = Zlo; b = Zhi;
        x = fmin(fmax(Z, a), b);
        okp = false;
        need_setup = false;
      }
      ok = c2p_residual(m, w, x, f);
      ++res.evals;
      // ---- inner: bracketed secant / bisection on Z; invariant g(a) < 0 < g(b) -----------------
      bool inner_conv = false, inner_stop = false;
      if (ok && f == 0.0) {
        inner_conv = true;
      } else {
        if (!ok || f < 0.0) a = x; else b = x;
        if (ok && okp && f != fp && x != xp) slope = (f - fp) / (x - xp);
        const double delta = ok ? f / slope : 0.0;          // predicted distance to the root
        if (ok && fabs(delta) <= tol * fabs(x)) inner_conv = true;
        else if (ok && (b - a) <= tol * fabs(x)) inner_conv = true;
        else if (res.evals >= maxit) inner_stop = true;
        else {
          double xn = ok ? x - delta : 0.5 * (a + b);
          if (!(xn > a && xn < b)) xn = 0.5 * (a + b);      // bisection safeguard
          xp = x; fp = f; okp = ok;
          x = xn;
        }
      }
      if (inner_conv || inner_stop) {
        Z = x; state_ok = ok;
        if (!inner_conv || !ok) {
          done = true;
        } else {
          // ---- outer: update (s, kE) from the new v ------------------------------------------------
          const double Wnew = w.W;
          const double kEnew = dot3(w.vU, EstarD) / (1.0 + s0 / Wnew);
          const bool same = fabs(Wnew - W) <= tol * Wnew && fabs(kEnew - kE) <= tol * escale;
          if (s0 == 0.0 || same) {
            converged = true; done = true;
          } else {
            // Anderson(1) acceleration of x -> G(x), x = (W, kE/escale)
            const double es = escale > 0.0 ? escale : 1.0;
            const double fW = Wnew - W, fk = (kEnew - kE) / es;
            double Wnext = Wnew, knext = kEnew;
            if (outer > 0) {
              const double dW = fW - fW_prev, dk = fk - fk_prev, den = dW * dW + dk * dk;
              if (den > 0.0) {
                const double theta = (fW * dW + fk * dk) / den;
                const double Wa = Wnew - theta * (Wnew - GW_prev), ka = kEnew - theta * (kEnew - Gk_prev);
                if (isfinite(Wa) && isfinite(ka) && Wa >= 1.0 && fabs(theta) < 10.0) { Wnext = Wa; knext = ka; }
              }
            }
            fW_prev = fW; fk_prev = fk; GW_prev = Wnew; Gk_prev = kEnew;
            W = Wnext; kE = knext;
            ++outer;
            if (outer >= max_outer || res.evals >= maxit) done = true;
            else need_setup = true;
          }
        }
      }
    }
    if (__all_sync(__activemask(), done)) break;            // warp-vote exit
  }
  res.failed = converged ? 0 : 1;
  if (state_ok) {
    P[RHO] = w.rho; P[PRS] = w.p;
#pragma unroll
    for (int i = 0; i < 3; ++i) { P[VX + i] = w.vU[i]; P[EX + i] = w.EU[i]; }
  } else {
    double EU[3];
    implicit_E_closed(m, vgU, Wg, s0 * Wg, w.EstarU, w.BD, EU);
    P[EX] = EU[0]; P[EY] = EU[1]; P[EZ] = EU[2];
  }
  return res;
}

// a6 over the grid.  Ust = stage vector (its calE entries are X*), guess = current G.P.  Writes G.P,
// the conduction current G.jc (reading R3) and, if Xout != null, the stage calE = sqrt(gamma) E.
// Floor rule: reading R9; write_back_floor only in the final recovery of a step.
struct C2PArgs {
  double* Ust[NCONS];
  double* Xout[3];
  double adt;
  int write_back_floor;
  int has_xout;
};

__global__ void __launch_bounds__(128)
k_c2p(const __grid_constant__ GridView G, const __grid_constant__ C2PArgs A, StatsDev* __restrict__ stats) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int evals = 0, failed = 0, floored = 0;
  if (t < nint) {
    const int i = (int)(t % nx);
    const long long r = t / nx;
    const int j = (int)(r % ny), k = (int)(r / ny);
    const long long c = cell_index(G, i, j, k);
    Met m;
    load_met_cell(G, c, m);
    double U[NCONS], P[NPRIM];
#pragma unroll
    for (int v = 0; v < NCONS; ++v) U[v] = A.Ust[v][c];
#pragma unroll
    for (int v = 0; v < 5; ++v) P[v] = G.P[v][c];
    const double Dh = U[CD] / m.sg;
    const double sigma = (A.adt > 0.0) ? sigma_of(G, Dh, c) : 0.0;
    C2POut r2 = c2p_solve(m, G.Gamma, U, A.adt, sigma, G.tol, G.maxit, P);
    evals = r2.evals; failed = r2.failed;
    if (G.rho_floor > 0.0 && (r2.failed || !(P[RHO] > G.rho_floor * (1.0 + 1e-3)))) {
      // reading R9: atmosphere reset
      floored = 1;
      P[RHO] = G.rho_floor; P[VX] = P[VY] = P[VZ] = 0.0;
      P[PRS] = G.p_atmo;
      const double s = A.adt * m.alpha * sigma;
#pragma unroll
      for (int q = 0; q < 3; ++q) P[EX + q] = (U[CEX + q] / m.sg) / (1.0 + s);
      if (A.write_back_floor) {
        double Unew[NCONS];
        prim2cons(m, G.Gamma, P, Unew);
        A.Ust[CD][c] = Unew[CD]; A.Ust[CTAU][c] = Unew[CTAU];
#pragma unroll
        for (int q = 0; q < 3; ++q) A.Ust[CSX + q][c] = Unew[CSX + q];
      }
    }
#pragma unroll
    for (int v = 0; v < NPRIM; ++v) G.P[v][c] = P[v];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      if (A.has_xout) A.Xout[q][c] = m.sg * P[EX + q];
      G.jc[q][c] = (A.adt > 0.0) ? (U[CEX + q] / m.sg - P[EX + q]) / (A.adt * m.alpha) : 0.0;
    }
  }
  // stats: warp reduce, one atomic per warp
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

// ---- launchers -----------------------------------------------------------------------------------
cudaError_t launch_c2p(const GridView& G, double* const Ust[NCONS], double* const Xout[3], double adt,
                       bool write_back_floor, StatsDev* stats, cudaStream_t st) {
  C2PArgs A;
  for (int v = 0; v < NCONS; ++v) A.Ust[v] = Ust[v];
  for (int q = 0; q < 3; ++q) A.Xout[q] = Xout ? Xout[q] : nullptr;
  A.adt = adt; A.write_back_floor = write_back_floor ? 1 : 0; A.has_xout = Xout ? 1 : 0;
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  const int threads = 128;
  const unsigned blocks = (unsigned)((nint + threads - 1) / threads);
  k_c2p<<<blocks, threads, 0, st>>>(G, A, stats);
  return cudaGetLastError();
}

cudaError_t launch_prim2cons(const GridView& G, cudaStream_t st) {
  const int threads = 256;
  const unsigned blocks = (unsigned)((G.ntot + threads - 1) / threads);
  k_prim2cons<<<blocks, threads, 0, st>>>(G);
  return cudaGetLastError();
}

}  // namespace rg
