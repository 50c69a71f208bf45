// rgrmhd_c2p.cu -- a6: implicit Ohm's-law update of the electric field fused with the 1D
// conservative-to-primitive recovery (Eq. 42-50), one thread per cell, all
// iterations in registers; followed, in the same thread, by the point-wise half of the right-hand side
// of that stage: explicit sources (a4) and the point-wise part of the stage combine (a5), which need
// nothing but the primitives just recovered.  Also here: a0 (prim -> cons at set_prims).
//
// The result is DEFINED (reading R8) as the root (E, v, p) of
//   (1+s) E - s (v.E) v + s v x B = Estar^,  s = a_ii dt alpha sigma W            [Eq. 42, R7]
//   Z v_i = S^_i - (E x B)_i,  Z = tau^ + D^ + p - (E^2+B^2)/2                    [Eq. 44, G2]
//   rho = D^/W,  p = (Gamma-1)/Gamma (Z/W^2 - rho)                                [Eq. 45-49]
// found by eliminating E from the momentum relation for frozen scalars (s, kE = v.E) and driving the
// scalar residual g(Z) to zero with a bracketed secant; an outer Anderson(1) fixed point updates
// (W, kE).  The system is tensorial, so it is solved in an orthonormal triad of the cell's gamma_ij
// (Cholesky factor, gamma = L L^T): every dot and cross product in the loop is Euclidean and the
// metric is touched only before and after.  The solver is ONE loop whose body holds exactly one
// residual evaluation, so lanes in different inner/outer phases still execute the expensive part
// convergently; the loop ends for a warp when every lane is done (warp vote).
#include "rgrmhd_sources.cuh"

namespace rg {

struct C2POut {
  int evals;
  int failed;
};

// Orthonormal triad of gamma_ij: lower Cholesky factor L (gamma = L L^T) and the reciprocals of its
// diagonal.  a^ = L^T a for contravariant, a^ = L^-1 a for covariant components; a.b and a x b are then
// Euclidean (det L > 0: the triad is right handed, so [ijk]/sqrt(gamma) -> [abc]).
struct Triad {
  double l11, l21, l31, l22, l32, l33, i11, i22, i33;
};
__device__ __forceinline__ void triad_make(const double g[6], Triad& t) {
  sqrt_rsqrt_fast(g[0], t.l11, t.i11);
  t.l21 = g[1] * t.i11; t.l31 = g[2] * t.i11;
  sqrt_rsqrt_fast(g[3] - t.l21 * t.l21, t.l22, t.i22);
  t.l32 = (g[4] - t.l31 * t.l21) * t.i22;
  sqrt_rsqrt_fast(g[5] - t.l31 * t.l31 - t.l32 * t.l32, t.l33, t.i33);
}
__device__ __forceinline__ void triad_from_contra(const Triad& t, double a0, double a1, double a2, double h[3]) {
  h[0] = t.l11 * a0 + t.l21 * a1 + t.l31 * a2;
  h[1] = t.l22 * a1 + t.l32 * a2;
  h[2] = t.l33 * a2;
}
__device__ __forceinline__ void triad_from_cov(const Triad& t, double a0, double a1, double a2, double h[3]) {
  h[0] = a0 * t.i11;
  h[1] = (a1 - t.l21 * h[0]) * t.i22;
  h[2] = (a2 - t.l31 * h[0] - t.l32 * h[1]) * t.i33;
}
__device__ __forceinline__ void triad_to_contra(const Triad& t, const double h[3], double a[3]) {
  a[2] = h[2] * t.i33;
  a[1] = (h[1] - t.l32 * a[2]) * t.i22;
  a[0] = (h[0] - t.l21 * a[1] - t.l31 * a[2]) * t.i11;
}
__device__ __forceinline__ void cross3(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

// closed form of Eq. 42 at fixed v (reading R7), triad components
__device__ __forceinline__ void implicit_E_closed(const double v[3], double W, double s, const double Es[3],
                                                  const double B[3], double E[3]) {
  double vxB[3];
  cross3(v, B, vxB);
  const double kE = dot3(v, Es) / (1.0 + s / (W * W)), i1s = 1.0 / (1.0 + s);
#pragma unroll
  for (int i = 0; i < 3; ++i) E[i] = (Es[i] - s * vxB[i] + s * kE * v[i]) * i1s;
}

// P holds the guess (rho, p, v^i) on entry and all 14 primitives on return.  sg = sqrt(gamma).
__device__ __forceinline__ C2POut c2p_solve(const Triad& t, double isg, double alpha, double Gamma, double gog1,
                                            double gm1og, const double U[NCONS], double adt, double sigma, double tol,
                                            int maxit, unsigned lanes, double P[NPRIM]) {
  const double Dh = U[CD] * isg, tauh = U[CTAU] * isg;
  double Sh[3], Es[3], B[3], EsxB[3];
  triad_from_cov(t, U[CSX] * isg, U[CSY] * isg, U[CSZ] * isg, Sh);
  // EM fields that do not depend on the solve
#pragma unroll
  for (int i = 0; i < 3; ++i) P[BX + i] = U[CBX + i] * isg;
  P[PSI] = U[CPSI] * isg; P[PHI] = U[CPHI] * isg; P[QCH] = U[CQ] * isg;
  triad_from_contra(t, U[CEX] * isg, U[CEY] * isg, U[CEZ] * isg, Es);
  triad_from_contra(t, P[BX], P[BY], P[BZ], B);
  const double B2 = dot3(B, B);
  cross3(Es, B, EsxB);
  const double s0 = adt * alpha * sigma;
  const double em2 = dot3(Es, Es) + B2;
  double escale, ies;
  if (em2 > 1e-280) sqrt_rsqrt_fast(em2, escale, ies);
  else { escale = sqrt(em2); ies = escale > 0.0 ? 1.0 / escale : 1.0; }
  C2POut res = {0, 1};
  const double Zlo = Dh, Zhi = Gamma * (tauh + Dh - 0.5 * B2);
  // guess
  double vg[3];
  triad_from_contra(t, P[VX], P[VY], P[VZ], vg);
  double v2g = dot3(vg, vg);
  if (!(v2g < 1.0)) { vg[0] = vg[1] = vg[2] = 0.0; v2g = 0.0; }
  const double Wg = rsqrt_fast(1.0 - v2g);
  double W = Wg;
  double kE = dot3(vg, Es) * W * rcp_fast(W + s0);          // (v.E*)/(1 + s/W^2), s = s0 W
  if (!(Dh > 0.0) || !(Zhi > Zlo)) {   // no physical bracket: keep the guess, E from the guess v
    double Eh[3], EU[3];
    implicit_E_closed(vg, W, s0 * W, Es, B, Eh);
    triad_to_contra(t, Eh, EU);
    P[EX] = EU[0]; P[EY] = EU[1]; P[EZ] = EU[2];
    return res;
  }
  double Z = (P[RHO] + gog1 * P[PRS]) * W * W;
  bool converged = false, state_ok = false;
  const int max_outer = 50;
  // inverse slope of g for the first secant step: dg/dZ ~ 1 - (Gamma-1)/Gamma / W^2 at fixed v (exact in the
  // unmagnetised, slow limit), instead of 1
  double fW_prev = 0, fk_prev = 0, GW_prev = 0, Gk_prev = 0, step_prev = 0, islope = rcp_fast(1.0 - gm1og * (1.0 - v2g));
  // frozen per outer pass
  double s = 0, r = 0, i1s = 1, Npar[3] = {0, 0, 0}, Nperp[3] = {0, 0, 0}, BxN[3] = {0, 0, 0};
  // last evaluation
  double v[3] = {0, 0, 0}, E[3] = {0, 0, 0}, Wv = 1, rho = 0, p = 0;
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
        s = s0 * W; i1s = rcp_fast(1.0 + s); r = s * i1s;
        double N[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) N[i] = Sh[i] - EsxB[i] * i1s;
        const double fpar = (B2 > 1e-280) ? dot3(N, B) * rcp_fast(B2) : (B2 > 0.0) ? dot3(N, B) / B2 : 0.0;
#pragma unroll
        for (int i = 0; i < 3; ++i) { Npar[i] = fpar * B[i]; Nperp[i] = N[i] - Npar[i]; }
        cross3(B, Nperp, BxN);
        a = Zlo; b = Zhi;
        x = fmin(fmax(Z, a), b);
        okp = false;
        need_setup = false;
      }
      // ---- residual g(x) for frozen (s, kE); v^2 >= 1 counts as g = -infinity ------------------
      {
        const double A = x + r * B2, c = r * kE;
        const double iden = rcp_fast(A * A + c * c * B2), iZ = rcp_fast(x);
#pragma unroll
        for (int i = 0; i < 3; ++i) v[i] = Npar[i] * iZ + (A * Nperp[i] + c * BxN[i]) * iden;
        const double v2 = dot3(v, v);
        ok = v2 < 1.0;
        const double omv2 = ok ? 1.0 - v2 : 1.0;
        double iW;
        sqrt_rsqrt_fast(omv2, iW, Wv);                                   // 1/W, W
        double vxB[3];
        cross3(v, B, vxB);
        const double skE = s * kE;
#pragma unroll
        for (int i = 0; i < 3; ++i) E[i] = (Es[i] - s * vxB[i] + skE * v[i]) * i1s;
        rho = Dh * iW;                                                   // Eq. 45
        p = gm1og * (x * omv2 - rho);                                    // Eq. 47-49
        f = x - (tauh + Dh + p - 0.5 * (dot3(E, E) + B2));
      }
      ++res.evals;
      // ---- inner: bracketed secant / bisection on Z; invariant g(a) < 0 < g(b) -----------------
      bool inner_conv = false, inner_stop = false;
      if (ok && f == 0.0) {
        inner_conv = true;
      } else {
        if (!ok || f < 0.0) a = x; else b = x;
        const bool sec = ok && okp && f != fp && x != xp;
        const double isl = (x - xp) * rcp_fast(sec ? f - fp : 1.0);
        if (sec) islope = isl;
        const double delta = ok ? f * islope : 0.0;          // predicted distance to the root
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
          const double Wnew = Wv;
          const double kEnew = dot3(v, Es) * Wnew * rcp_fast(Wnew + s0);
          const bool same = fabs(Wnew - W) <= tol * Wnew && fabs(kEnew - kE) <= tol * escale;
          // round-off stagnation: the fixed-point residual no longer shrinks and is below 1000 tol
          const double step = fmax(fabs(Wnew - W) * rcp_fast(Wnew), fabs(kEnew - kE) * ies);
          const bool stalled = outer >= 2 && step >= step_prev && step <= 1000.0 * tol;
          step_prev = step;
          if (s0 == 0.0 || same || stalled) {
            converged = true; done = true;
          } else {
            // Anderson(1) acceleration of x -> G(x), x = (W, kE/escale)
            const double fW = Wnew - W, fk = (kEnew - kE) * ies;
            double Wnext = Wnew, knext = kEnew;
            if (outer > 0) {
              const double dW = fW - fW_prev, dk = fk - fk_prev, den = dW * dW + dk * dk;
              if (den > 0.0) {
                const double theta = (fW * dW + fk * dk) * rcp_fast(den);
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
    if (__all_sync(lanes, done)) break;                     // warp-vote exit over the lanes that entered the solve
  }
  res.failed = converged ? 0 : 1;
  double EU[3];
  if (state_ok) {
    double vU[3];
    triad_to_contra(t, v, vU);
    triad_to_contra(t, E, EU);
    P[RHO] = rho; P[PRS] = p;
#pragma unroll
    for (int i = 0; i < 3; ++i) P[VX + i] = vU[i];
  } else {
    double Eh[3];
    implicit_E_closed(vg, Wg, s0 * Wg, Es, B, Eh);
    triad_to_contra(t, Eh, EU);
  }
  P[EX] = EU[0]; P[EY] = EU[1]; P[EZ] = EU[2];
  return res;
}

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
  const bool in_range = i < G.n[0] && j < G.n[1];
  const unsigned lanes = __ballot_sync(0xffffffffu, in_range);   // the lanes that take part in the solver's warp votes
  if (in_range) {
    const long long c = cell_index(G, i, j, k);
    double g6[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) g6[q] = __ldg(G.met[MGXX + q] + c);
    const double alpha = __ldg(G.met[MALP] + c);
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
      C2POut r0 = c2p_solve(t, isg, alpha, G.Gamma, G.gog1, G.gm1og, U, 0.0, 0.0, G.tol, G.maxit, lanes, P);
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
    const double sigma = (STAGE == 3) ? 0.0 : sigma_of(G, U[CD] * isg, c);
    // The point-wise right-hand side after the solve reads ~57 more fields of this cell.  Start those loads
    // now as asynchronous copies into a thread-private shared-memory column: no registers are held and
    // the solve below hides their DRAM latency.
    extern __shared__ double pf_smem[];
    double* const pf = pf_smem + threadIdx.x;              // pf[q * NTH]: conflict-free, private to this thread
    constexpr int NTH = C2P_TX * C2P_TY;
    if (STAGE != 3) {
      // fields that are identically zero on this grid (zero shift, K_ij = 0, diagonal metric, ...) are not read
      const unsigned long long nz = __ldg(G.src_mask);
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
    C2POut r2 = c2p_solve(t, isg, alpha, G.Gamma, G.gog1, G.gm1og, U, adt, sigma, G.tol, G.maxit, lanes, P);
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

// Static source coefficients of every interior cell (once per set_metric).
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
#pragma unroll
    for (int q = 0; q < NSRC; ++q) {
      G.src[q][c] = out[q];
      if (out[q] != 0.0) nz |= 1ull << q;
    }
#pragma unroll
    for (int q = 0; q < 6; ++q)
      if (__ldg(G.met[MKXX + q] + c) != 0.0) nz |= 1ull << (NSRC + q);
  }
  // which fields are not identically zero: warp OR, one atomic per warp
  unsigned lo = (unsigned)nz, hi = (unsigned)(nz >> 32);
  lo = __reduce_or_sync(0xffffffffu, lo);
  hi = __reduce_or_sync(0xffffffffu, hi);
  if ((threadIdx.x & 31) == 0 && (lo | hi)) atomicOr(mask, ((unsigned long long)hi << 32) | lo);
}

cudaError_t launch_metric_coeffs(const GridView& G, cudaStream_t st) {
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  unsigned long long* mask = const_cast<unsigned long long*>(G.src_mask);
  cudaError_t e = cudaMemsetAsync(mask, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess) return e;
  k_metric_coeffs<<<(unsigned)((nint + 127) / 128), 128, 0, st>>>(G, mask);
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
