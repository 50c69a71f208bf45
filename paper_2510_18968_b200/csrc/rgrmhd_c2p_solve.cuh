// rgrmhd_c2p_solve.cuh -- a6, one cell: the implicit Ohm's-law update of the electric field fused with the 1D
// conservative-to-primitive recovery (Eq. 42-50), all iterations in registers.  Shared by the
// recovery kernels of the IMEX-SSP2(2,2,2) path (rgrmhd_c2p.cu) and of the general tableau driver (rgrmhd_imex_gen.cu).
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
// convergently; a lane leaves the loop when it is done and waits for the rest of its warp at the loop's exit (an
// explicit warp vote per trip, the round-1 version, measured 3 % slower for the whole kernel).
#pragma once
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
                                            int maxit, double P[NPRIM]) {
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
  // no physical bracket: a failure; keep the guess, E from the guess v (the tail below does exactly that for a lane
  // without a valid state): such a lane never enters the loop.
  const bool no_bracket = !(Dh > 0.0) || !(Zhi > Zlo);
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
  bool need_setup = true, done = no_bracket;
  // ONE loop, one residual evaluation per trip.
  while (!done) {
    {
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

}  // namespace rg
