// tangent1d_kernel.cuh — the fused Runge-Kutta stage of stage1d_kernel.cuh carried together with its TANGENT:
// every quantity is a pair (value, derivative along one direction of perturbation of U^n and gamma), so that a run
// of stages applies the chain of Jacobians of PAPER.md Eq. 16,
//     prod_j dU^{n+j}/dU^{n+j-1}   and   dU^{n+k}/dgamma,
// to that direction.  With the loss of Eq. 14 this gives dL/dgamma = <dL/dU, Udot>: the paper's inference of the
// specific-heat ratio from Sod data (Fig. 3b).  SURVEY.md section 8(f) rank 3, forward mode: for a
// handful of scalar parameters it costs one extra pass per parameter and needs no stored trajectory (R21).
//
// One thread per cell, 128-thread CTAs that produce 126 cells (threads 0 and 127 are support cells, recomputed by
// the neighbouring CTA with identical arithmetic).  Same discretisation as the primal kernels — WENO5-JS on
// (rho, u, v, p) (Eq. 8-9, R3, R4), HLLC with Davis speeds (Eq. 3-7, R1, R2), positivity guard (R15), viscous flux
// (R8), nu Lap_h(U) (Eq. 10), the Runge-Kutta combine (R5) — written once on pairs; comparisons look at the value
// only, so min / max / sign / the guard carry the derivative of the branch the value selects.
// HBM traffic per cell-stage: 2 x (64 / 96 B) — the state and its tangent, in and out.
#pragma once
#include "stage_kernel.cuh"

namespace jxs {

constexpr int T1D_TB = 128;          // threads per CTA
constexpr int T1D_OUT = T1D_TB - 2;  // cells produced per CTA

struct Tangent1dArgs {
  const double* Uin;      // padded [4][7][pitch], ghosts filled
  const double* Uin_dot;  // its tangent, same layout, ghosts filled with the linearised boundary conditions
  const double* U0;       // U^n of the step and its tangent (read only when rk_a != 0)
  const double* U0_dot;
  double* Uout;
  double* Uout_dot;
  const double* dt;  // device scalar (a constant of the differentiation)
  long long plane;
  int nx, pitch;
  double gamma, gamma_dot, dxi, mu, Pr, nu, rk_a, rk_b;
};

// ------------------------------------------------------------------ pairs (value, derivative)
struct Dual {
  double v, d;
};
__device__ __forceinline__ Dual dual(double v, double d = 0.0) { return Dual{v, d}; }
__device__ __forceinline__ Dual operator+(Dual a, Dual b) { return Dual{a.v + b.v, a.d + b.d}; }
__device__ __forceinline__ Dual operator-(Dual a, Dual b) { return Dual{a.v - b.v, a.d - b.d}; }
__device__ __forceinline__ Dual operator-(Dual a) { return Dual{-a.v, -a.d}; }
__device__ __forceinline__ Dual operator*(Dual a, Dual b) { return Dual{a.v * b.v, fma(a.v, b.d, a.d * b.v)}; }
__device__ __forceinline__ Dual operator*(double a, Dual b) { return Dual{a * b.v, a * b.d}; }
__device__ __forceinline__ Dual operator+(Dual a, double b) { return Dual{a.v + b, a.d}; }
__device__ __forceinline__ Dual operator-(Dual a, double b) { return Dual{a.v - b, a.d}; }
// 1/b and a/b: (1/b)' = -b'/b^2, (a/b)' = (a' - (a/b) b')/b
__device__ __forceinline__ Dual rcp_dual(Dual b) {
  const double r = rcp_(b.v);
  return Dual{r, -b.d * r * r};
}
__device__ __forceinline__ Dual operator/(Dual a, Dual b) {
  const double r = rcp_(b.v), q = a.v * r;
  return Dual{q, fma(-q, b.d, a.d) * r};
}
__device__ __forceinline__ Dual sqrt_dual(Dual x) {  // sqrt(x)' = x'/(2 sqrt(x))
  const double rs = rsqrt_(x.v);
  return Dual{x.v * rs, 0.5 * x.d * rs};
}
__device__ __forceinline__ Dual min_dual(Dual a, Dual b) { return b.v < a.v ? b : a; }
__device__ __forceinline__ Dual max_dual(Dual a, Dual b) { return a.v < b.v ? b : a; }
__device__ __forceinline__ Dual fma_dual(double a, Dual b, Dual c) { return Dual{fma(a, b.v, c.v), fma(a, b.d, c.d)}; }

// WENO5-JS of one variable at one cell from (a, b, c, d, e) = cells i-2 .. i+2: the left-biased value at face i+1/2
// (Lp) and the right-biased value at face i-1/2 (Rm).  The two share the smoothness indicators (the mirrored
// stencil has beta_0 and beta_2 exchanged).  eps = 1e-6, linear weights 0.1 / 0.6 / 0.3, exponent 2 (R4).
__device__ __forceinline__ void weno5_dual(Dual a, Dual b, Dual c, Dual d, Dual e, Dual& Lp, Dual& Rm) {
  const Dual s0 = a - 2.0 * b + c, t0 = a - 4.0 * b + 3.0 * c;
  const Dual s1 = b - 2.0 * c + d, t1 = b - d;
  const Dual s2 = c - 2.0 * d + e, t2 = 3.0 * c - 4.0 * d + e;
  // (eps + beta)^2 with beta = 13/12 s^2 + 1/4 t^2, its derivative 2 (13/12 s s' + 1/4 t t') written out
  auto eps_beta_sq = [](Dual s, Dual t) {
    const double ms = (13.0 / 12.0) * s.v, mt = 0.25 * t.v;
    const double x = fma(mt, t.v, fma(ms, s.v, 1e-6));
    const double xd = 2.0 * fma(ms, s.d, mt * t.d);
    return Dual{x * x, (x + x) * xd};
  };
  const Dual e0 = eps_beta_sq(s0, t0), e1 = eps_beta_sq(s1, t1), e2 = eps_beta_sq(s2, t2);
  // alpha_k = d_k / (eps + beta_k)^2 over their sum, with the common denominator multiplied through (one division
  // per side instead of four); the 1/6 of the candidate values is folded into the linear weights
  const Dual w0 = e1 * e2, w1 = e0 * e2, w2 = e0 * e1;
  auto blend = [](Dual wa, Dual wb, Dual wc, Dual qa, Dual qb, Dual qc) {  // weights 0.1, 0.6, 0.3 on (wa, wb, wc)
    const Dual na = wa * qa, nb = wb * qb, nc = wc * qc;
    const Dual N{fma(0.1 / 6.0, na.v, fma(0.6 / 6.0, nb.v, (0.3 / 6.0) * nc.v)),
                 fma(0.1 / 6.0, na.d, fma(0.6 / 6.0, nb.d, (0.3 / 6.0) * nc.d))};
    const Dual D{fma(0.1, wa.v, fma(0.6, wb.v, 0.3 * wc.v)), fma(0.1, wa.d, fma(0.6, wb.d, 0.3 * wc.d))};
    return N / D;
  };
  // left-biased at i+1/2, and right-biased at i-1/2 = the same formula on (e, d, c, b, a)
  Lp = blend(w0, w1, w2, 2.0 * a - 7.0 * b + 11.0 * c, 5.0 * c - b + 2.0 * d, 2.0 * c + 5.0 * d - e);
  Rm = blend(w2, w1, w0, 2.0 * e - 7.0 * d + 11.0 * c, 5.0 * c - d + 2.0 * b, 2.0 * c + 5.0 * b - a);
}

// one side K of the HLLC flux (Eq. 3-4, R1): F_K + s_K^clip (U*_K - U_K) with
// U*_K = rho_K chi [1, s*, v_K, E_K/rho_K + (s* - u_K)(s* + p_K / (rho_K (s_K - u_K)))], chi = (s_K - u_K)/(s_K - s*)
__device__ __forceinline__ void hllc_side_dual(Dual r, Dual u, Dual v, Dual p, Dual sK, Dual sS, Dual sclip, Dual g1inv,
                                               Dual F[4]) {
  const Dual E = p * g1inv + 0.5 * (r * (u * u + v * v));
  const Dual ru = r * u;
  const Dual du = sK - u;
  const Dual chi = du / (sK - sS);
  const Dual rc = r * chi;
  const Dual Es = rc * (E / r + (sS - u) * (sS + p / (r * du)));
  F[0] = ru + sclip * (rc - r);
  F[1] = ru * u + p + sclip * (rc * sS - ru);
  F[2] = ru * v + sclip * (rc * v - r * v);
  F[3] = u * (E + p) + sclip * (Es - E);
}

// HLLC flux along x from primitive left / right states (Eq. 3, 5-7); sign(s*) = 0 averages the two sides (R2)
__device__ __forceinline__ void hllc_dual(const Dual L[4], const Dual R[4], Dual gamma, Dual g1inv, Dual F[4]) {
  const Dual aL = sqrt_dual(gamma * L[3] / L[0]), aR = sqrt_dual(gamma * R[3] / R[0]);
  const Dual sL = min_dual(L[1] - aL, R[1] - aR);  // Eq. 6
  const Dual sR = max_dual(L[1] + aL, R[1] + aR);
  const Dual mL = L[0] * (sL - L[1]), mR = R[0] * (sR - R[1]);
  const Dual sS = (R[3] - L[3] + mL * L[1] - mR * R[1]) / (mL - mR);  // Eq. 7
  const Dual sm = min_dual(dual(0.0), sL), sp = max_dual(dual(0.0), sR);  // Eq. 5
  if (sS.v > 0.0) hllc_side_dual(L[0], L[1], L[2], L[3], sL, sS, sm, g1inv, F);
  else if (sS.v < 0.0) hllc_side_dual(R[0], R[1], R[2], R[3], sR, sS, sp, g1inv, F);
  else {
    Dual G[4];
    hllc_side_dual(L[0], L[1], L[2], L[3], sL, sS, sm, g1inv, F);
    hllc_side_dual(R[0], R[1], R[2], R[3], sR, sS, sp, g1inv, G);
#pragma unroll
    for (int k = 0; k < 4; ++k) F[k] = 0.5 * (F[k] + G[k]);
  }
}

__global__ void __launch_bounds__(T1D_TB) tangent1d_kernel(const Tangent1dArgs A) {
  __shared__ Dual prim[5][T1D_TB + 4];  // (rho, u, v, p, T) of padded columns c0-2 .. c0+129 (T only with mu > 0)
  __shared__ Dual rmS[4][T1D_TB];       // right-biased state at each cell's left face
  __shared__ Dual fS[4][T1D_TB];        // flux through each cell's right face
  const int t = threadIdx.x;
  const int c0 = T1D_OUT * blockIdx.x + 2;  // padded column of thread 0
  const int col = c0 + t;
  const size_t row = 3 * (size_t)A.pitch;  // the one interior row of the padded buffers
  const Dual gamma = dual(A.gamma, A.gamma_dot);
  const Dual g1 = gamma - 1.0, g1inv = rcp_dual(g1);
  const bool visc = A.mu != 0.0;

  // ---- S3: conserved -> primitives of my column and (threads 0-3) of one halo column
  Dual Uc[4];
  auto to_prim = [&](int c, int slot, bool keep) {
    const size_t o = row + (size_t)min(c, A.pitch - 1);
    Dual U[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) U[k] = dual(A.Uin[k * A.plane + o], A.Uin_dot[k * A.plane + o]);
    if (keep) {
#pragma unroll
      for (int k = 0; k < 4; ++k) Uc[k] = U[k];
    }
    const Dual ri = rcp_dual(U[0]);
    const Dual u = U[1] * ri, v = U[2] * ri;
    const Dual p = g1 * (U[3] - 0.5 * (U[1] * u + U[2] * v));  // Eq. 2
    prim[0][slot] = U[0]; prim[1][slot] = u; prim[2][slot] = v; prim[3][slot] = p;
    if (visc) prim[4][slot] = p * ri;
  };
  to_prim(col, t + 2, true);
  if (t < 4) to_prim(t < 2 ? c0 - 2 + t : c0 + T1D_TB + (t - 2), t < 2 ? t : T1D_TB + t, false);
  __syncthreads();

  // ---- S4: WENO5-JS of my cell -> right-biased state at my left face, left-biased at my right face
  Dual wc[4], Lp[4];
  {
    Dual Rm[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      wc[k] = prim[k][t + 2];
      weno5_dual(prim[k][t], prim[k][t + 1], wc[k], prim[k][t + 3], prim[k][t + 4], Lp[k], Rm[k]);
    }
    const bool badR = !(Rm[0].v > 0.0) || !(Rm[3].v > 0.0);  // positivity guard (R15): fall back to the cell
    const bool badL = !(Lp[0].v > 0.0) || !(Lp[3].v > 0.0);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      rmS[k][t] = badR ? wc[k] : Rm[k];
      if (badL) Lp[k] = wc[k];
    }
  }
  __syncthreads();

  // ---- S5 (+S6): flux through my right face (thread 127 has no right neighbour in the tile: its flux is not used)
  Dual F[4];
  {
    const int tn = min(t + 1, T1D_TB - 1);
    const Dual R[4] = {rmS[0][tn], rmS[1][tn], rmS[2][tn], rmS[3][tn]};
    hllc_dual(Lp, R, gamma, g1inv, F);
    if (visc) {  // R8 at the face between my cell and the next; the cross differences of a planar flow vanish
      const int c = t + 2;
      const Dual kappa = (A.mu / A.Pr) * (gamma * g1inv);
      const Dual ux = A.dxi * (prim[1][c + 1] - prim[1][c]), vx = A.dxi * (prim[2][c + 1] - prim[2][c]);
      const Dual Tx = A.dxi * (prim[4][c + 1] - prim[4][c]);
      const Dual ub = 0.5 * (prim[1][c] + prim[1][c + 1]), vb = 0.5 * (prim[2][c] + prim[2][c + 1]);
      const Dual txx = (4.0 / 3.0 * A.mu) * ux, txy = A.mu * vx;
      F[1] = F[1] - txx;
      F[2] = F[2] - txy;
      F[3] = F[3] - (ub * txx + vb * txy + kappa * Tx);
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) fS[k][t] = F[k];
  }
  __syncthreads();

  // ---- S7: divergence (+ nu Lap_h(U), Eq. 10), S8: the Runge-Kutta combine, on the pair
  const int ic = col - 3;  // interior index
  const bool ok = t >= 1 && t <= T1D_OUT && ic < A.nx;
  Dual Lc[4];
  {
    const int tl = max(t - 1, 0);
#pragma unroll
    for (int k = 0; k < 4; ++k) Lc[k] = A.dxi * (fS[k][tl] - F[k]);
    if (A.nu != 0.0) {
      auto cons = [&](int c, Dual* U) {
        const Dual r = prim[0][c], u = prim[1][c], v = prim[2][c], p = prim[3][c];
        U[0] = r; U[1] = r * u; U[2] = r * v; U[3] = p * g1inv + 0.5 * (r * (u * u + v * v));
      };
      Dual Um[4], Uxm[4], Uxp[4];
      cons(t + 2, Um); cons(t + 1, Uxm); cons(t + 3, Uxp);
      const double ax = A.nu * A.dxi * A.dxi;
#pragma unroll
      for (int k = 0; k < 4; ++k) Lc[k] = Lc[k] + ax * (Uxp[k] - 2.0 * Um[k] + Uxm[k]);
    }
  }
  const double dtv = *A.dt;
  Dual Un[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) Un[k] = fma_dual(dtv, Lc[k], Uc[k]);
  if (A.rk_a != 0.0 && ok) {
    const size_t o = row + col;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const Dual U0 = dual(A.U0[k * A.plane + o], A.U0_dot[k * A.plane + o]);
      Un[k] = fma_dual(A.rk_a, U0, A.rk_b * Un[k]);
    }
  }
  if (ok) {
    const size_t o = row + col;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      A.Uout[k * A.plane + o] = Un[k].v;
      A.Uout_dot[k * A.plane + o] = Un[k].d;
    }
  }
}

// ------------------------------------------------------------------ the loss of Eq. 14 and its derivative
// L = mean((U - Utarget)^2), dL = mean(2 (U - Utarget) Udot) (R22).  Two launches, fixed summation order: every CTA
// sums a strided share, CTA 0 of the second launch sums the partial sums.
constexpr int MSE_TB = 256;

__device__ __forceinline__ void mse_block_sum(double& a, double& b) {
  __shared__ double sa[MSE_TB / 32], sb[MSE_TB / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
  if ((threadIdx.x & 31) == 0) { sa[threadIdx.x >> 5] = a; sb[threadIdx.x >> 5] = b; }
  __syncthreads();
  if (threadIdx.x < 32) {
    a = threadIdx.x < MSE_TB / 32 ? sa[threadIdx.x] : 0.0;
    b = threadIdx.x < MSE_TB / 32 ? sb[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
      a += __shfl_xor_sync(0xffffffffu, a, o);
      b += __shfl_xor_sync(0xffffffffu, b, o);
    }
  }
}

__global__ void __launch_bounds__(MSE_TB) mse_partial_kernel(const double* U, const double* Udot, const double* Ut,
                                                             long long n, double* partial) {
  double a = 0.0, b = 0.0;
  for (long long i = (long long)blockIdx.x * MSE_TB + threadIdx.x; i < n; i += (long long)gridDim.x * MSE_TB) {
    const double r = U[i] - Ut[i];
    a = fma(r, r, a);
    b = fma(2.0 * r, Udot[i], b);
  }
  mse_block_sum(a, b);
  if (threadIdx.x == 0) { partial[2 * blockIdx.x] = a; partial[2 * blockIdx.x + 1] = b; }
}

__global__ void __launch_bounds__(MSE_TB) mse_final_kernel(const double* partial, int nparts, double inv_n, double* out) {
  double a = 0.0, b = 0.0;
  for (int i = threadIdx.x; i < nparts; i += MSE_TB) { a += partial[2 * i]; b += partial[2 * i + 1]; }
  mse_block_sum(a, b);
  if (threadIdx.x == 0) { out[0] = a * inv_n; out[1] = b * inv_n; }
}

}  // namespace jxs
