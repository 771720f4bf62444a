// stage1d_kernel.cuh — the fused Runge-Kutta stage for ONE-dimensional problems (ny = 1): the paper's Sod
// shock-tube workload (Eq. 17; its scaling study runs up to 9e6 degrees of freedom).
// SURVEY.md section 8(f) rank 2.  Same discretisation as stage_kernel.cuh restricted to x — the same device
// routines (weno5_n, hllc_n, rcp_n, rsqrt_n) — so a planar problem run through the 2D path and through this
// one agree to round-off: the y-fluxes of identical rows cancel exactly.
//
// One thread per cell, 256-thread CTAs that produce 254 cells: thread t owns padded column 254 b + 2 + t,
// threads 0 and 255 are support cells recomputed by the neighbouring CTA with identical arithmetic.
// Primitives of the tile (+2 halo columns per side), the right-biased states and the face fluxes go through
// shared memory once each; nothing but U crosses HBM (24 B per cell-stage for (rho, rho u, E) would be the
// floor; this kernel also carries rho v so that the C ABI keeps one layout: 64 / 96 B per cell-stage).
// With mu > 0 the viscous flux of stage_kernel.cuh (R8) is added at the face, its cross terms being zero.
#pragma once
#include "stage_kernel.cuh"

namespace jxs {

constexpr int S1D_TB = 256;          // threads per CTA
constexpr int S1D_OUT = S1D_TB - 2;  // cells produced per CTA

#define JXS_V _Pragma("unroll") for (int k = 0; k < N; ++k)

template <typename T>
__global__ void __launch_bounds__(S1D_TB) stage1d_kernel(const StageArgs<T> A) {
  __shared__ T prim[5][S1D_TB + 4];  // (rho, u, v, p, T) of padded columns c0-2 .. c0+257 (T only with mu > 0)
  __shared__ T rmS[4][S1D_TB];       // right-biased state at each cell's left face
  __shared__ T fS[4][S1D_TB];        // flux through each cell's right face
  const int t = threadIdx.x;
  const int c0 = S1D_OUT * blockIdx.x + 2;  // padded column of thread 0
  const int col = c0 + t;
  const T* row = A.Uin + 3 * (size_t)A.pitch;  // the one interior row of the padded buffer
  const T g1 = A.g1, g1inv = A.g1inv, gamma = A.gamma;
  const bool visc = A.mu != T(0);

  // U^n of my cell for the Runge-Kutta combine: requested first, used last
  T U0c[4] = {T(0), T(0), T(0), T(0)};
  if (A.mode == 0 && A.rk_a != T(0)) {
    const T* row0 = A.U0 + 3 * (size_t)A.pitch + min(col, A.pitch - 1);
#pragma unroll
    for (int k = 0; k < 4; ++k) U0c[k] = row0[k * A.plane];
  }
  // ---- S3: conserved -> primitives of my column and (threads 0-3) of one halo column
  T Uc[4];
  {
    constexpr int N = 2;
    const int hc = t < 2 ? c0 - 2 + t : c0 + S1D_TB + (t - 2);  // halo column of threads 0..3
    const int cc[N] = {min(col, A.pitch - 1), min(t < 4 ? hc : col, A.pitch - 1)};
    T r[N], ru[N], rv[N], E[N], ri[N], u[N], v[N], p[N];
    JXS_V { r[k] = row[cc[k]]; ru[k] = row[A.plane + cc[k]]; rv[k] = row[2 * A.plane + cc[k]]; E[k] = row[3 * A.plane + cc[k]]; }
    Uc[0] = r[0]; Uc[1] = ru[0]; Uc[2] = rv[0]; Uc[3] = E[0];
    rcp_n<T, N>(r, ri);
    JXS_V u[k] = ru[k] * ri[k];
    JXS_V v[k] = rv[k] * ri[k];
    JXS_V p[k] = rv[k] * v[k];
    JXS_V p[k] = fma_(ru[k], u[k], p[k]);
    JXS_V p[k] = fma_(T(-0.5), p[k], E[k]);
    JXS_V p[k] = g1 * p[k];
    prim[0][t + 2] = r[0]; prim[1][t + 2] = u[0]; prim[2][t + 2] = v[0]; prim[3][t + 2] = p[0];
    if (visc) prim[4][t + 2] = p[0] * ri[0];
    if (t < 4) {
      const int o = t < 2 ? t : S1D_TB + t;
      prim[0][o] = r[1]; prim[1][o] = u[1]; prim[2][o] = v[1]; prim[3][o] = p[1];
      if (visc) prim[4][o] = p[1] * ri[1];
    }
  }
  __syncthreads();

  // ---- S4: WENO5-JS of my cell -> right-biased state at my left face, left-biased at my right face
  T wc[4], Rm[4], Lp[4];
  {
    constexpr int N = 4;
    T a[N], b[N], d[N], e[N];
    JXS_V { a[k] = prim[k][t]; b[k] = prim[k][t + 1]; wc[k] = prim[k][t + 2]; d[k] = prim[k][t + 3]; e[k] = prim[k][t + 4]; }
    weno5_n<T, N>(a, b, wc, d, e, A, Rm, Lp);
    const bool badR = any_not_positive(Rm[0], Rm[3]);  // positivity guard (R15)
    const bool badL = any_not_positive(Lp[0], Lp[3]);
    JXS_V { Rm[k] = badR ? wc[k] : Rm[k]; Lp[k] = badL ? wc[k] : Lp[k]; }
    JXS_V rmS[k][t] = Rm[k];
  }
  __syncthreads();

  // ---- S5: HLLC at my right face (thread 255 has no right neighbour in the tile: its flux is not used)
  T F[4];
  {
    constexpr int N = 1;
    const int tn = min(t + 1, S1D_TB - 1);
    const T rL[N] = {Lp[0]}, unL[N] = {Lp[1]}, utL[N] = {Lp[2]}, pL[N] = {Lp[3]};
    const T rR[N] = {rmS[0][tn]}, unR[N] = {rmS[1][tn]}, utR[N] = {rmS[2][tn]}, pR[N] = {rmS[3][tn]};
    T f0[N], f1[N], f2[N], f3[N];
    hllc_n<T, N>(rL, unL, utL, pL, rR, unR, utR, pR, gamma, g1inv, f0, f1, f2, f3);
    if (visc) {  // S6 (R8) at my right face; the cross differences of a planar flow vanish
      const int c = t + 2;
      const T dn[N] = {prim[1][c + 1] - prim[1][c]}, dt_[N] = {prim[2][c + 1] - prim[2][c]}, zero[N] = {T(0)};
      const T sn[N] = {prim[1][c] + prim[1][c + 1]}, st[N] = {prim[2][c] + prim[2][c + 1]};
      const T dT[N] = {prim[4][c + 1] - prim[4][c]};
      const T cn[N] = {A.vx_n}, cc[N] = {A.vx_c}, cs[N] = {A.vx_s}, ct[N] = {A.vx_t}, cq[N] = {A.vx_q};
      viscous_n<T, N>(dn, dt_, zero, zero, sn, st, dT, cn, cc, cs, ct, cq, f1, f2, f3);
    }
    F[0] = f0[0]; F[1] = f1[0]; F[2] = f2[0]; F[3] = f3[0];
    if (A.dF1d) {  // Eq. 11: + F^Neural of this face (mlp1d_kernel.cuh)
      const size_t o = 3 * (size_t)A.pitch + min(col, A.pitch - 1);
#pragma unroll
      for (int k = 0; k < 4; ++k) F[k] += T(A.dF1d[k * A.plane + o]);
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) fS[k][t] = F[k];
  }
  __syncthreads();

  // ---- S7: divergence (+ the nu Lap_h(U) term of Eq. 10), S8: combine, S9: wavespeed of the new state
  const int ic = col - 3;  // interior index
  const bool ok = t >= 1 && t <= S1D_OUT && ic < A.nx;
  T Lc[4];
  {
    const int tl = max(t - 1, 0);
#pragma unroll
    for (int k = 0; k < 4; ++k) Lc[k] = (fS[k][tl] - F[k]) * A.dxi;
    if (A.nu != T(0)) {
      auto cons = [&](int c, T* U) {
        const T r = prim[0][c], u = prim[1][c], v = prim[2][c], p = prim[3][c];
        U[0] = r; U[1] = r * u; U[2] = r * v; U[3] = fma_(T(0.5) * r, fma_(u, u, v * v), p * g1inv);
      };
      T Um[4], Uxm[4], Uxp[4];
      cons(t + 2, Um); cons(t + 1, Uxm); cons(t + 3, Uxp);
      const T ax = A.nu * A.dxi * A.dxi;
#pragma unroll
      for (int k = 0; k < 4; ++k) Lc[k] += ax * (Uxp[k] - T(2) * Um[k] + Uxm[k]);
    }
  }
  T smax = T(0);
  if (A.mode == 1) {
    if (ok) {
#pragma unroll
      for (int k = 0; k < 4; ++k) A.Uout[(size_t)k * A.nx + ic] = Lc[k];
    }
  } else {
    const T dtv = T(*A.dt);
    T Un[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) Un[k] = fma_(dtv, Lc[k], Uc[k]);
    if (A.rk_a != T(0)) {
#pragma unroll
      for (int k = 0; k < 4; ++k) Un[k] = fma_(A.rk_a, U0c[k], A.rk_b * Un[k]);
    }
    if (ok) {
      T* o = A.Uout + 3 * (size_t)A.pitch + col;
#pragma unroll
      for (int k = 0; k < 4; ++k) o[k * A.plane] = Un[k];
    }
    if (A.smax_bits) {
      const T ri = rcp_(Un[0]);
      const T u = Un[1] * ri, v = Un[2] * ri;
      const T p = g1 * fma_(T(-0.5), fma_(Un[1], u, Un[2] * v), Un[3]);
      const T gp = gamma * p;
      const T a = gp * rsqrt_(gp * Un[0]);
      const T s = max_(abs_(u), abs_(v)) + a;
      if (ok) smax = s;  // NaN propagates through the reduction below
    }
  }
  if (A.smax_bits) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const T other = __shfl_xor_sync(0xffffffffu, smax, o);
      smax = (other > smax || other != other) ? other : smax;
    }
    // one atomic per CTA: the warp maxima go through shared memory (rmS was last read before the previous barrier)
    if ((t & 31) == 0) rmS[0][t >> 5] = smax;
    __syncthreads();
    if (t < 32) {
      T m = t < S1D_TB / 32 ? rmS[0][t] : T(0);
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) {
        const T other = __shfl_xor_sync(0xffffffffu, m, o);
        m = (other > m || other != other) ? other : m;
      }
      if (t == 0) atomic_max_pos(A.smax_bits, (double)m);
    }
  }
}

#undef JXS_V

}  // namespace jxs
