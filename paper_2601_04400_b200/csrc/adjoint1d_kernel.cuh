// adjoint1d_kernel.cuh — the ADJOINT (reverse mode) of the one-dimensional Euler stage: Eq. 15-16:
// "gradients ... are computed via backpropagation through the full sequence of unrolled solver steps".  For the stage
//     U_out = b (U + dt L(U; gamma))        (+ a U0, whose adjoint a Ubar_out the caller adds)
// and an adjoint Ubar_out of its result, this kernel returns
//     Ubar_in = b (Ubar_out + dt (dL/dU)^T Ubar_out)   and   gamma_bar += b dt <dL/dgamma, Ubar_out>,
// the transposed Jacobians of PAPER.md Eq. 16 applied from the left.  SURVEY.md section 8(f) rank 3 (R21,
// R24).  Hand-derived reverse sweep through S8 -> S7 -> S5 (HLLC, Eq. 3-7) -> S4 (WENO5-JS) -> S3 (primitives); every
// branch of the forward sweep (min / max of the wave speeds, sign of s*, the positivity guard) is re-taken from the
// stored stage state, and carries the derivative of the branch taken, as in tangent1d_kernel.cuh.
//
// One thread per PADDED cell (ghost cells included: their adjoints are folded onto the cells the boundary conditions
// copy them from by adjoint1d_fold_kernel), 128-thread CTAs that produce 122 cells: a cell's adjoint collects
// contributions from the reconstructions of cells c-2 .. c+2, which need the flux adjoints of faces c-3+1/2 .. c+2+1/2.
// Scatter is turned into gather through shared memory: no atomics, fixed summation order.
// With mu > 0 the viscous flux of the 1D stage (R8, kappa depends on gamma) and with nu > 0 the nu Lap_h(U) term
// are reversed as well.  fp64.
#pragma once
#include "aux_kernels.cuh"
#include "stage_kernel.cuh"

namespace jxs {

constexpr int A1D_TB = 128;          // threads per CTA
constexpr int A1D_OUT = A1D_TB - 6;  // cells produced per CTA

struct Adjoint1dArgs {
  const double* U;         // padded row (compact: [4][pitch]), ghosts filled: the stage's input state
  const double* Ubar_out;  // adjoint of the stage's result, same layout, zero outside the interior
  double* Ubar_in;         // adjoint of the stage's input, same layout, ghost columns included
  const double* E1;        // optional: Ubar_in += e1 E1 + e2 E2 on interior cells (the a U0 terms of later stages)
  const double* E2;
  const double* Wmlp;      // optional: adjoint of the primitives through the network input (mlp1d_backward_kernel)
  double* gbar_partial;    // [gridDim.x] this launch's contributions to gamma_bar
  double dt;               // the step size (a constant of the differentiation)
  long long plane;         // pitch (compact layout)
  int nx, pitch;
  double gamma, dxi, b, e1, e2;
  double mu, Pr, nu;       // viscous flux (R8) and the nu Lap_h(U) term of Eq. 10; 0 = absent
};

// WENO5-JS values of one variable at one cell (as weno5_dual in tangent1d_kernel.cuh, values only) and, given the
// adjoints (Lb, Rb) of the two results, the adjoints of the five cell values
__device__ __forceinline__ void weno5_val(double a, double b, double c, double d, double e, double& Lp, double& Rm,
                                          double& Di, double& Ei) {
  const double s0 = a - 2.0 * b + c, t0 = a - 4.0 * b + 3.0 * c;
  const double s1 = b - 2.0 * c + d, t1 = b - d;
  const double s2 = c - 2.0 * d + e, t2 = 3.0 * c - 4.0 * d + e;
  const double c1 = 13.0 / 12.0;
  const double x0 = fma(0.25 * t0, t0, fma(c1 * s0, s0, 1e-6));
  const double x1 = fma(0.25 * t1, t1, fma(c1 * s1, s1, 1e-6));
  const double x2 = fma(0.25 * t2, t2, fma(c1 * s2, s2, 1e-6));
  const double e0 = x0 * x0, e1 = x1 * x1, e2 = x2 * x2;
  const double w0 = e1 * e2, w1 = e0 * e2, w2 = e0 * e1;
  const double k0 = 0.1 / 6.0, k1 = 0.6 / 6.0, k2 = 0.3 / 6.0;
  Di = rcp_(0.1 * w0 + 0.6 * w1 + 0.3 * w2);  // the two reciprocals are kept for the reverse sweep
  Ei = rcp_(0.1 * w2 + 0.6 * w1 + 0.3 * w0);
  Lp = (k0 * w0 * (2.0 * a - 7.0 * b + 11.0 * c) + k1 * w1 * (5.0 * c - b + 2.0 * d) + k2 * w2 * (2.0 * c + 5.0 * d - e)) * Di;
  Rm = (k0 * w2 * (2.0 * e - 7.0 * d + 11.0 * c) + k1 * w1 * (5.0 * c - d + 2.0 * b) + k2 * w0 * (2.0 * c + 5.0 * b - a)) * Ei;
}

// (Lp, Rm, Di, Ei: the forward values and reciprocals of weno5_val; they multiply Lb / Rb only, so after the
// positivity guard, which zeroes the adjoint it replaces, any finite numbers do)
__device__ __forceinline__ void weno5_adjoint(double a, double b, double c, double d, double e, double Lb, double Rb,
                                              double Lp, double Rm, double Di, double Ei, double g[5]) {
  const double s0 = a - 2.0 * b + c, t0 = a - 4.0 * b + 3.0 * c;
  const double s1 = b - 2.0 * c + d, t1 = b - d;
  const double s2 = c - 2.0 * d + e, t2 = 3.0 * c - 4.0 * d + e;
  const double c1 = 13.0 / 12.0;
  const double x0 = fma(0.25 * t0, t0, fma(c1 * s0, s0, 1e-6));
  const double x1 = fma(0.25 * t1, t1, fma(c1 * s1, s1, 1e-6));
  const double x2 = fma(0.25 * t2, t2, fma(c1 * s2, s2, 1e-6));
  const double e0 = x0 * x0, e1 = x1 * x1, e2 = x2 * x2;
  const double w0 = e1 * e2, w1 = e0 * e2, w2 = e0 * e1;
  const double k0 = 0.1 / 6.0, k1 = 0.6 / 6.0, k2 = 0.3 / 6.0;
  // left-biased value Lp = N / D
  const double Q0 = 2.0 * a - 7.0 * b + 11.0 * c, Q1 = 5.0 * c - b + 2.0 * d, Q2 = 2.0 * c + 5.0 * d - e;
  const double Nb = Lb * Di, Db = -Nb * Lp;
  double w0b = Nb * k0 * Q0 + Db * 0.1, w1b = Nb * k1 * Q1 + Db * 0.6, w2b = Nb * k2 * Q2 + Db * 0.3;
  const double Q0b = Nb * k0 * w0, Q1b = Nb * k1 * w1, Q2b = Nb * k2 * w2;
  // right-biased value Rm = N' / D' (the mirrored stencil: w0 and w2 exchanged)
  const double P0 = 2.0 * e - 7.0 * d + 11.0 * c, P1 = 5.0 * c - d + 2.0 * b, P2 = 2.0 * c + 5.0 * b - a;
  const double Mb = Rb * Ei, Eb = -Mb * Rm;
  w2b += Mb * k0 * P0 + Eb * 0.1; w1b += Mb * k1 * P1 + Eb * 0.6; w0b += Mb * k2 * P2 + Eb * 0.3;
  const double P0b = Mb * k0 * w2, P1b = Mb * k1 * w1, P2b = Mb * k2 * w0;
  // weights -> (eps + beta)^2 -> s, t
  const double e0b = w1b * e2 + w2b * e1, e1b = w0b * e2 + w2b * e0, e2b = w0b * e1 + w1b * e0;
  const double x0b = 2.0 * x0 * e0b, x1b = 2.0 * x1 * e1b, x2b = 2.0 * x2 * e2b;
  const double s0b = 2.0 * c1 * s0 * x0b, t0b = 0.5 * t0 * x0b;
  const double s1b = 2.0 * c1 * s1 * x1b, t1b = 0.5 * t1 * x1b;
  const double s2b = 2.0 * c1 * s2 * x2b, t2b = 0.5 * t2 * x2b;
  // the linear maps, transposed
  g[0] = s0b + t0b + 2.0 * Q0b - P2b;
  g[1] = -2.0 * s0b - 4.0 * t0b + s1b + t1b - 7.0 * Q0b - Q1b + 2.0 * P1b + 5.0 * P2b;
  g[2] = s0b + 3.0 * t0b - 2.0 * s1b + s2b + 3.0 * t2b + 11.0 * Q0b + 5.0 * Q1b + 2.0 * Q2b + 11.0 * P0b + 5.0 * P1b + 2.0 * P2b;
  g[3] = s1b - t1b - 2.0 * s2b - 4.0 * t2b + 2.0 * Q1b + 5.0 * Q2b - 7.0 * P0b - P1b;
  g[4] = s2b + t2b - Q2b + 2.0 * P0b;
}

// adjoint of one side K of the HLLC flux (hllc_side_dual in tangent1d_kernel.cuh): given the flux adjoint f, add to
// the adjoints of the side's state W = (rho, u, v, p), of the wave speeds sK, s*, of the clipped speed sc and of
// g = 1/(gamma-1)
__device__ __forceinline__ void hllc_side_adjoint(const double W[4], double ri, double sK, double sS, double sc, double g,
                                                  const double f[4], double Wb[4], double& sKb, double& sSb, double& scb,
                                                  double& gb) {  // ri = 1 / rho
  const double r = W[0], u = W[1], v = W[2], p = W[3];
  const double q = u * u + v * v;
  const double E = p * g + 0.5 * r * q;
  const double ru = r * u, du = sK - u, den = sK - sS;
  const double deni = rcp_(den);
  const double chi = du * deni, rc = r * chi;
  const double A = r * du, Ai = rcp_(A), B = p * Ai;
  const double Cc = sS + B, Dd = sS - u;
  const double H = E * ri + Dd * Cc, Es = rc * H;
  double rb = 0.0, ub = 0.0, vb = 0.0, pb = 0.0, Eb = 0.0, rub = 0.0, rcb = 0.0;
  // F3 = u (E + p) + sc (Es - E)
  ub += f[3] * (E + p); Eb += f[3] * (u - sc); pb += f[3] * u; scb += f[3] * (Es - E);
  const double Esb = f[3] * sc;
  // F2 = ru v + sc (rc v - r v)
  rub += f[2] * v; vb += f[2] * (ru + sc * (rc - r)); scb += f[2] * (rc * v - r * v); rcb += f[2] * sc * v; rb -= f[2] * sc * v;
  // F1 = ru u + p + sc (rc sS - ru)
  rub += f[1] * (u - sc); ub += f[1] * ru; pb += f[1]; scb += f[1] * (rc * sS - ru); rcb += f[1] * sc * sS; sSb += f[1] * sc * rc;
  // F0 = ru + sc (rc - r)
  rub += f[0]; scb += f[0] * (rc - r); rcb += f[0] * sc; rb -= f[0] * sc;
  // Es = rc H, H = E / r + Dd Cc
  rcb += Esb * H;
  const double Hb = Esb * rc;
  Eb += Hb * ri; rb -= Hb * E * ri * ri;
  const double Ddb = Hb * Cc, Ccb = Hb * Dd;
  sSb += Ddb + Ccb; ub -= Ddb;
  // B = p / A, A = r du
  pb += Ccb * Ai;
  const double Ab = -Ccb * B * Ai;
  rb += Ab * du;
  double dub = Ab * r;
  // rc = r chi, chi = du / den, den = sK - sS, du = sK - u
  rb += rcb * chi;
  const double chib = rcb * r;
  dub += chib * deni;
  const double denb = -chib * chi * deni;
  sKb += denb + dub; sSb -= denb; ub -= dub;
  // ru = r u;  E = p g + r q / 2;  q = u^2 + v^2
  rb += rub * u; ub += rub * r;
  pb += Eb * g; gb += Eb * p; rb += 0.5 * Eb * q;
  const double qb = 0.5 * Eb * r;
  ub += 2.0 * qb * u; vb += 2.0 * qb * v;
  Wb[0] += rb; Wb[1] += ub; Wb[2] += vb; Wb[3] += pb;
}

// adjoint of the HLLC flux F(WL, WR; gamma) (hllc_dual): Lb, Rb = adjoints of the two states, returns gamma_bar
__device__ __forceinline__ double hllc_adjoint(const double L[4], const double R[4], double gamma, const double f[4],
                                               double Lb[4], double Rb[4]) {
  const double g = rcp_(gamma - 1.0);
  const double rLi = rcp_(L[0]), rRi = rcp_(R[0]);
  const double zL = gamma * L[3] * rLi, zR = gamma * R[3] * rRi;
  const double aLi = rsqrt_(zL), aRi = rsqrt_(zR), aL = zL * aLi, aR = zR * aRi;
  const double xa = L[1] - aL, xb = R[1] - aR, ya = L[1] + aL, yb = R[1] + aR;
  const bool sL_from_R = xb < xa, sR_from_R = ya < yb;
  const double sL = sL_from_R ? xb : xa, sR = sR_from_R ? yb : ya;
  const double mL = L[0] * (sL - L[1]), mR = R[0] * (sR - R[1]);
  const double dn = mL - mR, dni = rcp_(dn);
  const double sS = (R[3] - L[3] + mL * L[1] - mR * R[1]) * dni;
  const double sm = sL < 0.0 ? sL : 0.0, sp = 0.0 < sR ? sR : 0.0;
#pragma unroll
  for (int k = 0; k < 4; ++k) { Lb[k] = 0.0; Rb[k] = 0.0; }
  double sLb = 0.0, sRb = 0.0, sSb = 0.0, smb = 0.0, spb = 0.0, gb = 0.0;
  if (sS > 0.0) hllc_side_adjoint(L, rLi, sL, sS, sm, g, f, Lb, sLb, sSb, smb, gb);
  else if (sS < 0.0) hllc_side_adjoint(R, rRi, sR, sS, sp, g, f, Rb, sRb, sSb, spb, gb);
  else {
    const double h[4] = {0.5 * f[0], 0.5 * f[1], 0.5 * f[2], 0.5 * f[3]};
    hllc_side_adjoint(L, rLi, sL, sS, sm, g, h, Lb, sLb, sSb, smb, gb);
    hllc_side_adjoint(R, rRi, sR, sS, sp, g, h, Rb, sRb, sSb, spb, gb);
  }
  if (sL < 0.0) sLb += smb;  // sm = min(0, sL), sp = max(0, sR)
  if (0.0 < sR) sRb += spb;
  // s* = num / dn
  const double numb = sSb * dni, dnb = -numb * sS;
  double mLb = dnb + numb * L[1], mRb = -dnb - numb * R[1];
  Rb[3] += numb; Lb[3] -= numb; Lb[1] += numb * mL; Rb[1] -= numb * mR;
  // mL = rL (sL - uL), mR = rR (sR - uR)
  Lb[0] += mLb * (sL - L[1]); sLb += mLb * L[0]; Lb[1] -= mLb * L[0];
  Rb[0] += mRb * (sR - R[1]); sRb += mRb * R[0]; Rb[1] -= mRb * R[0];
  // sL = min(uL - aL, uR - aR), sR = max(uL + aL, uR + aR)
  double aLb = 0.0, aRb = 0.0;
  if (sL_from_R) { Rb[1] += sLb; aRb -= sLb; } else { Lb[1] += sLb; aLb -= sLb; }
  if (sR_from_R) { Rb[1] += sRb; aRb += sRb; } else { Lb[1] += sRb; aLb += sRb; }
  // a = sqrt(z), z = gamma p / rho
  double gammab = 0.0;
  {
    const double zb = 0.5 * aLb * aLi;
    gammab += zb * L[3] * rLi; Lb[3] += zb * gamma * rLi; Lb[0] -= zb * zL * rLi;
  }
  {
    const double zb = 0.5 * aRb * aRi;
    gammab += zb * R[3] * rRi; Rb[3] += zb * gamma * rRi; Rb[0] -= zb * zR * rRi;
  }
  return gammab - gb * g * g;  // g = 1 / (gamma - 1)
}

// NS: the viscous flux and / or the nu-term are present (mu > 0 or nu > 0)
template <bool NS>
__global__ void __launch_bounds__(A1D_TB) adjoint1d_kernel(const Adjoint1dArgs A) {
  __shared__ double prim[4][A1D_TB + 4];   // (rho, u, v, p) of padded columns pc0-2 .. pc0+129
  __shared__ double rmS[4][A1D_TB];        // right-biased state at each cell's left face (values)
  __shared__ double LbS[4][A1D_TB];        // adjoint of L at each cell: b dt Ubar_out on interior cells, else 0
  __shared__ double rmB[4][A1D_TB + 1];    // adjoint of the right-biased state at each cell's left face
  __shared__ double con[4][5][A1D_TB];     // each cell's reconstruction adjoints for cells c-2 .. c+2
  __shared__ double visN[4][A1D_TB + 1];   // viscous flux: adjoint of (rho, u, v, p) of the cell right of each face
  __shared__ double red[A1D_TB / 32];
  const int t = threadIdx.x;
  const int pc0 = A1D_OUT * blockIdx.x - 3;  // padded column of thread 0
  const int pc = pc0 + t;
  const int last = A.nx + 5;                 // last padded column
  const double g1 = A.gamma - 1.0;
  const double bdt = A.b * A.dt;
  const bool interior = pc >= 3 && pc <= A.nx + 2;

  // ---- forward: primitives of the tile, my L adjoint
  auto to_prim = [&](int c, int slot) {
    const size_t o = (size_t)min(max(c, 0), last);
    const double r = A.U[o], ru = A.U[A.plane + o], rv = A.U[2 * A.plane + o], E = A.U[3 * A.plane + o];
    const double ri = rcp_(r), u = ru * ri, v = rv * ri;
    prim[0][slot] = r; prim[1][slot] = u; prim[2][slot] = v; prim[3][slot] = g1 * (E - 0.5 * (ru * u + rv * v));
  };
  to_prim(pc, t + 2);
  if (t < 4) to_prim(t < 2 ? pc0 - 2 + t : pc0 + A1D_TB + (t - 2), t < 2 ? t : A1D_TB + t);
  double Ub[4] = {0.0, 0.0, 0.0, 0.0};
  if (interior) {
#pragma unroll
    for (int k = 0; k < 4; ++k) Ub[k] = A.Ubar_out[k * A.plane + pc];
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) LbS[k][t] = bdt * Ub[k];
  if (t == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) { rmB[k][0] = 0.0; visN[k][0] = 0.0; }
  }
  __syncthreads();

  // ---- forward: my reconstruction (cells pc-2 .. pc+2 must exist), the guard's decisions
  const bool stencil = pc >= 2 && pc <= A.nx + 3;
  double wc[4], Lp[4], Rm[4];
  bool badL = false, badR = false;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    wc[k] = prim[k][t + 2];
    Lp[k] = Rm[k] = wc[k];
    double Di = 0.0, Ei = 0.0;
    if (stencil) weno5_val(prim[k][t], prim[k][t + 1], wc[k], prim[k][t + 3], prim[k][t + 4], Lp[k], Rm[k], Di, Ei);
    con[k][0][t] = Di;  // my own slots of the gather array, free until my reverse sweep fills them
    con[k][1][t] = Ei;
  }
  if (stencil) {
    badR = !(Rm[0] > 0.0) || !(Rm[3] > 0.0);
    badL = !(Lp[0] > 0.0) || !(Lp[3] > 0.0);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (badR) Rm[k] = wc[k];
    if (badL) Lp[k] = wc[k];
    rmS[k][t] = Rm[k];
  }
  __syncthreads();

  // ---- reverse S7 + S5: the face to my right (between pc and pc+1) carries flux adjoint (Lbar_{pc+1} - Lbar_pc)/dx
  const bool face = pc >= 2 && pc <= A.nx + 2 && t < A1D_TB - 1;
  const bool mine = t >= 3 && t <= A1D_TB - 4 && pc <= last;  // the cells (and faces) this CTA accounts for
  double Lpb[4] = {0.0, 0.0, 0.0, 0.0}, gbar = 0.0;
  double vo[4] = {0.0, 0.0, 0.0, 0.0};  // viscous flux of this face: adjoint of my cell's (rho, u, v, p)
  {
    double Rnb[4] = {0.0, 0.0, 0.0, 0.0}, vn[4] = {0.0, 0.0, 0.0, 0.0};
    if (face) {
      double f[4], R[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { f[k] = A.dxi * (LbS[k][t + 1] - LbS[k][t]); R[k] = rmS[k][t + 1]; }
      double gb = hllc_adjoint(Lp, R, A.gamma, f, Lpb, Rnb);
      if (NS && A.mu != 0.0) {
        // F -= (0, txx, txy, ub txx + vb txy + kappa Tx), txx = 4/3 mu ux, txy = mu vx, T = p / rho (R8, 1D)
        const int c = t + 2;
        const double rc_ = prim[0][c], rn = prim[0][c + 1], rci = rcp_(rc_), rni = rcp_(rn);
        const double Tc = prim[3][c] * rci, Tn = prim[3][c + 1] * rni;
        const double kappa = A.mu / A.Pr * A.gamma * rcp_(g1);
        const double ux = A.dxi * (prim[1][c + 1] - prim[1][c]), vx = A.dxi * (prim[2][c + 1] - prim[2][c]);
        const double Tx = A.dxi * (Tn - Tc);
        const double ub = 0.5 * (prim[1][c] + prim[1][c + 1]), vb = 0.5 * (prim[2][c] + prim[2][c + 1]);
        const double txx = 4.0 / 3.0 * A.mu * ux, txy = A.mu * vx;
        const double uxb = -(4.0 / 3.0 * A.mu) * (f[1] + f[3] * ub) * A.dxi, vxb = -A.mu * (f[2] + f[3] * vb) * A.dxi;
        const double ubb = -0.5 * f[3] * txx, vbb = -0.5 * f[3] * txy, Txb = -f[3] * kappa * A.dxi;
        vo[1] = ubb - uxb; vn[1] = ubb + uxb;
        vo[2] = vbb - vxb; vn[2] = vbb + vxb;
        vo[3] = -Txb * rci; vo[0] = Txb * Tc * rci;   // T = p / rho
        vn[3] = Txb * rni; vn[0] = -Txb * Tn * rni;
        gb += f[3] * Tx * (A.mu / A.Pr) * rcp_(g1 * g1);  // kappa = mu gamma / ((gamma-1) Pr)
      }
      if (mine) gbar += gb;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      rmB[k][t + 1] = Rnb[k];
      if (NS) visN[k][t + 1] = vn[k];
    }
  }
  __syncthreads();

  // ---- reverse S4: my reconstruction's adjoints for cells pc-2 .. pc+2 (the guard sends them to my own cell)
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    double g[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    const double Rb = rmB[k][t];
    if (stencil) {
      weno5_adjoint(prim[k][t], prim[k][t + 1], wc[k], prim[k][t + 3], prim[k][t + 4], badL ? 0.0 : Lpb[k], badR ? 0.0 : Rb,
                    Lp[k], rmS[k][t], con[k][0][t], con[k][1][t], g);
      g[2] += (badL ? Lpb[k] : 0.0) + (badR ? Rb : 0.0);
    }
#pragma unroll
    for (int j = 0; j < 5; ++j) con[k][j][t] = g[j];
  }
  // the U0 terms of the Shu-Osher combine: requested before the barrier, used after the gather
  double Ex[4] = {0.0, 0.0, 0.0, 0.0};
  if (interior && mine) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (A.E1) Ex[k] = A.e1 * A.E1[k * A.plane + pc];
      if (A.E2) Ex[k] = fma(A.e2, A.E2[k * A.plane + pc], Ex[k]);
    }
  }
  __syncthreads();

  // ---- gather, reverse S3 (primitives -> conserved), S8
  if (mine) {
    double Wb[4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
      Wb[k] = con[k][0][t + 2] + con[k][1][t + 1] + con[k][2][t] + con[k][3][t - 1] + con[k][4][t - 2] +
              (NS ? vo[k] + visN[k][t] : 0.0);
    if (A.Wmlp) {
#pragma unroll
      for (int k = 0; k < 4; ++k) Wb[k] += A.Wmlp[k * A.plane + pc];
    }
    const double r = wc[0], u = wc[1], v = wc[2], p = wc[3], ri = rcp_(r);
    // u = ru / r, v = rv / r, p = g1 (E - (ru u + rv v) / 2)
    double out[4];
    out[3] = g1 * Wb[3];
    out[1] = Wb[1] * ri - g1 * u * Wb[3];
    out[2] = Wb[2] * ri - g1 * v * Wb[3];
    out[0] = Wb[0] - (Wb[1] * u + Wb[2] * v) * ri + 0.5 * g1 * (u * u + v * v) * Wb[3];
    gbar += Wb[3] * p * rcp_(g1);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double x = out[k];
      if (NS && A.nu != 0.0)  // L += nu Lap_h(U) (Eq. 10): the Laplacian is its own transpose
        x = fma(A.nu * A.dxi * A.dxi, LbS[k][t - 1] - 2.0 * LbS[k][t] + LbS[k][t + 1], x);
      if (interior) x = fma(A.b, Ub[k], x) + Ex[k];
      A.Ubar_in[k * A.plane + pc] = x;
    }
  }
  // gamma_bar of this CTA, fixed order
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) gbar += __shfl_xor_sync(0xffffffffu, gbar, o);
  if ((t & 31) == 0) red[t >> 5] = gbar;
  __syncthreads();
  if (t == 0) A.gbar_partial[blockIdx.x] = (red[0] + red[1]) + (red[2] + red[3]);
}

// After adjoint1d_kernel: (1) the ghost columns' adjoints go to the cells the boundary conditions copy them from
// (transposed ghost fill: periodic / transmissive copy, reflective copy with the normal momentum negated; an inflow
// ghost is a constant of U whose energy p/(gamma-1) + ... moves with gamma), (2) gamma_bar += the launch's partial
// sums, in a fixed order.  One CTA.
constexpr int A1D_FOLD_TB = 1024;
__global__ void __launch_bounds__(A1D_FOLD_TB) adjoint1d_fold_kernel(double* Ubar, long long plane, int nx, int xlo,
                                                                     int xhi, double p_inflow, double gamma,
                                                                     const double* partial, int nparts,
                                                                     double* gamma_bar) {
  __shared__ double red[A1D_FOLD_TB / 32];
  double a = 0.0;
  for (int i = threadIdx.x; i < nparts; i += A1D_FOLD_TB) a += partial[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = a;
  __syncthreads();
  // ghost columns: one thread per (side, component); its three ghost cells are read together, then added to their
  // source cells one after the other (all three may share one: a transmissive end)
  __shared__ double gin[8];
  if (threadIdx.x < 8) {
    const int side = threadIdx.x >> 2, k = threadIdx.x & 3;
    const double g1 = gamma - 1.0;
    double x[3], gi = 0.0;
    int idx[3];
#pragma unroll
    for (int g = 0; g < 3; ++g) {
      idx[g] = side == 0 ? g - 3 : nx + g;  // interior index of the ghost cell
      x[g] = Ubar[k * plane + idx[g] + 3];
      Ubar[k * plane + idx[g] + 3] = 0.0;
    }
#pragma unroll
    for (int g = 0; g < 3; ++g) {
      int src, sgn;
      bc_map(idx[g], nx, xlo, xhi, src, sgn);
      if (src < 0) { if (k == 3) gi -= x[g] * p_inflow / (g1 * g1); }
      else Ubar[k * plane + src + 3] += (k == 1 && sgn < 0) ? -x[g] : x[g];
    }
    gin[threadIdx.x] = gi;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double gb = 0.0;
    for (int w = 0; w < A1D_FOLD_TB / 32; ++w) gb += red[w];
    for (int w = 0; w < 8; ++w) gb += gin[w];
    *gamma_bar += gb;
  }
}

// The loss of PAPER.md Eq. 14 inside the reverse sweep: L = (1/m) sum_s mean((U^{n+s} - target_s)^2).  For one s:
// Ubar (+)= coef (U - target), coef = 2 / (m 4 nx), on the interior cells of the compact padded row, and
// loss_acc += sum (U - target)^2 (one fp64 atomic per CTA).  target: [4][nx] interior layout.
__global__ void __launch_bounds__(256) mse_inject_kernel(const double* __restrict__ Urow, long long plane,
                                                         const double* __restrict__ target, int nx, double coef,
                                                         double* Xrow, int accumulate, double* loss_acc) {
  __shared__ double red[8];
  double a = 0.0;
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < 4LL * nx; i += (long long)gridDim.x * 256) {
    const int k = (int)(i / nx), c = (int)(i - (long long)k * nx);
    const double r = Urow[k * plane + c + 3] - target[i];
    double* x = Xrow + k * plane + c + 3;
    *x = accumulate ? fma(coef, r, *x) : coef * r;
    a = fma(r, r, a);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red[w];
    atomicAdd(loss_acc, t);
  }
}

}  // namespace jxs
