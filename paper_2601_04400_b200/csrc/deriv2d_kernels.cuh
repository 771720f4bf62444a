// deriv2d_kernels.cuh — the derivatives of the TWO-dimensional stage (PAPER.md L115-128
// Eq. 15-16, L170 Fig. 5d-f: the inference of gamma on the shock-cylinder case; R21, R24, R25): forward mode
// (the stage on (value, derivative) pairs) and reverse mode (the transposed Jacobians applied from the left),
// including the immersed-boundary fill, walls, inflow and the viscous cross derivatives.  fp64.
//
// The right-hand side is a sum of operators on the primitives W(U):
//     L = Lx + Ly + Lv,   Lx / Ly: WENO5 + HLLC (+ the nu-term's second difference) along the rows / the columns,
//                         Lv: the viscous fluxes of both directions (R8), with their cross derivatives.
// Lx and Ly are one-dimensional operators applied to every line of the grid, so both modes run the LINE kernels below
// — the per-cell device routines of tangent1d_kernel.cuh / adjoint1d_kernel.cuh (weno5_dual, hllc_dual, weno5_adjoint,
// hllc_adjoint), one thread per cell of a line — on the rows of the state and, for Ly, on the rows of a TRANSPOSED copy
// of it with the two momenta exchanged (the y-flux is the x-flux with u and v interchanged), so that both
// passes read and write coalesced rows.  Lv is a nine-point operator on (u, v, T) and has kernels of its own: forward
// on pairs, and in reverse as a GATHER (every cell sums the adjoint coefficients of the 12 faces that touch it), so
// there are no atomics and the result is reproducible bit for bit.  The boundary conditions and the immersed-boundary
// fill are part of the differentiated map: their tangents are the linearised fills, their adjoints the transposed
// fills (ghost adjoints folded onto the cells they were copied from, in a fixed order).
#pragma once
#include "adjoint1d_kernel.cuh"
#include "aux_kernels.cuh"
#include "stage_kernel.cuh"
#include "tangent1d_kernel.cuh"

namespace jxs {

// A set of lines inside a padded SoA buffer [4][rows][pitch]: component k of padded position pc (0 .. n+5) of line l
// (l = 0 .. nlines-1) lies at k * plane + (l + 3) * pitch + pc.
struct LineSet {
  long long plane;
  int pitch;
  int n;       // interior cells along a line
  int nlines;  // interior lines
};

// ------------------------------------------------------------------ forward mode, one direction
struct TangentLineArgs {
  const double* U;      // padded, ghosts filled: the stage's input state ...
  const double* Udot;   // ... and its tangent (ghosts filled with the linearised boundary conditions)
  double* L;            // out: the directional part of L at interior cells, same layout (other cells untouched)
  double* Ldot;
  LineSet g;
  double gamma, gamma_dot, dhi, nu;  // dhi = 1 / spacing along the line
  int accumulate;                    // add to L / Ldot instead of overwriting
};

// tangent1d_kernel's sweep (S3-S5, S7 without the combine) on every line of the set; blockIdx.y = line
__global__ void __launch_bounds__(T1D_TB) tangent_line_kernel(const TangentLineArgs A) {
  __shared__ Dual prim[4][T1D_TB + 4];
  __shared__ Dual rmS[4][T1D_TB];
  __shared__ Dual fS[4][T1D_TB];
  const int t = threadIdx.x;
  const int c0 = T1D_OUT * blockIdx.x + 2;
  const int col = c0 + t;
  const size_t row = (size_t)(blockIdx.y + 3) * A.g.pitch;
  const int last = A.g.n + 5;
  const Dual gamma = dual(A.gamma, A.gamma_dot);
  const Dual g1 = gamma - 1.0, g1inv = rcp_dual(g1);

  auto to_prim = [&](int c, int slot) {
    const size_t o = row + (size_t)min(max(c, 0), last);
    Dual U[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) U[k] = dual(A.U[k * A.g.plane + o], A.Udot[k * A.g.plane + o]);
    const Dual ri = rcp_dual(U[0]);
    const Dual u = U[1] * ri, v = U[2] * ri;
    const Dual p = g1 * (U[3] - 0.5 * (U[1] * u + U[2] * v));
    prim[0][slot] = U[0]; prim[1][slot] = u; prim[2][slot] = v; prim[3][slot] = p;
  };
  to_prim(col, t + 2);
  if (t < 4) to_prim(t < 2 ? c0 - 2 + t : c0 + T1D_TB + (t - 2), t < 2 ? t : T1D_TB + t);
  __syncthreads();

  Dual wc[4], Lp[4];
  {
    Dual Rm[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      wc[k] = prim[k][t + 2];
      weno5_dual(prim[k][t], prim[k][t + 1], wc[k], prim[k][t + 3], prim[k][t + 4], Lp[k], Rm[k]);
    }
    const bool badR = !(Rm[0].v > 0.0) || !(Rm[3].v > 0.0);
    const bool badL = !(Lp[0].v > 0.0) || !(Lp[3].v > 0.0);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      rmS[k][t] = badR ? wc[k] : Rm[k];
      if (badL) Lp[k] = wc[k];
    }
  }
  __syncthreads();
  Dual F[4];
  {
    const int tn = min(t + 1, T1D_TB - 1);
    const Dual R[4] = {rmS[0][tn], rmS[1][tn], rmS[2][tn], rmS[3][tn]};
    hllc_dual(Lp, R, gamma, g1inv, F);
#pragma unroll
    for (int k = 0; k < 4; ++k) fS[k][t] = F[k];
  }
  __syncthreads();
  const int ic = col - 3;
  const bool ok = t >= 1 && t <= T1D_OUT && ic < A.g.n;
  if (!ok) return;
  Dual Lc[4];
  const int tl = t - 1;
#pragma unroll
  for (int k = 0; k < 4; ++k) Lc[k] = A.dhi * (fS[k][tl] - F[k]);
  if (A.nu != 0.0) {
    auto cons = [&](int c, Dual* U) {
      const Dual r = prim[0][c], u = prim[1][c], v = prim[2][c], p = prim[3][c];
      U[0] = r; U[1] = r * u; U[2] = r * v; U[3] = p * g1inv + 0.5 * (r * (u * u + v * v));
    };
    Dual Um[4], Uxm[4], Uxp[4];
    cons(t + 2, Um); cons(t + 1, Uxm); cons(t + 3, Uxp);
    const double ax = A.nu * A.dhi * A.dhi;
#pragma unroll
    for (int k = 0; k < 4; ++k) Lc[k] = Lc[k] + ax * (Uxp[k] - 2.0 * Um[k] + Uxm[k]);
  }
  const size_t o = row + col;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (A.accumulate) {
      A.L[k * A.g.plane + o] += Lc[k].v;
      A.Ldot[k * A.g.plane + o] += Lc[k].d;
    } else {
      A.L[k * A.g.plane + o] = Lc[k].v;
      A.Ldot[k * A.g.plane + o] = Lc[k].d;
    }
  }
}

// ------------------------------------------------------------------ transposes between the two layouts
// natural: [4][ny+6][pitch] (x fastest);  transposed: [4][nx+6][pitch_t] (y fastest) with the momenta exchanged, so
// that a column of the grid is a line whose normal velocity sits in component 1.  32 x 32 tiles through shared memory.
struct TransposeArgs {
  const double* src;
  double* dst;
  long long plane_s, plane_d;
  int pitch_s, pitch_d;
  int r_lo, r_hi, c_lo, c_hi;  // the region of src that moves: rows [r_lo, r_hi) x columns [c_lo, c_hi)
  int accumulate;              // dst += instead of dst =
};
__global__ void __launch_bounds__(256) transpose_swap_kernel(const TransposeArgs A) {
  __shared__ double tile[32][33];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
  const int c0 = A.c_lo + blockIdx.x * 32, r0 = A.r_lo + blockIdx.y * 32;
  const int k = blockIdx.z, kd = k == 1 ? 2 : (k == 2 ? 1 : k);
  for (int r = ty; r < 32; r += 8) {
    const int rr = r0 + r, cc = c0 + tx;
    tile[r][tx] = (rr < A.r_hi && cc < A.c_hi) ? A.src[k * A.plane_s + (long long)rr * A.pitch_s + cc] : 0.0;
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int rd = c0 + r, cd = r0 + tx;  // dst row = src column, dst column = src row
    if (rd < A.c_hi && cd < A.r_hi) {
      double* p = A.dst + kd * A.plane_d + (long long)rd * A.pitch_d + cd;
      *p = A.accumulate ? *p + tile[tx][r] : tile[tx][r];
    }
  }
}

// ------------------------------------------------------------------ Lv, forward mode
// The viscous fluxes of both directions on pairs (oracle O6 / R8, term by term) and their divergence, ADDED to L, Ldot
// at interior cells.  One thread per cell of a 32 x 8 tile; (u, v, T) of the tile and a one-cell halo in shared memory.
struct Visc2dArgs {
  const double* U;
  const double* Udot;
  double* L;
  double* Ldot;
  long long plane;
  int nx, ny, pitch;
  double gamma, gamma_dot, mu, Pr, dxi, dyi;
};
constexpr int V2_TX = 32, V2_TY = 8;
__global__ void __launch_bounds__(V2_TX * V2_TY) viscous2d_tangent_kernel(const Visc2dArgs A) {
  __shared__ Dual W[3][V2_TY + 2][V2_TX + 2];  // u, v, T
  const int tx = threadIdx.x % V2_TX, ty = threadIdx.x / V2_TX;
  const int i0 = blockIdx.x * V2_TX, j0 = blockIdx.y * V2_TY;  // interior index of the tile's first cell
  const Dual gamma = dual(A.gamma, A.gamma_dot), g1 = gamma - 1.0;
  for (int s = threadIdx.x; s < (V2_TX + 2) * (V2_TY + 2); s += V2_TX * V2_TY) {
    const int lx = s % (V2_TX + 2), ly = s / (V2_TX + 2);
    const int ip = min(i0 + lx - 1, A.nx) + 3, jp = min(j0 + ly - 1, A.ny) + 3;  // padded, clamped to the first ghost layer
    const size_t o = (size_t)jp * A.pitch + ip;
    Dual U[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) U[k] = dual(A.U[k * A.plane + o], A.Udot[k * A.plane + o]);
    const Dual ri = rcp_dual(U[0]);
    const Dual u = U[1] * ri, v = U[2] * ri;
    const Dual p = g1 * (U[3] - 0.5 * (U[1] * u + U[2] * v));
    W[0][ly][lx] = u; W[1][ly][lx] = v; W[2][ly][lx] = p * ri;
  }
  __syncthreads();
  const int i = i0 + tx, j = j0 + ty;
  if (i >= A.nx || j >= A.ny) return;
  const Dual kap = (A.mu / A.Pr) * (gamma * rcp_dual(g1));
  const int cx = tx + 1, cy = ty + 1;
  auto u = [&](int dx, int dy) { return W[0][cy + dy][cx + dx]; };
  auto v = [&](int dx, int dy) { return W[1][cy + dy][cx + dx]; };
  auto T = [&](int dx, int dy) { return W[2][cy + dy][cx + dx]; };
  // x-face between (i + s - 1, j) and (i + s, j), s = 0 (my left face), 1 (my right face)
  Dual Fv[2][3], Gv[2][3];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int a = s - 1, b = s;  // the two cells' x offsets
    const Dual ux = A.dxi * (u(b, 0) - u(a, 0)), vx = A.dxi * (v(b, 0) - v(a, 0)), Tx = A.dxi * (T(b, 0) - T(a, 0));
    const Dual uy = (0.25 * A.dyi) * ((u(a, 1) - u(a, -1)) + (u(b, 1) - u(b, -1)));
    const Dual vy = (0.25 * A.dyi) * ((v(a, 1) - v(a, -1)) + (v(b, 1) - v(b, -1)));
    const Dual ub = 0.5 * (u(a, 0) + u(b, 0)), vb = 0.5 * (v(a, 0) + v(b, 0));
    const Dual txx = A.mu * ((4.0 / 3.0) * ux - (2.0 / 3.0) * vy), txy = A.mu * (uy + vx);
    Fv[s][0] = txx; Fv[s][1] = txy; Fv[s][2] = ub * txx + vb * txy + kap * Tx;
  }
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int a = s - 1, b = s;  // the two cells' y offsets
    const Dual uy = A.dyi * (u(0, b) - u(0, a)), vy = A.dyi * (v(0, b) - v(0, a)), Ty = A.dyi * (T(0, b) - T(0, a));
    const Dual ux = (0.25 * A.dxi) * ((u(1, a) - u(-1, a)) + (u(1, b) - u(-1, b)));
    const Dual vx = (0.25 * A.dxi) * ((v(1, a) - v(-1, a)) + (v(1, b) - v(-1, b)));
    const Dual ub = 0.5 * (u(0, a) + u(0, b)), vb = 0.5 * (v(0, a) + v(0, b));
    const Dual tyy = A.mu * ((4.0 / 3.0) * vy - (2.0 / 3.0) * ux), txy = A.mu * (uy + vx);
    Gv[s][0] = txy; Gv[s][1] = tyy; Gv[s][2] = ub * txy + vb * tyy + kap * Ty;
  }
  const size_t o = (size_t)(j + 3) * A.pitch + i + 3;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const Dual d = A.dxi * (Fv[1][k] - Fv[0][k]) + A.dyi * (Gv[1][k] - Gv[0][k]);
    A.L[(k + 1) * A.plane + o] += d.v;
    A.Ldot[(k + 1) * A.plane + o] += d.d;
  }
}

// ------------------------------------------------------------------ forward mode: the Runge-Kutta combine on pairs
// Uout = a U0 + b (U + dt fl L) at interior cells (fl = 0 at non-fluid cells: they keep their state, S7)
struct Combine2dArgs {
  const double *U, *Udot, *U0, *U0dot, *L, *Ldot;
  double *Uout, *Uoutdot;
  const uint8_t* fluid;
  const double* dt;
  long long plane;
  int nx, ny, pitch;
  double a, b;
};
__global__ void __launch_bounds__(256) combine2d_tangent_kernel(const Combine2dArgs A) {
  const long long n = (long long)A.nx * A.ny;
  const double dt = *A.dt;
  for (long long t = blockIdx.x * 256LL + threadIdx.x; t < n; t += (long long)gridDim.x * 256) {
    const int j = (int)(t / A.nx), i = (int)(t - (long long)j * A.nx);
    const size_t o = (size_t)(j + 3) * A.pitch + i + 3;
    const double dtf = (!A.fluid || A.fluid[t]) ? dt : 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double x = fma(dtf, A.L[k * A.plane + o], A.U[k * A.plane + o]);
      double xd = fma(dtf, A.Ldot[k * A.plane + o], A.Udot[k * A.plane + o]);
      if (A.a != 0.0) {
        x = fma(A.a, A.U0[k * A.plane + o], A.b * x);
        xd = fma(A.a, A.U0dot[k * A.plane + o], A.b * xd);
      }
      A.Uout[k * A.plane + o] = x;
      A.Uoutdot[k * A.plane + o] = xd;
    }
  }
}

// ------------------------------------------------------------------ the immersed-boundary fill on pairs (R9 I6)
// one thread per ghost cell: the fill of ghost_fill_kernel written on (value, derivative); writes the TANGENT of the
// ghost state only (the value was written by ghost_fill_kernel)
__device__ __forceinline__ void ibm_fill_dual(const Dual (&Ud)[4][4], const double (&w)[4], double nx_, double ny_,
                                              Dual gamma, Dual (&out)[4]) {
  const Dual g1 = gamma - 1.0;
  Dual WI[4] = {dual(0.0), dual(0.0), dual(0.0), dual(0.0)};
#pragma unroll
  for (int d = 0; d < 4; ++d) {
    if (w[d] == 0.0) continue;
    const Dual ri = rcp_dual(Ud[d][0]);
    const Dual u = Ud[d][1] * ri, v = Ud[d][2] * ri;
    const Dual p = g1 * (Ud[d][3] - 0.5 * (Ud[d][0] * (u * u + v * v)));
    WI[0] = WI[0] + w[d] * Ud[d][0]; WI[1] = WI[1] + w[d] * u; WI[2] = WI[2] + w[d] * v; WI[3] = WI[3] + w[d] * p;
  }
  const Dual un = nx_ * WI[1] + ny_ * WI[2];
  const Dual r = WI[0], u = WI[1] - (2.0 * nx_) * un, v = WI[2] - (2.0 * ny_) * un, p = WI[3];
  out[0] = r; out[1] = r * u; out[2] = r * v; out[3] = p * rcp_dual(g1) + 0.5 * (r * (u * u + v * v));
}
__global__ void __launch_bounds__(128) ibm_fill_tangent_kernel(const double* __restrict__ U, double* __restrict__ Udot,
                                                               long long plane, IbmList ibm, double gamma, double gamma_dot) {
  const int q = blockIdx.x * 128 + threadIdx.x;
  if (q >= ibm.n) return;
  Dual Ud[4][4];
  double w[4];
#pragma unroll
  for (int d = 0; d < 4; ++d) {
    w[d] = ibm.w[4 * q + d];
    const long long o = ibm.donor[4 * q + d];
#pragma unroll
    for (int k = 0; k < 4; ++k) Ud[d][k] = dual(U[k * plane + o], Udot[k * plane + o]);
  }
  Dual out[4];
  ibm_fill_dual(Ud, w, ibm.nrm[2 * q], ibm.nrm[2 * q + 1], dual(gamma, gamma_dot), out);
  const long long o = ibm.cell[q];
#pragma unroll
  for (int k = 0; k < 4; ++k) Udot[k * plane + o] = out[k].d;
}

// ------------------------------------------------------------------ reverse mode, one direction
struct AdjointLineArgs {
  const double* U;         // padded, ghosts filled: the stage's input state (natural or transposed layout)
  const double* Ubar_out;  // adjoint of the stage's result, same layout, zero outside the interior
  double* Ubar_in;         // out: this direction's part of the adjoint of the stage's input, ghost positions of the lines included
  const double* E1;        // with identity: Ubar_in += e1 E1 + e2 E2 on interior cells
  const double* E2;
  const uint8_t* fluid;    // [nlines][n] in the layout's own orientation, 1 = fluid; nullptr = all fluid
  double* gbar_partial;    // [gridDim.y * gridDim.x] contributions to gamma_bar
  LineSet g;
  double dt, gamma, dhi, b, e1, e2, nu;
  int identity;            // 1: Ubar_in = b Ubar_out + (this direction) + E terms; 0: this direction only
};

// adjoint1d_kernel's reverse sweep on every line of the set (blockIdx.y = line), without the 1D viscous flux
__global__ void __launch_bounds__(A1D_TB) adjoint_line_kernel(const AdjointLineArgs A) {
  __shared__ double prim[4][A1D_TB + 4];
  __shared__ double rmS[4][A1D_TB];
  __shared__ double LbS[4][A1D_TB];
  __shared__ double rmB[4][A1D_TB + 1];
  __shared__ double con[4][5][A1D_TB];
  __shared__ double red[A1D_TB / 32];
  const int t = threadIdx.x;
  const int pc0 = A1D_OUT * blockIdx.x - 3;
  const int pc = pc0 + t;
  const int last = A.g.n + 5;
  const size_t row = (size_t)(blockIdx.y + 3) * A.g.pitch;
  const double g1 = A.gamma - 1.0;
  const double bdt = A.b * A.dt;
  const bool interior = pc >= 3 && pc <= A.g.n + 2;

  auto to_prim = [&](int c, int slot) {
    const size_t o = row + (size_t)min(max(c, 0), last);
    const double r = A.U[o], ru = A.U[A.g.plane + o], rv = A.U[2 * A.g.plane + o], E = A.U[3 * A.g.plane + o];
    const double ri = rcp_(r), u = ru * ri, v = rv * ri;
    prim[0][slot] = r; prim[1][slot] = u; prim[2][slot] = v; prim[3][slot] = g1 * (E - 0.5 * (ru * u + rv * v));
  };
  to_prim(pc, t + 2);
  if (t < 4) to_prim(t < 2 ? pc0 - 2 + t : pc0 + A1D_TB + (t - 2), t < 2 ? t : A1D_TB + t);
  double Ub[4] = {0.0, 0.0, 0.0, 0.0};
  bool fl = false;
  if (interior) {
#pragma unroll
    for (int k = 0; k < 4; ++k) Ub[k] = A.Ubar_out[k * A.g.plane + row + pc];
    fl = !A.fluid || A.fluid[(size_t)blockIdx.y * A.g.n + (pc - 3)];
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) LbS[k][t] = fl ? bdt * Ub[k] : 0.0;  // L = 0 at non-fluid cells (S7)
  if (t == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) rmB[k][0] = 0.0;
  }
  __syncthreads();

  const bool stencil = pc >= 2 && pc <= A.g.n + 3;
  double wc[4], Lp[4], Rm[4];
  bool badL = false, badR = false;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    wc[k] = prim[k][t + 2];
    Lp[k] = Rm[k] = wc[k];
    double Di = 0.0, Ei = 0.0;
    if (stencil) weno5_val(prim[k][t], prim[k][t + 1], wc[k], prim[k][t + 3], prim[k][t + 4], Lp[k], Rm[k], Di, Ei);
    con[k][0][t] = Di;
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

  const bool face = pc >= 2 && pc <= A.g.n + 2 && t < A1D_TB - 1;
  const bool mine = t >= 3 && t <= A1D_TB - 4 && pc <= last;
  double Lpb[4] = {0.0, 0.0, 0.0, 0.0}, gbar = 0.0;
  {
    double Rnb[4] = {0.0, 0.0, 0.0, 0.0};
    if (face) {
      double f[4], R[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { f[k] = A.dhi * (LbS[k][t + 1] - LbS[k][t]); R[k] = rmS[k][t + 1]; }
      const double gb = hllc_adjoint(Lp, R, A.gamma, f, Lpb, Rnb);
      if (mine) gbar += gb;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) rmB[k][t + 1] = Rnb[k];
  }
  __syncthreads();

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
  double Ex[4] = {0.0, 0.0, 0.0, 0.0};
  if (A.identity && interior && mine) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (A.E1) Ex[k] = A.e1 * A.E1[k * A.g.plane + row + pc];
      if (A.E2) Ex[k] = fma(A.e2, A.E2[k * A.g.plane + row + pc], Ex[k]);
    }
  }
  __syncthreads();

  if (mine) {
    double Wb[4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
      Wb[k] = con[k][0][t + 2] + con[k][1][t + 1] + con[k][2][t] + con[k][3][t - 1] + con[k][4][t - 2];
    const double r = wc[0], u = wc[1], v = wc[2], p = wc[3], ri = rcp_(r);
    double out[4];
    out[3] = g1 * Wb[3];
    out[1] = Wb[1] * ri - g1 * u * Wb[3];
    out[2] = Wb[2] * ri - g1 * v * Wb[3];
    out[0] = Wb[0] - (Wb[1] * u + Wb[2] * v) * ri + 0.5 * g1 * (u * u + v * v) * Wb[3];
    gbar += Wb[3] * p * rcp_(g1);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double x = out[k];
      if (A.nu != 0.0) x = fma(A.nu * A.dhi * A.dhi, LbS[k][t - 1] - 2.0 * LbS[k][t] + LbS[k][t + 1], x);
      if (A.identity && interior) x = fma(A.b, Ub[k], x) + Ex[k];
      A.Ubar_in[k * A.g.plane + row + pc] = x;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) gbar += __shfl_xor_sync(0xffffffffu, gbar, o);
  if ((t & 31) == 0) red[t >> 5] = gbar;
  __syncthreads();
  if (t == 0) A.gbar_partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = (red[0] + red[1]) + (red[2] + red[3]);
}

// ------------------------------------------------------------------ Lv, reverse mode
// Pass 1, one thread per face: the adjoint coefficients of the face's viscous flux.  With phi = the flux adjoint
// (differences of b dt Ubar_out at the two cells, fluid cells only) of an x-face between cells a = (i, j), b = (i+1, j):
//   txx_bar = phi1 + phi3 ub,  txy_bar = phi2 + phi3 vb,  ub_bar = phi3 txx,  vb_bar = phi3 txy,  Tx_bar = phi3 kappa
//   ux_bar = 4/3 mu txx_bar,  vy_bar = -2/3 mu txx_bar,  uy_bar = vx_bar = mu txy_bar
// and the seven numbers kept per face are what the six cells of its stencil receive:
//   [0] u: normal difference (+ at b, - at a)    ux_bar / h_n          [1] u: average (both cells)   ub_bar / 2
//   [2] u: tangential differences (+ at j+1, - at j-1, both columns)   uy_bar / (4 h_t)
//   [3], [4], [5] the same for v (vx_bar, vb_bar, vy_bar);             [6] T: normal difference      Tx_bar / h_n
// y-faces likewise with the roles of the axes exchanged.  gamma enters through kappa: gamma_bar partial sums per CTA.
struct Visc2dAdjArgs {
  const double* U;         // padded, ghosts filled
  const double* Ubar_out;  // padded
  const uint8_t* fluid;    // [ny][nx] or nullptr
  double* Cx;              // [7][ny][nx+1]: x-face f of row j between cells f-1 and f
  double* Cy;              // [7][ny+1][nx]
  double* Ubar_in;         // padded: += the viscous part (pass 2)
  double* gbar_partial;
  long long plane;
  int nx, ny, pitch;
  double gamma, mu, Pr, dxi, dyi, bdt;
};
__device__ __forceinline__ void visc_prim(const double* U, long long plane, size_t o, double g1, double& u, double& v,
                                          double& T, double& r) {
  r = U[o];
  const double ri = rcp_(r), ru = U[plane + o], rv = U[2 * plane + o], E = U[3 * plane + o];
  u = ru * ri; v = rv * ri;
  T = g1 * (E - 0.5 * (ru * u + rv * v)) * ri;
}
__global__ void __launch_bounds__(256) viscous2d_adjoint_faces_kernel(const Visc2dAdjArgs A) {
  __shared__ double red[8];
  const long long nfx = (long long)A.ny * (A.nx + 1), nfy = (long long)(A.ny + 1) * A.nx;
  const double g1 = A.gamma - 1.0, kap = A.mu / A.Pr * A.gamma / g1;
  double gbar = 0.0;
  for (long long t = blockIdx.x * 256LL + threadIdx.x; t < nfx + nfy; t += (long long)gridDim.x * 256) {
    const bool xf = t < nfx;
    int i, j;  // the lower / left cell of the face (interior index, may be -1)
    if (xf) { j = (int)(t / (A.nx + 1)); i = (int)(t - (long long)j * (A.nx + 1)) - 1; }
    else { const long long s = t - nfx; j = (int)(s / A.nx) - 1; i = (int)(s - (long long)(j + 1) * A.nx); }
    const int di = xf ? 1 : 0, dj = xf ? 0 : 1;
    const size_t oa = (size_t)(j + 3) * A.pitch + i + 3, ob = oa + (size_t)dj * A.pitch + di;
    // flux adjoint: L_a += h (Fv_face), L_b -= h (Fv_face) (L = ... + dFv/dx), fluid cells only
    auto Lbar = [&](int ii, int jj, size_t o, int k) -> double {
      if (ii < 0 || ii >= A.nx || jj < 0 || jj >= A.ny) return 0.0;
      if (A.fluid && !A.fluid[(size_t)jj * A.nx + ii]) return 0.0;
      return A.bdt * A.Ubar_out[k * A.plane + o];
    };
    const double hn = xf ? A.dxi : A.dyi, ht = xf ? A.dyi : A.dxi;
    double phi[4];
#pragma unroll
    for (int k = 1; k < 4; ++k) phi[k] = hn * (Lbar(i, j, oa, k) - Lbar(i + di, j + dj, ob, k));
    double ua, va, Ta, ra, ub_, vb_, Tb, rb;
    visc_prim(A.U, A.plane, oa, g1, ua, va, Ta, ra);
    visc_prim(A.U, A.plane, ob, g1, ub_, vb_, Tb, rb);
    // tangential differences of u and v across the face's two cells
    const size_t st = xf ? (size_t)A.pitch : 1;  // one step along the tangential axis
    double ut = 0.0, vt = 0.0;
    {
      double u1, v1, T1, r1, u2, v2, T2, r2;
      visc_prim(A.U, A.plane, oa + st, g1, u1, v1, T1, r1); visc_prim(A.U, A.plane, oa - st, g1, u2, v2, T2, r2);
      ut += u1 - u2; vt += v1 - v2;
      visc_prim(A.U, A.plane, ob + st, g1, u1, v1, T1, r1); visc_prim(A.U, A.plane, ob - st, g1, u2, v2, T2, r2);
      ut += u1 - u2; vt += v1 - v2;
    }
    ut *= 0.25 * ht; vt *= 0.25 * ht;
    const double un_ = hn * (ub_ - ua), vn_ = hn * (vb_ - va), Tn_ = hn * (Tb - Ta);
    const double uavg = 0.5 * (ua + ub_), vavg = 0.5 * (va + vb_);
    double c[7];
    if (xf) {  // Fv = (0, txx, txy, ub txx + vb txy + kap Tx), txx = mu (4/3 ux - 2/3 vy), txy = mu (uy + vx)
      const double txx = A.mu * (4.0 / 3.0 * un_ - 2.0 / 3.0 * vt), txy = A.mu * (ut + vn_);
      const double txxb = phi[1] + phi[3] * uavg, txyb = phi[2] + phi[3] * vavg;
      c[0] = (4.0 / 3.0) * A.mu * txxb * hn; c[1] = 0.5 * phi[3] * txx; c[2] = A.mu * txyb * 0.25 * ht;
      c[3] = A.mu * txyb * hn; c[4] = 0.5 * phi[3] * txy; c[5] = -(2.0 / 3.0) * A.mu * txxb * 0.25 * ht;
      c[6] = phi[3] * kap * hn;
      gbar += phi[3] * Tn_ * (-(A.mu / A.Pr) / (g1 * g1));  // d kappa / d gamma = -mu / (Pr (gamma-1)^2)
    } else {   // Gv = (0, txy, tyy, ub txy + vb tyy + kap Ty), tyy = mu (4/3 vy - 2/3 ux), txy = mu (uy + vx)
      const double tyy = A.mu * (4.0 / 3.0 * vn_ - 2.0 / 3.0 * ut), txy = A.mu * (un_ + vt);
      const double txyb = phi[1] + phi[3] * uavg, tyyb = phi[2] + phi[3] * vavg;
      c[0] = A.mu * txyb * hn; c[1] = 0.5 * phi[3] * txy; c[2] = -(2.0 / 3.0) * A.mu * tyyb * 0.25 * ht;
      c[3] = (4.0 / 3.0) * A.mu * tyyb * hn; c[4] = 0.5 * phi[3] * tyy; c[5] = A.mu * txyb * 0.25 * ht;
      c[6] = phi[3] * kap * hn;
      gbar += phi[3] * Tn_ * (-(A.mu / A.Pr) / (g1 * g1));
    }
    double* C = xf ? A.Cx : A.Cy;
    const long long nf = xf ? nfx : nfy, f = xf ? t : t - nfx;
#pragma unroll
    for (int q = 0; q < 7; ++q) C[q * nf + f] = c[q];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) gbar += __shfl_xor_sync(0xffffffffu, gbar, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = gbar;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < 8; ++w) s += red[w];
    A.gbar_partial[blockIdx.x] = s;
  }
}
// Pass 2, one thread per cell of [-1, nx] x [-1, ny]: gather the coefficients of the faces whose stencils hold the
// cell (fixed order), convert the adjoint of (u, v, T) to that of the conserved variables, add to Ubar_in.
__global__ void __launch_bounds__(256) viscous2d_adjoint_gather_kernel(const Visc2dAdjArgs A) {
  const int nxe = A.nx + 2, nye = A.ny + 2;
  const long long n = (long long)nxe * nye;
  const long long nfx = (long long)A.ny * (A.nx + 1), nfy = (long long)(A.ny + 1) * A.nx;
  const double g1 = A.gamma - 1.0;
  for (long long t = blockIdx.x * 256LL + threadIdx.x; t < n; t += (long long)gridDim.x * 256) {
    const int j = (int)(t / nxe) - 1, i = (int)(t - (long long)(j + 1) * nxe) - 1;
    // x-face f (between cells f-1 and f) of row jj exists for 0 <= f <= nx, 0 <= jj < ny
    auto cx = [&](int q, int f, int jj) -> double {
      return (f < 0 || f > A.nx || jj < 0 || jj >= A.ny) ? 0.0 : A.Cx[q * nfx + (long long)jj * (A.nx + 1) + f];
    };
    // y-face f (between rows f-1 and f) of column ii exists for 0 <= f <= ny, 0 <= ii < nx
    auto cy = [&](int q, int ii, int f) -> double {
      return (f < 0 || f > A.ny || ii < 0 || ii >= A.nx) ? 0.0 : A.Cy[q * nfy + (long long)f * A.nx + ii];
    };
    // my right x-face is f = i+1 (I am its cell a), my left x-face f = i (I am its cell b)
    double ub = (cx(0, i, j) - cx(0, i + 1, j)) + (cx(1, i, j) + cx(1, i + 1, j)) +
                ((cx(2, i, j - 1) + cx(2, i + 1, j - 1)) - (cx(2, i, j + 1) + cx(2, i + 1, j + 1)));
    double vb = (cx(3, i, j) - cx(3, i + 1, j)) + (cx(4, i, j) + cx(4, i + 1, j)) +
                ((cx(5, i, j - 1) + cx(5, i + 1, j - 1)) - (cx(5, i, j + 1) + cx(5, i + 1, j + 1)));
    double Tb = cx(6, i, j) - cx(6, i + 1, j);
    // my top y-face is f = j+1 (cell a), my bottom y-face f = j (cell b); tangential axis = x
    ub += (cy(0, i, j) - cy(0, i, j + 1)) + (cy(1, i, j) + cy(1, i, j + 1)) +
          ((cy(2, i - 1, j) + cy(2, i - 1, j + 1)) - (cy(2, i + 1, j) + cy(2, i + 1, j + 1)));
    vb += (cy(3, i, j) - cy(3, i, j + 1)) + (cy(4, i, j) + cy(4, i, j + 1)) +
          ((cy(5, i - 1, j) + cy(5, i - 1, j + 1)) - (cy(5, i + 1, j) + cy(5, i + 1, j + 1)));
    Tb += cy(6, i, j) - cy(6, i, j + 1);
    const size_t o = (size_t)(j + 3) * A.pitch + i + 3;
    double u, v, T, r;
    visc_prim(A.U, A.plane, o, g1, u, v, T, r);
    const double ri = rcp_(r);
    // T = p / rho: p_bar = T_bar / rho, rho_bar = -T_bar T / rho; then (u, v, p) -> conserved as in the line kernel
    const double pb = Tb * ri, rb0 = -Tb * T * ri;
    double out[4];
    out[3] = g1 * pb;
    out[1] = ub * ri - g1 * u * pb;
    out[2] = vb * ri - g1 * v * pb;
    out[0] = rb0 - (ub * u + vb * v) * ri + 0.5 * g1 * (u * u + v * v) * pb;
#pragma unroll
    for (int k = 0; k < 4; ++k) A.Ubar_in[k * A.plane + o] += out[k];
  }
}
// (the pressure's own dependence on gamma inside T: p = (gamma-1)(E - ...) gives gamma_bar += p_bar p / (gamma-1))
__global__ void __launch_bounds__(256) viscous2d_adjoint_gamma_kernel(const Visc2dAdjArgs A, double* partial) {
  __shared__ double red[8];
  const int nxe = A.nx + 2, nye = A.ny + 2;
  const long long n = (long long)nxe * nye;
  const long long nfx = (long long)A.ny * (A.nx + 1), nfy = (long long)(A.ny + 1) * A.nx;
  const double g1 = A.gamma - 1.0;
  double gbar = 0.0;
  for (long long t = blockIdx.x * 256LL + threadIdx.x; t < n; t += (long long)gridDim.x * 256) {
    const int j = (int)(t / nxe) - 1, i = (int)(t - (long long)(j + 1) * nxe) - 1;
    auto cx = [&](int f, int jj) -> double {
      return (f < 0 || f > A.nx || jj < 0 || jj >= A.ny) ? 0.0 : A.Cx[6 * nfx + (long long)jj * (A.nx + 1) + f];
    };
    auto cy = [&](int ii, int f) -> double {
      return (f < 0 || f > A.ny || ii < 0 || ii >= A.nx) ? 0.0 : A.Cy[6 * nfy + (long long)f * A.nx + ii];
    };
    const double Tb = (cx(i, j) - cx(i + 1, j)) + (cy(i, j) - cy(i, j + 1));
    const size_t o = (size_t)(j + 3) * A.pitch + i + 3;
    double u, v, T, r;
    visc_prim(A.U, A.plane, o, g1, u, v, T, r);
    gbar += Tb * T / g1;  // p_bar p / g1 = (T_bar / rho) (T rho) / g1
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) gbar += __shfl_xor_sync(0xffffffffu, gbar, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = gbar;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < 8; ++w) s += red[w];
    partial[blockIdx.x] = s;
  }
}

// ------------------------------------------------------------------ the transposed fills
// Immersed boundary, pass 1 (one thread per ghost cell): columns of the fill's Jacobian by forward mode (one pair run
// per donor entry and one for gamma, a few dozen flops each), paired with the ghost cell's adjoint:
//   contrib[q][d][k] = <dU_G / dU_{donor d, component k}, Ubar_G>,   gcontrib[q] = <dU_G / dgamma, Ubar_G>
// and the ghost cell's own adjoint is cleared (its value before the fill has no influence on anything).
__global__ void __launch_bounds__(128) ibm_adjoint_ghost_kernel(const double* __restrict__ U, double* __restrict__ Ubar,
                                                                long long plane, IbmList ibm, double gamma,
                                                                double* __restrict__ contrib, double* __restrict__ gcontrib) {
  const int q = blockIdx.x * 128 + threadIdx.x;
  if (q >= ibm.n) return;
  double w[4], Uv[4][4], Gb[4];
  const long long og = ibm.cell[q];
#pragma unroll
  for (int k = 0; k < 4; ++k) { Gb[k] = Ubar[k * plane + og]; Ubar[k * plane + og] = 0.0; }
#pragma unroll
  for (int d = 0; d < 4; ++d) {
    w[d] = ibm.w[4 * q + d];
    const long long o = ibm.donor[4 * q + d];
#pragma unroll
    for (int k = 0; k < 4; ++k) Uv[d][k] = U[k * plane + o];
  }
  const double nx_ = ibm.nrm[2 * q], ny_ = ibm.nrm[2 * q + 1];
  for (int col = 0; col < 17; ++col) {  // 16 donor entries, then gamma
    Dual Ud[4][4];
#pragma unroll
    for (int d = 0; d < 4; ++d)
#pragma unroll
      for (int k = 0; k < 4; ++k) Ud[d][k] = dual(Uv[d][k], (col < 16 && col == 4 * d + k) ? 1.0 : 0.0);
    Dual out[4];
    double val = 0.0;
    if (col == 16 || w[col >> 2] != 0.0) {
      ibm_fill_dual(Ud, w, nx_, ny_, dual(gamma, col == 16 ? 1.0 : 0.0), out);
      val = (out[0].d * Gb[0] + out[1].d * Gb[1]) + (out[2].d * Gb[2] + out[3].d * Gb[3]);
    }
    if (col < 16) contrib[(size_t)q * 16 + col] = val;
    else gcontrib[q] = val;
  }
}
// pass 2 (one thread per donor cell): sum the contributions of the ghost cells it feeds, in list order.
// rows[c] .. rows[c+1]: entries of donor c; entry = 16 q + 4 d (the four components follow each other)
__global__ void __launch_bounds__(128) ibm_adjoint_donor_kernel(double* __restrict__ Ubar, long long plane,
                                                                const int* __restrict__ dcell, const int* __restrict__ rows,
                                                                const int* __restrict__ entry, int ndonor,
                                                                const double* __restrict__ contrib) {
  const int c = blockIdx.x * 128 + threadIdx.x;
  if (c >= ndonor) return;
  double s[4] = {0.0, 0.0, 0.0, 0.0};
  for (int e = rows[c]; e < rows[c + 1]; ++e) {
    const int base = entry[e];
#pragma unroll
    for (int k = 0; k < 4; ++k) s[k] += contrib[base + k];
  }
  const long long o = dcell[c];
#pragma unroll
  for (int k = 0; k < 4; ++k) Ubar[k * plane + o] += s[k];
}

// Domain frame: the transposed ghost fill.  The fill runs x sides (interior rows) and then y sides over the
// x-extended range (R11), so its transpose folds the ghost ROWS first (axis = 1: one thread per padded column and
// side) and then the ghost COLUMNS of the interior rows (axis = 0: one thread per interior row and side).  A thread
// reads its three ghost cells, clears them and adds them to their source cells one after the other (a transmissive
// side maps all three onto one cell).  Inflow ghosts are constants of U whose energy moves with gamma.
__global__ void __launch_bounds__(128) frame_fold_kernel(double* __restrict__ Ubar, GridDims g, BcSpec bc, int axis,
                                                         double p_inflow, double gamma, double* __restrict__ gpartial) {
  const int nline = axis == 1 ? g.nx + 6 : g.ny;
  const int t = blockIdx.x * 128 + threadIdx.x;
  double gi = 0.0;
  if (t < 2 * nline) {
    const int side = t / nline, l = t % nline;
    const int n = axis == 1 ? g.ny : g.nx;
    const int lo = axis == 1 ? bc.ylo : bc.xlo, hi = axis == 1 ? bc.yhi : bc.xhi;
    const double g1 = gamma - 1.0;
    auto off = [&](int pos) -> long long {  // padded offset of interior position `pos` along the axis on my line
      return axis == 1 ? (long long)(pos + 3) * g.pitch + l : (long long)(l + 3) * g.pitch + pos + 3;
    };
    for (int k = 0; k < 4; ++k) {
      double x[3];
      int idx[3];
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        idx[q] = side == 0 ? q - 3 : n + q;
        x[q] = Ubar[k * g.plane + off(idx[q])];
        Ubar[k * g.plane + off(idx[q])] = 0.0;
      }
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        int src, sgn;
        bc_map(idx[q], n, lo, hi, src, sgn);
        if (src < 0) { if (k == 3) gi -= x[q] * p_inflow / (g1 * g1); }
        else Ubar[k * g.plane + off(src)] += (k == 1 + axis && sgn < 0) ? -x[q] : x[q];
      }
    }
  }
  gpartial[t < 2 * nline ? t : 2 * nline] = gi;  // slot 2 * nline: scratch for the idle threads
}

// gamma_bar += sum of n partial sums, in a fixed order (one CTA)
__global__ void __launch_bounds__(1024) sum_partials_kernel(const double* __restrict__ p, long long n, double* out) {
  __shared__ double red[32];
  double a = 0.0;
  for (long long i = threadIdx.x; i < n; i += 1024) a += p[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < 32; ++w) s += red[w];
    *out += s;
  }
}

// The loss of PAPER.md Eq. 14 inside the 2D reverse sweep (as mse_inject_kernel): Ubar (+)= coef (U - target) on the
// interior cells of the padded buffers, partial[blockIdx.x] = this CTA's sum of (U - target)^2 (summed in a fixed order
// by sum_partials_kernel).  target: interior layout [4][ny][nx].
__global__ void __launch_bounds__(256) mse_inject2d_kernel(const double* __restrict__ U, const double* __restrict__ target,
                                                           double* __restrict__ X, GridDims g, double coef, int accumulate,
                                                           double* __restrict__ partial) {
  __shared__ double red[8];
  const long long n = (long long)g.nx * g.ny;
  double a = 0.0;
  for (long long t = blockIdx.x * 256LL + threadIdx.x; t < 4 * n; t += (long long)gridDim.x * 256) {
    const int k = (int)(t / n);
    const long long r0 = t - k * n;
    const int j = (int)(r0 / g.nx), i = (int)(r0 - (long long)j * g.nx);
    const long long o = k * g.plane + (long long)(j + 3) * g.pitch + i + 3;
    const double r = U[o] - target[t];
    X[o] = accumulate ? fma(coef, r, X[o]) : coef * r;
    a = fma(r, r, a);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red[w];
    partial[blockIdx.x] = t;
  }
}

}  // namespace jxs
