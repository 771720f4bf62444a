// jxo.cpp — the CPU ORACLE.  TEST INFRASTRUCTURE ONLY (see jxo.h).
//
// Plain nested loops over padded arrays [4][ny+6][nx+6], one thread, no SIMD
// intrinsics, no blocking, no fusion; compiled with -O2 -ffp-contract=off so
// that every add and multiply is rounded separately.  Templated on the scalar
// so the same source runs in double, in float and with a counting scalar.
//
// Passages followed (P:Lnn = /root/reference/PAPER.md line nn; Rn = reading n
// in DESIGN.md "Readings of the paper", used where the paper is silent/garbled):
//   O1  ghost frame          P:L162 (inflow / outflow / reflective walls); R11
//   O2  IBM ghost-cell fill  P:L109-111 (ghost-cell IBM, slip wall); R9
//   O3  primitives           P:L41 Eq. 2
//   O4  WENO5-JS             P:L46; constants R4
//   O5  HLLC                 P:L54-72 Eq. 3-7; star state R1, sign(0) R2
//   O6  viscous fluxes       P:L9 ("Navier-Stokes"), Eq. 10; R7, R8
//   O7  divergence           P:L85 Eq. 10
//   O8  SSP-RK3              R5 (paper: forward Euler, Eq. 10)
//   O9  CFL time step        R6 (paper silent)
//   O10 per-face MLP         P:L96 Eq. 11; R14
//   O11 CNN neural flux (2D)  P:L94 (3 conv layers, ReLU/ReLU/tanh, SAME padding, 6,388 parameters), Eq. 11-13
//                             (shared between x and y); readings R18-R20 of DESIGN.md
//   O12 tangent of the step   P:L115-128 Eq. 15-16 (the chain of Jacobians, applied to one direction), P:L149 (gamma
//                             inference); the solver run on the Dual scalar; R21-R23
//   O13 adjoint of the step   the transpose of O12 from its definition, one tangent run per entry (jxo.py:
//                             Oracle.step_fixed_dt_adjoint); R24
//
// PARITY UNPINNED against the paper (no external definition exists; the rules
// are shared definitions constrained only by invariants):
//   the dt rule (O9), the viscous discretisation (O6), the IBM interpolation
//   choices (O2) and the MLP input/output conventions (O10).
#include "jxo.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

namespace {

constexpr int NG = 3;  // ghost layers: the 6-cell WENO5 stencil reaches 3 cells

// ---------------------------------------------------------------------------
// counting scalar: a double that tallies the arithmetic performed on it
// ---------------------------------------------------------------------------
struct Tally {
  long long add = 0, mul = 0, div = 0, sqrt_ = 0, cmp = 0;
};
Tally g_tally;

struct Counted {
  double v;
  Counted() : v(0) {}
  Counted(double x) : v(x) {}
  explicit operator double() const { return v; }
};
inline Counted operator+(Counted a, Counted b) { g_tally.add++; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { g_tally.add++; return Counted(a.v - b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }
inline Counted operator*(Counted a, Counted b) { g_tally.mul++; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { g_tally.div++; return Counted(a.v / b.v); }
inline Counted& operator+=(Counted& a, Counted b) { a = a + b; return a; }
inline Counted& operator-=(Counted& a, Counted b) { a = a - b; return a; }
inline bool operator<(Counted a, Counted b) { g_tally.cmp++; return a.v < b.v; }
inline bool operator>(Counted a, Counted b) { g_tally.cmp++; return a.v > b.v; }
inline bool operator<=(Counted a, Counted b) { g_tally.cmp++; return a.v <= b.v; }
inline bool operator>=(Counted a, Counted b) { g_tally.cmp++; return a.v >= b.v; }

inline double s_sqrt(double x) { return std::sqrt(x); }
inline float s_sqrt(float x) { return std::sqrt(x); }
inline Counted s_sqrt(Counted x) { g_tally.sqrt_++; return Counted(std::sqrt(x.v)); }
inline double s_abs(double x) { return std::fabs(x); }
inline float s_abs(float x) { return std::fabs(x); }
inline Counted s_abs(Counted x) { g_tally.cmp++; return Counted(std::fabs(x.v)); }
template <class T> inline T s_min(T a, T b) { return (b < a) ? b : a; }
template <class T> inline T s_max(T a, T b) { return (a < b) ? b : a; }
inline double to_double(double x) { return x; }
inline double to_double(float x) { return (double)x; }
inline double to_double(Counted x) { return x.v; }

// ---------------------------------------------------------------------------
// dual number: a value and its derivative along ONE direction of perturbation.
// Running the solver on it applies the chain of Jacobians of PAPER.md Eq. 16,
//   prod_j dU^{n+j}/dU^{n+j-1}  and  dU^{n+k}/d(parameter),
// to that direction (forward-mode differentiation; R21).  Every rule below is
// the textbook derivative of the operation; comparisons look at the value only,
// so min / max / sign / the positivity guard take the derivative of the branch
// the value selects, and |x| has derivative sign(x) (0 at x = 0).
// ---------------------------------------------------------------------------
struct Dual {
  double v, d;
  Dual() : v(0), d(0) {}
  Dual(double x) : v(x), d(0) {}
  Dual(double x, double dx) : v(x), d(dx) {}
  explicit operator double() const { return v; }
};
inline Dual operator+(Dual a, Dual b) { return Dual(a.v + b.v, a.d + b.d); }
inline Dual operator-(Dual a, Dual b) { return Dual(a.v - b.v, a.d - b.d); }
inline Dual operator-(Dual a) { return Dual(-a.v, -a.d); }
inline Dual operator*(Dual a, Dual b) { return Dual(a.v * b.v, a.d * b.v + a.v * b.d); }
inline Dual operator/(Dual a, Dual b) { return Dual(a.v / b.v, (a.d * b.v - a.v * b.d) / (b.v * b.v)); }
inline Dual& operator+=(Dual& a, Dual b) { a = a + b; return a; }
inline Dual& operator-=(Dual& a, Dual b) { a = a - b; return a; }
inline bool operator<(Dual a, Dual b) { return a.v < b.v; }
inline bool operator>(Dual a, Dual b) { return a.v > b.v; }
inline bool operator<=(Dual a, Dual b) { return a.v <= b.v; }
inline bool operator>=(Dual a, Dual b) { return a.v >= b.v; }
inline Dual s_sqrt(Dual x) { const double r = std::sqrt(x.v); return Dual(r, x.d / (2.0 * r)); }
inline Dual s_tanh(Dual x) { const double t = std::tanh(x.v); return Dual(t, (1.0 - t * t) * x.d); }
inline Dual s_abs(Dual x) { return Dual(std::fabs(x.v), x.v > 0 ? x.d : (x.v < 0 ? -x.d : 0.0)); }
inline double to_double(Dual x) { return x.v; }

// ---------------------------------------------------------------------------
// O4  WENO5-JS, left-biased value at i+1/2 from (a,b,c,d,e) = v[i-2..i+2]
//     ("WENO ... convex reconstruction of candidate stencils"; R4:
//     eps = 1e-6, linear weights 0.1/0.6/0.3, classical smoothness indicators,
//     exponent 2 — BASELINE.json configs[0])
// ---------------------------------------------------------------------------
template <class T>
T weno5(T a, T b, T c, T d, T e) {
  const T eps = T(1e-6);
  const T q0 = (T(2) * a - T(7) * b + T(11) * c) / T(6);
  const T q1 = (-b + T(5) * c + T(2) * d) / T(6);
  const T q2 = (T(2) * c + T(5) * d - e) / T(6);
  const T s0 = a - T(2) * b + c, t0 = a - T(4) * b + T(3) * c;
  const T s1 = b - T(2) * c + d, t1 = b - d;
  const T s2 = c - T(2) * d + e, t2 = T(3) * c - T(4) * d + e;
  const T c1312 = T(13) / T(12), c14 = T(1) / T(4);
  const T b0 = c1312 * (s0 * s0) + c14 * (t0 * t0);
  const T b1 = c1312 * (s1 * s1) + c14 * (t1 * t1);
  const T b2 = c1312 * (s2 * s2) + c14 * (t2 * t2);
  const T a0 = T(0.1) / ((eps + b0) * (eps + b0));
  const T a1 = T(0.6) / ((eps + b1) * (eps + b1));
  const T a2 = T(0.3) / ((eps + b2) * (eps + b2));
  return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
}

// ---------------------------------------------------------------------------
// O5  HLLC flux along x from primitive states W = (rho,u,v,p)
//     Eq. 3 (blend with sign(s*)), Eq. 5-6 (Davis speeds), Eq. 7 (contact speed)
//     Eq. 4 is garbled in the source; R1: the standard star state of the cited
//     source family (Toro; Johnsen & Colonius [6]):
//       U*k = rho_k chi_k [1, s*, v_k, E_k/rho_k + (s*-u_k)(s* + p_k/(rho_k (s_k-u_k)))]
//       chi_k = (s_k-u_k)/(s_k-s*)
//     R2: sign(0) = 0.
// ---------------------------------------------------------------------------
template <class T>
struct HllcDetail {
  T sL, sR, sS;
  T UsL[4], UsR[4];
};

template <class T>
void hllc_x(const T WL[4], const T WR[4], T gamma, T F[4], HllcDetail<T>* det = nullptr) {
  const T rL = WL[0], uL = WL[1], vL = WL[2], pL = WL[3];
  const T rR = WR[0], uR = WR[1], vR = WR[2], pR = WR[3];
  const T aL = s_sqrt(gamma * pL / rL);
  const T aR = s_sqrt(gamma * pR / rR);
  const T sL = s_min(uL - aL, uR - aR);                                     // Eq. 6
  const T sR = s_max(uL + aL, uR + aR);
  const T sS = (pR - pL + rL * uL * (sL - uL) - rR * uR * (sR - uR)) /      // Eq. 7
               (rL * (sL - uL) - rR * (sR - uR));
  const T sm = s_min(T(0), sL), sp = s_max(T(0), sR);                       // Eq. 5
  const T g1 = gamma - T(1);
  const T EL = pL / g1 + T(0.5) * rL * (uL * uL + vL * vL);
  const T ER = pR / g1 + T(0.5) * rR * (uR * uR + vR * vR);
  const T UL[4] = {rL, rL * uL, rL * vL, EL};
  const T UR[4] = {rR, rR * uR, rR * vR, ER};
  const T FL[4] = {rL * uL, rL * uL * uL + pL, rL * uL * vL, uL * (EL + pL)};
  const T FR[4] = {rR * uR, rR * uR * uR + pR, rR * uR * vR, uR * (ER + pR)};
  const T chiL = (sL - uL) / (sL - sS), chiR = (sR - uR) / (sR - sS);
  const T UsL[4] = {rL * chiL, rL * chiL * sS, rL * chiL * vL,
                    rL * chiL * (EL / rL + (sS - uL) * (sS + pL / (rL * (sL - uL))))};
  const T UsR[4] = {rR * chiR, rR * chiR * sS, rR * chiR * vR,
                    rR * chiR * (ER / rR + (sS - uR) * (sS + pR / (rR * (sR - uR))))};
  T sg = T(0);
  if (sS > T(0)) sg = T(1);
  else if (sS < T(0)) sg = T(-1);
  const T wl = (T(1) + sg) / T(2), wr = (T(1) - sg) / T(2);                 // Eq. 3
  for (int k = 0; k < 4; ++k)
    F[k] = wl * (FL[k] + sm * (UsL[k] - UL[k])) + wr * (FR[k] + sp * (UsR[k] - UR[k]));
  if (det) {
    det->sL = sL; det->sR = sR; det->sS = sS;
    for (int k = 0; k < 4; ++k) { det->UsL[k] = UsL[k]; det->UsR[k] = UsR[k]; }
  }
}

// bf16 round-to-nearest-even of a double (via float), used by the emulating MLP
inline double bf16_round(double x) {
  float f = (float)x;
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return (double)f;  // inf / nan
  const uint32_t lsb = (u >> 16) & 1u;
  u += 0x7fffu + lsb;
  u &= 0xffff0000u;
  std::memcpy(&f, &u, 4);
  return (double)f;
}

struct Mlp {
  bool on = false, bf16 = false;
  std::vector<double> W1, b1, W2, b2, W3, b3;  // W1[64][24], W2[64][64], W3[4][64]
  double in_scale[4] = {1, 1, 1, 1}, out_scale[4] = {1, 1, 1, 1};
  // direction of perturbation of the parameters for the tangent O12 (same layout; empty = the parameters do not move)
  std::vector<double> dW1, db1, dW2, db2, dW3, db3;
  // O10 on the dual scalar (exact mode only): the same three layers, every parameter carrying its direction
  void eval_dual(const Dual x[24], Dual y[4]) const {
    const bool dir = !dW1.empty();
    auto par = [&](const std::vector<double>& w, const std::vector<double>& d, size_t i) { return Dual(w[i], dir ? d[i] : 0.0); };
    Dual h1[64], h2[64];
    for (int o = 0; o < 64; ++o) {
      Dual s = par(b1, db1, o);
      for (int k = 0; k < 24; ++k) s += par(W1, dW1, o * 24 + k) * x[k];
      h1[o] = s_tanh(s);
    }
    for (int o = 0; o < 64; ++o) {
      Dual s = par(b2, db2, o);
      for (int k = 0; k < 64; ++k) s += par(W2, dW2, o * 64 + k) * h1[k];
      h2[o] = s_tanh(s);
    }
    for (int o = 0; o < 4; ++o) {
      Dual s = par(b3, db3, o);
      for (int k = 0; k < 64; ++k) s += par(W3, dW3, o * 64 + k) * h2[k];
      y[o] = s;
    }
  }
  // O10: h1 = tanh(W1 x + b1), h2 = tanh(W2 h1 + b2), y = W3 h2 + b3 (linear)
  void eval(const double x_in[24], double y[4]) const {
    double x[24], h1[64], h2[64];
    for (int k = 0; k < 24; ++k) x[k] = bf16 ? bf16_round(x_in[k]) : x_in[k];
    for (int o = 0; o < 64; ++o) {
      double s = b1[o];
      for (int k = 0; k < 24; ++k) s += W1[o * 24 + k] * x[k];
      h1[o] = std::tanh(s);
      if (bf16) h1[o] = bf16_round(h1[o]);
    }
    for (int o = 0; o < 64; ++o) {
      double s = b2[o];
      for (int k = 0; k < 64; ++k) s += W2[o * 64 + k] * h1[k];
      h2[o] = std::tanh(s);
      if (bf16) h2[o] = bf16_round(h2[o]);
    }
    for (int o = 0; o < 4; ++o) {
      double s = b3[o];
      for (int k = 0; k < 64; ++k) s += W3[o * 64 + k] * h2[k];
      y[o] = s;
    }
  }
};

// O11: the paper's fully convolutional neural flux: three 3x3 convolutions 4 -> 32 -> 16 -> 4 with biases
// (1184 + 4624 + 580 = 6,388 parameters, the count the paper prints), ReLU, ReLU, tanh, zero ("SAME") padding at
// every layer.  A field is in[c][a][b], a = index along the face's TANGENTIAL direction, b = along its NORMAL
// direction (R19: the same weights serve x- and y-faces, Eq. 13).  Cross-correlation, as in JAX / PyTorch:
//   out[o][a][b] = act( bias[o] + sum_c sum_{da,db = -1..1} W[o][c][da+1][db+1] * in[c][a+da][b+db] ).
struct Cnn {
  bool on = false, bf16 = false;
  std::vector<double> W1, b1, W2, b2, W3, b3;  // W1[32][4][3][3], W2[16][32][3][3], W3[4][16][3][3]
  double in_scale[4] = {1, 1, 1, 1}, out_scale[4] = {1, 1, 1, 1};
  static void conv(const std::vector<double>& in, int cin, int na, int nb, const std::vector<double>& W,
                   const std::vector<double>& b, int cout, int act, bool round_out, std::vector<double>& out) {
    out.assign((size_t)cout * na * nb, 0.0);
    for (int o = 0; o < cout; ++o)
      for (int a = 0; a < na; ++a)
        for (int bb = 0; bb < nb; ++bb) {
          double s = b[o];
          for (int c = 0; c < cin; ++c)
            for (int da = -1; da <= 1; ++da)
              for (int db = -1; db <= 1; ++db) {
                const int a2 = a + da, b2 = bb + db;
                if (a2 < 0 || a2 >= na || b2 < 0 || b2 >= nb) continue;  // zero padding
                s += W[(((size_t)o * cin + c) * 3 + (da + 1)) * 3 + (db + 1)] * in[((size_t)c * na + a2) * nb + b2];
              }
          s = act == 0 ? (s > 0.0 ? s : 0.0) : std::tanh(s);
          out[((size_t)o * na + a) * nb + bb] = round_out ? bf16_round(s) : s;
        }
  }
  // in[4][na][nb] (already normalised) -> out[4][na][nb] in (-1,1)
  void apply(const std::vector<double>& in, int na, int nb, std::vector<double>& out) const {
    std::vector<double> x(in), h1, h2;
    if (bf16) for (double& v : x) v = bf16_round(v);
    conv(x, 4, na, nb, W1, b1, 32, 0, bf16, h1);
    conv(h1, 32, na, nb, W2, b2, 16, 0, bf16, h2);
    conv(h2, 16, na, nb, W3, b3, 4, 1, false, out);
  }
};

struct IbmGhost {
  int i, j;          // the ghost cell
  int di[4], dj[4];  // bilinear donors (i0,j0),(i0+1,j0),(i0,j0+1),(i0+1,j0+1)
  double w[4];       // weights, zero at non-fluid donors, renormalised
  double nx, ny;     // unit normal pointing into the fluid
};

struct Config {
  int nx, ny;
  double dx, dy, gamma, mu, Pr, nu;
  jxo_bc bc;
  double gamma_dot = 0;  // perturbation of gamma carried by the Dual scalar (jxo_step_fixed_dt_tangent), else unused
};

// gamma as the solver's scalar: for Dual it carries the direction of perturbation
template <class T> inline T gamma_of(const Config& c) { return T(c.gamma); }
template <> inline Dual gamma_of<Dual>(const Config& c) { return Dual(c.gamma, c.gamma_dot); }

// ---------------------------------------------------------------------------
// the solver, templated on the scalar
// ---------------------------------------------------------------------------
template <class T>
struct Core {
  const Config& c;
  const std::vector<unsigned char>& type;  // 0 fluid 1 ghost 2 solid (interior)
  const std::vector<IbmGhost>& ghosts;
  const Mlp& mlp;
  const Cnn* cnn = nullptr;
  std::vector<double>* cap[4] = {nullptr, nullptr, nullptr, nullptr};  // observers: Xx, Xy, Yx, Yy of the last rhs (O11)
  long long guard = 0;
  int nxp, nyp;
  size_t plane;

  Core(const Config& cfg, const std::vector<unsigned char>& ty, const std::vector<IbmGhost>& gh,
       const Mlp& m)
      : c(cfg), type(ty), ghosts(gh), mlp(m) {
    nxp = c.nx + 2 * NG;
    nyp = c.ny + 2 * NG;
    plane = (size_t)nxp * nyp;
  }
  inline size_t at(int i, int j) const { return (size_t)(j + NG) * nxp + (i + NG); }

  void pad(const T* U, std::vector<T>& Up) const {
    Up.assign(4 * plane, T(0));
    for (int k = 0; k < 4; ++k)
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) Up[k * plane + at(i, j)] = U[((size_t)k * c.ny + j) * c.nx + i];
  }
  void unpad(const std::vector<T>& Up, T* U) const {
    for (int k = 0; k < 4; ++k)
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) U[((size_t)k * c.ny + j) * c.nx + i] = Up[k * plane + at(i, j)];
  }

  // O1: three ghost layers per side; x sides first for j in [0,ny), then the y
  // sides over the x-extended range i in [-3,nx+3) (this fills the corners).
  void fill_side(std::vector<T>& Up, int axis, int side, int g, int lo, int hi) const {
    const int n = axis == 0 ? c.nx : c.ny;
    const int kind = axis == 0 ? (side == 0 ? c.bc.xlo : c.bc.xhi) : (side == 0 ? c.bc.ylo : c.bc.yhi);
    const int dst = side == 0 ? -g : n - 1 + g;
    int src = 0;
    switch (kind) {
      case JXO_BC_PERIODIC: src = side == 0 ? n - g : g - 1; break;
      case JXO_BC_TRANSMISSIVE: src = side == 0 ? 0 : n - 1; break;
      case JXO_BC_REFLECTIVE: src = side == 0 ? g - 1 : n - g; break;
      default: break;
    }
    T inflow[4];
    {
      const T r = T(c.bc.inflow[0]), u = T(c.bc.inflow[1]), v = T(c.bc.inflow[2]), p = T(c.bc.inflow[3]);
      inflow[0] = r; inflow[1] = r * u; inflow[2] = r * v;
      inflow[3] = p / (gamma_of<T>(c) - T(1)) + T(0.5) * r * (u * u + v * v);
    }
    for (int t = lo; t < hi; ++t) {
      for (int k = 0; k < 4; ++k) {
        const size_t d = axis == 0 ? at(dst, t) : at(t, dst);
        const size_t s = axis == 0 ? at(src, t) : at(t, src);
        T val;
        if (kind == JXO_BC_INFLOW) val = inflow[k];
        else {
          val = Up[k * plane + s];
          // reflective wall: negate the wall-normal momentum
          if (kind == JXO_BC_REFLECTIVE && k == 1 + axis) val = -val;
        }
        Up[k * plane + d] = val;
      }
    }
  }
  void fill_frame(std::vector<T>& Up) const {
    for (int g = 1; g <= NG; ++g) {
      fill_side(Up, 0, 0, g, 0, c.ny);
      fill_side(Up, 0, 1, g, 0, c.ny);
    }
    for (int g = 1; g <= NG; ++g) {
      fill_side(Up, 1, 0, g, -NG, c.nx + NG);
      fill_side(Up, 1, 1, g, -NG, c.nx + NG);
    }
  }

  // O3 / Eq. 2: conserved -> primitive at one padded cell
  inline void prim_at(const std::vector<T>& Up, size_t a, T W[4]) const {
    const T r = Up[a], ru = Up[plane + a], rv = Up[2 * plane + a], E = Up[3 * plane + a];
    const T u = ru / r, v = rv / r;
    W[0] = r; W[1] = u; W[2] = v;
    W[3] = (gamma_of<T>(c) - T(1)) * (E - T(0.5) * r * (u * u + v * v));
  }

  // O2 / I6: gather primitives at the donors, interpolate to the image point,
  // reflect the velocity about the normal (slip wall), store conserved.
  void fill_ibm(std::vector<T>& Up) const {
    for (const IbmGhost& g : ghosts) {
      T WI[4] = {T(0), T(0), T(0), T(0)};
      for (int d = 0; d < 4; ++d) {
        if (g.w[d] == 0.0) continue;
        T W[4];
        prim_at(Up, at(g.di[d], g.dj[d]), W);
        for (int k = 0; k < 4; ++k) WI[k] += T(g.w[d]) * W[k];
      }
      const T nx_ = T(g.nx), ny_ = T(g.ny);
      const T un = WI[1] * nx_ + WI[2] * ny_;
      const T r = WI[0], u = WI[1] - T(2) * un * nx_, v = WI[2] - T(2) * un * ny_, p = WI[3];
      const size_t a = at(g.i, g.j);
      Up[a] = r;
      Up[plane + a] = r * u;
      Up[2 * plane + a] = r * v;
      Up[3 * plane + a] = p / (gamma_of<T>(c) - T(1)) + T(0.5) * r * (u * u + v * v);
    }
  }

  // L(U) on a padded, ghost-filled array.  L is interior [4][ny][nx].
  void rhs(const std::vector<T>& Up, T* L) {
    const int nx = c.nx, ny = c.ny;
    const T gamma = gamma_of<T>(c);
    // O3: primitives at all padded cells
    std::vector<T> W(4 * plane);
    for (int j = -NG; j < ny + NG; ++j)
      for (int i = -NG; i < nx + NG; ++i) {
        T w[4];
        prim_at(Up, at(i, j), w);
        for (int k = 0; k < 4; ++k) W[k * plane + at(i, j)] = w[k];
      }
    auto Wv = [&](int k, int i, int j) -> T { return W[k * plane + at(i, j)]; };

    // x-faces: Fx[k][j][f], f = 0..nx is the face between cells f-1 and f
    std::vector<T> Fx((size_t)4 * ny * (nx + 1)), Gy((size_t)4 * (ny + 1) * nx);
    // O11 (R19): the network's input at a face = mean of the left and right reconstructed states, as conservative
    // variables (rho, rho u_n, rho u_t, E), divided by in_scale.  Xx[c][j][f] (tangential j, normal f),
    // Xy[c][i][f] (tangential i, normal f).
    const bool cnn_on = cnn && cnn->on;
    std::vector<double> Xx, Xy;
    if (cnn_on) { Xx.assign((size_t)4 * ny * (nx + 1), 0.0); Xy.assign((size_t)4 * nx * (ny + 1), 0.0); }
    auto face_input = [&](const T* SL, const T* SR, double* x4) {  // S = (rho, u_n, u_t, p)
      double m[4] = {0, 0, 0, 0};
      for (int side = 0; side < 2; ++side) {
        const T* S = side == 0 ? SL : SR;
        const double r = to_double(S[0]), un = to_double(S[1]), ut = to_double(S[2]), p = to_double(S[3]);
        m[0] += r; m[1] += r * un; m[2] += r * ut; m[3] += p / (c.gamma - 1.0) + 0.5 * r * (un * un + ut * ut);
      }
      for (int k = 0; k < 4; ++k) x4[k] = 0.5 * m[k] / cnn->in_scale[k];
    };
    for (int j = 0; j < ny; ++j)
      for (int f = 0; f <= nx; ++f) {
        const int i = f - 1;  // face i+1/2
        T WL[4], WR[4];
        for (int k = 0; k < 4; ++k) {  // O4, component-wise on (rho,u,v,p) (R3)
          WL[k] = weno5(Wv(k, i - 2, j), Wv(k, i - 1, j), Wv(k, i, j), Wv(k, i + 1, j), Wv(k, i + 2, j));
          WR[k] = weno5(Wv(k, i + 3, j), Wv(k, i + 2, j), Wv(k, i + 1, j), Wv(k, i, j), Wv(k, i - 1, j));
        }
        // positivity guard (R15): a side with rho<=0 or p<=0 falls back to its cell
        if (WL[0] <= T(0) || WL[3] <= T(0)) { ++guard; for (int k = 0; k < 4; ++k) WL[k] = Wv(k, i, j); }
        if (WR[0] <= T(0) || WR[3] <= T(0)) { ++guard; for (int k = 0; k < 4; ++k) WR[k] = Wv(k, i + 1, j); }
        T F[4];
        hllc_x(WL, WR, gamma, F);
        if (mlp.on) {  // O10: cells i-2..i+3, each (rho,u,v,p)/in_scale
          if constexpr (std::is_same<T, Dual>::value) {  // O12: the network's inputs and parameters carry their directions
            Dual x[24], y[4];
            for (int cc = 0; cc < 6; ++cc)
              for (int k = 0; k < 4; ++k) x[4 * cc + k] = Wv(k, i - 2 + cc, j) / Dual(mlp.in_scale[k]);
            mlp.eval_dual(x, y);
            for (int k = 0; k < 4; ++k) F[k] += Dual(mlp.out_scale[k]) * y[k];
          } else {
            double x[24], y[4];
            for (int cc = 0; cc < 6; ++cc)
              for (int k = 0; k < 4; ++k) x[4 * cc + k] = to_double(Wv(k, i - 2 + cc, j)) / mlp.in_scale[k];
            mlp.eval(x, y);
            for (int k = 0; k < 4; ++k) F[k] += T(mlp.out_scale[k] * y[k]);  // Eq. 11
          }
        }
        if (cnn_on) {
          double x4[4];
          face_input(WL, WR, x4);
          for (int k = 0; k < 4; ++k) Xx[((size_t)k * ny + j) * (nx + 1) + f] = x4[k];
        }
        for (int k = 0; k < 4; ++k) Fx[((size_t)k * ny + j) * (nx + 1) + f] = F[k];
      }
    // y-faces: the same routine with u and v interchanged
    for (int f = 0; f <= ny; ++f)
      for (int i = 0; i < nx; ++i) {
        const int j = f - 1;
        T WL[4], WR[4];
        for (int k = 0; k < 4; ++k) {
          WL[k] = weno5(Wv(k, i, j - 2), Wv(k, i, j - 1), Wv(k, i, j), Wv(k, i, j + 1), Wv(k, i, j + 2));
          WR[k] = weno5(Wv(k, i, j + 3), Wv(k, i, j + 2), Wv(k, i, j + 1), Wv(k, i, j), Wv(k, i, j - 1));
        }
        if (WL[0] <= T(0) || WL[3] <= T(0)) { ++guard; for (int k = 0; k < 4; ++k) WL[k] = Wv(k, i, j); }
        if (WR[0] <= T(0) || WR[3] <= T(0)) { ++guard; for (int k = 0; k < 4; ++k) WR[k] = Wv(k, i, j + 1); }
        const T SL[4] = {WL[0], WL[2], WL[1], WL[3]}, SR[4] = {WR[0], WR[2], WR[1], WR[3]};
        T F[4];
        hllc_x(SL, SR, gamma, F);
        if (mlp.on) {  // normal velocity first: (rho, v, u, p)
          static const int perm[4] = {0, 2, 1, 3};
          if constexpr (std::is_same<T, Dual>::value) {
            Dual x[24], y[4];
            for (int cc = 0; cc < 6; ++cc)
              for (int k = 0; k < 4; ++k) x[4 * cc + k] = Wv(perm[k], i, j - 2 + cc) / Dual(mlp.in_scale[k]);
            mlp.eval_dual(x, y);
            for (int k = 0; k < 4; ++k) F[k] += Dual(mlp.out_scale[k]) * y[k];
          } else {
            double x[24], y[4];
            for (int cc = 0; cc < 6; ++cc)
              for (int k = 0; k < 4; ++k) x[4 * cc + k] = to_double(Wv(perm[k], i, j - 2 + cc)) / mlp.in_scale[k];
            mlp.eval(x, y);
            for (int k = 0; k < 4; ++k) F[k] += T(mlp.out_scale[k] * y[k]);
          }
        }
        if (cnn_on) {
          double x4[4];
          face_input(SL, SR, x4);
          for (int k = 0; k < 4; ++k) Xy[((size_t)k * nx + i) * (ny + 1) + f] = x4[k];
        }
        Gy[((size_t)0 * (ny + 1) + f) * nx + i] = F[0];
        Gy[((size_t)1 * (ny + 1) + f) * nx + i] = F[2];  // x-momentum = tangential
        Gy[((size_t)2 * (ny + 1) + f) * nx + i] = F[1];  // y-momentum = normal
        Gy[((size_t)3 * (ny + 1) + f) * nx + i] = F[3];
      }

    if (cnn_on) {  // Eq. 11-13: F^Neural = out_scale o CNN(field), same weights for both directions
      std::vector<double> Y;
      cnn->apply(Xx, ny, nx + 1, Y);
      if (cap[0]) { *cap[0] = Xx; *cap[1] = Xy; *cap[2] = Y; }
      for (int k = 0; k < 4; ++k)
        for (int j = 0; j < ny; ++j)
          for (int f = 0; f <= nx; ++f)
            Fx[((size_t)k * ny + j) * (nx + 1) + f] += T(cnn->out_scale[k] * Y[((size_t)k * ny + j) * (nx + 1) + f]);
      cnn->apply(Xy, nx, ny + 1, Y);
      if (cap[3]) *cap[3] = Y;
      static const int to_cons[4] = {0, 2, 1, 3};  // (mass, normal = rho v, tangential = rho u, energy) -> conserved slot
      for (int k = 0; k < 4; ++k)
        for (int i = 0; i < nx; ++i)
          for (int f = 0; f <= ny; ++f)
            Gy[((size_t)to_cons[k] * (ny + 1) + f) * nx + i] += T(cnn->out_scale[k] * Y[((size_t)k * nx + i) * (ny + 1) + f]);
    }

    // O6: viscous fluxes (R7, R8), constant mu, Stokes hypothesis, T = p/rho,
    // k = mu*gamma/((gamma-1) Pr); face-centred second-order central differences
    std::vector<T> Fv, Gv;
    const bool visc = c.mu > 0.0;
    if (visc) {
      const T mu = T(c.mu), kap = T(c.mu) * gamma / ((gamma - T(1)) * T(c.Pr));
      const T dx = T(c.dx), dy = T(c.dy);
      auto Tm = [&](int i, int j) -> T { return Wv(3, i, j) / Wv(0, i, j); };
      Fv.assign((size_t)4 * ny * (nx + 1), T(0));
      Gv.assign((size_t)4 * (ny + 1) * nx, T(0));
      for (int j = 0; j < ny; ++j)
        for (int f = 0; f <= nx; ++f) {
          const int i = f - 1;  // face between (i,j) and (i+1,j)
          const T ux = (Wv(1, i + 1, j) - Wv(1, i, j)) / dx;
          const T vx = (Wv(2, i + 1, j) - Wv(2, i, j)) / dx;
          const T Tx = (Tm(i + 1, j) - Tm(i, j)) / dx;
          const T uy = T(0.25) * ((Wv(1, i, j + 1) - Wv(1, i, j - 1)) + (Wv(1, i + 1, j + 1) - Wv(1, i + 1, j - 1))) / dy;
          const T vy = T(0.25) * ((Wv(2, i, j + 1) - Wv(2, i, j - 1)) + (Wv(2, i + 1, j + 1) - Wv(2, i + 1, j - 1))) / dy;
          const T ub = T(0.5) * (Wv(1, i, j) + Wv(1, i + 1, j)), vb = T(0.5) * (Wv(2, i, j) + Wv(2, i + 1, j));
          const T txx = mu * (T(4) / T(3) * ux - T(2) / T(3) * vy);
          const T txy = mu * (uy + vx);
          const size_t o = (size_t)j * (nx + 1) + f, st = (size_t)ny * (nx + 1);
          Fv[st + o] = txx;
          Fv[2 * st + o] = txy;
          Fv[3 * st + o] = ub * txx + vb * txy + kap * Tx;
        }
      for (int f = 0; f <= ny; ++f)
        for (int i = 0; i < nx; ++i) {
          const int j = f - 1;  // face between (i,j) and (i,j+1)
          const T uy = (Wv(1, i, j + 1) - Wv(1, i, j)) / dy;
          const T vy = (Wv(2, i, j + 1) - Wv(2, i, j)) / dy;
          const T Ty = (Tm(i, j + 1) - Tm(i, j)) / dy;
          const T ux = T(0.25) * ((Wv(1, i + 1, j) - Wv(1, i - 1, j)) + (Wv(1, i + 1, j + 1) - Wv(1, i - 1, j + 1))) / dx;
          const T vx = T(0.25) * ((Wv(2, i + 1, j) - Wv(2, i - 1, j)) + (Wv(2, i + 1, j + 1) - Wv(2, i - 1, j + 1))) / dx;
          const T ub = T(0.5) * (Wv(1, i, j) + Wv(1, i, j + 1)), vb = T(0.5) * (Wv(2, i, j) + Wv(2, i, j + 1));
          const T tyy = mu * (T(4) / T(3) * vy - T(2) / T(3) * ux);
          const T txy = mu * (uy + vx);
          const size_t o = (size_t)f * nx + i, st = (size_t)(ny + 1) * nx;
          Gv[st + o] = txy;
          Gv[2 * st + o] = tyy;
          Gv[3 * st + o] = ub * txy + vb * tyy + kap * Ty;
        }
    }

    // O7: L = -dF/dx - dG/dy + dFv/dx + dGv/dy + nu * Laplacian_h(U); 0 at non-fluid cells
    const T dx = T(c.dx), dy = T(c.dy), nu = T(c.nu);
    for (int k = 0; k < 4; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const size_t o = ((size_t)k * ny + j) * nx + i;
          if (type[(size_t)j * nx + i] != 0) { L[o] = T(0); continue; }
          const size_t fx = ((size_t)k * ny + j) * (nx + 1) + i;
          const size_t gy = ((size_t)k * (ny + 1) + j) * nx + i;
          T v = -(Fx[fx + 1] - Fx[fx]) / dx - (Gy[gy + nx] - Gy[gy]) / dy;
          if (visc) v += (Fv[fx + 1] - Fv[fx]) / dx + (Gv[gy + nx] - Gv[gy]) / dy;
          if (c.nu != 0.0) {
            const T* u = &Up[k * plane];
            const T lap = (u[at(i + 1, j)] - T(2) * u[at(i, j)] + u[at(i - 1, j)]) / (dx * dx) +
                          (u[at(i, j + 1)] - T(2) * u[at(i, j)] + u[at(i, j - 1)]) / (dy * dy);
            v += nu * lap;
          }
          L[o] = v;
        }
  }

  // O9: s_max over fluid interior cells of max(|u|+a, |v|+a)
  T max_wavespeed(const std::vector<T>& Up) const {
    T smax = T(0);
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) {
        if (type[(size_t)j * c.nx + i] != 0) continue;
        T w[4];
        prim_at(Up, at(i, j), w);
        const T a = s_sqrt(gamma_of<T>(c) * w[3] / w[0]);
        smax = s_max(smax, s_max(s_abs(w[1]) + a, s_abs(w[2]) + a));
      }
    return smax;
  }

  // one ghost fill + L
  void fill_and_rhs(std::vector<T>& Up, T* L) {
    fill_frame(Up);
    fill_ibm(Up);
    rhs(Up, L);
  }

  // O8: SSP-RK3 (Shu-Osher); ghost fills before every L
  void rk3_step(std::vector<T>& U0, T dt) {
    const size_t n = (size_t)c.nx * c.ny;
    std::vector<T> L(4 * n), U1(U0), U2;
    fill_and_rhs(U0, L.data());
    for (int k = 0; k < 4; ++k)
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) {
          const size_t a = k * plane + at(i, j);
          U1[a] = U0[a] + dt * L[(k * (size_t)c.ny + j) * c.nx + i];
        }
    fill_and_rhs(U1, L.data());
    U2 = U1;
    for (int k = 0; k < 4; ++k)
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) {
          const size_t a = k * plane + at(i, j);
          U2[a] = T(0.75) * U0[a] + T(0.25) * (U1[a] + dt * L[(k * (size_t)c.ny + j) * c.nx + i]);
        }
    fill_and_rhs(U2, L.data());
    for (int k = 0; k < 4; ++k)
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) {
          const size_t a = k * plane + at(i, j);
          U0[a] = T(1) / T(3) * U0[a] + T(2) / T(3) * (U2[a] + dt * L[(k * (size_t)c.ny + j) * c.nx + i]);
        }
  }
};

}  // namespace

// ---------------------------------------------------------------------------
// handle
// ---------------------------------------------------------------------------
struct jxo_solver {
  Config c;
  int dtype;
  std::vector<unsigned char> type;  // interior cell types
  std::vector<IbmGhost> ghosts;
  Mlp mlp;
  Cnn cnn;
  long long guard = 0;
  double t = 0, last_dt = 0;
  std::string err;
};

namespace {

bool all_finite(const double* p, size_t n) {
  for (size_t i = 0; i < n; ++i)
    if (!std::isfinite(p[i])) return false;
  return true;
}

// O2 setup (I1-I5), once per phi
int build_ibm(jxo_solver* s, const double* phi) {
  const int nx = s->c.nx, ny = s->c.ny;
  const double dx = s->c.dx, dy = s->c.dy;
  s->type.assign((size_t)nx * ny, 0);
  s->ghosts.clear();
  if (!phi) return JXO_OK;
  auto P = [&](int i, int j) { return phi[(size_t)j * nx + i]; };
  auto fluid = [&](int i, int j) { return i >= 0 && i < nx && j >= 0 && j < ny && P(i, j) > 0.0; };
  // I1: fluid <=> phi > 0; bodies must stay >= 8 cells away from the domain edges
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i)
      if (!(P(i, j) > 0.0)) {
        if (i < 8 || i >= nx - 8 || j < 8 || j >= ny - 8) {
          s->err = "IBM body closer than 8 cells to a domain edge";
          return JXO_EINVAL;
        }
        s->type[(size_t)j * nx + i] = 2;
      }
  // I2: ghost <=> non-fluid with a fluid cell at axis-aligned offset <= 3 or in the 3x3 box
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      if (s->type[(size_t)j * nx + i] == 0) continue;
      bool g = false;
      for (int k = 1; k <= 3 && !g; ++k)
        g = fluid(i - k, j) || fluid(i + k, j) || fluid(i, j - k) || fluid(i, j + k);
      g = g || fluid(i - 1, j - 1) || fluid(i + 1, j - 1) || fluid(i - 1, j + 1) || fluid(i + 1, j + 1);
      if (g) s->type[(size_t)j * nx + i] = 1;
    }
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      if (s->type[(size_t)j * nx + i] != 1) continue;
      IbmGhost g;
      g.i = i; g.j = j;
      // I3: n = grad(phi)/|grad(phi)| by central differences of the sampled phi
      double gx = (P(i + 1, j) - P(i - 1, j)) / (2.0 * dx);
      double gy = (P(i, j + 1) - P(i, j - 1)) / (2.0 * dy);
      const double gn = std::sqrt(gx * gx + gy * gy);
      if (!(gn > 0.0)) { s->err = "IBM: zero level-set gradient at a ghost cell"; return JXO_EINVAL; }
      gx /= gn; gy /= gn;
      g.nx = gx; g.ny = gy;
      // I4: image point x_I = x_G + 2 |phi_G| n
      const double xg = (i + 0.5) * dx, yg = (j + 0.5) * dy;
      double xi = xg + 2.0 * std::fabs(P(i, j)) * gx, yi = yg + 2.0 * std::fabs(P(i, j)) * gy;
      // I5: bilinear donors; zero non-fluid donors and renormalise; if no fluid
      // donor is left push the image point outward by min(dx,dy) n, <= 8 times
      bool ok = false;
      for (int attempt = 0; attempt <= 8 && !ok; ++attempt) {
        const double fx = xi / dx - 0.5, fy = yi / dy - 0.5;
        const int i0 = (int)std::floor(fx), j0 = (int)std::floor(fy);
        const double tx = fx - i0, ty = fy - j0;
        const double w[4] = {(1 - tx) * (1 - ty), tx * (1 - ty), (1 - tx) * ty, tx * ty};
        const int di[4] = {i0, i0 + 1, i0, i0 + 1}, dj[4] = {j0, j0, j0 + 1, j0 + 1};
        double sum = 0;
        for (int d = 0; d < 4; ++d) {
          g.di[d] = di[d]; g.dj[d] = dj[d];
          g.w[d] = fluid(di[d], dj[d]) ? w[d] : 0.0;
          sum += g.w[d];
        }
        if (sum > 0.0) {
          for (int d = 0; d < 4; ++d) {
            g.w[d] /= sum;
            if (g.w[d] == 0.0) { g.di[d] = i; g.dj[d] = j; }  // unused donor: any valid index
          }
          ok = true;
        } else {
          const double h = std::min(dx, dy);
          xi += h * gx; yi += h * gy;
        }
      }
      if (!ok) { s->err = "IBM: ghost cell without a fluid donor"; return JXO_EINVAL; }
      s->ghosts.push_back(g);
    }
  return JXO_OK;
}

template <class T>
int do_rhs(jxo_solver* s, const void* U, void* dUdt) {
  Core<T> core(s->c, s->type, s->ghosts, s->mlp);
  core.cnn = &s->cnn;
  std::vector<T> Up;
  core.pad((const T*)U, Up);
  core.fill_and_rhs(Up, (T*)dUdt);
  s->guard += core.guard;
  return JXO_OK;
}

template <class T>
int do_wavespeed(jxo_solver* s, const void* U, double* smax) {
  Core<T> core(s->c, s->type, s->ghosts, s->mlp);
  core.cnn = &s->cnn;
  std::vector<T> Up;
  core.pad((const T*)U, Up);
  *smax = to_double(core.max_wavespeed(Up));
  return JXO_OK;
}

template <class T>
int do_step(jxo_solver* s, void* U, double cfl, double fixed_dt, int nsteps) {
  Core<T> core(s->c, s->type, s->ghosts, s->mlp);
  core.cnn = &s->cnn;
  std::vector<T> Up;
  core.pad((T*)U, Up);
  int rc = JXO_OK;
  for (int n = 0; n < nsteps; ++n) {
    T dt;
    if (fixed_dt > 0) dt = T(fixed_dt);
    else {
      // O9: dt = cfl * min(dx,dy) / s_max, once per step on U^n
      const T smax = core.max_wavespeed(Up);
      if (!std::isfinite(to_double(smax)) || !(to_double(smax) > 0)) { rc = JXO_ENUMERIC; break; }
      dt = T(cfl) * T(std::min(s->c.dx, s->c.dy)) / smax;
    }
    core.rk3_step(Up, dt);
    s->t += to_double(dt);
    s->last_dt = to_double(dt);
  }
  core.unpad(Up, (T*)U);
  s->guard += core.guard;
  if (rc == JXO_OK) {
    const size_t n = (size_t)4 * s->c.nx * s->c.ny;
    const T* u = (const T*)U;
    for (size_t i = 0; i < n; ++i)
      if (!std::isfinite(to_double(u[i]))) { rc = JXO_ENUMERIC; break; }
  }
  if (rc == JXO_ENUMERIC) s->err = "non-finite state";
  return rc;
}

}  // namespace

extern "C" {

int jxo_create(int nx, int ny, double dx, double dy, double gamma, double mu, double Pr,
               const jxo_bc* bc, int dtype, jxo_solver** out) {
  if (!out || !bc) return JXO_EINVAL;
  *out = nullptr;
  if (nx < 8 || ny < 8 || !(dx > 0) || !(dy > 0) || !(gamma > 1) || mu < 0 || (mu > 0 && !(Pr > 0)))
    return JXO_EINVAL;
  if (dtype != JXO_F64 && dtype != JXO_F32) return JXO_EINVAL;
  const int k[4] = {bc->xlo, bc->xhi, bc->ylo, bc->yhi};
  for (int q = 0; q < 4; ++q)
    if (k[q] < 0 || k[q] > 3) return JXO_EINVAL;
  if ((bc->xlo == JXO_BC_PERIODIC) != (bc->xhi == JXO_BC_PERIODIC)) return JXO_EINVAL;
  if ((bc->ylo == JXO_BC_PERIODIC) != (bc->yhi == JXO_BC_PERIODIC)) return JXO_EINVAL;
  if (!all_finite(bc->inflow, 4)) return JXO_EINVAL;
  jxo_solver* s = new (std::nothrow) jxo_solver;
  if (!s) return JXO_ENOMEM;
  s->c = Config{nx, ny, dx, dy, gamma, mu, Pr, 0.0, *bc};
  s->dtype = dtype;
  s->type.assign((size_t)nx * ny, 0);
  *out = s;
  return JXO_OK;
}

void jxo_destroy(jxo_solver* s) { delete s; }
const char* jxo_last_error(const jxo_solver* s) { return s ? s->err.c_str() : "null handle"; }

int jxo_set_ibm(jxo_solver* s, const double* phi) {
  if (!s) return JXO_EINVAL;
  return build_ibm(s, phi);
}

int jxo_set_flux_mlp(jxo_solver* s, const float* w, const double in_scale[4], const double out_scale[4],
                     int emulate_bf16) {
  if (!s) return JXO_EINVAL;
  if (!w) { s->mlp.on = false; return JXO_OK; }
  if (!in_scale || !out_scale) return JXO_EINVAL;
  Mlp& m = s->mlp;
  m.bf16 = emulate_bf16 != 0;
  auto take = [&](std::vector<double>& dst, size_t n, bool round) {
    dst.resize(n);
    for (size_t i = 0; i < n; ++i) dst[i] = (round && m.bf16) ? bf16_round((double)w[i]) : (double)w[i];
    w += n;
  };
  // weights are rounded to bf16 in the emulating mode, biases stay fp32
  take(m.W1, 64 * 24, true); take(m.b1, 64, false);
  take(m.W2, 64 * 64, true); take(m.b2, 64, false);
  take(m.W3, 4 * 64, true);  take(m.b3, 4, false);
  for (int k = 0; k < 4; ++k) {
    if (!(in_scale[k] > 0)) return JXO_EINVAL;
    m.in_scale[k] = in_scale[k];
    m.out_scale[k] = out_scale[k];
  }
  m.dW1.clear(); m.db1.clear(); m.dW2.clear(); m.db2.clear(); m.dW3.clear(); m.db3.clear();
  m.on = true;
  return JXO_OK;
}

// direction of perturbation of the MLP's parameters for O12 (6020 doubles in the order of the weights); NULL = none.
// jxo_set_flux_mlp clears it.
int jxo_set_flux_mlp_direction(jxo_solver* s, const double* d) {
  if (!s) return JXO_EINVAL;
  Mlp& m = s->mlp;
  if (!d) { m.dW1.clear(); m.db1.clear(); m.dW2.clear(); m.db2.clear(); m.dW3.clear(); m.db3.clear(); return JXO_OK; }
  auto take = [&](std::vector<double>& dst, size_t n) { dst.assign(d, d + n); d += n; };
  take(m.dW1, 64 * 24); take(m.db1, 64); take(m.dW2, 64 * 64); take(m.db2, 64); take(m.dW3, 4 * 64); take(m.db3, 4);
  return JXO_OK;
}

int jxo_set_artificial_viscosity(jxo_solver* s, double nu) {
  if (!s || nu < 0) return JXO_EINVAL;
  s->c.nu = nu;
  return JXO_OK;
}

int jxo_rhs(jxo_solver* s, const void* U, void* dUdt) {
  if (!s || !U || !dUdt) return JXO_EINVAL;
  return s->dtype == JXO_F64 ? do_rhs<double>(s, U, dUdt) : do_rhs<float>(s, U, dUdt);
}

int jxo_max_wavespeed(jxo_solver* s, const void* U, double* smax) {
  if (!s || !U || !smax) return JXO_EINVAL;
  return s->dtype == JXO_F64 ? do_wavespeed<double>(s, U, smax) : do_wavespeed<float>(s, U, smax);
}

int jxo_step(jxo_solver* s, void* U, double cfl, int nsteps) {
  if (!s || !U || !(cfl > 0) || nsteps < 0) return JXO_EINVAL;
  return s->dtype == JXO_F64 ? do_step<double>(s, U, cfl, 0.0, nsteps) : do_step<float>(s, U, cfl, 0.0, nsteps);
}

int jxo_step_fixed_dt(jxo_solver* s, void* U, double dt, int nsteps) {
  if (!s || !U || !(dt > 0) || nsteps < 0) return JXO_EINVAL;
  return s->dtype == JXO_F64 ? do_step<double>(s, U, 0.0, dt, nsteps) : do_step<float>(s, U, 0.0, dt, nsteps);
}

int jxo_get_time(const jxo_solver* s, double* t, double* last_dt) {
  if (!s) return JXO_EINVAL;
  if (t) *t = s->t;
  if (last_dt) *last_dt = s->last_dt;
  return JXO_OK;
}

double jxo_weno5(const double v[5]) { return weno5<double>(v[0], v[1], v[2], v[3], v[4]); }

void jxo_hllc(const double WL[4], const double WR[4], double gamma, double F[4]) {
  hllc_x<double>(WL, WR, gamma, F);
}

void jxo_hllc_star(const double WL[4], const double WR[4], double gamma, double speeds[3],
                   double UstarL[4], double UstarR[4]) {
  double F[4];
  HllcDetail<double> d;
  hllc_x<double>(WL, WR, gamma, F, &d);
  speeds[0] = d.sL; speeds[1] = d.sR; speeds[2] = d.sS;
  for (int k = 0; k < 4; ++k) { UstarL[k] = d.UsL[k]; UstarR[k] = d.UsR[k]; }
}

// O12 (R21): the tangent of jxo_step_fixed_dt.  On return U = S^n(U; gamma) and
//   Udot = dS^n/dU . Udot + dS^n/dgamma . gamma_dot      (the Jacobian products of PAPER.md Eq. 16),
// computed by running the same templated solver on Dual scalars.  fp64 handles without a network.
int jxo_step_fixed_dt_tangent(jxo_solver* s, double* U, double* Udot, double gamma_dot, double dt, int nsteps) {
  if (!s || !U || !Udot || !(dt > 0) || nsteps < 0) return JXO_EINVAL;
  if (s->dtype != JXO_F64) { s->err = "the tangent is fp64 only"; return JXO_EINVAL; }
  if ((s->mlp.on && s->mlp.bf16) || s->cnn.on) { s->err = "the tangent differentiates the exact (fp64) MLP only"; return JXO_ESTATE; }
  const size_t n = (size_t)4 * s->c.nx * s->c.ny;
  std::vector<Dual> Ud(n), Up;
  for (size_t i = 0; i < n; ++i) Ud[i] = Dual(U[i], Udot[i]);
  s->c.gamma_dot = gamma_dot;
  Core<Dual> core(s->c, s->type, s->ghosts, s->mlp);
  core.pad(Ud.data(), Up);
  for (int k = 0; k < nsteps; ++k) {
    core.rk3_step(Up, Dual(dt));
    s->t += dt;
    s->last_dt = dt;
  }
  core.unpad(Up, Ud.data());
  s->c.gamma_dot = 0;
  s->guard += core.guard;
  int rc = JXO_OK;
  for (size_t i = 0; i < n; ++i) {
    U[i] = Ud[i].v;
    Udot[i] = Ud[i].d;
    if (!std::isfinite(U[i]) || !std::isfinite(Udot[i])) rc = JXO_ENUMERIC;
  }
  if (rc == JXO_ENUMERIC) s->err = "non-finite state or tangent";
  return rc;
}

// L(U) and its tangent: the building block of O12 for a caller-written time integrator (the forward-Euler update of
// PAPER.md Eq. 10 written out in jxo.py).  L, Ldot: [4][ny][nx] doubles, out.
int jxo_rhs_tangent(jxo_solver* s, const double* U, const double* Udot, double gamma_dot, double* L, double* Ldot) {
  if (!s || !U || !Udot || !L || !Ldot) return JXO_EINVAL;
  if (s->dtype != JXO_F64) { s->err = "the tangent is fp64 only"; return JXO_EINVAL; }
  if ((s->mlp.on && s->mlp.bf16) || s->cnn.on) { s->err = "the tangent differentiates the exact (fp64) MLP only"; return JXO_ESTATE; }
  const size_t n = (size_t)4 * s->c.nx * s->c.ny;
  std::vector<Dual> Ud(n), Ld(n), Up;
  for (size_t i = 0; i < n; ++i) Ud[i] = Dual(U[i], Udot[i]);
  s->c.gamma_dot = gamma_dot;
  Core<Dual> core(s->c, s->type, s->ghosts, s->mlp);
  core.pad(Ud.data(), Up);
  core.fill_and_rhs(Up, Ld.data());
  s->c.gamma_dot = 0;
  s->guard += core.guard;
  for (size_t i = 0; i < n; ++i) { L[i] = Ld[i].v; Ldot[i] = Ld[i].d; }
  return JXO_OK;
}

// pointwise tangents of O4 and O5, for the closed-form pins
void jxo_weno5_tangent(const double v[5], const double vdot[5], double out[2]) {
  const Dual r = weno5<Dual>(Dual(v[0], vdot[0]), Dual(v[1], vdot[1]), Dual(v[2], vdot[2]), Dual(v[3], vdot[3]),
                             Dual(v[4], vdot[4]));
  out[0] = r.v; out[1] = r.d;
}

void jxo_hllc_tangent(const double WL[4], const double WR[4], const double WLdot[4], const double WRdot[4],
                      double gamma, double gamma_dot, double F[4], double Fdot[4]) {
  Dual L[4], R[4], f[4];
  for (int k = 0; k < 4; ++k) { L[k] = Dual(WL[k], WLdot[k]); R[k] = Dual(WR[k], WRdot[k]); }
  hllc_x<Dual>(L, R, Dual(gamma, gamma_dot), f);
  for (int k = 0; k < 4; ++k) { F[k] = f[k].v; Fdot[k] = f[k].d; }
}

int jxo_fill_ghosts(jxo_solver* s, const void* U, void* Upad) {
  if (!s || !U || !Upad) return JXO_EINVAL;
  if (s->dtype == JXO_F64) {
    Core<double> core(s->c, s->type, s->ghosts, s->mlp);
    core.cnn = &s->cnn;
    std::vector<double> Up;
    core.pad((const double*)U, Up);
    core.fill_frame(Up);
    core.fill_ibm(Up);
    std::memcpy(Upad, Up.data(), Up.size() * sizeof(double));
  } else {
    Core<float> core(s->c, s->type, s->ghosts, s->mlp);
    core.cnn = &s->cnn;
    std::vector<float> Up;
    core.pad((const float*)U, Up);
    core.fill_frame(Up);
    core.fill_ibm(Up);
    std::memcpy(Upad, Up.data(), Up.size() * sizeof(float));
  }
  return JXO_OK;
}

int jxo_ibm_ghosts(const jxo_solver* s, int* cell, int* donors, double* weights, double* normal) {
  if (!s) return -1;
  const int nx = s->c.nx;
  for (size_t g = 0; g < s->ghosts.size(); ++g) {
    const IbmGhost& G = s->ghosts[g];
    if (cell) cell[g] = G.j * nx + G.i;
    for (int d = 0; d < 4; ++d) {
      if (donors) donors[4 * g + d] = G.dj[d] * nx + G.di[d];
      if (weights) weights[4 * g + d] = G.w[d];
    }
    if (normal) { normal[2 * g] = G.nx; normal[2 * g + 1] = G.ny; }
  }
  return (int)s->ghosts.size();
}

int jxo_cell_types(const jxo_solver* s, unsigned char* type) {
  if (!s || !type) return JXO_EINVAL;
  std::memcpy(type, s->type.data(), s->type.size());
  return JXO_OK;
}

long long jxo_guard_count(const jxo_solver* s) { return s ? s->guard : -1; }

int jxo_count_ops(jxo_solver* s, const double* U, long long counts[5]) {
  if (!s || !U || !counts) return JXO_EINVAL;
  const size_t n = (size_t)4 * s->c.nx * s->c.ny;
  std::vector<Counted> Uc(n), L(n);
  for (size_t i = 0; i < n; ++i) Uc[i] = Counted(U[i]);
  Core<Counted> core(s->c, s->type, s->ghosts, s->mlp);
  core.cnn = &s->cnn;
  std::vector<Counted> Up;
  core.pad(Uc.data(), Up);
  core.fill_frame(Up);
  core.fill_ibm(Up);
  g_tally = Tally();
  core.rhs(Up, L.data());
  // one RK combine of the general form a*U0 + b*(U + dt*L)
  const Counted a(0.75), b(0.25), dt(1e-3);
  for (size_t i = 0; i < n; ++i) Uc[i] = a * Uc[i] + b * (Uc[i] + dt * L[i]);
  // the wavespeed reduction
  (void)core.max_wavespeed(Up);
  counts[0] = g_tally.add; counts[1] = g_tally.mul; counts[2] = g_tally.div;
  counts[3] = g_tally.sqrt_; counts[4] = g_tally.cmp;
  return JXO_OK;
}

int jxo_set_flux_cnn(jxo_solver* s, const float* w, const double in_scale[4], const double out_scale[4],
                     int emulate_bf16) {
  if (!s) return JXO_EINVAL;
  if (!w) { s->cnn.on = false; return JXO_OK; }
  if (!in_scale || !out_scale) return JXO_EINVAL;
  for (int i = 0; i < 6388; ++i)
    if (!std::isfinite(w[i])) return JXO_EINVAL;
  for (int k = 0; k < 4; ++k)
    if (!(in_scale[k] > 0)) return JXO_EINVAL;
  Cnn& m = s->cnn;
  m.bf16 = emulate_bf16 != 0;
  auto take = [&](std::vector<double>& dst, size_t n, bool round) {
    dst.resize(n);
    for (size_t i = 0; i < n; ++i) dst[i] = round && m.bf16 ? bf16_round((double)w[i]) : (double)w[i];
    w += n;
  };
  // PyTorch / JAX OIHW order: W1[32][4][3][3], b1[32], W2[16][32][3][3], b2[16], W3[4][16][3][3], b3[4]
  take(m.W1, 32 * 4 * 9, true); take(m.b1, 32, false);
  take(m.W2, 16 * 32 * 9, true); take(m.b2, 16, false);
  take(m.W3, 4 * 16 * 9, true); take(m.b3, 4, false);
  for (int k = 0; k < 4; ++k) { m.in_scale[k] = in_scale[k]; m.out_scale[k] = out_scale[k]; }
  m.on = true;
  return JXO_OK;
}

int jxo_cnn_fields(jxo_solver* s, const double* U, double* Xx, double* Xy, double* Yx, double* Yy) {
  if (!s || !s->cnn.on || s->dtype != JXO_F64 || !U || !Xx || !Xy || !Yx || !Yy) return JXO_ESTATE;
  Core<double> core(s->c, s->type, s->ghosts, s->mlp);
  core.cnn = &s->cnn;
  std::vector<double> f[4], Up, L((size_t)4 * s->c.nx * s->c.ny);
  for (int q = 0; q < 4; ++q) core.cap[q] = &f[q];
  core.pad(U, Up);
  core.fill_and_rhs(Up, L.data());
  double* out[4] = {Xx, Xy, Yx, Yy};
  for (int q = 0; q < 4; ++q) std::copy(f[q].begin(), f[q].end(), out[q]);
  return JXO_OK;
}

int jxo_cnn_apply(const jxo_solver* s, const double* in, int na, int nb, double* out) {
  if (!s || !s->cnn.on || !in || !out || na < 1 || nb < 1) return JXO_ESTATE;
  std::vector<double> x(in, in + (size_t)4 * na * nb), y;
  s->cnn.apply(x, na, nb, y);
  std::copy(y.begin(), y.end(), out);
  return JXO_OK;
}

int jxo_mlp_eval(const jxo_solver* s, const double x[24], double y[4]) {
  if (!s || !s->mlp.on) return JXO_ESTATE;
  s->mlp.eval(x, y);
  return JXO_OK;
}

}  // extern "C"
