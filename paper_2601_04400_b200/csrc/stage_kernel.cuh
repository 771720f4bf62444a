// stage_kernel.cuh — the fused Runge-Kutta-stage kernel (S3-S9 of DESIGN.md §1) for sm_100a.
//
// Work decomposition: the grid is cut into column strips of 32 cells, one per
// WARP and one cell per LANE, and each strip into row segments.  A warp marches its strip upwards
// one row per iteration, completely independently of every other warp (no block-level barrier
// exists in this kernel; the CTA is only a container of 4 warps):
//   * rows of conserved variables arrive in shared memory by TMA bulk copies (cp.async.bulk +
//     mbarrier), the next row in flight while the current one is used; the Runge-Kutta operands
//     of the output row (U_in and U^n) arrive the same way one iteration ahead, so the row loop
//     holds no global load;
//   * a row is converted to primitives (+ temperature) once and kept in a 5-row per-warp ring;
//   * WENO5 is evaluated in CELL-CENTRED form: the smoothness indicators of a cell are computed
//     once and give both the left state of its upper face and the right state of its lower face
//     (y from the ring's 5 rows, x from the 5-cell row window of the lane);
//   * every face flux is computed exactly once: y-face fluxes are carried in registers from one
//     iteration to the next, x-face fluxes are exchanged between neighbouring lanes with warp
//     shuffles; lanes 0 and 31 are support cells recomputed by the neighbouring strip with
//     identical arithmetic (so conservation holds to round-off);
//   * viscous fluxes are subtracted from the inviscid ones at the face; the divergence, the
//     Runge-Kutta combine and (last stage) the wavespeed of the new state are fused behind.
// Neither reconstructed states nor fluxes ever leave the SM.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace jxs {

constexpr int LW = 32;           // cells per warp strip (1 per lane)
constexpr int CW = LW + 4;       // + 2 halo cells per side
constexpr int RING = 5;          // rows of primitives kept per warp
constexpr int STAGE_WARPS = 1;   // one warp per CTA: everything derived from blockIdx is warp-uniform

template <typename T> struct Cfg;
// output cells per strip = lanes 1..SOUT; strips must start on 16-byte boundaries (TMA)
template <> struct Cfg<double> { static constexpr int SOUT = 30; };
template <> struct Cfg<float> { static constexpr int SOUT = 28; };

template <typename T>
struct StageArgs {
  const T* Uin;          // padded [4][ny+6][pitch], ghosts filled
  const T* U0;           // padded, U^n of the step (read only when rk_a != 0)
  T* Uout;               // mode 0: padded; mode 1: interior [4][ny][nx] (dUdt)
  const uint8_t* fluid;  // [ny][nx], 1 = fluid; nullptr = all fluid
  const double* dt;      // device scalar
  unsigned long long* smax_bits;  // non-null: atomicMax of the wavespeed of the new state
  long long plane;       // (ny+6)*pitch
  int nx, ny, pitch;
  int nstrips, rows_per_seg, ntasks;
  int mode;
  T gamma, g1, g1inv, dxi, dyi, mu, kappa, nu;
  T rk_a, rk_b;          // Uout = a*U0 + b*(Uin + dt*L)
  // Literals that are not exact in the upper 32 bits of a double cannot be SASS immediates; as
  // kernel parameters they are constant-bank operands (no registers, no moves).
  T c133, eps4, sixth;  // 13/3, 4e-6, 1/6
  // viscous-flux coefficients with mu, kappa, the grid spacings and the 1/4 of the averaged tangential
  // derivative folded in (R8): normal stress, cross derivative in the normal stress, shear (normal and
  // tangential part), heat flux; n = the face's normal direction
  T vy_n, vy_c, vy_s, vy_t, vy_q;  // y-faces: 4/3 mu/dy, (2/3) mu/(4 dx), mu/dy, mu/(4 dx), kappa/dy
  T vx_n, vx_c, vx_s, vx_t, vx_q;  // x-faces: 4/3 mu/dx, (2/3) mu/(4 dy), mu/dx, mu/(4 dy), kappa/dx
  // S5' (optional): network outputs y per face from flux_mlp_kernel, padded indexing [4][ny+6][pitch]:
  // dF = right face, dG = top face of the cell; k = (mass, normal, tangential momentum, energy) (R14)
  const float* dF;
  const float* dG;
  T oscale[4];
};


// ------------------------------------------------------------------ small PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void tma_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  } while (!ok);
}

// one lane of the (converged) warp, chosen by the hardware: ptxas then keeps the bulk copies on the
// uniform datapath instead of looping over "every active lane"
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(pred));
  return pred != 0;
}

// ------------------------------------------------------------------ scalar helpers
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double min_(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float min_(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double max_(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double abs_(double a) { return fabs(a); }
__device__ __forceinline__ float abs_(float a) { return fabsf(a); }
// Branch-free reciprocal and reciprocal square root.  MUFU.RCP64H / MUFU.RSQ64H are accurate to
// 2^-20 (measured on B200), so ONE cubic Newton step reaches 1 ulp (max rel. error 2.2e-16 /
// 2.7e-16 measured over 2^26 arguments).  No slow path: arguments here are densities, pressures,
// wave-speed differences and WENO denominators, all normal and far from the range limits.
__device__ __forceinline__ double rcp_(double b) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
  double e = fma(-b, r, 1.0);
  e = fma(e, e, e);
  return fma(r, e, r);
}
__device__ __forceinline__ float rcp_(float b) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(b));
  return r;
}
__device__ __forceinline__ double rsqrt_(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double f = fma(-(0.5 * x) * y, y, 0.5);
  return fma(y, f * fma(1.5, f, 1.0), y);
}
__device__ __forceinline__ float rsqrt_(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// !(x > 0) on the integer pipe (the FP64 pipe is the bottleneck): true for x <= 0 and NaN
__device__ __forceinline__ bool not_positive(double x) {
  return (unsigned long long)(__double_as_longlong(x) - 1ll) >= 0x7FF0000000000000ull;
}
__device__ __forceinline__ bool not_positive(float x) {
  return (unsigned)(__float_as_int(x) - 1) >= 0x7F800000u;
}

// ------------------------------------------------------------------ S4: WENO5-JS, cell-centred
// (a,b,c,d,e) = v[i-2..i+2].  vm = right-biased value at i-1/2, vp = left-biased value at i+1/2.
// Same scheme as the paper's (L46; eps 1e-6, weights .1/.6/.3, R4), rearranged for the FP64 pipe:
// first differences, smoothness indicators scaled by 4 (Bk = 4(beta_k + eps)), the un-normalised
// weights multiplied through by (B0 B1 B2)^2 so that each side needs ONE reciprocal, and the
// candidate values taken relative to the central one q1:
//   vp = q1 + [ P12 (q0-q1) + 3 P01 (q2-q1) ] / [P12 + 6 P02 + 3 P01],   Pjk = (Bj Bk)^2,
//   q0-q1 = (s0-s1)/3,  q2-q1 = (s1-s2)/6,  q1 = c + (d2 + 2 d3)/6   (sk = second differences)
// and the mirror image for vm; with A = P12 (s0-s1), C = P01 (s1-s2) everything is in sixths.
template <typename T>
__device__ __forceinline__ void weno5_cell(T a, T b, T c, T d, T e, const StageArgs<T>& K, T& vm, T& vp) {
  const T d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  const T s0 = d2 - d1, s1 = d3 - d2, s2 = d4 - d3;
  const T t0 = fma_(T(3), d2, -d1), t1 = d2 + d3, t2 = fma_(T(-3), d3, d4);
  const T B0 = fma_(K.c133 * s0, s0, fma_(t0, t0, K.eps4));
  const T B1 = fma_(K.c133 * s1, s1, fma_(t1, t1, K.eps4));
  const T B2 = fma_(K.c133 * s2, s2, fma_(t2, t2, K.eps4));
  const T D0 = B0 * B0, D1 = B1 * B1, D2 = B2 * B2;
  const T P12 = D1 * D2, P02 = D0 * D2, P01 = D0 * D1;
  const T h = fma_(T(6), P02, P12 + P01);
  const T denp = fma_(T(2), P01, h), denm = fma_(T(2), P12, h);
  const T A = P12 * (s0 - s1), C = P01 * (s1 - s2);
  // 6 (vp - c) = (d2 + 2 d3) + (2A + 3C)/denp,   6 (c - vm) = (d3 + 2 d2) + (2C + 3A)/denm
  const T S = A + C;
  const T np = fma_(T(2), S, C), nm = fma_(T(2), S, A);
  T rp, rm;
  if (sizeof(T) == 8) {  // one reciprocal for both sides (the product stays far inside the fp64 range)
    const T r = rcp_(denp * denm);
    rp = r * denm; rm = r * denp;
  } else {
    rp = rcp_(denp); rm = rcp_(denm);
  }
  const T ep = fma_(np, rp, fma_(T(2), d3, d2));
  const T em = fma_(nm, rm, fma_(T(2), d2, d3));
  vp = fma_(K.sixth, ep, c);
  vm = fma_(-K.sixth, em, c);
}

// ------------------------------------------------------------------ S5: HLLC, one-sided
// Normal velocity un, tangential ut.  Eq. 3-7 with the star state of reading R1; for s* != 0 the
// sign blend of Eq. 3 is exact branch selection, at s* = 0 the left branch is taken (R2).
// Returns (mass, normal momentum, tangential momentum, energy) flux.
template <typename T>
__device__ __forceinline__ void hllc(T rL, T unL, T utL, T pL, T rR, T unR, T utR, T pR, T gamma, T g1inv,
                                     T& f0, T& f1, T& f2, T& f3) {
  // a = sqrt(gamma p / rho) = (gamma p) * rsqrt(gamma p rho)
  const T gpL = gamma * pL, gpR = gamma * pR;
  const T aL = gpL * rsqrt_(gpL * rL), aR = gpR * rsqrt_(gpR * rR);
  const T sL = min_(unL - aL, unR - aR), sR = max_(unL + aL, unR + aR);  // Eq. 6
  const T mL = rL * (sL - unL), mR = rR * (sR - unR);
  const T sS = fma_(mL, unL, fma_(-mR, unR, pR - pL)) * rcp_(mL - mR);    // Eq. 7
  const bool left = !(sS < T(0));
  const T r = left ? rL : rR, un = left ? unL : unR, ut = left ? utL : utR, p = left ? pL : pR;
  const T sk = left ? sL : sR;
  const T sc = left ? min_(T(0), sL) : max_(T(0), sR);                    // Eq. 5
  const T E = fma_(T(0.5) * r, fma_(un, un, ut * ut), p * g1inv);
  const T ru = r * un;
  const T rinv = rcp_(sk - sS);
  const T chi = (sk - un) * rinv;
  const T rchi = r * chi;
  const T dm = fma_(r, chi, -r);                                 // rho* - rho
  const T dn = fma_(rchi, sS, -ru);                              // (rho u)* - rho u
  const T dt_ = ut * dm;                                         // (rho v)* - rho v
  const T dE = fma_(sS - un, fma_(rchi, sS, p * rinv), fma_(chi, E, -E));  // E* - E
  f0 = fma_(sc, dm, ru);
  f1 = fma_(sc, dn, fma_(ru, un, p));
  f2 = fma_(sc, dt_, ru * ut);
  f3 = fma_(sc, dE, un * (E + p));
}

template <typename T>
__device__ __forceinline__ T shfl_down1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }
template <typename T>
__device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

__device__ __forceinline__ void atomic_max_pos(unsigned long long* addr, double v) {
  // v >= 0 (or NaN, whose bit pattern compares above +inf): unsigned order == numeric order
  atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

// Runge-Kutta operand rows: fp64 strips start on even columns, so the 32 owned columns can be
// fetched alone (16-byte aligned); fp32 fetches the CW-wide window like the raw rows.
template <typename T> struct Epi { static constexpr int W = sizeof(T) == 8 ? LW : CW, OFF = sizeof(T) == 8 ? 0 : 2; };
// per-warp shared memory: ring [RING][NV][CW] | raw row [4][CW] | RK operands [2][4][Epi::W] | 2 mbarriers
template <typename T, int NV>
__host__ __device__ constexpr size_t stage_smem_per_warp() {
  return (size_t)((RING * NV + 4) * CW + 8 * Epi<T>::W) * sizeof(T) + 16;
}

// ------------------------------------------------------------------ the kernel
template <typename T, bool VISC, bool ARTV, bool MLP, int MINB>
__global__ void __launch_bounds__(STAGE_WARPS * 32, MINB) stage_kernel(const StageArgs<T> A) {
  constexpr int SOUT = Cfg<T>::SOUT;
  constexpr int NV = VISC ? 5 : 4;
  extern __shared__ __align__(16) unsigned char smem_raw[];

  constexpr int EW = Epi<T>::W, EOFF = Epi<T>::OFF;
  const int lane = threadIdx.x;
  const int task = blockIdx.x;
  const int strip = task % A.nstrips, seg = task / A.nstrips;
  const int jbeg = 3 + seg * A.rows_per_seg;             // first output row (padded index)
  const int jend = min(jbeg + A.rows_per_seg, 3 + A.ny);  // one past the last
  if (jbeg >= jend) return;
  const int w0 = 2 + SOUT * strip;  // padded column of lane 0's cell
  const int ic = w0 + lane - 3;     // interior x index of my cell
  const int q = lane + 2;           // my column inside the per-warp rows

  T* ring = reinterpret_cast<T*>(smem_raw);  // [RING][NV][CW]
  T* raw = ring + RING * NV * CW;            // [4][CW]
  T* epi = raw + 4 * CW;                     // [2][4][EW]
  const uint32_t bar_raw = smem_u32(epi + 8 * EW), bar_epi = bar_raw + 8;
  const uint32_t raw_u32 = smem_u32(raw), epi_u32 = smem_u32(epi);
  constexpr uint32_t ROWB = CW * sizeof(T), EROWB = EW * sizeof(T);

  if (lane == 0) {
    mbar_init(bar_raw, 1);
    mbar_init(bar_epi, 1);
    mbar_fence_init();
  }
  __syncwarp();

  const int nfirst = jbeg - 3, nlast = jend + 2;  // rows to stream, inclusive
  const bool use_u0 = A.rk_a != T(0);
  const size_t soff = (size_t)(w0 - 2);
  auto issue_row = [&](int n) {  // lane 0 only: conserved row n -> raw
    mbar_expect_tx(bar_raw, 4 * ROWB);
    const T* s = A.Uin + soff + (size_t)n * A.pitch;
#pragma unroll
    for (int k = 0; k < 4; ++k) tma_bulk_g2s(raw_u32 + k * ROWB, s + k * A.plane, ROWB, bar_raw);
  };
  auto issue_epi = [&](int j) {  // lane 0 only: Runge-Kutta operands of output row j -> epi
    mbar_expect_tx(bar_epi, (use_u0 ? 8 : 4) * EROWB);
    const size_t o = (size_t)(w0 - EOFF) + (size_t)j * A.pitch;
#pragma unroll
    for (int k = 0; k < 4; ++k) tma_bulk_g2s(epi_u32 + k * EROWB, A.Uin + o + k * A.plane, EROWB, bar_epi);
    if (use_u0) {
#pragma unroll
      for (int k = 0; k < 4; ++k) tma_bulk_g2s(epi_u32 + (4 + k) * EROWB, A.U0 + o + k * A.plane, EROWB, bar_epi);
    }
  };
  if (elect_one()) issue_row(nfirst);

  const T gamma = A.gamma, g1inv = A.g1inv, g1 = A.g1;
  const T dtv = T(*A.dt);

  // state carried from one row to the next
  T Ly[4];  // left state (rho,u,v,p) at the face below the next centre row
  T Gp[4];  // total y-flux (rho, rho u, rho v, E) through the face below the output row
#pragma unroll
  for (int k = 0; k < 4; ++k) { Ly[k] = T(0); Gp[k] = T(0); }
  T cuP = T(0), cvP = T(0);
  T smax = T(0);
  unsigned fl_next = 1;  // fluid flag of my cell in the next output row, fetched one iteration ahead

  // Ring rows as loop-carried per-lane pointers (to my column q), rotated once per iteration: the row
  // accesses below become LDS with immediate offsets, no slot arithmetic.  pN = slot written next.
  T* pN = ring + q;
  const T *pA = ring + 1 * NV * CW + q, *pB = ring + 2 * NV * CW + q, *pC = ring + 3 * NV * CW + q,
          *pD = ring + 4 * NV * CW + q;
  const int hoff = lane < 2 ? -2 : LW - 2;  // my halo column (lanes 0-3 convert one each), relative to q
  for (int n = nfirst; n <= nlast; ++n) {
    const int it = n - nfirst;
    // ---------------------------------------------------------------- S3: new row -> primitives
    __syncwarp();  // every lane is done reading the ring slot that is overwritten now
    mbar_wait(bar_raw, it & 1);
    {
      auto convert = [&](int o) {  // o = column relative to q
        const T* src = raw + q + o;
        const T r = src[0], ru = src[CW], rv = src[2 * CW], E = src[3 * CW];
        const T ri = rcp_(r);
        const T u = ru * ri, v = rv * ri;
        const T p = g1 * fma_(T(-0.5), fma_(ru, u, rv * v), E);
        T* dst = pN + o;
        dst[0] = r;
        dst[CW] = u;
        dst[2 * CW] = v;
        dst[3 * CW] = p;
        if (VISC) dst[4 * CW] = p * ri;
      };
      convert(0);
      if (lane < 4) convert(hoff);
      __syncwarp();
      if (n < nlast && elect_one()) issue_row(n + 1);
    }
    // ring rows n-4 .. n  (valid once it >= 4): A = n-4, B = n-3 = jo (output row), C = n-2 = jc
    // (centre of the y stencil), D = n-1, E = n
    const T *rowA = pA - q, *rowB = pB - q, *rowC = pC - q, *rowD = pD - q, *rowE = pN - q;
    {
      T* const oldest = const_cast<T*>(pA);
      pA = pB; pB = pC; pC = pD; pD = pN; pN = oldest;
    }
    if (it < 4) continue;

    const int jo = n - 3;
    const bool do_out = it >= 6;  // rows jo >= jbeg
    const unsigned fl = fl_next;
    if (it >= 5 && n < nlast && A.fluid && ic < A.nx) fl_next = A.fluid[(size_t)(jo + 1 - 3) * A.nx + ic];
    float yF[4], yG[4];  // S5': network outputs at my right face and my top face (row jo)
    if (MLP && it >= 5) {
      const size_t o = (size_t)jo * A.pitch + (w0 + lane);
#pragma unroll
      for (int k = 0; k < 4; ++k) { yF[k] = __ldg(A.dF + k * A.plane + o); yG[k] = __ldg(A.dG + k * A.plane + o); }
    }

    // ---------------------------------------------------------------- S4/S5 along y
    T Ly_div[4];  // G_bottom - G_top of the output row, per component
    {
      T Ry[4], Lnew[4];
#pragma unroll
      for (int k = 0; k < 4; ++k)
        weno5_cell(rowA[k * CW + q], rowB[k * CW + q], rowC[k * CW + q], rowD[k * CW + q], rowE[k * CW + q], A, Ry[k],
                   Lnew[k]);
      // positivity guard (R15): a side with rho <= 0 or p <= 0 falls back to its cell (row jc);
      // one warp vote keeps the (never taken in practice) repair off the common path
      const bool badR = not_positive(Ry[0]) | not_positive(Ry[3]);
      const bool badL = not_positive(Lnew[0]) | not_positive(Lnew[3]);
      if (__any_sync(0xffffffffu, badR | badL)) {
        asm volatile("" ::: "memory");  // keeps this (never taken in practice) block a branch, not 16 selects
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const T cv = rowC[k * CW + q];
          Ry[k] = badR ? cv : Ry[k];
          Lnew[k] = badL ? cv : Lnew[k];
        }
      }
      T cuC, cvC;  // x-centred differences of u, v in row jc; cuP, cvP: the same for row jo (carried)
      if (VISC) {
        cuC = rowC[CW + q + 1] - rowC[CW + q - 1];
        cvC = rowC[2 * CW + q + 1] - rowC[2 * CW + q - 1];
      }
      if (it >= 5) {
        T f0, f1, f2, f3;  // face between rows jo and jc: normal = y
        hllc(Ly[0], Ly[2], Ly[1], Ly[3], Ry[0], Ry[2], Ry[1], Ry[3], gamma, g1inv, f0, f1, f2, f3);
        T G[4] = {f0, f2, f1, f3};
        if (MLP) {  // Eq. 11: normal momentum of a y-face is rho*v
          G[0] = fma_(A.oscale[0], T(yG[0]), G[0]); G[1] = fma_(A.oscale[2], T(yG[2]), G[1]);
          G[2] = fma_(A.oscale[1], T(yG[1]), G[2]); G[3] = fma_(A.oscale[3], T(yG[3]), G[3]);
        }
        if (VISC) {  // S6 (R8): G^v = (0, tau_xy, tau_yy, u tau_xy + v tau_yy + k T_y)
          const T uB = rowB[CW + q], uC = rowC[CW + q], vB = rowB[2 * CW + q], vC = rowC[2 * CW + q];
          const T dT = rowC[4 * CW + q] - rowB[4 * CW + q];
          const T tyy = fma_(A.vy_n, vC - vB, -(A.vy_c * (cuP + cuC)));
          const T txy = fma_(A.vy_s, uC - uB, A.vy_t * (cvP + cvC));
          G[1] -= txy;
          G[2] -= tyy;
          const T w = fma_(vB + vC, tyy, (uB + uC) * txy);  // 2 (u tau_xy + v tau_yy) at the face
          G[3] = fma_(-A.vy_q, dT, fma_(T(-0.5), w, G[3]));
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) { Ly_div[k] = Gp[k] - G[k]; Gp[k] = G[k]; }
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) Ly[k] = Lnew[k];
      if (VISC) { cuP = cuC; cvP = cvC; }
    }

    if (do_out) {
      // -------------------------------------------------------------- S4/S5 along x, row jo
      T F[4];   // total x-flux through my right face i+1/2
      T wc[4];  // my primitives
      {
        T Rm[4], Lp[4];  // right state at my left face, left state at my right face
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const T* r = rowB + k * CW + q;
          wc[k] = r[0];
          weno5_cell(r[-2], r[-1], r[0], r[1], r[2], A, Rm[k], Lp[k]);
        }
        const bool badR = not_positive(Rm[0]) | not_positive(Rm[3]);
        const bool badL = not_positive(Lp[0]) | not_positive(Lp[3]);
        if (__any_sync(0xffffffffu, badR | badL)) {
          asm volatile("" ::: "memory");
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            Rm[k] = badR ? wc[k] : Rm[k];
            Lp[k] = badL ? wc[k] : Lp[k];
          }
        }
        const T r0 = shfl_down1(Rm[0]), r1 = shfl_down1(Rm[1]), r2 = shfl_down1(Rm[2]), r3 = shfl_down1(Rm[3]);
        hllc(Lp[0], Lp[1], Lp[2], Lp[3], r0, r1, r2, r3, gamma, g1inv, F[0], F[1], F[2], F[3]);
        if (MLP) {
#pragma unroll
          for (int k = 0; k < 4; ++k) F[k] = fma_(A.oscale[k], T(yF[k]), F[k]);  // Eq. 11
        }
      }
      if (VISC) {  // S6 (R8): F^v = (0, tau_xx, tau_xy, u tau_xx + v tau_xy + k T_x) at my right face
        const T u1 = rowB[CW + q + 1], v1 = rowB[2 * CW + q + 1];
        const T dT = rowB[4 * CW + q + 1] - rowB[4 * CW + q];
        // y-centred differences (rows jo+1 = jc and jo-1) at my cell; the right neighbour's come by shuffle
        // (lane 31 gets its own back: its face flux is not used)
        const T cu0 = rowC[CW + q] - rowA[CW + q], cv0 = rowC[2 * CW + q] - rowA[2 * CW + q];
        const T cu1 = shfl_down1(cu0), cv1 = shfl_down1(cv0);
        const T txx = fma_(A.vx_n, u1 - wc[1], -(A.vx_c * (cv0 + cv1)));
        const T txy = fma_(A.vx_s, v1 - wc[2], A.vx_t * (cu0 + cu1));
        F[1] -= txx;
        F[2] -= txy;
        const T w = fma_(wc[2] + v1, txy, (wc[1] + u1) * txx);
        F[3] = fma_(-A.vx_q, dT, fma_(T(-0.5), w, F[3]));
      }

      // -------------------------------------------------------------- S7-S9: divergence, combine, store
      T Lc[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const T Fl = shfl_up1(F[k]);
        Lc[k] = fma_(Fl - F[k], A.dxi, Ly_div[k] * A.dyi);
      }
      if (ARTV) {  // nu * Lap_h(U) on the conserved variables (Eq. 10), rebuilt from the primitives
        auto cons = [&](const T* row, int c, T* U) {
          const T r = row[c], u = row[CW + c], v = row[2 * CW + c], p = row[3 * CW + c];
          U[0] = r; U[1] = r * u; U[2] = r * v; U[3] = fma_(T(0.5) * r, fma_(u, u, v * v), p * g1inv);
        };
        T Um[4], Uxm[4], Uxp[4], Ud[4], Uu[4];
        cons(rowB, q, Um); cons(rowB, q - 1, Uxm); cons(rowB, q + 1, Uxp); cons(rowA, q, Ud); cons(rowC, q, Uu);
        const T ax = A.nu * A.dxi * A.dxi, ay = A.nu * A.dyi * A.dyi;
#pragma unroll
        for (int k = 0; k < 4; ++k)
          Lc[k] += ax * (Uxp[k] - T(2) * Um[k] + Uxm[k]) + ay * (Uu[k] - T(2) * Um[k] + Ud[k]);
      }
      const bool ok = lane >= 1 && lane <= SOUT && ic < A.nx;  // lanes 0 and > SOUT are support cells
      if (A.mode == 1) {
        const size_t o = (size_t)(jo - 3) * A.nx + ic, pl = (size_t)A.nx * A.ny;
        if (ok) {
#pragma unroll
          for (int k = 0; k < 4; ++k) A.Uout[k * pl + o] = fl ? Lc[k] : T(0);
        }
      } else {
        mbar_wait(bar_epi, it & 1);
        const T dtf = fl ? dtv : T(0);  // non-fluid cells keep their state
        T Un[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          T v = fma_(dtf, Lc[k], epi[k * EW + lane + EOFF]);
          if (use_u0) v = fma_(A.rk_a, epi[(4 + k) * EW + lane + EOFF], A.rk_b * v);
          Un[k] = v;
        }
        if (ok) {
          T* o = A.Uout + (size_t)jo * A.pitch + (w0 + lane);
#pragma unroll
          for (int k = 0; k < 4; ++k) o[k * A.plane] = Un[k];
        }
        if (A.smax_bits) {  // S9 on the new state (it is U^n of the next step), fluid cells only
          const T ri = rcp_(Un[0]);
          const T u = Un[1] * ri, v = Un[2] * ri;
          const T p = g1 * fma_(T(-0.5), fma_(Un[1], u, Un[2] * v), Un[3]);
          const T gp = gamma * p;
          const T a = gp * rsqrt_(gp * Un[0]);
          const T s = max_(abs_(u), abs_(v)) + a;
          if (ok && fl) smax = (s > smax || s != s) ? s : smax;  // NaN propagates
        }
      }
    }
    // the Runge-Kutta operands of the next output row, one iteration ahead
    if (A.mode == 0 && it >= 5 && n < nlast) {
      __syncwarp();  // every lane has read epi
      if (elect_one()) issue_epi(jo + 1);
    }
  }
  if (A.smax_bits) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const T other = __shfl_xor_sync(0xffffffffu, smax, o);
      smax = (other > smax || other != other) ? other : smax;
    }
    if (lane == 0) atomic_max_pos(A.smax_bits, (double)smax);
  }
}

}  // namespace jxs
