// stage_kernel.cuh — the fused Runge-Kutta-stage kernel (S3-S9 of DESIGN.md §1) for sm_100a.
//
// Work decomposition: the grid is cut into column strips of 64 cells, one per
// WARP, and each strip into row segments.  A warp marches its strip upwards one row per
// iteration, completely independently of every other warp (no block-level barrier exists in
// this kernel).  Lane l owns the two adjacent columns w0+2l, w0+2l+1:
//   * rows of conserved variables arrive in shared memory by TMA bulk copies
//     (cp.async.bulk + mbarrier), two rows in flight;
//   * they are converted to primitives once and kept in a 5-row per-warp ring;
//   * WENO5 is evaluated in CELL-CENTRED form: the smoothness indicators of a cell are
//     computed once and give both the left state of its upper face and the right state of its
//     lower face (y from the ring's 5 rows, x from the 6-cell row window of the lane);
//   * every face flux is computed exactly once: y-face fluxes are carried in registers from
//     one iteration to the next, x-face fluxes are exchanged between neighbouring lanes with
//     warp shuffles; the strip's first and last column are support cells recomputed by the
//     neighbouring strip with identical arithmetic (so conservation holds to round-off);
//   * viscous fluxes are subtracted from the inviscid ones at the face, the divergence, the
//     Runge-Kutta combine and (last stage) the wavespeed of the new state are fused behind.
// Neither reconstructed states nor fluxes ever leave the SM.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace jxs {

constexpr int SW = 64;    // cells reconstructed per warp strip (2 per lane)
constexpr int CW = 68;    // + 2 halo cells per side
constexpr int RING = 5;   // rows of primitives kept per warp
constexpr int NSTG = 2;   // raw rows in flight

template <typename T> struct Cfg;
template <> struct Cfg<double> { using V2 = double2; static constexpr int SOUT = 62; };
// fp32: strips start on 16-byte boundaries only if the output width is a multiple of 4
template <> struct Cfg<float> { using V2 = float2; static constexpr int SOUT = 60; };

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

// ------------------------------------------------------------------ scalar helpers
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double min_(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float min_(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double max_(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double sqrt_(double a) { return sqrt(a); }
__device__ __forceinline__ float sqrt_(float a) { return sqrtf(a); }
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
__device__ __forceinline__ double2 mk2(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 mk2(float a, float b) { return make_float2(a, b); }

// ------------------------------------------------------------------ S4: WENO5-JS, cell-centred
// (a,b,c,d,e) = v[i-2..i+2].  vm = right-biased value at i-1/2, vp = left-biased value at i+1/2.
// Same scheme as the paper's (L46; eps 1e-6, weights .1/.6/.3, R4), rearranged: first differences,
// smoothness indicators scaled by 4, one common denominator per side:
//   vp = c + [P12 n0 + P02 n1 + P01 n2] / [P12 + 6 P02 + 3 P01],   Pjk = (Bj Bk)^2
template <typename T>
__device__ __forceinline__ void weno5_cell(T a, T b, T c, T d, T e, T& vm, T& vp) {
  const T d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  const T s0 = d2 - d1, s1 = d3 - d2, s2 = d4 - d3;
  const T t0 = fma_(T(3), d2, -d1), t1 = d2 + d3, t2 = fma_(T(-3), d3, d4);
  const T eps4 = T(4e-6), c133 = T(13.0 / 3.0);
  const T B0 = fma_(c133 * s0, s0, fma_(t0, t0, eps4));
  const T B1 = fma_(c133 * s1, s1, fma_(t1, t1, eps4));
  const T B2 = fma_(c133 * s2, s2, fma_(t2, t2, eps4));
  const T D0 = B0 * B0, D1 = B1 * B1, D2 = B2 * B2;
  const T P12 = D1 * D2, P02 = D0 * D2, P01 = D0 * D1;
  // left-biased at i+1/2: sub-stencil values minus c, times (6 d_k / 6)
  const T n0 = fma_(T(5.0 / 6.0), d2, T(-1.0 / 3.0) * d1);
  const T n1 = fma_(T(2), d3, d2);
  const T n2 = fma_(T(2), d3, T(-0.5) * d4);
  const T nump = fma_(P12, n0, fma_(P02, n1, P01 * n2));
  const T denp = fma_(T(3), P01, fma_(T(6), P02, P12));
  // right-biased at i-1/2: the mirror image
  const T m0 = fma_(T(-5.0 / 6.0), d3, T(1.0 / 3.0) * d4);
  const T m1 = -fma_(T(2), d2, d3);
  const T m2 = fma_(T(-2), d2, T(0.5) * d1);
  const T numm = fma_(P01, m0, fma_(P02, m1, P12 * m2));
  const T denm = fma_(T(3), P12, fma_(T(6), P02, P01));
  vp = fma_(nump, rcp_(denp), c);
  vm = fma_(numm, rcp_(denm), c);
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

template <int NV>
__host__ __device__ constexpr size_t stage_smem_per_warp(size_t elem) {
  return (size_t)(RING * NV + NSTG * 4) * CW * elem + 16;  // + NSTG mbarriers
}

// ------------------------------------------------------------------ the kernel
template <typename T, bool VISC, bool ARTV, int WARPS>
__global__ void __launch_bounds__(WARPS * 32) stage_kernel(const StageArgs<T> A) {
  using V2 = typename Cfg<T>::V2;
  constexpr int SOUT = Cfg<T>::SOUT;
  constexpr int NV = VISC ? 5 : 4;
  constexpr int ROWV = CW / 2;  // V2 per row
  extern __shared__ __align__(16) unsigned char smem_raw[];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int task = blockIdx.x * (blockDim.x >> 5) + warp;  // WARPS only bounds the block size
  if (task >= A.ntasks) return;  // warp-uniform
  const int strip = task % A.nstrips, seg = task / A.nstrips;
  const int jbeg = 3 + seg * A.rows_per_seg;             // first output row (padded index)
  const int jend = min(jbeg + A.rows_per_seg, 3 + A.ny);  // one past the last
  if (jbeg >= jend) return;
  const int w0 = 2 + SOUT * strip;  // padded column of lane 0's first cell (even)
  const int c0 = w0 + 2 * lane;     // my first column

  unsigned char* wbase = smem_raw + (size_t)warp * stage_smem_per_warp<NV>(sizeof(T));
  V2* ring = reinterpret_cast<V2*>(wbase);                                  // [RING][NV][ROWV]
  V2* stg = ring + RING * NV * ROWV;                                        // [NSTG][4][ROWV]
  const uint32_t bar0 = smem_u32(stg + NSTG * 4 * ROWV);                    // NSTG x 8 bytes
  const uint32_t stg_u32 = smem_u32(stg);
  constexpr uint32_t ROWB = CW * sizeof(T);

  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < NSTG; ++s) mbar_init(bar0 + 8 * s, 1);
    mbar_fence_init();
  }
  __syncwarp();

  const int nfirst = jbeg - 3, nlast = jend + 2;  // rows to stream, inclusive
  const T* src0 = A.Uin + (size_t)(w0 - 2);
  auto issue_row = [&](int n) {  // lane 0 only
    const int s = (n - nfirst) % NSTG;
    mbar_expect_tx(bar0 + 8 * s, 4 * ROWB);
#pragma unroll
    for (int k = 0; k < 4; ++k)
      tma_bulk_g2s(stg_u32 + (s * 4 + k) * ROWB, src0 + k * A.plane + (size_t)n * A.pitch, ROWB, bar0 + 8 * s);
  };
  if (lane == 0) {
    issue_row(nfirst);
    if (nfirst + 1 <= nlast) issue_row(nfirst + 1);
  }

  const T gamma = A.gamma, g1inv = A.g1inv, g1 = A.g1;
  const T dtv = T(*A.dt);

  // state carried from one row to the next (per owned cell e = 0,1)
  T Ly[4][2];  // left state (rho,u,v,p) at the face below the next centre row
  T Gp[4][2];  // total y-flux (rho, rho u, rho v, E) through the face below the output row
  T cdx_u[2], cdx_v[2];  // x-centred differences of u, v at the previous centre row (viscous)
#pragma unroll
  for (int k = 0; k < 4; ++k) { Ly[k][0] = Ly[k][1] = T(0); Gp[k][0] = Gp[k][1] = T(0); }
  cdx_u[0] = cdx_u[1] = cdx_v[0] = cdx_v[1] = T(0);
  T smax = T(0);

  int slot = 0;  // ring slot of the newest row
  for (int n = nfirst; n <= nlast; ++n) {
    const int it = n - nfirst;
    // ---------------------------------------------------------------- S3: new row -> primitives
    {
      const int s = it % NSTG;
      mbar_wait(bar0 + 8 * s, (it / NSTG) & 1);
      const V2* raw = stg + s * 4 * ROWV;
      V2* dst = ring + slot * NV * ROWV;
      auto convert = [&](int q) {
        const V2 r = raw[q], ru = raw[ROWV + q], rv = raw[2 * ROWV + q], E = raw[3 * ROWV + q];
        const T i0 = rcp_(r.x), i1 = rcp_(r.y);
        const T u0 = ru.x * i0, u1 = ru.y * i1, v0 = rv.x * i0, v1 = rv.y * i1;
        const T p0 = g1 * fma_(T(-0.5), fma_(ru.x, u0, rv.x * v0), E.x);
        const T p1 = g1 * fma_(T(-0.5), fma_(ru.y, u1, rv.y * v1), E.y);
        dst[q] = r;
        dst[ROWV + q] = mk2(u0, u1);
        dst[2 * ROWV + q] = mk2(v0, v1);
        dst[3 * ROWV + q] = mk2(p0, p1);
        if (VISC) dst[4 * ROWV + q] = mk2(p0 * i0, p1 * i1);
      };
      convert(lane + 1);
      if (lane < 2) convert(lane == 0 ? 0 : ROWV - 1);
      __syncwarp();
      if (lane == 0 && n + NSTG <= nlast) issue_row(n + NSTG);
    }
    // ring slots of rows n-4 .. n  (valid once it >= 4)
    int sl[5];
#pragma unroll
    for (int d = 0; d < 5; ++d) { int t = slot - d; sl[d] = t < 0 ? t + RING : t; }
    const V2* rowE = ring + sl[0] * NV * ROWV;  // n
    const V2* rowD = ring + sl[1] * NV * ROWV;  // n-1
    const V2* rowC = ring + sl[2] * NV * ROWV;  // n-2 = jc (centre of the y stencil)
    const V2* rowB = ring + sl[3] * NV * ROWV;  // n-3 = jo (output row)
    const V2* rowA = ring + sl[4] * NV * ROWV;  // n-4
    slot = slot + 1 == RING ? 0 : slot + 1;
    if (it < 4) continue;

    // issue the global loads the epilogue needs early (L2 hits: this warp streamed the row)
    const int jo = n - 3;
    const bool do_out = it >= 6;  // rows jo >= jbeg
    V2 uin[4], u0v[4];
    unsigned fl0 = 1, fl1 = 1;
    const int i0c = c0 - 3;  // interior x index of my first cell
    if (do_out) {
      const size_t o = (size_t)jo * A.pitch + c0;
#pragma unroll
      for (int k = 0; k < 4; ++k) uin[k] = *reinterpret_cast<const V2*>(A.Uin + k * A.plane + o);
      if (A.rk_a != T(0)) {
#pragma unroll
        for (int k = 0; k < 4; ++k) u0v[k] = *reinterpret_cast<const V2*>(A.U0 + k * A.plane + o);
      }
      if (A.fluid) {
        const size_t fo = (size_t)(jo - 3) * A.nx;
        if (i0c >= 0 && i0c < A.nx) fl0 = A.fluid[fo + i0c];
        if (i0c + 1 >= 0 && i0c + 1 < A.nx) fl1 = A.fluid[fo + i0c + 1];
      }
    }

    // ---------------------------------------------------------------- S4/S5 along y
    T Ry[4][2], Lnew[4][2];
    T cdy_u[2], cdy_v[2];  // W(jo+1) - W(jo-1) at my cells, for the x-face viscous fluxes
    T uB[2], vB[2], uC[2], vC[2];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const V2 a = rowA[k * ROWV + lane + 1], b = rowB[k * ROWV + lane + 1], c = rowC[k * ROWV + lane + 1],
               d = rowD[k * ROWV + lane + 1], e = rowE[k * ROWV + lane + 1];
      weno5_cell(a.x, b.x, c.x, d.x, e.x, Ry[k][0], Lnew[k][0]);
      weno5_cell(a.y, b.y, c.y, d.y, e.y, Ry[k][1], Lnew[k][1]);
      if (k == 1) { cdy_u[0] = c.x - a.x; cdy_u[1] = c.y - a.y; uB[0] = b.x; uB[1] = b.y; uC[0] = c.x; uC[1] = c.y; }
      if (k == 2) { cdy_v[0] = c.x - a.x; cdy_v[1] = c.y - a.y; vB[0] = b.x; vB[1] = b.y; vC[0] = c.x; vC[1] = c.y; }
    }
    // positivity guard (R15): a side with rho <= 0 or p <= 0 falls back to its cell (row jc)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const bool badR = !(Ry[0][e] > T(0)) || !(Ry[3][e] > T(0));
      const bool badL = !(Lnew[0][e] > T(0)) || !(Lnew[3][e] > T(0));
      if (badR || badL) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const V2 c = rowC[k * ROWV + lane + 1];
          const T cv = e == 0 ? c.x : c.y;
          if (badR) Ry[k][e] = cv;
          if (badL) Lnew[k][e] = cv;
        }
      }
    }
    // centred x differences at row jc for the y-face viscous flux
    T cdxu_c[2] = {T(0), T(0)}, cdxv_c[2] = {T(0), T(0)};
    if (VISC) {
      const V2 ul = rowC[ROWV + lane], ur = rowC[ROWV + lane + 2];
      const V2 vl = rowC[2 * ROWV + lane], vr = rowC[2 * ROWV + lane + 2];
      cdxu_c[0] = uC[1] - ul.y; cdxu_c[1] = ur.x - uC[0];
      cdxv_c[0] = vC[1] - vl.y; cdxv_c[1] = vr.x - vC[0];
    }
    T Ly_div[4][2];  // -(G_top - G_bottom) of the output row, per component
    if (it >= 5) {
      V2 Tb, Tc;
      if (VISC) { Tb = rowB[4 * ROWV + lane + 1]; Tc = rowC[4 * ROWV + lane + 1]; }
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        T f0, f1, f2, f3;  // face between rows jo and jc: normal = y
        hllc(Ly[0][e], Ly[2][e], Ly[1][e], Ly[3][e], Ry[0][e], Ry[2][e], Ry[1][e], Ry[3][e], gamma, g1inv,
             f0, f1, f2, f3);
        T G[4] = {f0, f2, f1, f3};
        if (VISC) {  // S6 (R8): G^v = (0, tau_xy, tau_yy, u tau_xy + v tau_yy + k T_y)
          const T uy = (uC[e] - uB[e]) * A.dyi, vy = (vC[e] - vB[e]) * A.dyi;
          const T Ty = ((e == 0 ? Tc.x : Tc.y) - (e == 0 ? Tb.x : Tb.y)) * A.dyi;
          const T ux = T(0.25) * (cdx_u[e] + cdxu_c[e]) * A.dxi, vx = T(0.25) * (cdx_v[e] + cdxv_c[e]) * A.dxi;
          const T tyy = A.mu * fma_(T(4.0 / 3.0), vy, T(-2.0 / 3.0) * ux);
          const T txy = A.mu * (uy + vx);
          const T ub = T(0.5) * (uB[e] + uC[e]), vb = T(0.5) * (vB[e] + vC[e]);
          G[1] -= txy;
          G[2] -= tyy;
          G[3] -= fma_(ub, txy, fma_(vb, tyy, A.kappa * Ty));
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) { Ly_div[k][e] = Gp[k][e] - G[k]; Gp[k][e] = G[k]; }
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) { Ly[k][0] = Lnew[k][0]; Ly[k][1] = Lnew[k][1]; }
    if (VISC) { cdx_u[0] = cdxu_c[0]; cdx_u[1] = cdxu_c[1]; cdx_v[0] = cdxv_c[0]; cdx_v[1] = cdxv_c[1]; }
    if (!do_out) continue;

    // ---------------------------------------------------------------- S4/S5 along x, row jo
    T Rm[4][2], Lp[4][2];  // right state at the cell's left face, left state at its right face
    T w2[4];               // primitives of the right neighbour cell (first cell of lane+1)
    T wl[4];               // primitives of the left neighbour cell
    T wc[4][2];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const V2 a = rowB[k * ROWV + lane], b = rowB[k * ROWV + lane + 1], c = rowB[k * ROWV + lane + 2];
      weno5_cell(a.x, a.y, b.x, b.y, c.x, Rm[k][0], Lp[k][0]);
      weno5_cell(a.y, b.x, b.y, c.x, c.y, Rm[k][1], Lp[k][1]);
      wc[k][0] = b.x; wc[k][1] = b.y; w2[k] = c.x; wl[k] = a.y;
    }
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const bool badR = !(Rm[0][e] > T(0)) || !(Rm[3][e] > T(0));
      const bool badL = !(Lp[0][e] > T(0)) || !(Lp[3][e] > T(0));
      if (badR || badL) {  // rare
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (badR) Rm[k][e] = wc[k][e];
          if (badL) Lp[k][e] = wc[k][e];
        }
      }
    }
    T Fa[4], Fb[4];
    hllc(Lp[0][0], Lp[1][0], Lp[2][0], Lp[3][0], Rm[0][1], Rm[1][1], Rm[2][1], Rm[3][1], gamma, g1inv,
         Fa[0], Fa[1], Fa[2], Fa[3]);
    {
      const T r0 = shfl_down1(Rm[0][0]), r1 = shfl_down1(Rm[1][0]), r2 = shfl_down1(Rm[2][0]),
              r3 = shfl_down1(Rm[3][0]);
      hllc(Lp[0][1], Lp[1][1], Lp[2][1], Lp[3][1], r0, r1, r2, r3, gamma, g1inv, Fb[0], Fb[1], Fb[2], Fb[3]);
    }
    if (VISC) {  // S6 (R8): F^v = (0, tau_xx, tau_xy, u tau_xx + v tau_xy + k T_x) at faces a and b
      const V2 Tq = rowB[4 * ROWV + lane + 1];
      const T T2 = rowB[4 * ROWV + lane + 2].x;
      // y-centred differences at the right neighbour cell (rows jo+1 = jc and jo-1)
      const T cu2 = rowC[ROWV + lane + 2].x - rowA[ROWV + lane + 2].x;
      const T cv2 = rowC[2 * ROWV + lane + 2].x - rowA[2 * ROWV + lane + 2].x;
      const T uu[3] = {wc[1][0], wc[1][1], w2[1]}, vv[3] = {wc[2][0], wc[2][1], w2[2]};
      const T TT[3] = {Tq.x, Tq.y, T2};
      const T cu[3] = {cdy_u[0], cdy_u[1], cu2}, cv[3] = {cdy_v[0], cdy_v[1], cv2};
#pragma unroll
      for (int f = 0; f < 2; ++f) {
        const T ux = (uu[f + 1] - uu[f]) * A.dxi, vx = (vv[f + 1] - vv[f]) * A.dxi;
        const T Tx = (TT[f + 1] - TT[f]) * A.dxi;
        const T uy = T(0.25) * (cu[f] + cu[f + 1]) * A.dyi, vy = T(0.25) * (cv[f] + cv[f + 1]) * A.dyi;
        const T txx = A.mu * fma_(T(4.0 / 3.0), ux, T(-2.0 / 3.0) * vy);
        const T txy = A.mu * (uy + vx);
        const T ub = T(0.5) * (uu[f] + uu[f + 1]), vb = T(0.5) * (vv[f] + vv[f + 1]);
        T* F = f == 0 ? Fa : Fb;
        F[1] -= txx;
        F[2] -= txy;
        F[3] -= fma_(ub, txx, fma_(vb, txy, A.kappa * Tx));
      }
    }
    T Fl[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) Fl[k] = shfl_up1(Fb[k]);

    // ---------------------------------------------------------------- S7-S9: divergence, combine, store
    T Lc[4][2];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      Lc[k][0] = fma_(Fl[k] - Fa[k], A.dxi, Ly_div[k][0] * A.dyi);
      Lc[k][1] = fma_(Fa[k] - Fb[k], A.dxi, Ly_div[k][1] * A.dyi);
    }
    if (ARTV) {  // nu * Lap_h(U) on the conserved variables (Eq. 10), rebuilt from the primitives
      auto cons = [&](T r, T u, T v, T p, T* U) {
        U[0] = r; U[1] = r * u; U[2] = r * v; U[3] = fma_(T(0.5) * r, fma_(u, u, v * v), p * g1inv);
      };
      T Ul[4], U0c[4], U1c[4], Ur[4], Ud[4], Uu[4];
      cons(wl[0], wl[1], wl[2], wl[3], Ul);
      cons(wc[0][0], wc[1][0], wc[2][0], wc[3][0], U0c);
      cons(wc[0][1], wc[1][1], wc[2][1], wc[3][1], U1c);
      cons(w2[0], w2[1], w2[2], w2[3], Ur);
      const T ax = A.nu * A.dxi * A.dxi, ay = A.nu * A.dyi * A.dyi;
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const V2 ra = rowA[lane + 1], ua = rowA[ROWV + lane + 1], va = rowA[2 * ROWV + lane + 1], pa = rowA[3 * ROWV + lane + 1];
        const V2 rc = rowC[lane + 1], uc = rowC[ROWV + lane + 1], vc = rowC[2 * ROWV + lane + 1], pc = rowC[3 * ROWV + lane + 1];
        cons(e ? ra.y : ra.x, e ? ua.y : ua.x, e ? va.y : va.x, e ? pa.y : pa.x, Ud);
        cons(e ? rc.y : rc.x, e ? uc.y : uc.x, e ? vc.y : vc.x, e ? pc.y : pc.x, Uu);
        const T* Um = e ? U1c : U0c;
        const T* Uxm = e ? U0c : Ul;
        const T* Uxp = e ? Ur : U1c;
#pragma unroll
        for (int k = 0; k < 4; ++k)
          Lc[k][e] += ax * (Uxp[k] - T(2) * Um[k] + Uxm[k]) + ay * (Uu[k] - T(2) * Um[k] + Ud[k]);
      }
    }
    const bool ok0 = lane >= 1 && i0c >= 0 && i0c < A.nx;                   // lane 0's first cell is support
    const bool ok1 = (2 * lane + 1 <= SOUT) && i0c + 1 >= 0 && i0c + 1 < A.nx;  // cells past w0+SOUT are support
    const bool ok0s = ok0 && (2 * lane <= SOUT);
    if (A.mode == 1) {
      const size_t o = (size_t)(jo - 3) * A.nx + i0c;
      const size_t pl = (size_t)A.nx * A.ny;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (ok0s) A.Uout[k * pl + o] = fl0 ? Lc[k][0] : T(0);
        if (ok1) A.Uout[k * pl + o + 1] = fl1 ? Lc[k][1] : T(0);
      }
    } else {
      T Un[4][2];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        T n0 = uin[k].x + (fl0 ? dtv * Lc[k][0] : T(0));
        T n1 = uin[k].y + (fl1 ? dtv * Lc[k][1] : T(0));
        if (A.rk_a != T(0)) {
          n0 = fma_(A.rk_a, u0v[k].x, A.rk_b * n0);
          n1 = fma_(A.rk_a, u0v[k].y, A.rk_b * n1);
        }
        Un[k][0] = n0; Un[k][1] = n1;
      }
      const size_t o = (size_t)jo * A.pitch + c0;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (ok0s && ok1) *reinterpret_cast<V2*>(A.Uout + k * A.plane + o) = mk2(Un[k][0], Un[k][1]);
        else {
          if (ok0s) A.Uout[k * A.plane + o] = Un[k][0];
          if (ok1) A.Uout[k * A.plane + o + 1] = Un[k][1];
        }
      }
      if (A.smax_bits) {  // S9 on the new state (it is U^n of the next step), fluid cells only
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const bool use = (e == 0 ? ok0s : ok1) && (e == 0 ? fl0 : fl1);
          const T ri = rcp_(Un[0][e]);
          const T u = Un[1][e] * ri, v = Un[2][e] * ri;
          const T p = g1 * fma_(T(-0.5), fma_(Un[1][e], u, Un[2][e] * v), Un[3][e]);
          const T gp = gamma * p;
          const T a = gp * rsqrt_(gp * Un[0][e]);
          const T s = max_(abs_(u), abs_(v)) + a;
          if (use) smax = (s > smax || s != s) ? s : smax;  // NaN propagates
        }
      }
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
