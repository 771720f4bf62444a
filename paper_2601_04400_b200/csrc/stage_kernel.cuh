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
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace jxs {

constexpr int LW = 32;           // cells per warp strip (1 per lane)
constexpr int CW = LW + 4;       // + 2 halo cells per side
constexpr int RING = 5;          // rows of primitives kept per warp
constexpr int STAGE_WARPS = 1;   // one warp per CTA: everything derived from blockIdx is warp-uniform

// output cells per strip = lanes 1..SOUT; the first column of a TMA box must lie on a 16-byte boundary
// (measured: a tiled copy from an unaligned column raises "illegal instruction"), so strips start on
// multiples of 2 doubles / 4 floats
template <typename T> struct Cfg;
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
  int nseg_a, rows_b;    // the first nseg_a row segments of a strip have rows_per_seg rows, the later ones rows_b
  // batch (BATCH instantiations): nb members stacked along y, nseg row segments per strip and member; dt and
  // smax_bits of member m lie state_stride bytes further on per member, its ten viscous coefficients (the order of
  // vy_n .. vx_q below) at vtab[10 m], its fluid mask and (mode 1) output at member strides
  int nb, nseg;
  long long state_stride;
  const T* vtab;
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
  // S5' (optional): network outputs y per face from flux_mlp_kernel / the CNN's last layer, one uint4 per padded cell
  // [rows][pitch]: eight fp16 values {right face: 4, top face: 4}, k = (mass, normal, tangential momentum, energy) (R14).
  // 16 bytes per cell-stage instead of the 32 of fp32 planes; fp16 keeps 11 bits (5e-4) of a correction held to 1e-2.
  const uint4* dFG;
  T oscale[4];
  // one-dimensional problems (stage1d_kernel.cuh): the per-face MLP's flux correction from mlp1d_kernel.cuh, already
  // scaled, indexed like U (right face of the cell); nullptr = none
  const double* dF1d;
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
// TMA tiled copy of a [4 variables][1 row][W columns] box of a padded SoA buffer (tensor map: dim 0 = column,
// 1 = row, 2 = variable) global -> shared: ONE instruction and three integer coordinates per row instead of four
// bulk copies with 64-bit address arithmetic each
__device__ __forceinline__ void tma_box_g2s(uint32_t dst, const CUtensorMap* tm, int col, int row, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(dst), "l"(tm), "r"(col), "r"(row), "r"(0), "r"(bar) : "memory");
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
// x <= 0 for both of two values, tested on the integer pipe (the FP64 pipe is the bottleneck) through the words that
// hold the sign: a word <= 0 means x <= 0 (including -0) or, for a double, 0 <= x < 2^-1042 (a density or pressure
// that small is zero for every purpose here; the oracle's test is x <= 0).  NaN is not flagged, as in the oracle.
__device__ __forceinline__ int sign_word(double x) { return __double2hiint(x); }
__device__ __forceinline__ int sign_word(float x) { return __float_as_int(x); }
template <typename T>
__device__ __forceinline__ bool any_not_positive(T a, T b) { return min(sign_word(a), sign_word(b)) <= 0; }

// sign bit and halving on the integer pipe (arguments are normal numbers; -0.0 counts as negative)
__device__ __forceinline__ bool is_negative(double x) { return __double2hiint(x) < 0; }
__device__ __forceinline__ bool is_negative(float x) { return __float_as_int(x) < 0; }
__device__ __forceinline__ double half_of(double x) {
  return __hiloint2double(__double2hiint(x) - 0x00100000, __double2loint(x));
}
__device__ __forceinline__ float half_of(float x) { return 0.5f * x; }

// ------------------------------------------------------------------ lock-step arithmetic
// The FP64 pipe of sm_100 accepts one warp instruction every 2 cycles and returns it after ~8; measured
// on B200 it only stays busy when every warp's OWN stream holds >= 4 independent
// FP64 instructions between a result and its use - more resident warps do not make up for a shorter
// distance (3 -> 72 %, 4 -> 92 % of the pipe).  So every routine below is written N-wide: each
// statement is applied to N independent problems (the 4 primitive variables of a reconstruction, the
// y- and the x-face of the Riemann solver, the cell and its halo cell of the conversion) before the
// next statement starts, which is the order ptxas keeps.
#define JXS_V _Pragma("unroll") for (int k = 0; k < N; ++k)

// Branch-free reciprocal and reciprocal square root.  MUFU.RCP64H / MUFU.RSQ64H are accurate to
// 2^-20 (measured on B200), so ONE cubic Newton step reaches 1 ulp (max rel. error 2.2e-16 /
// 2.7e-16 measured over 2^26 arguments).  No slow path: arguments here are densities, pressures,
// wave-speed differences and WENO denominators, all normal and far from the range limits.
__device__ __forceinline__ double rcp_seed(double b) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
  return r;
}
__device__ __forceinline__ float rcp_seed(float b) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(b));
  return r;
}
__device__ __forceinline__ double rsqrt_seed(double b) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
  return r;
}
__device__ __forceinline__ float rsqrt_seed(float b) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(b));
  return r;
}
template <typename T, int N>
__device__ __forceinline__ void rcp_n(const T (&b)[N], T (&r)[N]) {
  T x[N];
  JXS_V x[k] = rcp_seed(b[k]);
  if (sizeof(T) == 8) {
    T e[N];
    JXS_V e[k] = fma_(-b[k], x[k], T(1));
    JXS_V e[k] = fma_(e[k], e[k], e[k]);
    JXS_V r[k] = fma_(x[k], e[k], x[k]);
  } else {
    JXS_V r[k] = x[k];
  }
}
template <typename T, int N>
__device__ __forceinline__ void rsqrt_n(const T (&b)[N], T (&r)[N]) {
  T y[N];
  JXS_V y[k] = rsqrt_seed(b[k]);
  if (sizeof(T) == 8) {
    T h[N], f[N], g[N];
    JXS_V h[k] = half_of(b[k]);
    JXS_V h[k] = h[k] * y[k];
    JXS_V f[k] = fma_(-h[k], y[k], T(0.5));
    JXS_V g[k] = fma_(T(1.5), f[k], T(1));
    JXS_V f[k] = f[k] * g[k];
    JXS_V r[k] = fma_(y[k], f[k], y[k]);
  } else {
    JXS_V r[k] = y[k];
  }
}
template <typename T>
__device__ __forceinline__ T rcp_(T b) {
  T bb[1] = {b}, r[1];
  rcp_n<T, 1>(bb, r);
  return r[0];
}
template <typename T>
__device__ __forceinline__ T rsqrt_(T b) {
  T bb[1] = {b}, r[1];
  rsqrt_n<T, 1>(bb, r);
  return r[0];
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
// N problems in lock step (the primitive variables).
// The part of the reconstruction behind the smoothness terms: Bk = 4 (beta_k + eps) on entry.
template <typename T, int N>
__device__ __forceinline__ void weno5_tail_n(const T (&d2)[N], const T (&d3)[N], const T (&s0)[N], const T (&s1)[N],
                                             const T (&s2)[N], T (&B0)[N], T (&B1)[N], T (&B2)[N], const T (&c)[N],
                                             const StageArgs<T>& K, T (&vm)[N], T (&vp)[N]) {
  JXS_V B0[k] = B0[k] * B0[k];
  JXS_V B1[k] = B1[k] * B1[k];
  JXS_V B2[k] = B2[k] * B2[k];
  T P12[N], P02[N], P01[N], h[N], denp[N], denm[N], A[N], C[N], np[N], nm[N];
  JXS_V P12[k] = B1[k] * B2[k];
  JXS_V P02[k] = B0[k] * B2[k];
  JXS_V P01[k] = B0[k] * B1[k];
  JXS_V h[k] = P12[k] + P01[k];
  JXS_V A[k] = s0[k] - s1[k];
  JXS_V C[k] = s1[k] - s2[k];
  JXS_V h[k] = fma_(T(6), P02[k], h[k]);
  JXS_V A[k] = P12[k] * A[k];
  JXS_V C[k] = P01[k] * C[k];
  JXS_V denp[k] = fma_(T(2), P01[k], h[k]);
  JXS_V denm[k] = fma_(T(2), P12[k], h[k]);
  // 6 (vp - c) = (d2 + 2 d3) + (2A + 3C)/denp,   6 (c - vm) = (d3 + 2 d2) + (2C + 3A)/denm
  T S[N], rp[N], rm[N], ep[N], em[N];
  JXS_V S[k] = A[k] + C[k];
  if (sizeof(T) == 8) {  // one reciprocal for both sides (the product stays far inside the fp64 range)
    T dd[N], r[N];
    JXS_V dd[k] = denp[k] * denm[k];
    rcp_n<T, N>(dd, r);
    JXS_V rp[k] = r[k] * denm[k];
    JXS_V rm[k] = r[k] * denp[k];
  } else {
    rcp_n<T, N>(denp, rp);
    rcp_n<T, N>(denm, rm);
  }
  JXS_V np[k] = fma_(T(2), S[k], C[k]);
  JXS_V nm[k] = fma_(T(2), S[k], A[k]);
  JXS_V ep[k] = fma_(T(2), d3[k], d2[k]);
  JXS_V em[k] = fma_(T(2), d2[k], d3[k]);
  JXS_V ep[k] = fma_(np[k], rp[k], ep[k]);
  JXS_V em[k] = fma_(nm[k], rm[k], em[k]);
  JXS_V vp[k] = fma_(K.sixth, ep[k], c[k]);
  JXS_V vm[k] = fma_(-K.sixth, em[k], c[k]);
}

template <typename T, int N>
__device__ __forceinline__ void weno5_n(const T (&a)[N], const T (&b)[N], const T (&c)[N], const T (&d)[N],
                                        const T (&e)[N], const StageArgs<T>& K, T (&vm)[N], T (&vp)[N]) {
  T d1[N], d2[N], d3[N], d4[N], s0[N], s1[N], s2[N], t0[N], t1[N], t2[N];
  JXS_V d1[k] = b[k] - a[k];
  JXS_V d2[k] = c[k] - b[k];
  JXS_V d3[k] = d[k] - c[k];
  JXS_V d4[k] = e[k] - d[k];
  JXS_V s0[k] = d2[k] - d1[k];
  JXS_V s1[k] = d3[k] - d2[k];
  JXS_V s2[k] = d4[k] - d3[k];
  JXS_V t0[k] = fma_(T(3), d2[k], -d1[k]);
  JXS_V t1[k] = d2[k] + d3[k];
  JXS_V t2[k] = fma_(T(-3), d3[k], d4[k]);
  T B0[N], B1[N], B2[N], u0[N], u1[N], u2[N];
  JXS_V u0[k] = K.c133 * s0[k];
  JXS_V u1[k] = K.c133 * s1[k];
  JXS_V u2[k] = K.c133 * s2[k];
  JXS_V B0[k] = fma_(t0[k], t0[k], K.eps4);
  JXS_V B1[k] = fma_(t1[k], t1[k], K.eps4);
  JXS_V B2[k] = fma_(t2[k], t2[k], K.eps4);
  JXS_V B0[k] = fma_(u0[k], s0[k], B0[k]);
  JXS_V B1[k] = fma_(u1[k], s1[k], B1[k]);
  JXS_V B2[k] = fma_(u2[k], s2[k], B2[k]);
  weno5_tail_n<T, N>(d2, d3, s0, s1, s2, B0, B1, B2, c, K, vm, vp);
}

// The same reconstruction along the direction a warp MARCHES in (y): consecutive cells of a column share their first
// differences, second differences and the (13/3) s^2 + 4 eps part of the smoothness terms, so these are carried in
// registers from one row to the next instead of being recomputed (19 -> 10 FP64 instructions per variable before the
// common tail, 2 shared-memory loads per variable instead of 5).  For the stencil rows (a,b,c,d,e):
//   older = {d2 = c-b, s0, W0},  newer = {d3 = d-c, s1, W1},  Wk = (13/3) sk^2 + 4 eps;  dprev = d,  e = the new row.
// t0 = 3 d2 - d1 = 2 d2 + s0 and t2 = d4 - 3 d3 = s2 - 2 d3 need neither d1 nor d4.  On return `older` holds
// {d4, s2, W2}: it is the next row's `newer`, and this row's `newer` the next row's `older`.
template <typename T, int N> struct YCarry { T d[N], s[N], w[N]; };

template <typename T, int N>
__device__ __forceinline__ void weno5_carry_n(YCarry<T, N>& older, const YCarry<T, N>& newer, const T (&c)[N],
                                              const T (&dprev)[N], const T (&e)[N], const StageArgs<T>& K, T (&vm)[N],
                                              T (&vp)[N]) {
  T d4[N], s2[N], t0[N], t1[N], t2[N], u2[N], W2[N], B0[N], B1[N], B2[N];
  JXS_V d4[k] = e[k] - dprev[k];
  JXS_V t0[k] = fma_(T(2), older.d[k], older.s[k]);
  JXS_V t1[k] = older.d[k] + newer.d[k];
  JXS_V s2[k] = d4[k] - newer.d[k];
  JXS_V B0[k] = fma_(t0[k], t0[k], older.w[k]);
  JXS_V B1[k] = fma_(t1[k], t1[k], newer.w[k]);
  JXS_V t2[k] = fma_(T(-2), newer.d[k], s2[k]);
  JXS_V u2[k] = K.c133 * s2[k];
  JXS_V W2[k] = fma_(u2[k], s2[k], K.eps4);
  JXS_V B2[k] = fma_(t2[k], t2[k], W2[k]);
  weno5_tail_n<T, N>(older.d, newer.d, older.s, newer.s, s2, B0, B1, B2, c, K, vm, vp);
  JXS_V { older.d[k] = d4[k]; older.s[k] = s2[k]; older.w[k] = W2[k]; }
}
// the carried state before the first row of a segment, from the stencil rows (a, b, c, d)
template <typename T, int N>
__device__ __forceinline__ void weno5_carry_init_n(const T (&a)[N], const T (&b)[N], const T (&c)[N], const T (&d)[N],
                                                   const StageArgs<T>& K, YCarry<T, N>& older, YCarry<T, N>& newer) {
  T d1[N], u0[N], u1[N];
  JXS_V d1[k] = b[k] - a[k];
  JXS_V older.d[k] = c[k] - b[k];
  JXS_V newer.d[k] = d[k] - c[k];
  JXS_V older.s[k] = older.d[k] - d1[k];
  JXS_V newer.s[k] = newer.d[k] - older.d[k];
  JXS_V u0[k] = K.c133 * older.s[k];
  JXS_V u1[k] = K.c133 * newer.s[k];
  JXS_V older.w[k] = fma_(u0[k], older.s[k], K.eps4);
  JXS_V newer.w[k] = fma_(u1[k], newer.s[k], K.eps4);
}

// ------------------------------------------------------------------ S5: HLLC, one-sided
// Normal velocity un, tangential ut.  Eq. 3-7 with the star state of reading R1; for s* != 0 the
// sign blend of Eq. 3 is exact branch selection, at s* = 0 the left branch is taken (R2).
// Returns (mass, normal momentum, tangential momentum, energy) flux.  N faces in lock step.
template <typename T, int N>
__device__ __forceinline__ void hllc_n(const T (&rL)[N], const T (&unL)[N], const T (&utL)[N], const T (&pL)[N],
                                       const T (&rR)[N], const T (&unR)[N], const T (&utR)[N], const T (&pR)[N],
                                       T gamma, T g1inv, T (&f0)[N], T (&f1)[N], T (&f2)[N], T (&f3)[N]) {
  // a = sqrt(gamma p / rho) = (gamma p) * rsqrt(gamma p rho): both sides of all faces in one 2N-wide pass
  T gp[2 * N], x[2 * N], y[2 * N];
  JXS_V gp[k] = gamma * pL[k];
  JXS_V gp[N + k] = gamma * pR[k];
  JXS_V x[k] = gp[k] * rL[k];
  JXS_V x[N + k] = gp[N + k] * rR[k];
  rsqrt_n<T, 2 * N>(x, y);
  T aL[N], aR[N], sL[N], sR[N], mL[N], mR[N], q[N], den[N], sS[N];
  JXS_V aL[k] = gp[k] * y[k];
  JXS_V aR[k] = gp[N + k] * y[N + k];
  JXS_V sL[k] = min_(unL[k] - aL[k], unR[k] - aR[k]);  // Eq. 6
  JXS_V sR[k] = max_(unL[k] + aL[k], unR[k] + aR[k]);
  JXS_V mL[k] = sL[k] - unL[k];
  JXS_V mR[k] = sR[k] - unR[k];
  JXS_V mL[k] = rL[k] * mL[k];
  JXS_V mR[k] = rR[k] * mR[k];
  JXS_V q[k] = pR[k] - pL[k];
  JXS_V den[k] = mL[k] - mR[k];
  JXS_V q[k] = fma_(-mR[k], unR[k], q[k]);
  rcp_n<T, N>(den, den);
  JXS_V q[k] = fma_(mL[k], unL[k], q[k]);
  JXS_V sS[k] = q[k] * den[k];  // Eq. 7
  T r[N], un[N], ut[N], p[N], sk[N], sc[N];
  JXS_V {
    const bool left = !is_negative(sS[k]);
    r[k] = left ? rL[k] : rR[k]; un[k] = left ? unL[k] : unR[k]; ut[k] = left ? utL[k] : utR[k];
    p[k] = left ? pL[k] : pR[k]; sk[k] = left ? sL[k] : sR[k];
    // Eq. 5: min(0, sL) on the left, max(0, sR) on the right = the selected speed where its sign says so
    sc[k] = is_negative(sk[k]) == left ? sk[k] : T(0);
  }
  T E[N], ru[N], rinv[N], chi[N], rchi[N], w[N], dm[N], dn[N], dt_[N], dE[N], z[N];
  JXS_V rinv[k] = sk[k] - sS[k];
  JXS_V E[k] = ut[k] * ut[k];
  JXS_V w[k] = T(0.5) * r[k];
  JXS_V z[k] = p[k] * g1inv;
  rcp_n<T, N>(rinv, rinv);
  JXS_V E[k] = fma_(un[k], un[k], E[k]);
  JXS_V ru[k] = r[k] * un[k];
  JXS_V chi[k] = sk[k] - un[k];
  JXS_V E[k] = fma_(w[k], E[k], z[k]);
  JXS_V chi[k] = chi[k] * rinv[k];
  JXS_V w[k] = p[k] * rinv[k];
  JXS_V z[k] = sS[k] - un[k];
  JXS_V rchi[k] = r[k] * chi[k];
  JXS_V dE[k] = fma_(chi[k], E[k], -E[k]);
  JXS_V dm[k] = fma_(r[k], chi[k], -r[k]);      // rho* - rho
  JXS_V w[k] = fma_(rchi[k], sS[k], w[k]);
  JXS_V dn[k] = fma_(rchi[k], sS[k], -ru[k]);   // (rho u)* - rho u
  JXS_V dt_[k] = ut[k] * dm[k];                 // (rho v)* - rho v
  JXS_V dE[k] = fma_(z[k], w[k], dE[k]);        // E* - E
  JXS_V f1[k] = fma_(ru[k], un[k], p[k]);
  JXS_V f2[k] = ru[k] * ut[k];
  JXS_V f3[k] = E[k] + p[k];
  JXS_V f0[k] = fma_(sc[k], dm[k], ru[k]);
  JXS_V f3[k] = un[k] * f3[k];
  JXS_V f1[k] = fma_(sc[k], dn[k], f1[k]);
  JXS_V f2[k] = fma_(sc[k], dt_[k], f2[k]);
  JXS_V f3[k] = fma_(sc[k], dE[k], f3[k]);
}

// four fp16 values in two 32-bit words -> floats
__device__ __forceinline__ void unpack_half4(uint32_t lo, uint32_t hi, float (&y)[4]) {
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&lo)), b = __half22float2(*reinterpret_cast<const __half2*>(&hi));
  y[0] = a.x; y[1] = a.y; y[2] = b.x; y[3] = b.y;
}

template <typename T>
__device__ __forceinline__ T shfl_down1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }
template <typename T>
__device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

__device__ __forceinline__ void atomic_max_pos(unsigned long long* addr, double v) {
  // v >= 0 (or NaN, whose bit pattern compares above +inf): unsigned order == numeric order
  atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

// S6 (R8): viscous flux through N faces in lock step, subtracted from the fluxes (f1 = normal momentum,
// f2 = tangential momentum, f3 = energy).  dn, dt_: differences of the normal / tangential velocity across
// the face; xt, xn: sums of the two adjacent centred cross-differences of the tangential / normal
// velocity; sn, st: sums of the two adjacent velocities; dT: temperature difference.  Coefficients
// (StageArgs v?_*) per face: cn = 4/3 mu/h_n, cc = (2/3) mu/(4 h_t), cs = mu/h_n, ct = mu/(4 h_t), cq = kappa/h_n.
template <typename T, int N>
__device__ __forceinline__ void viscous_n(const T (&dn)[N], const T (&dt_)[N], const T (&xt)[N], const T (&xn)[N],
                                          const T (&sn)[N], const T (&st)[N], const T (&dT)[N], const T (&cn)[N],
                                          const T (&cc)[N], const T (&cs)[N], const T (&ct)[N], const T (&cq)[N],
                                          T (&f1)[N], T (&f2)[N], T (&f3)[N]) {
  T tnn[N], tnt[N], w[N];
  JXS_V tnn[k] = cc[k] * xt[k];
  JXS_V tnt[k] = ct[k] * xn[k];
  JXS_V tnn[k] = fma_(cn[k], dn[k], -tnn[k]);
  JXS_V tnt[k] = fma_(cs[k], dt_[k], tnt[k]);
  JXS_V w[k] = st[k] * tnt[k];
  JXS_V f1[k] -= tnn[k];
  JXS_V f2[k] -= tnt[k];
  JXS_V w[k] = fma_(sn[k], tnn[k], w[k]);  // 2 (u_n tau_nn + u_t tau_nt) at the face
  JXS_V f3[k] = fma_(T(-0.5), w[k], f3[k]);
  JXS_V f3[k] = fma_(-cq[k], dT[k], f3[k]);
}

// Runge-Kutta operand rows: fp64 strips start on even columns, so the 32 owned columns can be
// fetched alone (16-byte aligned); fp32 fetches the CW-wide window like the raw rows.
template <typename T> struct Epi { static constexpr int W = sizeof(T) == 8 ? LW : CW, OFF = sizeof(T) == 8 ? 0 : 2; };
// per-warp shared memory: raw rows 2 x [4][CW] | RK operands 2 x [4][Epi::W] | 2 mbarriers | ring [RING][NV][CW]
// (the TMA destinations first: tiled copies need 128-byte aligned destinations)
template <typename T> __host__ __device__ constexpr size_t stage_smem_raw() { return (size_t)4 * CW * sizeof(T); }
template <typename T> __host__ __device__ constexpr size_t stage_smem_epihalf() {
  return ((size_t)4 * Epi<T>::W * sizeof(T) + 127) / 128 * 128;
}
template <typename T> __host__ __device__ constexpr size_t stage_smem_epi() { return 2 * stage_smem_epihalf<T>(); }
template <typename T> __host__ __device__ constexpr size_t stage_smem_rawslot() { return (stage_smem_raw<T>() + 127) / 128 * 128; }
// one ring row [NV][CW], padded to 128 bytes: the first rows of a segment land in the ring directly
template <typename T, int NV> __host__ __device__ constexpr size_t stage_smem_ringslot() {
  return ((size_t)NV * CW * sizeof(T) + 127) / 128 * 128;
}
template <typename T, int NV>
__host__ __device__ constexpr size_t stage_smem_per_warp() {
  return 2 * stage_smem_rawslot<T>() + stage_smem_epi<T>() + 128 + (size_t)RING * stage_smem_ringslot<T, NV>();
}

// ------------------------------------------------------------------ the kernel
template <typename T, bool VISC, bool ARTV, bool MLP, int MINB, bool BATCH = false>
__global__ void __launch_bounds__(STAGE_WARPS * 32, MINB)
stage_kernel(const StageArgs<T> A, const __grid_constant__ CUtensorMap tm_row, const __grid_constant__ CUtensorMap tm_epi,
             const __grid_constant__ CUtensorMap tm_epi0) {
  // tm_row: boxes [4][1][CW] of Uin; tm_epi / tm_epi0: boxes [4][1][Epi::W] of Uin / U^n
  constexpr int SOUT = Cfg<T>::SOUT;
  constexpr int NV = VISC ? 5 : 4;
  extern __shared__ __align__(128) unsigned char smem_raw[];

  constexpr int EW = Epi<T>::W, EOFF = Epi<T>::OFF;
  const int lane = threadIdx.x;
  const int task = blockIdx.x;
  const int strip = task % A.nstrips, seg_all = task / A.nstrips;
  const int member = BATCH ? seg_all / A.nseg : 0, seg = BATCH ? seg_all - member * A.nseg : seg_all;
  const int rb = BATCH ? member * (A.ny + 6) : 0;  // first padded row of my member
  // first output row (padded index) and one past the last; tasks are handed out in blockIdx order, segment-major, and
  // the last segments are the short ones: the kernel's tail (SMs running out of tasks) shrinks with the task length
  const bool seg_long = seg < A.nseg_a;
  const int jbeg = rb + 3 + (seg_long ? seg * A.rows_per_seg : A.nseg_a * A.rows_per_seg + (seg - A.nseg_a) * A.rows_b);
  const int jend = min(jbeg + (seg_long ? A.rows_per_seg : A.rows_b), rb + 3 + A.ny);
  if (jbeg >= jend) return;
  const int w0 = 2 + SOUT * strip;  // padded column of lane 0's cell
  const int ic = w0 + lane - 3;     // interior x index of my cell
  const int q = lane + 2;           // my column inside the per-warp rows
  const bool in_x = (unsigned)ic < (unsigned)A.nx;  // my cell is an interior column (lane 0 of strip 0 is column -1)

  constexpr uint32_t RAWSLOT = (uint32_t)stage_smem_rawslot<T>();
  T* raw = reinterpret_cast<T*>(smem_raw);                                                  // [2] x [4][CW]
  T* epi = reinterpret_cast<T*>(smem_raw + 2 * RAWSLOT);                                    // U_in rows [4][EW]
  T* epi0 = reinterpret_cast<T*>(smem_raw + 2 * RAWSLOT + stage_smem_epihalf<T>());         // U^n rows [4][EW]
  T* ring = reinterpret_cast<T*>(smem_raw + 2 * RAWSLOT + stage_smem_epi<T>() + 128);       // [RING][NV][CW]
  const uint32_t raw_u32 = smem_u32(raw), epi_u32 = smem_u32(epi);
  const uint32_t bar_raw = epi_u32 + (uint32_t)stage_smem_epi<T>(), bar_epi = bar_raw + 8;
  constexpr uint32_t ROWB = CW * sizeof(T), EROWB = EW * sizeof(T);

  if (lane == 0) {
    mbar_init(bar_raw, 1);
    mbar_init(bar_epi, 1);
    mbar_fence_init();
  }
  __syncwarp();

  const int nfirst = jbeg - 3, nlast = jend + 2;  // rows to stream, inclusive
  const bool use_u0 = A.rk_a != T(0);
  auto issue_row = [&](int n, int slot) {  // one lane: conserved row n -> raw[slot]
    mbar_expect_tx(bar_raw, 4 * ROWB);
    tma_box_g2s(raw_u32 + slot * RAWSLOT, &tm_row, w0 - 2, n, bar_raw);
  };
  auto issue_epi = [&](int j) {  // one lane: Runge-Kutta operands of output row j -> epi
    mbar_expect_tx(bar_epi, (use_u0 ? 8 : 4) * EROWB);
    tma_box_g2s(epi_u32, &tm_epi, w0 - EOFF, j, bar_epi);
    if (use_u0) tma_box_g2s(epi_u32 + (uint32_t)stage_smem_epihalf<T>(), &tm_epi0, w0 - EOFF, j, bar_epi);
  };
  // The first five rows of the segment go straight into the ring (phase 0 of bar_epi), the sixth into raw slot 1
  // (phase 0 of bar_raw): one memory latency for the whole warm-up instead of one per row.
  if (elect_one()) {
    mbar_expect_tx(bar_epi, 5 * 4 * ROWB);
#pragma unroll
    for (int r = 0; r < 5; ++r)
      tma_box_g2s(smem_u32(ring) + r * (uint32_t)stage_smem_ringslot<T, NV>(), &tm_row, w0 - 2, nfirst + r, bar_epi);
    issue_row(nfirst + 5, 1);
  }

  const T gamma = A.gamma, g1inv = A.g1inv, g1 = A.g1;
  const T dtv = T(*reinterpret_cast<const double*>(reinterpret_cast<const char*>(A.dt) + (BATCH ? member * A.state_stride : 0)));
  const uint8_t* const fluid = A.fluid ? A.fluid + (BATCH ? (size_t)member * A.nx * A.ny : 0) : nullptr;
  // viscous-flux coefficients: kernel parameters (constant-bank operands), or this member's row of the table
  T vc[10] = {A.vy_n, A.vy_c, A.vy_s, A.vy_t, A.vy_q, A.vx_n, A.vx_c, A.vx_s, A.vx_t, A.vx_q};
  if (BATCH && VISC) {
#pragma unroll
    for (int c = 0; c < 10; ++c) vc[c] = A.vtab[10 * member + c];
  }

  // state carried from one row to the next
  T Ly[4];  // left state (rho,u,v,p) at the face below the next centre row
  T Gp[4];  // total y-flux (mass, normal = rho v, tangential = rho u, energy) through the face below the output row
#pragma unroll
  for (int k = 0; k < 4; ++k) { Ly[k] = T(0); Gp[k] = T(0); }
  T cuP = T(0), cvP = T(0);
  // the y-reconstruction's carried differences (weno5_carry_n) and the primitives of my cell in the two newest rows
  YCarry<T, 4> ycA, ycB;
  T Ep0[4], Ep1[4];
  T smax = T(0);
  unsigned fl_next = 1;  // fluid flag of my cell in the next output row, fetched one iteration ahead
  uint4 y_next = make_uint4(0, 0, 0, 0);  // S5': the network outputs of my cell in the next output row

  // Ring rows as loop-carried per-lane pointers (to my column q), rotated once per iteration: the row
  // accesses below become LDS with immediate offsets, no slot arithmetic.  pN = slot written next.
  constexpr int RS = (int)(stage_smem_ringslot<T, NV>() / sizeof(T));  // ring slot stride in elements
  const T *pA = ring + q, *pB = ring + 1 * RS + q, *pC = ring + 2 * RS + q, *pD = ring + 3 * RS + q;
  T* pN = ring + 4 * RS + q;
  // my halo column, relative to q (lanes 0-3 convert one each; the others redo their own and drop it)
  const int hoff = lane < 2 ? -2 : (lane < 4 ? LW - 2 : 0);

  // ---------------------------------------------------------------- S3: row n -> primitives, ring rotation
  // One warp-level barrier per row: after it every lane is done with the ring slot, the raw-row slot and the
  // Runge-Kutta operand rows that are overwritten next, so one elected lane issues the next TMA copies.
  auto take_row = [&](int n, int it, bool want_epi, T (&mine)[4]) {  // mine: (rho, u, v, p) of my cell in row n
    __syncwarp();
    mbar_wait(bar_raw, (it + 1) & 1);  // row nfirst+5 was phase 0
    if (elect_one()) {
      if (n < nlast) issue_row(n + 1, (it + 1) & 1);
      if (want_epi) issue_epi(n - 3);
    }
    const T* src = reinterpret_cast<const T*>(smem_raw + (it & 1) * RAWSLOT) + q;
    constexpr int N = 2;  // my cell and my halo cell in lock step
    T r[N], ru[N], rv[N], E[N], ri[N], u[N], v[N], p[N];
    const int o[N] = {0, hoff};
    JXS_V { r[k] = src[o[k]]; ru[k] = src[CW + o[k]]; rv[k] = src[2 * CW + o[k]]; E[k] = src[3 * CW + o[k]]; }
    rcp_n<T, N>(r, ri);
    JXS_V u[k] = ru[k] * ri[k];
    JXS_V v[k] = rv[k] * ri[k];
    JXS_V p[k] = rv[k] * v[k];
    JXS_V p[k] = fma_(ru[k], u[k], p[k]);
    JXS_V p[k] = fma_(T(-0.5), p[k], E[k]);
    JXS_V p[k] = g1 * p[k];
    JXS_V {
      if (k == 0 || lane < 4) {
        T* dst = pN + o[k];
        dst[0] = r[k]; dst[CW] = u[k]; dst[2 * CW] = v[k]; dst[3 * CW] = p[k];
        if (VISC) dst[4 * CW] = p[k] * ri[k];
      }
    }
    mine[0] = r[0]; mine[1] = u[0]; mine[2] = v[0]; mine[3] = p[0];
  };
  // ring rows until the next rotation: pA = row n-4, pB = n-3 (output row jo), pC = n-2 (centre of the y
  // stencil, jc), pD = n-1, pN = n (just written)
  auto rotate = [&]() {
    T* const oldest = const_cast<T*>(pA);
    pA = pB; pB = pC; pC = pD; pD = pN; pN = oldest;
  };

  // ---------------------------------------------------------------- S4 along y (and the carried cross differences)
  // older / newer: the carried state (see weno5_carry_n; they exchange roles every row), dprev / e: my cell in rows
  // n-1 and n, the centre row jc = n-2 comes from the ring
  auto weno_y = [&](YCarry<T, 4>& older, const YCarry<T, 4>& newer, const T (&dprev)[4], const T (&e)[4], T (&Ry)[4],
                    T (&Lnew)[4], T& cuC, T& cvC) {
    constexpr int N = 4;
    T c[N];
    JXS_V c[k] = pC[k * CW];
    weno5_carry_n<T, N>(older, newer, c, dprev, e, A, Ry, Lnew);
    // positivity guard (R15): a side with rho <= 0 or p <= 0 falls back to its cell (row jc);
    // one warp vote keeps the (never taken in practice) repair off the common path
    const bool badR = any_not_positive(Ry[0], Ry[3]);
    const bool badL = any_not_positive(Lnew[0], Lnew[3]);
    if (__any_sync(0xffffffffu, badR | badL)) {
      asm volatile("" ::: "memory");  // keeps this (never taken in practice) block a branch, not 16 selects
      JXS_V { Ry[k] = badR ? c[k] : Ry[k]; Lnew[k] = badL ? c[k] : Lnew[k]; }
    }
    if (VISC) {  // x-centred differences of u, v in row jc
      cuC = pC[CW + 1] - pC[CW - 1];
      cvC = pC[2 * CW + 1] - pC[2 * CW - 1];
    }
  };

  // ---------------------------------------------------------------- prologue: rows nfirst .. nfirst+5
  // rows nfirst .. nfirst+4 are converted in place in the ring (5 rows in lock step, then their halo columns);
  // then the left state at the face below row jbeg (it = 4) and the flux through it (it = 5)
  mbar_wait(bar_epi, 0);
  {
    constexpr int N = 5;
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
      const int o = pass == 0 ? 0 : hoff;
      T* const base = ring + q + o;
      T r[N], ru[N], rv[N], E[N], ri[N], u[N], v[N], p[N];
      JXS_V { const T* src = base + k * RS; r[k] = src[0]; ru[k] = src[CW]; rv[k] = src[2 * CW]; E[k] = src[3 * CW]; }
      rcp_n<T, N>(r, ri);
      JXS_V u[k] = ru[k] * ri[k];
      JXS_V v[k] = rv[k] * ri[k];
      JXS_V p[k] = rv[k] * v[k];
      JXS_V p[k] = fma_(ru[k], u[k], p[k]);
      JXS_V p[k] = fma_(T(-0.5), p[k], E[k]);
      JXS_V p[k] = g1 * p[k];
      if (pass == 0 || lane < 4) {
        JXS_V {
          T* dst = base + k * RS;
          dst[CW] = u[k]; dst[2 * CW] = v[k]; dst[3 * CW] = p[k];
          if (VISC) dst[4 * CW] = p[k] * ri[k];
        }
      }
    }
  }
  __syncwarp();  // the cross differences below read the neighbours' columns
  {  // it = 4: the left state at the face below row jbeg; the carried differences start from ring rows 0 .. 3
    constexpr int N = 4;
    T a[N], b[N], c[N], d[N];
    JXS_V { a[k] = pA[k * CW]; b[k] = pB[k * CW]; c[k] = pC[k * CW]; d[k] = pD[k * CW]; Ep0[k] = pN[k * CW]; }
    weno5_carry_init_n<T, N>(a, b, c, d, A, ycA, ycB);
    T Ry[4], cuC = T(0), cvC = T(0);
    weno_y(ycA, ycB, d, Ep0, Ry, Ly, cuC, cvC);
    if (VISC) { cuP = cuC; cvP = cvC; }
    rotate();
  }
  {  // it = 5: the flux through that face
    const int n = nfirst + 5;
    take_row(n, 5, false, Ep1);
    const int jo = n - 3;
    T Ry[4], Lnew[4], cuC = T(0), cvC = T(0);
    weno_y(ycB, ycA, Ep0, Ep1, Ry, Lnew, cuC, cvC);
    {
      constexpr int N = 1;
      T f0[N], f1[N], f2[N], f3[N];
      const T rL[N] = {Ly[0]}, unL[N] = {Ly[2]}, utL[N] = {Ly[1]}, pL[N] = {Ly[3]};
      const T rR[N] = {Ry[0]}, unR[N] = {Ry[2]}, utR[N] = {Ry[1]}, pR[N] = {Ry[3]};
      hllc_n<T, N>(rL, unL, utL, pL, rR, unR, utR, pR, gamma, g1inv, f0, f1, f2, f3);
      if (MLP) {  // Eq. 11
        const uint4 y8 = __ldg(A.dFG + (size_t)jo * A.pitch + (w0 + lane));
        float yG[4];
        unpack_half4(y8.z, y8.w, yG);
        f0[0] = fma_(A.oscale[0], T(yG[0]), f0[0]);
        f1[0] = fma_(A.oscale[1], T(yG[1]), f1[0]);
        f2[0] = fma_(A.oscale[2], T(yG[2]), f2[0]);
        f3[0] = fma_(A.oscale[3], T(yG[3]), f3[0]);
        y_next = __ldg(A.dFG + (size_t)(jo + 1) * A.pitch + (w0 + lane));
      }
      if (VISC) {
        const T dn[N] = {pC[2 * CW] - pB[2 * CW]}, dt_[N] = {pC[CW] - pB[CW]}, xt[N] = {cuP + cuC}, xn[N] = {cvP + cvC};
        const T sn[N] = {pB[2 * CW] + pC[2 * CW]}, st[N] = {pB[CW] + pC[CW]}, dT[N] = {pC[4 * CW] - pB[4 * CW]};
        const T cn[N] = {vc[0]}, cc[N] = {vc[1]}, cs[N] = {vc[2]}, ct[N] = {vc[3]}, cq[N] = {vc[4]};
        viscous_n<T, N>(dn, dt_, xt, xn, sn, st, dT, cn, cc, cs, ct, cq, f1, f2, f3);
      }
      Gp[0] = f0[0]; Gp[1] = f1[0]; Gp[2] = f2[0]; Gp[3] = f3[0];
      if (fluid && in_x) fl_next = fluid[(size_t)(jo + 1 - 3 - rb) * A.nx + ic];
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) Ly[k] = Lnew[k];
    if (VISC) { cuP = cuC; cvP = cvC; }
    rotate();
  }

  // ---------------------------------------------------------------- main loop: one output row per iteration
  // LyI / GpI / cuI / cvI / EpI: the carried state read by this row, ..O: where the next row finds it; older / newer:
  // the y-reconstruction's carried differences.  Two rows alternate between two sets of registers (the loop below is
  // unrolled by two), so no register copies rotate the carried state (measured: 20 moves per row, 1.6 % of the time).
  auto body = [&](const int n, const T (&LyI)[4], T (&LyO)[4], const T (&GpI)[4], T (&GpO)[4], const T& cuI, const T& cvI,
                  T& cuO, T& cvO, YCarry<T, 4>& older, const YCarry<T, 4>& newer, const T (&EpI)[4], T (&EpO)[4]) {
    const int it = n - nfirst;
    take_row(n, it, A.mode == 0, EpO);
    const int jo = n - 3;  // output row = pB; pC = jc
    const unsigned fl = fl_next;
    if (n < nlast && fluid && in_x) fl_next = fluid[(size_t)(jo + 1 - 3 - rb) * A.nx + ic];
    // S5': network outputs at my right face and my top face (row jo): one 16-byte load per cell, fetched a whole row
    // ahead (like the fluid flag) so that its latency never meets the use
    const uint4 y8 = y_next;
    if (MLP && n < nlast) y_next = __ldg(A.dFG + (size_t)(jo + 1) * A.pitch + (w0 + lane));

    // -------------------------------------------------------------- S4 along y (centre jc) and along x (row jo)
    T Ry[4], Lnew[4], cuC = T(0), cvC = T(0);
    weno_y(older, newer, EpI, EpO, Ry, Lnew, cuC, cvC);
    T wc[4], Rm[4], Lp[4];  // my primitives; right state at my left face, left state at my right face
    {
      constexpr int N = 4;
      T a[N], b[N], d[N], e[N];
      JXS_V { a[k] = pB[k * CW - 2]; b[k] = pB[k * CW - 1]; wc[k] = pB[k * CW]; d[k] = pB[k * CW + 1]; e[k] = pB[k * CW + 2]; }
      weno5_n<T, N>(a, b, wc, d, e, A, Rm, Lp);
      const bool badR = any_not_positive(Rm[0], Rm[3]);
      const bool badL = any_not_positive(Lp[0], Lp[3]);
      if (__any_sync(0xffffffffu, badR | badL)) {
        asm volatile("" ::: "memory");
        JXS_V { Rm[k] = badR ? wc[k] : Rm[k]; Lp[k] = badL ? wc[k] : Lp[k]; }
      }
    }

    // -------------------------------------------------------------- S5 (+S5', S6): the face above row jo (0) and my right face (1)
    T f0[2], f1[2], f2[2], f3[2];  // (mass, normal momentum, tangential momentum, energy)
    {
      constexpr int N = 2;
      const T rL[N] = {LyI[0], Lp[0]}, unL[N] = {LyI[2], Lp[1]}, utL[N] = {LyI[1], Lp[2]}, pL[N] = {LyI[3], Lp[3]};
      const T rR[N] = {Ry[0], shfl_down1(Rm[0])}, unR[N] = {Ry[2], shfl_down1(Rm[1])},
              utR[N] = {Ry[1], shfl_down1(Rm[2])}, pR[N] = {Ry[3], shfl_down1(Rm[3])};
      hllc_n<T, N>(rL, unL, utL, pL, rR, unR, utR, pR, gamma, g1inv, f0, f1, f2, f3);
      if (MLP) {  // Eq. 11
        float yF[4], yG[4];
        unpack_half4(y8.x, y8.y, yF);
        unpack_half4(y8.z, y8.w, yG);
        f0[0] = fma_(A.oscale[0], T(yG[0]), f0[0]); f0[1] = fma_(A.oscale[0], T(yF[0]), f0[1]);
        f1[0] = fma_(A.oscale[1], T(yG[1]), f1[0]); f1[1] = fma_(A.oscale[1], T(yF[1]), f1[1]);
        f2[0] = fma_(A.oscale[2], T(yG[2]), f2[0]); f2[1] = fma_(A.oscale[2], T(yF[2]), f2[1]);
        f3[0] = fma_(A.oscale[3], T(yG[3]), f3[0]); f3[1] = fma_(A.oscale[3], T(yF[3]), f3[1]);
      }
      if (VISC) {
        // y-face between rows jo and jc: normal velocity v.  x-face at my right: normal velocity u; the
        // y-centred cross differences (rows jo+1 = jc and jo-1) of the right neighbour come by shuffle
        // (lane 31 gets its own back: its face flux is not used)
        const T u1 = pB[CW + 1], v1 = pB[2 * CW + 1];
        const T cu0 = pC[CW] - pA[CW], cv0 = pC[2 * CW] - pA[2 * CW];
        const T cu1 = shfl_down1(cu0), cv1 = shfl_down1(cv0);
        const T dn[N] = {pC[2 * CW] - pB[2 * CW], u1 - wc[1]}, dt_[N] = {pC[CW] - pB[CW], v1 - wc[2]};
        const T xt[N] = {cuI + cuC, cv0 + cv1}, xn[N] = {cvI + cvC, cu0 + cu1};
        const T sn[N] = {pB[2 * CW] + pC[2 * CW], wc[1] + u1}, st[N] = {pB[CW] + pC[CW], wc[2] + v1};
        const T dT[N] = {pC[4 * CW] - pB[4 * CW], pB[4 * CW + 1] - pB[4 * CW]};
        const T cn[N] = {vc[0], vc[5]}, cc[N] = {vc[1], vc[6]}, cs[N] = {vc[2], vc[7]}, ct[N] = {vc[3], vc[8]},
                cq[N] = {vc[4], vc[9]};
        viscous_n<T, N>(dn, dt_, xt, xn, sn, st, dT, cn, cc, cs, ct, cq, f1, f2, f3);
      }
    }

    // -------------------------------------------------------------- S7: divergence (conserved order rho, rho u, rho v, E)
    T Lc[4];
    {
      const T Fx[4] = {f0[1], f1[1], f2[1], f3[1]};
      const T Gy[4] = {f0[0], f2[0], f1[0], f3[0]};
      const T Gb[4] = {GpI[0], GpI[2], GpI[1], GpI[3]};
      T dy_[4], Fl[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) Fl[k] = shfl_up1(Fx[k]);
#pragma unroll
      for (int k = 0; k < 4; ++k) dy_[k] = Gb[k] - Gy[k];
#pragma unroll
      for (int k = 0; k < 4; ++k) Fl[k] = Fl[k] - Fx[k];
#pragma unroll
      for (int k = 0; k < 4; ++k) dy_[k] = dy_[k] * A.dyi;
#pragma unroll
      for (int k = 0; k < 4; ++k) Lc[k] = fma_(Fl[k], A.dxi, dy_[k]);
      GpO[0] = f0[0]; GpO[1] = f1[0]; GpO[2] = f2[0]; GpO[3] = f3[0];
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) LyO[k] = Lnew[k];
    if (VISC) { cuO = cuC; cvO = cvC; }

    if (ARTV) {  // nu * Lap_h(U) on the conserved variables (Eq. 10), rebuilt from the primitives
      auto cons = [&](const T* row, int c, T* U) {
        const T r = row[c], u = row[CW + c], v = row[2 * CW + c], p = row[3 * CW + c];
        U[0] = r; U[1] = r * u; U[2] = r * v; U[3] = fma_(T(0.5) * r, fma_(u, u, v * v), p * g1inv);
      };
      T Um[4], Uxm[4], Uxp[4], Ud[4], Uu[4];
      cons(pB, 0, Um); cons(pB, -1, Uxm); cons(pB, 1, Uxp); cons(pA, 0, Ud); cons(pC, 0, Uu);
      const T ax = A.nu * A.dxi * A.dxi, ay = A.nu * A.dyi * A.dyi;
#pragma unroll
      for (int k = 0; k < 4; ++k)
        Lc[k] += ax * (Uxp[k] - T(2) * Um[k] + Uxm[k]) + ay * (Uu[k] - T(2) * Um[k] + Ud[k]);
    }

    // -------------------------------------------------------------- S8, S9: combine, store, wavespeed
    const bool ok = lane >= 1 && lane <= SOUT && in_x;  // lanes 0 and > SOUT are support cells
    if (A.mode == 1) {
      const size_t pl = (size_t)A.nx * A.ny, o = (size_t)(jo - 3 - rb) * A.nx + ic + (BATCH ? 4 * pl * member : 0);
      if (ok) {
#pragma unroll
        for (int k = 0; k < 4; ++k) A.Uout[k * pl + o] = fl ? Lc[k] : T(0);
      }
    } else {
      mbar_wait(bar_epi, (it + 1) & 1);  // phase 0 was the warm-up rows
      const T dtf = fl ? dtv : T(0);  // non-fluid cells keep their state
      T Un[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) Un[k] = fma_(dtf, Lc[k], epi[k * EW + lane + EOFF]);
      if (use_u0) {
#pragma unroll
        for (int k = 0; k < 4; ++k) Un[k] = A.rk_b * Un[k];
#pragma unroll
        for (int k = 0; k < 4; ++k) Un[k] = fma_(A.rk_a, epi0[k * EW + lane + EOFF], Un[k]);
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
    rotate();
  };
  {
    T LyB[4] = {T(0), T(0), T(0), T(0)}, GpB[4] = {T(0), T(0), T(0), T(0)}, cuB = T(0), cvB = T(0);
#pragma unroll 1
    for (int n = nfirst + 6; n <= nlast; n += 2) {
      body(n, Ly, LyB, Gp, GpB, cuP, cvP, cuB, cvB, ycA, ycB, Ep1, Ep0);
      if (n + 1 > nlast) break;
      body(n + 1, LyB, Ly, GpB, Gp, cuB, cvB, cuP, cvP, ycB, ycA, Ep0, Ep1);
    }
  }
  if (A.smax_bits) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const T other = __shfl_xor_sync(0xffffffffu, smax, o);
      smax = (other > smax || other != other) ? other : smax;
    }
    if (lane == 0)
      atomic_max_pos(reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(A.smax_bits) + (BATCH ? member * A.state_stride : 0)),
                     (double)smax);
  }
}

#undef JXS_V

}  // namespace jxs
