// flux_mlp_kernel.cuh — S5' of DESIGN.md §1: the per-face neural flux correction (Eq. 11,
// L109; BASELINE.json configs[4]; reading R14) on the 5th-generation tensor cores of sm_100a.
//
//   x (24 stencil primitives / in_scale, bf16) -> tanh(W1 x + b1) -> tanh(W2 h1 + b2) -> W3 h2 + b3
//
// One CTA = 4 warps = 128 threads marches a strip of 128 cells upwards, one row per iteration.  Thread
// t owns the cell in column c0+t and evaluates the network for TWO faces of that cell: its right face
// (x-face i+1/2: cells i-2..i+3 of the row) and its top face (y-face j+1/2: rows j-2..j+3 of the column,
// normal velocity first).  The two sets of 128 faces are the M = 128 rows of two tcgen05.mma tiles:
//   layer 1  D[128 x 64] = A1[128 x 32] W1^T     (K = 24 padded to 32, 2 MMAs of K = 16 per tile)
//   layer 2  D[128 x 64] = A2[128 x 64] W2^T     (4 MMAs per tile)
//   layer 3  D[128 x 16] = A2[128 x 64] W3^T     (N = 4 padded to 16, 4 MMAs per tile)
// A operands are written by the threads into shared memory in the canonical K-major no-swizzle layout
// (8 x 16-byte core matrices), weights sit there for the whole kernel, accumulators live in TMEM
// (128 columns per CTA: two 64-column tiles, reused by every layer).  TMEM lane m = face m = thread m,
// so tcgen05.ld (32x32b) hands every thread the pre-activations of its own face; bias, tanh
// (tanh.approx.f32, then one rounding to bf16 — the rounding points of the oracle's emulating mode; the
// packed tanh.approx.bf16x2 was measured: SASS splits it into two MUFU operations, so it is no faster,
// and its extra input rounding costs 1e-2 of accuracy) and the store of the next A operand follow in
// registers.  Completion of the MMAs is tracked with
// tcgen05.commit on an mbarrier.
// The scaled bf16 primitives of the last 6 rows are kept in a shared-memory ring; a row is converted
// once.  Output: y (before out_scale) per face as fp16, one uint4 per padded cell (row, col): {right face: 4, top
// face: 4}, k = (mass, normal, tangential momentum, energy).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace jxs {

constexpr int MLP_TILE = 128;               // faces per MMA tile = threads per CTA
constexpr int MLP_RING = 6;                 // rows of bf16 primitives kept
constexpr int MLP_RW = MLP_TILE + 5;        // ring row width: 2 halo cells left, 3 right
constexpr int MLP_TMEM_COLS = 128;
// shared-memory carve-up (bytes)
constexpr int MLP_OFF_W1 = 0;                         // [64 x 32] bf16 canonical, 4 KB
constexpr int MLP_OFF_W2 = MLP_OFF_W1 + 64 * 32 * 2;  // [64 x 64] 8 KB
constexpr int MLP_OFF_W3 = MLP_OFF_W2 + 64 * 64 * 2;  // [16 x 64] 2 KB
constexpr int MLP_WBLOB = MLP_OFF_W3 + 16 * 64 * 2;   // 14336 B of weights, then 132 floats of biases
constexpr int MLP_OFF_BIAS = MLP_WBLOB;               // b1[64] b2[64] b3[4]
constexpr int MLP_BLOB = MLP_OFF_BIAS + 132 * 4;      // what jxs_set_flux_mlp uploads
constexpr int MLP_OFF_A1 = 14976;                     // 2 tiles [128 x 32] bf16, 8 KB each ...
constexpr int MLP_OFF_A2 = MLP_OFF_A1;                // ... inside the 2 tiles [128 x 64] bf16, 16 KB each, of the
                                                      // hidden layers (written after layer 1 has read its operands):
                                                      // 54 KB per CTA, 4 CTAs = 16 warps and all 512 TMEM columns per SM
constexpr int MLP_OFF_RING = MLP_OFF_A2 + 2 * 16384;  // [6][133] uint2
constexpr int MLP_OFF_BAR = MLP_OFF_RING + MLP_RING * MLP_RW * 8 + 8;
constexpr int MLP_SMEM = MLP_OFF_BAR + 16;
static_assert(MLP_OFF_A1 >= MLP_BLOB && MLP_OFF_A1 % 128 == 0, "A tiles must not overlap the weights");
static_assert(MLP_OFF_BAR % 8 == 0, "mbarrier alignment");

template <typename T>
struct MlpArgs {
  const T* U;            // padded [4][ny+6][pitch], ghosts filled
  uint4* dFG;            // [rows][pitch]: per padded cell eight fp16 network outputs {right face: 4, top face: 4}
  const uint8_t* blob;   // MLP_BLOB bytes: canonical bf16 weights + fp32 biases
  long long plane;
  int nx, ny, pitch;
  int nstrips, rows_per_seg;
  int nseg;              // row segments per strip and member of a batch (members are stacked along y, ny+6 rows each)
  T g1;                  // gamma - 1
  T inv_scale[4];        // 1 / in_scale of (rho, u_n, u_t, p)
  float bias[132];       // b1[64] b2[64] b3[4]: kernel parameters, i.e. constant-bank operands of the bias adds
};

// ---- tcgen05 / TMEM wrappers (PTX ISA: tcgen05.*) ------------------------------------------------
__device__ __forceinline__ void tmem_alloc(uint32_t slot_smem, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot_smem), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// D[tmem] (+)= A[smem] * B[smem]^T, bf16 in, fp32 accumulate; issued by ONE thread
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
               ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrive on the mbarrier when every MMA issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// 32 lanes x 32 consecutive fp32 columns: thread t of the warp receives lane (lane_base + t)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
      "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&r)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr) : "memory");
}

// Shared-memory matrix descriptor, K-major, no swizzle: element (m, k) of a bf16 tile at
//   (m / 8) * SBO + (k / 8) * LBO + (m % 8) * 16 + (k % 8) * 2     (8 x 16-byte core matrices)
// bits [0,14) address >> 4, [16,30) LBO >> 4, [32,46) SBO >> 4, [46,48) version = 1, [61,64) swizzle = 0
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | (1ull << 46);
}
// Instruction descriptor of kind::f16: fp32 accumulate (bits 4-5 = 1), A and B bf16 (bits 7-9, 10-12 = 1),
// both K-major (bits 15, 16 = 0), N >> 3 in bits 17-22, M >> 4 in bits 24-28
__host__ __device__ constexpr uint32_t umma_idesc(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ float tanh_f32(float x) {
  float d;
  asm("tanh.approx.f32 %0, %1;" : "=f"(d) : "f"(x));
  return d;
}
__device__ __forceinline__ void mbar_wait_spin(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  } while (!ok);
}

// hidden layer epilogue of one tile: 64 pre-activations of my face (TMEM) -> + bias -> tanh -> bf16 -> A2 row
__device__ __forceinline__ void hidden_epilogue(uint32_t taddr, const float (&bias)[64], unsigned char* a2_tile, int m) {
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    uint32_t v[32];
    tmem_ld32(taddr + half * 32, v);
    tmem_ld_wait();
#pragma unroll
    for (int c = 0; c < 4; ++c) {  // 16-byte chunk = 8 activations k = 32*half + 8c .. +7
      uint32_t w[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int k = 8 * c + 2 * e;
        const float s0 = __uint_as_float(v[k]) + bias[32 * half + k];
        const float s1 = __uint_as_float(v[k + 1]) + bias[32 * half + k + 1];
        w[e] = pack_bf16(tanh_f32(s0), tanh_f32(s1));
      }
      *reinterpret_cast<uint4*>(a2_tile + (4 * half + c) * 2048 + m * 16) = make_uint4(w[0], w[1], w[2], w[3]);
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(MLP_TILE, 4) flux_mlp_kernel(const MlpArgs<T> A) {
  extern __shared__ __align__(128) unsigned char sm[];
  __shared__ uint32_t tmem_slot;
  const int t = threadIdx.x, warp = t >> 5;
  const int strip = blockIdx.x % A.nstrips, seg_all = blockIdx.x / A.nstrips;
  const int member = seg_all / A.nseg, seg = seg_all - member * A.nseg;
  const int rb = member * (A.ny + 6);  // first padded row of my member
  // cell rows whose faces this CTA evaluates: padded rows [rbeg, rend) of this member's [2, ny+3)
  const int rbeg = rb + 2 + seg * A.rows_per_seg;
  const int rend = min(rbeg + A.rows_per_seg, rb + A.ny + 3);
  if (rbeg >= rend) return;
  const int c0 = 2 + MLP_TILE * strip;  // padded column of thread 0's cell
  const int col = c0 + t;

  const uint32_t sm_u32 = (uint32_t)__cvta_generic_to_shared(sm);
  const uint32_t bar = sm_u32 + MLP_OFF_BAR;
  float b1[64], b2[64];  // compile-time indexed below: they stay constant-bank operands
#pragma unroll
  for (int k = 0; k < 64; ++k) { b1[k] = A.bias[k]; b2[k] = A.bias[64 + k]; }
  uint2* ring = reinterpret_cast<uint2*>(sm + MLP_OFF_RING);

  // ---- one-time set-up: weights -> smem, zero the K padding of the layer-1 A tiles, TMEM, mbarrier
  for (int i = t; i < MLP_BLOB / 16; i += MLP_TILE)
    reinterpret_cast<uint4*>(sm)[i] = reinterpret_cast<const uint4*>(A.blob)[i];
  if (t == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(1) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) tmem_alloc((uint32_t)__cvta_generic_to_shared(&tmem_slot), MLP_TMEM_COLS);
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t tlane = tmem + ((uint32_t)(32 * warp) << 16);  // my warp's lane quarter

  constexpr uint32_t IDESC_H = umma_idesc(128, 64), IDESC_O = umma_idesc(128, 16);
  uint32_t phase = 0;

  // conserved row n, ring column x -> scaled bf16 primitives (rho, u, v, p)
  auto load_row = [&](int n, int x, T (&q)[4]) {
    const int gc = min(c0 - 2 + x, A.pitch - 1);
    const T* s = A.U + (size_t)n * A.pitch + gc;
#pragma unroll
    for (int k = 0; k < 4; ++k) q[k] = s[k * A.plane];
  };
  auto convert = [&](const T (&q)[4]) -> uint2 {
    const T ri = T(1) / q[0];
    const T u = q[1] * ri, v = q[2] * ri;
    const T p = A.g1 * (q[3] - T(0.5) * (q[1] * u + q[2] * v));
    uint2 o;
    o.x = pack_bf16((float)(q[0] * A.inv_scale[0]), (float)(u * A.inv_scale[1]));
    o.y = pack_bf16((float)(v * A.inv_scale[2]), (float)(p * A.inv_scale[3]));
    return o;
  };

  const int nfirst = rbeg - 2, nlast = rend + 2;  // rows to stream, inclusive
  T q0[4], q1[4];
  load_row(nfirst, t, q0);
  if (t < 5) load_row(nfirst, MLP_TILE + t, q1);

  for (int n = nfirst; n <= nlast; ++n) {
    const int it = n - nfirst;
    const int slot = it % MLP_RING;
    // ---- S3': new row -> ring (the slot was last read two barriers ago)
    ring[slot * MLP_RW + t] = convert(q0);
    if (t < 5) ring[slot * MLP_RW + MLP_TILE + t] = convert(q1);
    if (n < nlast) {  // next row's loads fly during this iteration
      load_row(n + 1, t, q0);
      if (t < 5) load_row(n + 1, MLP_TILE + t, q1);
    }
    __syncthreads();
    if (it < 5) continue;
    const int r = n - 3;  // the cell row whose right and top faces are evaluated

    // ---- layer-1 A operands: x tile (cells c-2..c+3 of row r), y tile (rows r-2..r+3, normal first)
    {
      const int sr = (it - 3) % MLP_RING;
      const uint2* rx = ring + sr * MLP_RW + t;
      unsigned char* a1x = sm + MLP_OFF_A1 + t * 16;
      unsigned char* a1y = a1x + 8192;
      // K = 24 padded to 32: the last chunk is zero (the hidden layers' operands overwrite it every row)
      *reinterpret_cast<uint4*>(a1x + 3 * 2048) = make_uint4(0, 0, 0, 0);
      *reinterpret_cast<uint4*>(a1y + 3 * 2048) = make_uint4(0, 0, 0, 0);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const uint2 e0 = rx[2 * c], e1 = rx[2 * c + 1];
        *reinterpret_cast<uint4*>(a1x + c * 2048) = make_uint4(e0.x, e0.y, e1.x, e1.y);
        const uint2 f0 = ring[((it - 5 + 2 * c) % MLP_RING) * MLP_RW + t + 2];
        const uint2 f1 = ring[((it - 4 + 2 * c) % MLP_RING) * MLP_RW + t + 2];
        *reinterpret_cast<uint4*>(a1y + c * 2048) =
            make_uint4(__byte_perm(f0.x, f0.y, 0x5410), __byte_perm(f0.x, f0.y, 0x7632),
                       __byte_perm(f1.x, f1.y, 0x5410), __byte_perm(f1.x, f1.y, 0x7632));
      }
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (t == 0) {
      tc_fence_after();
#pragma unroll
      for (int tile = 0; tile < 2; ++tile)
#pragma unroll
        for (int ks = 0; ks < 2; ++ks)
          umma_bf16(tmem + 64 * tile, umma_desc(sm_u32 + MLP_OFF_A1 + tile * 8192 + ks * 4096, 2048, 128),
                    umma_desc(sm_u32 + MLP_OFF_W1 + ks * 2048, 1024, 128), IDESC_H, ks);
      umma_commit(bar);
    }
    mbar_wait_spin(bar, phase); phase ^= 1;
    tc_fence_after();

    // ---- hidden layer 1 -> A2, layer 2
    hidden_epilogue(tlane, b1, sm + MLP_OFF_A2, t);
    hidden_epilogue(tlane + 64, b1, sm + MLP_OFF_A2 + 16384, t);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (t == 0) {
      tc_fence_after();
#pragma unroll
      for (int tile = 0; tile < 2; ++tile)
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          umma_bf16(tmem + 64 * tile, umma_desc(sm_u32 + MLP_OFF_A2 + tile * 16384 + ks * 4096, 2048, 128),
                    umma_desc(sm_u32 + MLP_OFF_W2 + ks * 2048, 1024, 128), IDESC_H, ks);
      umma_commit(bar);
    }
    mbar_wait_spin(bar, phase); phase ^= 1;
    tc_fence_after();

    // ---- hidden layer 2 -> A2 (layer 2 has finished reading it), output layer (N = 16)
    hidden_epilogue(tlane, b2, sm + MLP_OFF_A2, t);
    hidden_epilogue(tlane + 64, b2, sm + MLP_OFF_A2 + 16384, t);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (t == 0) {
      tc_fence_after();
#pragma unroll
      for (int tile = 0; tile < 2; ++tile)
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          umma_bf16(tmem + 64 * tile, umma_desc(sm_u32 + MLP_OFF_A2 + tile * 16384 + ks * 4096, 2048, 128),
                    umma_desc(sm_u32 + MLP_OFF_W3 + ks * 512, 256, 128), IDESC_O, ks);
      umma_commit(bar);
    }
    mbar_wait_spin(bar, phase); phase ^= 1;
    tc_fence_after();

    // ---- y = W3 h2 + b3 of my two faces -> HBM
    {
      uint32_t yx[4], yy[4];
      tmem_ld4(tlane, yx);
      tmem_ld4(tlane + 64, yy);
      tmem_ld_wait();
      if (col <= A.nx + 2) {
        float fx[4], fy[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          fx[k] = __uint_as_float(yx[k]) + A.bias[128 + k];
          fy[k] = __uint_as_float(yy[k]) + A.bias[128 + k];
        }
        A.dFG[(size_t)r * A.pitch + col] = make_uint4(pack_half2(fx[0], fx[1]), pack_half2(fx[2], fx[3]),
                                                      pack_half2(fy[0], fy[1]), pack_half2(fy[2], fy[3]));
      }
    }
    tc_fence_before();  // the next iteration's MMAs overwrite the columns just read
  }
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, MLP_TMEM_COLS);
}

}  // namespace jxs
