// flux_mlp_kernel.cuh — S5' of DESIGN.md §1: the per-face neural flux correction (Eq. 11,
// L109; BASELINE.json configs[4]; reading R14) on the 5th-generation tensor cores of sm_100a.
//
//   x (24 stencil primitives / in_scale, bf16) -> tanh(W1 x + b1) -> tanh(W2 h1 + b2) -> W3 h2 + b3
//
// One CTA = 8 warps = two warpgroups marches a strip of 128 cells upwards, one row per iteration.  Thread lt
// (0..127) of warpgroup 0 owns the RIGHT face of the cell in column c0+lt (x-face i+1/2: cells i-2..i+3 of the
// row), thread lt of warpgroup 1 its TOP face (y-face j+1/2: rows j-2..j+3 of the column, normal velocity
// first).  The 128 faces of a warpgroup are the M = 128 rows of its own chain of tcgen05.mma tiles:
//   layer 1  D[128 x 64] = A1[128 x 32] W1^T     (K = 24 padded to 32, 2 MMAs of K = 16)
//   layer 2  D[128 x 64] = A2[128 x 64] W2^T     (4 MMAs)
//   layer 3  D[128 x 16] = A3[128 x 64] W3^T     (N = 4 padded to 16, 4 MMAs)
// The A operands live in TENSOR MEMORY (tcgen05.mma with [a_tmem]: lane m = row m, 32-bit column c = the bf16
// pair k = 2c, 2c+1): every thread writes the row of its own face with tcgen05.st and the tensor core reads
// it from there, so an MMA fetches only its 0.5-2 KB weight tile from shared memory and runs at the
// 128 N / 256-cycle floor (32 cycles for N = 64) instead of the ~100 cycles that the 4 KB A tile in shared
// memory cost (profiles/r02_flux_mlp.md).  Per warpgroup 96 TMEM columns: X = [0, 32) the A operand of the
// current layer, Y = [32, 96) its accumulator; TMEM lane m = face m = thread m, so tcgen05.ld (32x32b)
// hands every thread the pre-activations of its own face; bias, tanh (tanh.approx.f32, then one rounding to
// bf16 — the rounding points of the oracle's emulating mode; the packed tanh.approx.bf16x2 was measured: SASS
// splits it into two MUFU operations, so it is no faster, and its extra input rounding costs 1e-2 of
// accuracy) and the tcgen05.st of the next A operand follow in registers.  The two warpgroups run their
// chains independently (a named barrier and an mbarrier each) and meet once per row, when the new row of
// primitives enters the ring; two CTAs per SM (all 512 TMEM columns) = four independent chains that keep the
// SFU (tanh: the binding unit, 128 per face) busy while one of them waits for its MMAs.
// The scaled bf16 primitives of the last 7 rows are kept in a shared-memory ring; a row is converted
// once.  Output: y (before out_scale) per face as fp16, one uint4 per padded cell (row, col): {right face: 4, top
// face: 4}, k = (mass, normal, tangential momentum, energy).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace jxs {

constexpr int MLP_TILE = 128;               // faces per MMA tile = threads per warpgroup
constexpr int MLP_THREADS = 2 * MLP_TILE;   // warpgroup 0: x-faces, warpgroup 1: y-faces
constexpr int MLP_RING = 7;                 // rows of bf16 primitives kept (6 read + the one being written)
constexpr int MLP_RW = MLP_TILE + 5;        // ring row width: 2 halo cells left, 3 right
constexpr int MLP_TMEM_COLS = 256;          // 128 per warpgroup, 96 used: X = [0, 32), Y = [32, 96)
// shared-memory carve-up (bytes)
constexpr int MLP_OFF_W1 = 0;                         // [64 x 32] bf16 canonical, 4 KB
constexpr int MLP_OFF_W2 = MLP_OFF_W1 + 64 * 32 * 2;  // [64 x 64] 8 KB
constexpr int MLP_OFF_W3 = MLP_OFF_W2 + 64 * 64 * 2;  // [16 x 64] 2 KB
constexpr int MLP_WBLOB = MLP_OFF_W3 + 16 * 64 * 2;   // 14336 B of weights, then 132 floats of biases
constexpr int MLP_OFF_BIAS = MLP_WBLOB;               // b1[64] b2[64] b3[4]
constexpr int MLP_BLOB = MLP_OFF_BIAS + 132 * 4;      // what jxs_set_flux_mlp uploads
constexpr int MLP_OFF_RING = 14976;                   // [7][133] uint2
constexpr int MLP_OFF_BAR = MLP_OFF_RING + MLP_RING * MLP_RW * 8 + 8;  // one mbarrier per warpgroup
constexpr int MLP_SMEM = MLP_OFF_BAR + 16;
static_assert(MLP_OFF_RING >= MLP_BLOB && MLP_OFF_RING % 16 == 0, "the ring must not overlap the weights");
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

// D[tmem] (+)= A[tmem] * B[smem]^T: the A operand is read from tensor memory (lane = row, 8 columns per K = 16)
__device__ __forceinline__ void umma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n}"
               ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// 16 consecutive 32-bit columns of my lane <- w[0..15]
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&w)[16]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
               ::"r"(taddr), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]), "r"(w[8]),
                 "r"(w[9]), "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void wg_barrier(int wg) { asm volatile("bar.sync %0, 128;" ::"r"(1 + wg) : "memory"); }

