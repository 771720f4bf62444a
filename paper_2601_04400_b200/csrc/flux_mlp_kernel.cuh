// flux_mlp_kernel.cuh — S5' of DESIGN.md §1: the per-face neural flux correction (Eq. 11,
// L109; BASELINE.json configs[4]; reading R14) on the 5th-generation tensor cores of sm_100a.
//
//   x (24 stencil primitives / in_scale, bf16) -> tanh(W1 x + b1) -> tanh(W2 h1 + b2) -> W3 h2 + b3
//
// One CTA per SM = 26 warps marches a strip of 128 cells upwards.  The 128 RIGHT faces of a cell row (x-face i+1/2:
// cells i-2..i+3 of the row) and its 128 TOP faces (y-face j+1/2: rows j-2..j+3 of the column, normal velocity
// first) are the M = 128 rows of two chains (directions g = 0, 1) of tcgen05.mma tiles:
//   layer 1  D[128 x 64] = A1[128 x 32] W1^T     (K = 24 padded to 32, 2 MMAs of K = 16)
//   layer 2  D[128 x 64] = A2[128 x 64] W2^T     (4 MMAs)
//   layer 3  D[128 x 16] = A3[128 x 64] W3^T     (N = 4 padded to 16, 4 MMAs)
// and each direction works on TWO rows at once (tile slots s = 0: even rows of the segment, s = 1: odd rows): four
// independent chains, so that the MMAs of one (and the ~230 cycles a commit takes to come back) run under the tanh of
// the others.  What binds is the SFU (128 tanh per face at 16 per clock and SM); the schedule exists to keep
// MUFU.TANH issuing.
// The A operands live in TENSOR MEMORY (tcgen05.mma with [a_tmem]: lane m = row m, 32-bit column c = the bf16
// pair k = 2c, 2c+1): threads write the row of their own face with tcgen05.st and the tensor core reads it there;
// only the 0.5-2 KB weight tile of an MMA comes from shared memory.  A slot owns 128 of the SM's 512 TMEM columns:
//   X  = [0, 32)     A operand of layers 2 and 3 (the bf16 hidden activations)
//   Y  = [32, 96)    accumulator of layers 1 and 2 (64 pre-activations per face)
//   A1 = [96, 112)   layer-1 operand of the slot's NEXT row (24 inputs + padding)
//   O  = [112, 128)  accumulator of the output layer
// TMEM lane m = face m, so tcgen05.ld (32x32b) hands a thread the pre-activations of its own face; bias, tanh
// (tanh.approx.f32, then one rounding to bf16 - the rounding points of the oracle's emulating mode; the packed
// tanh.approx.bf16x2 was measured: SASS splits it into two MUFU operations, so it is no faster, and its extra input
// rounding costs 1e-2 of accuracy) and the tcgen05.st of the next operand follow in registers.
// Warp roles:
//   warps 0-15   four tanh warpgroups, (direction g, half h of the 64 hidden units): wait d_full[g][s] -> load 32
//                pre-activations -> tanh -> store 16 packed columns of X -> arrive a_full[g][s]; slots alternate
//   warps 16-19  the builder warpgroup, both directions, off the critical path: once layer 1 of a row has read A1
//                (l1_done) it builds the slot's next row there from the ring (a1_full); it reads the output layer's
//                accumulator (o_full), frees it (o_free) and writes y + b3 as fp16 to HBM
//   warps 20, 21 one lane each issues the MMAs of a direction as their operands become ready and commits them
//   warps 22-25  producers: conserved row n (n = p mod 4 for producer p) from HBM -> scaled bf16 primitives (fp32
//                arithmetic: they are rounded to 8 bits next) in a 10-row shared-memory ring (ring_full / ring_empty)
// Hand-over is by mbarriers only, one arrival per warp; nothing in the loop is a CTA-wide barrier.
// Output: y (before out_scale) per face as fp16, one uint4 per padded cell (row, col): {right face: 4, top
// face: 4}, k = (mass, normal, tangential momentum, energy).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace jxs {

constexpr int MLP_TILE = 128;               // faces per MMA tile = threads per warpgroup
constexpr int MLP_PRODUCERS = 4;           // producer warps: warp p converts the rows n = p (mod 4) of the segment
constexpr int MLP_THREADS = 5 * MLP_TILE + (2 + MLP_PRODUCERS) * 32;  // four tanh warpgroups, one builder warpgroup, two MMA warps, the producers
constexpr int MLP_RING = 10;                // rows of bf16 primitives kept (rows r-2 .. r+4 of a row pair + slack)
constexpr int MLP_RW = MLP_TILE + 5;        // ring row width: 2 halo cells left, 3 right
// nanoseconds between two polls of an mbarrier, by role (tanh warps, builders, producers, MMA lanes): a waiting warp
// should not crowd the SM's MIO queue, through which the working warps' MUFU and tcgen05.ld / st go as well (measured
// neutral against plain spinning: 0.675 against 0.677 ms)
constexpr unsigned PAUSE_T = 32, PAUSE_B = 64, PAUSE_P = 128, PAUSE_M = 20;
constexpr int MLP_TMEM_COLS = 512;          // [warpgroup][slot] x 128, 96 used: X = [0, 32), Y = [32, 96)
// shared-memory carve-up (bytes)
constexpr int MLP_OFF_W1 = 0;                         // [64 x 32] bf16 canonical, 4 KB
constexpr int MLP_OFF_W2 = MLP_OFF_W1 + 64 * 32 * 2;  // [64 x 64] 8 KB
constexpr int MLP_OFF_W3 = MLP_OFF_W2 + 64 * 64 * 2;  // [16 x 64] 2 KB
constexpr int MLP_WBLOB = MLP_OFF_W3 + 16 * 64 * 2;   // 14336 B of weights, then 132 floats of biases
constexpr int MLP_OFF_BIAS = MLP_WBLOB;               // b1[64] b2[64] b3[4]
constexpr int MLP_BLOB = MLP_OFF_BIAS + 132 * 4;      // what jxs_set_flux_mlp uploads
constexpr int MLP_OFF_RING = 14976;                   // [10][133] uint2
// mbarriers: a_full, d_full, o_full, a1_full, l1_done, o_free (each [2 directions][2 slots]), ring_full[MLP_RING], ring_empty[MLP_RING]
constexpr int MLP_OFF_BAR = MLP_OFF_RING + MLP_RING * MLP_RW * 8 + 8;
constexpr int MLP_SMEM = MLP_OFF_BAR + (24 + 2 * MLP_RING) * 8;
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
// wait with a pause between the polls: a waiting warp must not crowd the SM's MIO queue, through which the working warps'
// MUFU, tcgen05.ld / st and shared-memory instructions are issued as well
template <unsigned NS>
__device__ __forceinline__ void mbar_wait_pause(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  for (;;) {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) break;
    __nanosleep(NS);
  }
}
__device__ __forceinline__ void mlp_bar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
// one arrival for the whole warp: 128 or 256 separate arrivals on one barrier serialise in the shared-memory atomic unit
__device__ __forceinline__ void mbar_arrive_warp(uint32_t bar) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive2(uint32_t bar) {  // counts as two arrivals
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], 2;" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}


// hidden layer epilogue of one tile slot, column half H: 32 of the 64 pre-activations of my face (TMEM columns
// y + 32 H ..) -> + bias -> tanh -> bf16 pairs -> my half of the next layer's A operand (TMEM columns x + 16 H ..)
template <int H>
__device__ __forceinline__ void hidden_epilogue_ts(uint32_t y, uint32_t x, const float (&bias)[64]) {
  uint32_t v[32];
  tmem_ld32(y + 32 * H, v);
  tmem_ld_wait();
  uint32_t w[16];
#pragma unroll
  for (int e = 0; e < 16; ++e)
    w[e] = pack_bf16(tanh_f32(__uint_as_float(v[2 * e]) + bias[32 * H + 2 * e]),
                     tanh_f32(__uint_as_float(v[2 * e + 1]) + bias[32 * H + 2 * e + 1]));
  tmem_st16(x + 16 * H, w);
}

template <typename T>
__global__ void __launch_bounds__(MLP_THREADS, 1) flux_mlp_kernel(const MlpArgs<T> A) {
  extern __shared__ __align__(128) unsigned char sm[];
  __shared__ uint32_t tmem_slot;
  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
  const int strip = blockIdx.x % A.nstrips, seg_all = blockIdx.x / A.nstrips;
  const int member = seg_all / A.nseg, seg = seg_all - member * A.nseg;
  const int rb = member * (A.ny + 6);  // first padded row of my member
  // cell rows whose faces this CTA evaluates: padded rows [rbeg, rend) of this member's [2, ny+3)
  const int rbeg = rb + 2 + seg * A.rows_per_seg;
  const int rend = min(rbeg + A.rows_per_seg, rb + A.ny + 3);
  if (rbeg >= rend) return;
  const int c0 = 2 + MLP_TILE * strip;            // padded column of the cell of lt = 0
  const int nfirst = rbeg - 2, nlast = rend + 2;  // rows the producer streams, inclusive
  const int n0 = (rend - rbeg + 1) / 2, n1 = (rend - rbeg) / 2;  // rows of tile slot 0 (even) and 1 (odd)

  const uint32_t sm_u32 = (uint32_t)__cvta_generic_to_shared(sm);
  const uint32_t bars = sm_u32 + MLP_OFF_BAR;
  auto bar6 = [&](int kind, int g, int s) { return bars + 8 * (4 * kind + 2 * g + s); };
  auto a_full = [&](int g, int s) { return bar6(0, g, s); };   // 8 warps: the A operand of layer 2 / 3 is in X (tanh warps)
  auto d_full = [&](int g, int s) { return bar6(1, g, s); };   // commit: layer 1 / 2 has written Y
  auto o_full = [&](int g, int s) { return bar6(2, g, s); };   // commit: layer 3 has written O
  auto a1_full = [&](int g, int s) { return bar6(3, g, s); };  // 4 warps: the next row's layer-1 operand is in A1 (builders)
  auto l1_done = [&](int g, int s) { return bar6(4, g, s); };  // commit: layer 1 has read A1
  auto o_free = [&](int g, int s) { return bar6(5, g, s); };   // 4 warps: the builders have read O
  auto ring_full = [&](int slot) { return bars + 8 * (24 + slot); };
  auto ring_empty = [&](int slot) { return bars + 8 * (24 + MLP_RING + slot); };
  uint2* ring = reinterpret_cast<uint2*>(sm + MLP_OFF_RING);

  // ---- one-time set-up: weights -> smem, TMEM, mbarriers
  for (int i = t; i < MLP_BLOB / 16; i += MLP_THREADS)
    reinterpret_cast<uint4*>(sm)[i] = reinterpret_cast<const uint4*>(A.blob)[i];
  if (t == 0) {
    for (int q = 0; q < 4; ++q) {
      mlp_bar_init(a_full(q >> 1, q & 1), 8); mlp_bar_init(d_full(q >> 1, q & 1), 1);
      mlp_bar_init(o_full(q >> 1, q & 1), 1); mlp_bar_init(a1_full(q >> 1, q & 1), 4);
      mlp_bar_init(l1_done(q >> 1, q & 1), 1); mlp_bar_init(o_free(q >> 1, q & 1), 4);
    }
    for (int q = 0; q < MLP_RING; ++q) { mlp_bar_init(ring_full(q), 1); mlp_bar_init(ring_empty(q), 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) tmem_alloc((uint32_t)__cvta_generic_to_shared(&tmem_slot), MLP_TMEM_COLS);
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;

  if (warp >= 22) {
    // ================= producers: conserved row n -> scaled bf16 primitives (rho, u, v, p) of ring columns lane + 32 q
    constexpr int NQ = (MLP_RW + 31) / 32;
    T q[NQ][4];
    for (int n = nfirst + (warp - 22); n <= nlast; n += MLP_PRODUCERS) {
      const int it = n - nfirst, slot = it % MLP_RING;
#pragma unroll
      for (int c = 0; c < NQ; ++c) {
        const int gc = min(c0 - 2 + lane + 32 * c, A.pitch - 1);
        const T* src = A.U + (size_t)n * A.pitch + gc;
#pragma unroll
        for (int k = 0; k < 4; ++k) q[c][k] = src[k * A.plane];
      }
      if (it >= MLP_RING) mbar_wait_pause<PAUSE_P>(ring_empty(slot), (uint32_t)((it / MLP_RING - 1) & 1));
#pragma unroll
      for (int c = 0; c < NQ; ++c) {
        // fp32 is plenty ahead of a rounding to bf16 (8 significant bits), and the fp64 division was what made the
        // producers the slowest stage of the pipeline
        const float r = (float)q[c][0], ru = (float)q[c][1], rv = (float)q[c][2], E = (float)q[c][3];
        const float ri = 1.0f / r;
        const float u = ru * ri, v = rv * ri;
        const float p = (float)A.g1 * (E - 0.5f * (ru * u + rv * v));
        uint2 o;
        o.x = pack_bf16(r * (float)A.inv_scale[0], u * (float)A.inv_scale[1]);
        o.y = pack_bf16(v * (float)A.inv_scale[2], p * (float)A.inv_scale[3]);
        if (lane + 32 * c < MLP_RW) ring[slot * MLP_RW + lane + 32 * c] = o;
      }
      mbar_arrive_warp(ring_full(slot));
    }
  } else if (warp >= 20 && warp < 22) {
    // ================= MMA issue for direction g: one lane, in the order the warpgroup fills its A operands
    const int g = warp - 20;
    if (lane == 0) {
      constexpr uint32_t IDESC_H = umma_idesc(128, 64), IDESC_O = umma_idesc(128, 16);
      uint32_t pa[2] = {0, 0}, p1[2] = {0, 0}, pf[2] = {0, 0};
      int rows3[2] = {0, 0};  // output layers issued per slot
      auto layer1 = [&](int s) {  // A1 = [96, 112) -> Y
        const uint32_t base = tmem + 256 * g + 128 * s;
        mbar_wait_pause<PAUSE_M>(a1_full(g, s), p1[s]); p1[s] ^= 1;
        tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < 2; ++ks)
          umma_bf16_ts(base + 32, base + 96 + 8 * ks, umma_desc(sm_u32 + MLP_OFF_W1 + ks * 2048, 1024, 128), IDESC_H, ks);
        umma_commit(d_full(g, s));
        umma_commit(l1_done(g, s));
      };
      auto layer2 = [&](int s) {  // X -> Y
        const uint32_t base = tmem + 256 * g + 128 * s;
        mbar_wait_pause<PAUSE_M>(a_full(g, s), pa[s]); pa[s] ^= 1;
        tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          umma_bf16_ts(base + 32, base + 8 * ks, umma_desc(sm_u32 + MLP_OFF_W2 + ks * 2048, 1024, 128), IDESC_H, ks);
        umma_commit(d_full(g, s));
      };
      auto layer3 = [&](int s) {  // X -> O = [112, 128), once the builders have read the previous row's output
        const uint32_t base = tmem + 256 * g + 128 * s;
        mbar_wait_pause<PAUSE_M>(a_full(g, s), pa[s]); pa[s] ^= 1;
        if (rows3[s] > 0) { mbar_wait_pause<PAUSE_M>(o_free(g, s), pf[s]); pf[s] ^= 1; }
        ++rows3[s];
        tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          umma_bf16_ts(base + 112, base + 8 * ks, umma_desc(sm_u32 + MLP_OFF_W3 + ks * 512, 256, 128), IDESC_O, ks);
        umma_commit(o_full(g, s));
      };
      // per slot: layer 1, 2, 3 of a row, and layer 1 of the slot's next row right behind layer 3 (its operand A1 was
      // built long before and Y is free as soon as the tanh warps have read it for layer 3's operand)
      layer1(0);
      if (n1 > 0) layer1(1);
      for (int i = 0; i < n0; ++i) {
        layer2(0);
        if (i < n1) layer2(1);
        layer3(0);
        if (i + 1 < n0) layer1(0);
        if (i < n1) {
          layer3(1);
          if (i + 1 < n1) layer1(1);
        }
      }
    }
    __syncwarp();
  } else if (warp < 16) {
    // ================= four tanh warpgroups: g = 0 right faces, g = 1 top faces; h = which 32 of the 64 hidden units.
    // lt = my face = my TMEM lane; warps w, w + 8 (and builder warp 16 + w % 4) reach the same lanes 32 (w % 4) .. + 31.
    const int g = (warp >> 2) & 1, h = warp >> 3;
    const uint32_t lane_base = tmem + 256 * g + ((uint32_t)(32 * (warp & 3)) << 16);  // my lane quarter, slot 0
    uint32_t ph[2] = {0, 0};
    float b1[64], b2[64];  // compile-time indexed below: they stay constant-bank operands
#pragma unroll
    for (int q = 0; q < 64; ++q) { b1[q] = A.bias[q]; b2[q] = A.bias[64 + q]; }
    auto hidden = [&](int s, const float (&bias)[64]) {
      mbar_wait_pause<PAUSE_T>(d_full(g, s), ph[s]); ph[s] ^= 1;
      tc_fence_after();
      if (h == 0) hidden_epilogue_ts<0>(lane_base + 128 * s + 32, lane_base + 128 * s, bias);
      else hidden_epilogue_ts<1>(lane_base + 128 * s + 32, lane_base + 128 * s, bias);
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive_warp(a_full(g, s));
    };
    // Slot 0 takes the even rows of the segment, slot 1 the odd ones; the steps alternate between the slots, so that the
    // MMAs a step asks for have the other slot's step to complete in.
    for (int i = 0; i < n0; ++i) {
      hidden(0, b1);
      if (i < n1) hidden(1, b1);
      hidden(0, b2);
      if (i < n1) hidden(1, b2);
    }
  } else {
    // ================= the builder warpgroup (warps 16-19), both directions, off the critical path: the layer-1 operand
    // of a slot's NEXT row goes to the columns A1 = [96, 112) as soon as layer 1 of the current row has read them, and the
    // output layer writes to its own columns O = [112, 128), which are read here
    const int lt = 32 * (warp & 3) + lane, col = c0 + lt;
    const uint32_t lane_q = (uint32_t)(32 * (warp & 3)) << 16;
    uint32_t pl[2][2] = {{0, 0}, {0, 0}}, po[2][2] = {{0, 0}, {0, 0}};
    // layer-1 A operand of face lt of cell row r: 24 inputs as 12 bf16 pairs, K padded to 32 with zeros
    auto build_a1 = [&](int g, int s, int r) {
      const int it = r - nfirst;  // ring rows are numbered from nfirst
      uint32_t w[16];
      if (g == 0) {  // cells c-2 .. c+3 of row r
        mbar_wait_pause<PAUSE_B>(ring_full(it % MLP_RING), (uint32_t)((it / MLP_RING) & 1));
        const uint2* rx = ring + (it % MLP_RING) * MLP_RW + lt;
#pragma unroll
        for (int c = 0; c < 6; ++c) { const uint2 e = rx[c]; w[2 * c] = e.x; w[2 * c + 1] = e.y; }
        mbar_arrive_warp(ring_empty(it % MLP_RING));  // the x-faces of row r were the last right-face reader of ring row r
      } else {       // rows r-2 .. r+3 of column c, normal velocity first: (rho, v, u, p)
        // the producers fill the ring rows out of order: the first top-face row waits for all six rows it reads, every
        // later one for the one row that is new to it
        for (int q = (r == rbeg ? it - 2 : it + 3); q <= it + 3; ++q)
          mbar_wait_pause<PAUSE_B>(ring_full(q % MLP_RING), (uint32_t)((q / MLP_RING) & 1));
#pragma unroll
        for (int c = 0; c < 6; ++c) {
          const uint2 f = ring[((it - 2 + c) % MLP_RING) * MLP_RW + lt + 2];
          w[2 * c] = __byte_perm(f.x, f.y, 0x5410); w[2 * c + 1] = __byte_perm(f.x, f.y, 0x7632);
        }
        mbar_arrive_warp(ring_empty((it - 2) % MLP_RING));  // row r-2 is not read again by the top faces
      }
      w[12] = w[13] = w[14] = w[15] = 0u;
      tmem_st16(tmem + 256 * g + 128 * s + 96 + lane_q, w);
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive_warp(a1_full(g, s));
    };
    // y = W3 h2 + b3 of face lt -> its half of the cell's uint4 (x-faces: the first 8 bytes, y-faces: the second)
    auto output = [&](int g, int s, int r) {
      mbar_wait_pause<PAUSE_B>(o_full(g, s), po[g][s]); po[g][s] ^= 1;
      tc_fence_after();
      uint32_t y[4];
      tmem_ld4(tmem + 256 * g + 128 * s + 112 + lane_q, y);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive_warp(o_free(g, s));
      if (col <= A.nx + 2) {
        float f[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) f[q] = __uint_as_float(y[q]) + A.bias[128 + q];
        uint2* o = reinterpret_cast<uint2*>(A.dFG + (size_t)r * A.pitch + col) + g;
        *o = make_uint2(pack_half2(f[0], f[1]), pack_half2(f[2], f[3]));
      }
    };
    // ring rows rbeg-2, rbeg-1 have no right-face reader: release them for that direction
    mbar_arrive_warp(ring_empty(0));
    mbar_arrive_warp(ring_empty(1));
#pragma unroll
    for (int g = 0; g < 2; ++g) {
      build_a1(g, 0, rbeg);
      if (n1 > 0) build_a1(g, 1, rbeg + 1);
    }
    for (int i = 0; i < n0; ++i) {
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        if (s == 1 && i >= n1) break;
        const int r = rbeg + 2 * i + s;
        const bool next = s == 0 ? i + 1 < n0 : i + 1 < n1;
#pragma unroll
        for (int g = 0; g < 2; ++g) {
          if (next) {  // layer 1 of row r has read A1: build row r + 2's
            mbar_wait_pause<PAUSE_B>(l1_done(g, s), pl[g][s]); pl[g][s] ^= 1;
            tc_fence_after();
            build_a1(g, s, r + 2);
          }
        }
#pragma unroll
        for (int g = 0; g < 2; ++g) output(g, s, r);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, MLP_TMEM_COLS);
}

}  // namespace jxs
