// flux_cnn_kernel.cuh — the paper's two-dimensional neural flux (Eq. 11-13; SURVEY.md section 8(f)
// rank 1; readings R18-R20 of DESIGN.md) on the 5th-generation tensor cores of sm_100a.
//
//   F^Neural = out_scale o tanh(conv3x3(relu(conv3x3(relu(conv3x3(X; 4->32)); 32->16)); 16->4)),  zero padding
//
// where X is, at every face of one direction, the mean of the left and right WENO5 states as conservative
// variables (rho, rho u_n, rho u_t, E) / in_scale (R19).  Two kernels:
//
//   cnn_recon_kernel   U (padded, ghosts filled) -> the two input fields, bf16, 16 bytes per face
//   cnn_fused_kernel   one launch per direction: the three 3x3 convolutions as implicit GEMMs on tcgen05, the hidden
//                      activations kept in shared memory (see the kernel's comment)
//
// The input fields in HBM have a one-face border of zeros all around: element (row r, chunk c, face p) is the uint4 at
//   ((r + 1) * C + c) * nbp + (p + 1),      r in [-1, na], p in [-1, nbp - 2].
// Rows are indexed along the field's first axis, faces along its second.  x-faces: rows = j (tangential), faces
// = f (normal).  y-faces are kept in their natural order, rows = f (normal), faces = i (tangential), and use the
// TRANSPOSED 3x3 kernels instead (packed on the host), which is the same convolution.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux_mlp_kernel.cuh"
#include "stage_kernel.cuh"

namespace jxs {

constexpr int CNN_TILE = 128;           // faces per MMA tile = threads per CTA
constexpr int CNN_ROWP = CNN_TILE + 8;  // faces per shared-memory row buffer (window of 130, padded)

struct CnnField {      // one activation field in HBM
  uint4* data;         // base (row -1, chunk 0, face -1)
  int na, nb, nbp, C;  // rows, faces, padded faces per row (incl. the border), 8-channel chunks
  __host__ __device__ size_t at(int r, int c, int p) const { return ((size_t)(r + 1) * C + c) * nbp + (p + 1); }
};

// ------------------------------------------------------------------ pass 1: the input fields
template <typename S>
struct CnnReconArgs {
  const S* U;  // padded [4][ny+6][pitch], ghosts filled
  long long plane;
  int nx, ny, pitch;
  float g1, g1inv;
  float inv_scale[4];  // 1 / in_scale of (rho, rho u_n, rho u_t, E)
  float c133, eps4, sixth;  // WENO constants of stage_kernel.cuh (13/3, 4e-6, 1/6)
  CnnField Xx, Xy; // Xx: rows j, faces f = 0..nx;  Xy: rows f = 0..ny, faces i
};

// One thread per cell of a 32 x 8 tile; neighbouring tiles overlap by one cell in each direction, so that every
// face between two cells of a tile gets its left state from one thread and its right state from the next (through
// shared memory): 31 x 8 x-faces and 32 x 7 y-faces per CTA.  Cell-centred WENO5 of stage_kernel.cuh (weno5_n),
// evaluated in fp32 whatever the state's type: the field is rounded to bf16 (8 significant bits) right after.
constexpr int CNN_RX = 32, CNN_RY = 8;

template <typename S>
__global__ void __launch_bounds__(CNN_RX * CNN_RY) cnn_recon_kernel(const CnnReconArgs<S> A) {
  using T = float;
  __shared__ T W[4][CNN_RY + 4][CNN_RX + 4];  // primitives of cells [i0-2, i0+33] x [j0-2, j0+9]
  __shared__ T Rx[4][CNN_RY][CNN_RX];         // right-biased state at each cell's left face (rho, u, v, p)
  __shared__ T Ry[4][CNN_RY][CNN_RX];         // right-biased state at each cell's bottom face
  const int tx = threadIdx.x % CNN_RX, ty = threadIdx.x / CNN_RX;
  const int i0 = blockIdx.x * (CNN_RX - 1) - 1, j0 = blockIdx.y * (CNN_RY - 1) - 1;  // tile origin (cells start at -1)
  for (int q = threadIdx.x; q < (CNN_RY + 4) * (CNN_RX + 4); q += CNN_RX * CNN_RY) {
    const int cx = q % (CNN_RX + 4), cy = q / (CNN_RX + 4);
    const int ip = min(max(i0 - 2 + cx + 3, 0), A.nx + 5), jp = min(max(j0 - 2 + cy + 3, 0), A.ny + 5);
    const S* s = A.U + (size_t)jp * A.pitch + ip;
    const T r = (T)s[0], ru = (T)s[A.plane], rv = (T)s[2 * A.plane], E = (T)s[3 * A.plane];
    const T ri = rcp_(r);
    const T u = ru * ri, v = rv * ri;
    W[0][cy][cx] = r; W[1][cy][cx] = u; W[2][cy][cx] = v;
    W[3][cy][cx] = A.g1 * fma_(T(-0.5), fma_(ru, u, rv * v), E);
  }
  __syncthreads();
  const int cx = tx + 2, cy = ty + 2;
  StageArgs<T> K;  // only the three WENO constants are read
  K.c133 = A.c133; K.eps4 = A.eps4; K.sixth = A.sixth;
  T wc[4], Lx[4], Ly[4];  // my primitives; left-biased states at my right and top faces
  {
    T a[4], b[4], d[4], e[4], Rm[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { a[k] = W[k][cy][cx - 2]; b[k] = W[k][cy][cx - 1]; wc[k] = W[k][cy][cx]; d[k] = W[k][cy][cx + 1]; e[k] = W[k][cy][cx + 2]; }
    weno5_n<T, 4>(a, b, wc, d, e, K, Rm, Lx);
    const bool badR = any_not_positive(Rm[0], Rm[3]), badL = any_not_positive(Lx[0], Lx[3]);  // R15
#pragma unroll
    for (int k = 0; k < 4; ++k) { Rx[k][ty][tx] = badR ? wc[k] : Rm[k]; Lx[k] = badL ? wc[k] : Lx[k]; }
#pragma unroll
    for (int k = 0; k < 4; ++k) { a[k] = W[k][cy - 2][cx]; b[k] = W[k][cy - 1][cx]; d[k] = W[k][cy + 1][cx]; e[k] = W[k][cy + 2][cx]; }
    weno5_n<T, 4>(a, b, wc, d, e, K, Rm, Ly);
    const bool badRy = any_not_positive(Rm[0], Rm[3]), badLy = any_not_positive(Ly[0], Ly[3]);
#pragma unroll
    for (int k = 0; k < 4; ++k) { Ry[k][ty][tx] = badRy ? wc[k] : Rm[k]; Ly[k] = badLy ? wc[k] : Ly[k]; }
  }
  __syncthreads();
  // mean of the two states at a face as conservative variables (rho, rho u_n, rho u_t, E) / in_scale -> 4 bf16 + 4 zeros
  auto face_input = [&](T rl, T unl, T utl, T pl, T rr, T unr, T utr, T pr) -> uint4 {
    const T eL = fma_(T(0.5) * rl, fma_(unl, unl, utl * utl), pl * A.g1inv);
    const T eR = fma_(T(0.5) * rr, fma_(unr, unr, utr * utr), pr * A.g1inv);
    const float m0 = (float)(T(0.5) * (rl + rr) * A.inv_scale[0]);
    const float m1 = (float)(T(0.5) * fma_(rl, unl, rr * unr) * A.inv_scale[1]);
    const float m2 = (float)(T(0.5) * fma_(rl, utl, rr * utr) * A.inv_scale[2]);
    const float m3 = (float)(T(0.5) * (eL + eR) * A.inv_scale[3]);
    return make_uint4(pack_bf16(m0, m1), pack_bf16(m2, m3), 0u, 0u);
  };
  const int i = i0 + tx, j = j0 + ty;  // my cell
  // x-face f = i+1 of row j, between me and my right neighbour in the tile
  if (tx < CNN_RX - 1 && i + 1 <= A.nx && j >= 0 && j < A.ny)
    A.Xx.data[A.Xx.at(j, 0, i + 1)] =
        face_input(Lx[0], Lx[1], Lx[2], Lx[3], Rx[0][ty][tx + 1], Rx[1][ty][tx + 1], Rx[2][ty][tx + 1], Rx[3][ty][tx + 1]);
  // y-face f = j+1 of column i: normal velocity v first
  if (ty < CNN_RY - 1 && j + 1 <= A.ny && i >= 0 && i < A.nx)
    A.Xy.data[A.Xy.at(j + 1, 0, i)] =
        face_input(Ly[0], Ly[2], Ly[1], Ly[3], Ry[0][ty + 1][tx], Ry[2][ty + 1][tx], Ry[1][ty + 1][tx], Ry[3][ty + 1][tx]);
}

// test / inspection: the bf16 input fields -> float arrays in the oracle's layout, Xx[4][ny][nx+1] (row j, face f)
// and Xy[4][nx][ny+1] (column i, face f)
__global__ void cnn_inputs_gather_kernel(CnnField fx, CnnField fy, float* __restrict__ Xx, float* __restrict__ Xy, int nx, int ny) {
  const long long nfx = (long long)ny * (nx + 1), nfy = (long long)nx * (ny + 1);
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < nfx + nfy; t += (long long)gridDim.x * blockDim.x) {
    uint4 v;
    float* dst;
    long long stride;
    if (t < nfx) {
      const int j = (int)(t / (nx + 1)), f = (int)(t % (nx + 1));
      v = fx.data[fx.at(j, 0, f)]; dst = Xx + t; stride = nfx;
    } else {
      const long long u = t - nfx;
      const int i = (int)(u / (ny + 1)), f = (int)(u % (ny + 1));
      v = fy.data[fy.at(f, 0, i)]; dst = Xy + u; stride = nfy;
    }
    dst[0] = __uint_as_float(v.x << 16); dst[stride] = __uint_as_float(v.x & 0xffff0000u);
    dst[2 * stride] = __uint_as_float(v.y << 16); dst[3 * stride] = __uint_as_float(v.y & 0xffff0000u);
  }
}

// ------------------------------------------------------------------ the three 3x3 convolutions
// KC = 16-channel K steps per tap (input channels / 16, at least 1), NOUT = output channels padded to 16.
template <int KC>
__host__ __device__ constexpr int cnn_slot_bytes() { return 2 * KC * CNN_ROWP * 16; }  // one row buffer: 2 chunks per K step

// A 128 x N x 16 MMA with N <= 64 costs ~50 cycles whatever it computes, so a layer with one MMA per tap would be bound
// by its 9 * KC MMAs per row.  Input row r feeds THREE output rows (r+1 with row tap 0, r with tap 1, r-1 with tap 2)
// from the same shifted windows, so one MMA with the three taps' weights side by side (N = 3 * NOUT) does the work of
// three: 3 * KC MMAs per row.  The three accumulators (TMEM column groups g = output row mod 3) are always
// accumulated into; the group whose output row is complete after input row r (row r-1) is read by the epilogue and
// zeroed with tcgen05.st.  Which tap a group needs depends on r mod 3, hence three permutations of the weight tiles
// (packed on the host):
//   blob of a layer = [3 permutations][3 face taps db][KC][3 NOUT x 16] tiles in the K-major no-swizzle canonical layout
//   (element (n, k) at (n/8)*128 + (k/8)*(N*16) + (n%8)*16 + (k%8)*2), then NOUT fp32 biases;
//   in permutation q = r mod 3, rows g * NOUT .. of a tile hold row tap da = (q + 1 - g) mod 3.
// Face tap db of the convolution is an MMA whose A descriptor points 16*db bytes into the row buffer (layout
// [8-channel chunk][face][16 B]): im2col without a copy.
template <int KC, int NOUT>
__host__ __device__ constexpr int cnn3_wbytes() { return 3 * 3 * KC * 3 * NOUT * 16 * 2; }

template <int NCOL>
__device__ __forceinline__ void tmem_zero(uint32_t taddr) {  // NCOL (multiple of 16) columns of my lane <- 0
#pragma unroll
  for (int h = 0; h < NCOL / 16; ++h)
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1,%1,%1,%1,%1,%1,%1,%1,%1};"
                 ::"r"(taddr + 16 * h), "r"(0u) : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// ------------------------------------------------------------------ all three layers in one kernel
// The hidden fields (32 and 16 channels, 64 + 32 B per face) never leave the SM: a CTA marches a strip of faces row by
// row and keeps, in shared memory, the one row of each hidden layer that the next layer's MMAs read.  With the row taps
// stacked along N (above), input row r of a layer completes output row r-1, so one step of the march is
//   X row r -> [layer 1] -> H1 row r-1 -> [layer 2, one step later] -> H2 row r-3 -> [layer 3, one step later] -> out row r-5.
// The MMAs of the three layers of a step (1 + 6 + 3) are issued back to back and committed ONCE: layer 2 reads the H1
// row that the previous step's epilogue wrote, layer 3 the H2 row likewise, so a step costs one MMA round trip instead
// of three.  A layer's 3-wide face taps eat one face on each side: the 128-face tile yields 128 faces of H1, 126 valid
// faces of H2 and CNNF_OUT = 124 valid output faces, so the strips advance by 124 (3 % recomputed).  The "SAME" zero
// padding of every layer: hidden values at faces or rows outside the field are stored as zeros (not as the layer's
// response to padded inputs).  8 extra steps per row segment fill and drain the pipeline.
constexpr int CNNF_OUT = CNN_TILE - 4;
constexpr int CNNF_W1T = 3 * 96 * 16 * 2;  // layer 1: one [96 x 16] tile per permutation (its 3 face taps x 4 channels share one K step)
constexpr int CNNF_W1 = CNNF_W1T + 32 * 4, CNNF_W2 = cnn3_wbytes<2, 16>() + 16 * 4, CNNF_W3 = cnn3_wbytes<1, 16>() + 16 * 4;
constexpr int cnnf_align(int x) { return (x + 127) / 128 * 128; }
constexpr int CNNF_OFF_W2 = cnnf_align(CNNF_W1), CNNF_OFF_W3 = CNNF_OFF_W2 + cnnf_align(CNNF_W2);
constexpr int CNNF_XS = 3;                                             // X row ring slots
constexpr int CNNF_OFF_X = CNNF_OFF_W3 + cnnf_align(CNNF_W3);          // X row ring (K = 16: 2 chunks per row)
constexpr int CNNF_OFF_H1 = CNNF_OFF_X + CNNF_XS * cnn_slot_bytes<1>();  // two H1 rows (4 chunks each)
constexpr int CNNF_OFF_H2 = CNNF_OFF_H1 + 2 * cnn_slot_bytes<2>();     // two H2 rows (2 chunks each)
// mbarriers: x_full[XS], x_empty[XS], acc_full[3] (a layer's MMAs of a step are complete), eps_done[3] (its epilogue has
// read the accumulator, zeroed it and written its row)
constexpr int CNNF_OFF_BAR = CNNF_OFF_H2 + 2 * cnn_slot_bytes<1>();
constexpr int CNNF_SMEM = CNNF_OFF_BAR + (2 * CNNF_XS + 6) * 8;
constexpr int CNNF_TCOLS = 256;  // accumulators: layer 1 [0, 96), layer 2 [96, 144), layer 3 [144, 192)
constexpr int CNNF_THREADS = 3 * CNN_TILE + 64;  // one epilogue warpgroup per layer, the X producer warp, the MMA warp

struct CnnFusedArgs {
  CnnField in;                 // the input field X of this direction
  const uint8_t* blob[3];      // the three layers' blobs (layer 1: [3 permutations][96 x 16 tile], its taps side by side in K)
  int rows_per_seg, nstrips;
  uint4* dst;                  // as CnnLayerArgs (last layer)
  int slot, pitch, row_off, col_off;
};

__device__ __forceinline__ void tmem_ld16u(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                 "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
               : "r"(taddr) : "memory");
}
// 16 accumulator columns of my face -> + bias -> ReLU -> bf16 -> two 16-byte chunks of a row buffer (zeros if !keep)
__device__ __forceinline__ void cnnf_hidden16(uint32_t taddr, const float* bias, unsigned char* rowbuf, int chunk0, int m, bool keep) {
  uint32_t v[16];
  tmem_ld16u(taddr, v);
  tmem_ld_wait();
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    uint32_t w[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int k = 8 * c + 2 * e;
      w[e] = pack_bf16(fmaxf(__uint_as_float(v[k]) + bias[k], 0.f), fmaxf(__uint_as_float(v[k + 1]) + bias[k + 1], 0.f));
    }
    *reinterpret_cast<uint4*>(rowbuf + (chunk0 + c) * (CNN_ROWP * 16) + m * 16) = keep ? make_uint4(w[0], w[1], w[2], w[3]) : make_uint4(0, 0, 0, 0);
  }
}


// Roles of the 14 warps (two CTAs per SM): warps 0-3 / 4-7 / 8-11 are the epilogue warpgroups of layers 1 / 2 / 3 (thread
// m of a warpgroup owns tile row m = TMEM lane m), warp 12 streams the X rows from HBM into a ring, one lane of warp 13
// issues every MMA.  A layer's cycle is: MMAs of step r -> commit -> its warpgroup reads the completed group, zeroes
// it, writes its row (bias, ReLU, bf16, zeros outside the field) into one of two row buffers -> the MMAs of step r + 1 of
// this layer (the group is free) and of the next layer (its input row is there) may be issued.  The three cycles run
// against each other, so the tensor pipe works on one layer while the other two are in their epilogues; MMAs of one
// thread complete in issue order, which is also what keeps a row buffer from being overwritten while it is still read.
__global__ void __launch_bounds__(CNNF_THREADS, 2) cnn_fused_kernel(const CnnFusedArgs A) {
  extern __shared__ __align__(128) unsigned char sm[];
  __shared__ uint32_t tmem_slot;
  constexpr int LBO_A = CNN_ROWP * 16;
  constexpr int SLOTX = cnn_slot_bytes<1>(), SLOTH1 = cnn_slot_bytes<2>(), SLOTH2 = cnn_slot_bytes<1>();
  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
  const int strip = blockIdx.x % A.nstrips, seg = blockIdx.x / A.nstrips;
  const int na = A.in.na, nb = A.in.nb;
  const int abeg = seg * A.rows_per_seg, aend = min(abeg + A.rows_per_seg, na);
  if (abeg >= aend) return;
  const int b0 = strip * CNNF_OUT;  // first output face of the strip
  const uint32_t sm_u32 = (uint32_t)__cvta_generic_to_shared(sm);
  const uint32_t bars = sm_u32 + CNNF_OFF_BAR;
  auto x_full = [&](int s) { return bars + 8 * s; };
  auto x_empty = [&](int s) { return bars + 8 * (CNNF_XS + s); };
  auto acc_full = [&](int l) { return bars + 8 * (2 * CNNF_XS + l); };
  auto eps_done = [&](int l) { return bars + 8 * (2 * CNNF_XS + 3 + l); };
  const float* bias1 = reinterpret_cast<const float*>(sm + CNNF_W1T);
  const float* bias2 = reinterpret_cast<const float*>(sm + CNNF_OFF_W2 + cnn3_wbytes<2, 16>());
  const float* bias3 = reinterpret_cast<const float*>(sm + CNNF_OFF_W3 + cnn3_wbytes<1, 16>());

  for (int i = t; i < CNNF_W1 / 16; i += CNNF_THREADS) reinterpret_cast<uint4*>(sm)[i] = reinterpret_cast<const uint4*>(A.blob[0])[i];
  for (int i = t; i < CNNF_W2 / 16; i += CNNF_THREADS) reinterpret_cast<uint4*>(sm + CNNF_OFF_W2)[i] = reinterpret_cast<const uint4*>(A.blob[1])[i];
  for (int i = t; i < CNNF_W3 / 16; i += CNNF_THREADS) reinterpret_cast<uint4*>(sm + CNNF_OFF_W3)[i] = reinterpret_cast<const uint4*>(A.blob[2])[i];
  for (int i = t; i < (CNNF_OFF_BAR - CNNF_OFF_X) / 16; i += CNNF_THREADS) reinterpret_cast<uint4*>(sm + CNNF_OFF_X)[i] = make_uint4(0, 0, 0, 0);
  if (t == 0) {
    for (int s = 0; s < CNNF_XS; ++s) { mlp_bar_init(x_full(s), 1); mlp_bar_init(x_empty(s), 1); }
    for (int l = 0; l < 3; ++l) { mlp_bar_init(acc_full(l), 1); mlp_bar_init(eps_done(l), 4); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) tmem_alloc((uint32_t)__cvta_generic_to_shared(&tmem_slot), CNNF_TCOLS);
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t tlane = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
  if (warp < 4) tmem_zero<96>(tlane);
  else if (warp < 8) tmem_zero<48>(tlane + 96);
  else if (warp < 12) tmem_zero<48>(tlane + 144);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const int r_first = abeg - 3, r_last = aend + 4;  // X rows of the march; out row r - 5 completes at step r

  if (warp == 12) {
    // ================= X producer: ring entry i = face b0 - 3 + i, i = 0 .. 129 (lane + 32 k); zeros outside the field.
    // The loads of a row are issued two rows before its stores.
    uint4 pre[2][5];
    auto fetch_row = [&](int r, int q) {
      const bool row_in = r >= 0 && r < na;
#pragma unroll
      for (int k = 0; k < 5; ++k) {
        const int i = lane + 32 * k, p = b0 - 3 + i;
        pre[q][k] = (row_in && i < CNN_TILE + 2 && p >= 0 && p < nb) ? A.in.data[A.in.at(r, 0, p)] : make_uint4(0, 0, 0, 0);
      }
    };
    auto put_row = [&](int r, int q) {
      const int k0 = r - r_first, s = k0 % CNNF_XS;
      if (k0 >= CNNF_XS) mbar_wait_spin(x_empty(s), (uint32_t)((k0 / CNNF_XS - 1) & 1));
      // layer 1's im2col along the faces: the K = 16 operand row of ring entry i is (X[i], X[i+1]) in chunk 0 and
      // (X[i+2], 0) in chunk 1, 4 channels = 8 bytes each: the three face taps of the first layer in ONE MMA
      uint4* c0 = reinterpret_cast<uint4*>(sm + CNNF_OFF_X + s * SLOTX);
      uint4* c1 = c0 + CNN_ROWP;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint2 me = make_uint2(pre[q][k].x, pre[q][k].y), up = make_uint2(pre[q][k + 1].x, pre[q][k + 1].y);
        uint2 n1, n2, w0, w1;
        n1.x = __shfl_down_sync(0xffffffffu, me.x, 1); n1.y = __shfl_down_sync(0xffffffffu, me.y, 1);
        n2.x = __shfl_down_sync(0xffffffffu, me.x, 2); n2.y = __shfl_down_sync(0xffffffffu, me.y, 2);
        w0.x = __shfl_sync(0xffffffffu, up.x, 0); w0.y = __shfl_sync(0xffffffffu, up.y, 0);   // entry 32 (k + 1)
        w1.x = __shfl_sync(0xffffffffu, up.x, 1); w1.y = __shfl_sync(0xffffffffu, up.y, 1);   // entry 32 (k + 1) + 1
        if (lane == 31) { n1 = w0; n2 = w1; }
        if (lane == 30) n2 = w0;
        c0[lane + 32 * k] = make_uint4(me.x, me.y, n1.x, n1.y);
        c1[lane + 32 * k] = make_uint4(n2.x, n2.y, 0u, 0u);
      }
      if (r + 2 <= r_last) fetch_row(r + 2, q);
      fence_async_smem();
      mbar_arrive_warp(x_full(s));
    };
    fetch_row(r_first, 0);
    fetch_row(r_first + 1, 1);
    for (int r = r_first; r <= r_last; r += 2) {
      put_row(r, 0);
      if (r + 1 <= r_last) put_row(r + 1, 1);
    }
  } else if (warp == 13) {
    // ================= MMA issue
    if (lane == 0) {
      constexpr uint32_t ID1 = umma_idesc(128, 96), ID2 = umma_idesc(128, 48);
      constexpr int PERM1 = 96 * 32, PERM2 = 3 * 2 * 48 * 32, PERM3 = 3 * 1 * 48 * 32;
      uint32_t pe[3] = {0, 0, 0};
      for (int r = r_first; r <= r_last; ++r) {
        const int k0 = r - r_first, s = k0 % CNNF_XS;
        const bool first = r == r_first;
        // layer 1: X row r; its accumulator group of output row r + 2 was read and zeroed by epilogue 1 of step r - 1
        mbar_wait_spin(x_full(s), (uint32_t)((k0 / CNNF_XS) & 1));
        if (!first) { mbar_wait_spin(eps_done(0), pe[0]); pe[0] ^= 1; }
        tc_fence_after();
        {
          const uint32_t xb = sm_u32 + CNNF_OFF_X + s * SLOTX, w1 = sm_u32 + ((r + 12) % 3) * PERM1;
          umma_bf16(tmem, umma_desc(xb, LBO_A, 128), umma_desc(w1, 96 * 16, 128), ID1, 1u);
          umma_commit(acc_full(0));
          umma_commit(x_empty(s));
        }
        // layer 2: H1 row r - 2 (written by epilogue 1 of step r - 1, waited for above)
        if (!first) { mbar_wait_spin(eps_done(1), pe[1]); pe[1] ^= 1; }
        tc_fence_after();
        {
          const uint32_t hb = sm_u32 + CNNF_OFF_H1 + ((r - 2) & 1) * SLOTH1, w2 = sm_u32 + CNNF_OFF_W2 + ((r - 2 + 12) % 3) * PERM2;
#pragma unroll
          for (int db = 0; db < 3; ++db)
#pragma unroll
            for (int ks = 0; ks < 2; ++ks)
              umma_bf16(tmem + 96, umma_desc(hb + ks * 2 * LBO_A + db * 16, LBO_A, 128),
                        umma_desc(w2 + (db * 2 + ks) * 48 * 32, 48 * 16, 128), ID2, 1u);
          umma_commit(acc_full(1));
        }
        // layer 3: H2 row r - 4 (written by epilogue 2 of step r - 1, waited for above)
        if (!first) { mbar_wait_spin(eps_done(2), pe[2]); pe[2] ^= 1; }
        tc_fence_after();
        {
          const uint32_t hb = sm_u32 + CNNF_OFF_H2 + ((r - 4) & 1) * SLOTH2, w3 = sm_u32 + CNNF_OFF_W3 + ((r - 4 + 12) % 3) * PERM3;
#pragma unroll
          for (int db = 0; db < 3; ++db)
            umma_bf16(tmem + 144, umma_desc(hb + db * 16, LBO_A, 128), umma_desc(w3 + db * 48 * 32, 48 * 16, 128), ID2, 1u);
          umma_commit(acc_full(2));
        }
      }
    }
    __syncwarp();
  } else {
    // ================= the three epilogue warpgroups
    const int layer = warp >> 2, m = t & (CNN_TILE - 1);
    uint32_t pf = 0;
    for (int r = r_first; r <= r_last; ++r) {
      mbar_wait_spin(acc_full(layer), pf); pf ^= 1;
      tc_fence_after();
      if (layer == 0) {         // H1 row r - 1 (group (r - 1) mod 3): tile row m = face b0 - 2 + m
        const int row = r - 1, p = b0 - 2 + m;
        const bool keep = row >= 0 && row < na && p >= 0 && p < nb;
        const uint32_t tg = tlane + ((row + 12) % 3) * 32;
        unsigned char* buf = sm + CNNF_OFF_H1 + (row & 1) * SLOTH1;
        cnnf_hidden16(tg, bias1, buf, 0, m, keep);
        cnnf_hidden16(tg + 16, bias1 + 16, buf, 2, m, keep);
        tmem_zero<32>(tg);
      } else if (layer == 1) {  // H2 row r - 3: tile row m = face b0 - 1 + m
        const int row = r - 3, p = b0 - 1 + m;
        const bool keep = row >= 0 && row < na && p >= 0 && p < nb;
        const uint32_t tg = tlane + 96 + ((row + 12) % 3) * 16;
        cnnf_hidden16(tg, bias2, sm + CNNF_OFF_H2 + (row & 1) * SLOTH2, 0, m, keep);
        tmem_zero<16>(tg);
      } else {                  // out row r - 5: tile row m = face b0 + m, of which the first CNNF_OUT are valid
        const int row = r - 5, p = b0 + m;
        const uint32_t tg = tlane + 144 + ((row + 12) % 3) * 16;
        uint32_t y[4];
        tmem_ld4(tg, y);
        tmem_ld_wait();
        tmem_zero<16>(tg);
        if (row >= abeg && row < aend && m < CNNF_OUT && p < nb) {
          uint2* o = reinterpret_cast<uint2*>(A.dst + (size_t)(row + A.row_off) * A.pitch + p + A.col_off) + A.slot;
          float t4[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) t4[k] = tanh_f32(__uint_as_float(y[k]) + bias3[k]);
          *o = make_uint2(pack_half2(t4[0], t4[1]), pack_half2(t4[2], t4[3]));
        }
      }
      fence_async_smem();
      tc_fence_before();
      mbar_arrive_warp(eps_done(layer));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, CNNF_TCOLS);
}

}  // namespace jxs
