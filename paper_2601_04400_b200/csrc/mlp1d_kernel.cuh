// mlp1d_kernel.cuh — the per-face MLP neural flux for ONE-dimensional problems: PAPER.md L109 ("For the
// one-dimensional Sod shock-tube simulation, a multilayer perceptron (MLP) network is used to predict the neural
// flux", Fig. 1b), Eq. 11 (F = F^HLLC + F^Neural), with the conventions of the 2D path's S5' (R14): the input of face
// i+1/2 is the six cells i-2 .. i+3, each (rho, u, v, p) / in_scale; 24 -> 64 -> 64 -> 4 with tanh on the two hidden
// layers; Delta F = out_scale o y on the (mass, x-momentum, y-momentum, energy) fluxes.
//
// Evaluated in fp64 on the CUDA cores, one warp per face (lane l owns hidden units l and l + 32; activations travel
// between layers by warp shuffles): the differentiated 1D path (tangent1d / adjoint1d) is an fp64 path end to end, and
// at the sizes the paper trains on (N = 500 .. 1000) the step is bound by launches, not by these 11.8 kflop per face.
// mlp1d_backward_kernel is the reverse of the same evaluation for the training of P:L112-128 (Eq. 14-16).
#pragma once
#include "stage_kernel.cuh"

namespace jxs {

constexpr int MLP1D_NPARAM = 6020;  // W1[64][24], b1[64], W2[64][64], b2[64], W3[4][64], b3[4]
constexpr int MLP1D_W1 = 0, MLP1D_B1 = 1536, MLP1D_W2 = 1600, MLP1D_B2 = 5696, MLP1D_W3 = 5760, MLP1D_B3 = 6016;
// the device copy of the parameters carries W1 and W2 a second time, transposed (W1T[24][64], W2T[64][64]): with lane
// l owning hidden units l and l + 32 the forward pass reads a column of W per step, which is a row of the transpose
constexpr int MLP1D_W1T = 6020, MLP1D_W2T = 6020 + 1536, MLP1D_NDEV = 6020 + 1536 + 4096;

struct Mlp1dArgs {
  const void* U;        // padded state, ghosts filled (row 3 of [4][.][pitch])
  const double* theta;  // MLP1D_NDEV doubles: the 6020 parameters in the order of jxs_set_flux_mlp, then W1T, W2T
  double* dF;           // [4] planes, same indexing as U: the correction of the flux through the RIGHT face of a cell
  long long plane;
  int nx, pitch;
  double g1, inv_in[4], out_scale[4];
  // backward only
  const double* Ubar_out;  // adjoint of the stage's result (zero outside the interior)
  double* Wbar;            // [4] planes: += adjoint of the cells' primitives (rho, u, v, p) through the network input
  double* theta_bar;       // [6020] += weights' gradient
  double bdt, dxi;         // b dt of the stage, 1/dx
};

// the 24 inputs of the face right of padded column c: lane l < 24 holds variable l % 4 of cell c - 2 + l / 4
template <typename T>
__device__ __forceinline__ double mlp1d_input(const Mlp1dArgs& A, int c, int lane, double& r_out, double& u_out,
                                              double& v_out) {
  double x = 0.0;
  r_out = 1.0; u_out = 0.0; v_out = 0.0;
  if (lane < 24) {
    const T* U = (const T*)A.U + 3 * (size_t)A.pitch + (c - 2 + (lane >> 2));
    const double r = (double)U[0], ru = (double)U[A.plane], rv = (double)U[2 * A.plane], E = (double)U[3 * A.plane];
    const double ri = 1.0 / r, u = ru * ri, v = rv * ri;
    const double p = A.g1 * (E - 0.5 * (ru * u + rv * v));
    const int var = lane & 3;
    x = (var == 0 ? r : var == 1 ? u : var == 2 ? v : p) * A.inv_in[var];
    r_out = r; u_out = u; v_out = v;
  }
  return x;
}

// forward evaluation for one face by one warp; returns the hidden activations of this lane's units (l, l + 32)
__device__ __forceinline__ void mlp1d_forward(const double* __restrict__ th, double x, int lane, double& h1a, double& h1b,
                                              double& h2a, double& h2b, double y[4]) {
  double z0 = th[MLP1D_B1 + lane], z1 = th[MLP1D_B1 + lane + 32];
#pragma unroll
  for (int i = 0; i < 24; ++i) {
    const double xi = __shfl_sync(0xffffffffu, x, i);
    z0 = fma(th[MLP1D_W1T + i * 64 + lane], xi, z0);
    z1 = fma(th[MLP1D_W1T + i * 64 + lane + 32], xi, z1);
  }
  h1a = tanh(z0); h1b = tanh(z1);
  z0 = th[MLP1D_B2 + lane]; z1 = th[MLP1D_B2 + lane + 32];
#pragma unroll 8
  for (int i = 0; i < 32; ++i) {
    const double a = __shfl_sync(0xffffffffu, h1a, i), b = __shfl_sync(0xffffffffu, h1b, i);
    z0 = fma(th[MLP1D_W2T + i * 64 + lane], a, fma(th[MLP1D_W2T + (i + 32) * 64 + lane], b, z0));
    z1 = fma(th[MLP1D_W2T + i * 64 + lane + 32], a, fma(th[MLP1D_W2T + (i + 32) * 64 + lane + 32], b, z1));
  }
  h2a = tanh(z0); h2b = tanh(z1);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    double s = fma(th[MLP1D_W3 + k * 64 + lane], h2a, th[MLP1D_W3 + k * 64 + lane + 32] * h2b);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    y[k] = s + th[MLP1D_B3 + k];
  }
}

// dF of every face (right faces of padded columns 2 .. nx+2)
template <typename T>
__global__ void __launch_bounds__(128) mlp1d_kernel(const Mlp1dArgs A) {
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  for (int c = 2 + warp; c <= A.nx + 2; c += nwarps) {
    double r, u, v, h1a, h1b, h2a, h2b, y[4];
    const double x = mlp1d_input<T>(A, c, lane, r, u, v);
    mlp1d_forward(A.theta, x, lane, h1a, h1b, h2a, h2b, y);
    if (lane < 4) A.dF[lane * A.plane + 3 * (size_t)A.pitch + c] = A.out_scale[lane] * y[lane];
  }
}

// The reverse of the same evaluation.  The flux adjoint of the face right of column c is (Lbar_{c+1} - Lbar_c) / dx
// with Lbar = b dt Ubar_out (as in adjoint1d_kernel); ybar = out_scale o Fbar; then layer by layer:
//   W3bar += ybar h2^T, h2bar = W3^T ybar, z2bar = h2bar (1 - h2^2), W2bar += z2bar h1^T, h1bar = W2^T z2bar, ...
// and xbar / in_scale is the adjoint of the six cells' primitives (added to Wbar for adjoint1d_kernel to convert).
// The weights' gradient: every warp adds the contributions of its faces into a slot of its own in shared memory
// (4 x 6020 doubles, dynamic; plain stores, every entry belongs to one lane), the CTA sums its four slots and adds
// the result to the global gradient with one fp64 atomic per parameter; the adjoint of the network's input, which
// neighbouring faces share, goes through fp64 atomics as well (24 per face).  The order of those additions is not
// fixed: results agree to round-off.
constexpr int MLP1D_BWD_SMEM = 4 * MLP1D_NPARAM * (int)sizeof(double);

__global__ void __launch_bounds__(128) mlp1d_backward_kernel(const Mlp1dArgs A) {
  extern __shared__ double slots[];
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const double* th = A.theta;
  double* tb = slots + (threadIdx.x >> 5) * MLP1D_NPARAM;  // this warp's slot
  bool first = true;  // the first face of a warp writes its slot, the later ones add to it (every face touches all of it)
  if (2 + warp > A.nx + 2)
    for (int i = lane; i < MLP1D_NPARAM; i += 32) tb[i] = 0.0;  // a warp without a face
  auto add = [&](double* p, double v) { *p = first ? v : *p + v; };
  for (int c = 2 + warp; c <= A.nx + 2; c += nwarps) {
    double r, u, v, h1a, h1b, h2a, h2b, y[4];
    const double x = mlp1d_input<double>(A, c, lane, r, u, v);
    mlp1d_forward(th, x, lane, h1a, h1b, h2a, h2b, y);
    // flux adjoint of this face (interior cells are padded columns 3 .. nx+2)
    double yb[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const size_t o = k * A.plane + 3 * (size_t)A.pitch + c;
      const double lo = (c >= 3 && c <= A.nx + 2) ? A.Ubar_out[o] : 0.0;
      const double hi = (c + 1 >= 3 && c + 1 <= A.nx + 2) ? A.Ubar_out[o + 1] : 0.0;
      yb[k] = A.out_scale[k] * A.bdt * A.dxi * (hi - lo);
    }
    // output layer
    double h2ab = 0.0, h2bb = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      add(tb + MLP1D_W3 + k * 64 + lane, yb[k] * h2a);
      add(tb + MLP1D_W3 + k * 64 + lane + 32, yb[k] * h2b);
      h2ab = fma(th[MLP1D_W3 + k * 64 + lane], yb[k], h2ab);
      h2bb = fma(th[MLP1D_W3 + k * 64 + lane + 32], yb[k], h2bb);
    }
    if (lane < 4) add(tb + MLP1D_B3 + lane, yb[lane]);
    // second hidden layer: my units j = lane, lane + 32
    const double z2a = h2ab * (1.0 - h2a * h2a), z2b = h2bb * (1.0 - h2b * h2b);
    add(tb + MLP1D_B2 + lane, z2a);
    add(tb + MLP1D_B2 + lane + 32, z2b);
    double h1ab = 0.0, h1bb = 0.0;  // adjoint of h1 units lane, lane + 32: sum over all 64 units j of W2[j][.] z2bar_j
    for (int i = 0; i < 32; ++i) {
      const double a = __shfl_sync(0xffffffffu, h1a, i), b = __shfl_sync(0xffffffffu, h1b, i);
      // (the slot keeps W1 and W2 transposed, [input][unit]: neighbouring lanes, neighbouring words)
      add(tb + MLP1D_W2 + i * 64 + lane, z2a * a);
      add(tb + MLP1D_W2 + (i + 32) * 64 + lane, z2a * b);
      add(tb + MLP1D_W2 + i * 64 + lane + 32, z2b * a);
      add(tb + MLP1D_W2 + (i + 32) * 64 + lane + 32, z2b * b);
      const double za = __shfl_sync(0xffffffffu, z2a, i), zb = __shfl_sync(0xffffffffu, z2b, i);  // units i, i + 32
      h1ab = fma(th[MLP1D_W2 + i * 64 + lane], za, fma(th[MLP1D_W2 + (i + 32) * 64 + lane], zb, h1ab));
      h1bb = fma(th[MLP1D_W2 + i * 64 + lane + 32], za, fma(th[MLP1D_W2 + (i + 32) * 64 + lane + 32], zb, h1bb));
    }
    // first hidden layer
    const double z1a = h1ab * (1.0 - h1a * h1a), z1b = h1bb * (1.0 - h1b * h1b);
    add(tb + MLP1D_B1 + lane, z1a);
    add(tb + MLP1D_B1 + lane + 32, z1b);
    double xb = 0.0;  // adjoint of input lane (< 24)
    for (int i = 0; i < 24; ++i) {
      const double xi = __shfl_sync(0xffffffffu, x, i);
      add(tb + MLP1D_W1 + i * 64 + lane, z1a * xi);
      add(tb + MLP1D_W1 + i * 64 + lane + 32, z1b * xi);
    }
    for (int j = 0; j < 32; ++j) {
      const double za = __shfl_sync(0xffffffffu, z1a, j), zb = __shfl_sync(0xffffffffu, z1b, j);  // units j, j + 32
      if (lane < 24) xb = fma(th[MLP1D_W1 + j * 24 + lane], za, fma(th[MLP1D_W1 + (j + 32) * 24 + lane], zb, xb));
    }
    if (lane < 24) {
      const int var = lane & 3;
      atomicAdd(A.Wbar + var * A.plane + 3 * (size_t)A.pitch + (c - 2 + (lane >> 2)), xb * A.inv_in[var]);
    }
    first = false;
    __syncwarp();
  }
  __syncthreads();
  for (int q = threadIdx.x; q < MLP1D_NPARAM; q += blockDim.x) {
    int p = q;  // slot position -> parameter: the W1 and W2 blocks of a slot are transposed
    if (q < MLP1D_B1) p = MLP1D_W1 + (q & 63) * 24 + (q >> 6);
    else if (q >= MLP1D_W2 && q < MLP1D_B2) p = MLP1D_W2 + ((q - MLP1D_W2) & 63) * 64 + ((q - MLP1D_W2) >> 6);
    atomicAdd(A.theta_bar + p, (slots[q] + slots[MLP1D_NPARAM + q]) + (slots[2 * MLP1D_NPARAM + q] + slots[3 * MLP1D_NPARAM + q]));
  }
}

}  // namespace jxs
