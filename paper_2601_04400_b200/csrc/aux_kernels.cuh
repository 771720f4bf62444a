// aux_kernels.cuh — the small kernels around the fused stage kernel:
//   pad / unpad copies between the caller's interior arrays and the padded RK buffers,
//   S1 domain ghost-frame fill + S2 immersed-boundary ghost gather (one launch),
//   S9 stand-alone wavespeed reduction, the per-step device-side dt computation,
//   and the register-resident DFMA loop that measures the FP64 roofline denominator.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace jxs {

// A handle holds nb >= 1 independent grids of the same size (a batch: BASELINE.json configs[4]), stacked along y in
// one padded buffer: member m owns the padded rows [m (ny+6), (m+1) (ny+6)), each with its own ghost frame.
struct GridDims {
  int nx, ny, pitch;
  long long plane;  // nb*(ny+6)*pitch
  int nb;           // members of the batch
};

// interior [nb][4][ny][nx] -> padded [4][nb (ny+6)][pitch] (interior cell (i,j) of member m at row m (ny+6) + j+3,
// column i+3)
__device__ __forceinline__ long long padded_offset(const GridDims& g, long long t) {
  const long long n = (long long)g.nx * g.ny;
  const int mk = (int)(t / n), m = mk >> 2, k = mk & 3;
  const long long r = t - mk * n;
  const int j = (int)(r / g.nx), i = (int)(r - (long long)j * g.nx);
  return k * g.plane + ((long long)m * (g.ny + 6) + j + 3) * g.pitch + i + 3;
}
// one piece of a row of one variable of one member at a time (the index arithmetic once per piece, not per element);
// rows are cut into pieces of PAD_PIECE elements so that one-dimensional problems (4 rows in all) still fill the GPU
constexpr int PAD_PIECE = 4096;
template <typename T>
__global__ void pad_kernel(const T* __restrict__ src, T* __restrict__ dst, GridDims g) {
  const int npiece = (g.nx + PAD_PIECE - 1) / PAD_PIECE;
  const long long nitems = 4LL * g.ny * g.nb * npiece;
  for (long long it = blockIdx.x; it < nitems; it += gridDim.x) {
    const int L = (int)(it / npiece), i0 = (int)(it - (long long)L * npiece) * PAD_PIECE, i1 = min(i0 + PAD_PIECE, g.nx);
    const int mk = L / g.ny, j = L - mk * g.ny, m = mk >> 2, k = mk & 3;
    const T* a = src + (long long)L * g.nx;
    T* b = dst + k * g.plane + ((long long)m * (g.ny + 6) + j + 3) * g.pitch + 3;
    for (int i = i0 + threadIdx.x; i < i1; i += blockDim.x) b[i] = a[i];
  }
}
template <typename T>
__global__ void unpad_kernel(const T* __restrict__ src, T* __restrict__ dst, GridDims g) {
  const int npiece = (g.nx + PAD_PIECE - 1) / PAD_PIECE;
  const long long nitems = 4LL * g.ny * g.nb * npiece;
  for (long long it = blockIdx.x; it < nitems; it += gridDim.x) {
    const int L = (int)(it / npiece), i0 = (int)(it - (long long)L * npiece) * PAD_PIECE, i1 = min(i0 + PAD_PIECE, g.nx);
    const int mk = L / g.ny, j = L - mk * g.ny, m = mk >> 2, k = mk & 3;
    const T* a = src + k * g.plane + ((long long)m * (g.ny + 6) + j + 3) * g.pitch + 3;
    T* b = dst + (long long)L * g.nx;
    for (int i = i0 + threadIdx.x; i < i1; i += blockDim.x) b[i] = a[i];
  }
}
// every element of the padded buffers starts as a benign state so that support cells outside the
// frame never feed denormals/NaNs into the division slow paths
template <typename T>
__global__ void fill_benign_kernel(T* U, GridDims g, T e_rest) {
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < 4 * g.plane; t += (long long)gridDim.x * blockDim.x) {
    const int k = (int)(t / g.plane);
    U[t] = k == 0 ? T(1) : (k == 3 ? e_rest : T(0));
  }
}

// network outputs in padded indexing -> the caller's face arrays, scaled by out_scale (Eq. 11):
// dFx[4][ny][nx+1] (face f of row j lies between cells f-1 and f), dGy[4][ny+1][nx]; components are
// corrections to the (rho, rho u, rho v, E) fluxes (the y-faces' normal momentum is rho v)
__global__ void gather_faces_kernel(const uint4* __restrict__ dFG, float* __restrict__ dFx,
                                    float* __restrict__ dGy, GridDims g, double s0, double s1, double s2, double s3) {
  const double sc[4] = {s0, s1, s2, s3};
  const long long nfx = (long long)g.ny * (g.nx + 1), nfy = (long long)(g.ny + 1) * g.nx;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < 4 * (nfx + nfy);
       t += (long long)gridDim.x * blockDim.x) {
    if (t < 4 * nfx) {
      const int k = (int)(t / nfx);
      const long long r = t - k * nfx;
      const int j = (int)(r / (g.nx + 1)), f = (int)(r - (long long)j * (g.nx + 1));
      const __half* h = reinterpret_cast<const __half*>(dFG + (long long)(j + 3) * g.pitch + f + 2);
      dFx[t] = (float)(sc[k] * (double)__half2float(h[k]));
    } else {
      const long long u = t - 4 * nfx;
      const int k = (int)(u / nfy);  // conserved component; network output index swaps the momenta
      const int ko = k == 1 ? 2 : (k == 2 ? 1 : k);
      const long long r = u - k * nfy;
      const int f = (int)(r / g.nx), i = (int)(r - (long long)f * g.nx);
      const __half* h = reinterpret_cast<const __half*>(dFG + (long long)(f + 2) * g.pitch + i + 3);
      dGy[u] = (float)(sc[ko] * (double)__half2float(h[4 + ko]));
    }
  }
}

struct BcSpec {
  int xlo, xhi, ylo, yhi;
  double inflow_cons[4];
};

// index map of one axis: ghost index -> (interior source index, sign of the wall-normal momentum);
// src = -1 marks an inflow side.  (R11)
__device__ __forceinline__ void bc_map(int i, int n, int lo, int hi, int& src, int& sgn) {
  src = i; sgn = 1;
  if (i >= 0 && i < n) return;
  const bool low = i < 0;
  const int kind = low ? lo : hi;
  const int g = low ? -i : i - (n - 1);
  if (kind == 0) src = low ? n - g : g - 1;          // periodic
  else if (kind == 1) src = low ? 0 : n - 1;         // transmissive
  else if (kind == 2) { src = low ? g - 1 : n - g; sgn = -1; }  // reflective
  else src = -1;                                     // inflow
}

struct IbmList {
  const int* cell;      // padded offset row*pitch+col of the ghost cell
  const int* donor;     // [4*n] padded offsets of the donors
  const double* w;      // [4*n] weights
  const double* nrm;    // [2*n] unit normal into the fluid
  int n;
};

// S1 + S2 in one launch.  Threads [0, nframe) fill one frame cell each by composing the two axis
// maps (x sides first, then y sides over the x-extended range == y-map applied on top of x-map);
// threads [nframe, nframe + ibm.n) fill one IBM ghost cell each (R9 I6): gather primitives at the
// fluid donors, interpolate to the image point, reflect the velocity, store conserved.
// IBM donors are interior fluid cells, so the two parts do not depend on each other.
// inflow_tab: per-member inflow states (conserved, [nb][4]) of a batch whose members differ there; nullptr = bc's
template <typename T>
__global__ void ghost_fill_kernel(T* __restrict__ U, GridDims g, BcSpec bc, IbmList ibm, T gamma,
                                  const double* __restrict__ inflow_tab = nullptr) {
  const int nxp = g.nx + 6, nyp = g.ny + 6;
  const int side_cells = 6 * g.ny;            // x-ghost columns of the interior rows
  // + full ghost rows (incl. corners); a one-dimensional problem (ny = 1) has no use for them
  const int nframe = side_cells + (g.ny > 1 ? 6 * nxp : 0);
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nframe * g.nb) {
    const int member = t / nframe;
    t -= member * nframe;
    U += (long long)member * nyp * g.pitch;  // this member's rows
    if (inflow_tab) {
      for (int k = 0; k < 4; ++k) bc.inflow_cons[k] = inflow_tab[4 * member + k];
    }
    int ip, jp;  // padded indices in [0,nxp) x [0,nyp)
    if (t < side_cells) {
      jp = 3 + t / 6;
      const int c = t % 6;
      ip = c < 3 ? c : g.nx + c;
    } else {
      const int r = (t - side_cells) / nxp;
      ip = (t - side_cells) % nxp;
      jp = r < 3 ? r : g.ny + r;
    }
    const int i = ip - 3, j = jp - 3;
    int si, sj, sgx, sgy;
    bc_map(j, g.ny, bc.ylo, bc.yhi, sj, sgy);
    T v[4];
    if (sj < 0) {
      for (int k = 0; k < 4; ++k) v[k] = T(bc.inflow_cons[k]);
    } else {
      bc_map(i, g.nx, bc.xlo, bc.xhi, si, sgx);
      if (si < 0) {
        for (int k = 0; k < 4; ++k) v[k] = T(bc.inflow_cons[k]);
      } else {
        const long long o = (long long)(sj + 3) * g.pitch + si + 3;
        for (int k = 0; k < 4; ++k) v[k] = U[k * g.plane + o];
        if (sgx < 0) v[1] = -v[1];
      }
      if (sgy < 0) v[2] = -v[2];
    }
    const long long o = (long long)jp * g.pitch + ip;
    for (int k = 0; k < 4; ++k) U[k * g.plane + o] = v[k];
    (void)nyp;
    return;
  }
  const int q = t - nframe * g.nb;
  if (q >= ibm.n) return;
  T WI[4] = {T(0), T(0), T(0), T(0)};
  for (int d = 0; d < 4; ++d) {
    const T w = T(ibm.w[4 * q + d]);
    if (w == T(0)) continue;
    const long long o = ibm.donor[4 * q + d];
    const T r = U[o], ru = U[g.plane + o], rv = U[2 * g.plane + o], E = U[3 * g.plane + o];
    const T u = ru / r, v = rv / r;
    const T p = (gamma - T(1)) * (E - T(0.5) * r * (u * u + v * v));
    WI[0] += w * r; WI[1] += w * u; WI[2] += w * v; WI[3] += w * p;
  }
  const T nx_ = T(ibm.nrm[2 * q]), ny_ = T(ibm.nrm[2 * q + 1]);
  const T un = WI[1] * nx_ + WI[2] * ny_;
  const T r = WI[0], u = WI[1] - T(2) * un * nx_, v = WI[2] - T(2) * un * ny_, p = WI[3];
  const long long o = ibm.cell[q];
  U[o] = r;
  U[g.plane + o] = r * u;
  U[2 * g.plane + o] = r * v;
  U[3 * g.plane + o] = p / (gamma - T(1)) + T(0.5) * r * (u * u + v * v);
}

__device__ __forceinline__ void atomic_max_bits(unsigned long long* addr, double v) {
  atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

// S9 stand-alone: max over fluid interior cells of max(|u|+a, |v|+a) from a padded buffer; blockIdx.y = member of the
// batch, whose result goes to the word out_stride bytes further on
template <typename T>
__global__ void wavespeed_kernel(const T* __restrict__ U, GridDims g, const uint8_t* __restrict__ fluid, T gamma,
                                 unsigned long long* out_bits, long long out_stride = 0) {
  const long long n = (long long)g.nx * g.ny;
  const int member = blockIdx.y;
  U += (long long)member * (g.ny + 6) * g.pitch;
  if (fluid) fluid += member * n;
  out_bits = reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(out_bits) + member * out_stride);
  T smax = T(0);
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    if (fluid && !fluid[t]) continue;
    const int j = (int)(t / g.nx), i = (int)(t - (long long)j * g.nx);
    const long long o = (long long)(j + 3) * g.pitch + i + 3;
    const T r = U[o], ru = U[g.plane + o], rv = U[2 * g.plane + o], E = U[3 * g.plane + o];
    const T u = ru / r, v = rv / r;
    const T p = (gamma - T(1)) * (E - T(0.5) * r * (u * u + v * v));
    const T a = sqrt(gamma * p / r);
    const T s = max(fabs(u), fabs(v)) + a;
    smax = (s > smax || s != s) ? s : smax;
  }
  for (int o = 16; o > 0; o >>= 1) {
    const T other = __shfl_xor_sync(0xffffffffu, smax, o);
    smax = (other > smax || other != other) ? other : smax;
  }
  __shared__ T wmax[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) wmax[warp] = smax;
  __syncthreads();
  if (warp == 0) {
    smax = lane < (int)(blockDim.x >> 5) ? wmax[lane] : T(0);
    for (int o = 16; o > 0; o >>= 1) {
      const T other = __shfl_xor_sync(0xffffffffu, smax, o);
      smax = (other > smax || other != other) ? other : smax;
    }
    if (lane == 0) atomic_max_bits(out_bits, (double)smax);
  }
}

// pad_kernel and wavespeed_kernel in one pass over the caller's array (jxs_step with a CFL step: the state is read once
// instead of twice).  The per-cell arithmetic and the reduction are wavespeed_kernel's, so s_max has the same bits.
template <typename T>
__global__ void pad_wavespeed_kernel(const T* __restrict__ src, T* __restrict__ dst, GridDims g, const uint8_t* __restrict__ fluid,
                                     T gamma, unsigned long long* out_bits, long long out_stride) {
  const long long n = (long long)g.nx * g.ny;
  const int member = blockIdx.y;
  src += 4 * n * member;
  dst += (long long)member * (g.ny + 6) * g.pitch;
  if (fluid) fluid += member * n;
  out_bits = reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(out_bits) + member * out_stride);
  T smax = T(0);
  const int npiece = (g.nx + PAD_PIECE - 1) / PAD_PIECE;
  for (long long it = blockIdx.x; it < (long long)g.ny * npiece; it += gridDim.x)   // one piece of a row at a time
  for (int j = (int)(it / npiece), i0 = (int)(it - (long long)j * npiece) * PAD_PIECE, i = i0 + threadIdx.x;
       i < min(i0 + PAD_PIECE, g.nx); i += blockDim.x) {
    const long long t = (long long)j * g.nx + i;
    const long long o = (long long)(j + 3) * g.pitch + i + 3;
    const T r = src[t], ru = src[n + t], rv = src[2 * n + t], E = src[3 * n + t];
    dst[o] = r; dst[g.plane + o] = ru; dst[2 * g.plane + o] = rv; dst[3 * g.plane + o] = E;
    if (fluid && !fluid[t]) continue;
    const T u = ru / r, v = rv / r;
    const T p = (gamma - T(1)) * (E - T(0.5) * r * (u * u + v * v));
    const T a = sqrt(gamma * p / r);
    const T s = max(fabs(u), fabs(v)) + a;
    smax = (s > smax || s != s) ? s : smax;
  }
  for (int o = 16; o > 0; o >>= 1) {
    const T other = __shfl_xor_sync(0xffffffffu, smax, o);
    smax = (other > smax || other != other) ? other : smax;
  }
  __shared__ T wmax[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) wmax[warp] = smax;
  __syncthreads();
  if (warp == 0) {
    smax = lane < (int)(blockDim.x >> 5) ? wmax[lane] : T(0);
    for (int o = 16; o > 0; o >>= 1) {
      const T other = __shfl_xor_sync(0xffffffffu, smax, o);
      smax = (other > smax || other != other) ? other : smax;
    }
    if (lane == 0) atomic_max_bits(out_bits, (double)smax);
  }
}

// device-resident stepping state
struct StepState {
  unsigned long long smax_bits[2];  // wavespeed of U^n (cur) and accumulator for U^{n+1} (next)
  double dt;
  double t;
  int bad;                           // set when a non-finite / non-positive wavespeed was met
  int pad;
};

// once per step, before stage 1: dt = cfl*h/smax (R6) or the fixed dt; advance the clock; reset the
// accumulator the last stage of this step will fill.
__global__ void prepare_step_kernel(StepState* st, int cur, double cfl_h, double fixed_dt, int nb = 1) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;  // one thread per member of the batch
  if (m >= nb) return;
  st += m;
  double dt = fixed_dt;
  if (!(fixed_dt > 0.0)) {
    const double smax = __longlong_as_double((long long)st->smax_bits[cur]);
    if (!(smax > 0.0) || isinf(smax) || isnan(smax)) { st->bad = 1; dt = 0.0; }
    else dt = cfl_h / smax;
  }
  st->dt = dt;
  st->t += dt;
  st->smax_bits[cur ^ 1] = 0ull;
}

// FP64 roofline denominator: 8 independent DFMA chains per thread, register-resident
__global__ void dfma_peak_kernel(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  const double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
  if (s == 123.456) out[0] = s;  // never true; keeps the loop alive
}

// The same loop with three DISTINCT register operands per DFMA (x = p * q + x, p and q varying from one instruction to
// the next): the register file hands the FP64 pipe two 64-bit operands per issue slot, so such a DFMA occupies the pipe for 3
// cycles instead of 2 (measured: 24.8 against 37.2 TFLOP/s).  Real code is a mix of the two forms.
__global__ void dfma3_peak_kernel(double* out, int iters, const double* in) {
  double x[8], p[8], q[8];
#pragma unroll
  // p and q depend on the thread: uniform values would be kept in uniform registers, which are not register-file reads
  for (int k = 0; k < 8; ++k) { x[k] = threadIdx.x + k; p[k] = in[k] + 1e-13 * threadIdx.x; q[k] = in[8 + k] * (1.0 + 1e-13 * threadIdx.x); }
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fma(p[k], q[k], x[k]);
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k];
  if (s == 123.456) out[0] = s;
}
// MUFU.TANH rate (the roofline denominator of the flux-MLP kernel): 8 independent chains of tanh.approx.f32
__global__ void tanh_peak_kernel(double* out, int iters) {
  float x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = 0.1f * k + 1e-3f * threadIdx.x;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) asm volatile("tanh.approx.f32 %0, %0;" : "+f"(x[k]));
  }
  float s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k];
  if (s == 123.456f) out[0] = s;
}

// y-slab sharding: rows [row0, row0 + nrows) x the interior columns x the 4 fields of a padded
// buffer <-> a contiguous array [4][nrows][nx] that the caller sends to / receives from the neighbouring rank.
// row0 is an interior row index (0 = the first interior row).
template <typename T>
__global__ void rows_copy_kernel(T* __restrict__ U, T* __restrict__ rows, GridDims g, int row0, int nrows, int unpack) {
  const long long n = (long long)g.nx * nrows;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < 4 * n; t += (long long)gridDim.x * blockDim.x) {
    const int k = (int)(t / n);
    const long long r = t - k * n;
    const int j = (int)(r / g.nx), i = (int)(r - (long long)j * g.nx);
    T* p = U + k * g.plane + (long long)(row0 + j + 3) * g.pitch + i + 3;
    if (unpack) *p = rows[t];
    else rows[t] = *p;
  }
}
// s_max as a double <-> its bit pattern in the stepping state (for the MAX all-reduce over the ranks)
__global__ void smax_copy_kernel(unsigned long long* bits, double* v, int set) {
  if (set) *bits = (unsigned long long)__double_as_longlong(*v);
  else *v = __longlong_as_double((long long)*bits);
}

}  // namespace jxs
