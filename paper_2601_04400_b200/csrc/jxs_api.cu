// jxs_api.cu — the C ABI of include/jxs.h: handle, argument checks, host-side set-up (work
// decomposition, immersed-boundary classification and gather list), kernel launches.
// Every step of the hot path runs in the kernels of stage_kernel.cuh / aux_kernels.cuh.
#include "../../include/jxs.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <new>
#include <string>
#include <vector>

#include "aux_kernels.cuh"
#include "flux_mlp_kernel.cuh"
#include "flux_cnn_kernel.cuh"
#include "stage_kernel.cuh"
#include "stage1d_kernel.cuh"
#include "tangent1d_kernel.cuh"
#include "adjoint1d_kernel.cuh"
#include "mlp1d_kernel.cuh"
#include "deriv2d_kernels.cuh"

using namespace jxs;

namespace {
constexpr int MAX_EVENTS = 8192;
// resident one-warp CTAs per SM the stage kernel is compiled for (registers <= 65536 / (32 * minb)).  Measured on
// B200 (4096 x 2048, ms per stage launch) with the y-reconstruction's differences carried in registers: fp64 12 warps
// at 168 registers 0.3829, 16 warps at 128 registers (spilling) 0.4975; without the carried state 16 warps at 122
// registers 0.3975, 12 at 156 0.4026, 10 at 157 0.4121, 8 at 157 0.4091 (the FP64 pipe is fed by each warp's own
// independent instructions, not by the number of warps).  fp32: 20 warps at 96 registers 0.2299, 24 at 80 (spilling) 0.2438.
#ifndef JXS_MINB_F64
#define JXS_MINB_F64 12
#endif
#ifndef JXS_MINB_F32
#define JXS_MINB_F32 20
#endif
template <typename T> constexpr int stage_minb() { return sizeof(T) == 8 ? JXS_MINB_F64 : JXS_MINB_F32; }
}

struct jxs_solver {
  int nx = 0, ny = 0, dtype = 0;
  // batch (jxs_create_batch): nb independent grids of the same size stacked along y in every padded buffer; per member
  // the viscosity, the inflow state, the immersed boundary, the time step and the clock
  int nb = 1;
  std::vector<double> mu_b, t_b, dt_b;
  std::vector<jxs_bc> bc_b;
  double* d_inflow_tab = nullptr;  // [nb][4] conserved inflow states
  void* d_vtab = nullptr;          // [nb][10] viscous coefficients in the handle's dtype
  int mlp_nseg = 1;
  // y-slab sharding: rows outside [act_lo, act_hi) are inactive (overlap rows refreshed from the neighbouring rank before
  // every stage: L = 0 there and they do not enter s_max); shard_cur = which s_max slot is current
  int act_lo = 0, act_hi = 0;
  bool act_set = false;
  std::vector<uint8_t> fluid_host;  // the fluid mask as jxs_set_ibm built it (all ones without a body)
  int shard_cur = 0;
  bool shard_open = false;
  double dx = 0, dy = 0, gamma = 0, mu = 0, Pr = 0, nu = 0;
  jxs_bc bc{};
  cudaStream_t stream = nullptr;
  int num_sms = 0;
  int dev = 0;  // the device the handle was created on (and every call must be made on)
  // padded layout
  int pitch = 0;
  long long plane = 0;
  size_t elem = 8;
  void* buf[3] = {nullptr, nullptr, nullptr};
  void* stage_io = nullptr;  // interior-sized staging for the *_host entry points
  // tangent of the state (tangent1d_kernel.cuh): three padded buffers like buf[], allocated at the first
  // jxs_step_fixed_dt_tangent call; d_mse = partial sums and result of jxs_mse_tangent
  void* bufd[3] = {nullptr, nullptr, nullptr};
  double* d_mse = nullptr;
  // per-face MLP flux of one-dimensional problems (mlp1d_kernel.cuh): parameters, flux corrections, and for the
  // reverse sweep the weights' gradient and the adjoint of the primitives through the network input
  bool mlp1d_on = false;
  double* d_theta = nullptr;
  double* d_dF1d = nullptr;
  double* d_theta_bar = nullptr;
  double* d_Wmlp = nullptr;
  cudaGraphExec_t tan_exec = nullptr;  // one tangent step (10 launches), replayed: small grids are launch-bound
  // the whole recorded forward sweep and the whole reverse sweep of the 1D path as graphs (run_sweep): a sweep whose
  // parameters equal those of the call before is captured, and replayed from then on (22 launches per unrolled step)
  struct SweepGraph {
    cudaGraphExec_t exec = nullptr;
    std::vector<long long> key, seen;
    long long launches = 0;
  } rec_graph, adj_graph, rec2_graph, adj2_graph;   // 1D and 2D sweeps
  double tan_dt = 0, tan_gdot = 0;
  long long tan_launches = 0;
  // recorded trajectory and adjoint buffers of the one-dimensional reverse sweep (adjoint1d_kernel.cuh), compact
  // layout [4][pitch] per state: tape = the 3 stage inputs of every recorded step + the final state
  double* tape = nullptr;
  int tape_steps = 0;
  int tape_scheme = JXS_SSPRK3;  // the integrator the recording was made with
  int checkpoint = 0;            // jxs_set_adjoint_checkpointing: keep one state per step, recompute the stages
  int tape_ckpt = 0;             // ... as the recording was made
  double* ckpt = nullptr;        // the two recomputed stage states (compact layout)
  size_t tape_bytes = 0;
  double tape_dt = 0;
  double* adj = nullptr;  // 4 adjoint states, then the gamma_bar partial sums, then gamma_bar
  int adj_parts = 0;
  // two-dimensional derivatives (deriv2d_kernels.cuh): transposed scratch fields [4][nx+6][pitch_t], L and its tangent
  // in the natural layout, the viscous adjoint's face coefficients, the immersed boundary's transposed gather
  // (donor cell -> the ghost entries it feeds), the fluid mask transposed, partial sums of gamma_bar
  int pitch_t = 0;
  long long plane_t = 0;
  double* tr[4] = {nullptr, nullptr, nullptr, nullptr};
  double* Lnat[2] = {nullptr, nullptr};
  double* visc_C = nullptr;
  uint8_t* d_fluid_t = nullptr;
  int n_donor = 0;
  int* d_dcell = nullptr;
  int* d_drows = nullptr;
  int* d_dentry = nullptr;
  double* d_contrib = nullptr;
  double* d_gpart = nullptr;
  size_t gpart_n = 0;
  double* tape2 = nullptr;   // recorded padded states of the 2D reverse sweep (4 * plane doubles each)
  size_t tape2_bytes = 0;
  double* adj2 = nullptr;    // 4 padded adjoint states + gamma_bar + loss accumulator
  // TMA descriptors of the three padded buffers: boxes [4][1][CW] (stencil rows) and [4][1][Epi::W] (RK operand rows)
  CUtensorMap tm_row[3], tm_epi[3];
  // immersed boundary
  uint8_t* d_fluid = nullptr;
  int n_ghost = 0;
  int* d_cell = nullptr;
  int* d_donor = nullptr;
  double* d_w = nullptr;
  double* d_nrm = nullptr;
  // per-face MLP flux correction (S5')
  bool mlp_on = false;
  uint8_t* d_mlp_blob = nullptr;
  uint4* d_dFG = nullptr;  // [rows][pitch]: per padded cell eight fp16 network outputs {right face: 4, top face: 4}
  double in_scale[4] = {1, 1, 1, 1}, out_scale[4] = {1, 1, 1, 1};
  float mlp_bias[132] = {0};
  // the paper's 2D CNN flux (flux_cnn_kernel.cuh): per direction (x, y) the input field, the two hidden fields and
  // the three layers' weight blobs; shares d_dFG / out_scale with the MLP path (one of the two at a time)
  bool cnn_on = false;
  CnnField cnn_X[2] = {};
  uint8_t* d_cnn_blob3[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};  // per direction and layer, for cnn_fused_kernel
  double cnn_in_scale[4] = {1, 1, 1, 1};
  int mlp_strips = 0, mlp_rows_per_seg = 0, mlp_grid = 0;
  double mlp_ms = 0;
  long long mlp_launches = 0;
  std::vector<cudaEvent_t> mlp_events;
  int mlp_events_used = 0;
  // stepping state
  StepState* d_state = nullptr;
  double t = 0, last_dt = 0;
  int scheme = JXS_SSPRK3;
  // CUDA graph of TWO consecutive steps (after two steps the s_max slot and, for forward Euler, the buffer roles are
  // back where they started), replayed by jxs_step* when per-kernel profiling is off: small grids are launch-bound
  cudaStream_t cap_stream = nullptr;
  cudaGraphExec_t pair_exec = nullptr;
  double pair_cfl_h = 0, pair_fixed_dt = 0;
  long long pair_launches = 0;
  int pending_steps = 0;  // steps enqueued by jxs_step_async and not yet waited for
  // work decomposition of the stage kernel
  int nstrips = 0, rows_per_seg = 0, nseg = 0, ntasks = 0, warps = 0, grid = 0;
  int nseg_a = 0, rows_b = 0;  // the first nseg_a segments of a strip have rows_per_seg rows, the rest rows_b (short tail tasks)
  int share = 1;  // handles of about this size that step concurrently (jxs_set_concurrent_handles)
  bool tuned = false;  // rows_per_seg measured on this device (tune_decomposition)
  int rows_fixed = 0;  // jxs_set_rows_per_segment: > 0 overrides the heuristic and the measurement
  double tail_frac = 0.0;  // fraction of the rows cut into half-length segments (chosen by tune_decomposition)
  bool use_graph = true;  // jxs_set_graph_replay
  // bookkeeping
  long long launches = 0;
  bool profiling = false;
  std::vector<cudaEvent_t> events;
  int events_used = 0;
  double stage_ms = 0;
  long long stage_launches = 0;
  mutable std::string err;
};

namespace {

int fail(const jxs_solver* s, int code, const std::string& msg) {
  if (s) s->err = msg;
  return code;
}
int cuda_fail(const jxs_solver* s, cudaError_t e, const char* what) {
  return fail(s, e == cudaErrorMemoryAllocation ? JXS_ENOMEM : JXS_ECUDA,
              std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                             \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return cuda_fail(s, e_, #call);   \
  } while (0)

// cudaFuncSetAttribute is per device: one flag per (kernel instantiation, device)
constexpr int MAX_DEVICES = 64;
template <typename K>
cudaError_t configure_smem(const jxs_solver* s, K kern, bool (&done)[MAX_DEVICES], int smem) {
  const int d = s->dev;
  if (d < 0 || d >= MAX_DEVICES) return cudaErrorInvalidDevice;
  if (done[d]) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  if (e == cudaSuccess) done[d] = true;
  return e;
}
// every entry point that enqueues work checks that the caller is on the handle's device
int check_device(const jxs_solver* s) {
  int d = -1;
  if (cudaGetDevice(&d) != cudaSuccess) return fail(s, JXS_ECUDA, "cudaGetDevice failed");
  if (d != s->dev) return fail(s, JXS_ESTATE, "the current CUDA device is not the one the handle was created on");
  return JXS_OK;
}
#define DEV(s)                              \
  do {                                      \
    const int rc_ = check_device(s);        \
    if (rc_ != JXS_OK) return rc_;          \
  } while (0)

GridDims dims(const jxs_solver* s) { return GridDims{s->nx, s->ny, s->pitch, s->plane, s->nb}; }

BcSpec bcspec(const jxs_solver* s) {
  BcSpec b;
  b.xlo = s->bc.xlo; b.xhi = s->bc.xhi; b.ylo = s->bc.ylo; b.yhi = s->bc.yhi;
  const double r = s->bc.inflow[0], u = s->bc.inflow[1], v = s->bc.inflow[2], p = s->bc.inflow[3];
  b.inflow_cons[0] = r; b.inflow_cons[1] = r * u; b.inflow_cons[2] = r * v;
  b.inflow_cons[3] = p / (s->gamma - 1.0) + 0.5 * r * (u * u + v * v);
  return b;
}

template <typename T> constexpr int sout() { return Cfg<T>::SOUT; }

// cuTensorMapEncodeTiled through the runtime's driver entry point (libcuda is not linked)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}
// descriptor of boxes [4 variables][1 row][box_w columns] of a padded SoA buffer [4][ny+6][pitch]
bool make_tensor_map(const jxs_solver* s, void* base, int box_w, CUtensorMap* out) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const cuuint64_t gdim[3] = {(cuuint64_t)s->pitch, (cuuint64_t)s->nb * (s->ny + 6), 4};
  const cuuint64_t gstride[2] = {(cuuint64_t)s->pitch * s->elem, (cuuint64_t)s->plane * s->elem};
  const cuuint32_t box[3] = {(cuuint32_t)box_w, 1, 4};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(out, s->dtype == JXS_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, gdim,
             gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Strips x row segments = one-warp tasks.  The warp schedulers are greedy (a warp that can issue keeps the
// issue port), so the resident warps of an SM drift apart and a single wave of equal tasks ends ragged
// (measured: mean task lifetime 75 % of the kernel's).  Many short tasks handed out dynamically by the
// block scheduler keep every slot busy; the price is the ~2 row-equivalents of warm-up per task.
// cost model: rows of work per slot, plus half a task of tail per slot
// tail_frac > 0: the last tail_frac of the rows are cut into segments of half the length.  Tasks are handed out in
// blockIdx order (segment-major), so these are the tasks the kernel ends on, and the time during which SMs run out of
// work scales with their length; their extra warm-up rows are paid on that fraction only.
void set_rows_per_seg(jxs_solver* s, int rps, double tail_frac = 0.0) {
  s->rows_per_seg = rps;
  s->rows_b = rps;
  s->nseg_a = (s->ny + rps - 1) / rps;
  int nseg_b = 0;
  if (tail_frac > 0.0 && rps >= 16) {
    const int rb = std::max(8, rps / 2);
    const int na = std::max(0, (int)((1.0 - tail_frac) * s->ny) / rps);
    const int left = s->ny - na * rps;
    if (left > 0) { s->nseg_a = na; s->rows_b = rb; nseg_b = (left + rb - 1) / rb; }
  }
  s->nseg = s->nseg_a + nseg_b;
  s->ntasks = s->nseg * s->nstrips * s->nb;
  s->grid = s->ntasks;
}

void choose_decomposition(jxs_solver* s) {
  const int SOUT = s->dtype == JXS_F64 ? sout<double>() : sout<float>();
  s->nstrips = (s->nx + SOUT - 1) / SOUT;
  const int minb = s->dtype == JXS_F64 ? stage_minb<double>() : stage_minb<float>();
  const double slots = std::max(1.0, (double)s->num_sms * minb / s->share);  // this handle's share of the warp slots
  const int lo = std::min(s->ny, 8);
  std::vector<double> cost(s->ny + 1, 0.0);
  double best = 1e300;
  for (int rps = lo; rps <= s->ny; ++rps) {
    const double tasks = (double)((s->ny + rps - 1) / rps) * s->nstrips * s->nb;
    const double len = rps + 2.0;
    // one wave: the FP64 pipe of an SM is saturated by about 8 warps, fewer tasks run at full speed each
    cost[rps] = tasks <= slots ? 1.15 * len * std::max(1.0, tasks * s->share / (8.0 * s->num_sms))
                               : tasks / slots * len * (1.0 + 0.5 * slots / tasks);
    best = std::min(best, cost[rps]);
  }
  int best_rps = lo;
  for (int rps = lo; rps <= s->ny; ++rps)
    if (cost[rps] <= 1.01 * best) best_rps = rps;  // the longest segments among the near-optimal
  if (s->rows_fixed > 0) best_rps = std::max(1, std::min(s->ny, s->rows_fixed));
  set_rows_per_seg(s, best_rps);
  s->warps = STAGE_WARPS;
  s->tuned = s->rows_fixed > 0;
}

template <typename T, bool VISC, bool ARTV, bool MLP, bool BATCH = false>
cudaError_t launch_stage_t(jxs_solver* s, const StageArgs<T>& a) {
  auto kern = stage_kernel<T, VISC, ARTV, MLP, stage_minb<T>(), BATCH>;
  constexpr int NV = VISC ? 5 : 4;
  const size_t smem = stage_smem_per_warp<T, NV>();
  static bool configured[MAX_DEVICES] = {false};
  if (cudaError_t e = configure_smem(s, kern, configured, (int)smem); e != cudaSuccess) return e;
  int bi = 0;  // which padded buffer is U_in
  while (bi < 3 && s->buf[bi] != (const void*)a.Uin) ++bi;
  if (bi == 3) return cudaErrorInvalidValue;
  kern<<<s->grid, s->warps * 32, smem, s->stream>>>(a, s->tm_row[bi], s->tm_epi[bi], s->tm_epi[0]);
  return cudaGetLastError();
}

template <typename T>
cudaError_t launch_stage(jxs_solver* s, const void* Uin, const void* U0, void* Uout, int mode, double a, double b,
                         unsigned long long* smax_bits) {
  StageArgs<T> A;
  A.Uin = (const T*)Uin; A.U0 = (const T*)U0; A.Uout = (T*)Uout;
  A.fluid = s->d_fluid;
  A.dt = &s->d_state->dt;
  A.smax_bits = smax_bits;
  A.plane = s->plane; A.nx = s->nx; A.ny = s->ny; A.pitch = s->pitch;
  A.nstrips = s->nstrips; A.rows_per_seg = s->rows_per_seg; A.ntasks = s->ntasks;
  A.nseg_a = s->nseg_a; A.rows_b = s->rows_b;
  A.nb = s->nb; A.nseg = s->nseg; A.state_stride = (long long)sizeof(StepState); A.vtab = (const T*)s->d_vtab;
  A.mode = mode;
  A.gamma = (T)s->gamma; A.g1 = (T)(s->gamma - 1.0); A.g1inv = (T)(1.0 / (s->gamma - 1.0));
  A.dxi = (T)(1.0 / s->dx); A.dyi = (T)(1.0 / s->dy);
  A.mu = (T)s->mu;
  A.kappa = (T)(s->mu > 0 ? s->mu * s->gamma / ((s->gamma - 1.0) * s->Pr) : 0.0);
  A.nu = (T)s->nu;
  A.rk_a = (T)a; A.rk_b = (T)b;
  A.c133 = (T)(13.0 / 3.0); A.eps4 = (T)4e-6; A.sixth = (T)(1.0 / 6.0);
  {
    const double mu = s->mu, kap = s->mu > 0 ? s->mu * s->gamma / ((s->gamma - 1.0) * s->Pr) : 0.0;
    const double dxi = 1.0 / s->dx, dyi = 1.0 / s->dy;
    A.vy_n = (T)(4.0 / 3.0 * mu * dyi); A.vy_c = (T)(2.0 / 3.0 * mu * 0.25 * dxi); A.vy_s = (T)(mu * dyi);
    A.vy_t = (T)(mu * 0.25 * dxi); A.vy_q = (T)(kap * dyi);
    A.vx_n = (T)(4.0 / 3.0 * mu * dxi); A.vx_c = (T)(2.0 / 3.0 * mu * 0.25 * dyi); A.vx_s = (T)(mu * dxi);
    A.vx_t = (T)(mu * 0.25 * dyi); A.vx_q = (T)(kap * dxi);
  }
  A.dFG = (s->mlp_on || s->cnn_on) ? s->d_dFG : nullptr;
  for (int k = 0; k < 4; ++k) A.oscale[k] = (T)s->out_scale[k];
  A.dF1d = s->mlp1d_on ? s->d_dF1d : nullptr;
  const bool visc = s->mu > 0, artv = s->nu > 0;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (s->profiling && mode == 0 && s->events_used + 2 <= (int)s->events.size()) {
    e0 = s->events[s->events_used++];
    e1 = s->events[s->events_used++];
    cudaEventRecord(e0, s->stream);
  }
  cudaError_t e;
  if (s->ny == 1) {  // one-dimensional problems: stage1d_kernel.cuh
    stage1d_kernel<T><<<(s->nx + S1D_OUT - 1) / S1D_OUT, S1D_TB, 0, s->stream>>>(A);
    e = cudaGetLastError();
  } else if (s->nb > 1) {  // batch: one launch over all members (no nu-term: jxs_set_artificial_viscosity refuses)
    if (s->mlp_on) e = visc ? launch_stage_t<T, true, false, true, true>(s, A) : launch_stage_t<T, false, false, true, true>(s, A);
    else e = visc ? launch_stage_t<T, true, false, false, true>(s, A) : launch_stage_t<T, false, false, false, true>(s, A);
  } else if (s->mlp_on || s->cnn_on) {
    if (visc) e = artv ? launch_stage_t<T, true, true, true>(s, A) : launch_stage_t<T, true, false, true>(s, A);
    else e = artv ? launch_stage_t<T, false, true, true>(s, A) : launch_stage_t<T, false, false, true>(s, A);
  } else {
    if (visc) e = artv ? launch_stage_t<T, true, true, false>(s, A) : launch_stage_t<T, true, false, false>(s, A);
    else e = artv ? launch_stage_t<T, false, true, false>(s, A) : launch_stage_t<T, false, false, false>(s, A);
  }
  if (e1) cudaEventRecord(e1, s->stream);
  s->launches++;
  return e;
}

cudaError_t stage(jxs_solver* s, const void* Uin, const void* U0, void* Uout, int mode, double a, double b,
                  unsigned long long* smax_bits) {
  return s->dtype == JXS_F64 ? launch_stage<double>(s, Uin, U0, Uout, mode, a, b, smax_bits)
                             : launch_stage<float>(s, Uin, U0, Uout, mode, a, b, smax_bits);
}

cudaError_t ghost_fill(jxs_solver* s, void* U) {
  const int nframe = 6 * s->ny + (s->ny > 1 ? 6 * (s->nx + 6) : 0);
  const int total = nframe * s->nb + s->n_ghost;
  IbmList L{s->d_cell, s->d_donor, s->d_w, s->d_nrm, s->n_ghost};
  const int bs = 128;
  if (s->dtype == JXS_F64)
    ghost_fill_kernel<double><<<(total + bs - 1) / bs, bs, 0, s->stream>>>((double*)U, dims(s), bcspec(s), L, s->gamma,
                                                                          s->d_inflow_tab);
  else
    ghost_fill_kernel<float><<<(total + bs - 1) / bs, bs, 0, s->stream>>>((float*)U, dims(s), bcspec(s), L, (float)s->gamma,
                                                                         s->d_inflow_tab);
  s->launches++;
  return cudaGetLastError();
}

// S5': network outputs of every face of the padded, ghost-filled state U -> d_dFG
template <typename T>
cudaError_t launch_flux_mlp(jxs_solver* s, const void* U) {
  MlpArgs<T> A;
  A.U = (const T*)U; A.dFG = s->d_dFG; A.blob = s->d_mlp_blob;
  A.plane = s->plane; A.nx = s->nx; A.ny = s->ny; A.pitch = s->pitch;
  A.nstrips = s->mlp_strips; A.rows_per_seg = s->mlp_rows_per_seg; A.nseg = s->mlp_nseg;
  A.g1 = (T)(s->gamma - 1.0);
  for (int k = 0; k < 4; ++k) A.inv_scale[k] = (T)(1.0 / s->in_scale[k]);
  std::memcpy(A.bias, s->mlp_bias, sizeof(A.bias));
  auto kern = flux_mlp_kernel<T>;
  static bool configured[MAX_DEVICES] = {false};
  if (cudaError_t e = configure_smem(s, kern, configured, MLP_SMEM); e != cudaSuccess) return e;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (s->profiling && s->mlp_events_used + 2 <= (int)s->mlp_events.size()) {
    e0 = s->mlp_events[s->mlp_events_used++];
    e1 = s->mlp_events[s->mlp_events_used++];
    cudaEventRecord(e0, s->stream);
  }
  kern<<<s->mlp_grid, MLP_THREADS, MLP_SMEM, s->stream>>>(A);
  if (e1) cudaEventRecord(e1, s->stream);
  s->launches++;
  return cudaGetLastError();
}
// the CNN flux of the padded, ghost-filled state U -> d_dFG: reconstruction pass, then one fused three-layer launch
// per direction
template <typename T>
cudaError_t launch_flux_cnn(jxs_solver* s, const void* U) {
  CnnReconArgs<T> R;
  R.U = (const T*)U; R.plane = s->plane; R.nx = s->nx; R.ny = s->ny; R.pitch = s->pitch;
  R.g1 = (float)(s->gamma - 1.0); R.g1inv = (float)(1.0 / (s->gamma - 1.0));
  for (int k = 0; k < 4; ++k) R.inv_scale[k] = (float)(1.0 / s->cnn_in_scale[k]);
  R.Xx = s->cnn_X[0]; R.Xy = s->cnn_X[1];
  R.c133 = (float)(13.0 / 3.0); R.eps4 = 4e-6f; R.sixth = (float)(1.0 / 6.0);
  // tiles overlap by one cell: 31 x-faces and 7 y-faces per tile and direction, cells from -1 to nx / ny
  const dim3 grid((s->nx + 2 + CNN_RX - 2) / (CNN_RX - 1), (s->ny + 2 + CNN_RY - 2) / (CNN_RY - 1));
  cnn_recon_kernel<T><<<grid, CNN_RX * CNN_RY, 0, s->stream>>>(R);
  s->launches++;
  cudaError_t e = cudaGetLastError();
  static bool configured[MAX_DEVICES] = {false};
  if (e == cudaSuccess) e = configure_smem(s, cnn_fused_kernel, configured, CNNF_SMEM);
  for (int d = 0; d < 2 && e == cudaSuccess; ++d) {  // one launch per direction: the three layers fused
    CnnFusedArgs A{};
    A.in = s->cnn_X[d];
    for (int l = 0; l < 3; ++l) A.blob[l] = s->d_cnn_blob3[d][l];
    A.nstrips = (A.in.nb + CNNF_OUT - 1) / CNNF_OUT;
    // two CTAs per SM, 8 extra steps per row segment: the segment count that minimises (waves of CTAs) x (steps per CTA)
    const long long slots = 2LL * s->num_sms;
    long long best = -1;
    int rps = A.in.na;
    for (int nseg = 1; nseg <= std::max(1, A.in.na / 16); ++nseg) {
      const int r = (A.in.na + nseg - 1) / nseg;
      const long long waves = ((long long)A.nstrips * ((A.in.na + r - 1) / r) + slots - 1) / slots;
      const long long cost = waves * (r + 8);
      if (best < 0 || cost < best) { best = cost; rps = r; }
    }
    A.rows_per_seg = rps;
    A.dst = s->d_dFG; A.slot = d; A.pitch = s->pitch;
    A.row_off = d == 0 ? 3 : 2; A.col_off = d == 0 ? 2 : 3;
    const int grid = A.nstrips * ((A.in.na + rps - 1) / rps);
    cnn_fused_kernel<<<grid, CNNF_THREADS, CNNF_SMEM, s->stream>>>(A);
    s->launches++;
    e = cudaGetLastError();
  }
  return e;
}
Mlp1dArgs mlp1d_args(const jxs_solver* s, const void* U) {
  Mlp1dArgs A{};
  A.U = U; A.theta = s->d_theta; A.dF = s->d_dF1d; A.plane = s->plane; A.nx = s->nx; A.pitch = s->pitch;
  A.g1 = s->gamma - 1.0;
  for (int k = 0; k < 4; ++k) { A.inv_in[k] = 1.0 / s->in_scale[k]; A.out_scale[k] = s->out_scale[k]; }
  return A;
}
int mlp1d_grid(const jxs_solver* s) { return std::min((s->nx + 1 + 3) / 4, s->num_sms * 16); }

cudaError_t flux_mlp(jxs_solver* s, const void* U) {  // whichever network is set
  if (s->mlp1d_on) {  // one-dimensional problems: mlp1d_kernel.cuh, one warp per face
    const Mlp1dArgs A = mlp1d_args(s, U);
    if (s->dtype == JXS_F64) mlp1d_kernel<double><<<mlp1d_grid(s), 128, 0, s->stream>>>(A);
    else mlp1d_kernel<float><<<mlp1d_grid(s), 128, 0, s->stream>>>(A);
    s->launches++;
    return cudaGetLastError();
  }
  if (s->cnn_on) {  // jxs_flux_mlp_time then reports the whole network pass (reconstruction + one fused launch per direction)
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (s->profiling && s->mlp_events_used + 2 <= (int)s->mlp_events.size()) {
      e0 = s->mlp_events[s->mlp_events_used++];
      e1 = s->mlp_events[s->mlp_events_used++];
      cudaEventRecord(e0, s->stream);
    }
    const cudaError_t e = s->dtype == JXS_F64 ? launch_flux_cnn<double>(s, U) : launch_flux_cnn<float>(s, U);
    if (e1) cudaEventRecord(e1, s->stream);
    return e;
  }
  if (!s->mlp_on) return cudaSuccess;
  return s->dtype == JXS_F64 ? launch_flux_mlp<double>(s, U) : launch_flux_mlp<float>(s, U);
}

// fp32 -> bf16 bits, round to nearest even (weights are finite)
uint16_t bf16_bits(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
// W[N][Kin] (row-major, [out][in]) -> canonical K-major no-swizzle tile [Npad x Kpad] (zero padded):
// element (n, k) at (n/8)*128 + (k/8)*(Npad*16) + (n%8)*16 + (k%8)*2
void pack_canonical(const float* W, int N, int Kin, int Npad, int Kpad, uint8_t* dst) {
  std::memset(dst, 0, (size_t)Npad * Kpad * 2);
  for (int n = 0; n < N; ++n)
    for (int k = 0; k < Kin; ++k) {
      const size_t off = (size_t)(n / 8) * 128 + (size_t)(k / 8) * (Npad * 16) + (n % 8) * 16 + (k % 8) * 2;
      const uint16_t b = bf16_bits(W[(size_t)n * Kin + k]);
      std::memcpy(dst + off, &b, 2);
    }
}

// W is OIHW [cout][cin][3 tangential taps][3 normal taps]; the kernel's tap (row offset, face offset) is
// (tangential, normal) for x-faces and (normal, tangential) for y-faces (transposed = true).
// one convolution layer's blob for cnn_fused_kernel: [3 permutations q][3 face taps dp][KC][3 NOUT x 16] tiles + NOUT biases; rows
// g * NOUT .. of a tile hold row tap dr = (q + 1 - g) mod 3
std::vector<uint8_t> pack_cnn_layer3(const float* W, const float* b, int cout, int cin, int KC, int NOUT, bool transposed) {
  const int N3 = 3 * NOUT;
  std::vector<uint8_t> blob((size_t)3 * 3 * KC * N3 * 32 + NOUT * 4, 0);
  std::vector<float> tile((size_t)N3 * 16);
  for (int q = 0; q < 3; ++q)
    for (int dp = 0; dp < 3; ++dp)
      for (int ks = 0; ks < KC; ++ks) {
        std::fill(tile.begin(), tile.end(), 0.f);
        for (int g = 0; g < 3; ++g) {
          const int dr = ((q + 1 - g) % 3 + 3) % 3;
          const int ta = transposed ? dp : dr, tb = transposed ? dr : dp;
          for (int n = 0; n < cout; ++n)
            for (int k = 0; k < 16 && 16 * ks + k < cin; ++k)
              tile[(size_t)(g * NOUT + n) * 16 + k] = W[(((size_t)n * cin + 16 * ks + k) * 3 + ta) * 3 + tb];
        }
        pack_canonical(tile.data(), N3, 16, N3, 16, blob.data() + ((size_t)(q * 3 + dp) * KC + ks) * N3 * 32);
      }
  std::memcpy(blob.data() + (size_t)3 * 3 * KC * N3 * 32, b, (size_t)cout * 4);
  return blob;
}

// the first layer's blob for cnn_fused_kernel: its 3 face taps x 4 channels fit one K = 16 step (k = 4 dp + channel), so one
// [3 NOUT x 16] tile per permutation q; rows g * NOUT .. hold row tap dr = (q + 1 - g) mod 3 as above
std::vector<uint8_t> pack_cnn_layer1_im2col(const float* W, const float* b, int cout, int cin, int NOUT, bool transposed) {
  const int N3 = 3 * NOUT;
  std::vector<uint8_t> blob((size_t)3 * N3 * 32 + NOUT * 4, 0);
  std::vector<float> tile((size_t)N3 * 16);
  for (int q = 0; q < 3; ++q) {
    std::fill(tile.begin(), tile.end(), 0.f);
    for (int g = 0; g < 3; ++g) {
      const int dr = ((q + 1 - g) % 3 + 3) % 3;
      for (int dp = 0; dp < 3; ++dp) {
        const int ta = transposed ? dp : dr, tb = transposed ? dr : dp;
        for (int n = 0; n < cout; ++n)
          for (int k = 0; k < cin; ++k)
            tile[(size_t)(g * NOUT + n) * 16 + 4 * dp + k] = W[(((size_t)n * cin + k) * 3 + ta) * 3 + tb];
      }
    }
    pack_canonical(tile.data(), N3, 16, N3, 16, blob.data() + (size_t)q * N3 * 32);
  }
  std::memcpy(blob.data() + (size_t)3 * N3 * 32, b, (size_t)cout * 4);
  return blob;
}

cudaError_t pad(jxs_solver* s, const void* U, void* dst) {
  const int bs = 256, gs = s->num_sms * 8;
  if (s->dtype == JXS_F64) pad_kernel<double><<<gs, bs, 0, s->stream>>>((const double*)U, (double*)dst, dims(s));
  else pad_kernel<float><<<gs, bs, 0, s->stream>>>((const float*)U, (float*)dst, dims(s));
  s->launches++;
  return cudaGetLastError();
}

cudaError_t unpad(jxs_solver* s, const void* src, void* U) {
  const int bs = 256, gs = s->num_sms * 8;
  if (s->dtype == JXS_F64) unpad_kernel<double><<<gs, bs, 0, s->stream>>>((const double*)src, (double*)U, dims(s));
  else unpad_kernel<float><<<gs, bs, 0, s->stream>>>((const float*)src, (float*)U, dims(s));
  s->launches++;
  return cudaGetLastError();
}

cudaError_t wavespeed(jxs_solver* s, const void* Upad, unsigned long long* out_bits) {
  // out_bits: the word of member 0; member m's lies m StepStates further on
  cudaError_t e = cudaMemset2DAsync(out_bits, sizeof(StepState), 0, sizeof(unsigned long long), s->nb, s->stream);
  if (e != cudaSuccess) return e;
  const int bs = 256;
  const dim3 gs(std::max(1, s->num_sms * 8 / s->nb), s->nb);
  if (s->dtype == JXS_F64)
    wavespeed_kernel<double><<<gs, bs, 0, s->stream>>>((const double*)Upad, dims(s), s->d_fluid, s->gamma, out_bits,
                                                       (long long)sizeof(StepState));
  else
    wavespeed_kernel<float><<<gs, bs, 0, s->stream>>>((const float*)Upad, dims(s), s->d_fluid, (float)s->gamma, out_bits,
                                                      (long long)sizeof(StepState));
  s->launches++;
  return cudaGetLastError();
}

// pad + wavespeed in one pass (the entry of jxs_step with a CFL step)
cudaError_t pad_wavespeed(jxs_solver* s, const void* U, void* dst, unsigned long long* out_bits) {
  cudaError_t e = cudaMemset2DAsync(out_bits, sizeof(StepState), 0, sizeof(unsigned long long), s->nb, s->stream);
  if (e != cudaSuccess) return e;
  const int bs = 256;
  const dim3 gs(std::max(1, s->num_sms * 8 / s->nb), s->nb);
  if (s->dtype == JXS_F64)
    pad_wavespeed_kernel<double><<<gs, bs, 0, s->stream>>>((const double*)U, (double*)dst, dims(s), s->d_fluid, s->gamma,
                                                           out_bits, (long long)sizeof(StepState));
  else
    pad_wavespeed_kernel<float><<<gs, bs, 0, s->stream>>>((const float*)U, (float*)dst, dims(s), s->d_fluid, (float)s->gamma,
                                                          out_bits, (long long)sizeof(StepState));
  s->launches++;
  return cudaGetLastError();
}

void free_ibm(jxs_solver* s) {
  cudaFree(s->d_fluid); cudaFree(s->d_cell); cudaFree(s->d_donor); cudaFree(s->d_w); cudaFree(s->d_nrm);
  s->d_fluid = nullptr; s->d_cell = nullptr; s->d_donor = nullptr; s->d_w = nullptr; s->d_nrm = nullptr;
  s->n_ghost = 0;
  cudaFree(s->d_fluid_t); cudaFree(s->d_dcell); cudaFree(s->d_drows); cudaFree(s->d_dentry); cudaFree(s->d_contrib);
  s->d_fluid_t = nullptr; s->d_dcell = nullptr; s->d_drows = nullptr; s->d_dentry = nullptr; s->d_contrib = nullptr;
  s->n_donor = 0;
  s->tape_steps = 0;  // a recording made with another body cannot be reversed
}

// one step, enqueued on s->stream.  cur = index of the valid s_max, at = buffer that holds U^n (forward Euler swaps
// the two buffers every step; SSP-RK3 always starts and ends in buf[0]).
// SSP-RK3 (R5): three stages.  Forward Euler (Eq. 10 as printed): one stage with (a,b) = (0,1).
int one_step(jxs_solver* s, double cfl_h, double fixed_dt, int& cur, int& at) {
  prepare_step_kernel<<<(s->nb + 63) / 64, 64, 0, s->stream>>>(s->d_state, cur, cfl_h, fixed_dt, s->nb);
  s->launches++;
  CU(cudaGetLastError());
  unsigned long long* next = &s->d_state->smax_bits[cur ^ 1];
  if (s->scheme == JXS_EULER) {
    CU(ghost_fill(s, s->buf[at]));
    CU(flux_mlp(s, s->buf[at]));
    CU(stage(s, s->buf[at], nullptr, s->buf[at ^ 1], 0, 0.0, 1.0, next));              // U^{n+1} = U^n + dt L(U^n)
    at ^= 1;
  } else {
    CU(ghost_fill(s, s->buf[0]));
    CU(flux_mlp(s, s->buf[0]));
    CU(stage(s, s->buf[0], nullptr, s->buf[1], 0, 0.0, 1.0, nullptr));                  // U1 = U0 + dt L(U0)
    CU(ghost_fill(s, s->buf[1]));
    CU(flux_mlp(s, s->buf[1]));
    CU(stage(s, s->buf[1], s->buf[0], s->buf[2], 0, 0.75, 0.25, nullptr));              // U2 = 3/4 U0 + 1/4 (U1 + dt L(U1))
    CU(ghost_fill(s, s->buf[2]));
    CU(flux_mlp(s, s->buf[2]));
    CU(stage(s, s->buf[2], s->buf[0], s->buf[0], 0, 1.0 / 3.0, 2.0 / 3.0, next));       // U0 = 1/3 U0 + 2/3 (U2 + dt L(U2))
  }
  cur ^= 1;
  return JXS_OK;
}

void drop_graph(jxs_solver* s) {
  if (s->pair_exec) cudaGraphExecDestroy(s->pair_exec);
  s->pair_exec = nullptr;
  if (s->tan_exec) cudaGraphExecDestroy(s->tan_exec);
  s->tan_exec = nullptr;
  for (jxs_solver::SweepGraph* g : {&s->rec_graph, &s->adj_graph, &s->rec2_graph, &s->adj2_graph}) {
    if (g->exec) cudaGraphExecDestroy(g->exec);
    g->exec = nullptr;
    g->key.clear();
    g->seen.clear();
  }
}

// Run `body` (stream-ordered launches on s->stream only: no allocation, no synchronisation) either as it is, or - when
// the call before had the same `key` - captured into a graph that is replayed from then on.  The key holds every
// value and pointer that the launches bake in.
template <typename Body>
int run_sweep(jxs_solver* s, jxs_solver::SweepGraph& G, const std::vector<long long>& key, Body body) {
  if (s->profiling || !s->use_graph) return body();
  if (G.exec && G.key == key) {
    CU(cudaGraphLaunch(G.exec, s->stream));
    s->launches += G.launches;
    return JXS_OK;
  }
  if (G.seen != key) {  // first sight of these parameters: plain launches (they also set the kernels' attributes)
    G.seen = key;
    return body();
  }
  if (G.exec) cudaGraphExecDestroy(G.exec);
  G.exec = nullptr;
  if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    return body();
  }
  cudaStream_t user = s->stream;
  const long long l0 = s->launches;
  s->stream = s->cap_stream;
  bool ok = cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (ok) {
    ok = body() == JXS_OK;
    cudaGraph_t g = nullptr;
    if (cudaStreamEndCapture(s->cap_stream, &g) != cudaSuccess) ok = false;
    if (ok && cudaGraphInstantiate(&G.exec, g, 0) != cudaSuccess) ok = false;
    if (g) cudaGraphDestroy(g);
  }
  s->stream = user;
  G.launches = s->launches - l0;
  s->launches = l0;
  if (!ok) {
    cudaGetLastError();
    if (G.exec) cudaGraphExecDestroy(G.exec);
    G.exec = nullptr;
    G.seen.clear();
    return body();
  }
  G.key = key;
  CU(cudaGraphLaunch(G.exec, s->stream));
  s->launches += G.launches;
  return JXS_OK;
}

// capture two steps (from the state cur = 0, at = 0) on a private stream; false = use plain launches
bool capture_pair(jxs_solver* s, double cfl_h, double fixed_dt) {
  drop_graph(s);
  if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  cudaStream_t user = s->stream;
  const long long l0 = s->launches;
  s->stream = s->cap_stream;
  bool ok = cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  int cur = 0, at = 0;
  if (ok) {
    ok = one_step(s, cfl_h, fixed_dt, cur, at) == JXS_OK && one_step(s, cfl_h, fixed_dt, cur, at) == JXS_OK;
    cudaGraph_t g = nullptr;
    if (cudaStreamEndCapture(s->cap_stream, &g) != cudaSuccess) ok = false;
    if (ok && cudaGraphInstantiate(&s->pair_exec, g, 0) != cudaSuccess) ok = false;
    if (g) cudaGraphDestroy(g);
  }
  s->stream = user;
  s->pair_launches = s->launches - l0;
  s->launches = l0;
  if (!ok) {
    cudaGetLastError();
    drop_graph(s);
    return false;
  }
  s->pair_cfl_h = cfl_h;
  s->pair_fixed_dt = fixed_dt;
  return true;
}

// advance the padded state in buf[0] by nsteps steps; returns in *where the buffer that holds the result
int run_steps(jxs_solver* s, double cfl, double fixed_dt, int nsteps, int* where, bool smax_ready = false) {
  const double cfl_h = cfl * std::min(s->dx, s->dy);
  int cur = 0, at = 0;
  s->events_used = 0;
  s->mlp_events_used = 0;
  if (!(fixed_dt > 0) && !smax_ready) CU(wavespeed(s, s->buf[0], &s->d_state->smax_bits[0]));
  int n = 0;
  if (!s->profiling && s->use_graph && nsteps >= 6) {
    // the first pair runs as plain launches (it also configures the kernels' attributes outside any capture)
    for (; n < 2; ++n) { const int rc = one_step(s, cfl_h, fixed_dt, cur, at); if (rc != JXS_OK) return rc; }
    if ((s->pair_exec && s->pair_cfl_h == cfl_h && s->pair_fixed_dt == fixed_dt) || capture_pair(s, cfl_h, fixed_dt)) {
      for (; n + 2 <= nsteps; n += 2) {
        CU(cudaGraphLaunch(s->pair_exec, s->stream));
        s->launches += s->pair_launches;
      }
    }
  }
  for (; n < nsteps; ++n) { const int rc = one_step(s, cfl_h, fixed_dt, cur, at); if (rc != JXS_OK) return rc; }
  *where = at;
  return JXS_OK;
}

int finish_steps(jxs_solver* s, int nsteps) {
  std::vector<StepState> sts(s->nb);
  CU(cudaMemcpyAsync(sts.data(), s->d_state, sizeof(StepState) * s->nb, cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  StepState st = sts[0];
  for (int m = 0; m < s->nb; ++m) {
    s->t_b[m] = sts[m].t;
    if (nsteps > 0) s->dt_b[m] = sts[m].dt;
    st.bad |= sts[m].bad;
  }
  s->t = st.t;
  if (nsteps > 0) s->last_dt = st.dt;
  if (s->profiling) {
    s->stage_ms = 0;
    s->stage_launches = s->events_used / 2;
    for (int i = 0; i + 1 < s->events_used; i += 2) {
      float ms = 0;
      cudaEventElapsedTime(&ms, s->events[i], s->events[i + 1]);
      s->stage_ms += ms;
    }
    s->mlp_ms = 0;
    s->mlp_launches = s->mlp_events_used / 2;
    for (int i = 0; i + 1 < s->mlp_events_used; i += 2) {
      float ms = 0;
      cudaEventElapsedTime(&ms, s->mlp_events[i], s->mlp_events[i + 1]);
      s->mlp_ms += ms;
    }
  }
  if (st.bad) {
    int zero = 0;
    for (int m = 0; m < s->nb; ++m)
      cudaMemcpyAsync(&s->d_state[m].bad, &zero, sizeof(int), cudaMemcpyHostToDevice, s->stream);
    return fail(s, JXS_ENUMERIC, "non-finite or non-positive wavespeed met while stepping");
  }
  const double sm = 0;  (void)sm;
  return JXS_OK;
}

// When the tasks make several waves, how a kernel ends depends on how the last wave falls (measured on C4: 0.4057 ms
// at 25 rows per task, 0.4188 at 26, 0.4067 at 28, 0.4177 at 29): no model predicts that, so the first jxs_step* call
// of a handle times one stage launch for every segment length around the heuristic's choice and keeps the best.
// The results do not depend on the segmentation (every row is computed with the same arithmetic).  buf[0] holds
// the padded state; buf[1] is scratch here.
int tune_decomposition(jxs_solver* s) {
  s->tuned = true;
  const int minb = s->dtype == JXS_F64 ? stage_minb<double>() : stage_minb<float>();
  if (s->ny == 1 || (long long)s->ntasks < 2LL * s->num_sms * minb / s->share) return JXS_OK;  // one wave: nothing to tune
  const int base = s->rows_per_seg;
  const bool prof = s->profiling;
  s->profiling = false;
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  CU(ghost_fill(s, s->buf[0]));
  int best = base;
  double best_tail = 0.0;
  float best_ms = 1e30f;
  cudaError_t err = cudaSuccess;
  bool first = true;
  for (int rps = std::max(8, base - 12); rps <= std::min(s->ny, base + 16) && err == cudaSuccess; ++rps)
    for (int variant = 0; variant < 3 && err == cudaSuccess; ++variant) {
      const double tail = variant == 0 ? 0.0 : (variant == 1 ? 0.15 : 0.3);
      set_rows_per_seg(s, rps, tail);
      if (variant > 0 && s->rows_b == rps) continue;  // no short segments at this length
      float ms = 1e30f;
      for (int rep = 0; rep < 2 && err == cudaSuccess; ++rep) {  // the very first launch also warms the caches
        cudaEventRecord(e0, s->stream);
        err = stage(s, s->buf[0], nullptr, s->buf[1], 0, 0.0, 1.0, nullptr);
        cudaEventRecord(e1, s->stream);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float t = 0;
        if (err == cudaSuccess) cudaEventElapsedTime(&t, e0, e1);
        if (rep == 1 || !first) ms = std::min(ms, t);
      }
      first = false;
      if (ms < best_ms) { best_ms = ms; best = rps; best_tail = tail; }
    }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  set_rows_per_seg(s, best, best_tail);
  s->tail_frac = best_tail;
  s->profiling = prof;
  if (err != cudaSuccess) return cuda_fail(s, err, "tune_decomposition");
  return JXS_OK;
}

int step_common(jxs_solver* s, void* U, double cfl, double fixed_dt, int nsteps, bool host, bool wait = true) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U) return fail(s, JXS_EINVAL, "U is NULL");
  if (nsteps < 0) return fail(s, JXS_EINVAL, "nsteps < 0");
  if (!(fixed_dt > 0) && !(cfl > 0)) return fail(s, JXS_EINVAL, "cfl must be > 0");
  const size_t bytes = (size_t)4 * s->nx * s->ny * s->nb * s->elem;
  const void* Ud = U;
  if (host) {
    CU(cudaMemcpyAsync(s->stage_io, U, bytes, cudaMemcpyHostToDevice, s->stream));
    Ud = s->stage_io;
  }
  // with a CFL step the wavespeed of the incoming state is taken in the same pass that pads it
  const bool fused_entry = !(fixed_dt > 0) && nsteps > 0;
  if (fused_entry) CU(pad_wavespeed(s, Ud, s->buf[0], &s->d_state->smax_bits[0]));
  else CU(pad(s, Ud, s->buf[0]));
  if (!s->tuned && nsteps > 0 && wait) {  // never inside jxs_step_async: it must only enqueue (jxs_tune does it explicitly)
    const int rc = tune_decomposition(s);
    if (rc != JXS_OK) return rc;
  }
  int at = 0;
  int rc = run_steps(s, cfl, fixed_dt, nsteps, &at, fused_entry);
  if (rc != JXS_OK) return rc;
  if (host) {
    CU(unpad(s, s->buf[at], s->stage_io));
    CU(cudaMemcpyAsync(U, s->stage_io, bytes, cudaMemcpyDeviceToHost, s->stream));
  } else {
    CU(unpad(s, s->buf[at], U));
  }
  if (!wait) {
    s->pending_steps += nsteps;
    return JXS_OK;
  }
  return finish_steps(s, nsteps);
}

// ---- tangent of the one-dimensional step (tangent1d_kernel.cuh)
constexpr int MSE_PARTS = 1024;

// ghosts of the tangent buffer: the boundary conditions are linear in the state (copies and sign flips), so the
// same kernel fills them; the inflow state is given in primitives, so only its energy moves with gamma
cudaError_t ghost_fill_tangent(jxs_solver* s, void* Udot, double gamma_dot) {
  BcSpec b = bcspec(s);
  const double g1 = s->gamma - 1.0;
  b.inflow_cons[0] = b.inflow_cons[1] = b.inflow_cons[2] = 0.0;
  b.inflow_cons[3] = -s->bc.inflow[3] / (g1 * g1) * gamma_dot;
  const int total = 6 * s->ny;
  IbmList none{nullptr, nullptr, nullptr, nullptr, 0};
  const int bs = 128;
  ghost_fill_kernel<double><<<(total + bs - 1) / bs, bs, 0, s->stream>>>((double*)Udot, dims(s), b, none, s->gamma);
  s->launches++;
  return cudaGetLastError();
}

cudaError_t tangent_stage(jxs_solver* s, int in, int out, double a, double b, double gamma_dot) {
  Tangent1dArgs A;
  A.Uin = (const double*)s->buf[in]; A.Uin_dot = (const double*)s->bufd[in];
  A.U0 = (const double*)s->buf[0]; A.U0_dot = (const double*)s->bufd[0];
  A.Uout = (double*)s->buf[out]; A.Uout_dot = (double*)s->bufd[out];
  A.dt = &s->d_state->dt;
  A.plane = s->plane; A.nx = s->nx; A.pitch = s->pitch;
  A.gamma = s->gamma; A.gamma_dot = gamma_dot; A.dxi = 1.0 / s->dx;
  A.mu = s->mu; A.Pr = s->Pr; A.nu = s->nu; A.rk_a = a; A.rk_b = b;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (s->profiling && s->events_used + 2 <= (int)s->events.size()) {
    e0 = s->events[s->events_used++];
    e1 = s->events[s->events_used++];
    cudaEventRecord(e0, s->stream);
  }
  tangent1d_kernel<<<(s->nx + T1D_OUT - 1) / T1D_OUT, T1D_TB, 0, s->stream>>>(A);
  if (e1) cudaEventRecord(e1, s->stream);
  s->launches++;
  return cudaGetLastError();
}

int tangent_one_step(jxs_solver* s, double gamma_dot, double dt) {
  prepare_step_kernel<<<1, 1, 0, s->stream>>>(s->d_state, 0, 0.0, dt);
  s->launches++;
  CU(cudaGetLastError());
  static const double ab[3][2] = {{0.0, 1.0}, {0.75, 0.25}, {1.0 / 3.0, 2.0 / 3.0}};  // R5
  static const int io[3][2] = {{0, 1}, {1, 2}, {2, 0}};
  for (int st = 0; st < 3; ++st) {
    CU(ghost_fill(s, s->buf[io[st][0]]));
    CU(ghost_fill_tangent(s, s->bufd[io[st][0]], gamma_dot));
    CU(tangent_stage(s, io[st][0], io[st][1], ab[st][0], ab[st][1], gamma_dot));
  }
  return JXS_OK;
}

// capture one tangent step on the private stream (as capture_pair); false = use plain launches
bool capture_tangent_step(jxs_solver* s, double gamma_dot, double dt) {
  if (s->tan_exec) cudaGraphExecDestroy(s->tan_exec);
  s->tan_exec = nullptr;
  if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  cudaStream_t user = s->stream;
  const long long l0 = s->launches;
  s->stream = s->cap_stream;
  bool ok = cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (ok) {
    ok = tangent_one_step(s, gamma_dot, dt) == JXS_OK;
    cudaGraph_t g = nullptr;
    if (cudaStreamEndCapture(s->cap_stream, &g) != cudaSuccess) ok = false;
    if (ok && cudaGraphInstantiate(&s->tan_exec, g, 0) != cudaSuccess) ok = false;
    if (g) cudaGraphDestroy(g);
  }
  s->stream = user;
  s->tan_launches = s->launches - l0;
  s->launches = l0;
  if (!ok) {
    cudaGetLastError();
    if (s->tan_exec) cudaGraphExecDestroy(s->tan_exec);
    s->tan_exec = nullptr;
    return false;
  }
  s->tan_dt = dt;
  s->tan_gdot = gamma_dot;
  return true;
}

int tangent2d_common(jxs_solver* s, void* U, void* Udot, double gamma_dot, double dt, int nsteps);
int record2d_common(jxs_solver* s, void* U, double dt, int nsteps);
int adjoint2d_common(jxs_solver* s, void* Ubar, double* gamma_bar, const double* targets, double* loss);

int tangent_common(jxs_solver* s, void* U, void* Udot, double gamma_dot, double dt, int nsteps) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !Udot) return fail(s, JXS_EINVAL, "U or Udot is NULL");
  if (nsteps < 0) return fail(s, JXS_EINVAL, "nsteps < 0");
  if (!(dt > 0)) return fail(s, JXS_EINVAL, "dt must be > 0");
  if (!std::isfinite(gamma_dot)) return fail(s, JXS_EINVAL, "gamma_dot is not finite");
  if (s->dtype != JXS_F64) return fail(s, JXS_EINVAL, "the tangent is fp64 only");
  if (s->nb > 1) return fail(s, JXS_EINVAL, "no derivatives on a batch handle");
  if (s->mlp_on || s->cnn_on || s->mlp1d_on) return fail(s, JXS_ESTATE, "the tangent does not differentiate the networks");
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  if (s->ny != 1) return tangent2d_common(s, U, Udot, gamma_dot, dt, nsteps);
  const size_t bytes = (size_t)4 * s->plane * s->elem;
  for (int b = 0; b < 3; ++b)
    if (!s->bufd[b]) {
      CU(cudaMalloc(&s->bufd[b], bytes));
      CU(cudaMemsetAsync(s->bufd[b], 0, bytes, s->stream));
    }
  CU(pad(s, U, s->buf[0]));
  CU(pad(s, Udot, s->bufd[0]));
  s->events_used = 0;
  s->mlp_events_used = 0;
  int n = 0;
  if (s->scheme == JXS_EULER) {  // Eq. 10 as printed: one stage with (a, b) = (0, 1); the two buffers swap roles
    int at = 0;
    for (; n < nsteps; ++n, at ^= 1) {
      prepare_step_kernel<<<1, 1, 0, s->stream>>>(s->d_state, 0, 0.0, dt);
      s->launches++;
      CU(cudaGetLastError());
      CU(ghost_fill(s, s->buf[at]));
      CU(ghost_fill_tangent(s, s->bufd[at], gamma_dot));
      CU(tangent_stage(s, at, at ^ 1, 0.0, 1.0, gamma_dot));
    }
    CU(unpad(s, s->buf[at], U));
    CU(unpad(s, s->bufd[at], Udot));
    return finish_steps(s, nsteps);
  }
  if (!s->profiling && s->use_graph && nsteps >= 4) {
    // the first step runs as plain launches; the rest replay one captured step (the buffers' roles return after it)
    int rc = tangent_one_step(s, gamma_dot, dt);
    if (rc != JXS_OK) return rc;
    n = 1;
    if ((s->tan_exec && s->tan_dt == dt && s->tan_gdot == gamma_dot) || capture_tangent_step(s, gamma_dot, dt))
      for (; n < nsteps; ++n) {
        CU(cudaGraphLaunch(s->tan_exec, s->stream));
        s->launches += s->tan_launches;
      }
  }
  for (; n < nsteps; ++n) {
    const int rc = tangent_one_step(s, gamma_dot, dt);
    if (rc != JXS_OK) return rc;
  }
  CU(unpad(s, s->buf[0], U));
  CU(unpad(s, s->bufd[0], Udot));
  return finish_steps(s, nsteps);
}

// ---- reverse mode of the one-dimensional Euler step (adjoint1d_kernel.cuh)
// The tape and the adjoint states hold only the one interior row of the padded layout ([4][pitch] per state).  The
// kernels address row 3 of a [4][7][pitch] buffer, so they are handed a pointer 3 rows before the compact state and a
// plane stride of one row; they never touch another row when ny = 1.
struct CompactLayout {
  jxs_solver* s;
  long long plane;
  explicit CompactLayout(jxs_solver* s_) : s(s_), plane(s_->plane) { s->plane = s->pitch; }
  ~CompactLayout() { s->plane = plane; }
};
double* compact_state(const jxs_solver* s, double* base, long long i) {
  return base + i * 4 * (long long)s->pitch - 3 * (long long)s->pitch;
}

int adjoint_checks(jxs_solver* s) {
  if (s->dtype != JXS_F64) return fail(s, JXS_EINVAL, "the adjoint is fp64 only");
  if (s->nb > 1) return fail(s, JXS_EINVAL, "no derivatives on a batch handle");
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  return JXS_OK;
}

int record_common(jxs_solver* s, void* U, double dt, int nsteps) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U) return fail(s, JXS_EINVAL, "U is NULL");
  if (nsteps < 1) return fail(s, JXS_EINVAL, "nsteps < 1");
  if (!(dt > 0)) return fail(s, JXS_EINVAL, "dt must be > 0");
  int rc = adjoint_checks(s);
  if (rc != JXS_OK) return rc;
  if (s->ny != 1) return record2d_common(s, U, dt, nsteps);
  s->tape_steps = 0;
  const size_t state = (size_t)4 * s->pitch * sizeof(double);
  const bool ckpt = s->checkpoint && s->scheme == JXS_SSPRK3;
  const int per_step = (s->scheme == JXS_EULER || ckpt) ? 1 : 3;  // recorded states per step
  if (ckpt && !s->ckpt) {
    CU(cudaMalloc(&s->ckpt, 2 * state));
    CU(cudaMemsetAsync(s->ckpt, 0, 2 * state, s->stream));
  }
  const size_t bytes = state * (per_step * (size_t)nsteps + 1);
  if (!s->tape || s->tape_bytes < bytes) {  // the tape is kept between calls and only ever grows
    cudaFree(s->tape);
    s->tape = nullptr;
    s->tape_bytes = 0;
    CU(cudaMalloc(&s->tape, bytes));
    s->tape_bytes = bytes;
  }
  // the columns past the padded row are never written; the kernels' clamped support reads must find numbers there
  if (s->pitch > s->nx + 6)
    CU(cudaMemset2DAsync(s->tape + s->nx + 6, (size_t)s->pitch * sizeof(double), 0,
                         (size_t)(s->pitch - s->nx - 6) * sizeof(double), 4 * (per_step * (size_t)nsteps + 1), s->stream));
  CompactLayout compact(s);
  auto T = [&](long long i) { return (void*)compact_state(s, s->tape, i); };
  CU(pad(s, U, T(0)));
  s->events_used = 0;
  s->mlp_events_used = 0;
  auto sweep = [&]() -> int {
  for (long long n = 0; n < nsteps; ++n) {
    prepare_step_kernel<<<1, 1, 0, s->stream>>>(s->d_state, 0, 0.0, dt);
    s->launches++;
    CU(cudaGetLastError());
    if (ckpt) {  // SSP-RK3 with only U^n kept: the two inner stage states live in scratch and are recomputed later
      void* S0 = compact_state(s, s->ckpt, 0);
      void* S1 = compact_state(s, s->ckpt, 1);
      CU(ghost_fill(s, T(n)));
      CU(flux_mlp(s, T(n)));
      CU(stage(s, T(n), nullptr, S0, 0, 0.0, 1.0, nullptr));
      CU(ghost_fill(s, S0));
      CU(flux_mlp(s, S0));
      CU(stage(s, S0, T(n), S1, 0, 0.75, 0.25, nullptr));
      CU(ghost_fill(s, S1));
      CU(flux_mlp(s, S1));
      CU(stage(s, S1, T(n), T(n + 1), 0, 1.0 / 3.0, 2.0 / 3.0, nullptr));
      continue;
    }
    if (per_step == 1) {  // forward Euler (Eq. 10)
      CU(ghost_fill(s, T(n)));
      CU(flux_mlp(s, T(n)));
      CU(stage(s, T(n), nullptr, T(n + 1), 0, 0.0, 1.0, nullptr));
      continue;
    }
    CU(ghost_fill(s, T(3 * n)));
    CU(flux_mlp(s, T(3 * n)));
    CU(stage(s, T(3 * n), nullptr, T(3 * n + 1), 0, 0.0, 1.0, nullptr));
    CU(ghost_fill(s, T(3 * n + 1)));
    CU(flux_mlp(s, T(3 * n + 1)));
    CU(stage(s, T(3 * n + 1), T(3 * n), T(3 * n + 2), 0, 0.75, 0.25, nullptr));
    CU(ghost_fill(s, T(3 * n + 2)));
    CU(flux_mlp(s, T(3 * n + 2)));
    CU(stage(s, T(3 * n + 2), T(3 * n), T(3 * n + 3), 0, 1.0 / 3.0, 2.0 / 3.0, nullptr));
  }
  return JXS_OK;
  };
  {
    long long dt_bits;
    std::memcpy(&dt_bits, &dt, 8);
    const std::vector<long long> key = {nsteps, dt_bits, s->scheme, ckpt, s->mlp1d_on, (long long)(size_t)s->tape,
                                        (long long)(size_t)s->ckpt};
    rc = run_sweep(s, s->rec_graph, key, sweep);
    if (rc != JXS_OK) return rc;
  }
  CU(unpad(s, T((long long)per_step * nsteps), U));
  rc = finish_steps(s, nsteps);
  if (rc != JXS_OK) return rc;
  s->tape_steps = nsteps;
  s->tape_scheme = s->scheme;
  s->tape_ckpt = ckpt;
  s->tape_dt = dt;
  return JXS_OK;
}

cudaError_t adjoint_stage(jxs_solver* s, const double* U, const double* out, double* in, double b, const double* E1,
                          double e1, const double* E2, double e2) {
  Adjoint1dArgs A;
  A.U = U + 3 * (long long)s->pitch; A.Ubar_out = out + 3 * (long long)s->pitch; A.Ubar_in = in + 3 * (long long)s->pitch;
  A.E1 = E1 ? E1 + 3 * (long long)s->pitch : nullptr; A.E2 = E2 ? E2 + 3 * (long long)s->pitch : nullptr;
  double* partial = s->adj + 4LL * 4 * s->pitch;
  A.gbar_partial = partial;
  A.dt = s->tape_dt; A.plane = s->pitch; A.nx = s->nx; A.pitch = s->pitch;
  A.gamma = s->gamma; A.dxi = 1.0 / s->dx; A.b = b; A.e1 = e1; A.e2 = e2;
  A.mu = s->mu; A.Pr = s->Pr; A.nu = s->nu;
  A.Wmlp = nullptr;
  if (s->mlp1d_on) {  // the network's reverse first: weights' gradient, and the adjoint of its input for the kernel below
    Mlp1dArgs M = mlp1d_args(s, U);  // (compact layout: U is the virtual pointer 3 rows before the state)
    M.Ubar_out = out; M.Wbar = s->d_Wmlp; M.theta_bar = s->d_theta_bar; M.bdt = b * s->tape_dt; M.dxi = 1.0 / s->dx;
    cudaError_t e = cudaMemsetAsync(s->d_Wmlp, 0, (size_t)4 * 4 * s->pitch * sizeof(double), s->stream);
    if (e != cudaSuccess) return e;
    static bool configured[MAX_DEVICES] = {false};
    e = configure_smem(s, mlp1d_backward_kernel, configured, MLP1D_BWD_SMEM);
    if (e != cudaSuccess) return e;
    // every CTA flushes its 6020 sums at its end: one face per warp on small grids (the paper's N = 500 .. 1000,
    // where latency counts), at most 2 CTAs per SM on large ones (where the flushes would)
    const int bgrid = std::max(1, std::min((s->nx + 1 + 3) / 4, s->num_sms * 2));
    mlp1d_backward_kernel<<<bgrid, 128, MLP1D_BWD_SMEM, s->stream>>>(M);
    s->launches++;
    A.Wmlp = s->d_Wmlp + 3 * (long long)s->pitch;
  }
  cudaEvent_t e0 = nullptr, e1v = nullptr;
  if (s->profiling && s->events_used + 2 <= (int)s->events.size()) {
    e0 = s->events[s->events_used++];
    e1v = s->events[s->events_used++];
    cudaEventRecord(e0, s->stream);
  }
  if (s->mu > 0 || s->nu > 0) adjoint1d_kernel<true><<<s->adj_parts, A1D_TB, 0, s->stream>>>(A);
  else adjoint1d_kernel<false><<<s->adj_parts, A1D_TB, 0, s->stream>>>(A);
  if (e1v) cudaEventRecord(e1v, s->stream);
  adjoint1d_fold_kernel<<<1, A1D_FOLD_TB, 0, s->stream>>>(A.Ubar_in, s->pitch, s->nx, s->bc.xlo, s->bc.xhi, s->bc.inflow[3],
                                                   s->gamma, partial, s->adj_parts, partial + s->adj_parts);
  s->launches += 2;
  return cudaGetLastError();
}

// targets != nullptr: the loss of Eq. 14 over the recorded steps drives the sweep (Ubar is output only, *loss too)
int adjoint_common(jxs_solver* s, void* Ubar, double* gamma_bar, const double* targets = nullptr, double* loss = nullptr) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!Ubar || !gamma_bar || (targets && !loss)) return fail(s, JXS_EINVAL, "NULL argument");
  int rc = adjoint_checks(s);
  if (rc != JXS_OK) return rc;
  if (s->ny != 1) return adjoint2d_common(s, Ubar, gamma_bar, targets, loss);
  if (!s->tape || s->tape_steps < 1) return fail(s, JXS_ESTATE, "no recorded steps: call jxs_step_fixed_dt_record first");
  const int parts = (s->nx + 6 + A1D_OUT - 1) / A1D_OUT;
  const size_t state = (size_t)4 * s->pitch;
  if (!s->adj || s->adj_parts != parts) {
    cudaFree(s->adj);
    s->adj = nullptr;
    CU(cudaMalloc(&s->adj, (4 * state + parts + 2) * sizeof(double)));
    s->adj_parts = parts;
  }
  CU(cudaMemsetAsync(s->adj, 0, (4 * state + parts + 2) * sizeof(double), s->stream));
  CompactLayout compact(s);
  auto T = [&](long long i) { return compact_state(s, s->tape, i); };
  auto B = [&](int i) { return compact_state(s, s->adj, i); };
  const int per_step = (s->tape_scheme == JXS_EULER || s->tape_ckpt) ? 1 : 3;
  const long long ncell4 = 4LL * s->nx;
  double* loss_acc = s->adj + 4 * state + parts + 1;
  // Eq. 14: the state after recorded step n is tape state per_step * n; its target is targets[n - 1]
  auto inject = [&](long long n, int into, int accumulate) {
    const int gs = (int)std::min<long long>((ncell4 + 255) / 256, s->num_sms * 4);
    mse_inject_kernel<<<gs, 256, 0, s->stream>>>(T(per_step * n) + 3 * (long long)s->pitch, s->pitch,
                                                 targets + (n - 1) * ncell4, s->nx, 2.0 / (s->tape_steps * (double)ncell4),
                                                 B(into) + 3 * (long long)s->pitch, accumulate, loss_acc);
    s->launches++;
    return cudaGetLastError();
  };
  if (targets) CU(inject(s->tape_steps, 0, 0));
  else CU(pad(s, Ubar, B(0)));
  if (s->mlp1d_on) CU(cudaMemsetAsync(s->d_theta_bar, 0, MLP1D_NPARAM * sizeof(double), s->stream));
  s->events_used = 0;
  int x = 0;  // which adjoint state holds the adjoint of U^{n+1}
  auto sweep = [&]() -> int {
  x = 0;
  for (long long n = s->tape_steps - 1; n >= 0; --n) {
    // (Eq. 14) the adjoint of U^{n+1} so far comes from the later steps: add this state's own term of the loss
    if (targets && n + 1 < s->tape_steps) CU(inject(n + 1, x, 1));
    if (s->tape_ckpt) {  // recompute the step's inner stage states from the kept U^n, then reverse the three stages
      double* S0 = compact_state(s, s->ckpt, 0);
      double* S1 = compact_state(s, s->ckpt, 1);
      CU(cudaMemcpyAsync(&s->d_state->dt, &s->tape_dt, sizeof(double), cudaMemcpyHostToDevice, s->stream));
      CU(flux_mlp(s, T(n)));
      CU(stage(s, T(n), nullptr, S0, 0, 0.0, 1.0, nullptr));
      CU(ghost_fill(s, S0));
      CU(flux_mlp(s, S0));
      CU(stage(s, S0, T(n), S1, 0, 0.75, 0.25, nullptr));
      CU(ghost_fill(s, S1));
      const int y2 = (x + 1) & 3, y1 = (x + 2) & 3, y0 = (x + 3) & 3;
      CU(adjoint_stage(s, S1, B(x), B(y2), 2.0 / 3.0, nullptr, 0.0, nullptr, 0.0));
      CU(adjoint_stage(s, S0, B(y2), B(y1), 0.25, nullptr, 0.0, nullptr, 0.0));
      CU(adjoint_stage(s, T(n), B(y1), B(y0), 1.0, B(x), 1.0 / 3.0, B(y2), 0.75));
      x = y0;
      continue;
    }
    if (s->tape_scheme == JXS_EULER) {  // U^{n+1} = U^n + dt L(U^n)
      CU(adjoint_stage(s, T(n), B(x), B(x ^ 1), 1.0, nullptr, 0.0, nullptr, 0.0));
      x ^= 1;
      continue;
    }
    const int y2 = (x + 1) & 3, y1 = (x + 2) & 3, y0 = (x + 3) & 3;
    // U^{n+1} = 1/3 U0 + 2/3 (U2 + dt L(U2));  U2 = 3/4 U0 + 1/4 (U1 + dt L(U1));  U1 = U0 + dt L(U0)   (R5)
    CU(adjoint_stage(s, T(3 * n + 2), B(x), B(y2), 2.0 / 3.0, nullptr, 0.0, nullptr, 0.0));
    CU(adjoint_stage(s, T(3 * n + 1), B(y2), B(y1), 0.25, nullptr, 0.0, nullptr, 0.0));
    CU(adjoint_stage(s, T(3 * n), B(y1), B(y0), 1.0, B(x), 1.0 / 3.0, B(y2), 0.75));
    x = y0;
  }
  return JXS_OK;
  };
  if (s->tape_ckpt) {  // the checkpointed sweep copies dt from a host variable inside the loop: plain launches
    rc = sweep();
  } else {
    long long dt_bits;
    std::memcpy(&dt_bits, &s->tape_dt, 8);
    const std::vector<long long> key = {s->tape_steps, dt_bits, s->tape_scheme, s->mlp1d_on, (long long)(size_t)s->tape,
                                        (long long)(size_t)s->adj, (long long)(size_t)targets, s->adj_parts};
    rc = run_sweep(s, s->adj_graph, key, sweep);
    if (rc == JXS_OK) {  // where the adjoint of U^0 ends up does not depend on how the sweep was run
      x = 0;
      if (s->tape_scheme == JXS_EULER) x = (int)(s->tape_steps & 1);
      else for (long long n = 0; n < s->tape_steps; ++n) x = (x + 3) & 3;
    }
  }
  if (rc != JXS_OK) return rc;
  CU(unpad(s, B(x), Ubar));
  double out[2];
  CU(cudaMemcpyAsync(out, s->adj + 4 * state + parts, sizeof(out), cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  *gamma_bar = out[0];
  if (loss) *loss = out[1] / (s->tape_steps * (double)ncell4);
  if (s->profiling) {
    s->stage_ms = 0;
    s->stage_launches = s->events_used / 2;
    for (int i = 0; i + 1 < s->events_used; i += 2) {
      float ms = 0;
      cudaEventElapsedTime(&ms, s->events[i], s->events[i + 1]);
      s->stage_ms += ms;
    }
  }
  return JXS_OK;
}

// ---- derivatives of the two-dimensional step (deriv2d_kernels.cuh)
int deriv2d_scratch(jxs_solver* s) {
  if (s->tr[0]) return JXS_OK;
  s->pitch_t = (s->ny + 6 + 15) / 16 * 16;
  s->plane_t = (long long)(s->nx + 6) * s->pitch_t;
  const size_t tb = (size_t)4 * s->plane_t * sizeof(double), nb = (size_t)4 * s->plane * sizeof(double);
  for (int q = 0; q < 4; ++q) { CU(cudaMalloc(&s->tr[q], tb)); CU(cudaMemsetAsync(s->tr[q], 0, tb, s->stream)); }
  for (int q = 0; q < 2; ++q) { CU(cudaMalloc(&s->Lnat[q], nb)); CU(cudaMemsetAsync(s->Lnat[q], 0, nb, s->stream)); }
  const size_t nf = (size_t)s->ny * (s->nx + 1) + (size_t)(s->ny + 1) * s->nx;
  CU(cudaMalloc(&s->visc_C, 7 * nf * sizeof(double)));
  // partial sums of gamma_bar: the line kernels' CTAs of both passes, the viscous kernels, the folds, the ghosts
  const size_t lines = (size_t)((s->nx + 6 + A1D_OUT - 1) / A1D_OUT) * s->ny + (size_t)((s->ny + 6 + A1D_OUT - 1) / A1D_OUT) * s->nx;
  s->gpart_n = lines + 2 * (size_t)s->num_sms * 8 + 4 * (size_t)(s->nx + s->ny + 16) + (size_t)s->n_ghost + 64;
  CU(cudaMalloc(&s->d_gpart, s->gpart_n * sizeof(double)));
  return JXS_OK;
}
LineSet lines_x(const jxs_solver* s) { return LineSet{s->plane, s->pitch, s->nx, s->ny}; }
LineSet lines_y(const jxs_solver* s) { return LineSet{s->plane_t, s->pitch_t, s->ny, s->nx}; }

// natural [4][ny+6][pitch] -> transposed [4][nx+6][pitch_t] (momenta exchanged), the whole padded field
cudaError_t to_transposed(jxs_solver* s, const double* src, double* dst) {
  TransposeArgs T{src, dst, s->plane, s->plane_t, s->pitch, s->pitch_t, 0, s->ny + 6, 0, s->nx + 6, 0};
  const dim3 grid((s->nx + 6 + 31) / 32, (s->ny + 6 + 31) / 32, 4);
  transpose_swap_kernel<<<grid, 256, 0, s->stream>>>(T);
  s->launches++;
  return cudaGetLastError();
}
// transposed -> natural, added: the lines 3 .. nx+2 of src (interior columns), positions [p_lo, p_hi) along them
cudaError_t add_from_transposed(jxs_solver* s, const double* src, double* dst, int p_lo, int p_hi) {
  TransposeArgs T{src, dst, s->plane_t, s->plane, s->pitch_t, s->pitch, 3, s->nx + 3, p_lo, p_hi, 1};
  const dim3 grid((p_hi - p_lo + 31) / 32, (s->nx + 31) / 32, 4);
  transpose_swap_kernel<<<grid, 256, 0, s->stream>>>(T);
  s->launches++;
  return cudaGetLastError();
}

// the tangent's ghosts: frame (the boundary conditions are linear; the inflow state's energy moves with gamma), then
// the immersed-boundary fill on pairs.  U must already hold its own ghosts.
cudaError_t ghost_fill_tangent2d(jxs_solver* s, const void* U, void* Udot, double gamma_dot) {
  BcSpec b = bcspec(s);
  const double g1 = s->gamma - 1.0;
  b.inflow_cons[0] = b.inflow_cons[1] = b.inflow_cons[2] = 0.0;
  b.inflow_cons[3] = -s->bc.inflow[3] / (g1 * g1) * gamma_dot;
  const int total = 6 * s->ny + 6 * (s->nx + 6);
  IbmList none{nullptr, nullptr, nullptr, nullptr, 0};
  ghost_fill_kernel<double><<<(total + 127) / 128, 128, 0, s->stream>>>((double*)Udot, dims(s), b, none, s->gamma);
  s->launches++;
  if (s->n_ghost > 0) {
    IbmList L{s->d_cell, s->d_donor, s->d_w, s->d_nrm, s->n_ghost};
    ibm_fill_tangent_kernel<<<(s->n_ghost + 127) / 128, 128, 0, s->stream>>>((const double*)U, (double*)Udot, s->plane, L,
                                                                             s->gamma, gamma_dot);
    s->launches++;
  }
  return cudaGetLastError();
}

// one stage on pairs: (buf[in], bufd[in]) -> (buf[out], bufd[out]) = a U0 + b (U + dt L), L = Lx + Ly + Lv
int tangent_stage2d(jxs_solver* s, int in, int out, double a, double b, double gamma_dot) {
  const double *U = (const double*)s->buf[in], *Ud = (const double*)s->bufd[in];
  CU(ghost_fill(s, s->buf[in]));
  CU(ghost_fill_tangent2d(s, U, s->bufd[in], gamma_dot));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (s->profiling && s->events_used + 2 <= (int)s->events.size()) {
    e0 = s->events[s->events_used++];
    e1 = s->events[s->events_used++];
    cudaEventRecord(e0, s->stream);
  }
  TangentLineArgs X{U, Ud, s->Lnat[0], s->Lnat[1], lines_x(s), s->gamma, gamma_dot, 1.0 / s->dx, s->nu, 0};
  tangent_line_kernel<<<dim3((s->nx + T1D_OUT - 1) / T1D_OUT, s->ny), T1D_TB, 0, s->stream>>>(X);
  s->launches++;
  CU(to_transposed(s, U, s->tr[0]));
  CU(to_transposed(s, Ud, s->tr[1]));
  TangentLineArgs Y{s->tr[0], s->tr[1], s->tr[2], s->tr[3], lines_y(s), s->gamma, gamma_dot, 1.0 / s->dy, s->nu, 0};
  tangent_line_kernel<<<dim3((s->ny + T1D_OUT - 1) / T1D_OUT, s->nx), T1D_TB, 0, s->stream>>>(Y);
  s->launches++;
  CU(add_from_transposed(s, s->tr[2], s->Lnat[0], 3, s->ny + 3));
  CU(add_from_transposed(s, s->tr[3], s->Lnat[1], 3, s->ny + 3));
  if (s->mu > 0) {
    Visc2dArgs V{U, Ud, s->Lnat[0], s->Lnat[1], s->plane, s->nx, s->ny, s->pitch, s->gamma, gamma_dot, s->mu, s->Pr,
                 1.0 / s->dx, 1.0 / s->dy};
    viscous2d_tangent_kernel<<<dim3((s->nx + V2_TX - 1) / V2_TX, (s->ny + V2_TY - 1) / V2_TY), V2_TX * V2_TY, 0, s->stream>>>(V);
    s->launches++;
  }
  Combine2dArgs C{U, Ud, (const double*)s->buf[0], (const double*)s->bufd[0], s->Lnat[0], s->Lnat[1], (double*)s->buf[out],
                  (double*)s->bufd[out], s->d_fluid, &s->d_state->dt, s->plane, s->nx, s->ny, s->pitch, a, b};
  combine2d_tangent_kernel<<<s->num_sms * 8, 256, 0, s->stream>>>(C);
  s->launches++;
  if (e1) cudaEventRecord(e1, s->stream);
  CU(cudaGetLastError());
  return JXS_OK;
}

int tangent2d_common(jxs_solver* s, void* U, void* Udot, double gamma_dot, double dt, int nsteps) {
  if (s->mlp_on || s->cnn_on) return fail(s, JXS_ESTATE, "the tangent does not differentiate the 2D networks");
  int rc = deriv2d_scratch(s);
  if (rc != JXS_OK) return rc;
  const size_t bytes = (size_t)4 * s->plane * s->elem;
  for (int b = 0; b < 3; ++b)
    if (!s->bufd[b]) {
      CU(cudaMalloc(&s->bufd[b], bytes));
      CU(cudaMemsetAsync(s->bufd[b], 0, bytes, s->stream));
    }
  CU(pad(s, U, s->buf[0]));
  CU(pad(s, Udot, s->bufd[0]));
  s->events_used = 0;
  s->mlp_events_used = 0;
  int at = 0;
  for (int n = 0; n < nsteps; ++n) {
    prepare_step_kernel<<<1, 1, 0, s->stream>>>(s->d_state, 0, 0.0, dt);
    s->launches++;
    CU(cudaGetLastError());
    if (s->scheme == JXS_EULER) {  // Eq. 10: one stage with (a, b) = (0, 1); the two buffers swap roles
      rc = tangent_stage2d(s, at, at ^ 1, 0.0, 1.0, gamma_dot);
      if (rc != JXS_OK) return rc;
      at ^= 1;
      continue;
    }
    static const double ab[3][2] = {{0.0, 1.0}, {0.75, 0.25}, {1.0 / 3.0, 2.0 / 3.0}};  // R5
    static const int io[3][2] = {{0, 1}, {1, 2}, {2, 0}};
    for (int st = 0; st < 3; ++st) {
      rc = tangent_stage2d(s, io[st][0], io[st][1], ab[st][0], ab[st][1], gamma_dot);
      if (rc != JXS_OK) return rc;
    }
  }
  CU(unpad(s, s->buf[at], U));
  CU(unpad(s, s->bufd[at], Udot));
  return finish_steps(s, nsteps);
}

// recorded forward sweep in 2D: the padded, ghost-filled input state of every stage is kept (3 per SSP-RK3 step, 1
// per forward-Euler step, or with checkpointing U^n only), plus the final state
int record2d_common(jxs_solver* s, void* U, double dt, int nsteps) {
  if (s->mlp_on || s->cnn_on) return fail(s, JXS_ESTATE, "the adjoint does not differentiate the 2D networks");
  int rc = deriv2d_scratch(s);
  if (rc != JXS_OK) return rc;
  s->tape_steps = 0;
  const size_t state = (size_t)4 * s->plane;
  const bool ckpt = s->checkpoint && s->scheme == JXS_SSPRK3;
  const int per_step = (s->scheme == JXS_EULER || ckpt) ? 1 : 3;
  const size_t bytes = state * sizeof(double) * (per_step * (size_t)nsteps + 1);
  if (!s->tape2 || s->tape2_bytes < bytes) {
    cudaFree(s->tape2);
    s->tape2 = nullptr;
    s->tape2_bytes = 0;
    if (cudaMalloc(&s->tape2, bytes) != cudaSuccess) {
      cudaGetLastError();
      return fail(s, JXS_ENOMEM, "the recorded trajectory does not fit in device memory");
    }
    s->tape2_bytes = bytes;
  }
  auto T = [&](long long i) { return (void*)(s->tape2 + i * state); };
  CU(pad(s, U, s->buf[0]));
  s->events_used = 0;
  s->mlp_events_used = 0;
  const size_t sb = state * sizeof(double);
  // The fused stage kernel reads through the tensor maps of buf[0..2]; the recording therefore steps in the handle's
  // buffers exactly like jxs_step_fixed_dt and copies each stage's (ghost-filled) input to the tape.
  auto sweep = [&]() -> int {
  long long rec = 0;
  for (long long n = 0; n < nsteps; ++n) {
    prepare_step_kernel<<<1, 1, 0, s->stream>>>(s->d_state, 0, 0.0, dt);
    s->launches++;
    CU(cudaGetLastError());
    if (s->scheme == JXS_EULER) {
      const int at = (int)(n & 1);
      CU(ghost_fill(s, s->buf[at]));
      CU(cudaMemcpyAsync(T(rec++), s->buf[at], sb, cudaMemcpyDeviceToDevice, s->stream));
      CU(stage(s, s->buf[at], nullptr, s->buf[at ^ 1], 0, 0.0, 1.0, nullptr));
      continue;
    }
    CU(ghost_fill(s, s->buf[0]));
    CU(cudaMemcpyAsync(T(rec++), s->buf[0], sb, cudaMemcpyDeviceToDevice, s->stream));
    CU(stage(s, s->buf[0], nullptr, s->buf[1], 0, 0.0, 1.0, nullptr));
    CU(ghost_fill(s, s->buf[1]));
    if (!ckpt) CU(cudaMemcpyAsync(T(rec++), s->buf[1], sb, cudaMemcpyDeviceToDevice, s->stream));
    CU(stage(s, s->buf[1], s->buf[0], s->buf[2], 0, 0.75, 0.25, nullptr));
    CU(ghost_fill(s, s->buf[2]));
    if (!ckpt) CU(cudaMemcpyAsync(T(rec++), s->buf[2], sb, cudaMemcpyDeviceToDevice, s->stream));
    CU(stage(s, s->buf[2], s->buf[0], s->buf[0], 0, 1.0 / 3.0, 2.0 / 3.0, nullptr));
  }
  const int at = s->scheme == JXS_EULER ? (nsteps & 1) : 0;
  CU(cudaMemcpyAsync(T(rec), s->buf[at], sb, cudaMemcpyDeviceToDevice, s->stream));
  return JXS_OK;
  };
  {
    long long dt_bits;
    std::memcpy(&dt_bits, &dt, 8);
    const std::vector<long long> key = {nsteps, dt_bits, s->scheme, ckpt, (long long)(size_t)s->tape2, s->rows_per_seg, s->grid};
    rc = run_sweep(s, s->rec2_graph, key, sweep);
    if (rc != JXS_OK) return rc;
  }
  const int at = s->scheme == JXS_EULER ? (nsteps & 1) : 0;
  CU(unpad(s, s->buf[at], U));
  rc = finish_steps(s, nsteps);
  if (rc != JXS_OK) return rc;
  s->tape_steps = nsteps;
  s->tape_scheme = s->scheme;
  s->tape_ckpt = ckpt;
  s->tape_dt = dt;
  return JXS_OK;
}

// gamma_bar accumulator: adj2 + 16 * plane; loss accumulator behind it
double* adj2_state(const jxs_solver* s, int i) { return s->adj2 + (size_t)i * 4 * s->plane; }
double* adj2_gbar(const jxs_solver* s) { return s->adj2 + (size_t)16 * s->plane; }

cudaError_t add_partials(jxs_solver* s, long long n) {
  sum_partials_kernel<<<1, 1024, 0, s->stream>>>(s->d_gpart, n, adj2_gbar(s));
  s->launches++;
  return cudaGetLastError();
}

// reverse of one 2D stage U_out = b (U + dt fl L(U)) (+ a U0): Ubar_in = b Ubar_out + b dt (dL/dU)^T (fl Ubar_out)
// + e1 E1 + e2 E2, then the transposed immersed-boundary fill and the transposed frame fill; gamma_bar accumulates
int adjoint_stage2d(jxs_solver* s, const double* U, const double* out, double* in, double b, const double* E1, double e1,
                    const double* E2, double e2) {
  const size_t sb = (size_t)4 * s->plane * sizeof(double);
  CU(cudaMemsetAsync(in, 0, sb, s->stream));
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  if (s->profiling && s->events_used + 2 <= (int)s->events.size()) {
    ev0 = s->events[s->events_used++];
    ev1 = s->events[s->events_used++];
    cudaEventRecord(ev0, s->stream);
  }
  // Lx: the rows
  const int px = (s->nx + 6 + A1D_OUT - 1) / A1D_OUT, py = (s->ny + 6 + A1D_OUT - 1) / A1D_OUT;
  AdjointLineArgs X{U, out, in, E1, E2, s->d_fluid, s->d_gpart, lines_x(s), s->tape_dt, s->gamma, 1.0 / s->dx, b, e1, e2, s->nu, 1};
  adjoint_line_kernel<<<dim3(px, s->ny), A1D_TB, 0, s->stream>>>(X);
  s->launches++;
  CU(add_partials(s, (long long)px * s->ny));
  // Ly: the rows of the transposed copies
  CU(to_transposed(s, U, s->tr[0]));
  CU(to_transposed(s, out, s->tr[1]));
  AdjointLineArgs Y{s->tr[0], s->tr[1], s->tr[2], nullptr, nullptr, s->d_fluid_t, s->d_gpart, lines_y(s), s->tape_dt, s->gamma,
                    1.0 / s->dy, b, 0.0, 0.0, s->nu, 0};
  adjoint_line_kernel<<<dim3(py, s->nx), A1D_TB, 0, s->stream>>>(Y);
  s->launches++;
  CU(add_partials(s, (long long)py * s->nx));
  CU(add_from_transposed(s, s->tr[2], in, 0, s->ny + 6));
  // Lv
  if (s->mu > 0) {
    const size_t nfx = (size_t)s->ny * (s->nx + 1);
    Visc2dAdjArgs V{U, out, s->d_fluid, s->visc_C, s->visc_C + 7 * nfx, in, s->d_gpart, s->plane, s->nx, s->ny, s->pitch,
                    s->gamma, s->mu, s->Pr, 1.0 / s->dx, 1.0 / s->dy, b * s->tape_dt};
    const int gs = s->num_sms * 8;
    viscous2d_adjoint_faces_kernel<<<gs, 256, 0, s->stream>>>(V);
    viscous2d_adjoint_gather_kernel<<<gs, 256, 0, s->stream>>>(V);
    viscous2d_adjoint_gamma_kernel<<<gs, 256, 0, s->stream>>>(V, s->d_gpart + gs);
    s->launches += 3;
    CU(add_partials(s, 2LL * gs));
  }
  if (ev1) cudaEventRecord(ev1, s->stream);
  // the transposed fills, in the reverse order of the fills
  if (s->n_ghost > 0) {
    IbmList L{s->d_cell, s->d_donor, s->d_w, s->d_nrm, s->n_ghost};
    double* gcontrib = s->d_contrib + (size_t)16 * s->n_ghost;
    ibm_adjoint_ghost_kernel<<<(s->n_ghost + 127) / 128, 128, 0, s->stream>>>(U, in, s->plane, L, s->gamma, s->d_contrib, gcontrib);
    ibm_adjoint_donor_kernel<<<(s->n_donor + 127) / 128, 128, 0, s->stream>>>(in, s->plane, s->d_dcell, s->d_drows, s->d_dentry,
                                                                           s->n_donor, s->d_contrib);
    sum_partials_kernel<<<1, 1024, 0, s->stream>>>(gcontrib, s->n_ghost, adj2_gbar(s));
    s->launches += 3;
  }
  for (int axis = 1; axis >= 0; --axis) {
    const int nline = axis == 1 ? s->nx + 6 : s->ny;
    frame_fold_kernel<<<(2 * nline + 127) / 128, 128, 0, s->stream>>>(in, dims(s), bcspec(s), axis, s->bc.inflow[3], s->gamma,
                                                                      s->d_gpart);
    s->launches++;
    CU(add_partials(s, 2LL * nline));
  }
  CU(cudaGetLastError());
  return JXS_OK;
}

int adjoint2d_common(jxs_solver* s, void* Ubar, double* gamma_bar, const double* targets, double* loss) {
  if (!s->tape2 || s->tape_steps < 1) return fail(s, JXS_ESTATE, "no recorded steps: call jxs_step_fixed_dt_record first");
  const size_t state = (size_t)4 * s->plane, sb = state * sizeof(double);
  if (!s->adj2) CU(cudaMalloc(&s->adj2, (4 * state + 2) * sizeof(double)));
  CU(cudaMemsetAsync(s->adj2, 0, (4 * state + 2) * sizeof(double), s->stream));
  auto T = [&](long long i) { return s->tape2 + i * state; };
  auto B = [&](int i) { return adj2_state(s, i); };
  const int per_step = (s->tape_scheme == JXS_EULER || s->tape_ckpt) ? 1 : 3;
  const long long ncell4 = 4LL * s->nx * s->ny;
  double* loss_acc = adj2_gbar(s) + 1;
  const int igs = s->num_sms * 4;
  auto inject = [&](long long n, int into, int accumulate) -> cudaError_t {  // Eq. 14: state after step n vs targets[n-1]
    mse_inject2d_kernel<<<igs, 256, 0, s->stream>>>(T(per_step * n), targets + (n - 1) * ncell4, B(into), dims(s),
                                                    2.0 / (s->tape_steps * (double)ncell4), accumulate, s->d_gpart);
    sum_partials_kernel<<<1, 1024, 0, s->stream>>>(s->d_gpart, igs, loss_acc);
    s->launches += 2;
    return cudaGetLastError();
  };
  if (targets) CU(inject(s->tape_steps, 0, 0));
  else CU(pad(s, Ubar, B(0)));
  s->events_used = 0;
  int x = 0;
  auto sweep = [&]() -> int {
  x = 0;
  for (long long n = s->tape_steps - 1; n >= 0; --n) {
    if (targets && n + 1 < s->tape_steps) CU(inject(n + 1, x, 1));
    int rc;
    if (s->tape_scheme == JXS_EULER) {
      rc = adjoint_stage2d(s, T(n), B(x), B(x ^ 1), 1.0, nullptr, 0.0, nullptr, 0.0);
      if (rc != JXS_OK) return rc;
      x ^= 1;
      continue;
    }
    const double *S0 = T(3 * n), *S1 = T(3 * n + 1), *S2 = T(3 * n + 2);
    if (s->tape_ckpt) {  // recompute the two inner stage states from the kept U^n (in the handle's own buffers)
      CU(cudaMemcpyAsync(s->buf[0], T(n), sb, cudaMemcpyDeviceToDevice, s->stream));
      CU(cudaMemcpyAsync(&s->d_state->dt, &s->tape_dt, sizeof(double), cudaMemcpyHostToDevice, s->stream));
      CU(stage(s, s->buf[0], nullptr, s->buf[1], 0, 0.0, 1.0, nullptr));
      CU(ghost_fill(s, s->buf[1]));
      CU(stage(s, s->buf[1], s->buf[0], s->buf[2], 0, 0.75, 0.25, nullptr));
      CU(ghost_fill(s, s->buf[2]));
      S0 = (const double*)s->buf[0]; S1 = (const double*)s->buf[1]; S2 = (const double*)s->buf[2];
    }
    const int y2 = (x + 1) & 3, y1 = (x + 2) & 3, y0 = (x + 3) & 3;
    // U^{n+1} = 1/3 U0 + 2/3 (U2 + dt L(U2));  U2 = 3/4 U0 + 1/4 (U1 + dt L(U1));  U1 = U0 + dt L(U0)   (R5)
    rc = adjoint_stage2d(s, S2, B(x), B(y2), 2.0 / 3.0, nullptr, 0.0, nullptr, 0.0);
    if (rc == JXS_OK) rc = adjoint_stage2d(s, S1, B(y2), B(y1), 0.25, nullptr, 0.0, nullptr, 0.0);
    if (rc == JXS_OK) rc = adjoint_stage2d(s, S0, B(y1), B(y0), 1.0, B(x), 1.0 / 3.0, B(y2), 0.75);
    if (rc != JXS_OK) return rc;
    x = y0;
  }
  return JXS_OK;
  };
  {
    int rc;
    if (s->tape_ckpt) {  // the checkpointed sweep copies dt from a host variable inside the loop: plain launches
      rc = sweep();
    } else {
      long long dt_bits;
      std::memcpy(&dt_bits, &s->tape_dt, 8);
      const std::vector<long long> key = {s->tape_steps, dt_bits, s->tape_scheme, (long long)(size_t)s->tape2,
                                          (long long)(size_t)s->adj2, (long long)(size_t)targets};
      rc = run_sweep(s, s->adj2_graph, key, sweep);
      if (rc == JXS_OK) {  // where the adjoint of U^0 ends up does not depend on how the sweep was run
        x = 0;
        if (s->tape_scheme == JXS_EULER) x = (int)(s->tape_steps & 1);
        else for (long long n = 0; n < s->tape_steps; ++n) x = (x + 3) & 3;
      }
    }
    if (rc != JXS_OK) return rc;
  }
  CU(unpad(s, B(x), Ubar));
  double out[2];
  CU(cudaMemcpyAsync(out, adj2_gbar(s), sizeof(out), cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  *gamma_bar = out[0];
  if (loss) *loss = out[1] / (s->tape_steps * (double)ncell4);
  if (s->profiling) {
    s->stage_ms = 0;
    s->stage_launches = s->events_used / 2;
    for (int i = 0; i + 1 < s->events_used; i += 2) {
      float ms = 0;
      cudaEventElapsedTime(&ms, s->events[i], s->events[i + 1]);
      s->stage_ms += ms;
    }
  }
  return JXS_OK;
}

}  // namespace

extern "C" {

static int create_common(int nb, int nx, int ny, double dx, double dy, double gamma, const double* mu_b, double Pr,
                         const jxs_bc* bc_b, int dtype, void* cuda_stream, jxs_solver** out) {
  if (!out) return JXS_EINVAL;
  *out = nullptr;
  if (!bc_b || !mu_b || nb < 1) return JXS_EINVAL;
  if (nb > 1 && ny == 1) return JXS_EINVAL;  // batches are two-dimensional
  if (nx < 8 || (ny < 8 && ny != 1) || !(dx > 0) || !(dy > 0) || !(gamma > 1)) return JXS_EINVAL;
  if (dtype != JXS_F64 && dtype != JXS_F32) return JXS_EINVAL;
  for (int m = 0; m < nb; ++m) {
    const jxs_bc* bc = bc_b + m;
    if (!(mu_b[m] >= 0) || (mu_b[m] > 0 && !(Pr > 0)) || (mu_b[m] > 0) != (mu_b[0] > 0)) return JXS_EINVAL;
    const int kinds[4] = {bc->xlo, bc->xhi, bc->ylo, bc->yhi};
    for (int k : kinds)
      if (k < 0 || k > 3) return JXS_EINVAL;
    if ((bc->xlo == JXS_BC_PERIODIC) != (bc->xhi == JXS_BC_PERIODIC)) return JXS_EINVAL;
    if ((bc->ylo == JXS_BC_PERIODIC) != (bc->yhi == JXS_BC_PERIODIC)) return JXS_EINVAL;
    for (int k = 0; k < 4; ++k)
      if (!std::isfinite(bc->inflow[k])) return JXS_EINVAL;
    // the members of a batch share the kinds of their boundary conditions; the inflow states may differ
    if (bc->xlo != bc_b->xlo || bc->xhi != bc_b->xhi || bc->ylo != bc_b->ylo || bc->yhi != bc_b->yhi) return JXS_EINVAL;
  }
  const jxs_bc* bc = bc_b;
  const double mu = mu_b[0];
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return JXS_ECUDA;
  jxs_solver* s = new (std::nothrow) jxs_solver;
  if (!s) return JXS_ENOMEM;
  s->nx = nx; s->ny = ny; s->dx = dx; s->dy = dy; s->gamma = gamma; s->mu = mu; s->Pr = Pr; s->bc = *bc;
  s->nb = nb;
  s->mu_b.assign(mu_b, mu_b + nb);
  s->bc_b.assign(bc_b, bc_b + nb);
  s->t_b.assign(nb, 0.0);
  s->dt_b.assign(nb, 0.0);
  if (ny == 1) s->bc.ylo = s->bc.yhi = JXS_BC_TRANSMISSIVE;  // the ghost rows of a single row are copies of it
  s->dtype = dtype;
  s->elem = dtype == JXS_F64 ? 8 : 4;
  s->stream = (cudaStream_t)cuda_stream;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { delete s; return JXS_ECUDA; }
  if (prop.major != 10 || prop.minor != 0) { delete s; return JXS_ECUDA; }  // the library holds sm_100a code only
  s->dev = dev;
  s->num_sms = prop.multiProcessorCount;
  choose_decomposition(s);
  const int SOUT = dtype == JXS_F64 ? sout<double>() : sout<float>();
  s->pitch = ((SOUT * s->nstrips + 6 + 15) / 16) * 16;
  s->plane = (long long)nb * (ny + 6) * s->pitch;
  if (s->plane > 0x7fffffffLL) { delete s; return JXS_EINVAL; }
  const size_t pbytes = (size_t)4 * s->plane * s->elem;
  cudaError_t e = cudaSuccess;
  for (int b = 0; b < 3 && e == cudaSuccess; ++b) e = cudaMalloc(&s->buf[b], pbytes);
  if (e == cudaSuccess) e = cudaMalloc(&s->stage_io, (size_t)4 * nx * ny * nb * s->elem);
  if (e == cudaSuccess) e = cudaMalloc(&s->d_state, sizeof(StepState) * nb);
  if (e == cudaSuccess) e = cudaMemsetAsync(s->d_state, 0, sizeof(StepState) * nb, s->stream);
  if (e == cudaSuccess && nb > 1) {  // per-member inflow states and viscous coefficients (the order of StageArgs)
    std::vector<double> inflow(4 * (size_t)nb), vt(10 * (size_t)nb);
    for (int m = 0; m < nb; ++m) {
      const double r = bc_b[m].inflow[0], u = bc_b[m].inflow[1], v = bc_b[m].inflow[2], p = bc_b[m].inflow[3];
      inflow[4 * m] = r; inflow[4 * m + 1] = r * u; inflow[4 * m + 2] = r * v;
      inflow[4 * m + 3] = p / (gamma - 1.0) + 0.5 * r * (u * u + v * v);
      const double mm = mu_b[m], kap = mm > 0 ? mm * gamma / ((gamma - 1.0) * Pr) : 0.0, dxi = 1.0 / dx, dyi = 1.0 / dy;
      const double c[10] = {4.0 / 3.0 * mm * dyi, 2.0 / 3.0 * mm * 0.25 * dxi, mm * dyi, mm * 0.25 * dxi, kap * dyi,
                            4.0 / 3.0 * mm * dxi, 2.0 / 3.0 * mm * 0.25 * dyi, mm * dxi, mm * 0.25 * dyi, kap * dxi};
      for (int q = 0; q < 10; ++q) vt[10 * m + q] = c[q];
    }
    e = cudaMalloc(&s->d_inflow_tab, inflow.size() * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(s->d_inflow_tab, inflow.data(), inflow.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&s->d_vtab, vt.size() * s->elem);
    if (e == cudaSuccess) {
      if (dtype == JXS_F64) e = cudaMemcpy(s->d_vtab, vt.data(), vt.size() * sizeof(double), cudaMemcpyHostToDevice);
      else {
        std::vector<float> vf(vt.begin(), vt.end());
        e = cudaMemcpy(s->d_vtab, vf.data(), vf.size() * sizeof(float), cudaMemcpyHostToDevice);
      }
    }
  }
  if (e != cudaSuccess) {
    const int rc = e == cudaErrorMemoryAllocation ? JXS_ENOMEM : JXS_ECUDA;
    jxs_destroy(s);
    cudaGetLastError();
    return rc;
  }
  for (int b = 0; b < 3; ++b)
    if (!make_tensor_map(s, s->buf[b], CW, &s->tm_row[b]) || !make_tensor_map(s, s->buf[b], dtype == JXS_F64 ? Epi<double>::W : Epi<float>::W, &s->tm_epi[b])) {
      jxs_destroy(s);
      return JXS_ECUDA;
    }
  const double e_rest = 1.0 / (gamma - 1.0);
  for (int b = 0; b < 3; ++b) {
    if (dtype == JXS_F64) fill_benign_kernel<double><<<s->num_sms * 4, 256, 0, s->stream>>>((double*)s->buf[b], dims(s), e_rest);
    else fill_benign_kernel<float><<<s->num_sms * 4, 256, 0, s->stream>>>((float*)s->buf[b], dims(s), (float)e_rest);
    s->launches++;
  }
  if (cudaGetLastError() != cudaSuccess) { jxs_destroy(s); return JXS_ECUDA; }
  *out = s;
  return JXS_OK;
}

int jxs_create(int nx, int ny, double dx, double dy, double gamma, double mu, double Pr, const jxs_bc* bc, int dtype,
               void* cuda_stream, jxs_solver** out) {
  return create_common(1, nx, ny, dx, dy, gamma, &mu, Pr, bc, dtype, cuda_stream, out);
}
int jxs_create_batch(int nbatch, int nx, int ny, double dx, double dy, double gamma, const double* mu, double Pr,
                     const jxs_bc* bc, int dtype, void* cuda_stream, jxs_solver** out) {
  return create_common(nbatch, nx, ny, dx, dy, gamma, mu, Pr, bc, dtype, cuda_stream, out);
}

void jxs_destroy(jxs_solver* s) {
  if (!s) return;
  cudaStreamSynchronize(s->stream);
  drop_graph(s);
  if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
  for (int b = 0; b < 3; ++b) cudaFree(s->buf[b]);
  cudaFree(s->stage_io);
  for (int b = 0; b < 3; ++b) cudaFree(s->bufd[b]);
  if (s->tan_exec) cudaGraphExecDestroy(s->tan_exec);
  cudaFree(s->d_mse);
  cudaFree(s->d_theta); cudaFree(s->d_dF1d); cudaFree(s->d_theta_bar); cudaFree(s->d_Wmlp);
  cudaFree(s->tape);
  cudaFree(s->tape2); cudaFree(s->adj2); cudaFree(s->visc_C); cudaFree(s->d_gpart);
  for (int q = 0; q < 4; ++q) cudaFree(s->tr[q]);
  cudaFree(s->Lnat[0]); cudaFree(s->Lnat[1]);
  cudaFree(s->ckpt);
  cudaFree(s->adj);
  cudaFree(s->d_state);
  cudaFree(s->d_inflow_tab); cudaFree(s->d_vtab);
  free_ibm(s);
  cudaFree(s->d_mlp_blob); cudaFree(s->d_dFG);
  for (int d = 0; d < 2; ++d) {
    cudaFree(s->cnn_X[d].data);
    for (int l = 0; l < 3; ++l) cudaFree(s->d_cnn_blob3[d][l]);
  }
  for (cudaEvent_t ev : s->events) cudaEventDestroy(ev);
  for (cudaEvent_t ev : s->mlp_events) cudaEventDestroy(ev);
  delete s;
}

const char* jxs_last_error(const jxs_solver* s) { return s ? s->err.c_str() : "null handle"; }

// the device mask = the body's fluid mask with the inactive rows cleared (single handles only)
static int apply_active_rows(jxs_solver* s) {
  std::vector<uint8_t> m = s->fluid_host.empty() ? std::vector<uint8_t>((size_t)s->nx * s->ny, 1) : s->fluid_host;
  for (int j = 0; j < s->ny; ++j)
    if (j < s->act_lo || j >= s->act_hi) std::fill(m.begin() + (size_t)j * s->nx, m.begin() + (size_t)(j + 1) * s->nx, 0);
  if (!s->d_fluid) CU(cudaMalloc(&s->d_fluid, m.size()));
  CU(cudaMemcpy(s->d_fluid, m.data(), m.size(), cudaMemcpyHostToDevice));
  return JXS_OK;
}

int jxs_set_ibm(jxs_solver* s, const double* phi) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  drop_graph(s);
  CU(cudaStreamSynchronize(s->stream));
  free_ibm(s);
  s->fluid_host.clear();
  if (!phi) return s->act_set ? apply_active_rows(s) : JXS_OK;
  if (s->ny == 1) return fail(s, JXS_EINVAL, "no immersed boundary in one-dimensional problems");
  const int nx = s->nx, ny = s->ny;
  const double dx = s->dx, dy = s->dy;
  // classification (R9 I1, I2): 1 = fluid in `fl`; ghost = non-fluid cell that some fluid cell's
  // WENO stencil (3 cells along an axis) or viscous stencil (3x3 box) touches
  std::vector<uint8_t> fl_all((size_t)nx * ny * s->nb);
  for (size_t c = 0; c < fl_all.size(); ++c) fl_all[c] = phi[c] > 0.0 ? 1 : 0;
  std::vector<int> cell, donor;
  std::vector<double> wts, nrm;
  const double* const phi_all = phi;
  for (int member = 0; member < s->nb; ++member) {  // a batch: one level set per member, [nb][ny][nx]
  const uint8_t* fl = fl_all.data() + (size_t)member * nx * ny;
  phi = phi_all + (size_t)member * nx * ny;
  const int moff = member * (ny + 6) * s->pitch;  // this member's rows in the padded buffers
  auto is_fluid = [&](int i, int j) { return i >= 0 && i < nx && j >= 0 && j < ny && fl[(size_t)j * nx + i]; };
  static const int off[16][2] = {{1, 0}, {-1, 0}, {0, 1}, {0, -1}, {2, 0}, {-2, 0}, {0, 2}, {0, -2},
                                 {3, 0}, {-3, 0}, {0, 3}, {0, -3}, {1, 1}, {-1, 1}, {1, -1}, {-1, -1}};
  const double h = std::min(dx, dy);
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      if (fl[(size_t)j * nx + i]) continue;
      // y-slab sharding: an edge behind inactive rows is a cut through the domain, not its boundary; bodies may cross
      // it, and ghost cells of inactive rows whose stencils leave the slab are skipped (their rows are refreshed from
      // the rank that owns them before every stage)
      const bool inactive = s->act_set && (j < s->act_lo || j >= s->act_hi);
      const bool cut_lo = s->act_set && s->act_lo > 0, cut_hi = s->act_set && s->act_hi < ny;
      if (i < 8 || i >= nx - 8 || (j < 8 && !cut_lo) || (j >= ny - 8 && !cut_hi))
        return fail(s, JXS_EINVAL, "IBM body closer than 8 cells to a domain edge");
      bool ghost = false;
      for (int q = 0; q < 16 && !ghost; ++q) ghost = is_fluid(i + off[q][0], j + off[q][1]);
      if (!ghost) continue;
      if (j == 0 || j == ny - 1) {
        if (inactive) continue;
        return fail(s, JXS_EINVAL, "IBM: a ghost cell of an active row lies on a slab edge (overlap too small)");
      }
      // I3: unit normal from central differences of the sampled level set
      const double px = (phi[(size_t)j * nx + i + 1] - phi[(size_t)j * nx + i - 1]) / (2.0 * dx);
      const double py = (phi[(size_t)(j + 1) * nx + i] - phi[(size_t)(j - 1) * nx + i]) / (2.0 * dy);
      const double pn = std::sqrt(px * px + py * py);
      if (!(pn > 0.0)) return fail(s, JXS_EINVAL, "IBM: zero level-set gradient at a ghost cell");
      const double n0 = px / pn, n1 = py / pn;
      // I4: image point, mirrored through the surface along the normal
      const double depth = std::fabs(phi[(size_t)j * nx + i]);
      // kept as its offset from the ghost cell's centre, in cells: x_I = (i + 0.5 + ox) dx.  The donors and weights
      // then do not depend on where the cell sits in the array (a slab of a sharded run builds the same list)
      double ox = 2.0 * depth * n0 / dx, oy = 2.0 * depth * n1 / dy;
      // I5: bilinear donors, non-fluid ones dropped, weights renormalised; probe outwards if empty
      int di[4], dj[4];
      double w[4], sum = 0.0;
      for (int attempt = 0; attempt < 9; ++attempt) {
        const double flx = std::floor(ox), fly = std::floor(oy);
        const int i0 = i + (int)flx, j0 = j + (int)fly;
        const double tx = ox - flx, ty = oy - fly;
        const double bw[4] = {(1 - tx) * (1 - ty), tx * (1 - ty), (1 - tx) * ty, tx * ty};
        sum = 0.0;
        for (int d = 0; d < 4; ++d) {
          di[d] = i0 + (d & 1); dj[d] = j0 + (d >> 1);
          w[d] = is_fluid(di[d], dj[d]) ? bw[d] : 0.0;
          sum += w[d];
        }
        if (sum > 0.0) break;
        ox += h * n0 / dx; oy += h * n1 / dy;
      }
      if (!(sum > 0.0)) {
        if (inactive) continue;
        return fail(s, JXS_EINVAL, "IBM: ghost cell without a fluid donor");
      }
      cell.push_back(moff + (j + 3) * s->pitch + i + 3);
      for (int d = 0; d < 4; ++d) {
        const double wd = w[d] / sum;
        wts.push_back(wd);
        donor.push_back(moff + (wd > 0.0 ? (dj[d] + 3) * s->pitch + di[d] + 3 : (j + 3) * s->pitch + i + 3));
      }
      nrm.push_back(n0); nrm.push_back(n1);
    }
  }  // members
  phi = phi_all;
  const std::vector<uint8_t>& fl = fl_all;
  const int ng = (int)cell.size();
  s->fluid_host = fl;
  CU(cudaMalloc(&s->d_fluid, fl.size()));
  CU(cudaMemcpy(s->d_fluid, fl.data(), fl.size(), cudaMemcpyHostToDevice));
  if (s->act_set) {
    const int rc_ = apply_active_rows(s);
    if (rc_ != JXS_OK) return rc_;
  }
  if (ng > 0) {
    CU(cudaMalloc(&s->d_cell, sizeof(int) * ng));
    CU(cudaMalloc(&s->d_donor, sizeof(int) * 4 * ng));
    CU(cudaMalloc(&s->d_w, sizeof(double) * 4 * ng));
    CU(cudaMalloc(&s->d_nrm, sizeof(double) * 2 * ng));
    CU(cudaMemcpy(s->d_cell, cell.data(), sizeof(int) * ng, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(s->d_donor, donor.data(), sizeof(int) * 4 * ng, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(s->d_w, wts.data(), sizeof(double) * 4 * ng, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(s->d_nrm, nrm.data(), sizeof(double) * 2 * ng, cudaMemcpyHostToDevice));
  }
  s->n_ghost = ng;
  // for the reverse sweep (deriv2d_kernels.cuh): the fluid mask transposed, and the gather list transposed —
  // every donor cell with the entries 16 q + 4 d of the ghost cells q it feeds, in increasing order (a fixed
  // summation order instead of atomics)
  if (s->nb == 1) {
    std::vector<uint8_t> flt((size_t)nx * ny);
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) flt[(size_t)i * ny + j] = fl[(size_t)j * nx + i];
    CU(cudaMalloc(&s->d_fluid_t, flt.size()));
    CU(cudaMemcpy(s->d_fluid_t, flt.data(), flt.size(), cudaMemcpyHostToDevice));
    std::vector<std::pair<int, int>> de;  // (donor cell offset, entry)
    for (int q = 0; q < ng; ++q)
      for (int d = 0; d < 4; ++d)
        if (wts[4 * q + d] > 0.0) de.emplace_back(donor[4 * q + d], 16 * q + 4 * d);
    std::sort(de.begin(), de.end());
    std::vector<int> dcell, rows, entry;
    for (size_t e = 0; e < de.size(); ++e) {
      if (e == 0 || de[e].first != de[e - 1].first) { dcell.push_back(de[e].first); rows.push_back((int)e); }
      entry.push_back(de[e].second);
    }
    rows.push_back((int)de.size());
    s->n_donor = (int)dcell.size();
    if (s->n_donor > 0) {
      CU(cudaMalloc(&s->d_dcell, sizeof(int) * dcell.size()));
      CU(cudaMalloc(&s->d_drows, sizeof(int) * rows.size()));
      CU(cudaMalloc(&s->d_dentry, sizeof(int) * entry.size()));
      CU(cudaMalloc(&s->d_contrib, sizeof(double) * 17 * (size_t)ng));
      CU(cudaMemcpy(s->d_dcell, dcell.data(), sizeof(int) * dcell.size(), cudaMemcpyHostToDevice));
      CU(cudaMemcpy(s->d_drows, rows.data(), sizeof(int) * rows.size(), cudaMemcpyHostToDevice));
      CU(cudaMemcpy(s->d_dentry, entry.data(), sizeof(int) * entry.size(), cudaMemcpyHostToDevice));
    }
  }
  return JXS_OK;
}

int jxs_set_flux_mlp(jxs_solver* s, const float* weights, const double in_scale[4], const double out_scale[4]) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  drop_graph(s);
  CU(cudaStreamSynchronize(s->stream));
  if (!weights) { s->mlp_on = false; s->mlp1d_on = false; s->tape_steps = 0; return JXS_OK; }
  if (s->cnn_on) return fail(s, JXS_ESTATE, "the CNN flux is set: disable it first (jxs_set_flux_cnn(NULL))");
  if (!in_scale || !out_scale) return fail(s, JXS_EINVAL, "in_scale / out_scale is NULL");
  for (int k = 0; k < 4; ++k)
    if (!(in_scale[k] > 0) || !std::isfinite(in_scale[k]) || !std::isfinite(out_scale[k]))
      return fail(s, JXS_EINVAL, "in_scale must be > 0 and out_scale finite");
  for (int i = 0; i < 6020; ++i)
    if (!std::isfinite(weights[i])) return fail(s, JXS_EINVAL, "non-finite MLP weight");
  if (s->ny == 1) {  // one-dimensional problems: the fp64 per-face MLP of mlp1d_kernel.cuh
    std::vector<double> th(MLP1D_NDEV);
    for (int i = 0; i < MLP1D_NPARAM; ++i) th[i] = (double)weights[i];
    for (int j = 0; j < 64; ++j) {  // the transposed copies the forward pass reads
      for (int i = 0; i < 24; ++i) th[MLP1D_W1T + i * 64 + j] = th[MLP1D_W1 + j * 24 + i];
      for (int i = 0; i < 64; ++i) th[MLP1D_W2T + i * 64 + j] = th[MLP1D_W2 + j * 64 + i];
    }
    const size_t fbytes = (size_t)4 * s->plane * sizeof(double);
    if (!s->d_theta) CU(cudaMalloc(&s->d_theta, MLP1D_NDEV * sizeof(double)));
    if (!s->d_theta_bar) CU(cudaMalloc(&s->d_theta_bar, MLP1D_NPARAM * sizeof(double)));
    if (!s->d_dF1d) { CU(cudaMalloc(&s->d_dF1d, fbytes)); CU(cudaMemset(s->d_dF1d, 0, fbytes)); }
    if (!s->d_Wmlp) { CU(cudaMalloc(&s->d_Wmlp, fbytes)); CU(cudaMemset(s->d_Wmlp, 0, fbytes)); }
    CU(cudaMemcpy(s->d_theta, th.data(), MLP1D_NDEV * sizeof(double), cudaMemcpyHostToDevice));
    CU(cudaMemset(s->d_theta_bar, 0, MLP1D_NPARAM * sizeof(double)));
    for (int k = 0; k < 4; ++k) { s->in_scale[k] = in_scale[k]; s->out_scale[k] = out_scale[k]; }
    s->mlp1d_on = true;
    s->tape_steps = 0;
    return JXS_OK;
  }
  // W1[64][24], b1[64], W2[64][64], b2[64], W3[4][64], b3[4] -> bf16 tiles in the tensor-core layout + fp32 biases
  std::vector<uint8_t> blob(MLP_BLOB, 0);
  const float *W1 = weights, *b1 = W1 + 64 * 24, *W2 = b1 + 64, *b2 = W2 + 64 * 64, *W3 = b2 + 64, *b3 = W3 + 4 * 64;
  pack_canonical(W1, 64, 24, 64, 32, blob.data() + MLP_OFF_W1);
  pack_canonical(W2, 64, 64, 64, 64, blob.data() + MLP_OFF_W2);
  pack_canonical(W3, 4, 64, 16, 64, blob.data() + MLP_OFF_W3);
  float* bias = reinterpret_cast<float*>(blob.data() + MLP_OFF_BIAS);
  std::memcpy(bias, b1, 64 * 4); std::memcpy(bias + 64, b2, 64 * 4); std::memcpy(bias + 128, b3, 4 * 4);
  std::memcpy(s->mlp_bias, bias, sizeof(s->mlp_bias));
  const size_t fbytes = (size_t)s->plane * sizeof(uint4);
  if (!s->d_mlp_blob) CU(cudaMalloc(&s->d_mlp_blob, MLP_BLOB));
  if (!s->d_dFG) { CU(cudaMalloc(&s->d_dFG, fbytes)); CU(cudaMemset(s->d_dFG, 0, fbytes)); }
  CU(cudaMemcpy(s->d_mlp_blob, blob.data(), MLP_BLOB, cudaMemcpyHostToDevice));
  for (int k = 0; k < 4; ++k) { s->in_scale[k] = in_scale[k]; s->out_scale[k] = out_scale[k]; }
  // strips of 128 cells x row segments: 1 resident CTA per SM, 5 extra rows per segment; the segment count
  // that minimises (waves of CTAs) x (rows a CTA streams)
  s->mlp_strips = (s->nx + 1 + MLP_TILE - 1) / MLP_TILE;
  const int nrows = s->ny + 1;
  const long long slots = (long long)s->num_sms, columns = (long long)s->mlp_strips * s->nb;
  long long best_cost = -1;
  int rps = nrows;
  for (int nseg = 1; nseg <= std::max(1, nrows / 8); ++nseg) {
    const int r = (nrows + nseg - 1) / nseg;
    const long long waves = (columns * ((nrows + r - 1) / r) + slots - 1) / slots;
    const long long cost = waves * (r + 5);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; rps = r; }
  }
  s->mlp_rows_per_seg = rps;
  s->mlp_nseg = (nrows + rps - 1) / rps;
  s->mlp_grid = s->mlp_strips * s->mlp_nseg * s->nb;
  s->mlp_on = true;
  return JXS_OK;
}

int jxs_set_flux_cnn(jxs_solver* s, const float* weights, const double in_scale[4], const double out_scale[4]) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  drop_graph(s);
  CU(cudaStreamSynchronize(s->stream));
  if (!weights) { s->cnn_on = false; return JXS_OK; }
  if (s->ny == 1) return fail(s, JXS_EINVAL, "no CNN flux in one-dimensional problems");
  if (s->nb > 1) return fail(s, JXS_EINVAL, "no CNN flux on a batch handle");
  if (s->mlp_on) return fail(s, JXS_ESTATE, "the flux MLP is set: disable it first (jxs_set_flux_mlp(NULL))");
  if (!in_scale || !out_scale) return fail(s, JXS_EINVAL, "in_scale / out_scale is NULL");
  for (int k = 0; k < 4; ++k)
    if (!(in_scale[k] > 0) || !std::isfinite(in_scale[k]) || !std::isfinite(out_scale[k]))
      return fail(s, JXS_EINVAL, "in_scale must be > 0 and out_scale finite");
  for (int i = 0; i < 6388; ++i)
    if (!std::isfinite(weights[i])) return fail(s, JXS_EINVAL, "non-finite CNN weight");
  // OIHW: W1[32][4][3][3], b1[32], W2[16][32][3][3], b2[16], W3[4][16][3][3], b3[4]
  const float *W1 = weights, *b1 = W1 + 32 * 4 * 9, *W2 = b1 + 32, *b2 = W2 + 16 * 32 * 9, *W3 = b2 + 16, *b3 = W3 + 4 * 16 * 9;
  for (int d = 0; d < 2; ++d) {
    const std::vector<uint8_t> blobs3[3] = {pack_cnn_layer1_im2col(W1, b1, 32, 4, 32, d == 1), pack_cnn_layer3(W2, b2, 16, 32, 2, 16, d == 1),
                                            pack_cnn_layer3(W3, b3, 4, 16, 1, 16, d == 1)};
    for (int l = 0; l < 3; ++l) {
      if (!s->d_cnn_blob3[d][l]) CU(cudaMalloc(&s->d_cnn_blob3[d][l], blobs3[l].size()));
      CU(cudaMemcpy(s->d_cnn_blob3[d][l], blobs3[l].data(), blobs3[l].size(), cudaMemcpyHostToDevice));
    }
    // fields: x-faces rows j (ny), faces f (nx+1); y-faces rows f (ny+1), faces i (nx); zero border all around
    const int na = d == 0 ? s->ny : s->ny + 1, nb = d == 0 ? s->nx + 1 : s->nx;
    const int nbp = (nb + CNN_TILE - 1) / CNN_TILE * CNN_TILE + 2;
    CnnField* f = &s->cnn_X[d];   // the hidden fields never leave the SM (cnn_fused_kernel)
    const size_t bytes = (size_t)(na + 2) * nbp * sizeof(uint4);
    if (!f->data) CU(cudaMalloc(&f->data, bytes));
    CU(cudaMemset(f->data, 0, bytes));
    f->na = na; f->nb = nb; f->nbp = nbp; f->C = 1;
  }
  const size_t fbytes = (size_t)s->plane * sizeof(uint4);
  if (!s->d_dFG) { CU(cudaMalloc(&s->d_dFG, fbytes)); CU(cudaMemset(s->d_dFG, 0, fbytes)); }
  for (int k = 0; k < 4; ++k) { s->cnn_in_scale[k] = in_scale[k]; s->out_scale[k] = out_scale[k]; }
  s->cnn_on = true;
  return JXS_OK;
}

int jxs_flux_cnn_inputs(jxs_solver* s, const void* U, float* Xx, float* Xy) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !Xx || !Xy) return fail(s, JXS_EINVAL, "NULL array");
  if (!s->cnn_on) return fail(s, JXS_ESTATE, "no CNN set (jxs_set_flux_cnn)");
  CU(pad(s, U, s->buf[0]));
  CU(ghost_fill(s, s->buf[0]));
  CU(flux_mlp(s, s->buf[0]));
  const int bs = 256, gs = s->num_sms * 8;
  cnn_inputs_gather_kernel<<<gs, bs, 0, s->stream>>>(s->cnn_X[0], s->cnn_X[1], Xx, Xy, s->nx, s->ny);
  s->launches++;
  CU(cudaGetLastError());
  return JXS_OK;
}

int jxs_set_artificial_viscosity(jxs_solver* s, double nu) {
  if (!s) return JXS_EINVAL;
  if (!(nu >= 0) || !std::isfinite(nu)) return fail(s, JXS_EINVAL, "nu must be finite and >= 0");
  if (s->nb > 1 && nu > 0) return fail(s, JXS_EINVAL, "no nu-term on a batch handle");
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  drop_graph(s);
  s->tape_steps = 0;  // a recording made with another nu cannot be reversed
  s->nu = nu;
  return JXS_OK;
}

int jxs_set_gamma(jxs_solver* s, double gamma) {
  if (!s) return JXS_EINVAL;
  if (!(gamma > 1) || !std::isfinite(gamma)) return fail(s, JXS_EINVAL, "gamma must be > 1");
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  drop_graph(s);
  s->tape_steps = 0;  // a recording made with another gamma cannot be reversed
  s->gamma = gamma;
  return JXS_OK;
}

int jxs_rhs(jxs_solver* s, const void* U, void* dUdt) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !dUdt) return fail(s, JXS_EINVAL, "NULL array");
  CU(pad(s, U, s->buf[0]));
  CU(ghost_fill(s, s->buf[0]));
  CU(flux_mlp(s, s->buf[0]));
  CU(stage(s, s->buf[0], nullptr, dUdt, 1, 0.0, 1.0, nullptr));
  return JXS_OK;
}

int jxs_rhs_host(jxs_solver* s, const void* U, void* dUdt) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !dUdt) return fail(s, JXS_EINVAL, "NULL array");
  const size_t bytes = (size_t)4 * s->nx * s->ny * s->nb * s->elem;
  CU(cudaMemcpyAsync(s->stage_io, U, bytes, cudaMemcpyHostToDevice, s->stream));
  CU(pad(s, s->stage_io, s->buf[0]));
  CU(ghost_fill(s, s->buf[0]));
  CU(flux_mlp(s, s->buf[0]));
  CU(stage(s, s->buf[0], nullptr, s->stage_io, 1, 0.0, 1.0, nullptr));
  CU(cudaMemcpyAsync(dUdt, s->stage_io, bytes, cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  return JXS_OK;
}

int jxs_max_wavespeed(jxs_solver* s, const void* U, double* smax) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !smax) return fail(s, JXS_EINVAL, "NULL argument");
  CU(pad(s, U, s->buf[1]));
  unsigned long long* bits = &s->d_state->smax_bits[0];
  CU(wavespeed(s, s->buf[1], bits));
  std::vector<unsigned long long> h(s->nb);
  CU(cudaMemcpy2DAsync(h.data(), sizeof(unsigned long long), bits, sizeof(StepState), sizeof(unsigned long long), s->nb,
                       cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  std::memcpy(smax, h.data(), sizeof(double) * s->nb);  // one value per member of a batch
  return JXS_OK;
}

int jxs_step(jxs_solver* s, void* U, double cfl, int nsteps) { return step_common(s, U, cfl, 0.0, nsteps, false); }
int jxs_step_fixed_dt(jxs_solver* s, void* U, double dt, int nsteps) {
  if (s && !(dt > 0)) return fail(s, JXS_EINVAL, "dt must be > 0");
  return step_common(s, U, 0.0, dt, nsteps, false);
}
int jxs_step_fixed_dt_tangent(jxs_solver* s, void* U, void* Udot, double gamma_dot, double dt, int nsteps) {
  return tangent_common(s, U, Udot, gamma_dot, dt, nsteps);
}

int jxs_step_fixed_dt_record(jxs_solver* s, void* U, double dt, int nsteps) { return record_common(s, U, dt, nsteps); }
int jxs_adjoint_steps(jxs_solver* s, void* Ubar, double* gamma_bar) { return adjoint_common(s, Ubar, gamma_bar); }
int jxs_adjoint_steps_mse(jxs_solver* s, const void* targets, void* Ubar, double* loss, double* gamma_bar) {
  if (s && !targets) return fail(s, JXS_EINVAL, "targets is NULL");
  return adjoint_common(s, Ubar, gamma_bar, (const double*)targets, loss);
}

int jxs_flux_mlp_gradient(jxs_solver* s, double* grad) {
  if (!s) return JXS_EINVAL;
  if (!grad) return fail(s, JXS_EINVAL, "grad is NULL");
  if (!s->mlp1d_on) return fail(s, JXS_ESTATE, "no flux MLP set on a one-dimensional handle");
  CU(cudaMemcpyAsync(grad, s->d_theta_bar, MLP1D_NPARAM * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  return JXS_OK;
}

int jxs_set_adjoint_checkpointing(jxs_solver* s, int on) {
  if (!s) return JXS_EINVAL;
  s->checkpoint = on != 0;
  return JXS_OK;
}

int jxs_mse_tangent(jxs_solver* s, const void* U, const void* Udot, const void* Utarget, double* loss, double* dloss) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !Udot || !Utarget || !loss || !dloss) return fail(s, JXS_EINVAL, "NULL argument");
  if (s->dtype != JXS_F64) return fail(s, JXS_EINVAL, "the tangent is fp64 only");
  if (!s->d_mse) CU(cudaMalloc(&s->d_mse, (2 * MSE_PARTS + 2) * sizeof(double)));
  const long long n = 4LL * s->nx * s->ny;
  const int parts = (int)std::min<long long>(MSE_PARTS, (n + MSE_TB - 1) / MSE_TB);
  mse_partial_kernel<<<parts, MSE_TB, 0, s->stream>>>((const double*)U, (const double*)Udot, (const double*)Utarget, n,
                                                     s->d_mse);
  mse_final_kernel<<<1, MSE_TB, 0, s->stream>>>(s->d_mse, parts, 1.0 / (double)n, s->d_mse + 2 * MSE_PARTS);
  s->launches += 2;
  CU(cudaGetLastError());
  double out[2];
  CU(cudaMemcpyAsync(out, s->d_mse + 2 * MSE_PARTS, sizeof(out), cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  *loss = out[0];
  *dloss = out[1];
  return JXS_OK;
}

// ---- the allocation-free variant of jxs_mse_tangent (include/jxs.h): the partial sums of the first launch live in a
// file-scope device array instead of a lazily cudaMalloc'ed buffer of the handle.  Every GPU that loads the library holds
// the array (16 KB) until exit.  In host code `g_mse_noalloc_scratch` is only a stand-in for the symbol: its device
// address is looked up once per device (with that device current) and it is that address the kernels are given.
constexpr long long MSE_NOALLOC_MAX_N = JXS_MSE_NOALLOC_MAX_N;
static __device__ __align__(256) double g_mse_noalloc_scratch[2 * MSE_PARTS];
static double* g_mse_noalloc_ptr[MAX_DEVICES] = {nullptr};

int jxs_mse_tangent_noalloc(jxs_solver* s, const void* U, const void* Udot, const void* Utarget, double* out_dev) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !Udot || !Utarget || !out_dev) return fail(s, JXS_EINVAL, "NULL argument");
  if (s->dtype != JXS_F64) return fail(s, JXS_EINVAL, "the tangent is fp64 only");
  const long long n = 4LL * s->nx * s->ny;  // as in jxs_mse_tangent
  if (n > MSE_NOALLOC_MAX_N)
    return fail(s, JXS_EINVAL, "jxs_mse_tangent_noalloc: 4 nx ny entries exceed JXS_MSE_NOALLOC_MAX_N (2^26), the size its "
                               "fixed scratch array is stated for; use jxs_mse_tangent");
  if (s->dev < 0 || s->dev >= MAX_DEVICES) return fail(s, JXS_EINVAL, "device index out of range");
  double* scratch = g_mse_noalloc_ptr[s->dev];
  if (!scratch) {  // set-up, once per device: the device address of the symbol on the CURRENT device (= s->dev, checked above)
    const cudaError_t e = cudaGetSymbolAddress((void**)&scratch, g_mse_noalloc_scratch);
    if (e != cudaSuccess || !scratch) return fail(s, JXS_ECUDA, cudaGetErrorString(e));
    g_mse_noalloc_ptr[s->dev] = scratch;
  }
  // same launches as jxs_mse_tangent: every partial sum that the second launch reads is written by the first one, so
  // nothing in the array has to start at zero and the contents the last call left behind are never read
  const int parts = (int)std::min<long long>(MSE_PARTS, (n + MSE_TB - 1) / MSE_TB);
  mse_partial_kernel<<<parts, MSE_TB, 0, s->stream>>>((const double*)U, (const double*)Udot, (const double*)Utarget, n, scratch);
  mse_final_kernel<<<1, MSE_TB, 0, s->stream>>>(scratch, parts, 1.0 / (double)n, out_dev);
  s->launches += 2;
  if (const cudaError_t e = cudaGetLastError(); e != cudaSuccess) return fail(s, JXS_ECUDA, cudaGetErrorString(e));
  return JXS_OK;
}

int jxs_step_host(jxs_solver* s, void* U, double cfl, int nsteps) { return step_common(s, U, cfl, 0.0, nsteps, true); }
int jxs_step_async(jxs_solver* s, void* U, double cfl, int nsteps) { return step_common(s, U, cfl, 0.0, nsteps, false, false); }
int jxs_wait(jxs_solver* s) {
  if (!s) return JXS_EINVAL;
  const int n = s->pending_steps;
  s->pending_steps = 0;
  return finish_steps(s, n);
}
int jxs_set_concurrent_handles(jxs_solver* s, int n) {
  if (!s) return JXS_EINVAL;
  if (n < 1) return fail(s, JXS_EINVAL, "n must be >= 1");
  drop_graph(s);
  s->share = n;
  choose_decomposition(s);  // the padded layout depends on the strips only, not on the row segments
  return JXS_OK;
}
int jxs_set_rows_per_segment(jxs_solver* s, int rows) {
  if (!s) return JXS_EINVAL;
  if (rows < 0) return fail(s, JXS_EINVAL, "rows must be >= 0");
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  drop_graph(s);
  s->rows_fixed = rows;
  choose_decomposition(s);
  return JXS_OK;
}
int jxs_set_graph_replay(jxs_solver* s, int on) {
  if (!s) return JXS_EINVAL;
  s->use_graph = on != 0;
  if (!s->use_graph) drop_graph(s);
  return JXS_OK;
}
int jxs_tune(jxs_solver* s) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  if (s->tuned) return JXS_OK;
  drop_graph(s);
  return tune_decomposition(s);
}
// ---- y-slab sharding: the pieces a multi-rank driver composes (paper_2601_04400_b200/sharded.py)
int jxs_set_active_rows(jxs_solver* s, int j_lo, int j_hi) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (s->nb > 1 || s->ny == 1) return fail(s, JXS_EINVAL, "active rows: single two-dimensional handles only");
  if (j_lo < 0 || j_hi > s->ny || j_lo >= j_hi) return fail(s, JXS_EINVAL, "bad row range");
  if (s->n_ghost > 0 || !s->fluid_host.empty()) return fail(s, JXS_ESTATE, "set the active rows before jxs_set_ibm");
  drop_graph(s);
  CU(cudaStreamSynchronize(s->stream));
  s->act_lo = j_lo; s->act_hi = j_hi;
  s->act_set = !(j_lo == 0 && j_hi == s->ny);
  if (!s->act_set) { cudaFree(s->d_fluid); s->d_fluid = nullptr; return JXS_OK; }
  return apply_active_rows(s);
}
static int shard_checks(jxs_solver* s) {
  if (s->nb > 1 || s->ny == 1) return fail(s, JXS_EINVAL, "sharded stepping: single two-dimensional handles only");
  if (s->scheme != JXS_SSPRK3) return fail(s, JXS_ESTATE, "sharded stepping is SSP-RK3");
  if (s->cnn_on) return fail(s, JXS_ESTATE, "no CNN flux in sharded stepping (its receptive field needs a deeper exchange)");
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  return JXS_OK;
}
int jxs_shard_begin(jxs_solver* s, const void* U) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U) return fail(s, JXS_EINVAL, "U is NULL");
  int rc = shard_checks(s);
  if (rc != JXS_OK) return rc;
  CU(pad(s, U, s->buf[0]));
  s->shard_cur = 0;
  CU(wavespeed(s, s->buf[0], &s->d_state->smax_bits[0]));
  s->shard_open = true;
  return JXS_OK;
}
int jxs_shard_smax(jxs_solver* s, double* d_smax, int set) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!d_smax) return fail(s, JXS_EINVAL, "d_smax is NULL");
  if (!s->shard_open) return fail(s, JXS_ESTATE, "jxs_shard_begin first");
  smax_copy_kernel<<<1, 1, 0, s->stream>>>(&s->d_state->smax_bits[s->shard_cur], d_smax, set);
  s->launches++;
  CU(cudaGetLastError());
  return JXS_OK;
}
int jxs_shard_step_begin(jxs_solver* s, double cfl, double fixed_dt) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!s->shard_open) return fail(s, JXS_ESTATE, "jxs_shard_begin first");
  if (!(fixed_dt > 0) && !(cfl > 0)) return fail(s, JXS_EINVAL, "cfl must be > 0");
  prepare_step_kernel<<<1, 64, 0, s->stream>>>(s->d_state, s->shard_cur, cfl * std::min(s->dx, s->dy), fixed_dt > 0 ? fixed_dt : 0.0, 1);
  s->launches++;
  CU(cudaGetLastError());
  return JXS_OK;
}
int jxs_shard_stage(jxs_solver* s, int k) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!s->shard_open) return fail(s, JXS_ESTATE, "jxs_shard_begin first");
  if (k < 0 || k > 2) return fail(s, JXS_EINVAL, "stage index 0..2");
  static const double ab[3][2] = {{0.0, 1.0}, {0.75, 0.25}, {1.0 / 3.0, 2.0 / 3.0}};
  const int in = k, out = (k + 1) % 3;
  CU(ghost_fill(s, s->buf[in]));
  CU(flux_mlp(s, s->buf[in]));
  unsigned long long* next = k == 2 ? &s->d_state->smax_bits[s->shard_cur ^ 1] : nullptr;
  CU(stage(s, s->buf[in], k == 0 ? nullptr : s->buf[0], s->buf[out], 0, ab[k][0], ab[k][1], next));
  if (k == 2) s->shard_cur ^= 1;
  return JXS_OK;
}
int jxs_shard_rows(jxs_solver* s, int k, int row0, int nrows, void* rows, int unpack) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!s->shard_open) return fail(s, JXS_ESTATE, "jxs_shard_begin first");
  if (!rows || k < 0 || k > 2 || nrows < 1 || row0 < 0 || row0 + nrows > s->ny) return fail(s, JXS_EINVAL, "bad rows");
  const int bs = 256, gs = std::max(1, std::min(s->num_sms * 4, (int)((4LL * s->nx * nrows + bs - 1) / bs)));
  if (s->dtype == JXS_F64) rows_copy_kernel<double><<<gs, bs, 0, s->stream>>>((double*)s->buf[k], (double*)rows, dims(s), row0, nrows, unpack);
  else rows_copy_kernel<float><<<gs, bs, 0, s->stream>>>((float*)s->buf[k], (float*)rows, dims(s), row0, nrows, unpack);
  s->launches++;
  CU(cudaGetLastError());
  return JXS_OK;
}
int jxs_shard_end(jxs_solver* s, void* U, int nsteps) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U) return fail(s, JXS_EINVAL, "U is NULL");
  if (!s->shard_open) return fail(s, JXS_ESTATE, "jxs_shard_begin first");
  s->shard_open = false;
  CU(unpad(s, s->buf[0], U));
  return finish_steps(s, nsteps);
}

int jxs_set_time_integrator(jxs_solver* s, int scheme) {
  if (!s) return JXS_EINVAL;
  drop_graph(s);
  if (scheme != JXS_SSPRK3 && scheme != JXS_EULER) return fail(s, JXS_EINVAL, "unknown time integrator");
  if (s->pending_steps) return fail(s, JXS_ESTATE, "jxs_wait first");
  s->scheme = scheme;
  return JXS_OK;
}

int jxs_get_time(const jxs_solver* s, double* t, double* last_dt) {
  if (!s) return JXS_EINVAL;
  if (t) *t = s->t;
  if (last_dt) *last_dt = s->last_dt;
  return JXS_OK;
}

int jxs_get_time_batch(const jxs_solver* s, double* t, double* last_dt) {
  if (!s) return JXS_EINVAL;
  for (int m = 0; m < s->nb; ++m) {
    if (t) t[m] = s->t_b[m];
    if (last_dt) last_dt[m] = s->dt_b[m];
  }
  return JXS_OK;
}
int jxs_batch_size(const jxs_solver* s) { return s ? s->nb : -1; }

long long jxs_launch_count(const jxs_solver* s) { return s ? s->launches : -1; }

int jxs_set_profiling(jxs_solver* s, int on) {
  if (!s) return JXS_EINVAL;
  s->profiling = on != 0;
  if (s->profiling && s->events.empty()) {
    s->events.resize(MAX_EVENTS);
    for (cudaEvent_t& ev : s->events) CU(cudaEventCreate(&ev));
    s->mlp_events.resize(MAX_EVENTS);
    for (cudaEvent_t& ev : s->mlp_events) CU(cudaEventCreate(&ev));
  }
  return JXS_OK;
}

int jxs_stage_time(const jxs_solver* s, double* ms_total, long long* launches) {
  if (!s) return JXS_EINVAL;
  if (ms_total) *ms_total = s->stage_ms;
  if (launches) *launches = s->stage_launches;
  return JXS_OK;
}

int jxs_ibm_ghost_count(const jxs_solver* s) { return s ? s->n_ghost : -1; }

int jxs_flux_mlp_time(const jxs_solver* s, double* ms_total, long long* launches) {
  if (!s) return JXS_EINVAL;
  if (ms_total) *ms_total = s->mlp_ms;
  if (launches) *launches = s->mlp_launches;
  return JXS_OK;
}

int jxs_flux_correction(jxs_solver* s, const void* U, float* dFx, float* dGy) {
  if (!s) return JXS_EINVAL;
  DEV(s);
  if (!U || !dFx || !dGy) return fail(s, JXS_EINVAL, "NULL array");
  if (!s->mlp_on && !s->cnn_on) return fail(s, JXS_ESTATE, "no flux network set (jxs_set_flux_mlp / jxs_set_flux_cnn)");
  if (s->nb > 1) return fail(s, JXS_EINVAL, "jxs_flux_correction inspects single handles");
  CU(pad(s, U, s->buf[0]));
  CU(ghost_fill(s, s->buf[0]));
  CU(flux_mlp(s, s->buf[0]));
  const int bs = 256, gs = s->num_sms * 8;
  gather_faces_kernel<<<gs, bs, 0, s->stream>>>(s->d_dFG, dFx, dGy, dims(s), s->out_scale[0], s->out_scale[1],
                                                 s->out_scale[2], s->out_scale[3]);
  s->launches++;
  CU(cudaGetLastError());
  return JXS_OK;
}

int jxs_measure_unit_rate(void* cuda_stream, int what, double ms, double* rate) {
  if (!rate || !(ms > 0) || what < 0 || what > 2) return JXS_EINVAL;
  int ndev = 0, dev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return JXS_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return JXS_ECUDA;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  double* d_out = nullptr;
  if (cudaMalloc(&d_out, 17 * sizeof(double)) != cudaSuccess) return JXS_ENOMEM;
  double seed[16];
  for (int k = 0; k < 16; ++k) seed[k] = k < 8 ? 1.0 + 1e-7 * (k + 1) : 1e-9 * (k - 7);
  cudaMemcpyAsync(d_out + 1, seed, sizeof(seed), cudaMemcpyHostToDevice, st);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int bs = 256, gs = prop.multiProcessorCount * 8;
  int iters = 2000;
  double best = 0;
  float el = 0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0, st);
    if (what == JXS_RATE_DFMA) dfma_peak_kernel<<<gs, bs, 0, st>>>(d_out, iters, 1.0000001, 1e-9);
    else if (what == JXS_RATE_DFMA3) dfma3_peak_kernel<<<gs, bs, 0, st>>>(d_out, iters, d_out + 1);
    else tanh_peak_kernel<<<gs, bs, 0, st>>>(d_out, iters);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    cudaEventElapsedTime(&el, e0, e1);
    // 64 operations per thread and trip; an FMA counts as 2 flop, a tanh as 1
    const double ops = (double)gs * bs * (double)iters * 64.0 * (what == JXS_RATE_TANH ? 1.0 : 2.0);
    if (rep > 0) best = std::max(best, ops / (el * 1e-3) / 1e12);
    if (el < ms) iters = (int)std::min(2.0e6, iters * std::max(1.5, ms / std::max(el, 1e-3f)));
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d_out);
  if (cudaGetLastError() != cudaSuccess) return JXS_ECUDA;
  *rate = best;
  return JXS_OK;
}

int jxs_measure_fp64_peak(void* cuda_stream, double ms, double* tflops) {
  return jxs_measure_unit_rate(cuda_stream, JXS_RATE_DFMA, ms, tflops);
}

}  // extern "C"
