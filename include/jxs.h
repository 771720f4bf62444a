/* jxs.h — C ABI of the B200-native (sm_100a) Runge-Kutta-stage library.
 *
 * One SSP-RK3 stage of the 2D compressible Euler / Navier-Stokes right-hand side
 * on a uniform Cartesian grid, as described in JAX-Shock (arXiv 2601.04400):
 *   ghost-frame and immersed-boundary ghost-cell fill,
 *   WENO5 reconstruction of primitive left/right face states (L46, L56),
 *   HLLC flux in x and y (L54-81, Eq. 3-9), flux divergence + viscous terms
 *   (L9, L83-85 Eq. 10), Runge-Kutta combine and CFL wavespeed reduction
 *   (BASELINE.json north_star), optional per-face MLP flux correction (L96 Eq. 11).
 * Widened since: the paper's 2D CNN flux (L94, Eq. 11-13), the forward-Euler update of Eq. 10,
 * one-dimensional problems (ny = 1: the Sod tube of L132-149) with their per-face MLP flux (L109), and for those
 * the derivatives the paper obtains from JAX (L92, L112-128, L149): the tangent of the step, its adjoint with the
 * trajectory kept in HBM, the loss of Eq. 14 and the gradient with respect to gamma and to the network's weights.
 * Where the paper is silent or garbled the readings R1-R24 of DESIGN.md apply.
 *
 * Conventions
 *   - every function returns an int status (JXS_OK = 0); nothing throws, aborts or prints;
 *     jxs_last_error() gives the detail of the last failure on a handle.
 *   - the handle is opaque and owns every internal buffer (padded RK buffers, IBM lists,
 *     MLP weights, device scalars).  The caller owns every array it passes; the library
 *     never frees or keeps them past the call.
 *   - field arrays are DEVICE pointers unless the function name ends in _host:
 *     SoA [4][ny][nx], x fastest, component order (rho, rho*u, rho*v, E), interior cells
 *     only, element type = the handle's dtype (JXS_F64 -> double, JXS_F32 -> float),
 *     16-byte aligned.
 *   - all device work is enqueued on the stream given to jxs_create (0 = default stream).
 *     Functions returning a host scalar synchronise that stream; jxs_rhs does not;
 *     jxs_step* synchronise once at the end to read the non-finite flag.
 *   - there is no CPU fallback: without a CUDA device jxs_create fails with JXS_ECUDA (also on a device that is
 *     not compute capability 10.0: the library holds sm_100a code only).  A handle belongs to the device that was
 *     current at jxs_create; calls made with another device current return JXS_ESTATE.
 */
#ifndef JXS_H
#define JXS_H
#ifdef __cplusplus
extern "C" {
#endif

enum {
  JXS_OK = 0,
  JXS_EINVAL = 1,   /* bad argument (see each function)                         */
  JXS_ENOMEM = 2,   /* host or device allocation failed                          */
  JXS_ECUDA = 3,    /* CUDA runtime error (no device, launch failure, ...)       */
  JXS_ESTATE = 4,   /* call not valid in the handle's current state              */
  JXS_ENUMERIC = 5  /* non-finite wavespeed / state detected during stepping     */
};
enum { JXS_BC_PERIODIC = 0, JXS_BC_TRANSMISSIVE = 1, JXS_BC_REFLECTIVE = 2, JXS_BC_INFLOW = 3 };
enum { JXS_F64 = 0, JXS_F32 = 1 };
enum { JXS_SSPRK3 = 0, JXS_EULER = 1 };

typedef struct jxs_solver jxs_solver;

/* Domain boundary conditions (inflow = left state, outflow, reflective walls;
 * transmissive for Sod, periodic for the vortex: BASELINE.json configs).  Three ghost layers
 * per side; x sides first, then y sides over the x-extended range (R11).                  */
typedef struct {
  int xlo, xhi, ylo, yhi; /* JXS_BC_*; PERIODIC must be set on both sides of an axis   */
  double inflow[4];       /* primitive (rho,u,v,p) imposed on JXS_BC_INFLOW sides       */
} jxs_bc;

/* Create a solver for an nx x ny grid of spacing (dx,dy), ideal gas gamma (Eq. 2), constant
 * dynamic viscosity mu >= 0 (0 = Euler) and Prandtl number Pr (R7, R8).
 * cuda_stream: a cudaStream_t cast to void*, or NULL.
 * ny = 1 selects the one-dimensional path (the paper's Sod tube): fields are
 * [4][1][nx] (rho v is carried along), the y boundary conditions are ignored, dy still enters the
 * CFL step as min(dx,dy) (pass dy = dx); no immersed boundary, no CNN flux (the per-face MLP is available).
 * JXS_EINVAL: nx < 8, ny < 8 and != 1, dx/dy <= 0, gamma <= 1, mu < 0, Pr <= 0 with mu > 0,
 * bad bc or dtype, NULL pointers.  JXS_ECUDA: no usable device.  JXS_ENOMEM: allocation failed. */
int jxs_create(int nx, int ny, double dx, double dy, double gamma, double mu, double Pr,
               const jxs_bc* bc, int dtype, void* cuda_stream, jxs_solver** out);
/* A BATCH of nbatch independent simulations on grids of one size (BASELINE.json configs[4]: 16 shock-cylinder runs;
 * SURVEY.md section 8(f) rank 4), advanced by ONE launch per kernel and stage: the members are stacked along y in the
 * handle's padded buffers, each with its own ghost frame, immersed boundary, time step and clock.
 *   mu[nbatch]  dynamic viscosity of every member (all zero or all positive); bc[nbatch]: the same kinds on every
 *               member, the inflow states may differ; nx, ny >= 8 (no one-dimensional batches)
 * On a batch handle every field argument is [nbatch][4][ny][nx] (member-major), jxs_set_ibm takes [nbatch][ny][nx]
 * level sets, jxs_max_wavespeed writes nbatch values, jxs_step evaluates the CFL step per member (jxs_get_time_batch),
 * the flux MLP (one set of weights) serves all members.  Results are bitwise those of nbatch separate handles.
 * Not available on a batch (JXS_EINVAL): the CNN flux, the nu-term, the derivatives, jxs_flux_correction.          */
int jxs_create_batch(int nbatch, int nx, int ny, double dx, double dy, double gamma, const double* mu, double Pr,
                     const jxs_bc* bc, int dtype, void* cuda_stream, jxs_solver** out);
int jxs_batch_size(const jxs_solver*);
/* t_host[nbatch], last_dt_host[nbatch] (either may be NULL): every member's clock (a single handle: one value) */
int jxs_get_time_batch(const jxs_solver*, double* t_host, double* last_dt_host);
void jxs_destroy(jxs_solver*);
/* Never NULL; "" when there was no error.  Valid until the next call on the handle.        */
const char* jxs_last_error(const jxs_solver*);

/* Immersed boundary (R9, R10).  phi_host: HOST array [ny][nx], signed
 * distance, > 0 in the fluid; NULL removes the body.  Builds the cell classification and the
 * ghost-cell gather list on the host and uploads them.  JXS_EINVAL: a non-fluid cell closer
 * than 8 cells to a domain edge, zero gradient at a ghost cell, or a ghost cell left without
 * a fluid donor (the previous body, if any, is then removed).                              */
int jxs_set_ibm(jxs_solver*, const double* phi_host);

/* Per-face MLP flux correction (Eq. 11; BASELINE.json configs[4]; R14).  weights_host: HOST
 * array of 6020 floats, W1[64][24], b1[64], W2[64][64], b2[64], W3[4][64], b3[4] (row-major,
 * [out][in]); NULL disables.  in_scale[4] > 0 divides (rho, u_n, u_t, p); out_scale[4]
 * multiplies the four outputs (mass, normal, tangential momentum, energy).  The network is
 * evaluated in bf16 with fp32 accumulation on the tensor cores.                             */
int jxs_set_flux_mlp(jxs_solver*, const float* weights_host, const double in_scale[4],
                     const double out_scale[4]);

/* The corrections themselves (Eq. 11), for inspection and parity tests: Delta F = out_scale o y of
 * every face of U after the ghost fills, as fp32 DEVICE arrays dFx[4][ny][nx+1] (face f of row j lies
 * between cells f-1 and f) and dGy[4][ny+1][nx], components = corrections to the (rho, rho u, rho v, E)
 * fluxes.  JXS_ESTATE without a network.  Asynchronous.                                     */
int jxs_flux_correction(jxs_solver*, const void* U, float* dFx, float* dGy);
/* The paper's two-dimensional neural flux (Eq. 11-13): a fully
 * convolutional network, three 3x3 convolutions 4 -> 32 -> 16 -> 4 with ReLU, ReLU, tanh and zero padding (6388
 * parameters, R18), applied to the field of normalised face states of each direction with the same weights (R19)
 * and added, times out_scale, to the HLLC flux (R20).  weights_host: 6388 floats in OIHW order W1[32][4][3][3],
 * b1[32], W2[16][32][3][3], b2[16], W3[4][16][3][3], b3[4] (first tap index along the face's tangential direction,
 * second along its normal); in_scale of (rho, rho u_n, rho u_t, E) > 0; out_scale of the (mass, normal momentum,
 * tangential momentum, energy) flux.  Evaluated in bf16 with fp32 accumulation on the tensor cores.  NULL weights
 * disable it.  JXS_ESTATE while the per-face MLP is set (one network at a time), JXS_EINVAL for ny = 1.
 * jxs_flux_correction returns its corrections; jxs_flux_cnn_inputs (inspection) returns the network's input
 * fields as floats, Xx[4][ny][nx+1] and Xy[4][nx][ny+1] (device pointers).                                   */
int jxs_set_flux_cnn(jxs_solver*, const float* weights_host, const double in_scale[4], const double out_scale[4]);
int jxs_flux_cnn_inputs(jxs_solver*, const void* U, float* Xx, float* Xy);

/* Change the specific-heat ratio of the handle (> 1, else JXS_EINVAL): the unknown of the paper's inference from
 * Sod data (Fig. 3b), so an optimisation loop keeps one handle.  Everything that depends on gamma is
 * evaluated at launch time; captured CUDA graphs and a recorded trajectory (jxs_step_fixed_dt_record) are dropped.
 * JXS_ESTATE with steps pending (jxs_wait).                                                   */
int jxs_set_gamma(jxs_solver*, double gamma);

/* Laplacian artificial viscosity nu * Lap_h(U) of PAPER.md Eq. 10; default 0 (R7).  Drops a recorded
 * trajectory.  JXS_EINVAL for nu < 0 or non-finite (nothing changes), JXS_ESTATE with steps pending. */
int jxs_set_artificial_viscosity(jxs_solver*, double nu);

/* dUdt = L(U): ghost fills on an internal copy of U, then the fused stage kernel with the
 * Runge-Kutta combine disabled.  dUdt is 0 at non-fluid cells.  Asynchronous.               */
int jxs_rhs(jxs_solver*, const void* U, void* dUdt);

/* smax = max over fluid interior cells of max(|u|+a, |v|+a) (R6).  Synchronises.            */
int jxs_max_wavespeed(jxs_solver*, const void* U, double* smax_host);

/* Advance U in place by nsteps SSP-RK3 steps (R5), dt = cfl*min(dx,dy)/smax evaluated on the
 * device at the start of every step (R6).  JXS_ENUMERIC if a non-finite or non-positive
 * wavespeed was met (U then holds the last state computed).  Synchronises once at the end.
 * For nsteps >= 6 (and jxs_set_profiling off) pairs of steps are replayed from a CUDA graph
 * captured on a private stream; results are identical to plain launches (jxs_set_graph_replay(h, 0) turns
 * the replay off).  The first synchronous stepping call of a handle on a large grid also times about forty
 * stage launches to choose the length of the row segments the grid is cut into (jxs_tune, below; it
 * synchronises the stream once; results do not depend on it).                                        */
int jxs_step(jxs_solver*, void* U, double cfl, int nsteps);
/* Same with a fixed time step.                                                              */
int jxs_step_fixed_dt(jxs_solver*, void* U, double dt, int nsteps);
/* Tangent (forward-mode derivative) of jxs_step_fixed_dt, in one and in two dimensions: PAPER.md Eq. 15-16 (the step
 * U^{n+k} = S(U^{n+k-1}, theta) and the chain of its Jacobians) applied to ONE direction of perturbation, for the
 * paper's inference of the specific-heat ratio from Sod data (L149, Fig. 3b; R21).
 * In 2D (ny > 1; Fig. 5d-f; R25) the boundary conditions and the immersed-boundary fill are
 * differentiated with the scheme (deriv2d_kernels.cuh); the 2D networks are not (JXS_ESTATE).
 *   U, Udot   DEVICE pointers, [4][ny][nx] doubles, read and overwritten: the state and a direction of perturbation
 *             of it (owned by the caller; Udot = 0 differentiates with respect to gamma at fixed conserved state,
 *             Udot[3] = -p/(gamma-1)^2 at fixed primitives)
 *   gamma_dot perturbation of gamma along the same direction
 *   dt        step size, a constant of the differentiation (> 0); nsteps >= 0 steps of the handle's time integrator
 *             (SSP-RK3, or the forward-Euler update of Eq. 10 with its nu-term: the update the paper differentiates)
 * On return U = S^nsteps(U; gamma) (the same arithmetic as the tangent's value part, equal to jxs_step_fixed_dt to
 * round-off) and Udot = dS^nsteps/dU . Udot + dS^nsteps/dgamma . gamma_dot.  Branches of the scheme (min / max of wave
 * speeds, sign of the contact speed, positivity guard) carry the derivative of the branch taken.
 * Errors: JXS_EINVAL for NULL pointers, dt <= 0, nsteps < 0, a non-finite gamma_dot, an fp32 or a batch handle;
 * JXS_ESTATE with a network set or with steps pending (jxs_wait);
 * JXS_ENOMEM / JXS_ECUDA from the first call's allocation of the tangent buffers.  Synchronises the stream.      */
int jxs_step_fixed_dt_tangent(jxs_solver*, void* U, void* Udot, double gamma_dot, double dt, int nsteps);

/* The loss of PAPER.md Eq. 14 for one target and its derivative along a tangent (R22):
 *   *loss = mean((U - Utarget)^2),  *dloss = mean(2 (U - Utarget) Udot)   over the 4 nx ny entries.
 * U, Udot, Utarget: DEVICE pointers, [4][ny][nx] doubles, read only; loss, dloss: HOST doubles.  With Udot from
 * jxs_step_fixed_dt_tangent, *dloss = dL/dgamma.  The summation order is fixed (two launches), so the result is
 * reproducible.  Errors: JXS_EINVAL for NULL pointers or an fp32 handle.  Synchronises the stream.               */
int jxs_mse_tangent(jxs_solver*, const void* U, const void* Udot, const void* Utarget, double* loss, double* dloss);

/* jxs_mse_tangent for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same two launches in the same fixed summation order, hence the same bits, but
 *   - the partial sums go to a file-scope device array of the library (2 x 1024 doubles = 16 KB, held by every GPU
 *     that loads the library until exit) instead of a buffer the handle allocates on first use;
 *   - the result goes to out_dev, a DEVICE array of 2 doubles the caller owns: out_dev[0] = mean((U - Utarget)^2),
 *     out_dev[1] = mean(2 (U - Utarget) Udot); nothing is copied to the host and the stream is NOT synchronised:
 *     the call only enqueues two kernels on the handle's stream.
 * It calls no cudaMalloc / cudaFree and no allocating library routine.  The first call on a device looks up the
 * array's device address (cudaGetSymbolAddress, no allocation): make one call before starting a graph capture.
 * U, Udot, Utarget: DEVICE pointers, [4][ny][nx] doubles, read only (as for jxs_mse_tangent).
 * Limit: 4 nx ny <= JXS_MSE_NOALLOC_MAX_N = 2^26 entries (twice the 4 x 4096 x 2048 of the largest BASELINE
 * configuration: the size the array is stated and tested for); beyond it JXS_EINVAL with a message naming the limit.
 * ALL calls on a device share the one array, which keeps the last call's partial sums (every value a call reads it
 * has written itself, so nothing needs clearing): calls that overlap on the GPU (different streams, or graph
 * launches running concurrently) race on it and return garbage - order them.
 * Errors: JXS_EINVAL (NULL pointers, fp32 handle, size beyond the limit), JXS_ESTATE (wrong current device),
 * JXS_ECUDA.                                                                                                       */
#define JXS_MSE_NOALLOC_MAX_N (1LL << 26)
int jxs_mse_tangent_noalloc(jxs_solver*, const void* U, const void* Udot, const void* Utarget, double* out_dev);

/* Reverse mode (adjoint) of jxs_step_fixed_dt, in one and in two dimensions (Euler or Navier-Stokes, nu-term; in 2D with the
 * immersed boundary and the frame's corners, R25): Eq. 15-16 —
 * "backpropagation through the full sequence of unrolled solver steps" (R21, R24).
 * Two calls: the forward sweep that records the trajectory, then the reverse sweep.
 *
 * jxs_step_fixed_dt_record: as jxs_step_fixed_dt (U: DEVICE pointer, [4][ny][nx] doubles, advanced in place by nsteps
 * >= 1 steps of size dt > 0 of the handle's time integrator), keeping the stage states of every step (3 for SSP-RK3, 1
 * for forward Euler) in device memory owned by the handle (32 nx bytes per state in 1D, a padded buffer of
 * 32 (nx+6..) (ny+6) bytes in 2D).
 * jxs_adjoint_steps: Ubar (DEVICE pointer, [4][ny][nx] doubles) holds on entry the adjoint of the final state, e.g.
 * dL/dU^{n+m} of the loss of Eq. 14; on return the adjoint of the initial state, (dU^{n+m}/dU^n)^T Ubar.
 * *gamma_bar (HOST) = <dU^{n+m}/dgamma at fixed initial conserved state, Ubar>.  For every direction (Udot, gamma_dot),
 * with Udot_end from jxs_step_fixed_dt_tangent: <Ubar on entry, Udot_end> = <Ubar on return, Udot> + gamma_bar gamma_dot.
 * May be called repeatedly on one recording.  Branches of the scheme carry the derivative of the branch taken.
 * Errors: JXS_EINVAL for NULL pointers, dt <= 0, nsteps < 1, an fp32 or a batch handle; JXS_ESTATE with a 2D network, steps
 * pending, or (adjoint) nothing recorded (changing gamma, nu or the network drops a recording); JXS_ENOMEM when the
 * trajectory does not fit.  With the per-face MLP set on the handle (see jxs_flux_mlp_gradient below) both calls include it.  The recording stays (and its memory is reused by the next record call) until jxs_destroy.  Both
 * synchronise the stream.                                                                                         */
int jxs_step_fixed_dt_record(jxs_solver*, void* U, double dt, int nsteps);
int jxs_adjoint_steps(jxs_solver*, void* Ubar, double* gamma_bar);
/* The reverse sweep driven by the loss of PAPER.md Eq. 14 itself, the mean over the m recorded steps of the mean
 * squared error against one target per step (R22):  L = (1/m) sum_{s=1..m} mean((U^{n+s} - targets[s-1])^2).
 *   targets  DEVICE, [m][4][ny][nx] doubles, m = the nsteps of the last jxs_step_fixed_dt_record: the downsampled
 *            reference states U~^{n+s} (read only)
 *   Ubar     DEVICE, [4][ny][nx] doubles, OUT: dL/dU^n
 *   loss, gamma_bar  HOST, OUT: L and dL/dgamma at fixed U^n; the weights' gradient dL/dtheta is read with
 *            jxs_flux_mlp_gradient
 * Every intermediate loss L_s enters the sweep where its state does (Eq. 16 summed over s), so the cost is that of
 * one jxs_adjoint_steps.  Errors as jxs_adjoint_steps, JXS_EINVAL for NULL.  Synchronises the stream.            */
int jxs_adjoint_steps_mse(jxs_solver*, const void* targets, void* Ubar, double* loss, double* gamma_bar);

/* One-dimensional handles accept jxs_set_flux_mlp as well ("For the one-dimensional Sod shock-tube
 * simulation, a multilayer perceptron (MLP) network is used to predict the neural flux"): same parameters, input
 * and output conventions as in 2D (R14), evaluated per face in fp64 and added to the HLLC flux of every stage (Eq. 11)
 * by all the stepping calls, jxs_rhs and jxs_step_fixed_dt_record.  jxs_adjoint_steps then also differentiates
 * through the network — its input's dependence on the state and on gamma enters Ubar and *gamma_bar — and accumulates
 * the weights' gradient (Eq. 16), which jxs_flux_mlp_gradient copies out:
 *   grad  HOST, 6020 doubles in the order of the weights: d<Ubar on entry, U^{n+m}>/d(theta) of the last
 *         jxs_adjoint_steps call (zero before any).  Sums over faces use fp64 atomics: reproducible to round-off.
 * JXS_ESTATE without a flux MLP on a one-dimensional handle, JXS_EINVAL for NULL.  The forward-mode tangent does not
 * cover the network (JXS_ESTATE).                                                                                  */
int jxs_flux_mlp_gradient(jxs_solver*, double* grad);

/* Checkpointing of the recording (default off): with on != 0 an SSP-RK3 recording keeps only U^n of every step (32 nx
 * bytes per step instead of 96) and jxs_adjoint_steps recomputes the two inner stage states of a step before it
 * reverses them: one third of the memory for two more stage launches per step, bit-identical results.  Applies to
 * recordings made after the call.                                                                                 */
int jxs_set_adjoint_checkpointing(jxs_solver*, int on);

/* Same two calls on HOST buffers (pageable or pinned): host->device copy, stepping,
 * device->host copy; used for end-to-end timing.                                            */
int jxs_step_host(jxs_solver*, void* U_host, double cfl, int nsteps);
int jxs_rhs_host(jxs_solver*, const void* U_host, void* dUdt_host);
/* jxs_step without the final synchronisation: only enqueues on the handle's stream, so that several handles
 * (BASELINE.json configs[4]: 16 independent simulations, one stream each) run concurrently.  jxs_wait
 * synchronises the stream, updates jxs_get_time and returns JXS_ENUMERIC like jxs_step would have.
 * U must stay valid until jxs_wait returns.                                                  */
int jxs_step_async(jxs_solver*, void* U, double cfl, int nsteps);
int jxs_wait(jxs_solver*);
/* The work decomposition of the fused stage kernel: the grid is cut into column strips and
 * each strip into row segments of `rows` rows, one task each.  Results never depend on it.
 *   jxs_tune                  times one stage launch per candidate segment length around the heuristic's choice on the
 *                             handle's own buffers (about forty launches, one stream synchronisation) and keeps the best;
 *                             jxs_step / jxs_step_fixed_dt / jxs_step_host do this themselves on their first call,
 *                             jxs_step_async never does (it only enqueues): call jxs_tune once before an async loop.
 *                             JXS_ESTATE with steps pending.
 *   jxs_set_rows_per_segment  rows > 0 fixes the segment length (no measurement); 0 returns to the heuristic + jxs_tune.
 *   jxs_set_graph_replay      on = 0: plain launches instead of the replayed two-step CUDA graph (default on).   */
int jxs_tune(jxs_solver*);
int jxs_set_rows_per_segment(jxs_solver*, int rows);
int jxs_set_graph_replay(jxs_solver*, int on);
/* Performance hint for such ensembles: n handles of about this size step concurrently, so this handle sizes
 * its tasks for 1/n of the GPU (longer row segments, fewer warm-up rows) instead of trying to fill it alone.
 * Results do not change.  Default 1.                                                           */
int jxs_set_concurrent_handles(jxs_solver*, int n);
/* y-slab sharding of ONE simulation over several GPUs: the pieces a multi-rank
 * driver composes — paper_2601_04400_b200/sharded.py does, with torch.distributed (NCCL) carrying the rows.  Every
 * rank runs an ordinary handle on its slab extended by 12 overlap rows per cut side.
 *   jxs_set_active_rows   rows outside [j_lo, j_hi) are the overlap: L = 0 there, they do not enter s_max, and an
 *                         immersed body may cross the slab edge behind them (the 8-cell edge rule applies to the
 *                         domain's real edges only).  Call before jxs_set_ibm (JXS_ESTATE otherwise).
 *   jxs_shard_begin       U (DEVICE, [4][ny][nx]) -> the handle's buffers; local s_max of the active rows
 *   jxs_shard_smax        set = 0: *d_smax (DEVICE double) <- the current local s_max; set = 1: the handle's s_max <-
 *                         *d_smax (after the MAX all-reduce over the ranks)
 *   jxs_shard_step_begin  dt = cfl min(dx,dy) / s_max (or fixed_dt > 0), clock advanced
 *   jxs_shard_rows        rows [row0, row0 + nrows) of the INPUT buffer of stage k (0..2) -> rows (DEVICE, contiguous
 *                         [4][nrows][nx]) (unpack = 0), or back (unpack = 1): the halo pack / unpack kernels
 *   jxs_shard_stage       ghost fills + [flux MLP] + the fused stage kernel of SSP-RK3 stage k
 *   jxs_shard_end         the result -> U; synchronises, returns JXS_ENUMERIC like jxs_step
 * All asynchronous on the handle's stream except jxs_shard_end.  JXS_EINVAL on batch or one-dimensional handles,
 * JXS_ESTATE out of order, with forward Euler, or with the CNN flux.                                              */
int jxs_set_active_rows(jxs_solver*, int j_lo, int j_hi);
int jxs_shard_begin(jxs_solver*, const void* U);
int jxs_shard_smax(jxs_solver*, double* d_smax, int set);
int jxs_shard_step_begin(jxs_solver*, double cfl, double fixed_dt);
int jxs_shard_rows(jxs_solver*, int k, int row0, int nrows, void* rows, int unpack);
int jxs_shard_stage(jxs_solver*, int k);
int jxs_shard_end(jxs_solver*, void* U, int nsteps);

/* Time integrator of jxs_step*: JXS_SSPRK3 (default, R5) or JXS_EULER, the forward-Euler update the paper
 * prints (Eq. 10; with jxs_set_artificial_viscosity it is Eq. 10 term by term) = one stage
 * with (a,b) = (0,1).  SURVEY.md section 8(f) rank 2.                                           */
int jxs_set_time_integrator(jxs_solver*, int scheme);

/* Simulated time since creation and the last time step taken.                               */
int jxs_get_time(const jxs_solver*, double* t_host, double* last_dt_host);

/* Number of kernel launches enqueued by this handle since creation (bench.py reports it).   */
long long jxs_launch_count(const jxs_solver*);
/* Device time (ms) of the stage kernels of the last jxs_step* call, measured with CUDA events
 * on the handle's stream, and how many stage launches that was.  Only recorded when
 * jxs_set_profiling(h, 1) is on (it adds two event records per stage launch).               */
int jxs_set_profiling(jxs_solver*, int on);
int jxs_stage_time(const jxs_solver*, double* ms_total, long long* launches);
/* Same for the flux-MLP kernel (S5').                                                        */
int jxs_flux_mlp_time(const jxs_solver*, double* ms_total, long long* launches);
/* Number of IBM ghost cells (0 without a body).                                             */
int jxs_ibm_ghost_count(const jxs_solver*);
/* Sustained FP64 FMA rate of the device, in TFLOP/s (2 flops per FMA), from a register-
 * resident DFMA loop run for about `ms` milliseconds: the ALU-roofline denominator.         */
int jxs_measure_fp64_peak(void* cuda_stream, double ms, double* tflops);
/* Sustained rate of one execution unit of the current device, from a register-resident loop run for about `ms`
 * milliseconds on `cuda_stream` (synchronous): the measured denominators of the "alu"-bound rooflines.
 *   JXS_RATE_DFMA   FP64 FMAs of the form x = x * a + b (two register operands), TFLOP/s at 2 flop per FMA: what
 *                   jxs_measure_fp64_peak returns; 64 per clock and SM;
 *   JXS_RATE_DFMA3  FP64 FMAs with three distinct vector-register operands (x = p * q + x), TFLOP/s: the register
 *                   file delivers two 64-bit operands per issue slot of the FP64 pipe, so these take 3 cycles
 *                   instead of 2 (measured 24.8 against 37.2 TFLOP/s); constants and uniform values do not count;
 *   JXS_RATE_TANH   MUFU.TANH (tanh.approx.f32), in 10^12 results per second: 16 per clock and SM.
 * Errors: JXS_EINVAL (rate NULL, ms <= 0, unknown `what`), JXS_ENOMEM, JXS_ECUDA.                              */
#define JXS_RATE_DFMA 0
#define JXS_RATE_DFMA3 1
#define JXS_RATE_TANH 2
int jxs_measure_unit_rate(void* cuda_stream, int what, double ms, double* rate);

#ifdef __cplusplus
}
#endif
#endif
