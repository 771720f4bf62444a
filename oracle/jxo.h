/* jxo.h — C ABI of the CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded reference implementation of one Runge-Kutta
 * stage of the 2D compressible Euler / Navier-Stokes right-hand side described
 * in JAX-Shock (arXiv 2601.04400; PAPER.md) with the readings listed in
 * DESIGN.md ("Readings of the paper").  It shares no code with the CUDA
 * library in paper_2601_04400_b200/csrc and must only be used by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * All arrays are HOST pointers, SoA [4][ny][nx], x fastest, component order
 * (rho, rho*u, rho*v, E), interior cells only, element type = the handle's
 * dtype (JXO_F64 -> double, JXO_F32 -> float).
 */
#ifndef JXO_H
#define JXO_H
#ifdef __cplusplus
extern "C" {
#endif

enum { JXO_OK = 0, JXO_EINVAL = 1, JXO_ENOMEM = 2, JXO_ESTATE = 4, JXO_ENUMERIC = 5 };
enum { JXO_BC_PERIODIC = 0, JXO_BC_TRANSMISSIVE = 1, JXO_BC_REFLECTIVE = 2, JXO_BC_INFLOW = 3 };
enum { JXO_F64 = 0, JXO_F32 = 1 };

typedef struct jxo_solver jxo_solver;
typedef struct {
  int xlo, xhi, ylo, yhi; /* JXO_BC_* per side                         */
  double inflow[4];       /* (rho,u,v,p) used by JXO_BC_INFLOW sides   */
} jxo_bc;

int jxo_create(int nx, int ny, double dx, double dy, double gamma, double mu, double Pr,
               const jxo_bc* bc, int dtype, jxo_solver** out);
void jxo_destroy(jxo_solver*);
const char* jxo_last_error(const jxo_solver*);

/* phi_host [ny][nx], signed distance, > 0 in the fluid; NULL removes the body. */
int jxo_set_ibm(jxo_solver*, const double* phi_host);
/* weights: W1[64][24], b1[64], W2[64][64], b2[64], W3[4][64], b3[4] (6020 floats);
 * NULL disables.  emulate_bf16 != 0 rounds weights, inputs and hidden
 * activations to bf16 (round-to-nearest-even) and accumulates in double.      */
int jxo_set_flux_mlp(jxo_solver*, const float* weights, const double in_scale[4],
                     const double out_scale[4], int emulate_bf16);
/* O11: the paper's 2D CNN neural flux (Eq. 11-13): weights in OIHW order W1[32][4][3][3], b1[32],
 * W2[16][32][3][3], b2[16], W3[4][16][3][3], b3[4] = 6388 floats; in_scale of (rho, rho u_n, rho u_t, E), out_scale
 * of the (mass, normal, tangential momentum, energy) flux.  NULL disables.  emulate_bf16 != 0 rounds weights, inputs
 * and the two hidden activation fields to bf16.  Can be combined with the per-face MLP (both are added).          */
int jxo_set_flux_cnn(jxo_solver*, const float* weights, const double in_scale[4],
                     const double out_scale[4], int emulate_bf16);
/* O12 through the exact (emulate_bf16 = 0) MLP: direction of perturbation of its 6020 parameters, doubles in the
 * order of the weights; NULL = the parameters do not move (default; jxo_set_flux_mlp resets it).                */
int jxo_set_flux_mlp_direction(jxo_solver*, const double* direction);
int jxo_set_artificial_viscosity(jxo_solver*, double nu);

int jxo_rhs(jxo_solver*, const void* U, void* dUdt);
int jxo_max_wavespeed(jxo_solver*, const void* U, double* smax);
int jxo_step(jxo_solver*, void* U, double cfl, int nsteps);
int jxo_step_fixed_dt(jxo_solver*, void* U, double dt, int nsteps);
int jxo_get_time(const jxo_solver*, double* t, double* last_dt);
/* O12: the tangent (forward-mode derivative) of jxo_step_fixed_dt: the Jacobian products of PAPER.md Eq. 16 applied
 * to one direction.  U, Udot: [4][ny][nx] doubles, in and out.  On return U = S^n(U; gamma) and
 * Udot = dS^n/dU . Udot + dS^n/dgamma . gamma_dot.  fp64 handles without a network (EINVAL / ESTATE).
 * With a loss L(U) (Eq. 14) this gives dL/dgamma = <dL/dU, Udot>: the paper's gamma inference (L149, Fig. 3b). */
int jxo_step_fixed_dt_tangent(jxo_solver*, double* U, double* Udot, double gamma_dot, double dt, int nsteps);
/* L(U) and its tangent along (Udot, gamma_dot), [4][ny][nx] doubles each: for the forward-Euler update of Eq. 10,
 * which jxo.py writes out with it.                                                                            */
int jxo_rhs_tangent(jxo_solver*, const double* U, const double* Udot, double gamma_dot, double* L, double* Ldot);

/* ---- introspection used only by the oracle's own pins ------------------- */
/* one left-biased WENO5-JS value at i+1/2 from (v[i-2..i+2]) in double          */
double jxo_weno5(const double v[5]);
/* HLLC flux in x from primitive (rho,u,v,p) left/right states                   */
void jxo_hllc(const double WL[4], const double WR[4], double gamma, double F[4]);
/* wave speeds sL,sR,s* and the two star states (conserved) of the same solver   */
void jxo_hllc_star(const double WL[4], const double WR[4], double gamma,
                   double speeds[3], double UstarL[4], double UstarR[4]);
/* tangents of the two routines above: out = {value, derivative along vdot}; F, Fdot along (WLdot, WRdot, gamma_dot) */
void jxo_weno5_tangent(const double v[5], const double vdot[5], double out[2]);
void jxo_hllc_tangent(const double WL[4], const double WR[4], const double WLdot[4], const double WRdot[4],
                      double gamma, double gamma_dot, double F[4], double Fdot[4]);
/* fill domain frame + IBM ghosts of U (interior array is copied into a padded
 * array, filled, and the padded array [4][ny+6][nx+6] is returned in Upad)      */
int jxo_fill_ghosts(jxo_solver*, const void* U, void* Upad);
/* number of IBM ghost cells; arrays may be NULL. cell = j*nx+i; donors 4 per
 * ghost as j*nx+i; weights 4 per ghost; normal 2 per ghost                      */
int jxo_ibm_ghosts(const jxo_solver*, int* cell, int* donors, double* weights, double* normal);
/* cell type per interior cell: 0 fluid, 1 ghost, 2 solid                        */
int jxo_cell_types(const jxo_solver*, unsigned char* type);
/* activations of the positivity guard since creation                            */
long long jxo_guard_count(const jxo_solver*);
/* arithmetic tally of ONE rhs + one RK combine on the given field, evaluated
 * with a counting scalar: counts = {add/sub, mul, div, sqrt, min/max/abs/cmp}   */
int jxo_count_ops(jxo_solver*, const double* U, long long counts[5]);
/* the per-face MLP alone: x[24] (already normalised) -> y[4]                    */
int jxo_mlp_eval(const jxo_solver*, const double x[24], double y[4]);
/* the CNN alone on a normalised field in[4][na][nb] (a tangential, b normal) -> out[4][na][nb]   */
int jxo_cnn_apply(const jxo_solver*, const double* in, int na, int nb, double* out);
/* observers of one rhs evaluation (fp64 handles): the network's input fields Xx[4][ny][nx+1], Xy[4][nx][ny+1]
 * (R19) and its outputs before out_scale, same shapes                                              */
int jxo_cnn_fields(jxo_solver*, const double* U, double* Xx, double* Xy, double* Yx, double* Yy);

#ifdef __cplusplus
}
#endif
#endif
