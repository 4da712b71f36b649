/*
 * fs_oracle.h -- C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded fp64 implementation of one fractional step of the
 * incompressible Navier-Stokes finite-volume solver of Diff-FlowFSI (arxiv 2505.23940,
 * /root/reference/PAPER.md section 2.3: Eq. 3-10, 12, 20-22) written from the paper and from
 * SURVEY.md section 8(c) (steps O1..O9).  It shares no code, header, table or helper with
 * the CUDA path under paper_2505_23940_b200/csrc and must never be imported by the product.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
 *
 * Array conventions (all fp64, x fastest, then y, then z):
 *   p, div   : nz * ny * nx
 *   u        : nz * ny * (nx+bx)      bx = 1 when the x direction is bounded (non-periodic)
 *   v        : nz * (ny+by) * nx
 *   w        : (nz+bz) * ny * nx
 *   u(i,j,k) sits at (x_f(i), y_c(j), z_c(k)) etc. (staggered grid).
 */
#ifndef FS_ORACLE_H
#define FS_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_BC_PERIODIC = 0, ORC_BC_NOSLIP = 1, ORC_BC_SLIP = 2, ORC_BC_INFLOW = 3, ORC_BC_OUTFLOW = 4 };
enum { ORC_TIME_EULER = 0, ORC_TIME_AB2 = 1, ORC_TIME_RK3 = 2 };   /* Eq. 4 / configs / "explicit Runge-Kutta" (L100, L431) */
enum { ORC_PC_NONE = 0, ORC_PC_JACOBI = 1, ORC_PC_GMG = 2 };
enum { ORC_DELTA_ROMA3 = 0, ORC_DELTA_PESKIN4 = 1 };
enum { ORC_CONV_CENTRAL = 0, ORC_CONV_UPWIND = 1 };   /* 2nd-order central or 1st-order upwind convection */
enum { ORC_U = 0, ORC_V, ORC_W, ORC_P, ORC_HU, ORC_HV, ORC_HW, ORC_DIV };

typedef struct {
  int nx, ny, nz;
  double x0, y0, z0, lx, ly, lz;
  const double* yf;          /* ny+1 face coordinates or NULL (uniform) */
  int bc[6];                 /* -x,+x,-y,+y,-z,+z */
  double bc_vel[6][3];
  double nu, rho, dt, body_force[3];
  int time_scheme;
  int precond; double rtol; int max_iter; int warm_start;
  int mg_nu1, mg_nu2, mg_coarse_sweeps; double mg_omega;
  int delta;
  uint64_t seed; double inflow_noise;
  int convection;            /* ORC_CONV_* */
  double cs;                 /* constant Smagorinsky coefficient C_s (L437, L638); 0 = no subgrid model */
  int wall_model;            /* != 0: equilibrium wall model (Spalding law, Eq. 27-29) on no-slip y walls */
  int coupling_max_iters;    /* strong FSI coupling (Algorithm 1): at most this many sub-iterations per step; <= 1: weak */
  double coupling_tol;       /* stop when || (w^k - w^{k-1}) / w^{k-1} ||^2 < tol (paper: 1e-5) */
  double cfl;                /* > 0: CFL-adaptive step size, dt = min(dt, cfl h_min / |u|_max) (L431); <= 0: fixed dt */
} orc_params;

typedef struct {
  int pcg_iters, converged, nan_flag;
  double rel_residual, true_rel_residual, max_abs_div;
  double body_force[3], body_disp[3], body_vel[3];
  long long step;
  double dt, time;           /* step size used by the last step, elapsed time */
  int coupling_iters; double coupling_xi;   /* Algorithm 1: sub-iterations of the last step and its final xi */
} orc_info;

typedef struct orc_sim orc_sim;

orc_sim* orc_create(const orc_params* p);           /* NULL on invalid parameters */
void     orc_destroy(orc_sim*);
long long orc_field_size(orc_sim*, int field);
int  orc_set_field(orc_sim*, int field, const double* src);
int  orc_get_field(orc_sim*, int field, double* dst);
int  orc_set_markers(orc_sim*, int n, const double* xyz, const double* vel, const double* dvol);
int  orc_set_body(orc_sim*, double m, double c, double k, int dof_mask);
/* eps-mask IBM of the paper (Eq. 5, 8-9, 18-19, 23; reading E1): eps_cells nz*ny*nx bytes (1 = solid cell), uc[3] the exact
 * solid velocity u_c (NULL = 0).  Switches the IBM from marker forcing to mask forcing; markers, if set, then only carry
 * the structure velocity to the IB points (Eq. 18-19).  eps_cells == NULL switches back. */
int  orc_set_solid_mask(orc_sim*, const unsigned char* eps_cells, const double* uc);
void orc_get_face_masks(orc_sim*, unsigned char* mu, unsigned char* mv, unsigned char* mw);   /* 0 fluid, 1 solid, 2 IB point */
/* Flexible beam (Eq. 11, 13-17, Newmark-beta; reading N2-2): a straight Euler-Bernoulli beam of n_nodes nodes in the x-y
 * plane (node_xy: n_nodes * 2), clamped at node 0, two degrees of freedom (deflection along the axis normal, rotation) per
 * free node; marker_node[l] = the node marker l rides on (call after orc_set_markers).  EI: bending stiffness, mu_s: mass
 * per unit length, zeta_s: damping ratio of Eq. 16 (Rayleigh damping from omega_1, omega_2 of Eq. 17). */
int  orc_set_beam(orc_sim*, int n_nodes, const double* node_xy, const int* marker_node, double EI, double mu_s, double zeta_s);
int  orc_beam_ndof(orc_sim*);                                     /* 2 (n_nodes - 1) */
void orc_beam_matrices(orc_sim*, double* K, double* M, double* C, double* coef /* alpha, beta, omega_1, omega_2 */);
void orc_get_beam_state(orc_sim*, double* w, double* v, double* a, double* Q);   /* ndof each; Q = load of the last step */
void orc_set_beam_state(orc_sim*, const double* w, const double* v, const double* a);
void orc_beam_newmark(orc_sim*, const double* Q, double dt);      /* one Newmark step with the given load (piece for the pins) */
int  orc_step(orc_sim*, int nsteps, orc_info* last, int* iters_per_step /* nsteps ints or NULL */);
int  orc_poisson_solve(orc_sim*, const double* rhs, double* p_inout, orc_info* info);
int  orc_set_history(orc_sim*, int have_history, long long step);   /* restart support */

/* pieces exposed so the tests can pin them one by one */
double orc_delta_phi(int kind, double r);                       /* Eq. 22 / Roma kernel, h factored out */
void orc_laplacian(orc_sim*, const double* p, double* out);     /* L p  (O6) */
void orc_apply_A(orc_sim*, const double* x, double* out);       /* A x = -dy_j L x */
void orc_divergence(orc_sim*, const double* u, const double* v, const double* w, double* out);
void orc_gradient(orc_sim*, const double* p, double* gu, double* gv, double* gw); /* 0 on boundary faces */
void orc_momentum_rhs(orc_sim*, double* hu, double* hv, double* hw); /* H^n of current u,v,w */
void orc_convection(orc_sim*, double* cu, double* cv, double* cw);   /* C only (nu=0, g=0) */
void orc_eddy_viscosity(orc_sim*, double* nut);                  /* Smagorinsky nu_t at the cell centres of the current u, v, w */
double orc_wall_utau(double U, double y, double nu);             /* u_tau of Spalding's law (Eq. 27) by Newton-Raphson */
/* The predicted field of the current state without advancing it: stage 0 = after O3 (predictor + prescribed
 * boundary-normal faces, incl. the convective-outflow update), 1 = after O4 (IBM direct forcing, u*),
 * 2 = after O5 (outflow flux correction).  Returns non-zero for an unknown stage. */
int  orc_predict(orc_sim*, int stage, double* us, double* vs, double* ws);
void orc_vcycle(orc_sim*, const double* r, double* z);          /* z = M^-1 r, GMG */
void orc_jacobi_diag(orc_sim*, double* diag);
/* IBM pieces: arrays sized by the current marker count n */
int  orc_marker_count(orc_sim*);
void orc_ibm_index(orc_sim*);                                   /* I-1: (re)build indices + cell list */
void orc_get_cell_list(orc_sim*, int* base /*3*n*3*/, int* perm /*n*/, int* keys /*n*/,
                       int* seg_start /*n+1*/, int* nseg);
void orc_interpolate(orc_sim*, const double* u, const double* v, const double* w, double* out /*n*3*/);
void orc_spread(orc_sim*, const double* F /*n*3*/, double* fu, double* fv, double* fw); /* adds f */
void orc_get_markers(orc_sim*, double* xyz, double* vel, double* force);
void orc_set_body_state(orc_sim*, const double* disp, const double* vel);
void orc_get_body_state(orc_sim*, double* disp, double* vel, double* force);
double orc_inflow_rand(uint64_t seed, long long step, int face, int a, int b);
void orc_rk4_body(double m, double c, double k, double F, double dt, double* w, double* wdot);

#ifdef __cplusplus
}
#endif
#endif
