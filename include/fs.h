/*
 * fs.h -- C ABI of the B200-native fractional-step Navier-Stokes / immersed-boundary library.
 *
 * One call of fs_step advances the incompressible Navier-Stokes finite-volume solver of
 * Diff-FlowFSI (arxiv 2505.23940; section 2.3.1) by one fractional step on a
 * staggered Cartesian grid (pressure at cell centres, velocity components on their faces, PAPER.md
 * L100):
 *
 *   predictor   u~ = u^n + dt (a0 H^n + a1 H^{n-1}),  H = -div(u u) + nu lap(u) + g   (Eq. 4)
 *   IBM         U_l = sum_x u~(x) delta_h(x - X_l) dv            (Eq. 3b; operator of Eq. 20)
 *               F_l = (U^b_l - U_l)/dt                           (Eq. 5, at the markers)
 *               u*  = u~ + dt sum_l F_l delta_h(x - X_l) dV_l    (Eq. 3a; Eq. 4)
 *   Poisson     lap p = (rho/dt) div u*                          (Eq. 7; Eq. 9 with eps = 0, L127-129)
 *   projection  u^{n+1} = u* - (dt/rho) grad p                   (Eq. 6/10, L114, L131)
 *   rigid body  m w'' + c w' + k w = F  by RK4                   (Eq. 12)
 *
 * All of it runs in hand-written CUDA kernels for sm_100a, replayed as one CUDA graph per step
 * (the PCG loop is a device-controlled conditional WHILE node).  There is no CPU fallback.
 *
 * Conventions
 *  - Every pointer argument says whether it is a HOST or a DEVICE pointer.  No torch types.
 *  - Eulerian arrays: x fastest, then y, then z; structure of arrays.  Extents:
 *        p, div       : nz * ny * nx
 *        u, hu        : nz * ny * (nx+bx)     bx = 1 if the x direction is bounded (non-periodic)
 *        v, hv        : nz * (ny+by) * nx
 *        w, hw        : (nz+bz) * ny * nx
 *    u(i,j,k) sits at (x_f(i), y_c(j), z_c(k)), v at (x_c, y_f(j), z_c), w at (x_c, y_c, z_f(k)).
 *  - Marker arrays are always fp64 (positions decide integer indices; see fs_set_ibm_markers).
 *  - Ownership: the library never allocates device memory.  The caller passes one workspace of
 *    fs_workspace_bytes() bytes (256-byte aligned) and the CUDA stream everything runs on; both
 *    must outlive the fs_grid.  The fs_grid host object (and its CUDA graphs) belongs to the
 *    library and is released by fs_grid_destroy.  All set calls copy; all get calls copy out.
 *  - Device: a grid lives on the CUDA device that owns its workspace, which must be the caller's current device
 *    when fs_grid_create is called (the stream belongs to it too).  Every later call makes that device current
 *    for its duration and restores the caller's, so grids on several GPUs can be driven from one thread.
 *  - Errors: every call returns fs_status; nothing throws or aborts across the ABI; out-parameters
 *    are untouched on failure.  Two documented exceptions, where the out-parameter IS filled because it
 *    describes the failure: fs_step(..., last) returning FS_ERR_NOT_CONVERGED / FS_ERR_UNSUPPORTED, and
 *    fs_poisson_solve(..., info) returning FS_ERR_NOT_CONVERGED.
 */
#ifndef FS_H
#define FS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct fs_grid fs_grid;   /* opaque */

typedef enum { FS_OK = 0, FS_ERR_INVALID_ARG, FS_ERR_BAD_STATE, FS_ERR_OOM, FS_ERR_CUDA,
               FS_ERR_NOT_CONVERGED, FS_ERR_UNSUPPORTED } fs_status;
typedef enum { FS_F32 = 0, FS_F64 = 1 } fs_dtype;
/* Boundary types of PAPER.md Table 1 (L429, L454-456). */
typedef enum { FS_BC_PERIODIC = 0, FS_BC_NOSLIP = 1, FS_BC_SLIP = 2, FS_BC_INFLOW = 3,
               FS_BC_OUTFLOW_CONVECTIVE = 4 } fs_bc;
typedef enum { FS_TIME_EULER = 0,   /* Eq. 4 as printed (L104) */
               FS_TIME_AB2 = 1,     /* u~ = u + dt (a0 H^n + a1 H^{n-1}); a0 = 1 + r/2, a1 = -r/2, r = dt_n / dt_{n-1} (configs) */
               FS_TIME_RK3 = 2      /* "explicit Runge-Kutta" (L100, L431, Table 1): three-stage SSP scheme, each stage a full
                                       fractional step E(u): u1 = E(u^n), u2 = 3/4 u^n + 1/4 E(u1), u^{n+1} = 1/3 u^n + 2/3 E(u2) */
             } fs_time;
typedef enum { FS_PC_NONE = 0, FS_PC_JACOBI = 1, FS_PC_GMG = 2 } fs_precond; /* CG: L449, L686 */
typedef enum { FS_DELTA_ROMA3 = 0, FS_DELTA_PESKIN4 = 1 } fs_delta;        /* Eq. 21-22 */
typedef enum { FS_EXEC_GRAPH = 0,   /* one CUDA-graph replay per step, PCG loop = conditional WHILE node */
               FS_EXEC_STREAM = 1   /* same kernels launched directly; host polls the PCG flag (debug) */
             } fs_exec;
typedef enum { FS_CONV_CENTRAL = 0,  /* 2nd-order central convective fluxes (the default of every config) */
               FS_CONV_UPWIND = 1    /* 1st-order upwind: transported value from the upwind side of each face (L100, Table 1) */
             } fs_conv;
typedef enum { FS_U = 0, FS_V, FS_W, FS_P, FS_HU, FS_HV, FS_HW, FS_DIV,
               FS_MARKER_X,      /* n*3 fp64 positions */
               FS_MARKER_U,      /* n*3 fp64 target velocities U^b */
               FS_MARKER_F,      /* n*3 fp64 forces F_l of the last step */
               FS_MARKER_BASE,   /* 3*n*3 int32: lowest support index [component][marker][direction] */
               FS_MARKER_PERM,   /* n int32: marker ids sorted by (cell key, id) */
               FS_MARKER_KEYS,   /* n int32: sorted cell keys */
               FS_MARKER_SEG,    /* nseg+1 int32 segment starts (call fs_marker_segments for nseg) */
               FS_BODY_STATE,    /* 9 fp64: displacement[3], velocity[3], force[3] */
               FS_MASK_U, FS_MASK_V, FS_MASK_W   /* uint8 per stored face of u / v / w: 0 fluid, 1 solid, 2 IB point (get only;
                                                    shapes of FS_U / FS_V / FS_W; eps-mask IBM, fs_set_solid_mask) */
             } fs_field;

typedef struct {
  int nx, ny, nz;
  double x0, y0, z0, lx, ly, lz;
  const double* yf;            /* HOST, ny+1 face coordinates; NULL = uniform (stretching is y-only) */
  fs_dtype dtype;              /* arithmetic / storage type of all Eulerian fields */
  fs_bc bc[6];                 /* -x,+x,-y,+y,-z,+z ; both faces of a direction periodic or neither */
  double bc_vel[6][3];         /* wall / inflow velocity; [outflow][normal] = convective speed U_c */
  double nu, rho, dt, body_force[3];
  fs_time time_scheme;
  fs_precond precond; double rtol; int max_iter; int warm_start;
  int mg_nu1, mg_nu2, mg_coarse_sweeps; double mg_omega;   /* GMG V(nu1,nu2), damped Jacobi */
  fs_delta delta; int max_markers;
  uint64_t seed; double inflow_noise;
  fs_exec exec_mode;
  fs_conv convection;          /* convective flux scheme of the momentum RHS */
  int solid_mask;              /* != 0: reserve workspace for the eps-mask IBM (fs_set_solid_mask) */
  double cs;                   /* constant Smagorinsky coefficient C_s (L437, L452, L638): nu_t = (C_s Delta)^2 |S|, Delta = (hx dy hz)^(1/3),
                                  diffusive term div[(nu + nu_t) grad u_i]; 0 = no subgrid model */
  int wall_model;              /* != 0: equilibrium wall model on no-slip y walls (Spalding's law, Eq. 27, kappa = 0.4, B = 5, by
                                  Newton-Raphson; nu_t of Eq. 28-29 on the wall face of the tangential components) */
  int coupling_max_iters;      /* strong FSI coupling (Algorithm 1): up to this many fluid + structure sweeps per step, each
                                  restarting the fluid from time level n with the structure's latest iterate; <= 1: weak coupling */
  double coupling_tol;         /* stop when xi = || (w^k - w^{k-1}) / w^{k-1} ||_2^2 < coupling_tol (paper: 1e-5, N <= 100) */
  double cfl;                  /* > 0: CFL-adaptive step (L431): dt = min(dt, cfl h_min / max|u,v,w|) from the field at the start
                                  of every step, h_min the smallest cell extent; <= 0: fixed dt */
  int max_beam_nodes;          /* > 0: reserve workspace for a flexible beam of up to this many nodes (fs_set_beam; <= 129) */
} fs_params;

typedef struct {
  int pcg_iters; int converged; int nan_flag;
  double rel_residual;        /* recurrence residual ||r|| / ||b|| that the stopping test used */
  double true_rel_residual;   /* ||b - A p|| / ||b|| recomputed from the projected field */
  double max_abs_div;         /* max |D u^{n+1}| */
  double body_force[3], body_disp[3], body_vel[3];
  long long step;
  long long unconverged_steps;  /* sticky, since fs_grid_create: steps whose PCG hit max_iter ...            */
  long long nan_steps;          /* ... and steps whose projected field held a NaN (also seen by async steps) */
  double dt, time;              /* step size of the last step (CFL-adaptive dt), elapsed time since the grid was created */
  int coupling_iters;           /* Algorithm 1: sweeps of the last step (1 = weak coupling) ... */
  double coupling_xi;           /* ... and its final xi; pcg_iters is then the sum over the sweeps */
} fs_step_info;
typedef struct { int iters; int converged; double rel_residual, true_rel_residual; } fs_poisson_info;

/* Bytes of device workspace fs_grid_create needs for these parameters: the fields of one fractional step (u, v, w,
 * u*, H^{n-1}, p: Eq. 4-10), the PCG vectors of the Poisson solve (Eq. 7; CG L449), the
 * GMG levels, and the marker arrays (Eq. 18 notation, L183-185).  HOST pointers.  FS_ERR_INVALID_ARG /
 * FS_ERR_UNSUPPORTED as for fs_grid_create; *bytes untouched then. */
fs_status fs_workspace_bytes(const fs_params* params, size_t* bytes);

/* Creates a grid: the staggered finite-volume arrangement of PAPER.md L100 (p at cell centres, velocity
 * components on their faces; uniform, or y-stretched through params->yf) with the boundary types of Table 1
 * (L429, L454-456).  params: HOST.  workspace: DEVICE memory of the CURRENT device, >= fs_workspace_bytes,
 * 256-byte aligned, owned by the caller, zeroed by this call.  cuda_stream: a cudaStream_t of the current
 * device (NULL = legacy default stream).  FS_ERR_INVALID_ARG: bad parameters, misaligned / too small / non-device
 * workspace or one that belongs to another device.  FS_ERR_UNSUPPORTED: GMG on a grid that is not uniform and
 * isotropic (periodic and bounded directions may be mixed: on a bounded one the boundary flux is dropped on every level);
 * more than 2^31 - 1 stored values per field. */
fs_status fs_grid_create(const fs_params* params, void* workspace, size_t bytes, void* cuda_stream,
                         fs_grid** out);
fs_status fs_grid_destroy(fs_grid* g);

/* Number of elements of a field (HOST out pointer). */
fs_status fs_field_size(fs_grid* g, fs_field f, long long* count);

/* Copy a whole field of the solver state (u, v, w on faces, p at centres; H = the explicit right-hand
 * side of Eq. 4; the marker arrays of Eq. 18) in / out.  src/dst is a HOST pointer when
 * *_on_device == 0, else a DEVICE pointer.  dtype applies to FS_U..FS_DIV (converted if it differs from the grid's); marker fields
 * are fp64 / int32 regardless.  Synchronises the stream.  FS_DIV is computed on demand (get only). */
fs_status fs_fields_set(fs_grid* g, fs_field f, const void* src, fs_dtype dtype, int src_on_device);
fs_status fs_fields_get(fs_grid* g, fs_field f, void* dst, fs_dtype dtype, int dst_on_device);

/* Asynchronous variants for pipelines -- e.g. several independent grids, each on its own stream, so that one grid's PCIe
 * traffic overlaps another grid's step (replicas): as fs_fields_set / fs_fields_get for FS_U .. FS_HW with a HOST
 * buffer of the GRID's dtype, but the copy is only enqueued on the grid's stream.  The buffer must be page-locked for the copy
 * to be asynchronous and must stay valid and untouched until the caller has synchronised that stream.  FS_ERR_INVALID_ARG
 * for other fields. */
fs_status fs_fields_set_async(fs_grid* g, fs_field f, const void* host_src);
fs_status fs_fields_get_async(fs_grid* g, fs_field f, void* host_dst);

/* Restart support: whether H^{n-1} is valid (AB2) and the step counter (inflow-noise hash). */
fs_status fs_set_history(fs_grid* g, int have_history, long long step);

/* Lagrangian markers (Eq. 18 notation: X_l, velocity, volume element dV_l; L183-185).  HOST
 * pointers, fp64: xyz n*3, vel n*3 (NULL = 0), dvol n (NULL = hx*hy*hz).  n = 0 removes them.
 * Rebuilds indices and the cell list.  FS_ERR_UNSUPPORTED on a y-stretched grid, and when the delta-function
 * support of a marker (3 or 4 nodes per direction, Eq. 21-22) reaches a prescribed boundary-normal face or leaves
 * the box in a non-periodic direction (the grid then keeps no markers); n > max_markers is FS_ERR_INVALID_ARG. */
fs_status fs_set_ibm_markers(fs_grid* g, int n, const double* xyz, const double* vel, const double* dvol);
fs_status fs_marker_segments(fs_grid* g, int* nseg);

/* Rigid body of Eq. 12 (L144-147): mass, damping, stiffness given directly; dof_mask bit0=x,1=y,2=z.
 * All markers translate with the body. */
fs_status fs_set_body(fs_grid* g, double m, double c, double k, int dof_mask);
fs_status fs_set_body_state(fs_grid* g, const double* disp3, const double* vel3);   /* HOST */

/* Flexible structure (Eq. 11, Eq. 13-17, Newmark-beta L177): a straight Euler-Bernoulli beam of
 * n_nodes nodes in the x-y plane, clamped at node 0 (the flexible plates of section 3.3), bending only (L149):
 * every free node carries the deflection w along the normal n of the reference axis and the rotation theta, the degrees of
 * freedom of the 4 x 4 element matrices of Eq. 13 (stiffness, EI / L_e^3) and Eq. 14 (consistent mass, mu_s L_e / 420).
 * Damping C = alpha M + beta K (Eq. 15) with alpha, beta from the two lowest modal frequencies of Eq. 17 and the damping
 * ratio zeta_s (Eq. 16).  Every step the nodal load Q_i = n . q_i, q_i = -rho sum_{l on node i} F_l dV_l (Eq. 20), drives
 * one Newmark-beta step (gamma = 1/2, beta = 1/4) of Eq. 11 on the device; markers follow their node, X_l = X_l^ref + w n,
 * U^b_l = dw/dt n.  With params.coupling_max_iters > 1 the sweeps of Algorithm 1 apply (xi over all degrees of freedom).
 * node_xy: HOST, n_nodes * 2 fp64, collinear and ordered along the axis; marker_node: HOST, one int per marker (call after
 * fs_set_ibm_markers; the current marker positions become the reference configuration).  FS_ERR_BAD_STATE without markers
 * or with params.max_beam_nodes < n_nodes; FS_ERR_UNSUPPORTED together with a rigid body, the eps mask or a CFL-adaptive
 * step; FS_ERR_INVALID_ARG for nodes that are not collinear / ordered, EI <= 0, mu_s <= 0, zeta_s < 0, a bad node index. */
fs_status fs_set_beam(fs_grid* g, int n_nodes, const double* node_xy, const int* marker_node, double EI, double mu_s, double zeta_s);
/* Beam state (HOST, fp64, 2 (n_nodes - 1) values each: w_1, theta_1, w_2, ...; any pointer may be NULL): displacement,
 * velocity, acceleration, the load vector of the last step; coef (4 values): alpha, beta (Eq. 16), omega_1, omega_2 (Eq. 17). */
fs_status fs_beam_state(fs_grid* g, double* w, double* v, double* a, double* Q, double* coef);

/* The paper's own IBM: volume-of-solid function eps (1 in solid cells, 0 in fluid cells,
 * L110) instead of marker forcing.  eps_cells: HOST, nz*ny*nx bytes; uc: HOST, 3 fp64, the exact velocity u_c of the
 * immersed solid (Eq. 8; NULL = at rest; a rigid body set with fs_set_body overrides it with its own velocity).
 *   predictor   u* = (1 - eps) u~ + eps u_s                       (Eq. 4 with the forcing of Eq. 5)
 *               u_s = u_c on faces of solid cells, u_IB at the IB points (Eq. 23)
 *   IB points   u_IB = sum_i wdot(X_i) delta_h(x - X_i) dV_i / F_Ni,  F_Ni = sum over the fluid nodes of the support
 *               of delta_h dv   (Eq. 18-19; only when markers are set: they carry the structure's velocity)
 *   Poisson     lap p = (rho/dt) div[(1 - eps) u* + eps u_c]      (Eq. 9; = Eq. 7 when eps = 0, L129)
 *   body force  -rho sum_x f(x) dv,  f = (u* - u~)/dt             (Eq. 20 summed over the body, L193)
 * A face is solid when either cell it separates is solid; IB points are fluid faces with a solid face among their six
 * same-component neighbours (L74); prescribed boundary-normal faces are never forced.  eps_cells == NULL returns to
 * marker forcing.  FS_ERR_BAD_STATE unless params.solid_mask != 0; FS_ERR_UNSUPPORTED on a y-stretched grid. */
fs_status fs_set_solid_mask(fs_grid* g, const unsigned char* eps_cells, const double* uc);

/* Advance nsteps fractional steps: predictor (Eq. 4) -> IBM interpolate / force / spread (Eq. 3b, 5, 3a;
 * L89-91, L108) -> Poisson (Eq. 7) by PCG (L449, L686) -> projection (Eq. 6/10, L114, L131) -> rigid body
 * (Eq. 12), one CUDA-graph replay per step.  last == NULL: fully asynchronous on the grid's stream.
 * last != NULL (HOST): synchronises and fills *last for the final step (also when it returns
 * FS_ERR_NOT_CONVERGED: that step's PCG hit max_iter; or FS_ERR_UNSUPPORTED: a moving body carried a marker
 * support into a non-periodic boundary).  unconverged_steps / nan_steps count such steps over ALL steps since the
 * grid was created, including asynchronous ones. */
fs_status fs_step(fs_grid* g, int nsteps, fs_step_info* last);

/* Solves lap p = rhs (Eq. 7 form; homogeneous Neumann on bounded faces, zero-mean solution) with
 * the grid's PCG.  rhs and p_inout: nz*ny*nx elements of `dtype`, HOST or DEVICE by on_device;
 * p_inout holds the initial guess when warm_start != 0.  Synchronises. */
fs_status fs_poisson_solve(fs_grid* g, const void* rhs, void* p_inout, fs_dtype dtype, int on_device,
                           fs_poisson_info* info);

/* Pieces of the path exposed for element-wise parity tests (DEVICE work, HOST pointers, fp64):
 *   fs_ibm_interpolate: out[n*3] = interpolation of the current u,v,w at the markers (Eq. 3b)
 *   fs_ibm_spread:      u,v,w += spread of F[n*3] (Eq. 3a, f = sum_l F_l delta_h dV_l, no dt) */
fs_status fs_ibm_interpolate(fs_grid* g, double* out);
fs_status fs_ibm_spread(fs_grid* g, const double* F);
/*   fs_gmg_vcycle: z = M^-1 r, one V-cycle of the GMG preconditioner (r, z: nz*ny*nx fp64, HOST);
 *   FS_ERR_BAD_STATE unless precond == FS_PC_GMG.  Clobbers the PCG scratch fields only. */
fs_status fs_gmg_vcycle(fs_grid* g, const double* r, double* z);
/*   fs_momentum_rhs: runs the S1 kernel alone on the current u,v,w: FS_HU/HV/HW := H^n (Eq. 4),
 *   overwriting the stored H^{n-1}; u,v,w,p are untouched (the predicted field goes to scratch). */
fs_status fs_momentum_rhs(fs_grid* g);

/* Per-kernel timing (measurement aid for bench.py's roofline block).  fs_profile_step advances nsteps
 * steps with the SAME kernels launched directly on the grid's stream (not the graph), each bracketed by
 * a CUDA event pair, and accumulates per kernel name: launches, milliseconds, and ALGORITHMIC bytes
 * (the field words that pass must move).  Synchronises.  Entries are read back
 * one by one (name: library-owned static string; all out pointers HOST). */
fs_status fs_profile_step(fs_grid* g, int nsteps);
fs_status fs_profile_count(fs_grid* g, int* n);
fs_status fs_profile_entry(fs_grid* g, int idx, const char** name, long long* launches, double* ms, double* bytes);
fs_status fs_profile_reset(fs_grid* g);

/* Number of kernel launches (graph kernel nodes incl. loop-body replays) issued so far. */
fs_status fs_launch_count(fs_grid* g, long long* launches);

/* Which kernel instantiations this grid has enqueued so far, as one ';'-separated string of names such as
 * "k_mg_down<f64,TR16,UPD>" (lets a parity test assert that it exercised the instantiation it was written for).
 * buf: HOST, cap bytes; *needed (HOST, may be NULL) = bytes including the terminator.  buf == NULL && cap == 0
 * only queries the size; a too small buf is FS_ERR_INVALID_ARG. */
fs_status fs_kernels_used(fs_grid* g, char* buf, size_t cap, size_t* needed);

const char* fs_status_string(fs_status s);

#ifdef __cplusplus
}
#endif
#endif
