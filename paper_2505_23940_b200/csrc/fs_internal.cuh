// fs_internal.cuh -- device-side data structures and launcher declarations shared by the CUDA
// translation units of libfs (the product).  Nothing here is shared with oracle/.
//
// Layout in HBM: structure of arrays, x fastest, then y, then z;
// a velocity component has n+1 entries along its own normal when that direction is bounded.
#pragma once
#include <cuda.h>            // CUtensorMap (the type and enums only: the driver entry point is looked up at run time)
#include <cuda_runtime.h>
#include <stdint.h>
#include <cstdlib>
#include "../../include/fs.h"

namespace fs {

constexpr int kMaxLevels = 12;
constexpr int kMaxPartials = 32768;   // partial sums per reduction slot (>= blocks of any reducing kernel)
constexpr int kRedSlots = 4;          // values reduced at once by one kernel

// Scalars that live in device memory so that a captured step never needs the host.
struct Scalars {
  // Poisson / PCG
  double mean_coef;      // sum(bhat_raw) / sum(dy)      (compatibility shift)
  double bnorm2, rr;     // ||bhat||^2, ||r||^2 (recurrence residual)
  double rho_cur, rho_prev, dq;
  double pmean;
  double rmean;         // fp32 only: mean of the recurrence residual, removed with one iteration of lag (null-space deflation)
  double sum_dy;         // sum over all cells of dy_j
  int iter, done, converged, first;
  int rsel, need_update; // rsel: which residual buffer (r / r2) is current; need_update: K2 of the last iteration still to do (k_mg_down<UPD>)
  int dsel, pending;     // pending: the x += alpha_prev d of the last k_pcg_update has not been applied yet
  double alpha_prev, sum_p, sum_d;   // deferred x update (k_pcg_dirapply / k_pflush)
  int body_runs;         // replays of the PCG loop body in the current solve (counted by the direction kernel)
  int ibm_oob;           // sticky: a marker support reached a non-periodic boundary (unsupported)
  int max_iter, pad0;
  double rtol;
  // step control
  double dt, dt_prev, time;   // step size of the current / previous step (CFL-adaptive dt lives on the device), elapsed time
  double umax;                // max |u|, |v|, |w| over all stored faces (k_dt_begin)
  int iter_acc, conv_acc, body_acc, pad4;   // Runge-Kutta: PCG iterations / convergence / body replays summed over the stages
  long long step; int have_hist; int nan_flag;
  double max_div, true_rr;
  long long total_iters, total_body;          // PCG iterations / loop-body replays of all steps so far
  long long unconverged_steps, nan_steps;     // sticky: steps whose PCG hit max_iter / whose projected field held a NaN
  // open-boundary flux correction (O5)
  double flux_phi, flux_aout;
  // IBM
  int nseg; int bbox_lo[3], bbox_hi[3]; int pad1;
  double body_force[3], body_disp[3], body_vel[3];
  double body_disp0[3], body_vel0[3];   // strong coupling: the body's state at time level n (every sweep's RK4 starts there)
  double beam_xi;                       // flexible beam: xi of Algorithm 1 of the last Newmark step
  // tickets for last-block reductions
  unsigned int ticket[8];
};

template <class T> struct Ctx {
  int nx, ny, nz, bx, by, bz, nxu, nyv, nzw;
  int bc[6];
  double bcv[6][3];
  double hx, hy, hz, dt, rho, nu, g[3];   // dt: the configured (maximum) step; kernels read the current one from S->dt
  double cfl, hmin;
  double cs; int wall_model;     // LES closures (constant Smagorinsky, Spalding wall model); nu_t lives in q before the Poisson solve
  double x0, y0, z0;
  T ihx, ihz, ihx2, ihz2;
  int time_scheme, precond, warm_start, delta, uniform_y, convection;
  uint64_t seed; double inflow_noise;
  // y metrics (device arrays of T unless noted)
  const T* dy;     // [ny+2]: dy[j+1] = DY(j), j in [-1, ny] (mirrored ghost at walls, wrapped if periodic)
  const T* idy;    // [ny+2] idy[j+1] = 1/DY(j)
  const T* idyc;   // [ny+1] 1/DYC(j): centre-to-centre distance across face j
  const T* wyl;    // [ny+1] weight of the value below face j in the linear interpolation to the face
  const T* wyh;    // [ny+1] weight of the value above
  const T* cyl;    // [ny]   Laplacian coefficient towards j-1 (0 at a bounded end)
  const T* cyh;    // [ny]   towards j+1
  const double* dy64;  // [ny] fp64 cell heights (reductions, flux areas)
  // fields
  T *u, *v, *w, *p, *us, *vs, *ws, *hu, *hv, *hw;
  T *q0u, *q0v, *q0w;    // u^n kept for the Runge-Kutta stage combinations (FS_TIME_RK3 only, else nullptr)
  T *r, *r2, *d, *d2, *q, *z, *bh;   // r2: second residual buffer (GMG fused update), else nullptr
  Scalars* S;
  double* partials;     // [kRedSlots][kMaxPartials]
};

// TMA descriptor of a dense (nx, ny, nz) field with a (boxx, boxy, 1) box; passed to kernels as a __grid_constant__ parameter
struct Tmap { CUtensorMap m; };
// false when the driver entry point is missing or the field / box does not qualify (then the kernel skips its prefetches)
bool tmap_encode(Tmap* out, const void* ptr, int esize, int nx, int ny, int nz, int boxx, int boxy);
// the fields one streaming kernel prefetches; n = 0: none (some map could not be encoded)
struct TmapSet { Tmap m[6]; int n; };
constexpr int kPfAhead = 4;          // planes between the L2 prefetch of a tile plane and the register loads of the same data

struct MgLevel { int nx, ny, nz; double h; void *e, *g, *t; };
template <class T> struct MgCtx {
  int nlev, nu1, nu2, coarse_sweeps; double omega;
  int bd;                      // bit d set: direction d is bounded (boundary fluxes dropped on every level, reading G1); 0: triply periodic
  MgLevel lev[kMaxLevels];
};

struct IbmCtx {
  int n, sw, delta;            // markers, support width (3 or 4)
  double org[3][3];            // node origin of component c along direction d
  double inv[3];               // 1/h per direction
  double o[3];                 // domain origin
  double ivol;                 // 1/(hx hy hz)
  double *X, *Ub, *dV, *Fl, *Ul, *wts;   // wts: [3][n][3][4]
  int *base, *perm, *keys, *keys_raw, *seg, *flags;
  // body (Eq. 12)
  int has_body, dof; double bm, bc, bk;
  int strong;                  // strong coupling (Algorithm 1): RK4 starts from body_disp0 / body_vel0
  // eps-mask IBM (Eq. 5, 8-9, 18-19, 23): cell mask, per-face classes (0 fluid, 1 solid, 2 IB point), u_c, scratch for u_IB
  int has_mask; double uc[3];
  unsigned char *eps, *mu, *mv, *mw;
  void *ibu, *ibv, *ibw;       // T*: u_IB spread from the markers (Eq. 18), velocity-shaped
  // flexible beam (Eq. 11, 13-17, Newmark-beta; reading N2-2): ndof = 2 (nodes - 1) degrees of freedom (w, theta per free node)
  int has_beam, nbn, ndof;
  double bnrm[2];              // unit normal of the straight reference axis (markers move along it)
  double nk[6];                // Newmark coefficients a0..a5 for the grid's (fixed) dt
  double *bw, *bv, *ba, *bw0, *bv0, *ba0, *bQ;   // state, state of time level n (strong coupling), load of the last step
  double *bL, *bM, *bC;        // band storage: Cholesky factor of K_eff [ndof][4] (columns r-3..r), M and C [ndof][7] (columns r-3..r+3)
  double *Xref;                // marker positions of the undeformed beam
  int *mnode, *nstart, *nlist; // node of each marker; markers of node i = nlist[nstart[i] .. nstart[i+1]) in ascending id
};
constexpr int kMaxBeamNodes = 129;   // 256 degrees of freedom: the Newmark step runs in one CTA's shared memory

// Per-kernel timing (measurement aid, fs_profile_step): when prof != nullptr every launch is bracketed
// by a CUDA event pair on the launching stream and tagged with its name and ALGORITHMIC bytes (the
// field words the pass must move; not what the hardware happened to move).
struct Prof;
void prof_begin(Prof* p, const char* name, double bytes, cudaStream_t s);
void prof_end(Prof* p, cudaStream_t s);
// Which kernel instantiations a grid has enqueued so far (always on; host side, recorded at launch / capture time):
// lets a parity test assert that it exercised the template instantiation it was written for (fs_kernels_used).
struct Seen;
void seen_add(Seen* s, const char* inst);
struct Launch { cudaStream_t s; cudaGraphConditionalHandle cond; int use_cond; Prof* prof; Seen* seen; };
// name: profile label (what the pass is); inst: the kernel instantiation that runs it
#define FS_LAUNCHI(L, name, inst, bytes, ...)                       \
  do {                                                              \
    if ((L).seen) seen_add((L).seen, inst);                         \
    if ((L).prof) prof_begin((L).prof, name, (double)(bytes), (L).s); \
    __VA_ARGS__;                                                    \
    if ((L).prof) prof_end((L).prof, (L).s);                        \
  } while (0)
#define FS_LAUNCH(L, name, bytes, ...) FS_LAUNCHI(L, name, name, bytes, __VA_ARGS__)
template <class T> constexpr const char* tname() { return sizeof(T) == 8 ? "f64" : "f32"; }


// z chunk length of a streaming kernel: xy tiles x chunks CTAs run in waves of `slots` (CTAs resident on the
// 148 SMs); every chunk marches its planes plus `halo` redundant ones.  Pick the chunk count that minimises
// waves x planes per chunk (a half-empty last wave costs as much as a full one), chunks of at least min_kz
// planes, at most kMaxPartials CTAs (one reduction partial each).
inline int pick_kz(long long tiles_xy, int nz, long long slots, int halo, int min_kz) {
  { static const int ov = [] { const char* e = getenv("FS_TUNE_MINKZ"); return e ? atoi(e) : 0; }(); if (ov > 0) min_kz = ov; }
  int best = nz; double best_cost = 1e300;
  for (int zc = 1; zc <= nz; ++zc) {
    const int kz = (nz + zc - 1) / zc;
    if (zc > 1 && kz < min_kz) break;
    if ((nz + kz - 1) / kz != zc) continue;              // same chunk count as a smaller zc: already seen
    if (tiles_xy * zc > kMaxPartials) break;
    const long long waves = (tiles_xy * zc + slots - 1) / slots;
    const double cost = (double)waves * (kz + halo);
    if (cost < best_cost * 0.999) { best_cost = cost; best = kz; }
  }
  return best;
}

// ---- launchers (one per kernel family; each returns the number of kernels it enqueued) ----------
template <class T> int launch_momentum(const Ctx<T>& c, const Launch& L);
// vectorised S1 kernel (fs_kernels_momv.cu): periodic x, nx a multiple of the vector width, no LES closure, y / z periodic or walls
template <class T> bool momentumv_applies(const Ctx<T>& c);
template <class T> int launch_momentumv(const Ctx<T>& c, const Launch& L);
template <class T> cudaError_t momv_configure_device();
template <class T> int launch_flux_correction(const Ctx<T>& c, const Launch& L);
template <class T> int launch_div_rhs(const Ctx<T>& c, const Launch& L);
template <class T> int launch_rhs_from_b(const Ctx<T>& c, const T* b, const Launch& L);
template <class T> int launch_project(const Ctx<T>& c, const Launch& L);
template <class T> int launch_divergence(const Ctx<T>& c, const T* u, const T* v, const T* w, T* out, const Launch& L);
template <class T> int launch_step_end(const Ctx<T>& c, const IbmCtx& ib, const Launch& L);
template <class T> int launch_step_begin(const Ctx<T>& c, const Launch& L);                      // CFL dt, Runge-Kutta u^n copy
template <class T> int launch_stage_end(const Ctx<T>& c, int stage, const Launch& L);           // Runge-Kutta stage combination
template <class TS, class TD> void launch_convert(const TS* src, TD* dst, long long n, cudaStream_t s);
template <class T> void launch_scale(T* x, double a, long long n, cudaStream_t s);

template <class T> int launch_pcg_init(const Ctx<T>& c, const Launch& L, bool need_bhat);
template <class T> int launch_pcg_body(const Ctx<T>& c, const MgCtx<T>& mg, const Launch& L);
template <class T> int launch_pcg_finish(const Ctx<T>& c, const Launch& L);
// the whole solve as one persistent cooperative kernel (fs_kernels_pcgc.cu): point preconditioners, L2-sized grids
template <class T> bool pcg_coop_applies(const Ctx<T>& c);
template <class T> int launch_pcg_coop(const Ctx<T>& c, const Launch& L);
template <class T> int launch_true_residual(const Ctx<T>& c, const Launch& L);
// dot_fused != nullptr asks for rho_cur = rhs . (zs out) from the last kernel; *dot_fused says whether it was done
// upd_fused != nullptr additionally asks the level-0 down kernel to perform the residual update of the previous
// PCG iteration (fs_kernels_mgf.cu k_mg_down<UPD>); *upd_fused says whether it was done
template <class T> int launch_vcycle(const Ctx<T>& c, const MgCtx<T>& mg, const T* rhs, T* out, const Launch& L, bool* dot_fused, T zs,
                                     bool* upd_fused = nullptr);
template <class T> int launch_mg_down(const Ctx<T>& c, const T* g, T* e, T* gc, int nx, int ny, int nz, double h, double omega,
                                      const char* name, const Launch& L, bool upd = false, T* g2 = nullptr, const T* q = nullptr);
template <class T> int launch_mg_up(const Ctx<T>& c, const T* ein, const T* ec, const T* g, T* eo, int nx, int ny, int nz, double h,
                                    double omega, bool dot, T zs, const char* name, const Launch& L, const T* g2 = nullptr);

// raises the dynamic shared-memory limit of every GMG kernel instantiation of type T on the CURRENT device
// (cudaFuncSetAttribute is per device: called by fs_grid_create for each grid, not once per process)
template <class T> cudaError_t mg_configure_device();
template <class T> cudaError_t mgf_configure_device();

template <class T> int launch_ibm_index(const Ctx<T>& c, const IbmCtx& ib, const Launch& L);
template <class T> int launch_ibm_interpolate(const Ctx<T>& c, const IbmCtx& ib, const T* u, const T* v, const T* w, double* out, const Launch& L);
template <class T> int launch_ibm_force(const Ctx<T>& c, const IbmCtx& ib, const Launch& L);
// scale < 0: the field receives (current dt) x the spread force (u* = u~ + dt f, Eq. 4); else scale x
template <class T> int launch_ibm_spread(const Ctx<T>& c, const IbmCtx& ib, const double* F, T* u, T* v, T* w, double scale, const Launch& L);
template <class T> int launch_mask_classify(const Ctx<T>& c, const IbmCtx& ib, const Launch& L);
template <class T> int launch_mask_forcing(const Ctx<T>& c, const IbmCtx& ib, const Launch& L);
template <class T> int launch_beam_step(const Ctx<T>& c, const IbmCtx& ib, const Launch& L);
// host side of fs_set_beam (fs_beam.cu): assembles Eq. 13-14, finds omega_1, omega_2 of Eq. 17, builds C (Eq. 15-16), factors
// K_eff = K + a0 M + a1 C; outputs in band storage as IbmCtx describes them.  false: M or K_eff not positive definite.
bool beam_build(int nb, const double* node_xy, double EI, double mus, double zeta, double dt,
                double* Lband, double* Mband, double* Cband, double* nk, double* coef /* alpha, beta, omega1, omega2 */);

// ---- device helpers ---------------------------------------------------------------------------------
#ifdef __CUDACC__
// two x-adjacent cells handled by one thread (16-byte accesses for fp64, 8-byte for fp32)
template <class T> struct V2T;
template <> struct V2T<double> { using type = double2; };
template <> struct V2T<float> { using type = float2; };
template <class T> struct V16T;
template <> struct V16T<double> { using type = double2; };
template <> struct V16T<float> { using type = float4; };
// L2 prefetch of one tile plane of a field through its tensor map (fs_tma.cu): one instruction, no register and no
// shared memory, so a streaming kernel can run its DRAM fetches several planes ahead of the register loads that
// follow (those then hit L2) without growing its register queue.  (x, y, z) = element coordinates of the box origin;
// parts of the box outside the array are skipped.  Called by ONE thread of the CTA.
__device__ __forceinline__ void tma_prefetch_plane(const Tmap& m, int x, int y, int z) {
  asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(reinterpret_cast<unsigned long long>(&m)), "r"(x), "r"(y), "r"(z)
               : "memory");
}
template <class T, class V> __device__ __forceinline__ V ldv2(const T* p) { return *reinterpret_cast<const V*>(p); }
template <class T, class V> __device__ __forceinline__ void stv2(T* p, const V& v) { *reinterpret_cast<V*>(p) = v; }

// one 16-byte vector of x-adjacent cells as an array (2 fp64 / 4 fp32 cells)
template <class T> struct Vec16 {
  static constexpr int VX = 16 / sizeof(T);
  alignas(16) T a[VX];
};
template <class T> __device__ __forceinline__ Vec16<T> ld16(const T* p) {
  Vec16<T> v; *reinterpret_cast<typename V16T<T>::type*>(v.a) = *reinterpret_cast<const typename V16T<T>::type*>(p); return v;
}
template <class T> __device__ __forceinline__ void st16(T* p, const Vec16<T>& v) {
  *reinterpret_cast<typename V16T<T>::type*>(p) = *reinterpret_cast<const typename V16T<T>::type*>(v.a);
}

__device__ __forceinline__ int wrapi(int i, int n) { i %= n; return i < 0 ? i + n : i; }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  return v;
}

// Block-wide sum of NV values; result valid in thread 0.  blockDim (flattened) <= 1024.
template <int NV> __device__ __forceinline__ void block_sum(double (&v)[NV], double* sh /*[NV*32]*/) {
  const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int nth = blockDim.x * blockDim.y * blockDim.z;
  const int lane = tid & 31, wid = tid >> 5, nw = (nth + 31) >> 5;
#pragma unroll
  for (int a = 0; a < NV; ++a) v[a] = warp_sum(v[a]);
  __syncthreads();
  if (lane == 0) {
#pragma unroll
    for (int a = 0; a < NV; ++a) sh[a * 32 + wid] = v[a];
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      double t = lane < nw ? sh[a * 32 + lane] : 0.0;
      v[a] = warp_sum(t);
    }
  }
}

// Deterministic grid-wide sum: every block stores its partial, the last block to arrive (ticket)
// adds the partials in a fixed order.  Returns true in ALL threads of that last block; v holds the
// totals in its thread 0.  No floating-point atomics, so results do not depend on block scheduling.
template <int NV> __device__ __forceinline__ bool grid_sum(double (&v)[NV], double* partials, unsigned int* ticket,
                                                          double* sh /*[NV*32]*/, int* sh_flag) {
  const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int nth = blockDim.x * blockDim.y * blockDim.z;
  const int bid = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
  const int nblk = gridDim.x * gridDim.y * gridDim.z;
  block_sum<NV>(v, sh);
  if (tid == 0) {
#pragma unroll
    for (int a = 0; a < NV; ++a) __stcg(&partials[a * kMaxPartials + bid], v[a]);
    __threadfence();
    unsigned int t = atomicAdd(ticket, 1u);
    *sh_flag = (t == (unsigned int)(nblk - 1));
  }
  __syncthreads();
  if (!*sh_flag) return false;
  __threadfence();
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    double t = 0.0;
    for (int b = tid; b < nblk; b += nth) t += __ldcg(&partials[a * kMaxPartials + b]);
    v[a] = t;
  }
  block_sum<NV>(v, sh);
  if (tid == 0) *ticket = 0u;
  return true;
}
#endif

}  // namespace fs
