// fs_api.cu -- the C ABI of include/fs.h: parameter validation, workspace carving, host-side metric
// tables, CUDA-graph capture of one fractional step (PCG loop = conditional WHILE node) and the
// field I/O calls.  No torch types; the caller owns device memory and the stream.
#include "fs_internal.cuh"
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace fs;

#define CK(x)                                                              \
  do {                                                                     \
    cudaError_t e_ = (x);                                                  \
    if (e_ != cudaSuccess) {                                               \
      std::fprintf(stderr, "libfs: CUDA error %s at %s:%d (%s)\n", cudaGetErrorString(e_), __FILE__, __LINE__, #x); \
      return FS_ERR_CUDA;                                                  \
    }                                                                      \
  } while (0)

// ---- per-kernel timing (fs_profile_step / fs_profile_entry) ---------------------------------------------
namespace fs {
struct ProfRec { const char* name; double bytes; cudaEvent_t e0, e1; };
struct ProfAgg { const char* name; long long launches; double ms, bytes; };
struct Prof { std::vector<ProfRec> recs; std::vector<ProfAgg> agg; };
void prof_begin(Prof* p, const char* name, double bytes, cudaStream_t s) {
  ProfRec r{name, bytes, nullptr, nullptr};
  cudaEventCreate(&r.e0); cudaEventCreate(&r.e1);
  cudaEventRecord(r.e0, s);
  p->recs.push_back(r);
}
void prof_end(Prof* p, cudaStream_t s) { cudaEventRecord(p->recs.back().e1, s); }
static void prof_collect(Prof* p) {     // caller has synchronised the stream
  for (ProfRec& r : p->recs) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, r.e0, r.e1);
    cudaEventDestroy(r.e0); cudaEventDestroy(r.e1);
    ProfAgg* a = nullptr;
    for (ProfAgg& x : p->agg) if (std::strcmp(x.name, r.name) == 0) { a = &x; break; }
    if (!a) { p->agg.push_back(ProfAgg{r.name, 0, 0.0, 0.0}); a = &p->agg.back(); }
    a->launches += 1; a->ms += ms; a->bytes += r.bytes;
  }
  p->recs.clear();
}
struct Seen { std::vector<const char*> names; };
void seen_add(Seen* s, const char* inst) {
  for (const char* n : s->names) if (n == inst || std::strcmp(n, inst) == 0) return;
  s->names.push_back(inst);
}
}  // namespace fs

struct fs_grid {
  fs_params P;
  int device = 0;                       // the CUDA device the workspace lives on; every entry point runs on it
  fs::Prof prof; bool profiling = false;
  fs::Seen seen;
  std::vector<double> yf;
  bool f64 = true;
  int bx = 0, by = 0, bz = 0, nxu = 0, nyv = 0, nzw = 0;
  double hx = 0, hy = 0, hz = 0;
  bool uniform_y = true;
  cudaStream_t stream = nullptr, cap = nullptr, cap2 = nullptr;
  char* ws = nullptr; size_t ws_bytes = 0;
  Ctx<float> cf; Ctx<double> cd;
  MgCtx<float> mf; MgCtx<double> md;
  IbmCtx ib;
  Scalars* S = nullptr;
  size_t nU = 0, nV = 0, nW = 0, nP = 0;
  void* fld[8] = {nullptr};           // device pointers of FS_U..FS_HW (+ none for FS_DIV)
  // graphs
  cudaGraphExec_t step_exec = nullptr, poisson_exec = nullptr;
  int step_fixed = 0, step_body = 0, poisson_fixed = 0, poisson_body = 0;
  long long fixed_launches = 0, body_iters_poisson = 0;
  int nl = 0; bool indexed = false;
  void* bak[7] = {nullptr};           // strong coupling: u, v, w, p, H^{n-1} of time level n (device, T)
  double beam_coef[4] = {0, 0, 0, 0}; // flexible beam: alpha, beta (Eq. 16), omega_1, omega_2 (Eq. 17)
  int last_sweeps = 1; double last_xi = 0.0; long long last_iters = 0;
};

namespace {

// Every entry point that takes an fs_grid makes the grid's device current for the call and restores the caller's
// device afterwards, so grids on several GPUs can be driven from one thread (replicas).
struct DeviceGuard {
  int prev = -1; bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; prev = -1; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define GUARD(g) DeviceGuard guard_((g)->device); if (!guard_.ok) return FS_ERR_CUDA

struct Bump {
  char* base; size_t off;
  template <class T> T* take(size_t n) {
    off = (off + 255) & ~size_t(255);
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
};

int mg_levels(int nx, int ny, int nz) {
  int L = 1;
  while (nx % 2 == 0 && ny % 2 == 0 && nz % 2 == 0 && std::min(nx, std::min(ny, nz)) / 2 >= 4) { nx /= 2; ny /= 2; nz /= 2; ++L; }
  return L;
}

fs_status validate(const fs_params* p) {
  if (!p) return FS_ERR_INVALID_ARG;
  if (p->nx < 2 || p->ny < 2 || p->nz < 2) return FS_ERR_INVALID_ARG;
  if (!(p->dt > 0) || !(p->rho > 0) || !(p->lx > 0) || !(p->ly > 0) || !(p->lz > 0) || !(p->nu >= 0)) return FS_ERR_INVALID_ARG;
  if (p->dtype != FS_F32 && p->dtype != FS_F64) return FS_ERR_INVALID_ARG;
  if (p->max_markers < 0 || p->max_iter < 0 || !(p->rtol >= 0)) return FS_ERR_INVALID_ARG;
  if (p->max_beam_nodes < 0 || p->max_beam_nodes == 1 || p->max_beam_nodes > kMaxBeamNodes) return FS_ERR_INVALID_ARG;
  for (int f = 0; f < 6; ++f) if ((int)p->bc[f] < 0 || (int)p->bc[f] > 4) return FS_ERR_INVALID_ARG;
  for (int d = 0; d < 3; ++d)
    if ((p->bc[2 * d] == FS_BC_PERIODIC) != (p->bc[2 * d + 1] == FS_BC_PERIODIC)) return FS_ERR_INVALID_ARG;
  if ((long long)(p->nx + 1) * (p->ny + 1) * (p->nz + 1) > (1LL << 31) - 1) return FS_ERR_UNSUPPORTED;   // int32 cell keys, 32-bit field offsets
  if ((long long)((p->nx + 29) / 30) * ((p->ny + 3) / 4) > kMaxPartials) return FS_ERR_UNSUPPORTED;   // one reduction partial per xy tile
  if (p->yf) for (int j = 0; j < p->ny; ++j) if (!(p->yf[j + 1] > p->yf[j])) return FS_ERR_INVALID_ARG;
  if ((int)p->convection < 0 || (int)p->convection > 1) return FS_ERR_INVALID_ARG;
  if ((int)p->time_scheme < 0 || (int)p->time_scheme > 2) return FS_ERR_INVALID_ARG;
  if (!(p->cs >= 0.0)) return FS_ERR_INVALID_ARG;
  if ((int)p->precond < 0 || (int)p->precond > 2 || (int)p->delta < 0 || (int)p->delta > 1) return FS_ERR_INVALID_ARG;
  if (p->precond == FS_PC_GMG) {
    const double hx = p->lx / p->nx, hy = p->ly / p->ny, hz = p->lz / p->nz;
    if (p->yf || std::fabs(hx - hy) > 1e-12 * hx || std::fabs(hx - hz) > 1e-12 * hx) return FS_ERR_UNSUPPORTED;   // uniform, isotropic
    if (p->mg_nu1 < 0 || p->mg_nu2 < 0 || p->mg_coarse_sweeps < 0) return FS_ERR_INVALID_ARG;
    if (mg_levels(p->nx, p->ny, p->nz) > kMaxLevels) return FS_ERR_UNSUPPORTED;
  }
  return FS_OK;
}

template <class T> Ctx<T>& ctx(fs_grid* g);
template <> Ctx<float>& ctx<float>(fs_grid* g) { return g->cf; }
template <> Ctx<double>& ctx<double>(fs_grid* g) { return g->cd; }
template <class T> MgCtx<T>& mgc(fs_grid* g);
template <> MgCtx<float>& mgc<float>(fs_grid* g) { return g->mf; }
template <> MgCtx<double>& mgc<double>(fs_grid* g) { return g->md; }

// Carves the workspace (base == nullptr: size pass only).
template <class T> size_t carve(fs_grid* g, char* base) {
  const fs_params& P = g->P;
  Ctx<T>& c = ctx<T>(g);
  MgCtx<T>& mg = mgc<T>(g);
  Bump b{base, 0};
  const int ny = P.ny;
  g->S = b.take<Scalars>(1);
  c.S = g->S;
  c.partials = b.take<double>((size_t)kRedSlots * kMaxPartials);
  T* dy = b.take<T>(ny + 2); T* idy = b.take<T>(ny + 2); T* idyc = b.take<T>(ny + 1);
  T* wyl = b.take<T>(ny + 1); T* wyh = b.take<T>(ny + 1); T* cyl = b.take<T>(ny); T* cyh = b.take<T>(ny);
  double* dy64 = b.take<double>(ny);
  c.dy = dy; c.idy = idy; c.idyc = idyc; c.wyl = wyl; c.wyh = wyh; c.cyl = cyl; c.cyh = cyh; c.dy64 = dy64;
  c.u = b.take<T>(g->nU); c.v = b.take<T>(g->nV); c.w = b.take<T>(g->nW);
  c.us = b.take<T>(g->nU); c.vs = b.take<T>(g->nV); c.ws = b.take<T>(g->nW);
  c.hu = b.take<T>(g->nU); c.hv = b.take<T>(g->nV); c.hw = b.take<T>(g->nW);
  c.p = b.take<T>(g->nP); c.r = b.take<T>(g->nP); c.d = b.take<T>(g->nP); c.d2 = b.take<T>(g->nP); c.q = b.take<T>(g->nP); c.bh = b.take<T>(g->nP);
  c.z = nullptr; c.r2 = nullptr;
  c.q0u = c.q0v = c.q0w = nullptr;
  for (int a = 0; a < 7; ++a) g->bak[a] = nullptr;
  if (P.coupling_max_iters > 1) {
    const size_t nb[7] = {g->nU, g->nV, g->nW, g->nP, g->nU, g->nV, g->nW};
    for (int a = 0; a < 7; ++a) g->bak[a] = b.take<T>(nb[a]);
  }
  if (P.time_scheme == FS_TIME_RK3) { c.q0u = b.take<T>(g->nU); c.q0v = b.take<T>(g->nV); c.q0w = b.take<T>(g->nW); }
  mg.nlev = 0;
  if (P.precond == FS_PC_GMG) {
    c.z = b.take<T>(g->nP);
    if (P.mg_nu1 == 2 && P.mg_nu2 == 2) c.r2 = b.take<T>(g->nP);   // second residual buffer of the fused update (k_mg_down<UPD>)
    mg.nlev = mg_levels(P.nx, P.ny, P.nz);
    mg.nu1 = P.mg_nu1; mg.nu2 = P.mg_nu2; mg.coarse_sweeps = P.mg_coarse_sweeps; mg.omega = P.mg_omega;
    mg.bd = (g->bx ? 1 : 0) | (g->by ? 2 : 0) | (g->bz ? 4 : 0);
    int nx = P.nx, nyy = P.ny, nz = P.nz; double h = g->hx;
    for (int l = 0; l < mg.nlev; ++l) {
      MgLevel& V = mg.lev[l];
      V.nx = nx; V.ny = nyy; V.nz = nz; V.h = h;
      const size_t N = (size_t)nx * nyy * nz;
      V.t = b.take<T>(N);
      V.e = l == 0 ? nullptr : (void*)b.take<T>(N);
      V.g = l == 0 ? nullptr : (void*)b.take<T>(N);
      nx /= 2; nyy /= 2; nz /= 2; h *= 2.0;
    }
  }
  IbmCtx& ib = g->ib;
  const size_t M = (size_t)P.max_markers;
  ib.X = b.take<double>(3 * M); ib.Ub = b.take<double>(3 * M); ib.dV = b.take<double>(M);
  ib.Fl = b.take<double>(3 * M); ib.Ul = b.take<double>(3 * M); ib.wts = b.take<double>(36 * M);
  ib.base = b.take<int>(9 * M); ib.perm = b.take<int>(M); ib.keys = b.take<int>(M); ib.keys_raw = b.take<int>(M);
  ib.seg = b.take<int>(M + 1); ib.flags = b.take<int>(M);
  ib.bw = ib.bv = ib.ba = ib.bw0 = ib.bv0 = ib.ba0 = ib.bQ = ib.bL = ib.bM = ib.bC = ib.Xref = nullptr; ib.mnode = ib.nstart = ib.nlist = nullptr;
  if (P.max_beam_nodes > 0) {             // flexible beam: state, band matrices, reference marker positions, node <-> marker maps
    const size_t nd = 2 * (size_t)(P.max_beam_nodes - 1);
    ib.bw = b.take<double>(nd); ib.bv = b.take<double>(nd); ib.ba = b.take<double>(nd);
    ib.bw0 = b.take<double>(nd); ib.bv0 = b.take<double>(nd); ib.ba0 = b.take<double>(nd); ib.bQ = b.take<double>(nd);
    ib.bL = b.take<double>(4 * nd); ib.bM = b.take<double>(7 * nd); ib.bC = b.take<double>(7 * nd);
    ib.Xref = b.take<double>(3 * M); ib.mnode = b.take<int>(M); ib.nstart = b.take<int>((size_t)P.max_beam_nodes + 1); ib.nlist = b.take<int>(M);
  }
  ib.eps = ib.mu = ib.mv = ib.mw = nullptr; ib.ibu = ib.ibv = ib.ibw = nullptr;
  if (P.solid_mask) {                     // eps-mask IBM: cell mask, face classes, and (with markers) the u_IB scratch fields
    ib.eps = b.take<unsigned char>(g->nP);
    ib.mu = b.take<unsigned char>(g->nU); ib.mv = b.take<unsigned char>(g->nV); ib.mw = b.take<unsigned char>(g->nW);
    if (M > 0) { ib.ibu = b.take<T>(g->nU); ib.ibv = b.take<T>(g->nV); ib.ibw = b.take<T>(g->nW); }
  }
  return (b.off + 255) & ~size_t(255);
}

void init_dims(fs_grid* g) {
  const fs_params& P = g->P;
  g->f64 = P.dtype == FS_F64;
  g->bx = P.bc[0] != FS_BC_PERIODIC; g->by = P.bc[2] != FS_BC_PERIODIC; g->bz = P.bc[4] != FS_BC_PERIODIC;
  g->nxu = P.nx + g->bx; g->nyv = P.ny + g->by; g->nzw = P.nz + g->bz;
  g->hx = P.lx / P.nx; g->hy = P.ly / P.ny; g->hz = P.lz / P.nz;
  g->uniform_y = P.yf == nullptr;
  g->nU = (size_t)g->nxu * P.ny * P.nz; g->nV = (size_t)P.nx * g->nyv * P.nz; g->nW = (size_t)P.nx * P.ny * g->nzw;
  g->nP = (size_t)P.nx * P.ny * P.nz;
}

// Host-side metric tables (SURVEY 8(c) "Grid"), uploaded once.
template <class T> fs_status upload_metrics(fs_grid* g) {
  const fs_params& P = g->P;
  Ctx<T>& c = ctx<T>(g);
  const int ny = P.ny;
  std::vector<double> dy(ny);
  for (int j = 0; j < ny; ++j) dy[j] = g->uniform_y ? g->hy : g->yf[j + 1] - g->yf[j];
  auto DY = [&](int j) {            // mirrored ghost at a bounded end, wrapped when periodic
    if (j < 0) return g->by ? dy[0] : dy[(j % ny + ny) % ny];
    if (j >= ny) return g->by ? dy[ny - 1] : dy[j % ny];
    return dy[j];
  };
  auto DYC = [&](int j) { return 0.5 * (DY(j - 1) + DY(j)); };
  std::vector<T> hdy(ny + 2), hidy(ny + 2), hidyc(ny + 1), hwl(ny + 1), hwh(ny + 1), hcl(ny), hch(ny);
  for (int j = -1; j <= ny; ++j) { hdy[j + 1] = (T)DY(j); hidy[j + 1] = (T)(1.0 / DY(j)); }
  for (int j = 0; j <= ny; ++j) {
    hidyc[j] = (T)(1.0 / DYC(j));
    const double dm = DY(j - 1), dp = DY(j);
    hwl[j] = (T)(dp / (dm + dp)); hwh[j] = (T)(dm / (dm + dp));
  }
  double sdy = 0.0;
  for (int j = 0; j < ny; ++j) {
    hcl[j] = (g->by && j == 0) ? (T)0 : (T)(1.0 / DYC(j));
    hch[j] = (g->by && j == ny - 1) ? (T)0 : (T)(1.0 / DYC(j + 1));
    sdy += dy[j];
  }
  CK(cudaMemcpyAsync((void*)c.dy, hdy.data(), sizeof(T) * (ny + 2), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync((void*)c.idy, hidy.data(), sizeof(T) * (ny + 2), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync((void*)c.idyc, hidyc.data(), sizeof(T) * (ny + 1), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync((void*)c.wyl, hwl.data(), sizeof(T) * (ny + 1), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync((void*)c.wyh, hwh.data(), sizeof(T) * (ny + 1), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync((void*)c.cyl, hcl.data(), sizeof(T) * ny, cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync((void*)c.cyh, hch.data(), sizeof(T) * ny, cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync((void*)c.dy64, dy.data(), sizeof(double) * ny, cudaMemcpyHostToDevice, g->stream));
  Scalars hs; std::memset(&hs, 0, sizeof hs);
  hs.sum_dy = sdy * (double)P.nx * (double)P.nz;
  hs.max_iter = P.max_iter; hs.rtol = P.rtol; hs.rho_prev = 1.0; hs.dq = 1.0;
  hs.dt = hs.dt_prev = P.dt; hs.conv_acc = 1;
  CK(cudaMemcpyAsync(g->S, &hs, sizeof hs, cudaMemcpyHostToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  // constants
  c.nx = P.nx; c.ny = P.ny; c.nz = P.nz; c.bx = g->bx; c.by = g->by; c.bz = g->bz;
  c.nxu = g->nxu; c.nyv = g->nyv; c.nzw = g->nzw;
  for (int f = 0; f < 6; ++f) { c.bc[f] = (int)P.bc[f]; for (int a = 0; a < 3; ++a) c.bcv[f][a] = P.bc_vel[f][a]; }
  c.hx = g->hx; c.hy = g->hy; c.hz = g->hz; c.dt = P.dt; c.rho = P.rho; c.nu = P.nu;
  for (int a = 0; a < 3; ++a) c.g[a] = P.body_force[a];
  c.x0 = P.x0; c.y0 = P.y0; c.z0 = P.z0;
  c.cs = P.cs; c.wall_model = P.wall_model;
  c.cfl = P.cfl; c.hmin = std::min(g->hx, g->hz);
  for (int j = 0; j < ny; ++j) c.hmin = std::min(c.hmin, dy[j]);
  c.ihx = (T)(1.0 / g->hx); c.ihz = (T)(1.0 / g->hz);
  c.ihx2 = (T)(1.0 / (g->hx * g->hx)); c.ihz2 = (T)(1.0 / (g->hz * g->hz));
  c.time_scheme = (int)P.time_scheme; c.precond = (int)P.precond; c.warm_start = P.warm_start; c.delta = (int)P.delta;
  c.uniform_y = g->uniform_y; c.convection = (int)P.convection; c.seed = P.seed; c.inflow_noise = P.inflow_noise;
  return FS_OK;
}

void init_ibm(fs_grid* g) {
  const fs_params& P = g->P;
  IbmCtx& ib = g->ib;
  ib.n = 0; ib.delta = (int)P.delta; ib.sw = P.delta == FS_DELTA_ROMA3 ? 3 : 4;
  const double o[3] = {P.x0, P.y0, P.z0}, h[3] = {g->hx, g->hy, g->hz};
  for (int d = 0; d < 3; ++d) {
    ib.o[d] = o[d]; ib.inv[d] = 1.0 / h[d];
    for (int c = 0; c < 3; ++c) ib.org[c][d] = d == c ? o[d] : o[d] + 0.5 * h[d];
  }
  ib.ivol = 1.0 / (g->hx * g->hy * g->hz);
  ib.has_body = 0; ib.dof = 0; ib.bm = 1.0; ib.bc = 0.0; ib.bk = 0.0;
  ib.has_mask = 0; ib.uc[0] = ib.uc[1] = ib.uc[2] = 0.0;
  ib.strong = 0;
  ib.has_beam = 0; ib.nbn = 0; ib.ndof = 0; ib.bnrm[0] = ib.bnrm[1] = 0.0;
  for (int a = 0; a < 6; ++a) ib.nk[a] = 0.0;
}


// ---- the step as three kernel sequences: before the PCG loop, the loop body, after the loop ---------
template <class T> int enqueue_pre(fs_grid* g, const Launch& L, bool poisson) {
  Ctx<T>& c = ctx<T>(g);
  int n = 0;
  if (poisson) {
    n += launch_rhs_from_b<T>(c, c.vs, L);
  } else {
    n += launch_momentum<T>(c, L);
    if (g->ib.has_mask) {                 // the paper's eps-mask forcing (markers only carry the structure velocity to the IB points)
      if (g->ib.n > 0 && (g->ib.has_body || g->ib.has_beam || !g->indexed)) n += launch_ibm_index<T>(c, g->ib, L);
      n += launch_mask_forcing<T>(c, g->ib, L);
    } else if (g->ib.n > 0) {
      if (g->ib.has_body || g->ib.has_beam || !g->indexed) n += launch_ibm_index<T>(c, g->ib, L);
      n += launch_ibm_interpolate<T>(c, g->ib, c.us, c.vs, c.ws, g->ib.Ul, L);
      n += launch_ibm_force<T>(c, g->ib, L);
      n += launch_ibm_spread<T>(c, g->ib, g->ib.Fl, c.us, c.vs, c.ws, -1.0, L);
    }
    n += launch_flux_correction<T>(c, L);
    n += launch_div_rhs<T>(c, L);
  }
  n += launch_pcg_init<T>(c, L, poisson);
  return n;
}
template <class T> int enqueue_body(fs_grid* g, const Launch& L) { return launch_pcg_body<T>(ctx<T>(g), mgc<T>(g), L); }
// stage / nstages: Runge-Kutta (FS_TIME_RK3) runs pre / loop / post three times per step, the other schemes once
template <class T> int enqueue_post(fs_grid* g, const Launch& L, bool poisson, int stage, int nstages) {
  Ctx<T>& c = ctx<T>(g);
  int n = launch_pcg_finish<T>(c, L);
  if (poisson) n += launch_true_residual<T>(c, L);
  else {
    n += launch_project<T>(c, L);
    if (nstages > 1) n += launch_stage_end<T>(c, stage, L);
    if (stage == nstages - 1) {
      if (g->ib.has_beam) n += launch_beam_step<T>(c, g->ib, L);
      n += launch_step_end<T>(c, g->ib, L);
    }
  }
  return n;
}
inline int num_stages(const fs_grid* g, bool poisson) { return (!poisson && g->P.time_scheme == FS_TIME_RK3) ? 3 : 1; }

template <class T> fs_status build_graph_impl(fs_grid* g, bool poisson, cudaGraphExec_t* out, int* n_fixed, int* n_body, bool* body_open) {
  cudaStream_t s = g->cap;
  cudaStreamCaptureStatus st; cudaGraph_t graph = nullptr; const cudaGraphNode_t* deps = nullptr; size_t nd = 0;
  CK(cudaStreamGetCaptureInfo_v2(s, &st, nullptr, &graph, &deps, &nd));
  const int nst = num_stages(g, poisson);
  int nfix = 0, nbody = 0;
  if (!poisson) { Launch L0{s, 0, 0, nullptr, &g->seen}; nfix += launch_step_begin<T>(ctx<T>(g), L0); CK(cudaGetLastError()); }
  const bool coop = pcg_coop_applies<T>(ctx<T>(g));    // L2-sized grids: the whole solve is one persistent cooperative kernel
  for (int stage = 0; stage < nst && coop; ++stage) {
    Launch L{s, 0, 0, nullptr, &g->seen};
    nfix += enqueue_pre<T>(g, L, poisson);
    nfix += launch_pcg_coop<T>(ctx<T>(g), L);
    nfix += enqueue_post<T>(g, L, poisson, stage, nst);
    CK(cudaGetLastError());
  }
  for (int stage = 0; stage < nst && !coop; ++stage) {  // one conditional WHILE node (one PCG solve) per stage
    cudaGraphConditionalHandle h;
    CK(cudaGraphConditionalHandleCreate(&h, graph, 0, cudaGraphCondAssignDefault));
    Launch L{s, h, 1, nullptr, &g->seen};
    nfix += enqueue_pre<T>(g, L, poisson);
    CK(cudaGetLastError());
    CK(cudaStreamGetCaptureInfo_v2(s, &st, nullptr, &graph, &deps, &nd));
    cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
    np.conditional.handle = h; np.conditional.type = cudaGraphCondTypeWhile; np.conditional.size = 1;
    cudaGraphNode_t node;
    CK(cudaGraphAddNode(&node, graph, deps, nd, &np));
    cudaGraph_t body = np.conditional.phGraph_out[0];
    CK(cudaStreamBeginCaptureToGraph(g->cap2, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    *body_open = true;
    Launch Lb{g->cap2, h, 1, nullptr, &g->seen};
    nbody = enqueue_body<T>(g, Lb);
    CK(cudaGetLastError());
    cudaGraph_t tmp = nullptr;
    *body_open = false;
    CK(cudaStreamEndCapture(g->cap2, &tmp));
    CK(cudaStreamUpdateCaptureDependencies(s, &node, 1, cudaStreamSetCaptureDependencies));
    nfix += enqueue_post<T>(g, L, poisson, stage, nst);
    CK(cudaGetLastError());
  }
  *n_fixed = nfix; *n_body = nbody;
  return FS_OK;
}

// Captures pre-loop kernels, the conditional WHILE node with the PCG body, and the post-loop kernels into one
// graph.  Whatever fails in between, both capture streams are taken out of capture mode and the partial graph
// is destroyed before the error is returned, so a later call starts from a clean state.
template <class T> fs_status build_graph(fs_grid* g, bool poisson, cudaGraphExec_t* out, int* n_fixed, int* n_body) {
  CK(cudaStreamBeginCapture(g->cap, cudaStreamCaptureModeRelaxed));
  bool body_open = false;
  fs_status st = build_graph_impl<T>(g, poisson, out, n_fixed, n_body, &body_open);
  cudaGraph_t graph = nullptr, tmp = nullptr;
  if (body_open) cudaStreamEndCapture(g->cap2, &tmp);           // the body graph is owned by the conditional node
  const cudaError_t ec = cudaStreamEndCapture(g->cap, &graph);
  if (st == FS_OK && ec != cudaSuccess) { std::fprintf(stderr, "libfs: graph capture failed: %s\n", cudaGetErrorString(ec)); st = FS_ERR_CUDA; }
  if (st == FS_OK) {
    if (*out) { cudaGraphExecDestroy(*out); *out = nullptr; }
    if (cudaGraphInstantiate(out, graph, 0) != cudaSuccess) { *out = nullptr; st = FS_ERR_CUDA; }
  }
  if (graph) cudaGraphDestroy(graph);
  if (st != FS_OK) cudaGetLastError();                          // clear the sticky-free error state of the failed capture
  return st;
}

// FS_EXEC_STREAM: same kernels, launched directly; the host polls the done flag between chunks.
template <class T> fs_status run_stream(fs_grid* g, bool poisson, int* n_fixed, int* n_body) {
  Launch L{g->stream, 0, 0, g->profiling ? &g->prof : nullptr, &g->seen};
  const int nst = num_stages(g, poisson);
  int nfix = 0, nbody = 0;
  if (!poisson) nfix += launch_step_begin<T>(ctx<T>(g), L);
  const bool coop = pcg_coop_applies<T>(ctx<T>(g));
  for (int stage = 0; stage < nst; ++stage) {
    nfix += enqueue_pre<T>(g, L, poisson);
    if (coop) nfix += launch_pcg_coop<T>(ctx<T>(g), L);
    else for (;;) {
      int done = 0;
      CK(cudaMemcpyAsync(&done, &g->S->done, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
      CK(cudaStreamSynchronize(g->stream));
      if (done) break;
      for (int a = 0; a < 4; ++a) nbody = enqueue_body<T>(g, L);
    }
    nfix += enqueue_post<T>(g, L, poisson, stage, nst);
  }
  CK(cudaGetLastError());
  *n_fixed = nfix; *n_body = nbody;
  return FS_OK;
}

template <class T> fs_status run_once(fs_grid* g, bool poisson) {
  if (g->P.exec_mode == FS_EXEC_STREAM || g->profiling) {
    int nf = 0, nb = 0;
    fs_status st = run_stream<T>(g, poisson, &nf, &nb);
    if (st != FS_OK) return st;
    (poisson ? g->poisson_fixed : g->step_fixed) = nf; (poisson ? g->poisson_body : g->step_body) = nb;
  } else {
    cudaGraphExec_t* ex = poisson ? &g->poisson_exec : &g->step_exec;
    if (!*ex) {
      fs_status st = build_graph<T>(g, poisson, ex, poisson ? &g->poisson_fixed : &g->step_fixed, poisson ? &g->poisson_body : &g->step_body);
      if (st != FS_OK) return st;
    }
    CK(cudaGraphLaunch(*ex, g->stream));
  }
  g->fixed_launches += poisson ? g->poisson_fixed : g->step_fixed;
  if (!poisson && g->ib.n > 0) g->indexed = true;
  return FS_OK;
}

// One time step.  Weak coupling / no body: one run of the step graph.  Strong coupling (Algorithm 1; reading
// N2-1): the fluid fields of time level n are kept, every sweep restarts from them with the structure's latest iterate
// (the markers already reflect it: k_step_end moved them), the structure is advanced from its time-level-n state with the
// sweep's force, and the host -- the loop is data dependent by nature -- stops on xi = ||(w^k - w^{k-1}) / w^{k-1}||^2.
template <class T> fs_status advance_step(fs_grid* g) {
  g->last_sweeps = 1; g->last_xi = 0.0; g->last_iters = -1;
  const int N = ((g->ib.has_body || g->ib.has_beam) && g->P.coupling_max_iters > 1) ? g->P.coupling_max_iters : 1;
  if (N == 1) return run_once<T>(g, false);
  if (g->ib.has_beam) {                   // the beam's state of time level n: every sweep's Newmark step starts there
    const size_t nb = (size_t)g->ib.ndof * sizeof(double);
    CK(cudaMemcpyAsync(g->ib.bw0, g->ib.bw, nb, cudaMemcpyDeviceToDevice, g->stream));
    CK(cudaMemcpyAsync(g->ib.bv0, g->ib.bv, nb, cudaMemcpyDeviceToDevice, g->stream));
    CK(cudaMemcpyAsync(g->ib.ba0, g->ib.ba, nb, cudaMemcpyDeviceToDevice, g->stream));
  }
  Ctx<T>& c = ctx<T>(g);
  Scalars h0;
  CK(cudaMemcpyAsync(&h0, g->S, sizeof(Scalars), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  CK(cudaMemcpyAsync(g->S->body_disp0, h0.body_disp, 3 * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(g->S->body_vel0, h0.body_vel, 3 * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  T* fld[7] = {c.u, c.v, c.w, c.p, c.hu, c.hv, c.hw};
  const size_t nb[7] = {g->nU, g->nV, g->nW, g->nP, g->nU, g->nV, g->nW};
  for (int a = 0; a < 7; ++a) CK(cudaMemcpyAsync(g->bak[a], fld[a], nb[a] * sizeof(T), cudaMemcpyDeviceToDevice, g->stream));
  double prev[3] = {h0.body_disp[0], h0.body_disp[1], h0.body_disp[2]};
  long long iters = 0; double xi = 0.0; int k = 1;
  for (k = 1; k <= N; ++k) {
    if (k > 1) {
      for (int a = 0; a < 7; ++a) CK(cudaMemcpyAsync(fld[a], g->bak[a], nb[a] * sizeof(T), cudaMemcpyDeviceToDevice, g->stream));
      CK(cudaMemcpyAsync(&g->S->step, &h0.step, sizeof(long long), cudaMemcpyHostToDevice, g->stream));
      CK(cudaMemcpyAsync(&g->S->have_hist, &h0.have_hist, sizeof(int), cudaMemcpyHostToDevice, g->stream));
      CK(cudaMemcpyAsync(&g->S->time, &h0.time, sizeof(double), cudaMemcpyHostToDevice, g->stream));
      CK(cudaMemcpyAsync(&g->S->dt_prev, &h0.dt_prev, sizeof(double), cudaMemcpyHostToDevice, g->stream));
    }
    fs_status st = run_once<T>(g, false); if (st != FS_OK) return st;
    Scalars hs;
    CK(cudaMemcpyAsync(&hs, g->S, sizeof(Scalars), cudaMemcpyDeviceToHost, g->stream));
    CK(cudaStreamSynchronize(g->stream));
    iters += hs.iter;
    xi = 0.0;
    for (int a = 0; a < 3; ++a) if (g->ib.has_body && (g->ib.dof & (1 << a))) {
      const double dw = hs.body_disp[a] - prev[a];
      if (!(dw == 0.0 && prev[a] == 0.0)) xi += (dw / prev[a]) * (dw / prev[a]);
      prev[a] = hs.body_disp[a];
    }
    if (g->ib.has_beam) xi = hs.beam_xi;   // summed over the degrees of freedom by k_beam_step
    if (xi < g->P.coupling_tol) break;
  }
  g->last_sweeps = k > N ? N : k; g->last_xi = xi; g->last_iters = iters;
  return FS_OK;
}

void invalidate(fs_grid* g) {
  if (g->step_exec) { cudaGraphExecDestroy(g->step_exec); g->step_exec = nullptr; }
}

fs_status read_scalars(fs_grid* g, Scalars* hs) {
  CK(cudaMemcpyAsync(hs, g->S, sizeof(Scalars), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

// copy a T-typed device field to / from a user buffer of `dtype`, host or device
template <class T> fs_status copy_out(fs_grid* g, const T* dev, size_t n, void* dst, fs_dtype dtype, int on_device) {
  const bool same = (dtype == FS_F64) == (sizeof(T) == 8);
  if (on_device) {
    if (same) CK(cudaMemcpyAsync(dst, dev, n * sizeof(T), cudaMemcpyDeviceToDevice, g->stream));
    else if (dtype == FS_F64) launch_convert<T, double>(dev, (double*)dst, (long long)n, g->stream);
    else launch_convert<T, float>(dev, (float*)dst, (long long)n, g->stream);
    CK(cudaStreamSynchronize(g->stream));
    return FS_OK;
  }
  if (same) { CK(cudaMemcpyAsync(dst, dev, n * sizeof(T), cudaMemcpyDeviceToHost, g->stream)); CK(cudaStreamSynchronize(g->stream)); return FS_OK; }
  std::vector<T> tmp(n);
  CK(cudaMemcpyAsync(tmp.data(), dev, n * sizeof(T), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if (dtype == FS_F64) { double* o = (double*)dst; for (size_t q = 0; q < n; ++q) o[q] = (double)tmp[q]; }
  else { float* o = (float*)dst; for (size_t q = 0; q < n; ++q) o[q] = (float)tmp[q]; }
  return FS_OK;
}
template <class T> fs_status copy_in(fs_grid* g, T* dev, size_t n, const void* src, fs_dtype dtype, int on_device) {
  const bool same = (dtype == FS_F64) == (sizeof(T) == 8);
  if (on_device) {
    if (same) CK(cudaMemcpyAsync(dev, src, n * sizeof(T), cudaMemcpyDeviceToDevice, g->stream));
    else if (dtype == FS_F64) launch_convert<double, T>((const double*)src, dev, (long long)n, g->stream);
    else launch_convert<float, T>((const float*)src, dev, (long long)n, g->stream);
    CK(cudaStreamSynchronize(g->stream));
    return FS_OK;
  }
  if (same) { CK(cudaMemcpyAsync(dev, src, n * sizeof(T), cudaMemcpyHostToDevice, g->stream)); CK(cudaStreamSynchronize(g->stream)); return FS_OK; }
  std::vector<T> tmp(n);
  if (dtype == FS_F64) { const double* i = (const double*)src; for (size_t q = 0; q < n; ++q) tmp[q] = (T)i[q]; }
  else { const float* i = (const float*)src; for (size_t q = 0; q < n; ++q) tmp[q] = (T)i[q]; }
  CK(cudaMemcpyAsync(dev, tmp.data(), n * sizeof(T), cudaMemcpyHostToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

template <class T> T* field_ptr(fs_grid* g, fs_field f, size_t* n) {
  Ctx<T>& c = ctx<T>(g);
  switch (f) {
    case FS_U: *n = g->nU; return c.u;   case FS_V: *n = g->nV; return c.v;   case FS_W: *n = g->nW; return c.w;
    case FS_P: *n = g->nP; return c.p;
    case FS_HU: *n = g->nU; return c.hu; case FS_HV: *n = g->nV; return c.hv; case FS_HW: *n = g->nW; return c.hw;
    case FS_DIV: *n = g->nP; return c.q;
    default: *n = 0; return nullptr;
  }
}

template <class T> fs_status fields_io(fs_grid* g, fs_field f, void* buf, fs_dtype dtype, int on_device, bool set) {
  size_t n; T* dev = field_ptr<T>(g, f, &n);
  if (!dev) return FS_ERR_INVALID_ARG;
  if (set) {
    if (f == FS_DIV) return FS_ERR_INVALID_ARG;
    return copy_in<T>(g, dev, n, buf, dtype, on_device);
  }
  if (f == FS_DIV) {
    Ctx<T>& c = ctx<T>(g);
    Launch L{g->stream, 0, 0, nullptr, &g->seen};
    launch_divergence<T>(c, c.u, c.v, c.w, c.q, L);
    CK(cudaGetLastError());
  }
  return copy_out<T>(g, dev, n, buf, dtype, on_device);
}

template <class T> fs_status poisson_impl(fs_grid* g, const void* rhs, void* p_inout, fs_dtype dtype, int on_device, fs_poisson_info* info) {
  Ctx<T>& c = ctx<T>(g);
  const size_t N = g->nP;
  // the flow state's pressure is parked in us (scratch between steps); rhs goes to vs
  CK(cudaMemcpyAsync(c.us, c.p, N * sizeof(T), cudaMemcpyDeviceToDevice, g->stream));
  fs_status st = copy_in<T>(g, c.vs, N, rhs, dtype, on_device); if (st != FS_OK) return st;
  st = copy_in<T>(g, c.p, N, p_inout, dtype, on_device); if (st != FS_OK) return st;
  st = run_once<T>(g, true); if (st != FS_OK) return st;
  Scalars hs; st = read_scalars(g, &hs); if (st != FS_OK) return st;
  g->body_iters_poisson += hs.body_runs;
  st = copy_out<T>(g, c.p, N, p_inout, dtype, on_device); if (st != FS_OK) return st;
  CK(cudaMemcpyAsync(c.p, c.us, N * sizeof(T), cudaMemcpyDeviceToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if (info) {
    info->iters = hs.iter; info->converged = hs.converged;
    info->rel_residual = hs.bnorm2 > 0 ? std::sqrt(hs.rr / hs.bnorm2) : 0.0;
    info->true_rel_residual = hs.bnorm2 > 0 ? std::sqrt(hs.true_rr / hs.bnorm2) : 0.0;
  }
  return hs.converged ? FS_OK : FS_ERR_NOT_CONVERGED;
}

}  // namespace

// ======================================================================================================
extern "C" {

const char* fs_status_string(fs_status s) {
  switch (s) {
    case FS_OK: return "ok"; case FS_ERR_INVALID_ARG: return "invalid argument"; case FS_ERR_BAD_STATE: return "bad state";
    case FS_ERR_OOM: return "out of memory"; case FS_ERR_CUDA: return "CUDA error"; case FS_ERR_NOT_CONVERGED: return "PCG not converged";
    case FS_ERR_UNSUPPORTED: return "unsupported configuration";
  }
  return "unknown";
}

fs_status fs_workspace_bytes(const fs_params* params, size_t* bytes) {
  if (!bytes) return FS_ERR_INVALID_ARG;
  fs_status st = validate(params); if (st != FS_OK) return st;
  fs_grid tmp; tmp.P = *params; init_dims(&tmp);
  *bytes = tmp.f64 ? carve<double>(&tmp, nullptr) : carve<float>(&tmp, nullptr);
  return FS_OK;
}

fs_status fs_grid_create(const fs_params* params, void* workspace, size_t bytes, void* cuda_stream, fs_grid** out) {
  if (!out || !workspace) return FS_ERR_INVALID_ARG;
  fs_status st = validate(params); if (st != FS_OK) return st;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return FS_ERR_INVALID_ARG;
  fs_grid* g = new (std::nothrow) fs_grid();
  if (!g) return FS_ERR_OOM;
  g->P = *params;
  if (params->yf) { g->yf.assign(params->yf, params->yf + params->ny + 1); }
  g->P.yf = params->yf ? g->yf.data() : nullptr;
  init_dims(g);
  const size_t need = g->f64 ? carve<double>(g, nullptr) : carve<float>(g, nullptr);
  if (bytes < need) { delete g; return FS_ERR_INVALID_ARG; }
  g->stream = (cudaStream_t)cuda_stream; g->ws = (char*)workspace; g->ws_bytes = bytes;
  if (g->f64) carve<double>(g, g->ws); else carve<float>(g, g->ws);
  auto fail = [&](fs_status s) { fs_grid_destroy(g); return s; };
  // the grid lives on the device that owns the workspace; that device must be the caller's current one (the
  // stream handle belongs to it too) and stays the grid's device for every later call, whatever is current then
  if (cudaGetDevice(&g->device) != cudaSuccess) { delete g; return FS_ERR_CUDA; }
  {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, workspace) != cudaSuccess) { cudaGetLastError(); delete g; return FS_ERR_INVALID_ARG; }
    if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) { delete g; return FS_ERR_INVALID_ARG; }
    if (pa.type == cudaMemoryTypeDevice && pa.device != g->device) { delete g; return FS_ERR_INVALID_ARG; }
  }
  if ((g->f64 ? momv_configure_device<double>() : momv_configure_device<float>()) != cudaSuccess) {
    std::fprintf(stderr, "libfs: cudaFuncSetAttribute(max dynamic shared memory) failed for the momentum kernel\n");
    delete g; return FS_ERR_CUDA;
  }
  if (g->P.precond == FS_PC_GMG) {
    const cudaError_t e1 = g->f64 ? mg_configure_device<double>() : mg_configure_device<float>();
    const cudaError_t e2 = g->f64 ? mgf_configure_device<double>() : mgf_configure_device<float>();
    if (e1 != cudaSuccess || e2 != cudaSuccess) {
      std::fprintf(stderr, "libfs: cudaFuncSetAttribute(max dynamic shared memory) failed: %s\n", cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
      delete g; return FS_ERR_CUDA;
    }
  }
  if (cudaStreamCreateWithFlags(&g->cap, cudaStreamNonBlocking) != cudaSuccess) return fail(FS_ERR_CUDA);
  if (cudaStreamCreateWithFlags(&g->cap2, cudaStreamNonBlocking) != cudaSuccess) return fail(FS_ERR_CUDA);
  if (cudaMemsetAsync(g->ws, 0, need, g->stream) != cudaSuccess) return fail(FS_ERR_CUDA);
  init_ibm(g);
  st = g->f64 ? upload_metrics<double>(g) : upload_metrics<float>(g);
  if (st != FS_OK) return fail(st);
  *out = g;
  return FS_OK;
}

fs_status fs_grid_destroy(fs_grid* g) {
  if (!g) return FS_ERR_INVALID_ARG;
  DeviceGuard guard_(g->device);
  if (g->stream || g->cap) cudaStreamSynchronize(g->stream);
  if (g->step_exec) cudaGraphExecDestroy(g->step_exec);
  if (g->poisson_exec) cudaGraphExecDestroy(g->poisson_exec);
  if (g->cap) cudaStreamDestroy(g->cap);
  if (g->cap2) cudaStreamDestroy(g->cap2);
  delete g;
  return FS_OK;
}

fs_status fs_field_size(fs_grid* g, fs_field f, long long* count) {
  if (!g || !count) return FS_ERR_INVALID_ARG;
  const long long n = g->ib.n;
  switch (f) {
    case FS_U: case FS_HU: *count = (long long)g->nU; break;
    case FS_V: case FS_HV: *count = (long long)g->nV; break;
    case FS_W: case FS_HW: *count = (long long)g->nW; break;
    case FS_P: case FS_DIV: *count = (long long)g->nP; break;
    case FS_MARKER_X: case FS_MARKER_U: case FS_MARKER_F: *count = 3 * n; break;
    case FS_MARKER_BASE: *count = 9 * n; break;
    case FS_MARKER_PERM: case FS_MARKER_KEYS: *count = n; break;
    case FS_MARKER_SEG: *count = n + 1; break;
    case FS_BODY_STATE: *count = 9; break;
    case FS_MASK_U: *count = (long long)g->nU; break;
    case FS_MASK_V: *count = (long long)g->nV; break;
    case FS_MASK_W: *count = (long long)g->nW; break;
    default: return FS_ERR_INVALID_ARG;
  }
  return FS_OK;
}

fs_status fs_fields_set(fs_grid* g, fs_field f, const void* src, fs_dtype dtype, int src_on_device) {
  if (!g || !src) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (f <= FS_DIV) return g->f64 ? fields_io<double>(g, f, const_cast<void*>(src), dtype, src_on_device, true)
                                 : fields_io<float>(g, f, const_cast<void*>(src), dtype, src_on_device, true);
  const cudaMemcpyKind kind = src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  const size_t n = (size_t)g->ib.n;
  if (f == FS_MARKER_X) { CK(cudaMemcpyAsync(g->ib.X, src, 3 * n * sizeof(double), kind, g->stream)); g->indexed = false; invalidate(g); }
  else if (f == FS_MARKER_U) CK(cudaMemcpyAsync(g->ib.Ub, src, 3 * n * sizeof(double), kind, g->stream));
  else if (f == FS_BODY_STATE) {
    CK(cudaMemcpyAsync(g->S->body_disp, src, 3 * sizeof(double), kind, g->stream));
    CK(cudaMemcpyAsync(g->S->body_vel, (const double*)src + 3, 3 * sizeof(double), kind, g->stream));
  } else return FS_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

static fs_status fields_async(fs_grid* g, fs_field f, void* host, bool set) {
  if (!g || !host || f > FS_HW) return FS_ERR_INVALID_ARG;
  GUARD(g);
  size_t n = 0;
  void* dev = g->f64 ? (void*)field_ptr<double>(g, f, &n) : (void*)field_ptr<float>(g, f, &n);
  if (!dev) return FS_ERR_INVALID_ARG;
  const size_t bytes = n * (g->f64 ? sizeof(double) : sizeof(float));
  if (set) CK(cudaMemcpyAsync(dev, host, bytes, cudaMemcpyHostToDevice, g->stream));
  else CK(cudaMemcpyAsync(host, dev, bytes, cudaMemcpyDeviceToHost, g->stream));
  return FS_OK;
}
fs_status fs_fields_set_async(fs_grid* g, fs_field f, const void* host_src) { return fields_async(g, f, const_cast<void*>(host_src), true); }
fs_status fs_fields_get_async(fs_grid* g, fs_field f, void* host_dst) { return fields_async(g, f, host_dst, false); }

fs_status fs_fields_get(fs_grid* g, fs_field f, void* dst, fs_dtype dtype, int dst_on_device) {
  if (!g || !dst) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (f <= FS_DIV) return g->f64 ? fields_io<double>(g, f, dst, dtype, dst_on_device, false)
                                 : fields_io<float>(g, f, dst, dtype, dst_on_device, false);
  const cudaMemcpyKind kind = dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  const size_t n = (size_t)g->ib.n;
  const void* src = nullptr; size_t bytes = 0;
  switch (f) {
    case FS_MARKER_X: src = g->ib.X; bytes = 3 * n * sizeof(double); break;
    case FS_MARKER_U: src = g->ib.Ub; bytes = 3 * n * sizeof(double); break;
    case FS_MARKER_F: src = g->ib.Fl; bytes = 3 * n * sizeof(double); break;
    case FS_MARKER_BASE: src = g->ib.base; bytes = 9 * n * sizeof(int); break;
    case FS_MARKER_PERM: src = g->ib.perm; bytes = n * sizeof(int); break;
    case FS_MARKER_KEYS: src = g->ib.keys; bytes = n * sizeof(int); break;
    case FS_MARKER_SEG: src = g->ib.seg; bytes = (n + 1) * sizeof(int); break;
    case FS_MASK_U: case FS_MASK_V: case FS_MASK_W:
      if (!g->ib.has_mask) return FS_ERR_BAD_STATE;
      src = f == FS_MASK_U ? g->ib.mu : (f == FS_MASK_V ? g->ib.mv : g->ib.mw);
      bytes = f == FS_MASK_U ? g->nU : (f == FS_MASK_V ? g->nV : g->nW);
      break;
    case FS_BODY_STATE: {
      CK(cudaMemcpyAsync(dst, g->S->body_disp, 3 * sizeof(double), kind, g->stream));
      CK(cudaMemcpyAsync((double*)dst + 3, g->S->body_vel, 3 * sizeof(double), kind, g->stream));
      CK(cudaMemcpyAsync((double*)dst + 6, g->S->body_force, 3 * sizeof(double), kind, g->stream));
      CK(cudaStreamSynchronize(g->stream));
      return FS_OK;
    }
    default: return FS_ERR_INVALID_ARG;
  }
  if (bytes) CK(cudaMemcpyAsync(dst, src, bytes, kind, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_set_history(fs_grid* g, int have_history, long long step) {
  if (!g) return FS_ERR_INVALID_ARG;
  GUARD(g);
  const int hh = have_history != 0;
  CK(cudaMemcpyAsync(&g->S->have_hist, &hh, sizeof(int), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(&g->S->step, &step, sizeof(long long), cudaMemcpyHostToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_set_ibm_markers(fs_grid* g, int n, const double* xyz, const double* vel, const double* dvol) {
  if (!g || n < 0 || (n > 0 && !xyz)) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (n > g->P.max_markers) return FS_ERR_INVALID_ARG;
  if (n > 0 && !g->uniform_y) return FS_ERR_UNSUPPORTED;
  IbmCtx& ib = g->ib;
  ib.n = n; g->nl = n; g->indexed = false;
  ib.has_beam = 0;                  // a beam rides on a particular marker set: it has to be set again (fs_set_beam)
  invalidate(g);
  if (n == 0) {
    double z[3] = {0, 0, 0};
    CK(cudaMemcpyAsync(g->S->body_force, z, sizeof z, cudaMemcpyHostToDevice, g->stream));
    CK(cudaStreamSynchronize(g->stream));
    return FS_OK;
  }
  CK(cudaMemcpyAsync(ib.X, xyz, 3 * (size_t)n * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  if (vel) CK(cudaMemcpyAsync(ib.Ub, vel, 3 * (size_t)n * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  else CK(cudaMemsetAsync(ib.Ub, 0, 3 * (size_t)n * sizeof(double), g->stream));
  std::vector<double> dv;
  if (dvol) dv.assign(dvol, dvol + n); else dv.assign(n, g->hx * g->hy * g->hz);
  CK(cudaMemcpyAsync(ib.dV, dv.data(), (size_t)n * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemsetAsync(ib.Fl, 0, 3 * (size_t)n * sizeof(double), g->stream));
  CK(cudaMemsetAsync(ib.Ul, 0, 3 * (size_t)n * sizeof(double), g->stream));
  CK(cudaMemsetAsync(&g->S->ibm_oob, 0, sizeof(int), g->stream));
  Launch L{g->stream, 0, 0, nullptr, &g->seen};
  g->fixed_launches += g->f64 ? launch_ibm_index<double>(g->cd, ib, L) : launch_ibm_index<float>(g->cf, ib, L);
  CK(cudaGetLastError());
  int oob = 0;
  CK(cudaMemcpyAsync(&oob, &g->S->ibm_oob, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if (oob) {                        // a support reaches a non-periodic boundary: refused, the grid keeps no markers
    const int zero = 0;
    ib.n = 0; g->nl = 0;
    CK(cudaMemcpyAsync(&g->S->ibm_oob, &zero, sizeof(int), cudaMemcpyHostToDevice, g->stream));
    CK(cudaStreamSynchronize(g->stream));
    return FS_ERR_UNSUPPORTED;
  }
  g->indexed = true;
  return FS_OK;
}

fs_status fs_marker_segments(fs_grid* g, int* nseg) {
  if (!g || !nseg) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (g->ib.n == 0) { *nseg = 0; return FS_OK; }
  int v = 0;
  CK(cudaMemcpyAsync(&v, &g->S->nseg, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  *nseg = v;
  return FS_OK;
}

fs_status fs_set_body(fs_grid* g, double m, double c, double k, int dof_mask) {
  if (!g || !(m > 0)) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (g->ib.has_beam) return FS_ERR_UNSUPPORTED;
  g->ib.has_body = 1; g->ib.bm = m; g->ib.bc = c; g->ib.bk = k; g->ib.dof = dof_mask;
  g->ib.strong = g->P.coupling_max_iters > 1;
  invalidate(g);
  return FS_OK;
}

fs_status fs_set_beam(fs_grid* g, int n_nodes, const double* node_xy, const int* marker_node, double EI, double mu_s, double zeta_s) {
  if (!g || n_nodes < 2 || !node_xy || !marker_node || !(EI > 0) || !(mu_s > 0) || zeta_s < 0) return FS_ERR_INVALID_ARG;
  GUARD(g);
  IbmCtx& ib = g->ib;
  if (ib.n <= 0 || g->P.max_beam_nodes < n_nodes) return FS_ERR_BAD_STATE;
  if (ib.has_body || ib.has_mask || g->P.cfl > 0.0) return FS_ERR_UNSUPPORTED;
  const double tx = node_xy[2 * (n_nodes - 1)] - node_xy[0], ty = node_xy[2 * (n_nodes - 1) + 1] - node_xy[1];
  const double len = std::sqrt(tx * tx + ty * ty);
  if (!(len > 0)) return FS_ERR_INVALID_ARG;
  for (int i = 1; i < n_nodes; ++i) {       // collinear and ordered along the axis
    const double ax = node_xy[2 * i] - node_xy[0], ay = node_xy[2 * i + 1] - node_xy[1];
    const double ex = node_xy[2 * i] - node_xy[2 * (i - 1)], ey = node_xy[2 * i + 1] - node_xy[2 * (i - 1) + 1];
    if (std::fabs(ax * ty - ay * tx) > 1e-12 * len * len || !(ex * tx + ey * ty > 0)) return FS_ERR_INVALID_ARG;
  }
  std::vector<int> start(n_nodes + 1, 0), list(ib.n);
  for (int l = 0; l < ib.n; ++l) { if (marker_node[l] < 0 || marker_node[l] >= n_nodes) return FS_ERR_INVALID_ARG; start[marker_node[l] + 1] += 1; }
  for (int i = 0; i < n_nodes; ++i) start[i + 1] += start[i];
  { std::vector<int> fill(start.begin(), start.end() - 1); for (int l = 0; l < ib.n; ++l) list[fill[marker_node[l]]++] = l; }
  const int nd = 2 * (n_nodes - 1);
  std::vector<double> Lb(4 * (size_t)nd), Mb(7 * (size_t)nd), Cb(7 * (size_t)nd);
  if (!beam_build(n_nodes, node_xy, EI, mu_s, zeta_s, g->P.dt, Lb.data(), Mb.data(), Cb.data(), ib.nk, g->beam_coef)) return FS_ERR_INVALID_ARG;
  invalidate(g);
  ib.has_beam = 1; ib.nbn = n_nodes; ib.ndof = nd; ib.bnrm[0] = -ty / len; ib.bnrm[1] = tx / len;
  ib.strong = g->P.coupling_max_iters > 1;
  double* zero7[7] = {ib.bw, ib.bv, ib.ba, ib.bw0, ib.bv0, ib.ba0, ib.bQ};
  for (double* z : zero7) CK(cudaMemsetAsync(z, 0, (size_t)nd * sizeof(double), g->stream));
  CK(cudaMemcpyAsync(ib.bL, Lb.data(), Lb.size() * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(ib.bM, Mb.data(), Mb.size() * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(ib.bC, Cb.data(), Cb.size() * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(ib.Xref, ib.X, 3 * (size_t)ib.n * sizeof(double), cudaMemcpyDeviceToDevice, g->stream));
  CK(cudaMemcpyAsync(ib.mnode, marker_node, (size_t)ib.n * sizeof(int), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(ib.nstart, start.data(), start.size() * sizeof(int), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(ib.nlist, list.data(), list.size() * sizeof(int), cudaMemcpyHostToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_beam_state(fs_grid* g, double* w, double* v, double* a, double* Q, double* coef) {
  if (!g) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (!g->ib.has_beam) return FS_ERR_BAD_STATE;
  const size_t nb = (size_t)g->ib.ndof * sizeof(double);
  if (w) CK(cudaMemcpyAsync(w, g->ib.bw, nb, cudaMemcpyDeviceToHost, g->stream));
  if (v) CK(cudaMemcpyAsync(v, g->ib.bv, nb, cudaMemcpyDeviceToHost, g->stream));
  if (a) CK(cudaMemcpyAsync(a, g->ib.ba, nb, cudaMemcpyDeviceToHost, g->stream));
  if (Q) CK(cudaMemcpyAsync(Q, g->ib.bQ, nb, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if (coef) for (int i = 0; i < 4; ++i) coef[i] = g->beam_coef[i];
  return FS_OK;
}

fs_status fs_set_solid_mask(fs_grid* g, const unsigned char* eps_cells, const double* uc) {
  if (!g) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (!g->P.solid_mask) return FS_ERR_BAD_STATE;
  if (!g->uniform_y || (eps_cells && g->ib.has_beam)) return FS_ERR_UNSUPPORTED;
  invalidate(g);
  IbmCtx& ib = g->ib;
  if (!eps_cells) { ib.has_mask = 0; return FS_OK; }
  CK(cudaMemcpyAsync(ib.eps, eps_cells, g->nP, cudaMemcpyHostToDevice, g->stream));
  for (int a = 0; a < 3; ++a) ib.uc[a] = uc ? uc[a] : 0.0;
  ib.has_mask = 1;
  Launch L{g->stream, 0, 0, nullptr, &g->seen};
  g->fixed_launches += g->f64 ? launch_mask_classify<double>(g->cd, ib, L) : launch_mask_classify<float>(g->cf, ib, L);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_set_body_state(fs_grid* g, const double* disp3, const double* vel3) {
  if (!g || !disp3 || !vel3) return FS_ERR_INVALID_ARG;
  GUARD(g);
  CK(cudaMemcpyAsync(g->S->body_disp, disp3, 3 * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(g->S->body_vel, vel3, 3 * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_step(fs_grid* g, int nsteps, fs_step_info* last) {
  if (!g || nsteps < 0) return FS_ERR_INVALID_ARG;
  GUARD(g);
  for (int s = 0; s < nsteps; ++s) {
    fs_status st = g->f64 ? advance_step<double>(g) : advance_step<float>(g);
    if (st != FS_OK) return st;
  }
  if (!last) return FS_OK;
  Scalars hs; fs_status st = read_scalars(g, &hs); if (st != FS_OK) return st;
  fs_step_info I;
  I.pcg_iters = hs.iter; I.converged = hs.converged; I.nan_flag = hs.nan_flag;
  I.rel_residual = hs.bnorm2 > 0 ? std::sqrt(hs.rr / hs.bnorm2) : 0.0;
  I.true_rel_residual = hs.bnorm2 > 0 ? std::sqrt(hs.true_rr / hs.bnorm2) : 0.0;
  I.max_abs_div = hs.max_div;
  for (int a = 0; a < 3; ++a) { I.body_force[a] = hs.body_force[a]; I.body_disp[a] = hs.body_disp[a]; I.body_vel[a] = hs.body_vel[a]; }
  I.step = hs.step;
  I.unconverged_steps = hs.unconverged_steps; I.nan_steps = hs.nan_steps;
  I.dt = hs.dt_prev; I.time = hs.time;
  I.coupling_iters = g->last_sweeps; I.coupling_xi = g->last_xi;
  if (g->last_iters >= 0) I.pcg_iters = (int)g->last_iters;
  *last = I;                        // valid for FS_OK, FS_ERR_NOT_CONVERGED and FS_ERR_UNSUPPORTED (fs.h)
  if (hs.ibm_oob) return FS_ERR_UNSUPPORTED;
  return (nsteps > 0 && !hs.converged) ? FS_ERR_NOT_CONVERGED : FS_OK;
}

fs_status fs_poisson_solve(fs_grid* g, const void* rhs, void* p_inout, fs_dtype dtype, int on_device, fs_poisson_info* info) {
  if (!g || !rhs || !p_inout) return FS_ERR_INVALID_ARG;
  GUARD(g);
  return g->f64 ? poisson_impl<double>(g, rhs, p_inout, dtype, on_device, info) : poisson_impl<float>(g, rhs, p_inout, dtype, on_device, info);
}

fs_status fs_ibm_interpolate(fs_grid* g, double* out) {
  if (!g || !out) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (g->ib.n == 0) return FS_ERR_BAD_STATE;
  Launch L{g->stream, 0, 0, nullptr, &g->seen};
  if (g->f64) g->fixed_launches += launch_ibm_interpolate<double>(g->cd, g->ib, g->cd.u, g->cd.v, g->cd.w, g->ib.Ul, L);
  else g->fixed_launches += launch_ibm_interpolate<float>(g->cf, g->ib, g->cf.u, g->cf.v, g->cf.w, g->ib.Ul, L);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, g->ib.Ul, 3 * (size_t)g->ib.n * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_ibm_spread(fs_grid* g, const double* F) {
  if (!g || !F) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (g->ib.n == 0) return FS_ERR_BAD_STATE;
  CK(cudaMemcpyAsync(g->ib.Fl, F, 3 * (size_t)g->ib.n * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  Launch L{g->stream, 0, 0, nullptr, &g->seen};
  if (g->f64) g->fixed_launches += launch_ibm_spread<double>(g->cd, g->ib, g->ib.Fl, g->cd.u, g->cd.v, g->cd.w, 1.0, L);
  else g->fixed_launches += launch_ibm_spread<float>(g->cf, g->ib, g->ib.Fl, g->cf.u, g->cf.v, g->cf.w, 1.0, L);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_gmg_vcycle(fs_grid* g, const double* r, double* z) {
  if (!g || !r || !z) return FS_ERR_INVALID_ARG;
  GUARD(g);
  if (g->P.precond != FS_PC_GMG) return FS_ERR_BAD_STATE;
  const int zero = 0;
  CK(cudaMemcpyAsync(&g->S->done, &zero, sizeof(int), cudaMemcpyHostToDevice, g->stream));
  Launch L{g->stream, 0, 0, nullptr, &g->seen};
  fs_status st;
  if (g->f64) {
    st = copy_in<double>(g, g->cd.r, g->nP, r, FS_F64, 0); if (st != FS_OK) return st;
    g->fixed_launches += launch_vcycle<double>(g->cd, g->md, g->cd.r, g->cd.z, L, nullptr, 1.0);
    launch_scale<double>(g->cd.z, 1.0 / g->hy, (long long)g->nP, g->stream);   // A = h (-L)  =>  M^-1 r = V(r) / h
    CK(cudaGetLastError());
    st = copy_out<double>(g, g->cd.z, g->nP, z, FS_F64, 0); if (st != FS_OK) return st;
  } else {
    st = copy_in<float>(g, g->cf.r, g->nP, r, FS_F64, 0); if (st != FS_OK) return st;
    g->fixed_launches += launch_vcycle<float>(g->cf, g->mf, g->cf.r, g->cf.z, L, nullptr, 1.0f);
    launch_scale<float>(g->cf.z, 1.0 / g->hy, (long long)g->nP, g->stream);
    CK(cudaGetLastError());
    st = copy_out<float>(g, g->cf.z, g->nP, z, FS_F64, 0); if (st != FS_OK) return st;
  }
  return FS_OK;
}

fs_status fs_momentum_rhs(fs_grid* g) {
  if (!g) return FS_ERR_INVALID_ARG;
  GUARD(g);
  Launch L{g->stream, 0, 0, nullptr, &g->seen};
  g->fixed_launches += g->f64 ? launch_momentum<double>(g->cd, L) : launch_momentum<float>(g->cf, L);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(g->stream));
  return FS_OK;
}

fs_status fs_profile_step(fs_grid* g, int nsteps) {
  if (!g || nsteps < 0) return FS_ERR_INVALID_ARG;
  GUARD(g);
  g->profiling = true;
  fs_status st = FS_OK;
  for (int s = 0; s < nsteps && st == FS_OK; ++s) {
    st = g->f64 ? advance_step<double>(g) : advance_step<float>(g);
    if (st == FS_OK && cudaStreamSynchronize(g->stream) != cudaSuccess) st = FS_ERR_CUDA;
    prof_collect(&g->prof);
  }
  g->profiling = false;
  return st;
}

fs_status fs_profile_count(fs_grid* g, int* n) {
  if (!g || !n) return FS_ERR_INVALID_ARG;
  *n = (int)g->prof.agg.size();
  return FS_OK;
}

fs_status fs_profile_entry(fs_grid* g, int idx, const char** name, long long* launches, double* ms, double* bytes) {
  if (!g || idx < 0 || idx >= (int)g->prof.agg.size() || !name || !launches || !ms || !bytes) return FS_ERR_INVALID_ARG;
  const ProfAgg& a = g->prof.agg[idx];
  *name = a.name; *launches = a.launches; *ms = a.ms; *bytes = a.bytes;
  return FS_OK;
}

fs_status fs_profile_reset(fs_grid* g) {
  if (!g) return FS_ERR_INVALID_ARG;
  g->prof.agg.clear();
  return FS_OK;
}

fs_status fs_kernels_used(fs_grid* g, char* buf, size_t cap, size_t* needed) {
  if (!g || (!buf && cap > 0)) return FS_ERR_INVALID_ARG;
  std::string all;
  for (const char* n : g->seen.names) { if (!all.empty()) all += ';'; all += n; }
  if (needed) *needed = all.size() + 1;
  if (cap < all.size() + 1) return buf ? FS_ERR_INVALID_ARG : FS_OK;
  std::memcpy(buf, all.c_str(), all.size() + 1);
  return FS_OK;
}

fs_status fs_launch_count(fs_grid* g, long long* launches) {
  if (!g || !launches) return FS_ERR_INVALID_ARG;
  GUARD(g);
  Scalars hs; fs_status st = read_scalars(g, &hs); if (st != FS_OK) return st;
  *launches = g->fixed_launches + hs.total_body * (long long)g->step_body + g->body_iters_poisson * (long long)g->poisson_body;
  return FS_OK;
}

}  // extern "C"
