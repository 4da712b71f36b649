// fs_kernels_pcg.cu -- pressure Poisson solve (S6 tail, S7): matrix-free 7-point operator
// A = -dy_j L (symmetric positive semi-definite) and textbook preconditioned CG (O7;
// solver family PAPER.md L449, CG L686).  The Laplacian apply is fused with the d.q dot product and
// the x/r update with the residual norm; all sums are deterministic (fs_internal.cuh grid_sum).
// Loop control lives in device memory: the last block of k_pcg_update decides whether the CUDA-graph
// WHILE node runs another iteration.
#include "fs_internal.cuh"
#include <cstring>
#include <cstdlib>

namespace fs {

struct ColGeom { dim3 grid, block; int kz; };
ColGeom col_geom(int nx, int ny, int nz);
constexpr int kFlatBlocks = 148 * 8;
static inline int flat_blocks(long long n) { long long b = (n + 255) / 256; return (int)(b < kFlatBlocks ? (b < 1 ? 1 : b) : kFlatBlocks); }

// Jacobi diagonal of A at (i,j,k): dy_j * (sum of the face coefficients that exist).
template <class T> __device__ __forceinline__ T diag_A(const Ctx<T>& c, int i, int j, int k) {
  const T cx = T((c.bx && i == 0 ? 0 : 1) + (c.bx && i == c.nx - 1 ? 0 : 1)) * c.ihx2;
  const T cz = T((c.bz && k == 0 ? 0 : 1) + (c.bz && k == c.nz - 1 ? 0 : 1)) * c.ihz2;
  const T cy = (c.cyh[j] + c.cyl[j]) * c.idy[j + 1];
  return (cx + cy + cz) * c.dy[j + 1];
}
// z = M^-1 r for the point preconditioners
template <class T> __device__ __forceinline__ T precond_point(const Ctx<T>& c, T r, int i, int j, int k) {
  return c.precond == FS_PC_JACOBI ? r / diag_A<T>(c, i, j, k) : r;
}

// Column-marching application of A: thread (i,j) walks k0..k1-1 keeping x(k-1), x(k), x(k+1) in
// registers; x+-1 / y+-1 neighbours come through L1.  Neighbour indices wrap (periodic) or clamp
// (bounded: the clamped difference is exactly zero = homogeneous Neumann flux dropped).
template <class T, class F> __device__ __forceinline__ void march_A(const Ctx<T>& c, const T* __restrict__ x, int i, int j, int k0, int k1, F&& f) {
  const int im = i > 0 ? i - 1 : (c.bx ? 0 : c.nx - 1), ip = i + 1 < c.nx ? i + 1 : (c.bx ? i : 0);
  const int jm = j > 0 ? j - 1 : (c.by ? 0 : c.ny - 1), jp = j + 1 < c.ny ? j + 1 : (c.by ? j : 0);
  const size_t pl = (size_t)c.nx * c.ny;
  const size_t oc = (size_t)i + (size_t)c.nx * j, ow = (size_t)im + (size_t)c.nx * j, oe = (size_t)ip + (size_t)c.nx * j;
  const size_t os = (size_t)i + (size_t)c.nx * jm, on = (size_t)i + (size_t)c.nx * jp;
  const T cyl = c.cyl[j], cyh = c.cyh[j], idy = c.idy[j + 1], ndy = -c.dy[j + 1];
  const int kb = k0 > 0 ? k0 - 1 : (c.bz ? 0 : c.nz - 1);
  T xb = x[oc + pl * kb], xc = x[oc + pl * k0];
  for (int k = k0; k < k1; ++k) {
    const int kt = k + 1 < c.nz ? k + 1 : (c.bz ? k : 0);
    const T xt = x[oc + pl * kt];
    const size_t o = pl * k;
    const T xw = x[ow + o], xe = x[oe + o], xs = x[os + o], xn = x[on + o];
    T acc = (xe - xc) * c.ihx2 - (xc - xw) * c.ihx2;
    const T fy = (xn - xc) * cyh - (xc - xs) * cyl;
    acc += fy * idy;
    acc += (xt - xc) * c.ihz2 - (xc - xb) * c.ihz2;
    f(k, oc + o, xc, acc * ndy);
    xb = xc; xc = xt;
  }
}

// ---- PCG start: r = (bhat_raw - mean_coef dy_j) - A x0 ; ||bhat||^2, ||r||^2, r.z -------------------
template <class T> __global__ void __launch_bounds__(256) k_pcg_init(const Ctx<T> c, int kz, Launch L) {
  __shared__ double sh[4 * 32]; __shared__ int flag;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  double v[4] = {0.0, 0.0, 0.0, 0.0};
  if (i < c.nx && j < c.ny) {
    const T shift = T(c.S->mean_coef) * c.dy[j + 1];
    march_A<T>(c, c.p, i, j, k0, k1, [&](int k, size_t q, T xc, T Ax) {
      const T bh = c.r[q] - shift;
      const T r = bh - Ax;
      c.r[q] = r;
      c.bh[q] = bh;
      const T z = precond_point<T>(c, r, i, j, k);
      v[0] += (double)bh * (double)bh; v[1] += (double)r * (double)r; v[2] += (double)r * (double)z; v[3] += (double)r;
    });
  }
  if (grid_sum<4>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0 && threadIdx.y == 0) {
      Scalars* S = c.S;
      S->bnorm2 = v[0]; S->rr = v[1]; S->rho_cur = v[2]; S->rho_prev = 1.0; S->dq = 1.0;
      S->iter = 0; S->body_runs = 0; S->first = 1; S->dsel = 0; S->pending = 0; S->rsel = 0; S->need_update = 0;
      S->rmean = v[3] / ((double)c.nx * c.ny * c.nz);
      const int conv = (v[0] == 0.0) || (sqrt(v[1]) <= S->rtol * sqrt(v[0]));
      S->converged = conv; S->done = conv || S->max_iter <= 0;
      if (L.use_cond) cudaGraphSetConditional(L.cond, S->done ? 0u : 1u);
    }
  }
}

// ---- K4 + K1 fused: d' = z + beta d, q = A d', d'.q -------------------------------------------------------
// 2.5-D streaming kernel (one thread per cell of a 32 x 16 extended tile, 30 x 14 results, z march with a
// register queue for the z neighbours and a double-buffered shared-memory plane for the x / y neighbours).
// d' is computed on the halo as well (from z and d there), so the separate direction pass and its 3 words
// per cell disappear: the pair moves 4 words (z, d in; d', q out) instead of 3 + 2.  d' goes to the OTHER
// direction buffer (a neighbouring CTA may still need the old d on its halo); Scalars::dsel says which of
// the two buffers holds the current direction and is toggled by k_pcg_update.
// PC: 0 none (z = r), 1 Jacobi (z = r / diag A), 2 GMG (z = zs * V-cycle output).
constexpr int kDaTX = 32, kDaTY = 16;

template <class T, int PC> __global__ void __launch_bounds__(kDaTX * kDaTY, 2) k_pcg_dirapply(const Ctx<T> c, T zs, int kz) {
  __shared__ T D[2][kDaTY][kDaTX];
  __shared__ double sh[3 * 32]; __shared__ int flag;
  const Scalars* S = c.S;
  if (blockIdx.x + blockIdx.y + blockIdx.z == 0 && threadIdx.x + threadIdx.y == 0) c.S->body_runs += 1;   // one writer: loop-body replays of this solve
  if (S->done) return;
  const bool first = S->first != 0;
  const T beta = first ? T(0) : T(S->rho_cur / S->rho_prev);
  const T* __restrict__ dold = S->dsel ? c.d2 : c.d;
  T* __restrict__ dnew = S->dsel ? c.d : c.d2;
  const T* __restrict__ zsrc = PC == 2 ? c.z : c.r;
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int iu = blockIdx.x * (kDaTX - 2) + tx - 1, ju = blockIdx.y * (kDaTY - 2) + ty - 1;
  // source cell of this thread: wrapped (periodic) or clamped (bounded: zero difference = dropped Neumann flux)
  const int i = c.bx ? min(max(iu, 0), c.nx - 1) : wrapi(iu, c.nx);
  const int j = c.by ? min(max(ju, 0), c.ny - 1) : wrapi(ju, c.ny);
  const bool own = tx >= 1 && tx <= kDaTX - 2 && ty >= 1 && ty <= kDaTY - 2 && iu < c.nx && ju < c.ny;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  const size_t pl = (size_t)c.nx * c.ny, oc = (size_t)i + (size_t)c.nx * j;
  const T cyl = c.cyl[j], cyh = c.cyh[j], idy = c.idy[j + 1], ndy = -c.dy[j + 1];
  // Jacobi diagonal pieces (same association as diag_A)
  const T dxy = T((c.bx && i == 0 ? 0 : 1) + (c.bx && i == c.nx - 1 ? 0 : 1)) * c.ihx2;
  const T dyy = (cyh + cyl) * idy;
  auto plane_src = [&](int k) { return c.bz ? min(max(k, 0), c.nz - 1) : wrapi(k, c.nz); };
  // Deferred x update (the x += alpha d of the PREVIOUS iteration rides on this kernel's read of the old d):
  // applied to the own cells when their d' is formed; sums of x and d' (volume weighted) for the final mean.
  const bool pend = S->pending != 0;
  const T alpha_p = pend ? T(S->alpha_prev) : T(0);
  double sp = 0.0, sd = 0.0;
  auto dir_at = [&](int k) {              // d' at (i, j, plane_src(k))
    const int ks = plane_src(k);
    const size_t o = oc + pl * ks;
    const bool upd = own && k >= k0 && k < k1;
    T pv = T(0);
    if (upd) pv = c.p[o];
    T z;
    if (PC == 2) z = zsrc[o] * zs;
    else if (PC == 1) {
      const T dzz = T((c.bz && ks == 0 ? 0 : 1) + (c.bz && ks == c.nz - 1 ? 0 : 1)) * c.ihz2;
      z = zsrc[o] / ((dxy + dyy + dzz) * c.dy[j + 1]);
    } else z = zsrc[o];
    const T dol = first ? T(0) : dold[o];
    const T dn = first ? z : z + beta * dol;
    if (upd) {
      if (pend) { pv += alpha_p * dol; c.p[o] = pv; }
      sp += (double)pv; sd += (double)dn;
    }
    return dn;
  };
  const int txm = max(tx - 1, 0), txp = min(tx + 1, kDaTX - 1), tym = max(ty - 1, 0), typ = min(ty + 1, kDaTY - 1);
  T dB = dir_at(k0 - 1), dC = dir_at(k0), dT = dir_at(k0 + 1);
  D[k0 & 1][ty][tx] = dC;
  __syncthreads();
  double v[1] = {0.0};
  for (int k = k0; k < k1; ++k) {
    T dN = T(0);
    if (k + 1 < k1) dN = dir_at(k + 2);   // in flight during the stencil
    const int s = k & 1;
    const T xw = D[s][ty][txm], xe = D[s][ty][txp], xs = D[s][tym][tx], xn = D[s][typ][tx];
    T acc = (xe - dC) * c.ihx2 - (dC - xw) * c.ihx2;
    const T fy = (xn - dC) * cyh - (dC - xs) * cyl;
    acc += fy * idy;
    acc += (dT - dC) * c.ihz2 - (dC - dB) * c.ihz2;
    const T Ax = acc * ndy;
    if (own) {
      const size_t o = oc + pl * k;
      dnew[o] = dC; c.q[o] = Ax;
      v[0] += (double)dC * (double)Ax;
    }
    D[s ^ 1][ty][tx] = dT;
    __syncthreads();
    dB = dC; dC = dT; dT = dN;
  }
  const double wy = c.dy64[j];
  double v3[3] = {v[0], sp * wy, sd * wy};
  if (grid_sum<3>(v3, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (tx == 0 && ty == 0) { c.S->dq = v3[0]; c.S->sum_p = v3[1]; c.S->sum_d = v3[2]; c.S->need_update = 1; }
  }
}

struct DaGeom { dim3 grid; int kz; };
static DaGeom da_geom(int nx, int ny, int nz) {
  const int bxn = (nx + kDaTX - 3) / (kDaTX - 2), byn = (ny + kDaTY - 3) / (kDaTY - 2);
  // z chunks: about 4 waves of 2 CTAs per SM, chunks of at least 16 planes (two halo planes per chunk)
  int kz = nz;
  while (kz > 16 && (long long)bxn * byn * ((nz + kz - 1) / kz) < 4LL * 296) kz = (kz + 1) / 2;
  while ((long long)bxn * byn * ((nz + kz - 1) / kz) > kMaxPartials && kz < nz) kz *= 2;
  DaGeom g; g.kz = kz; g.grid = dim3(bxn, byn, (nz + kz - 1) / kz);
  return g;
}

// Same operation, two x-adjacent cells per thread (nx even): 16-byte (fp64) / 8-byte (fp32) accesses, half
// the index arithmetic per cell, 64 x 16 extended tile -> 60 x 14 results, z loop unrolled by renaming.
constexpr int kDa2IX = 60, kDa2IY = kDaTY - 2, kDa2PL = kDaTY * 32;

template <class T, int PC> __global__ void __launch_bounds__(32 * kDaTY, 2) k_pcg_dirapply2(const Ctx<T> c, T zs, int kz) {
  using V = typename V2T<T>::type;
  __shared__ V D[2 * kDa2PL];
  __shared__ double sh[3 * 32]; __shared__ int flag;
  const Scalars* S = c.S;
  if (blockIdx.x + blockIdx.y + blockIdx.z == 0 && threadIdx.x + threadIdx.y == 0) c.S->body_runs += 1;   // one writer: loop-body replays of this solve
  if (S->done) return;
  const bool first = S->first != 0;
  const T beta = first ? T(0) : T(S->rho_cur / S->rho_prev);
  const T* __restrict__ dold = S->dsel ? c.d2 : c.d;
  T* __restrict__ dnew = S->dsel ? c.d : c.d2;
  const T* __restrict__ zsrc = PC == 2 ? c.z : c.r;
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = blockIdx.x * kDa2IX - 2 + 2 * lane, gy = blockIdx.y * kDa2IY - 1 + ty;
  const int sx = c.bx ? min(max(gx, 0), c.nx - 2) : wrapi(gx, c.nx);
  const int sy = c.by ? min(max(gy, 0), c.ny - 1) : wrapi(gy, c.ny);
  const bool fixl = c.bx && gx < 0, fixr = c.bx && gx >= c.nx;       // clamped halo pairs: both cells = the boundary cell
  const bool own = lane >= 1 && lane <= 30 && ty >= 1 && ty <= kDaTY - 2 && gx < c.nx && gy < c.ny;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  const unsigned pl = (unsigned)c.nx * c.ny, row = (unsigned)sx + (unsigned)c.nx * sy;
  const T cyl = c.cyl[sy], cyh = c.cyh[sy], idy = c.idy[sy + 1], ndy = -c.dy[sy + 1];
  const T ihx2 = c.ihx2, ihz2 = c.ihz2;
  T dgx = T(0), dgy = T(0);                // Jacobi: x + y parts of diag A / dy for the two cells
  T ivx_i = T(0), ivx_b = T(0), ivy_i = T(0), ivy_b = T(0);
  if (PC == 1) {
    const T dyy = (cyh + cyl) * idy;
    dgx = T((c.bx && sx == 0 ? 0 : 1) + 1) * ihx2 + dyy;
    dgy = T(1 + (c.bx && sx + 1 == c.nx - 1 ? 0 : 1)) * ihx2 + dyy;
    // reciprocal diagonals for the two kinds of plane (one or two z neighbours): one division per thread instead
    // of one per cell and plane; z = r * (1 / diag) differs from the oracle's r / diag by at most one rounding
    const T dyj_ = c.dy[sy + 1];
    ivx_i = T(1) / ((dgx + T(2) * ihz2) * dyj_); ivx_b = T(1) / ((dgx + T(1) * ihz2) * dyj_);
    ivy_i = T(1) / ((dgy + T(2) * ihz2) * dyj_); ivy_b = T(1) / ((dgy + T(1) * ihz2) * dyj_);
  }
  const int own_o = ty * 32 + lane;
  const int oS = (ty > 0 ? ty - 1 : 0) * 32 + lane, oN = (ty < kDaTY - 1 ? ty + 1 : ty) * 32 + lane;
  const int oW = ty * 32 + (lane > 0 ? lane - 1 : 0), oE = ty * 32 + (lane < 31 ? lane + 1 : 31);
  // Deferred x update: see k_pcg_dirapply.
  const bool pend = S->pending != 0;
  const T alpha_p = pend ? T(S->alpha_prev) : T(0);
  double sp = 0.0, sd = 0.0;
  V rz, rd, rp;                             // raw z, old d and x of the plane in flight
  int ksrc = 0; bool upd = false;
  auto fetch = [&](int k) {
    ksrc = c.bz ? min(max(k, 0), c.nz - 1) : (k < 0 ? k + c.nz : (k >= c.nz ? k - c.nz : k));
    const unsigned o = row + pl * (unsigned)ksrc;
    rz = ldv2<T, V>(zsrc + o);
    if (!first) rd = ldv2<T, V>(dold + o);
    upd = own && k >= k0 && k < k1;
    if (upd) rp = ldv2<T, V>(c.p + o);
  };
  auto make = [&]() {                       // d' of the fetched plane
    V z;
    if (PC == 2) { z.x = rz.x * zs; z.y = rz.y * zs; }
    else if (PC == 1) {
      const bool zb = c.bz && (ksrc == 0 || ksrc == c.nz - 1);
      z.x = rz.x * (zb ? ivx_b : ivx_i); z.y = rz.y * (zb ? ivy_b : ivy_i);
    } else z = rz;
    V d = z;
    if (!first) { d.x = z.x + beta * rd.x; d.y = z.y + beta * rd.y; }
    if (upd) {                              // own cells: never a clamped halo pair
      if (pend) { rp.x += alpha_p * rd.x; rp.y += alpha_p * rd.y; stv2<T, V>(c.p + (row + pl * (unsigned)ksrc), rp); }
      sp += (double)(rp.x + rp.y); sd += (double)(d.x + d.y);
    }
    if (fixl) d.y = d.x;
    if (fixr) d.x = d.y;
    return d;
  };
  rd.x = rd.y = T(0); rp = rd;
  V d0, d1, d2;
  fetch(k0 - 1); d0 = make();
  fetch(k0); d1 = make();
  int b = 0;
  D[own_o] = d1;
  fetch(k0 + 1);
  __syncthreads();
  double dot = 0.0;
  // dB, dC = d'(k-1), d'(k); dT receives d'(k+1)
  auto step = [&](int k, const V& dB, const V& dC, V& dT) {
    dT = make();
    if (k + 1 < k1) fetch(k + 2);
    const V* P = D + b;
    const V Sv = P[oS], Nv = P[oN];
    const T xw = P[oW].y, xe = P[oE].x;
    T ax = (dC.y - dC.x) * ihx2 - (dC.x - xw) * ihx2;
    T ay = (xe - dC.y) * ihx2 - (dC.y - dC.x) * ihx2;
    ax += ((Nv.x - dC.x) * cyh - (dC.x - Sv.x) * cyl) * idy;
    ay += ((Nv.y - dC.y) * cyh - (dC.y - Sv.y) * cyl) * idy;
    ax += (dT.x - dC.x) * ihz2 - (dC.x - dB.x) * ihz2;
    ay += (dT.y - dC.y) * ihz2 - (dC.y - dB.y) * ihz2;
    V q; q.x = ax * ndy; q.y = ay * ndy;
    if (own) {
      const unsigned o = row + pl * (unsigned)k;
      stv2<T, V>(dnew + o, dC); stv2<T, V>(c.q + o, q);
      dot += (double)(dC.x * q.x + dC.y * q.y);
    }
    b = kDa2PL - b;
    D[b + own_o] = dT;
    __syncthreads();
  };
  int k = k0;
  for (;;) {
    step(k, d0, d1, d2); if (++k >= k1) break;
    step(k, d1, d2, d0); if (++k >= k1) break;
    step(k, d2, d0, d1); if (++k >= k1) break;
  }
  const double wy = c.dy64[sy];
  double v[3] = {dot, sp * wy, sd * wy};
  if (grid_sum<3>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (lane == 0 && ty == 0) { c.S->dq = v[0]; c.S->sum_p = v[1]; c.S->sum_d = v[2]; c.S->need_update = 1; }
  }
}

static DaGeom da2_geom(int nx, int ny, int nz) {
  const int bxn = (nx + kDa2IX - 1) / kDa2IX, byn = (ny + kDa2IY - 1) / kDa2IY;
  const int kz = pick_kz((long long)bxn * byn, nz, 2LL * 148, 2, 16);
  DaGeom g; g.kz = kz; g.grid = dim3(bxn, byn, (nz + kz - 1) / kz);
  return g;
}

// Same operation, one 16-byte vector of x-adjacent cells per thread (fp32: VX = 4 cells; in fp64 the pair
// kernel above is the faster of the two and is the one used; nx a
// multiple of VX): vector global accesses, the index arithmetic shared by VX cells, a 32 VX x 16 extended
// tile -> 30 VX x 14 results (lanes 0 and 31 are halo), z loop unrolled by renaming.
constexpr int kDaVIY = kDaTY - 2;

template <class T, int PC> __global__ void __launch_bounds__(32 * kDaTY, 2) k_pcg_dirapplyv(const Ctx<T> c, T zs, int kz) {
  constexpr int VX = Vec16<T>::VX;
  constexpr int ROWE = 32 * VX;             // cells per shared-memory row
  constexpr int PLN = kDaTY * ROWE;
  using W = Vec16<T>;
  __shared__ __align__(16) T D[2 * PLN];
  __shared__ double sh[3 * 32]; __shared__ int flag;
  const Scalars* S = c.S;
  if (blockIdx.x + blockIdx.y + blockIdx.z == 0 && threadIdx.x + threadIdx.y == 0) c.S->body_runs += 1;   // one writer: loop-body replays of this solve
  if (S->done) return;
  const bool first = S->first != 0;
  const T beta = first ? T(0) : T(S->rho_cur / S->rho_prev);
  const T* __restrict__ dold = S->dsel ? c.d2 : c.d;
  T* __restrict__ dnew = S->dsel ? c.d : c.d2;
  const T* __restrict__ zsrc = PC == 2 ? c.z : c.r;
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = (blockIdx.x * 30 - 1 + lane) * VX, gy = blockIdx.y * kDaVIY - 1 + ty;
  const int sx = c.bx ? min(max(gx, 0), c.nx - VX) : wrapi(gx, c.nx);
  const int sy = c.by ? min(max(gy, 0), c.ny - 1) : wrapi(gy, c.ny);
  const bool fixl = c.bx && gx < 0, fixr = c.bx && gx >= c.nx;       // clamped halo vectors: every cell = the boundary cell
  const bool own = lane >= 1 && lane <= 30 && ty >= 1 && ty <= kDaTY - 2 && gx < c.nx && gy < c.ny;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  const unsigned pl = (unsigned)c.nx * c.ny, row = (unsigned)sx + (unsigned)c.nx * sy;
  const T cyl = c.cyl[sy], cyh = c.cyh[sy], idy = c.idy[sy + 1], dyj = c.dy[sy + 1], ndy = -dyj;
  const T ihx2 = c.ihx2, ihz2 = c.ihz2;
  T dg[VX], ivi[VX], ivb[VX];               // Jacobi: x + y parts of diag A / dy per cell, reciprocal diagonals
#pragma unroll
  for (int a = 0; a < VX; ++a) {
    const int i = sx + a;
    dg[a] = PC == 1 ? T((c.bx && i == 0 ? 0 : 1) + (c.bx && i == c.nx - 1 ? 0 : 1)) * ihx2 + (cyh + cyl) * idy : T(0);
    // reciprocal diagonals for planes with two / one z neighbours (see k_pcg_dirapply2)
    ivi[a] = PC == 1 ? T(1) / ((dg[a] + T(2) * ihz2) * dyj) : T(1);
    ivb[a] = PC == 1 ? T(1) / ((dg[a] + T(1) * ihz2) * dyj) : T(1);
  }
  const int o_own = ty * ROWE + lane * VX;
  const int o_s = (ty > 0 ? ty - 1 : 0) * ROWE + lane * VX, o_n = (ty < kDaTY - 1 ? ty + 1 : ty) * ROWE + lane * VX;
  const int o_w = ty * ROWE + (lane > 0 ? lane * VX - 1 : 0), o_e = ty * ROWE + (lane < 31 ? lane * VX + VX : 32 * VX - 1);
  // Deferred x update: see k_pcg_dirapply.
  const bool pend = S->pending != 0;
  const T alpha_p = pend ? T(S->alpha_prev) : T(0);
  double sp = 0.0, sd = 0.0;
  W rz, rd, rp;                             // raw z, old d and x of the plane in flight
#pragma unroll
  for (int a = 0; a < VX; ++a) { rd.a[a] = T(0); rp.a[a] = T(0); }
  int ksrc = 0; bool upd = false;
  auto fetch = [&](int k) {
    ksrc = c.bz ? min(max(k, 0), c.nz - 1) : (k < 0 ? k + c.nz : (k >= c.nz ? k - c.nz : k));
    const unsigned o = row + pl * (unsigned)ksrc;
    rz = ld16<T>(zsrc + o);
    if (!first) rd = ld16<T>(dold + o);
    upd = own && k >= k0 && k < k1;
    if (upd) rp = ld16<T>(c.p + o);
  };
  auto make = [&]() {                       // d' of the fetched plane
    W d;
    const bool zb = PC == 1 && c.bz && (ksrc == 0 || ksrc == c.nz - 1);
#pragma unroll
    for (int a = 0; a < VX; ++a) {
      T z;
      if (PC == 2) z = rz.a[a] * zs;
      else if (PC == 1) z = rz.a[a] * (zb ? ivb[a] : ivi[a]);
      else z = rz.a[a];
      d.a[a] = first ? z : z + beta * rd.a[a];
    }
    if (upd) {                              // own cells: never a clamped halo vector
      T s1 = T(0), s2 = T(0);
#pragma unroll
      for (int a = 0; a < VX; ++a) { if (pend) rp.a[a] += alpha_p * rd.a[a]; s1 += rp.a[a]; s2 += d.a[a]; }
      if (pend) st16<T>(c.p + (row + pl * (unsigned)ksrc), rp);
      sp += (double)s1; sd += (double)s2;
    }
    if (fixl) {
#pragma unroll
      for (int a = 1; a < VX; ++a) d.a[a] = d.a[0];
    }
    if (fixr) {
#pragma unroll
      for (int a = 0; a < VX - 1; ++a) d.a[a] = d.a[VX - 1];
    }
    return d;
  };
  W d0, d1, d2;
  fetch(k0 - 1); d0 = make();
  fetch(k0); d1 = make();
  int b = 0;
  st16<T>(D + o_own, d1);
  fetch(k0 + 1);
  __syncthreads();
  double dot = 0.0;
  // dB, dC = d'(k-1), d'(k); dT receives d'(k+1)
  auto step = [&](int k, const W& dB, const W& dC, W& dT) {
    dT = make();
    if (k + 1 < k1) fetch(k + 2);
    const T* P = D + b;
    const W Sv = ld16<T>(P + o_s), Nv = ld16<T>(P + o_n);
    const T xw0 = P[o_w], xeL = P[o_e];
    W q;
    T sdot = T(0);
#pragma unroll
    for (int a = 0; a < VX; ++a) {
      const T xc = dC.a[a];
      const T xw = a > 0 ? dC.a[a > 0 ? a - 1 : 0] : xw0;
      const T xe = a < VX - 1 ? dC.a[a < VX - 1 ? a + 1 : a] : xeL;
      T acc = (xe - xc) * ihx2 - (xc - xw) * ihx2;
      acc += ((Nv.a[a] - xc) * cyh - (xc - Sv.a[a]) * cyl) * idy;
      acc += (dT.a[a] - xc) * ihz2 - (xc - dB.a[a]) * ihz2;
      q.a[a] = acc * ndy;
      sdot += xc * q.a[a];
    }
    if (own) {
      const unsigned o = row + pl * (unsigned)k;
      st16<T>(dnew + o, dC); st16<T>(c.q + o, q);
      dot += (double)sdot;
    }
    b = PLN - b;
    st16<T>(D + b + o_own, dT);
    __syncthreads();
  };
  int k = k0;
  for (;;) {
    step(k, d0, d1, d2); if (++k >= k1) break;
    step(k, d1, d2, d0); if (++k >= k1) break;
    step(k, d2, d0, d1); if (++k >= k1) break;
  }
  const double wy = c.dy64[sy];
  double v[3] = {dot, sp * wy, sd * wy};
  if (grid_sum<3>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (lane == 0 && ty == 0) { c.S->dq = v[0]; c.S->sum_p = v[1]; c.S->sum_d = v[2]; c.S->need_update = 1; }
  }
}

template <class T> static DaGeom dav_geom(int nx, int ny, int nz) {
  const int ix = 30 * Vec16<T>::VX;
  const int bxn = (nx + ix - 1) / ix, byn = (ny + kDaVIY - 1) / kDaVIY;
  const int kz = pick_kz((long long)bxn * byn, nz, 2LL * 148, 2, 16);
  DaGeom g; g.kz = kz; g.grid = dim3(bxn, byn, (nz + kz - 1) / kz);
  return g;
}

// Same start, streaming form of k_pcg_dirapplyv (one 16-byte vector of cells per thread, A applied to x0
// through a shared plane and a register queue); bhat is only stored when the caller needs it later (WBH:
// fs_poisson_solve's true residual; fs_step gets that from the projection).
template <class T, int PC, bool WBH> __global__ void __launch_bounds__(32 * kDaTY, 2) k_pcg_initv(const Ctx<T> c, int kz, Launch L, const __grid_constant__ TmapSet tm) {
  constexpr int VX = Vec16<T>::VX;
  constexpr int ROWE = 32 * VX;
  constexpr int PLN = kDaTY * ROWE;
  using W = Vec16<T>;
  __shared__ __align__(16) T D[2 * PLN];
  __shared__ double sh[4 * 32]; __shared__ int flag;
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = (blockIdx.x * 30 - 1 + lane) * VX, gy = blockIdx.y * kDaVIY - 1 + ty;
  const int sx = c.bx ? min(max(gx, 0), c.nx - VX) : wrapi(gx, c.nx);
  const int sy = c.by ? min(max(gy, 0), c.ny - 1) : wrapi(gy, c.ny);
  const bool fixl = c.bx && gx < 0, fixr = c.bx && gx >= c.nx;
  const bool own = lane >= 1 && lane <= 30 && ty >= 1 && ty <= kDaTY - 2 && gx < c.nx && gy < c.ny;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  const unsigned pl = (unsigned)c.nx * c.ny, row = (unsigned)sx + (unsigned)c.nx * sy;
  const T cyl = c.cyl[sy], cyh = c.cyh[sy], idy = c.idy[sy + 1], dyj = c.dy[sy + 1], ndy = -dyj;
  const T ihx2 = c.ihx2, ihz2 = c.ihz2;
  const T shift = T(c.S->mean_coef) * dyj;
  T dg[VX], ivi[VX], ivb[VX];
#pragma unroll
  for (int a = 0; a < VX; ++a) {
    const int i = sx + a;
    dg[a] = PC == 1 ? T((c.bx && i == 0 ? 0 : 1) + (c.bx && i == c.nx - 1 ? 0 : 1)) * ihx2 + (cyh + cyl) * idy : T(0);
    // reciprocal diagonals for planes with two / one z neighbours (see k_pcg_dirapply2)
    ivi[a] = PC == 1 ? T(1) / ((dg[a] + T(2) * ihz2) * dyj) : T(1);
    ivb[a] = PC == 1 ? T(1) / ((dg[a] + T(1) * ihz2) * dyj) : T(1);
  }
  const int o_own = ty * ROWE + lane * VX;
  const int o_s = (ty > 0 ? ty - 1 : 0) * ROWE + lane * VX, o_n = (ty < kDaTY - 1 ? ty + 1 : ty) * ROWE + lane * VX;
  const int o_w = ty * ROWE + (lane > 0 ? lane * VX - 1 : 0), o_e = ty * ROWE + (lane < 31 ? lane * VX + VX : 32 * VX - 1);
  auto fetch = [&](int k) {
    const int ks = c.bz ? min(max(k, 0), c.nz - 1) : (k < 0 ? k + c.nz : (k >= c.nz ? k - c.nz : k));
    W d = ld16<T>(c.p + (row + pl * (unsigned)ks));
    if (fixl) {
#pragma unroll
      for (int a = 1; a < VX; ++a) d.a[a] = d.a[0];
    }
    if (fixr) {
#pragma unroll
      for (int a = 0; a < VX - 1; ++a) d.a[a] = d.a[VX - 1];
    }
    return d;
  };
  // tile planes of x0 and of the right-hand side go to L2 kPfAhead planes before the register loads (TMA, one thread)
  const bool pf_on = tm.n > 0 && lane == 0 && ty == 0;
  const int pf_x = (blockIdx.x * 30 - 1) * VX, pf_y = blockIdx.y * kDaVIY - 1;
  auto prefetch = [&](int k) {
    if (!pf_on || k > k1) return;
    tma_prefetch_plane(tm.m[0], pf_x, pf_y, c.bz ? min(k, c.nz - 1) : (k >= c.nz ? k - c.nz : k));
    if (k < k1) tma_prefetch_plane(tm.m[1], pf_x, pf_y, k);
  };
  for (int k = k0 + 2; k < k0 + 2 + kPfAhead; ++k) prefetch(k);
  W d0 = fetch(k0 - 1), d1 = fetch(k0), d2, nx1 = fetch(k0 + 1);
  W rb;                                     // raw right-hand side of the plane about to be processed
#pragma unroll
  for (int a = 0; a < VX; ++a) rb.a[a] = T(0);
  if (own) rb = ld16<T>(c.r + (row + pl * (unsigned)k0));
  int b = 0;
  st16<T>(D + o_own, d1);
  __syncthreads();
  double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0;
  auto step = [&](int k, const W& dB, const W& dC, W& dT) {
    dT = nx1;
    prefetch(k + 2 + kPfAhead);
    if (k + 1 < k1) nx1 = fetch(k + 2);
    const W rcur = rb;
    if (own && k + 1 < k1) rb = ld16<T>(c.r + (row + pl * (unsigned)(k + 1)));
    const T* P = D + b;
    const W Sv = ld16<T>(P + o_s), Nv = ld16<T>(P + o_n);
    const T xw0 = P[o_w], xeL = P[o_e];
    if (own) {
      const bool zb = PC == 1 && c.bz && (k == 0 || k == c.nz - 1);
      W r, bh;
      T s0 = T(0), s1 = T(0), s2 = T(0), s3 = T(0);
#pragma unroll
      for (int a = 0; a < VX; ++a) {
        const T xc = dC.a[a];
        const T xw = a > 0 ? dC.a[a > 0 ? a - 1 : 0] : xw0;
        const T xe = a < VX - 1 ? dC.a[a < VX - 1 ? a + 1 : a] : xeL;
        T acc = (xe - xc) * ihx2 - (xc - xw) * ihx2;
        acc += ((Nv.a[a] - xc) * cyh - (xc - Sv.a[a]) * cyl) * idy;
        acc += (dT.a[a] - xc) * ihz2 - (xc - dB.a[a]) * ihz2;
        bh.a[a] = rcur.a[a] - shift;
        r.a[a] = bh.a[a] - acc * ndy;
        const T z = PC == 1 ? r.a[a] * (zb ? ivb[a] : ivi[a]) : r.a[a];
        s0 += bh.a[a] * bh.a[a]; s1 += r.a[a] * r.a[a]; s2 += r.a[a] * z; s3 += r.a[a];
      }
      const unsigned o = row + pl * (unsigned)k;
      st16<T>(c.r + o, r);
      if (WBH) st16<T>(c.bh + o, bh);
      v0 += (double)s0; v1 += (double)s1; v2 += (double)s2; v3 += (double)s3;
    }
    b = PLN - b;
    st16<T>(D + b + o_own, dT);
    __syncthreads();
  };
  int k = k0;
  for (;;) {
    step(k, d0, d1, d2); if (++k >= k1) break;
    step(k, d1, d2, d0); if (++k >= k1) break;
    step(k, d2, d0, d1); if (++k >= k1) break;
  }
  double v[4] = {v0, v1, v2, v3};
  if (grid_sum<4>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (lane == 0 && ty == 0) {
      Scalars* S = c.S;
      S->bnorm2 = v[0]; S->rr = v[1]; S->rho_cur = v[2]; S->rho_prev = 1.0; S->dq = 1.0;
      S->iter = 0; S->body_runs = 0; S->first = 1; S->dsel = 0; S->pending = 0; S->rsel = 0; S->need_update = 0;
      S->rmean = v[3] / ((double)c.nx * c.ny * c.nz);
      const int conv = (v[0] == 0.0) || (sqrt(v[1]) <= S->rtol * sqrt(v[0]));
      S->converged = conv; S->done = conv || S->max_iter <= 0;
      if (L.use_cond) cudaGraphSetConditional(L.cond, S->done ? 0u : 1u);
    }
  }
}

// ---- K2: x += alpha d, r -= alpha q fused with ||r||^2 and r.z; loop control -------------------------
// fp32 only: rounding makes sum(q) != 0, so r slowly acquires a component along the null space of A
// (constants) that CG can never remove; once it dominates r the fp32 stencil differences lose all
// accuracy and the iteration diverges.  The mean of r measured by the previous pass is subtracted here
// (one iteration of lag; exactly zero in exact arithmetic, where sum(r) = 0).  fp64 follows O7 literally.
template <class T, bool GMG> __global__ void __launch_bounds__(256) k_pcg_update(const Ctx<T> c, Launch L) {
  __shared__ double sh[3 * 32]; __shared__ int flag;
  Scalars* S = c.S;
  if (S->done) return;
  const double alpha_d = S->rho_cur / S->dq;
  const T alpha = T(alpha_d);
  const long long N = (long long)c.nx * c.ny * c.nz;
  const T rm = sizeof(T) == 4 ? T(S->rmean) : T(0);
  double v[3] = {0.0, 0.0, 0.0};
  if (GMG) {
    // 16-byte accesses; per-vector partial sums in T, accumulated in fp64 (fp32: one conversion per 4 cells)
    constexpr int VW = 16 / sizeof(T);
    using V = typename V16T<T>::type;
    const long long NV = N / VW;
    const V* __restrict__ qv = reinterpret_cast<const V*>(c.q);
    V* __restrict__ rv = reinterpret_cast<V*>(c.r);
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < NV; q += (long long)gridDim.x * blockDim.x) {
      V r = rv[q]; const V qq = qv[q];
      T* re = reinterpret_cast<T*>(&r);
      const T* qe = reinterpret_cast<const T*>(&qq);
      T s2 = T(0), s1 = T(0);
#pragma unroll
      for (int a = 0; a < VW; ++a) {
        T t = re[a] - alpha * qe[a];
        if (sizeof(T) == 4) t -= rm;
        re[a] = t; s2 += t * t; s1 += t;
      }
      rv[q] = r;
      v[0] += (double)s2; v[2] += (double)s1;
    }
    for (long long q = NV * VW + blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
      T r = c.r[q] - alpha * c.q[q];
      if (sizeof(T) == 4) r -= rm;
      c.r[q] = r;
      v[0] += (double)r * (double)r; v[2] += (double)r;
    }
  } else {
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
      T r = c.r[q] - alpha * c.q[q];
      if (sizeof(T) == 4) r -= rm;
      c.r[q] = r;
      v[0] += (double)r * (double)r; v[2] += (double)r;
      const int i = (int)(q % c.nx); const long long t = q / c.nx; const int j = (int)(t % c.ny), k = (int)(t / c.ny);
      v[1] += (double)r * (double)precond_point<T>(c, r, i, j, k);
    }
  }
  if (grid_sum<3>(v, c.partials, &S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0) {
      S->rr = v[0]; S->rmean = v[2] / (double)N;
      S->iter += 1; S->first = 0; S->dsel ^= 1;
      S->alpha_prev = alpha_d; S->pending = 1;       // x += alpha d is applied by the next k_pcg_dirapply or by k_pflush
      S->rho_prev = S->rho_cur;
      if (!GMG) S->rho_cur = v[1];
      const int conv = sqrt(v[0]) <= S->rtol * sqrt(S->bnorm2);
      S->converged = conv;
      S->done = conv || S->iter >= S->max_iter;
      if (L.use_cond) cudaGraphSetConditional(L.cond, S->done ? 0u : 1u);
    }
  }
}

// K2 for the point preconditioners on grids with nx a multiple of the vector width: 3-D indexed (no integer
// division), one 16-byte vector of cells per thread, 32 x 8 threads per CTA marching a z chunk; r.z uses
// z = r / diag A (Jacobi) or z = r (none) with the diagonal assembled from per-cell / per-row / per-plane parts.
template <class T, int PC> __global__ void __launch_bounds__(256) k_pcg_updatev(const Ctx<T> c, int kz, Launch L) {
  constexpr int VX = Vec16<T>::VX;
  using W = Vec16<T>;
  __shared__ double sh[3 * 32]; __shared__ int flag;
  Scalars* S = c.S;
  if (S->done) return;
  const double alpha_d = S->rho_cur / S->dq;
  const T alpha = T(alpha_d);
  const T rm = sizeof(T) == 4 ? T(S->rmean) : T(0);
  const int gx = (blockIdx.x * 32 + threadIdx.x) * VX, gy = blockIdx.y * 8 + threadIdx.y;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  double v[3] = {0.0, 0.0, 0.0};
  if (gx < c.nx && gy < c.ny) {
    const unsigned pl = (unsigned)c.nx * c.ny, o0 = (unsigned)gx + (unsigned)c.nx * gy;
    const T dyj = c.dy[gy + 1];
    T dg[VX], ivi[VX], ivb[VX];
#pragma unroll
    for (int a = 0; a < VX; ++a) {
      const int i = gx + a;
      dg[a] = PC == 1 ? T((c.bx && i == 0 ? 0 : 1) + (c.bx && i == c.nx - 1 ? 0 : 1)) * c.ihx2 + (c.cyh[gy] + c.cyl[gy]) * c.idy[gy + 1] : T(0);
      ivi[a] = PC == 1 ? T(1) / ((dg[a] + T(2) * c.ihz2) * dyj) : T(1);
      ivb[a] = PC == 1 ? T(1) / ((dg[a] + T(1) * c.ihz2) * dyj) : T(1);
    }
#pragma unroll 2
    for (int k = k0; k < k1; ++k) {
      const unsigned o = o0 + pl * (unsigned)k;
      W r = ld16<T>(c.r + o);
      const W q = ld16<T>(c.q + o);
      const bool zb = PC == 1 && c.bz && (k == 0 || k == c.nz - 1);
      T s0 = T(0), s1 = T(0), s2 = T(0);
#pragma unroll
      for (int a = 0; a < VX; ++a) {
        T t = r.a[a] - alpha * q.a[a];
        if (sizeof(T) == 4) t -= rm;
        r.a[a] = t;
        const T z = PC == 1 ? t * (zb ? ivb[a] : ivi[a]) : t;
        s0 += t * t; s1 += t * z; s2 += t;
      }
      st16<T>(c.r + o, r);
      v[0] += (double)s0; v[1] += (double)s1; v[2] += (double)s2;
    }
  }
  if (grid_sum<3>(v, c.partials, &S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0 && threadIdx.y == 0) {
      const double N = (double)c.nx * c.ny * c.nz;
      S->rr = v[0]; S->rmean = v[2] / N;
      S->iter += 1; S->first = 0; S->dsel ^= 1;
      S->alpha_prev = alpha_d; S->pending = 1;
      S->rho_prev = S->rho_cur;
      S->rho_cur = v[1];
      const int conv = sqrt(v[0]) <= S->rtol * sqrt(S->bnorm2);
      S->converged = conv;
      S->done = conv || S->iter >= S->max_iter;
      if (L.use_cond) cudaGraphSetConditional(L.cond, S->done ? 0u : 1u);
    }
  }
}

// ---- GMG: rho = r . (zs z') after the V-cycle ----------------------------------------------------------
template <class T> __global__ void __launch_bounds__(256) k_dot_rz(const Ctx<T> c, T zs) {
  __shared__ double sh[32]; __shared__ int flag;
  if (c.S->done) return;
  const long long N = (long long)c.nx * c.ny * c.nz;
  double v[1] = {0.0};
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x)
    v[0] += (double)c.r[q] * (double)(c.z[q] * zs);
  if (grid_sum<1>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0) c.S->rho_cur = v[0];
  }
}

// tensor maps of n cell-shaped fields with a (boxx, boxy) tile plane box; .n = 0 when prefetching is off, a map cannot be encoded,
// or the periodic x direction is absent (bounded x: tiles are clamped, not prefetched)
template <class T> static TmapSet cell_maps(const Ctx<T>& c, const T* const* f, int n, int boxx, int boxy) {
  static const int on = [] { const char* e = getenv("FS_TUNE_PF2"); return e ? atoi(e) : 1; }();
  TmapSet tm; memset(&tm, 0, sizeof tm);
  if (!on || c.bx) return tm;
  for (int i = 0; i < n; ++i) if (!f[i] || !tmap_encode(&tm.m[i], f[i], sizeof(T), c.nx, c.ny, c.nz, boxx, boxy)) return tm;
  tm.n = n;
  return tm;
}

template <class T> int launch_pcg_init(const Ctx<T>& c, const Launch& L, bool need_bhat) {
  int n = 0;
  const double N = (double)c.nx * c.ny * c.nz;
  if (!c.warm_start) { FS_LAUNCH(L, "memset_p", 1.0 * sizeof(T) * N, cudaMemsetAsync(c.p, 0, sizeof(T) * (size_t)c.nx * c.ny * c.nz, L.s)); ++n; }
  if (c.nx % Vec16<T>::VX == 0) {
    const DaGeom G = dav_geom<T>(c.nx, c.ny, c.nz);
    const dim3 blk(32, kDaTY);
    const bool jac = c.precond == FS_PC_JACOBI;
    const T* pf_f[2] = {c.p, c.r};
    const TmapSet tm = cell_maps<T>(c, pf_f, 2, 32 * Vec16<T>::VX, kDaTY);
    FS_LAUNCHI(L, "pcg_init", sizeof(T) == 8 ? "k_pcg_initv<f64>" : "k_pcg_initv<f32>", (need_bhat ? 4.0 : 3.0) * sizeof(T) * N, {
      if (jac) { if (need_bhat) k_pcg_initv<T, 1, true><<<G.grid, blk, 0, L.s>>>(c, G.kz, L, tm); else k_pcg_initv<T, 1, false><<<G.grid, blk, 0, L.s>>>(c, G.kz, L, tm); }
      else { if (need_bhat) k_pcg_initv<T, 0, true><<<G.grid, blk, 0, L.s>>>(c, G.kz, L, tm); else k_pcg_initv<T, 0, false><<<G.grid, blk, 0, L.s>>>(c, G.kz, L, tm); }
    });
    return n + 1;
  }
  ColGeom g = col_geom(c.nx, c.ny, c.nz);
  FS_LAUNCHI(L, "pcg_init", sizeof(T) == 8 ? "k_pcg_init<f64>" : "k_pcg_init<f32>", 4.0 * sizeof(T) * N, k_pcg_init<T><<<g.grid, g.block, 0, L.s>>>(c, g.kz, L));
  return n + 1;
}

template <class T> int launch_pcg_body(const Ctx<T>& c, const MgCtx<T>& mg, const Launch& L) {
  const long long N = (long long)c.nx * c.ny * c.nz;
  int n = 0;
  bool upd_fused = false;                  // K2 done by the level-0 down kernel of the NEXT iteration (k_mg_down<UPD>)
  T zs = T(1);
  if (c.precond == FS_PC_GMG) {
    zs = T(1.0 / c.hy);
    bool fused = false;
    n += launch_vcycle<T>(c, mg, c.r, c.z, L, &fused, zs, &upd_fused);
    if (!fused) { FS_LAUNCH(L, "pcg_dot_rz", 2.0 * sizeof(T) * N, k_dot_rz<T><<<flat_blocks(N), 256, 0, L.s>>>(c, zs)); ++n; }
  }
  if (sizeof(T) == 8 && c.nx % 2 == 0) {
    const DaGeom G = da2_geom(c.nx, c.ny, c.nz);
    const dim3 blk(32, kDaTY);
    if (c.precond == FS_PC_GMG) FS_LAUNCHI(L, "pcg_dir_apply_dot", "k_pcg_dirapply2<f64>", 6.0 * sizeof(T) * N, k_pcg_dirapply2<T, 2><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    else if (c.precond == FS_PC_JACOBI) FS_LAUNCHI(L, "pcg_dir_apply_dot", "k_pcg_dirapply2<f64>", 6.0 * sizeof(T) * N, k_pcg_dirapply2<T, 1><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    else FS_LAUNCHI(L, "pcg_dir_apply_dot", "k_pcg_dirapply2<f64>", 6.0 * sizeof(T) * N, k_pcg_dirapply2<T, 0><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    ++n;
  } else if (sizeof(T) == 4 && c.nx % 4 == 0) {
    const DaGeom G = dav_geom<T>(c.nx, c.ny, c.nz);
    const dim3 blk(32, kDaTY);
    if (c.precond == FS_PC_GMG) FS_LAUNCHI(L, "pcg_dir_apply_dot", "k_pcg_dirapplyv<f32>", 6.0 * sizeof(T) * N, k_pcg_dirapplyv<T, 2><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    else if (c.precond == FS_PC_JACOBI) FS_LAUNCHI(L, "pcg_dir_apply_dot", "k_pcg_dirapplyv<f32>", 6.0 * sizeof(T) * N, k_pcg_dirapplyv<T, 1><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    else FS_LAUNCHI(L, "pcg_dir_apply_dot", "k_pcg_dirapplyv<f32>", 6.0 * sizeof(T) * N, k_pcg_dirapplyv<T, 0><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    ++n;
  } else {
    const DaGeom G = da_geom(c.nx, c.ny, c.nz);
    const dim3 blk(kDaTX, kDaTY);
    if (c.precond == FS_PC_GMG) FS_LAUNCHI(L, "pcg_dir_apply_dot", sizeof(T) == 8 ? "k_pcg_dirapply<f64>" : "k_pcg_dirapply<f32>", 6.0 * sizeof(T) * N, k_pcg_dirapply<T, 2><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    else if (c.precond == FS_PC_JACOBI) FS_LAUNCHI(L, "pcg_dir_apply_dot", sizeof(T) == 8 ? "k_pcg_dirapply<f64>" : "k_pcg_dirapply<f32>", 6.0 * sizeof(T) * N, k_pcg_dirapply<T, 1><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    else FS_LAUNCHI(L, "pcg_dir_apply_dot", sizeof(T) == 8 ? "k_pcg_dirapply<f64>" : "k_pcg_dirapply<f32>", 6.0 * sizeof(T) * N, k_pcg_dirapply<T, 0><<<G.grid, blk, 0, L.s>>>(c, zs, G.kz));
    ++n;
  }
  if (upd_fused) return n;
  if (c.precond == FS_PC_GMG) FS_LAUNCHI(L, "pcg_update_norm", sizeof(T) == 8 ? "k_pcg_update<f64,GMG>" : "k_pcg_update<f32,GMG>", 3.0 * sizeof(T) * N, k_pcg_update<T, true><<<flat_blocks(N), 256, 0, L.s>>>(c, L));
  else if (c.nx % Vec16<T>::VX == 0) {
    const int bxn = (c.nx + 32 * Vec16<T>::VX - 1) / (32 * Vec16<T>::VX), byn = (c.ny + 7) / 8;
    int kz = c.nz;
    while (kz > 4 && (long long)bxn * byn * ((c.nz + kz - 1) / kz) < 8LL * 148) kz = (kz + 1) / 2;
    while ((long long)bxn * byn * ((c.nz + kz - 1) / kz) > kMaxPartials) kz *= 2;
    const dim3 grid(bxn, byn, (c.nz + kz - 1) / kz), blk(32, 8);
    if (c.precond == FS_PC_JACOBI) FS_LAUNCHI(L, "pcg_update_norm", sizeof(T) == 8 ? "k_pcg_updatev<f64>" : "k_pcg_updatev<f32>", 3.0 * sizeof(T) * N, k_pcg_updatev<T, 1><<<grid, blk, 0, L.s>>>(c, kz, L));
    else FS_LAUNCHI(L, "pcg_update_norm", sizeof(T) == 8 ? "k_pcg_updatev<f64>" : "k_pcg_updatev<f32>", 3.0 * sizeof(T) * N, k_pcg_updatev<T, 0><<<grid, blk, 0, L.s>>>(c, kz, L));
  } else FS_LAUNCHI(L, "pcg_update_norm", sizeof(T) == 8 ? "k_pcg_update<f64>" : "k_pcg_update<f32>", 3.0 * sizeof(T) * N, k_pcg_update<T, false><<<flat_blocks(N), 256, 0, L.s>>>(c, L));
  ++n;
  return n;
}

// ---- after the loop: last deferred x update and zero-mean pressure (volume-weighted), SURVEY O6 -------
// With at least one iteration the mean of the final x follows from the sums k_pcg_dirapply left behind
// (sum x dV before the last update, sum d dV), so one pass does x += alpha d - mean.  With no iteration
// (converged at the start) the plain mean + shift kernels run instead; each kernel checks which case holds.
template <class T> __global__ void __launch_bounds__(256) k_pflush(const Ctx<T> c) {
  const Scalars* S = c.S;
  if (!S->pending) return;
  const long long N = (long long)c.nx * c.ny * c.nz;
  const double al = S->alpha_prev;
  const T alpha = T(al), m = T((S->sum_p + al * S->sum_d) / S->sum_dy);
  const T* __restrict__ dcur = S->dsel ? c.d2 : c.d;     // the direction of the last iteration
  constexpr int VW = 16 / sizeof(T);
  using V = typename V16T<T>::type;
  const long long NV = N / VW;
  const V* __restrict__ dv = reinterpret_cast<const V*>(dcur);
  V* __restrict__ pv = reinterpret_cast<V*>(c.p);
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < NV; q += (long long)gridDim.x * blockDim.x) {
    V p = pv[q]; const V d = dv[q];
    T* pe = reinterpret_cast<T*>(&p); const T* de = reinterpret_cast<const T*>(&d);
#pragma unroll
    for (int a = 0; a < VW; ++a) pe[a] = (pe[a] + alpha * de[a]) - m;
    pv[q] = p;
  }
  for (long long q = NV * VW + blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x)
    c.p[q] = (c.p[q] + alpha * dcur[q]) - m;
}
template <class T> __global__ void __launch_bounds__(256) k_pmean(const Ctx<T> c) {
  __shared__ double sh[32]; __shared__ int flag;
  if (c.S->pending) return;
  const long long N = (long long)c.nx * c.ny * c.nz;
  double v[1] = {0.0};
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    const int j = (int)((q / c.nx) % c.ny);
    v[0] += (double)c.p[q] * c.dy64[j];
  }
  if (grid_sum<1>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0) c.S->pmean = v[0] / c.S->sum_dy;
  }
}
template <class T> __global__ void __launch_bounds__(256) k_pshift(const Ctx<T> c) {
  if (c.S->pending) return;
  const long long N = (long long)c.nx * c.ny * c.nz;
  const T m = T(c.S->pmean);
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) c.p[q] -= m;
}
template <class T> __global__ void k_pflush_done(const Ctx<T> c) { c.S->pending = 0; }
template <class T> int launch_pcg_finish(const Ctx<T>& c, const Launch& L) {
  const long long N = (long long)c.nx * c.ny * c.nz;
  FS_LAUNCH(L, "p_mean", 0.0, k_pmean<T><<<flat_blocks(N), 256, 0, L.s>>>(c));
  FS_LAUNCH(L, "p_shift", 0.0, k_pshift<T><<<flat_blocks(N), 256, 0, L.s>>>(c));
  FS_LAUNCH(L, "p_flush_mean", 3.0 * sizeof(T) * N, k_pflush<T><<<flat_blocks(N), 256, 0, L.s>>>(c));
  FS_LAUNCH(L, "p_flush_mean", 0.0, k_pflush_done<T><<<1, 1, 0, L.s>>>(c));
  return 4;
}

// ---- true residual ||bhat - A p||^2 (fs_poisson_solve; fs_step gets it from the projection) ---------
template <class T> __global__ void __launch_bounds__(256) k_true_res(const Ctx<T> c, int kz) {
  __shared__ double sh[32]; __shared__ int flag;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  double v[1] = {0.0};
  if (i < c.nx && j < c.ny) {
    march_A<T>(c, c.p, i, j, k0, k1, [&](int k, size_t q, T xc, T Ax) {
      const double e = (double)c.bh[q] - (double)Ax;
      v[0] += e * e;
    });
  }
  if (grid_sum<1>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0 && threadIdx.y == 0) c.S->true_rr = v[0];
  }
}
template <class T> int launch_true_residual(const Ctx<T>& c, const Launch& L) {
  ColGeom g = col_geom(c.nx, c.ny, c.nz);
  FS_LAUNCH(L, "true_residual", 2.0 * sizeof(T) * c.nx * c.ny * c.nz, k_true_res<T><<<g.grid, g.block, 0, L.s>>>(c, g.kz));
  return 1;
}

#define INST(T)                                                                   \
  template int launch_pcg_init<T>(const Ctx<T>&, const Launch&, bool);                  \
  template int launch_pcg_body<T>(const Ctx<T>&, const MgCtx<T>&, const Launch&); \
  template int launch_pcg_finish<T>(const Ctx<T>&, const Launch&);                \
  template int launch_true_residual<T>(const Ctx<T>&, const Launch&);
INST(float)
INST(double)

}  // namespace fs
