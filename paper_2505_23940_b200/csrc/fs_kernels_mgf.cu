// fs_kernels_mgf.cu -- fused, temporally blocked kernels of the V(2,2) cycle (S7g).
//
// The unfused cycle moves 15.25 words per fine cell (first 2, sweep 3 x3, residual+restrict 2.125,
// prolong+correct 2.125); the two kernels here move 2.125 + 3.125:
//   k_mg_down : g -> e = two damped-Jacobi sweeps from a zero guess, gc = R (g - (-L) e)
//   k_mg_up   : e, ec, g -> e' = two sweeps applied to (e + P ec)   [level 0: also r . z for PCG]
// Both are 2.5-D streaming kernels: a CTA owns an xy tile and marches in z.  A thread owns two x-adjacent
// cells (16-byte loads for fp64, 8 for fp32), keeps the z neighbours of every pipeline stage in a register
// queue, gets the x and y neighbours
// through a double-buffered shared-memory plane (a warp is one row of the tile); one __syncthreads per plane.  Each later stage is valid on
// a tile one cell smaller per side (overlapped tiling: 64 x TY extended tile -> 60 x (TY-4) results); the
// halo re-reads hit L2.  All grids are periodic (GMG is only offered for triply periodic boxes).
#include "fs_internal.cuh"

namespace fs {


constexpr int kMgTY = 16;                 // rows of the extended tile
constexpr int kMgIX = 60, kMgIY = kMgTY - 4;

__device__ __forceinline__ int modp(int a, int n) { a %= n; return a < 0 ? a + n : a; }

struct MgGeom { dim3 grid; int zchunks; };
static MgGeom mg_geom(int nx, int ny, int nz) {
  const int bxn = (nx + kMgIX - 1) / kMgIX, byn = (ny + kMgIY - 1) / kMgIY;
  const long long slots = 2LL * 148;      // two CTAs of 512 threads per SM
  int best = 1; double best_cost = 1e300;
  for (int zc = 1; zc <= 64 && nz / zc >= 8; ++zc) {
    const long long blocks = (long long)bxn * byn * zc;
    if (blocks > kMaxPartials) break;
    const long long waves = (blocks + slots - 1) / slots;
    const double planes = (double)((nz / 2 + zc - 1) / zc * 2 + 4);
    const double cost = (double)waves * planes;
    if (cost < best_cost * 0.999) { best_cost = cost; best = zc; }
  }
  MgGeom g; g.zchunks = best; g.grid = dim3(bxn, byn, best);
  return g;
}
// even chunk boundaries
__device__ __forceinline__ int chunk_lo(int c, int nchunks, int nz) { return 2 * (int)(((long long)c * (nz / 2)) / nchunks); }


constexpr int kMgPL = kMgTY * 32;         // pairs per shared-memory plane

// Shared-memory positions of a thread: own pair, the rows below / above, the pairs left / right (clamped at
// the tile edge: edge results are never used).
struct MgPos { int own, s, n, w, e; };
__device__ __forceinline__ MgPos mg_pos(int lane, int ty) {
  MgPos p;
  p.own = ty * 32 + lane;
  p.s = (ty > 0 ? ty - 1 : 0) * 32 + lane;
  p.n = (ty < kMgTY - 1 ? ty + 1 : ty) * 32 + lane;
  p.w = ty * 32 + (lane > 0 ? lane - 1 : 0);
  p.e = ty * 32 + (lane < 31 ? lane + 1 : 31);
  return p;
}
// sum of the six neighbours of both cells of the pair c held at plane buffer P (the pair's own plane);
// zm / zp = the pairs below / above (register queue).
template <class T, class V> __device__ __forceinline__ V nb6(const V* __restrict__ P, const MgPos& q, const V& c, const V& zm, const V& zp) {
  const V S = P[q.s], N = P[q.n];
  const T left = P[q.w].y, right = P[q.e].x;
  V r;
  r.x = ((left + c.y) + (S.x + N.x)) + (zm.x + zp.x);
  r.y = ((c.x + right) + (S.y + N.y)) + (zm.y + zp.y);
  return r;
}

// ---- downward leg: e = S^2(0; g), gc = R (g - (-L) e) -----------------------------------------------------
// Two damped-Jacobi sweeps from a zero guess collapse to e = cg g + cn nb(g) with cg = 2 cw - 6 cw^2 / h^2,
// cn = cw^2 / h^2  (first sweep: cw g; second: cw g + cw (g - (6 cw g - cw nb) / h^2)).
// The z loop is unrolled three times so that the register queues rotate by renaming.
template <class T> __global__ void __launch_bounds__(32 * kMgTY, 2)
k_mg_down(const int* __restrict__ done, const T* __restrict__ g, T* __restrict__ eo, T* __restrict__ gc,
          int nx, int ny, int nz, T cg, T cn, T ih2) {
  using V = typename V2T<T>::type;
  if (done && *done) return;
  __shared__ V G[2 * kMgPL];
  __shared__ V E[2 * kMgPL];
  __shared__ T R[2 * kMgPL];
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = blockIdx.x * kMgIX - 2 + 2 * lane, gy = blockIdx.y * kMgIY - 2 + ty;
  const unsigned pl = (unsigned)nx * ny, row = (unsigned)modp(gx, nx) + (unsigned)nx * modp(gy, ny);
  const bool interior = lane >= 1 && lane <= 30 && ty >= 2 && ty < kMgTY - 2 && gx < nx && gy < ny;
  const bool comb = interior && ((ty & 1) == 0);
  const int z0 = chunk_lo(blockIdx.z, gridDim.z, nz), z1 = chunk_lo(blockIdx.z + 1, gridDim.z, nz);
  const int tend = z1 + 1;
  const MgPos q = mg_pos(lane, ty);
  const unsigned cpl = (unsigned)(nx >> 1) * (ny >> 1), crow = (unsigned)(gx >> 1) + (unsigned)(nx >> 1) * (gy >> 1);
  const T m6 = T(-6) * ih2;
  T acc = T(0);
  int zl = modp(z0 - 2, nz);              // plane of the load in flight
  int b = 0;                              // buffer of plane t (toggles); plane t-1 lives in kMgPL - b
  V nxt = ldv2<T, V>(g + (row + pl * zl));
  // one plane: gA, gB = g(t-2), g(t-1); gC receives g(t).  eA, eB = e(t-3), e(t-2); eC receives e(t-1).
  auto step = [&](int t, const V& gA, const V& gB, V& gC, const V& eA, const V& eB, V& eC) {
    gC = nxt;
    if (t < tend) { zl = zl + 1 == nz ? 0 : zl + 1; nxt = ldv2<T, V>(g + (row + pl * zl)); }
    const int pb = kMgPL - b;
    if (t >= z0) {            // e(t-1)
      const V nb = nb6<T, V>(G + pb, q, gB, gA, gC);
      eC.x = cg * gB.x + cn * nb.x; eC.y = cg * gB.y + cn * nb.y;
    }
    if (t >= z0 + 2) {        // residual at plane t-2, its x-pair sum, store of e(t-2)
      const V nb = nb6<T, V>(E + b, q, eB, eA, eC);
      const T rx = (gA.x + m6 * eB.x) + ih2 * nb.x;
      const T ry = (gA.y + m6 * eB.y) + ih2 * nb.y;
      R[b + q.own] = rx + ry;
      if (interior) stv2<T, V>(eo + (row + pl * (unsigned)(t - 2)), eB);
    }
    G[b + q.own] = gC;
    if (t >= z0) E[pb + q.own] = eC;
    __syncthreads();
    if (t >= z0 + 2 && comb) {
      acc += R[b + q.own] + R[b + q.own + 32];
      if ((t - z0) & 1) { gc[crow + cpl * (unsigned)((t - 2) >> 1)] = T(0.125) * acc; acc = T(0); }
    }
    b = pb;
  };
  const V zero = {T(0), T(0)};
  V g0 = zero, g1 = zero, g2 = zero, e0 = zero, e1 = zero, e2 = zero;
  int t = z0 - 2;
  for (;;) {
    step(t, g0, g1, g2, e0, e1, e2); if (++t > tend) break;
    step(t, g1, g2, g0, e1, e2, e0); if (++t > tend) break;
    step(t, g2, g0, g1, e2, e0, e1); if (++t > tend) break;
  }
}

// ---- upward leg: e' = S^2(e + P ec; g); DOT (level 0 inside PCG): rho = r . (zs e') ---------------------
// One sweep: e + cw (g - (6 e - nb) / h^2) = ce e + cw g + cn nb with ce = 1 - 6 cw / h^2, cn = cw / h^2.
template <class T, bool DOT> __global__ void __launch_bounds__(32 * kMgTY, 2)
k_mg_up(const int* __restrict__ done, const T* __restrict__ ein, const T* __restrict__ ec, const T* __restrict__ g,
        T* __restrict__ eo, int nx, int ny, int nz, T ce, T cw, T cn, T zs, Scalars* S_, double* partials) {
  using V = typename V2T<T>::type;
  if (done && *done) return;
  __shared__ V A[2 * kMgPL];
  __shared__ V B[2 * kMgPL];
  __shared__ double sh[32]; __shared__ int flag;
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = blockIdx.x * kMgIX - 2 + 2 * lane, gy = blockIdx.y * kMgIY - 2 + ty;
  const int gxw = modp(gx, nx), gyw = modp(gy, ny);
  const unsigned pl = (unsigned)nx * ny, row = (unsigned)gxw + (unsigned)nx * gyw;
  const bool interior = lane >= 1 && lane <= 30 && ty >= 2 && ty < kMgTY - 2 && gx < nx && gy < ny;
  const int z0 = chunk_lo(blockIdx.z, gridDim.z, nz), z1 = chunk_lo(blockIdx.z + 1, gridDim.z, nz);
  const int tend = z1 + 1;
  const MgPos q = mg_pos(lane, ty);
  const unsigned cpl = (unsigned)(nx >> 1) * (ny >> 1), crow = (unsigned)(gxw >> 1) + (unsigned)(nx >> 1) * (gyw >> 1);
  double dot = 0.0;
  int zl = modp(z0 - 2, nz);              // plane of the e / ec load in flight; the g load in flight is one plane behind
  int b = 0;
  V nxa = ldv2<T, V>(ein + (row + pl * zl));
  T nxc = ec[crow + cpl * (unsigned)(zl >> 1)];
  const V zero = {T(0), T(0)};
  V nxg = zero;
  // aA, aB = (e + P ec)(t-2), (t-1); aC receives plane t.  bA, bB = first post-sweep at t-3, t-2; bC receives t-1.
  // gA = g(t-2); gB receives g(t-1).
  auto step = [&](int t, const V& aA, const V& aB, V& aC, const V& bA, const V& bB, V& bC, const V& gA, V& gB) {
    aC.x = nxa.x + nxc; aC.y = nxa.y + nxc;
    gB = nxg;
    if (t < tend) {
      nxg = ldv2<T, V>(g + (row + pl * zl));           // plane t
      zl = zl + 1 == nz ? 0 : zl + 1;
      nxa = ldv2<T, V>(ein + (row + pl * zl));         // plane t+1
      nxc = ec[crow + cpl * (unsigned)(zl >> 1)];
    }
    const int pb = kMgPL - b;
    if (t >= z0) {            // first post-sweep at plane t-1
      const V nb = nb6<T, V>(A + pb, q, aB, aA, aC);
      bC.x = (ce * aB.x + cw * gB.x) + cn * nb.x;
      bC.y = (ce * aB.y + cw * gB.y) + cn * nb.y;
    }
    if (t >= z0 + 2) {        // second post-sweep at plane t-2
      const V nb = nb6<T, V>(B + b, q, bB, bA, bC);
      V o;
      o.x = (ce * bB.x + cw * gA.x) + cn * nb.x;
      o.y = (ce * bB.y + cw * gA.y) + cn * nb.y;
      if (interior) {
        stv2<T, V>(eo + (row + pl * (unsigned)(t - 2)), o);
        if (DOT) dot += (double)gA.x * (double)(o.x * zs) + (double)gA.y * (double)(o.y * zs);
      }
    }
    A[b + q.own] = aC;
    if (t >= z0) B[pb + q.own] = bC;
    __syncthreads();
    b = pb;
  };
  V a0 = zero, a1 = zero, a2 = zero, b0 = zero, b1 = zero, b2 = zero, g0 = zero, g1 = zero;
  int t = z0 - 2;
  for (;;) {
    step(t, a0, a1, a2, b0, b1, b2, g0, g1); if (++t > tend) break;
    step(t, a1, a2, a0, b1, b2, b0, g1, g0); if (++t > tend) break;
    step(t, a2, a0, a1, b2, b0, b1, g0, g1); if (++t > tend) break;
    step(t, a0, a1, a2, b0, b1, b2, g1, g0); if (++t > tend) break;
    step(t, a1, a2, a0, b1, b2, b0, g0, g1); if (++t > tend) break;
    step(t, a2, a0, a1, b2, b0, b1, g1, g0); if (++t > tend) break;
  }
  if (DOT) {
    double v[1] = {dot};
    if (grid_sum<1>(v, partials, &S_->ticket[0], sh, &flag)) {
      if (threadIdx.x == 0 && threadIdx.y == 0) S_->rho_cur = v[0];
    }
  }
}

template <class T> int launch_mg_down(const Ctx<T>& c, const T* g, T* e, T* gc, int nx, int ny, int nz, double h, double omega,
                                      const char* name, const Launch& L) {
  const MgGeom G = mg_geom(nx, ny, nz);
  const double N = (double)nx * ny * nz;
  const double ih2 = 1.0 / (h * h), cw = omega * h * h / 6.0;
  FS_LAUNCH(L, name, 2.125 * sizeof(T) * N,
            k_mg_down<T><<<G.grid, dim3(32, kMgTY), 0, L.s>>>(&c.S->done, g, e, gc, nx, ny, nz, T(2.0 * cw - 6.0 * cw * cw * ih2), T(cw * cw * ih2), T(ih2)));
  return 1;
}
template <class T> int launch_mg_up(const Ctx<T>& c, const T* ein, const T* ec, const T* g, T* eo, int nx, int ny, int nz, double h,
                                    double omega, bool dot, T zs, const char* name, const Launch& L) {
  const MgGeom G = mg_geom(nx, ny, nz);
  const double N = (double)nx * ny * nz;
  const double ih2d = 1.0 / (h * h), cwd = omega * h * h / 6.0;
  const T ce = T(1.0 - 6.0 * cwd * ih2d), cw = T(cwd), cn = T(cwd * ih2d);
  if (dot) FS_LAUNCH(L, name, 3.125 * sizeof(T) * N, k_mg_up<T, true><<<G.grid, dim3(32, kMgTY), 0, L.s>>>(&c.S->done, ein, ec, g, eo, nx, ny, nz, ce, cw, cn, zs, c.S, c.partials));
  else FS_LAUNCH(L, name, 3.125 * sizeof(T) * N, k_mg_up<T, false><<<G.grid, dim3(32, kMgTY), 0, L.s>>>(&c.S->done, ein, ec, g, eo, nx, ny, nz, ce, cw, cn, zs, c.S, c.partials));
  return 1;
}

#define INST(T)                                                                                                              \
  template int launch_mg_down<T>(const Ctx<T>&, const T*, T*, T*, int, int, int, double, double, const char*, const Launch&); \
  template int launch_mg_up<T>(const Ctx<T>&, const T*, const T*, const T*, T*, int, int, int, double, double, bool, T, const char*, const Launch&);
INST(float)
INST(double)

}  // namespace fs
