// fs_kernels_mgf.cu -- fused, temporally blocked kernels of the V(2,2) cycle (S7g).
//
// The unfused cycle moves 15.25 words per fine cell (first 2, sweep 3 x3, residual+restrict 2.125,
// prolong+correct 2.125); the two kernels here move 2.125 + 3.125:
//   k_mg_down : g -> e = two damped-Jacobi sweeps from a zero guess, gc = R (g - (-L) e)
//   k_mg_up   : e, ec, g -> e' = two sweeps applied to (e + P ec)   [level 0: also r . z for PCG]
// Both are 2.5-D streaming kernels: a CTA owns an xy tile and marches in z.  A thread owns a 2 x 2 patch of
// cells (two x-adjacent pairs: 16-byte global accesses for fp64, 8 for fp32; the patch is exactly one coarse
// cell, so restriction and prolongation need no exchange), keeps the z neighbours of every pipeline stage
// in a register queue that rotates by renaming (z loop unrolled), and exchanges only the patch edges through
// double-buffered shared-memory planes (separate planes for the even and the odd x column, so that every
// shared access is a compact row: the kernels are bound by shared-memory wavefronts, not by HBM, if the
// patch is smaller -- profiles/).  One __syncthreads per plane.  Each later stage is valid on a tile one
// cell smaller per side (overlapped tiling: 64 x 2TR extended tile -> 60 x (2TR-4) results); the halo
// re-reads hit L2.  All grids are periodic (GMG is only offered for triply periodic boxes).
#include "fs_internal.cuh"
#include <cstdlib>
#include <cstring>

namespace fs {

constexpr int kMgIX = 60;                 // result columns per tile (extended tile: 64 = 32 lanes x 2)
constexpr int kMgAhead = 4;               // k_mg_up: planes between an L2 prefetch and the register load of the same data
template <int TR> struct MgTile { static constexpr int ROWS = 2 * TR, IY = 2 * TR - 4, PL = 2 * TR * 32; };

__device__ __forceinline__ int modp(int a, int n) { a %= n; return a < 0 ? a + n : a; }

struct MgGeom { dim3 grid; int zchunks; };
static MgGeom mg_geom(int nx, int ny, int nz, int iy, int slots_per_sm) {
  const int bxn = (nx + kMgIX - 1) / kMgIX, byn = (ny + iy - 1) / iy;
  const long long slots = 148LL * slots_per_sm;
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

// A thread's 2 x 2 patch at one plane: lo = pair of row 2 ty, hi = pair of row 2 ty + 1.
template <class T> struct Quad { typename V2T<T>::type lo, hi; };

// Shared-memory offsets of a thread (elements of T inside one plane of ROWS x 32).
struct MgPos { int own0, s, n, w0, e0; };
template <int TR> __device__ __forceinline__ MgPos mg_pos(int lane, int ty) {
  const int r0 = 2 * ty, rs = r0 > 0 ? r0 - 1 : 0, rn = r0 + 2 < 2 * TR ? r0 + 2 : r0 + 1;
  MgPos p;
  p.own0 = r0 * 32 + lane; p.s = rs * 32 + lane; p.n = rn * 32 + lane;
  p.w0 = r0 * 32 + (lane > 0 ? lane - 1 : 0); p.e0 = r0 * 32 + (lane < 31 ? lane + 1 : 31);
  return p;
}
// Sum of the six neighbours of the four cells of patch c, whose plane is in the shared planes X (even
// columns) / Y (odd columns); zm / zp = the patches below / above (register queue).
template <class T> __device__ __forceinline__ Quad<T> nbq(const T* __restrict__ X, const T* __restrict__ Y, const MgPos& q,
                                                         const Quad<T>& c, const Quad<T>& zm, const Quad<T>& zp) {
  const T sx = X[q.s], sy = Y[q.s], nx_ = X[q.n], ny_ = Y[q.n];
  const T w0 = Y[q.w0], e0 = X[q.e0], w1 = Y[q.w0 + 32], e1 = X[q.e0 + 32];
  Quad<T> r;
  r.lo.x = ((w0 + c.lo.y) + (sx + c.hi.x)) + (zm.lo.x + zp.lo.x);
  r.lo.y = ((c.lo.x + e0) + (sy + c.hi.y)) + (zm.lo.y + zp.lo.y);
  r.hi.x = ((w1 + c.hi.y) + (c.lo.x + nx_)) + (zm.hi.x + zp.hi.x);
  r.hi.y = ((c.hi.x + e1) + (c.lo.y + ny_)) + (zm.hi.y + zp.hi.y);
  return r;
}
template <class T> __device__ __forceinline__ void stq(T* __restrict__ X, T* __restrict__ Y, const MgPos& q, const Quad<T>& c) {
  X[q.own0] = c.lo.x; Y[q.own0] = c.lo.y; X[q.own0 + 32] = c.hi.x; Y[q.own0 + 32] = c.hi.y;
}

// ---- downward leg: e = S^2(0; g), gc = R (g - (-L) e) -----------------------------------------------------
// Two damped-Jacobi sweeps from a zero guess collapse to e = cg g + cn nb(g) with cg = 2 cw - 6 cw^2 / h^2,
// cn = cw^2 / h^2  (first sweep: cw g; second: cw g + cw (g - (6 cw g - cw nb) / h^2)).
//
// UPD (level 0 inside PCG): the kernel also performs K2 of the PREVIOUS iteration on the fly, g = r - alpha q
// (halo included, so q is read with the same halo as r), stores the new r for the tile interior into the
// OTHER residual buffer (neighbouring CTAs still read the old one on their halos; Scalars::rsel says which
// buffer is current), and its last CTA does the loop control that k_pcg_update does in the unfused path:
// ||r||^2, iteration count, convergence flag, graph WHILE condition.  The separate update pass (3 words per
// cell) disappears; when the flag says "done" the remaining kernels of the iteration exit at once.
template <class T, int TR, bool UPD> __global__ void __launch_bounds__(32 * TR, (sizeof(T) == 4 ? 2 : 1) * (TR == 8 ? 2 : 1))
k_mg_down(const int* __restrict__ done, const T* __restrict__ g_a, T* __restrict__ g_b, const T* __restrict__ qv,
          T* __restrict__ eo, T* __restrict__ gc, int nx, int ny, int nz, T cg, T cn, T ih2, Scalars* S_, double* partials, Launch L) {
  using V = typename V2T<T>::type;
  constexpr int PL = MgTile<TR>::PL;
  if (done && *done) return;
  extern __shared__ __align__(16) unsigned char mg_smem[];
  T* GX = reinterpret_cast<T*>(mg_smem); T* GY = GX + 2 * PL; T* EX = GY + 2 * PL; T* EY = EX + 2 * PL;
  __shared__ double sh[2 * 32]; __shared__ int flag;
  const T* __restrict__ g = g_a; T* __restrict__ rout = nullptr;
  bool upd = false; T alpha = T(0), rm = T(0);
  if (UPD) {
    if (S_->rsel) { g = g_b; rout = const_cast<T*>(g_a); } else { g = g_a; rout = g_b; }
    upd = S_->need_update != 0;
    if (upd) { alpha = T(S_->rho_cur / S_->dq); rm = sizeof(T) == 4 ? T(S_->rmean) : T(0); }
  }
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = blockIdx.x * kMgIX - 2 + 2 * lane, gy = blockIdx.y * MgTile<TR>::IY - 2 + 2 * ty;
  const unsigned pl = (unsigned)nx * ny, gxw = (unsigned)modp(gx, nx);
  const unsigned row0 = gxw + (unsigned)nx * modp(gy, ny), row1 = gxw + (unsigned)nx * modp(gy + 1, ny);
  const bool interior = lane >= 1 && lane <= 30 && ty >= 1 && ty <= TR - 2 && gx < nx && gy < ny;
  const int z0 = chunk_lo(blockIdx.z, gridDim.z, nz), z1 = chunk_lo(blockIdx.z + 1, gridDim.z, nz);
  const int tend = z1 + 1;
  const MgPos q = mg_pos<TR>(lane, ty);
  const unsigned cpl = (unsigned)(nx >> 1) * (ny >> 1), crow = (unsigned)(gx >> 1) + (unsigned)(nx >> 1) * (gy >> 1);
  const T m6 = T(-6) * ih2;
  T acc = T(0);
  double s2 = 0.0, s1 = 0.0;
  int zl = modp(z0 - 2, nz);              // plane of the youngest load in flight
  int b = 0;                              // buffer of plane t (toggles); plane t-1 lives in PL - b
  // Two planes of global loads in flight, in two register buffers that alternate by renaming (the z loop is unrolled
  // 6 = lcm(3, 2) times): step t consumes the buffer that was filled two steps earlier and refills it with plane t + 2,
  // so no instruction touches a load before it is two planes old (a register copy between buffers would wait for it).
  Quad<T> l0g, l0q, l1g, l1q;
  l0q.lo.x = l0q.lo.y = l0q.hi.x = l0q.hi.y = T(0); l1q = l0q;
  auto fetch = [&](Quad<T>& gq, Quad<T>& qq) {
    const unsigned o = pl * zl;
    gq.lo = ldv2<T, V>(g + (row0 + o)); gq.hi = ldv2<T, V>(g + (row1 + o));
    if (UPD && upd) { qq.lo = ldv2<T, V>(qv + (row0 + o)); qq.hi = ldv2<T, V>(qv + (row1 + o)); }
  };
  fetch(l0g, l0q);
  zl = zl + 1 == nz ? 0 : zl + 1;
  fetch(l1g, l1q);
  // one plane: gA, gB = g(t-2), g(t-1); gC receives g(t) from the load buffer (lg, lq).  eA, eB = e(t-3), e(t-2); eC receives e(t-1).
  auto step = [&](int t, const Quad<T>& gA, const Quad<T>& gB, Quad<T>& gC, const Quad<T>& eA, const Quad<T>& eB, Quad<T>& eC,
                  Quad<T>& lg, Quad<T>& lq) {
    gC = lg;
    if (UPD && upd) {
      gC.lo.x = (gC.lo.x - alpha * lq.lo.x) - rm; gC.lo.y = (gC.lo.y - alpha * lq.lo.y) - rm;
      gC.hi.x = (gC.hi.x - alpha * lq.hi.x) - rm; gC.hi.y = (gC.hi.y - alpha * lq.hi.y) - rm;
    }
    if (t + 1 < tend) {
      zl = zl + 1 == nz ? 0 : zl + 1;
      fetch(lg, lq);
    }
    const int pb = PL - b;
    if (t >= z0) {            // e(t-1)
      const Quad<T> nb = nbq<T>(GX + pb, GY + pb, q, gB, gA, gC);
      eC.lo.x = cg * gB.lo.x + cn * nb.lo.x; eC.lo.y = cg * gB.lo.y + cn * nb.lo.y;
      eC.hi.x = cg * gB.hi.x + cn * nb.hi.x; eC.hi.y = cg * gB.hi.y + cn * nb.hi.y;
    }
    if (t >= z0 + 2) {        // residual at plane t-2 summed over the patch, store of e(t-2)
      const Quad<T> nb = nbq<T>(EX + b, EY + b, q, eB, eA, eC);
      const T r0 = ((gA.lo.x + m6 * eB.lo.x) + ih2 * nb.lo.x) + ((gA.lo.y + m6 * eB.lo.y) + ih2 * nb.lo.y);
      const T r1 = ((gA.hi.x + m6 * eB.hi.x) + ih2 * nb.hi.x) + ((gA.hi.y + m6 * eB.hi.y) + ih2 * nb.hi.y);
      acc += r0 + r1;
      if (interior) {
        const unsigned o = pl * (unsigned)(t - 2);
        stv2<T, V>(eo + (row0 + o), eB.lo); stv2<T, V>(eo + (row1 + o), eB.hi);
        if ((t - z0) & 1) gc[crow + cpl * (unsigned)((t - 2) >> 1)] = T(0.125) * acc;
        if (UPD && upd) {
          stv2<T, V>(rout + (row0 + o), gA.lo); stv2<T, V>(rout + (row1 + o), gA.hi);
          s2 += (double)((gA.lo.x * gA.lo.x + gA.lo.y * gA.lo.y) + (gA.hi.x * gA.hi.x + gA.hi.y * gA.hi.y));
          s1 += (double)((gA.lo.x + gA.lo.y) + (gA.hi.x + gA.hi.y));
        }
      }
      if ((t - z0) & 1) acc = T(0);
    }
    stq<T>(GX + b, GY + b, q, gC);
    if (t >= z0) stq<T>(EX + pb, EY + pb, q, eC);
    __syncthreads();
    b = pb;
  };
  Quad<T> g0, g1, g2, e0, e1, e2;
  g0.lo.x = g0.lo.y = g0.hi.x = g0.hi.y = T(0);
  g1 = g0; g2 = g0; e0 = g0; e1 = g0; e2 = g0;
  int t = z0 - 2;
  for (;;) {
    step(t, g0, g1, g2, e0, e1, e2, l0g, l0q); if (++t > tend) break;
    step(t, g1, g2, g0, e1, e2, e0, l1g, l1q); if (++t > tend) break;
    step(t, g2, g0, g1, e2, e0, e1, l0g, l0q); if (++t > tend) break;
    step(t, g0, g1, g2, e0, e1, e2, l1g, l1q); if (++t > tend) break;
    step(t, g1, g2, g0, e1, e2, e0, l0g, l0q); if (++t > tend) break;
    step(t, g2, g0, g1, e2, e0, e1, l1g, l1q); if (++t > tend) break;
  }
  if (UPD && upd) {           // what the last CTA of k_pcg_update does in the unfused path
    double v[2] = {s2, s1};
    if (grid_sum<2>(v, partials, &S_->ticket[0], sh, &flag)) {
      if (threadIdx.x == 0 && threadIdx.y == 0) {
        Scalars* S = S_;
        const double N = (double)nx * ny * nz;
        S->rr = v[0]; S->rmean = v[1] / N;
        S->alpha_prev = S->rho_cur / S->dq; S->pending = 1;
        S->iter += 1; S->first = 0; S->dsel ^= 1; S->rsel ^= 1; S->need_update = 0;
        S->rho_prev = S->rho_cur;
        const int conv = sqrt(v[0]) <= S->rtol * sqrt(S->bnorm2);
        S->converged = conv;
        S->done = conv || S->iter >= S->max_iter;
        if (L.use_cond) cudaGraphSetConditional(L.cond, S->done ? 0u : 1u);
      }
    }
  }
}

// ---- upward leg: e' = S^2(e + P ec; g); DOT (level 0 inside PCG): rho = r . (zs e') ---------------------
// One sweep: e + cw (g - (6 e - nb) / h^2) = ce e + cw g + cn nb with ce = 1 - 6 cw / h^2, cn = cw / h^2.
template <class T> __device__ __forceinline__ Quad<T> sweepq(const Quad<T>& e, const Quad<T>& nb, const Quad<T>& g, T ce, T cw, T cn) {
  Quad<T> o;
  o.lo.x = (ce * e.lo.x + cw * g.lo.x) + cn * nb.lo.x; o.lo.y = (ce * e.lo.y + cw * g.lo.y) + cn * nb.lo.y;
  o.hi.x = (ce * e.hi.x + cw * g.hi.x) + cn * nb.hi.x; o.hi.y = (ce * e.hi.y + cw * g.hi.y) + cn * nb.hi.y;
  return o;
}

template <class T, int TR, bool DOT> __global__ void __launch_bounds__(32 * TR, (sizeof(T) == 4 ? 2 : 1) * (TR == 8 ? 2 : 1))
k_mg_up(const int* __restrict__ done, const T* __restrict__ ein, const T* __restrict__ ec, const T* __restrict__ g_a,
        const T* __restrict__ g_b, T* __restrict__ eo, int nx, int ny, int nz, T ce, T cw, T cn, T zs, Scalars* S_, double* partials,
        const __grid_constant__ Tmap tm_e, const __grid_constant__ Tmap tm_c, const __grid_constant__ Tmap tm_ga,
        const __grid_constant__ Tmap tm_gb, int pf) {
  using V = typename V2T<T>::type;
  constexpr int PL = MgTile<TR>::PL;
  if (done && *done) return;
  const T* __restrict__ g = (g_b && S_->rsel) ? g_b : g_a;      // current residual buffer (k_mg_down<UPD> toggles rsel)
  extern __shared__ __align__(16) unsigned char mg_smem[];
  T* AX = reinterpret_cast<T*>(mg_smem); T* AY = AX + 2 * PL; T* BX = AY + 2 * PL; T* BY = BX + 2 * PL;
  __shared__ double sh[32]; __shared__ int flag;
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = blockIdx.x * kMgIX - 2 + 2 * lane, gy = blockIdx.y * MgTile<TR>::IY - 2 + 2 * ty;
  const int gxw = modp(gx, nx), gyw = modp(gy, ny);
  const unsigned pl = (unsigned)nx * ny;
  const unsigned row0 = (unsigned)gxw + (unsigned)nx * gyw, row1 = (unsigned)gxw + (unsigned)nx * modp(gy + 1, ny);
  const bool interior = lane >= 1 && lane <= 30 && ty >= 1 && ty <= TR - 2 && gx < nx && gy < ny;
  const int z0 = chunk_lo(blockIdx.z, gridDim.z, nz), z1 = chunk_lo(blockIdx.z + 1, gridDim.z, nz);
  const int tend = z1 + 1;
  const MgPos q = mg_pos<TR>(lane, ty);
  const unsigned cpl = (unsigned)(nx >> 1) * (ny >> 1), crow = (unsigned)(gxw >> 1) + (unsigned)(nx >> 1) * (gyw >> 1);
  double dot = 0.0;
  int zl = modp(z0 - 2, nz);              // plane of the e / ec load in flight; the g load in flight is one plane behind
  int b = 0;
  Quad<T> nxa, nxg;
  nxa.lo = ldv2<T, V>(ein + (row0 + pl * zl)); nxa.hi = ldv2<T, V>(ein + (row1 + pl * zl));
  T nxc = ec[crow + cpl * (unsigned)(zl >> 1)];
  nxg.lo.x = nxg.lo.y = nxg.hi.x = nxg.hi.y = T(0);
  // DRAM fetches run kMgAhead planes ahead of the register loads as L2 prefetches of whole tile planes (one TMA
  // instruction per field and plane, issued by one thread; fs_tma.cu): the register loads then hit L2, so one plane of
  // them in flight is enough and the register queue does not grow.
  constexpr int kAl = 16 / (int)sizeof(T);       // a TMA box must start on 16 bytes: x is rounded down to kAl cells, the box is that much wider
  const bool pf_on = pf && lane == 0 && ty == 0;
  const bool g_is_b = g == g_b;
  const int pf_x = blockIdx.x * kMgIX - 2, pf_y = blockIdx.y * MgTile<TR>::IY - 2;
  auto prefetch = [&](int t) {             // planes t + kMgAhead of e (and of ec on even planes), t + kMgAhead - 1 of g
    if (!pf_on || t + kMgAhead > tend) return;
    const int z = modp(t + kMgAhead, nz);
    tma_prefetch_plane(tm_e, pf_x & ~(kAl - 1), pf_y, z);
    tma_prefetch_plane(g_is_b ? tm_gb : tm_ga, pf_x & ~(kAl - 1), pf_y, z == 0 ? nz - 1 : z - 1);
    if (!(z & 1)) tma_prefetch_plane(tm_c, (pf_x >> 1) & ~(kAl - 1), pf_y >> 1, z >> 1);
  };
  for (int tt = z0 - 2 - kMgAhead + 1; tt < z0 - 2; ++tt) prefetch(tt);
  // aA, aB = (e + P ec)(t-2), (t-1); aC receives plane t.  bA, bB = first post-sweep at t-3, t-2; bC receives t-1.
  // gA = g(t-2); gB receives g(t-1).
  auto step = [&](int t, const Quad<T>& aA, const Quad<T>& aB, Quad<T>& aC, const Quad<T>& bA, const Quad<T>& bB, Quad<T>& bC,
                  const Quad<T>& gA, Quad<T>& gB) {
    aC.lo.x = nxa.lo.x + nxc; aC.lo.y = nxa.lo.y + nxc; aC.hi.x = nxa.hi.x + nxc; aC.hi.y = nxa.hi.y + nxc;
    gB = nxg;
    prefetch(t);
    if (t < tend) {
      const unsigned og = pl * zl;                     // plane t
      nxg.lo = ldv2<T, V>(g + (row0 + og)); nxg.hi = ldv2<T, V>(g + (row1 + og));
      zl = zl + 1 == nz ? 0 : zl + 1;
      const unsigned oa = pl * zl;                     // plane t+1
      nxa.lo = ldv2<T, V>(ein + (row0 + oa)); nxa.hi = ldv2<T, V>(ein + (row1 + oa));
      nxc = ec[crow + cpl * (unsigned)(zl >> 1)];
    }
    const int pb = PL - b;
    if (t >= z0) {            // first post-sweep at plane t-1
      const Quad<T> nb = nbq<T>(AX + pb, AY + pb, q, aB, aA, aC);
      bC = sweepq<T>(aB, nb, gB, ce, cw, cn);
    }
    if (t >= z0 + 2) {        // second post-sweep at plane t-2
      const Quad<T> nb = nbq<T>(BX + b, BY + b, q, bB, bA, bC);
      const Quad<T> o = sweepq<T>(bB, nb, gA, ce, cw, cn);
      if (interior) {
        const unsigned oo = pl * (unsigned)(t - 2);
        stv2<T, V>(eo + (row0 + oo), o.lo); stv2<T, V>(eo + (row1 + oo), o.hi);
        if (DOT) dot += (double)(((gA.lo.x * o.lo.x + gA.lo.y * o.lo.y) + (gA.hi.x * o.hi.x + gA.hi.y * o.hi.y)) * zs);
      }
    }
    stq<T>(AX + b, AY + b, q, aC);
    if (t >= z0) stq<T>(BX + pb, BY + pb, q, bC);
    __syncthreads();
    b = pb;
  };
  Quad<T> a0, a1, a2, b0, b1, b2, g0, g1;
  a0.lo.x = a0.lo.y = a0.hi.x = a0.hi.y = T(0);
  a1 = a0; a2 = a0; b0 = a0; b1 = a0; b2 = a0; g0 = a0; g1 = a0;
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

// Tile height: TR thread rows (2 TR cell rows; 16 on big levels: fewer halo rows per result, 8 below: more CTAs).
static int tune_env(const char* n, int d) { const char* e = getenv(n); return e ? atoi(e) : d; }
static int mg_tr(int ny) { static int thr = tune_env("FS_TUNE_TR16_NY", 384); return ny >= thr ? 16 : 8; }
template <class T, int TR> static int slots_per_sm() { return (sizeof(T) == 4 ? 2 : 1) * (TR == 8 ? 2 : 1); }
template <class K> static cudaError_t allow_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}
// Dynamic shared memory of the fused legs exceeds the 48 KB default at TR = 16 in fp64 (64 KB): the opt-in is a
// per-device function attribute, so it is (re)applied for the current device whenever a grid is created there.
template <class T, int TR> static cudaError_t configure_tr() {
  const size_t smem = 8 * (size_t)MgTile<TR>::PL * sizeof(T);
  cudaError_t e;
  if ((e = allow_smem(k_mg_down<T, TR, true>, smem)) != cudaSuccess) return e;
  if ((e = allow_smem(k_mg_down<T, TR, false>, smem)) != cudaSuccess) return e;
  if ((e = allow_smem(k_mg_up<T, TR, true>, smem)) != cudaSuccess) return e;
  return allow_smem(k_mg_up<T, TR, false>, smem);
}
template <class T> cudaError_t mgf_configure_device() {
  cudaError_t e = configure_tr<T, 8>();
  return e != cudaSuccess ? e : configure_tr<T, 16>();
}

template <class T, int TR, bool UPD> static void down_tr(const Ctx<T>& c, const T* g, T* g2, const T* q, T* e, T* gc, int nx, int ny, int nz,
                                                         T cg, T cn, T ih2, const Launch& L) {
  const MgGeom G = mg_geom(nx, ny, nz, MgTile<TR>::IY, slots_per_sm<T, TR>());
  const size_t smem = 8 * (size_t)MgTile<TR>::PL * sizeof(T);
  k_mg_down<T, TR, UPD><<<G.grid, dim3(32, TR), smem, L.s>>>(&c.S->done, g, g2, q, e, gc, nx, ny, nz, cg, cn, ih2, c.S, c.partials, L);
}
template <class T, int TR, bool DOT> static void up_tr(const Ctx<T>& c, const T* ein, const T* ec, const T* g, const T* g2, T* eo, int nx, int ny, int nz,
                                                       T ce, T cw, T cn, T zs, cudaStream_t s) {
  const MgGeom G = mg_geom(nx, ny, nz, MgTile<TR>::IY, slots_per_sm<T, TR>());
  const size_t smem = 8 * (size_t)MgTile<TR>::PL * sizeof(T);
  // tensor maps of the fields the kernel streams (extended tile planes: 64 x 2 TR fine cells, 32 x TR coarse cells)
  Tmap te, tc, tga, tgb;
  const int ROWS = MgTile<TR>::ROWS;
  // box origins are rounded down to 16 bytes in the kernel: fine tiles start at 60 bx - 2 (even), coarse ones at 30 bx - 1
  const int al = 16 / (int)sizeof(T), bxf = 64 + (al > 2 ? al : 0), bxc = 32 + al;
  int pf = tmap_encode(&te, ein, sizeof(T), nx, ny, nz, bxf, ROWS) && tmap_encode(&tc, ec, sizeof(T), nx / 2, ny / 2, nz / 2, bxc, ROWS / 2) &&
           tmap_encode(&tga, g, sizeof(T), nx, ny, nz, bxf, ROWS);
  if (pf && g2) pf = tmap_encode(&tgb, g2, sizeof(T), nx, ny, nz, bxf, ROWS); else if (pf) tgb = tga;
  if (!pf) { memset(&te, 0, sizeof te); tc = te; tga = te; tgb = te; }
  // measured at 512^3 / 256^3 (profiles/r2_tma_prefetch.md): removes the long-scoreboard stalls in both precisions, the fp64 leg
  // gains 0-5 % (it already moves its bytes at 0.88 of the copy rate), the fp32 leg with two CTAs per SM loses 5 %: fp64 only
  else { static int on = tune_env("FS_TUNE_PF", sizeof(T) == 8 ? 1 : 0); pf = on; }
  k_mg_up<T, TR, DOT><<<G.grid, dim3(32, TR), smem, s>>>(&c.S->done, ein, ec, g, g2, eo, nx, ny, nz, ce, cw, cn, zs, c.S, c.partials, te, tc, tga, tgb, pf);
}

// upd: level 0 inside PCG with the residual update of the previous iteration fused in (g2 = the other residual
// buffer, q = A d); the launch then moves 4.125 words per cell (r, q in; r, e, gc out)
template <class T> int launch_mg_down(const Ctx<T>& c, const T* g, T* e, T* gc, int nx, int ny, int nz, double h, double omega,
                                      const char* name, const Launch& L, bool upd, T* g2, const T* q) {
  const double N = (double)nx * ny * nz;
  const double ih2 = 1.0 / (h * h), cw = omega * h * h / 6.0;
  const T cg = T(2.0 * cw - 6.0 * cw * cw * ih2), cn = T(cw * cw * ih2);
  const bool big = mg_tr(ny) == 16;
  const char* inst = sizeof(T) == 8 ? (big ? (upd ? "k_mg_down<f64,TR16,UPD>" : "k_mg_down<f64,TR16>") : (upd ? "k_mg_down<f64,TR8,UPD>" : "k_mg_down<f64,TR8>"))
                                    : (big ? (upd ? "k_mg_down<f32,TR16,UPD>" : "k_mg_down<f32,TR16>") : (upd ? "k_mg_down<f32,TR8,UPD>" : "k_mg_down<f32,TR8>"));
  FS_LAUNCHI(L, name, inst, (upd ? 4.125 : 2.125) * sizeof(T) * N, {
    if (upd) { if (big) down_tr<T, 16, true>(c, g, g2, q, e, gc, nx, ny, nz, cg, cn, T(ih2), L); else down_tr<T, 8, true>(c, g, g2, q, e, gc, nx, ny, nz, cg, cn, T(ih2), L); }
    else { if (big) down_tr<T, 16, false>(c, g, nullptr, nullptr, e, gc, nx, ny, nz, cg, cn, T(ih2), L); else down_tr<T, 8, false>(c, g, nullptr, nullptr, e, gc, nx, ny, nz, cg, cn, T(ih2), L); }
  });
  return 1;
}
template <class T> int launch_mg_up(const Ctx<T>& c, const T* ein, const T* ec, const T* g, T* eo, int nx, int ny, int nz, double h,
                                    double omega, bool dot, T zs, const char* name, const Launch& L, const T* g2) {
  const double N = (double)nx * ny * nz;
  const double ih2d = 1.0 / (h * h), cwd = omega * h * h / 6.0;
  const T ce = T(1.0 - 6.0 * cwd * ih2d), cw = T(cwd), cn = T(cwd * ih2d);
  const bool big = mg_tr(ny) == 16;
  const char* inst = sizeof(T) == 8 ? (big ? (dot ? "k_mg_up<f64,TR16,DOT>" : "k_mg_up<f64,TR16>") : (dot ? "k_mg_up<f64,TR8,DOT>" : "k_mg_up<f64,TR8>"))
                                    : (big ? (dot ? "k_mg_up<f32,TR16,DOT>" : "k_mg_up<f32,TR16>") : (dot ? "k_mg_up<f32,TR8,DOT>" : "k_mg_up<f32,TR8>"));
  FS_LAUNCHI(L, name, inst, 3.125 * sizeof(T) * N, {
    if (big) { if (dot) up_tr<T, 16, true>(c, ein, ec, g, g2, eo, nx, ny, nz, ce, cw, cn, zs, L.s); else up_tr<T, 16, false>(c, ein, ec, g, g2, eo, nx, ny, nz, ce, cw, cn, zs, L.s); }
    else { if (dot) up_tr<T, 8, true>(c, ein, ec, g, g2, eo, nx, ny, nz, ce, cw, cn, zs, L.s); else up_tr<T, 8, false>(c, ein, ec, g, g2, eo, nx, ny, nz, ce, cw, cn, zs, L.s); }
  });
  return 1;
}

#define INST(T)                                                                                                              \
  template int launch_mg_down<T>(const Ctx<T>&, const T*, T*, T*, int, int, int, double, double, const char*, const Launch&, bool, T*, const T*); \
  template int launch_mg_up<T>(const Ctx<T>&, const T*, const T*, const T*, T*, int, int, int, double, double, bool, T, const char*, const Launch&, const T*);
INST(float)
INST(double)
template cudaError_t mgf_configure_device<float>();
template cudaError_t mgf_configure_device<double>();

}  // namespace fs
