// fs_kernels_mgf.cu -- fused, temporally blocked kernels of the V(2,2) cycle (S7g).
//
// The unfused cycle moves 15.25 words per fine cell (first 2, sweep 3 x3, residual+restrict 2.125,
// prolong+correct 2.125); the two kernels here move 2.125 + 3.125:
//   k_mg_down : g -> e = two damped-Jacobi sweeps from a zero guess, gc = R (g - (-L) e)
//   k_mg_up   : e, ec, g -> e' = two sweeps applied to (e + P ec)   [level 0: also r . z for PCG]
// Both are 2.5-D streaming kernels: a CTA owns an xy tile and marches in z.  A thread owns two x-adjacent
// cells (16-byte loads for fp64, 8 for fp32), keeps the z neighbours of every pipeline stage in a register
// queue, gets the x neighbours by warp shuffle (a warp is one row of the tile) and the y neighbours
// through a double-buffered shared-memory plane; one __syncthreads per plane.  Each later stage is valid on
// a tile one cell smaller per side (overlapped tiling: 64 x TY extended tile -> 60 x (TY-4) results); the
// halo re-reads hit L2.  All grids are periodic (GMG is only offered for triply periodic boxes).
#include "fs_internal.cuh"

namespace fs {

template <class T> struct V2T;
template <> struct V2T<double> { using type = double2; };
template <> struct V2T<float> { using type = float2; };

constexpr int kMgTY = 16;                 // rows of the extended tile
constexpr int kMgIX = 60, kMgIY = kMgTY - 4;

__device__ __forceinline__ int modp(int a, int n) { a %= n; return a < 0 ? a + n : a; }

// sum of the six neighbours of both cells of a pair: zm / zp = pairs below / above, S / N = pairs of the
// rows y-1 / y+1 (shared memory), x neighbours of the pair's outer sides by shuffle.
template <class T, class V> __device__ __forceinline__ V nb_sum(const V& c, const V& zm, const V& zp, const V& S, const V& N) {
  const T left = __shfl_up_sync(0xffffffffu, c.y, 1);
  const T right = __shfl_down_sync(0xffffffffu, c.x, 1);
  V r;
  r.x = left + c.y + S.x + N.x + zm.x + zp.x;
  r.y = c.x + right + S.y + N.y + zm.y + zp.y;
  return r;
}

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

template <class T, class V> __device__ __forceinline__ V ldv2(const T* p) { return *reinterpret_cast<const V*>(p); }
template <class T, class V> __device__ __forceinline__ void stv2(T* p, const V& v) { *reinterpret_cast<V*>(p) = v; }

// damped-Jacobi update of one cell: e + omega D^-1 (g - (-L) e), with nb = sum of the six neighbours
template <class T> __device__ __forceinline__ T jac(T e, T nb, T g, T ih2, T cw) { return e + cw * (g - (T(6) * e - nb) * ih2); }

// ---- downward leg: e = S^2(0; g), gc = R (g - (-L) e) -----------------------------------------------------
template <class T> __global__ void __launch_bounds__(32 * kMgTY, 2)
k_mg_down(const int* __restrict__ done, const T* __restrict__ g, T* __restrict__ eo, T* __restrict__ gc,
          int nx, int ny, int nz, T ih2, T cw) {
  using V = typename V2T<T>::type;
  if (done && *done) return;
  __shared__ V G[2][kMgTY][32];
  __shared__ V E[2][kMgTY][32];
  __shared__ T R[2][kMgTY][32];
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = blockIdx.x * kMgIX - 2 + 2 * lane, gy = blockIdx.y * kMgIY - 2 + ty;
  const int gxw = modp(gx, nx), gyw = modp(gy, ny);
  const size_t pl = (size_t)nx * ny;
  const size_t row = (size_t)gxw + (size_t)nx * gyw;
  const bool interior = lane >= 1 && lane <= 30 && ty >= 2 && ty < kMgTY - 2 && gx < nx && gy < ny;
  const bool comb = interior && ((ty & 1) == 0);
  const int z0 = chunk_lo(blockIdx.z, gridDim.z, nz), z1 = chunk_lo(blockIdx.z + 1, gridDim.z, nz);
  const int tys = ty > 0 ? ty - 1 : 0, tyn = ty < kMgTY - 1 ? ty + 1 : ty;
  const size_t crow = (size_t)(gx >> 1) + (size_t)(nx >> 1) * (size_t)(gy >> 1);
  const size_t cpl = (size_t)(nx >> 1) * (ny >> 1);
  V g0 = {T(0), T(0)}, g1 = g0, g2 = g0, e0 = g0, e1 = g0;
  T acc = T(0);
  V nxt = ldv2<T, V>(g + row + pl * modp(z0 - 2, nz));
  for (int t = z0 - 2; t <= z1 + 1; ++t) {
    g2 = nxt;
    if (t < z1 + 1) nxt = ldv2<T, V>(g + row + pl * modp(t + 1, nz));
    V en = g0;
    if (t >= z0) {            // e(t-1): first sweep from zero gives cw g, the second is applied to it
      const V S = G[(t - 1) & 1][tys][lane], N = G[(t - 1) & 1][tyn][lane];
      const V nb = nb_sum<T, V>(g1, g0, g2, S, N);
      en.x = jac<T>(cw * g1.x, cw * nb.x, g1.x, ih2, cw);
      en.y = jac<T>(cw * g1.y, cw * nb.y, g1.y, ih2, cw);
    }
    if (t >= z0 + 2) {        // residual at plane t-2, its x-pair sum, and the store of e(t-2)
      const V S = E[t & 1][tys][lane], N = E[t & 1][tyn][lane];
      const V nb = nb_sum<T, V>(e1, e0, en, S, N);
      const T rx = g0.x - (T(6) * e1.x - nb.x) * ih2;
      const T ry = g0.y - (T(6) * e1.y - nb.y) * ih2;
      R[t & 1][ty][lane] = rx + ry;
      if (interior) stv2<T, V>(eo + row + pl * (size_t)(t - 2), e1);
    }
    G[t & 1][ty][lane] = g2;
    if (t >= z0) E[(t - 1) & 1][ty][lane] = en;
    __syncthreads();
    if (t >= z0 + 2 && comb) {
      acc += R[t & 1][ty][lane] + R[t & 1][ty + 1][lane];
      if ((t - z0) & 1) { gc[crow + cpl * (size_t)((t - 2) >> 1)] = T(0.125) * acc; acc = T(0); }
    }
    g0 = g1; g1 = g2; e0 = e1; e1 = en;
  }
}

// ---- upward leg: e' = S^2(e + P ec; g); DOT (level 0 inside PCG): rho = r . (zs e') ---------------------
template <class T, bool DOT> __global__ void __launch_bounds__(32 * kMgTY, 2)
k_mg_up(const int* __restrict__ done, const T* __restrict__ ein, const T* __restrict__ ec, const T* __restrict__ g,
        T* __restrict__ eo, int nx, int ny, int nz, T ih2, T cw, T zs, Scalars* S_, double* partials) {
  using V = typename V2T<T>::type;
  if (done && *done) return;
  __shared__ V A[2][kMgTY][32];
  __shared__ V B[2][kMgTY][32];
  __shared__ double sh[32]; __shared__ int flag;
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = blockIdx.x * kMgIX - 2 + 2 * lane, gy = blockIdx.y * kMgIY - 2 + ty;
  const int gxw = modp(gx, nx), gyw = modp(gy, ny);
  const size_t pl = (size_t)nx * ny;
  const size_t row = (size_t)gxw + (size_t)nx * gyw;
  const bool interior = lane >= 1 && lane <= 30 && ty >= 2 && ty < kMgTY - 2 && gx < nx && gy < ny;
  const int z0 = chunk_lo(blockIdx.z, gridDim.z, nz), z1 = chunk_lo(blockIdx.z + 1, gridDim.z, nz);
  const int tys = ty > 0 ? ty - 1 : 0, tyn = ty < kMgTY - 1 ? ty + 1 : ty;
  const size_t crow = (size_t)(gxw >> 1) + (size_t)(nx >> 1) * (size_t)(gyw >> 1);
  const size_t cpl = (size_t)(nx >> 1) * (ny >> 1);
  const V zero = {T(0), T(0)};
  V a0 = zero, a1 = zero, a2 = zero, b0 = zero, b1 = zero, g0 = zero, g1 = zero;
  double v[1] = {0.0};
  int zt = modp(z0 - 2, nz);
  V nxa = ldv2<T, V>(ein + row + pl * zt);
  T nxc = ec[crow + cpl * (zt >> 1)];
  V nxg = zero;
  for (int t = z0 - 2; t <= z1 + 1; ++t) {
    a2.x = nxa.x + nxc; a2.y = nxa.y + nxc;          // e + P ec at plane t
    g1 = nxg;                                         // g at plane t-1
    if (t < z1 + 1) {
      const int zn = modp(t + 1, nz);
      nxa = ldv2<T, V>(ein + row + pl * zn);
      nxc = ec[crow + cpl * (zn >> 1)];
      nxg = ldv2<T, V>(g + row + pl * modp(t, nz));
    }
    V bn = zero;
    if (t >= z0) {            // first post-sweep at plane t-1
      const V S = A[(t - 1) & 1][tys][lane], N = A[(t - 1) & 1][tyn][lane];
      const V nb = nb_sum<T, V>(a1, a0, a2, S, N);
      bn.x = jac<T>(a1.x, nb.x, g1.x, ih2, cw);
      bn.y = jac<T>(a1.y, nb.y, g1.y, ih2, cw);
    }
    if (t >= z0 + 2) {        // second post-sweep at plane t-2
      const V S = B[t & 1][tys][lane], N = B[t & 1][tyn][lane];
      const V nb = nb_sum<T, V>(b1, b0, bn, S, N);
      V o;
      o.x = jac<T>(b1.x, nb.x, g0.x, ih2, cw);
      o.y = jac<T>(b1.y, nb.y, g0.y, ih2, cw);
      if (interior) {
        stv2<T, V>(eo + row + pl * (size_t)(t - 2), o);
        if (DOT) v[0] += (double)g0.x * (double)(o.x * zs) + (double)g0.y * (double)(o.y * zs);
      }
    }
    A[t & 1][ty][lane] = a2;
    if (t >= z0) B[(t - 1) & 1][ty][lane] = bn;
    __syncthreads();
    a0 = a1; a1 = a2; b0 = b1; b1 = bn; g0 = g1;
  }
  if (DOT) {
    if (grid_sum<1>(v, partials, &S_->ticket[0], sh, &flag)) {
      if (threadIdx.x == 0 && threadIdx.y == 0) S_->rho_cur = v[0];
    }
  }
}

template <class T> int launch_mg_down(const Ctx<T>& c, const T* g, T* e, T* gc, int nx, int ny, int nz, double h, double omega,
                                      const char* name, const Launch& L) {
  const MgGeom G = mg_geom(nx, ny, nz);
  const double N = (double)nx * ny * nz;
  FS_LAUNCH(L, name, 2.125 * sizeof(T) * N,
            k_mg_down<T><<<G.grid, dim3(32, kMgTY), 0, L.s>>>(&c.S->done, g, e, gc, nx, ny, nz, T(1.0 / (h * h)), T(omega * h * h / 6.0)));
  return 1;
}
template <class T> int launch_mg_up(const Ctx<T>& c, const T* ein, const T* ec, const T* g, T* eo, int nx, int ny, int nz, double h,
                                    double omega, bool dot, T zs, const char* name, const Launch& L) {
  const MgGeom G = mg_geom(nx, ny, nz);
  const double N = (double)nx * ny * nz;
  const T ih2 = T(1.0 / (h * h)), cw = T(omega * h * h / 6.0);
  if (dot) FS_LAUNCH(L, name, 3.125 * sizeof(T) * N, k_mg_up<T, true><<<G.grid, dim3(32, kMgTY), 0, L.s>>>(&c.S->done, ein, ec, g, eo, nx, ny, nz, ih2, cw, zs, c.S, c.partials));
  else FS_LAUNCH(L, name, 3.125 * sizeof(T) * N, k_mg_up<T, false><<<G.grid, dim3(32, kMgTY), 0, L.s>>>(&c.S->done, ein, ec, g, eo, nx, ny, nz, ih2, cw, zs, c.S, c.partials));
  return 1;
}

#define INST(T)                                                                                                              \
  template int launch_mg_down<T>(const Ctx<T>&, const T*, T*, T*, int, int, int, double, double, const char*, const Launch&); \
  template int launch_mg_up<T>(const Ctx<T>&, const T*, const T*, const T*, T*, int, int, int, double, double, bool, T, const char*, const Launch&);
INST(float)
INST(double)

}  // namespace fs
