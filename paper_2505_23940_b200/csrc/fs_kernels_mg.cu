// fs_kernels_mg.cu -- geometric-multigrid V-cycle preconditioner (S7g; not in the
// paper, named by BASELINE.json c5).  Uniform, isotropic grids; periodic or bounded (reading G1: boundary fluxes dropped).  Per level: nu1 damped-
// Jacobi sweeps from a zero guess, residual, 8-cell-average restriction, recursion, piecewise-constant
// prolongation + correction, nu2 sweeps; the coarsest level does a fixed number of sweeps.  The operator
// on every level is the rediscretised 7-point -L.  Jacobi is order independent, so the result matches
// the CPU oracle up to summation rounding.
#include "fs_internal.cuh"

namespace fs {

constexpr int kFlatBlocks = 148 * 8;
static inline int flat_blocks(long long n) { long long b = (n + 255) / 256; return (int)(b < kFlatBlocks ? (b < 1 ? 1 : b) : kFlatBlocks); }

// (-L) e at a cell.  bd: bit d set = direction d is bounded, the flux through a boundary face is dropped (reading G1): the cell
// then has nnb < 6 neighbours, returned through *nnb for the Jacobi diagonal nnb / h^2.  bd == 0: the periodic formulas.
template <class T> __device__ __forceinline__ T neg_lap(const T* __restrict__ e, int i, int j, int k, int nx, int ny, int nz, T ih2, int bd = 0, T* nnb = nullptr) {
  const size_t row = (size_t)nx * ((size_t)j + (size_t)ny * k);
  if (bd == 0) {
    const int ip = i + 1 == nx ? 0 : i + 1, im = i == 0 ? nx - 1 : i - 1;
    const int jp = j + 1 == ny ? 0 : j + 1, jm = j == 0 ? ny - 1 : j - 1;
    const int kp = k + 1 == nz ? 0 : k + 1, km = k == 0 ? nz - 1 : k - 1;
    const T nb = e[row + ip] + e[row + im] + e[(size_t)i + (size_t)nx * ((size_t)jp + (size_t)ny * k)] +
                 e[(size_t)i + (size_t)nx * ((size_t)jm + (size_t)ny * k)] + e[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * kp)] +
                 e[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * km)];
    if (nnb) *nnb = T(6);
    return (T(6) * e[row + i] - nb) * ih2;
  }
  // neighbours in the oracle's order (+x, -x, +y, -y, +z, -z); a missing one adds 0 and is counted out of nnb
  const bool bx = bd & 1, by = bd & 2, bz = bd & 4;
  const bool hxp = !(bx && i + 1 == nx), hxm = !(bx && i == 0), hyp = !(by && j + 1 == ny), hym = !(by && j == 0), hzp = !(bz && k + 1 == nz), hzm = !(bz && k == 0);
  const int ip = i + 1 == nx ? 0 : i + 1, im = i == 0 ? nx - 1 : i - 1;
  const int jp = j + 1 == ny ? 0 : j + 1, jm = j == 0 ? ny - 1 : j - 1;
  const int kp = k + 1 == nz ? 0 : k + 1, km = k == 0 ? nz - 1 : k - 1;
  const T xp = hxp ? e[row + ip] : T(0), xm = hxm ? e[row + im] : T(0);
  const T yp = hyp ? e[(size_t)i + (size_t)nx * ((size_t)jp + (size_t)ny * k)] : T(0), ym = hym ? e[(size_t)i + (size_t)nx * ((size_t)jm + (size_t)ny * k)] : T(0);
  const T zp = hzp ? e[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * kp)] : T(0), zm = hzm ? e[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * km)] : T(0);
  const T nb = xp + xm + yp + ym + zp + zm;
  const T n = T((int)hxp + (int)hxm + (int)hyp + (int)hym + (int)hzp + (int)hzm);
  if (nnb) *nnb = n;
  return (n * e[row + i] - nb) * ih2;
}
// number of neighbours of a cell (the Jacobi diagonal is nnb / h^2)
__device__ __forceinline__ int mg_nnb(int i, int j, int k, int nx, int ny, int nz, int bd) {
  int n = 6;
  if (bd & 1) n -= (i == 0) + (i + 1 == nx);
  if (bd & 2) n -= (j == 0) + (j + 1 == ny);
  if (bd & 4) n -= (k == 0) + (k + 1 == nz);
  return n;
}

// first sweep from a zero guess: e = omega D^-1 g   (cw = omega h^2 / 6; bounded grids: wh2 / nnb per cell, wh2 = omega h^2)
template <class T> __global__ void __launch_bounds__(256) k_mg_first(const int* __restrict__ done, const T* __restrict__ g, T* __restrict__ e, T cw, long long N,
                                                                    int nx, int ny, int nz, int bd, double wh2) {
  if (done && *done) return;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    T c = cw;
    if (bd) { const int i = (int)(q % nx); const long long t = q / nx; c = T(wh2 / (double)mg_nnb(i, (int)(t % ny), (int)(t / ny), nx, ny, nz, bd)); }
    e[q] = c * g[q];
  }
}
// damped-Jacobi sweep  dst = src + omega D^-1 (g - (-L) src)
template <class T> __global__ void __launch_bounds__(256) k_mg_sweep(const int* __restrict__ done, const T* __restrict__ g, const T* __restrict__ src,
                                                                    T* __restrict__ dst, int nx, int ny, int nz, T ih2, T cw, int bd, double wh2) {
  if (done && *done) return;
  const long long N = (long long)nx * ny * nz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % nx); const long long t = q / nx; const int j = (int)(t % ny), k = (int)(t / ny);
    T nnb;
    const T lap = neg_lap<T>(src, i, j, k, nx, ny, nz, ih2, bd, &nnb);
    const T c = bd ? T(wh2 / (double)nnb) : cw;
    dst[q] = src[q] + c * (g[q] - lap);
  }
}
// residual + restriction: gc = mean over the 8 children of (g - (-L) e); e == nullptr means e = 0
template <class T> __global__ void __launch_bounds__(256) k_mg_restrict(const int* __restrict__ done, const T* __restrict__ g, const T* __restrict__ e,
                                                                       T* __restrict__ gc, int nx, int ny, int nz, T ih2, int bd) {
  if (done && *done) return;
  const int cx = nx / 2, cy = ny / 2, cz = nz / 2;
  const long long Nc = (long long)cx * cy * cz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < Nc; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % cx); const long long t = q / cx; const int j = (int)(t % cy), k = (int)(t / cy);
    T a = T(0);
    for (int dk = 0; dk < 2; ++dk) for (int dj = 0; dj < 2; ++dj) for (int di = 0; di < 2; ++di) {
      const int fi = 2 * i + di, fj = 2 * j + dj, fk = 2 * k + dk;
      const size_t fq = (size_t)fi + (size_t)nx * ((size_t)fj + (size_t)ny * fk);
      a += e ? g[fq] - neg_lap<T>(e, fi, fj, fk, nx, ny, nz, ih2, bd) : g[fq];
    }
    gc[q] = T(0.125) * a;
  }
}
// piecewise-constant prolongation + correction: e += P ec   (e_in == nullptr: e = P ec)
template <class T> __global__ void __launch_bounds__(256) k_mg_prolong(const int* __restrict__ done, const T* __restrict__ ec, const T* __restrict__ e_in,
                                                                      T* __restrict__ e, int nx, int ny, int nz) {
  if (done && *done) return;
  const int cx = nx / 2, cy = ny / 2;
  const long long N = (long long)nx * ny * nz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % nx); const long long t = q / nx; const int j = (int)(t % ny), k = (int)(t / ny);
    const T cval = ec[(size_t)(i >> 1) + (size_t)cx * ((size_t)(j >> 1) + (size_t)cy * (k >> 1))];
    e[q] = e_in ? e_in[q] + cval : cval;
  }
}

// ---- tail of the V-cycle in ONE CTA ------------------------------------------------------------------
// Levels of at most kTailCells cells (16^3) and everything below them fit in shared memory together: one
// launch runs their downward legs, the coarsest-level sweeps and their upward legs, instead of ~20 launches
// that each do microseconds of work.  Same operations, in the same order, as the per-level kernels above.
constexpr int kTailCells = 4096;
struct MgTail { int nlev; int nx[kMaxLevels], ny[kMaxLevels], nz[kMaxLevels]; double h[kMaxLevels]; };

// cell index -> (i, j, k): shifts and masks when nx and ny are powers of two (the usual case: 16^3, 8^3, 4^3), two
// divisions otherwise; the tail runs on ONE SM and is issue bound, and the divisions were most of its instructions
__device__ __forceinline__ void tail_ijk(int q, int nx, int ny, int& i, int& j, int& k) {
  if (((nx & (nx - 1)) | (ny & (ny - 1))) == 0) {
    const int lx = 31 - __clz(nx), ly = 31 - __clz(ny);
    i = q & (nx - 1); j = (q >> lx) & (ny - 1); k = q >> (lx + ly);
  } else { i = q % nx; const int t = q / nx; j = t % ny; k = t / ny; }
}

template <class T> __device__ __forceinline__ T tail_neg_lap(const T* e, int q, int nx, int ny, int nz, T ih2) {
  int i, j, k;
  tail_ijk(q, nx, ny, i, j, k);
  const int ip = i + 1 == nx ? 0 : i + 1, im = i == 0 ? nx - 1 : i - 1;
  const int jp = j + 1 == ny ? 0 : j + 1, jm = j == 0 ? ny - 1 : j - 1;
  const int kp = k + 1 == nz ? 0 : k + 1, km = k == 0 ? nz - 1 : k - 1;
  const int row = nx * (j + ny * k);
  const T nb = e[row + ip] + e[row + im] + e[i + nx * (jp + ny * k)] + e[i + nx * (jm + ny * k)] + e[i + nx * (j + ny * kp)] + e[i + nx * (j + ny * km)];
  return (T(6) * e[q] - nb) * ih2;
}

template <class T> __global__ void __launch_bounds__(1024) k_mg_tail(const int* __restrict__ done, const T* __restrict__ g_in, T* __restrict__ e_out,
                                                                      MgTail a, int nu1, int nu2, int ncoarse, double omega) {
  if (done && *done) return;
  extern __shared__ __align__(16) unsigned char tail_smem[];
  T* base = reinterpret_cast<T*>(tail_smem);
  T* G[kMaxLevels]; T* E[kMaxLevels]; T* Tm[kMaxLevels]; T* cur[kMaxLevels];
  int N[kMaxLevels];
  {
    T* p = base;
    for (int l = 0; l < a.nlev; ++l) { N[l] = a.nx[l] * a.ny[l] * a.nz[l]; G[l] = p; p += N[l]; E[l] = p; p += N[l]; Tm[l] = p; p += N[l]; }
  }
  const int tid = threadIdx.x, nth = blockDim.x;
  for (int q = tid; q < N[0]; q += nth) G[0][q] = g_in[q];
  __syncthreads();
  const int last = a.nlev - 1;
  // sweeps from a zero guess: returns the buffer that holds the iterate (nullptr = still zero)
  auto smooth0 = [&](int l, int n) -> T* {
    if (n <= 0) return nullptr;
    const T ih2 = T(1.0 / (a.h[l] * a.h[l])), cw = T(omega * a.h[l] * a.h[l] / 6.0);
    T* x = E[l]; T* y = Tm[l];
    for (int q = tid; q < N[l]; q += nth) x[q] = cw * G[l][q];
    __syncthreads();
    for (int it = 1; it < n; ++it) {
      for (int q = tid; q < N[l]; q += nth) y[q] = x[q] + cw * (G[l][q] - tail_neg_lap<T>(x, q, a.nx[l], a.ny[l], a.nz[l], ih2));
      __syncthreads();
      T* t = x; x = y; y = t;
    }
    return x;
  };
  auto smooth = [&](int l, T* x, int n) -> T* {
    const T ih2 = T(1.0 / (a.h[l] * a.h[l])), cw = T(omega * a.h[l] * a.h[l] / 6.0);
    T* y = x == E[l] ? Tm[l] : E[l];
    for (int it = 0; it < n; ++it) {
      for (int q = tid; q < N[l]; q += nth) y[q] = x[q] + cw * (G[l][q] - tail_neg_lap<T>(x, q, a.nx[l], a.ny[l], a.nz[l], ih2));
      __syncthreads();
      T* t = x; x = y; y = t;
    }
    return x;
  };
  for (int l = 0; l < last; ++l) {        // downward legs
    cur[l] = smooth0(l, nu1);
    const int nx = a.nx[l], ny = a.ny[l], nz = a.nz[l], cx = nx / 2, cy = ny / 2;
    const T ih2 = T(1.0 / (a.h[l] * a.h[l]));
    for (int q = tid; q < N[l + 1]; q += nth) {
      int i, j, k;
      tail_ijk(q, cx, cy, i, j, k);
      T s = T(0);
      for (int dk = 0; dk < 2; ++dk) for (int dj = 0; dj < 2; ++dj) for (int di = 0; di < 2; ++di) {
        const int fq = (2 * i + di) + nx * ((2 * j + dj) + ny * (2 * k + dk));
        s += cur[l] ? G[l][fq] - tail_neg_lap<T>(cur[l], fq, nx, ny, nz, ih2) : G[l][fq];
      }
      G[l + 1][q] = T(0.125) * s;
    }
    __syncthreads();
  }
  cur[last] = smooth0(last, ncoarse);
  if (!cur[last]) { for (int q = tid; q < N[last]; q += nth) E[last][q] = T(0); __syncthreads(); cur[last] = E[last]; }
  for (int l = last - 1; l >= 0; --l) {   // upward legs
    const int nx = a.nx[l], ny = a.ny[l], cx = nx / 2, cy = ny / 2;
    T* x = cur[l] ? cur[l] : E[l];
    const T* ec = cur[l + 1];
    const bool add = cur[l] != nullptr;
    for (int q = tid; q < N[l]; q += nth) {
      int i, j, k;
      tail_ijk(q, nx, ny, i, j, k);
      const T cv = ec[(i >> 1) + cx * ((j >> 1) + cy * (k >> 1))];
      x[q] = add ? x[q] + cv : cv;
    }
    __syncthreads();
    cur[l] = smooth(l, x, nu2);
  }
  for (int q = tid; q < N[0]; q += nth) e_out[q] = cur[0][q];
}

// k_mg_tail needs up to 3 (4096 + 4096/7 + 8) words of dynamic shared memory (112 KB in fp64): per-device opt-in,
// applied by fs_grid_create for the device the grid lives on.
template <class T> cudaError_t mg_configure_device() {
  return cudaFuncSetAttribute(k_mg_tail<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(3 * (kTailCells + kTailCells / 7 + 8) * sizeof(T)));
}
template cudaError_t mg_configure_device<float>();
template cudaError_t mg_configure_device<double>();

// profile labels of the fused legs per level (bench.py sums the levels >= 1 and the tail into "mg_coarse")
static const char* const kDownName[kMaxLevels] = {"mg_down_l0", "mg_down_l1", "mg_down_l2", "mg_down_l3", "mg_down_l4", "mg_down_l5", "mg_down_l6", "mg_down_l7",
                                                  "mg_down_l8", "mg_down_l9", "mg_down_l10", "mg_down_l11"};
static const char* const kUpName[kMaxLevels] = {"mg_up_l0", "mg_up_l1", "mg_up_l2", "mg_up_l3", "mg_up_l4", "mg_up_l5", "mg_up_l6", "mg_up_l7",
                                                "mg_up_l8", "mg_up_l9", "mg_up_l10", "mg_up_l11"};

// Recursion unrolled on the host: emits the kernels of one V-cycle for rhs -> out (out = V(rhs)).
template <class T> int launch_vcycle(const Ctx<T>& c, const MgCtx<T>& mg, const T* rhs, T* out, const Launch& L, bool* dot_fused, T zs, bool* upd_fused) {
  int n = 0;
  const int* done = &c.S->done;
  const T* gl[kMaxLevels]; T* el[kMaxLevels]; T* tl[kMaxLevels]; T* cur[kMaxLevels];
  for (int l = 0; l < mg.nlev; ++l) {
    gl[l] = l == 0 ? rhs : (const T*)mg.lev[l].g;
    el[l] = l == 0 ? out : (T*)mg.lev[l].e;
    tl[l] = (T*)mg.lev[l].t;
  }
  const bool want_dot = dot_fused != nullptr;
  if (dot_fused) *dot_fused = false;
  if (upd_fused) *upd_fused = false;
  // Fast path, V(2,2) with at least two levels: two fused kernels per level (fs_kernels_mgf.cu).
  if (mg.nu1 == 2 && mg.nu2 == 2 && mg.nlev >= 2 && mg.bd == 0) {     // triply periodic: the fused legs (bounded grids: the per-sweep kernels below)
    const int last = mg.nlev - 1;
    // tail levels (small enough to live in one CTA's shared memory together): from level lt down
    int lt = last;
    while (lt > 1 && (long long)mg.lev[lt - 1].nx * mg.lev[lt - 1].ny * mg.lev[lt - 1].nz <= kTailCells) --lt;
    const bool tail_ok = (long long)mg.lev[lt].nx * mg.lev[lt].ny * mg.lev[lt].nz <= kTailCells;
    if (!tail_ok) lt = mg.nlev;          // no tail: the coarsest level is too big (cannot happen with >= 4-cell coarse boxes, kept for safety)
    const int top = tail_ok ? lt : last; // levels 0..top-1 run the fused per-level kernels
    for (int l = 0; l < top; ++l) {
      const MgLevel& V = mg.lev[l];
      const bool upd = l == 0 && upd_fused != nullptr && want_dot && c.r2 != nullptr && rhs == c.r;
      n += launch_mg_down<T>(c, gl[l], tl[l], (T*)mg.lev[l + 1].g, V.nx, V.ny, V.nz, V.h, mg.omega, kDownName[l], L,
                             upd, upd ? c.r2 : nullptr, upd ? c.q : nullptr);
      if (upd) *upd_fused = true;
    }
    const bool r_pingpong = upd_fused && *upd_fused;
    if (tail_ok) {
      MgTail a; a.nlev = mg.nlev - lt;
      size_t cells = 0;
      for (int l = lt; l < mg.nlev; ++l) {
        a.nx[l - lt] = mg.lev[l].nx; a.ny[l - lt] = mg.lev[l].ny; a.nz[l - lt] = mg.lev[l].nz; a.h[l - lt] = mg.lev[l].h;
        cells += (size_t)mg.lev[l].nx * mg.lev[l].ny * mg.lev[l].nz;
      }
      const size_t smem = 3 * cells * sizeof(T);
      FS_LAUNCH(L, "mg_tail", 2.0 * sizeof(T) * mg.lev[lt].nx * mg.lev[lt].ny * mg.lev[lt].nz,
                k_mg_tail<T><<<1, 1024, smem, L.s>>>(done, gl[lt], el[lt], a, mg.nu1, mg.nu2, mg.coarse_sweeps, mg.omega)); ++n;
    } else {
      const MgLevel& V = mg.lev[last];
      const long long N = (long long)V.nx * V.ny * V.nz;
      const T ih2 = T(1.0 / (V.h * V.h)), cw = T(mg.omega * V.h * V.h / 6.0);
      const int pre = mg.coarse_sweeps;
      if (pre <= 0) { FS_LAUNCH(L, "mg_coarse", 1.0 * sizeof(T) * N, cudaMemsetAsync(el[last], 0, sizeof(T) * (size_t)N, L.s)); ++n; }
      else {
        T* a = ((pre - 1) % 2 == 0) ? el[last] : tl[last];
        T* b = ((pre - 1) % 2 == 0) ? tl[last] : el[last];
        FS_LAUNCH(L, "mg_coarse", 2.0 * sizeof(T) * N, k_mg_first<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[last], a, cw, N, V.nx, V.ny, V.nz, 0, 0.0)); ++n;
        for (int it = 1; it < pre; ++it) {
          FS_LAUNCH(L, "mg_coarse", 3.0 * sizeof(T) * N, k_mg_sweep<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[last], a, b, V.nx, V.ny, V.nz, ih2, cw, 0, 0.0)); ++n;
          T* t = a; a = b; b = t;
        }
      }
    }
    for (int l = top - 1; l >= 0; --l) {
      const MgLevel& V = mg.lev[l];
      const bool dot = want_dot && l == 0;
      n += launch_mg_up<T>(c, tl[l], el[l + 1], gl[l], el[l], V.nx, V.ny, V.nz, V.h, mg.omega, dot, zs, kUpName[l], L,
                           (l == 0 && r_pingpong) ? c.r2 : nullptr);
      if (dot) *dot_fused = true;
    }
    return n;
  }
  // downward leg
  for (int l = 0; l < mg.nlev; ++l) {
    const MgLevel& V = mg.lev[l];
    const long long N = (long long)V.nx * V.ny * V.nz;
    const T ih2 = T(1.0 / (V.h * V.h)), cw = T(mg.omega * V.h * V.h / 6.0);
    const double wh2 = mg.omega * V.h * V.h;
    const bool coarsest = l == mg.nlev - 1;
    const int pre = coarsest ? mg.coarse_sweeps : mg.nu1;
    const int swaps = coarsest ? (pre > 0 ? pre - 1 : 0) : ((pre > 0 ? pre - 1 : 0) + mg.nu2);
    T* a = (swaps % 2 == 0) ? el[l] : tl[l];          // so that the level's final iterate lands in el[l]
    T* b = (swaps % 2 == 0) ? tl[l] : el[l];
    if (pre > 0) {
      FS_LAUNCH(L, l == 0 ? "mg_first_l0" : "mg_coarse", 2.0 * sizeof(T) * N, k_mg_first<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[l], a, cw, N, V.nx, V.ny, V.nz, mg.bd, wh2)); ++n;
      for (int it = 1; it < pre; ++it) {
        FS_LAUNCH(L, l == 0 ? "mg_sweep_l0" : "mg_coarse", 3.0 * sizeof(T) * N, k_mg_sweep<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[l], a, b, V.nx, V.ny, V.nz, ih2, cw, mg.bd, wh2)); ++n;
        T* t = a; a = b; b = t;
      }
      cur[l] = a;
    } else {
      cur[l] = nullptr;                                // e = 0
      if (coarsest) { FS_LAUNCH(L, "mg_coarse", 1.0 * sizeof(T) * N, cudaMemsetAsync(el[l], 0, sizeof(T) * (size_t)N, L.s)); ++n; cur[l] = el[l]; }
    }
    if (!coarsest) {
      const long long Nc = N / 8;
      FS_LAUNCH(L, l == 0 ? "mg_restrict_l0" : "mg_coarse", (cur[l] ? 2.125 : 1.125) * sizeof(T) * N, k_mg_restrict<T><<<flat_blocks(Nc), 256, 0, L.s>>>(done, gl[l], cur[l], (T*)mg.lev[l + 1].g, V.nx, V.ny, V.nz, ih2, mg.bd)); ++n;
    }
  }
  // upward leg
  for (int l = mg.nlev - 2; l >= 0; --l) {
    const MgLevel& V = mg.lev[l];
    const long long N = (long long)V.nx * V.ny * V.nz;
    const T ih2 = T(1.0 / (V.h * V.h)), cw = T(mg.omega * V.h * V.h / 6.0);
    const double wh2 = mg.omega * V.h * V.h;
    T* a = cur[l];
    T* dst = a ? a : ((mg.nu2 % 2 == 0) ? el[l] : tl[l]);
    FS_LAUNCH(L, l == 0 ? "mg_prolong_l0" : "mg_coarse", (a ? 2.125 : 1.125) * sizeof(T) * N, k_mg_prolong<T><<<flat_blocks(N), 256, 0, L.s>>>(done, el[l + 1], a, dst, V.nx, V.ny, V.nz)); ++n;
    a = dst;
    T* b = a == el[l] ? tl[l] : el[l];
    for (int it = 0; it < mg.nu2; ++it) {
      FS_LAUNCH(L, l == 0 ? "mg_sweep_l0" : "mg_coarse", 3.0 * sizeof(T) * N, k_mg_sweep<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[l], a, b, V.nx, V.ny, V.nz, ih2, cw, mg.bd, wh2)); ++n;
      T* t = a; a = b; b = t;
    }
    // a == el[l] by construction of the swap parity
  }
  return n;
}

template int launch_vcycle<float>(const Ctx<float>&, const MgCtx<float>&, const float*, float*, const Launch&, bool*, float, bool*);
template int launch_vcycle<double>(const Ctx<double>&, const MgCtx<double>&, const double*, double*, const Launch&, bool*, double, bool*);

}  // namespace fs
