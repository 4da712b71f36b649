// fs_kernels_mg.cu -- geometric-multigrid V-cycle preconditioner (S7g; not in the
// paper, named by BASELINE.json c5).  Uniform, isotropic, all-periodic grids.  Per level: nu1 damped-
// Jacobi sweeps from a zero guess, residual, 8-cell-average restriction, recursion, piecewise-constant
// prolongation + correction, nu2 sweeps; the coarsest level does a fixed number of sweeps.  The operator
// on every level is the rediscretised 7-point -L.  Jacobi is order independent, so the result matches
// the CPU oracle up to summation rounding.
#include "fs_internal.cuh"

namespace fs {

constexpr int kFlatBlocks = 148 * 8;
static inline int flat_blocks(long long n) { long long b = (n + 255) / 256; return (int)(b < kFlatBlocks ? (b < 1 ? 1 : b) : kFlatBlocks); }

template <class T> __device__ __forceinline__ T neg_lap(const T* __restrict__ e, int i, int j, int k, int nx, int ny, int nz, T ih2) {
  const int ip = i + 1 == nx ? 0 : i + 1, im = i == 0 ? nx - 1 : i - 1;
  const int jp = j + 1 == ny ? 0 : j + 1, jm = j == 0 ? ny - 1 : j - 1;
  const int kp = k + 1 == nz ? 0 : k + 1, km = k == 0 ? nz - 1 : k - 1;
  const size_t row = (size_t)nx * ((size_t)j + (size_t)ny * k);
  const T nb = e[row + ip] + e[row + im] + e[(size_t)i + (size_t)nx * ((size_t)jp + (size_t)ny * k)] +
               e[(size_t)i + (size_t)nx * ((size_t)jm + (size_t)ny * k)] + e[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * kp)] +
               e[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * km)];
  return (T(6) * e[row + i] - nb) * ih2;
}

// first sweep from a zero guess: e = omega D^-1 g
template <class T> __global__ void __launch_bounds__(256) k_mg_first(const int* __restrict__ done, const T* __restrict__ g, T* __restrict__ e, T cw, long long N) {
  if (done && *done) return;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) e[q] = cw * g[q];
}
// damped-Jacobi sweep  dst = src + omega D^-1 (g - (-L) src)
template <class T> __global__ void __launch_bounds__(256) k_mg_sweep(const int* __restrict__ done, const T* __restrict__ g, const T* __restrict__ src,
                                                                    T* __restrict__ dst, int nx, int ny, int nz, T ih2, T cw) {
  if (done && *done) return;
  const long long N = (long long)nx * ny * nz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % nx); const long long t = q / nx; const int j = (int)(t % ny), k = (int)(t / ny);
    dst[q] = src[q] + cw * (g[q] - neg_lap<T>(src, i, j, k, nx, ny, nz, ih2));
  }
}
// residual + restriction: gc = mean over the 8 children of (g - (-L) e); e == nullptr means e = 0
template <class T> __global__ void __launch_bounds__(256) k_mg_restrict(const int* __restrict__ done, const T* __restrict__ g, const T* __restrict__ e,
                                                                       T* __restrict__ gc, int nx, int ny, int nz, T ih2) {
  if (done && *done) return;
  const int cx = nx / 2, cy = ny / 2, cz = nz / 2;
  const long long Nc = (long long)cx * cy * cz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < Nc; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % cx); const long long t = q / cx; const int j = (int)(t % cy), k = (int)(t / cy);
    T a = T(0);
    for (int dk = 0; dk < 2; ++dk) for (int dj = 0; dj < 2; ++dj) for (int di = 0; di < 2; ++di) {
      const int fi = 2 * i + di, fj = 2 * j + dj, fk = 2 * k + dk;
      const size_t fq = (size_t)fi + (size_t)nx * ((size_t)fj + (size_t)ny * fk);
      a += e ? g[fq] - neg_lap<T>(e, fi, fj, fk, nx, ny, nz, ih2) : g[fq];
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

// Recursion unrolled on the host: emits the kernels of one V-cycle for rhs -> out (out = V(rhs)).
template <class T> int launch_vcycle(const Ctx<T>& c, const MgCtx<T>& mg, const T* rhs, T* out, const Launch& L, bool* dot_fused, T zs) {
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
  // Fast path, V(2,2) with at least two levels: two fused kernels per level (fs_kernels_mgf.cu).
  if (mg.nu1 == 2 && mg.nu2 == 2 && mg.nlev >= 2) {
    const int last = mg.nlev - 1;
    for (int l = 0; l < last; ++l) {
      const MgLevel& V = mg.lev[l];
      n += launch_mg_down<T>(c, gl[l], tl[l], (T*)mg.lev[l + 1].g, V.nx, V.ny, V.nz, V.h, mg.omega, l == 0 ? "mg_down_l0" : "mg_coarse", L);
    }
    {
      const MgLevel& V = mg.lev[last];
      const long long N = (long long)V.nx * V.ny * V.nz;
      const T ih2 = T(1.0 / (V.h * V.h)), cw = T(mg.omega * V.h * V.h / 6.0);
      const int pre = mg.coarse_sweeps;
      if (pre <= 0) { FS_LAUNCH(L, "mg_coarse", 1.0 * sizeof(T) * N, cudaMemsetAsync(el[last], 0, sizeof(T) * (size_t)N, L.s)); ++n; }
      else {
        T* a = ((pre - 1) % 2 == 0) ? el[last] : tl[last];
        T* b = ((pre - 1) % 2 == 0) ? tl[last] : el[last];
        FS_LAUNCH(L, "mg_coarse", 2.0 * sizeof(T) * N, k_mg_first<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[last], a, cw, N)); ++n;
        for (int it = 1; it < pre; ++it) {
          FS_LAUNCH(L, "mg_coarse", 3.0 * sizeof(T) * N, k_mg_sweep<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[last], a, b, V.nx, V.ny, V.nz, ih2, cw)); ++n;
          T* t = a; a = b; b = t;
        }
      }
    }
    for (int l = last - 1; l >= 0; --l) {
      const MgLevel& V = mg.lev[l];
      const bool dot = want_dot && l == 0;
      n += launch_mg_up<T>(c, tl[l], el[l + 1], gl[l], el[l], V.nx, V.ny, V.nz, V.h, mg.omega, dot, zs, l == 0 ? "mg_up_l0" : "mg_coarse", L);
      if (dot) *dot_fused = true;
    }
    return n;
  }
  // downward leg
  for (int l = 0; l < mg.nlev; ++l) {
    const MgLevel& V = mg.lev[l];
    const long long N = (long long)V.nx * V.ny * V.nz;
    const T ih2 = T(1.0 / (V.h * V.h)), cw = T(mg.omega * V.h * V.h / 6.0);
    const bool coarsest = l == mg.nlev - 1;
    const int pre = coarsest ? mg.coarse_sweeps : mg.nu1;
    const int swaps = coarsest ? (pre > 0 ? pre - 1 : 0) : ((pre > 0 ? pre - 1 : 0) + mg.nu2);
    T* a = (swaps % 2 == 0) ? el[l] : tl[l];          // so that the level's final iterate lands in el[l]
    T* b = (swaps % 2 == 0) ? tl[l] : el[l];
    if (pre > 0) {
      FS_LAUNCH(L, l == 0 ? "mg_first_l0" : "mg_coarse", 2.0 * sizeof(T) * N, k_mg_first<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[l], a, cw, N)); ++n;
      for (int it = 1; it < pre; ++it) {
        FS_LAUNCH(L, l == 0 ? "mg_sweep_l0" : "mg_coarse", 3.0 * sizeof(T) * N, k_mg_sweep<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[l], a, b, V.nx, V.ny, V.nz, ih2, cw)); ++n;
        T* t = a; a = b; b = t;
      }
      cur[l] = a;
    } else {
      cur[l] = nullptr;                                // e = 0
      if (coarsest) { FS_LAUNCH(L, "mg_coarse", 1.0 * sizeof(T) * N, cudaMemsetAsync(el[l], 0, sizeof(T) * (size_t)N, L.s)); ++n; cur[l] = el[l]; }
    }
    if (!coarsest) {
      const long long Nc = N / 8;
      FS_LAUNCH(L, l == 0 ? "mg_restrict_l0" : "mg_coarse", (cur[l] ? 2.125 : 1.125) * sizeof(T) * N, k_mg_restrict<T><<<flat_blocks(Nc), 256, 0, L.s>>>(done, gl[l], cur[l], (T*)mg.lev[l + 1].g, V.nx, V.ny, V.nz, ih2)); ++n;
    }
  }
  // upward leg
  for (int l = mg.nlev - 2; l >= 0; --l) {
    const MgLevel& V = mg.lev[l];
    const long long N = (long long)V.nx * V.ny * V.nz;
    const T ih2 = T(1.0 / (V.h * V.h)), cw = T(mg.omega * V.h * V.h / 6.0);
    T* a = cur[l];
    T* dst = a ? a : ((mg.nu2 % 2 == 0) ? el[l] : tl[l]);
    FS_LAUNCH(L, l == 0 ? "mg_prolong_l0" : "mg_coarse", (a ? 2.125 : 1.125) * sizeof(T) * N, k_mg_prolong<T><<<flat_blocks(N), 256, 0, L.s>>>(done, el[l + 1], a, dst, V.nx, V.ny, V.nz)); ++n;
    a = dst;
    T* b = a == el[l] ? tl[l] : el[l];
    for (int it = 0; it < mg.nu2; ++it) {
      FS_LAUNCH(L, l == 0 ? "mg_sweep_l0" : "mg_coarse", 3.0 * sizeof(T) * N, k_mg_sweep<T><<<flat_blocks(N), 256, 0, L.s>>>(done, gl[l], a, b, V.nx, V.ny, V.nz, ih2, cw)); ++n;
      T* t = a; a = b; b = t;
    }
    // a == el[l] by construction of the swap parity
  }
  return n;
}

template int launch_vcycle<float>(const Ctx<float>&, const MgCtx<float>&, const float*, float*, const Launch&, bool*, float);
template int launch_vcycle<double>(const Ctx<double>&, const MgCtx<double>&, const double*, double*, const Launch&, bool*, double);

}  // namespace fs
