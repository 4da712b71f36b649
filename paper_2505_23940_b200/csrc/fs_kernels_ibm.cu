// fs_kernels_ibm.cu -- direct-forcing immersed boundary between Eulerian faces and Lagrangian markers
// (S2-S5): support indices + cell list, interpolation (Eq. 3b; operator of Eq. 20), marker
// force (Eq. 5 at the markers, L108) with the body-force total (Eq. 12 sums, L147), and spreading
// (Eq. 3a) as a deterministic marker-sorted gather.  Regularised delta: tensor product (Eq. 21,
// L198-202) of the Roma 3-point kernel or the paper's 4-point kernel (Eq. 22).
// Marker data are always fp64; index arithmetic uses individually rounded operations (no FMA) so the
// integer results are bit-identical to any IEEE implementation that performs the same operations.
#include "fs_internal.cuh"

namespace fs {

// 1-D kernels with h factored out
__device__ __forceinline__ double phi_roma3(double r) {
  const double a = fabs(r);
  if (a <= 0.5) return (1.0 + sqrt(1.0 - 3.0 * a * a)) / 3.0;
  if (a <= 1.5) { const double q = 1.0 - a; return (5.0 - 3.0 * a - sqrt(1.0 - 3.0 * q * q)) / 6.0; }
  return 0.0;
}
__device__ __forceinline__ double phi_peskin4(double r) {
  const double a = fabs(r);
  if (a <= 1.0) return (3.0 - 2.0 * a + sqrt(1.0 + 4.0 * a - 4.0 * a * a)) / 8.0;
  if (a <= 2.0) return (5.0 - 2.0 * a - sqrt(-7.0 + 12.0 * a - 4.0 * a * a)) / 8.0;
  return 0.0;
}

// storage index of support node m of component c along direction d, or -1 (outside a bounded domain /
// a prescribed boundary-normal face)
template <class T> __device__ __forceinline__ int node_index(const Ctx<T>& c, int m, int comp, int d) {
  const int n = d == 0 ? c.nx : (d == 1 ? c.ny : c.nz);
  const int bd = d == 0 ? c.bx : (d == 1 ? c.by : c.bz);
  if (!bd) return wrapi(m, n);
  if (d == comp) return (m >= 1 && m <= n - 1) ? m : -1;
  return (m >= 0 && m <= n - 1) ? m : -1;
}
template <class T> __device__ __forceinline__ size_t comp_index(const Ctx<T>& c, int comp, int i, int j, int k) {
  const int ex = comp == 0 ? c.nxu : c.nx, ey = comp == 1 ? c.nyv : c.ny;
  return (size_t)i + (size_t)ex * ((size_t)j + (size_t)ey * (size_t)k);
}

// ---- I-1a: per marker: lowest support index per (component, direction), 1-D weights, cell key ------
template <class T> __global__ void k_ibm_index(const Ctx<T> c, const IbmCtx ib) {
  const int l = blockIdx.x * blockDim.x + threadIdx.x;
  if (l >= ib.n) return;
  const int n[3] = {c.nx, c.ny, c.nz}, bd[3] = {c.bx, c.by, c.bz};
  int ic[3];
  for (int d = 0; d < 3; ++d) {
    const double X = ib.X[3 * l + d];
    for (int comp = 0; comp < 3; ++comp) {
      const double sc = __dmul_rn(__dsub_rn(X, ib.org[comp][d]), ib.inv[d]);
      int base;
      if (ib.delta == FS_DELTA_ROMA3) base = (int)floor(__dadd_rn(sc, 0.5)) - 1;
      else base = (int)floor(sc) - 1;
      ib.base[((size_t)comp * ib.n + l) * 3 + d] = base;
      // a support that reaches a prescribed boundary-normal face or leaves a bounded box is unsupported
      // (sticky flag; fs_set_ibm_markers / fs_step report FS_ERR_UNSUPPORTED).  node_index keeps memory accesses safe.
      for (int a = 0; a < ib.sw; ++a) if (node_index<T>(c, base + a, comp, d) < 0) c.S->ibm_oob = 1;
      double* wt = ib.wts + (((size_t)comp * ib.n + l) * 3 + d) * 4;
      for (int a = 0; a < 4; ++a) {
        const double r = __dsub_rn(sc, (double)(base + a));
        wt[a] = a < ib.sw ? (ib.delta == FS_DELTA_ROMA3 ? phi_roma3(r) : phi_peskin4(r)) : 0.0;
      }
    }
    const int q = (int)floor(__dmul_rn(__dsub_rn(X, ib.o[d]), ib.inv[d]));
    ic[d] = bd[d] ? min(max(q, 0), n[d] - 1) : wrapi(q, n[d]);
  }
  ib.keys_raw[l] = ic[0] + c.nx * (ic[1] + c.ny * ic[2]);
}

// ---- I-1b: stable sort by (key, id) as a rank computation: rank = #{(key', id') < (key, id)} ---------
__global__ void __launch_bounds__(256) k_ibm_rank(const IbmCtx ib) {
  __shared__ int sk[256];
  const int l = blockIdx.x * blockDim.x + threadIdx.x;
  const int key = l < ib.n ? ib.keys_raw[l] : 0;
  int rank = 0;
  for (int t0 = 0; t0 < ib.n; t0 += 256) {
    const int m = t0 + threadIdx.x;
    sk[threadIdx.x] = m < ib.n ? ib.keys_raw[m] : 0x7fffffff;
    __syncthreads();
    const int lim = min(256, ib.n - t0);
    for (int a = 0; a < lim; ++a) {
      const int km = sk[a];
      rank += (km < key) || (km == key && t0 + a < l);
    }
    __syncthreads();
  }
  if (l < ib.n) { ib.perm[rank] = l; ib.keys[rank] = key; }
}

// ---- I-1c: segment starts over distinct keys (one block, chunked scan) + bounding box of supports ---
template <class T> __global__ void __launch_bounds__(1024) k_ibm_segments(const Ctx<T> c, const IbmCtx ib) {
  __shared__ int ssum[32]; __shared__ int carry; __shared__ int slo[3][32], shi[3][32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid == 0) carry = 0;
  __syncthreads();
  for (int t0 = 0; t0 < ib.n; t0 += 1024) {
    const int r = t0 + tid;
    const int flag = r < ib.n ? (r == 0 || ib.keys[r] != ib.keys[r - 1]) : 0;
    int x = flag;                                           // inclusive warp scan
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) ssum[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int s = ssum[lane];
      for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
      ssum[lane] = s;
    }
    __syncthreads();
    const int incl = x + (wid > 0 ? ssum[wid - 1] : 0) + carry;
    if (flag) ib.seg[incl - 1] = r;
    __syncthreads();
    if (tid == 1023) carry = incl;
    __syncthreads();
  }
  if (tid == 0) { ib.seg[carry] = ib.n; c.S->nseg = carry; }
  // bounding box (unwrapped node indices) of all supports, all components
  int lo[3] = {0x7fffffff, 0x7fffffff, 0x7fffffff}, hi[3] = {-0x7fffffff, -0x7fffffff, -0x7fffffff};
  for (int l = tid; l < ib.n; l += 1024)
    for (int comp = 0; comp < 3; ++comp) for (int d = 0; d < 3; ++d) {
      const int b = ib.base[((size_t)comp * ib.n + l) * 3 + d];
      lo[d] = min(lo[d], b); hi[d] = max(hi[d], b + ib.sw - 1);
    }
  for (int d = 0; d < 3; ++d) {
    for (int o = 16; o > 0; o >>= 1) { lo[d] = min(lo[d], __shfl_down_sync(0xffffffffu, lo[d], o)); hi[d] = max(hi[d], __shfl_down_sync(0xffffffffu, hi[d], o)); }
    if (lane == 0) { slo[d][wid] = lo[d]; shi[d][wid] = hi[d]; }
  }
  __syncthreads();
  if (tid == 0)
    for (int d = 0; d < 3; ++d) {
      int a = slo[d][0], b = shi[d][0];
      for (int w = 1; w < 32; ++w) { a = min(a, slo[d][w]); b = max(b, shi[d][w]); }
      c.S->bbox_lo[d] = a; c.S->bbox_hi[d] = b;
    }
}

template <class T> int launch_ibm_index(const Ctx<T>& c, const IbmCtx& ib, const Launch& L) {
  if (ib.n <= 0) return 0;
  const int nb = (ib.n + 255) / 256;
  FS_LAUNCH(L, "ibm_index", 0.0, k_ibm_index<T><<<nb, 256, 0, L.s>>>(c, ib));
  FS_LAUNCH(L, "ibm_rank", 0.0, k_ibm_rank<<<nb, 256, 0, L.s>>>(ib));
  FS_LAUNCH(L, "ibm_segments", 0.0, k_ibm_segments<T><<<1, 1024, 0, L.s>>>(c, ib));
  return 3;
}

// ---- I-2: U_l = sum over the support of u(node) * phi phi phi  (one thread per marker component) ----
template <class T> __global__ void __launch_bounds__(128) k_ibm_interp(const Ctx<T> c, const IbmCtx ib, const T* __restrict__ u,
                                                                      const T* __restrict__ v, const T* __restrict__ w, double* __restrict__ out) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 3 * ib.n) return;
  const int l = t / 3, comp = t - 3 * l;
  const T* __restrict__ f = comp == 0 ? u : (comp == 1 ? v : w);
  const int* base = ib.base + ((size_t)comp * ib.n + l) * 3;
  const double* wt = ib.wts + ((size_t)comp * ib.n + l) * 12;
  double acc = 0.0;
  for (int cc = 0; cc < ib.sw; ++cc) {
    const int kk = node_index<T>(c, base[2] + cc, comp, 2);
    for (int b = 0; b < ib.sw; ++b) {
      const int jj = node_index<T>(c, base[1] + b, comp, 1);
      for (int a = 0; a < ib.sw; ++a) {
        const int ii = node_index<T>(c, base[0] + a, comp, 0);
        if (ii < 0 || jj < 0 || kk < 0) continue;
        const double wgt = (wt[a] * wt[4 + b]) * wt[8 + cc];
        acc += (double)f[comp_index<T>(c, comp, ii, jj, kk)] * wgt;
      }
    }
  }
  out[t] = acc;
}
template <class T> int launch_ibm_interpolate(const Ctx<T>& c, const IbmCtx& ib, const T* u, const T* v, const T* w, double* out, const Launch& L) {
  if (ib.n <= 0) return 0;
  FS_LAUNCH(L, "ibm_interpolate", 3.0 * ib.sw * ib.sw * ib.sw * ib.n * sizeof(T), k_ibm_interp<T><<<(3 * ib.n + 127) / 128, 128, 0, L.s>>>(c, ib, u, v, w, out));
  return 1;
}

// ---- I-3: F_l = (U^b_l - U_l)/dt ; body force = -rho sum_l F_l dV_l (one block, fixed-order tree) ----
template <class T> __global__ void __launch_bounds__(1024) k_ibm_force(const Ctx<T> c, const IbmCtx ib) {
  __shared__ double sh[3 * 32];
  double v[3] = {0.0, 0.0, 0.0};
  for (int l = threadIdx.x; l < ib.n; l += blockDim.x)
    for (int a = 0; a < 3; ++a) {
      const double F = (ib.Ub[3 * l + a] - ib.Ul[3 * l + a]) / c.S->dt;
      ib.Fl[3 * l + a] = F;
      v[a] += F * ib.dV[l];
    }
  block_sum<3>(v, sh);
  if (threadIdx.x == 0) for (int a = 0; a < 3; ++a) c.S->body_force[a] = -c.rho * v[a];
}
template <class T> int launch_ibm_force(const Ctx<T>& c, const IbmCtx& ib, const Launch& L) {
  if (ib.n <= 0) return 0;
  FS_LAUNCH(L, "ibm_force", 0.0, k_ibm_force<T><<<1, 1024, 0, L.s>>>(c, ib));
  return 1;
}

// ---- I-4: spreading as a gather.  One thread per (component, node) of the support bounding box; it
// visits the candidate pressure cells in ascending key order and, inside a cell, the markers in cell-
// list order, so every node adds its contributions in exactly the order of the sorted marker list:
// deterministic, no atomics.   u(node) += scale * sum_l F_l phi phi phi dV_l / (hx hy hz)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int lower_bound_key(const int* __restrict__ keys, int n, int key) {
  int lo = 0, hi = n;
  while (lo < hi) { const int mid = (lo + hi) >> 1; if (keys[mid] < key) lo = mid + 1; else hi = mid; }
  return lo;
}
// candidate cell interval [m-3, m+3] along one direction as up to two ascending wrapped sub-intervals
__device__ __forceinline__ int cell_intervals(int m, int n, int bounded, int (&a)[2], int (&b)[2]) {
  int lo = m - 3, hi = m + 3;
  if (bounded) { lo = max(lo, 0); hi = min(hi, n - 1); if (lo > hi) return 0; a[0] = lo; b[0] = hi; return 1; }
  if (hi - lo + 1 >= n) { a[0] = 0; b[0] = n - 1; return 1; }
  lo = wrapi(lo, n); hi = wrapi(hi, n);
  if (lo <= hi) { a[0] = lo; b[0] = hi; return 1; }
  a[0] = 0; b[0] = hi; a[1] = lo; b[1] = n - 1; return 2;
}

template <class T> __global__ void __launch_bounds__(128) k_ibm_spread(const Ctx<T> c, const IbmCtx ib, const double* __restrict__ F,
                                                                      T* __restrict__ u, T* __restrict__ v, T* __restrict__ w, double scale) {
  const Scalars* S = c.S;
  if (scale < 0.0) scale = S->dt;          // u* = u~ + dt f with the step size of this step (Eq. 4)
  const int n[3] = {c.nx, c.ny, c.nz}, bd[3] = {c.bx, c.by, c.bz};
  int lo[3], ext[3];
  for (int d = 0; d < 3; ++d) {
    lo[d] = S->bbox_lo[d];
    ext[d] = S->bbox_hi[d] - lo[d] + 1;
    if (!bd[d]) ext[d] = min(ext[d], n[d]);       // never visit a wrapped node twice
    if (ext[d] < 0) ext[d] = 0;
  }
  const long long per = (long long)ext[0] * ext[1] * ext[2];
  const int nl = ib.n;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < 3 * per; t += (long long)gridDim.x * blockDim.x) {
    const int comp = (int)(t / per); long long r = t - comp * per;
    int m[3]; m[0] = lo[0] + (int)(r % ext[0]); r /= ext[0]; m[1] = lo[1] + (int)(r % ext[1]); m[2] = lo[2] + (int)(r / ext[1]);
    int id[3]; bool ok = true;
    for (int d = 0; d < 3; ++d) { id[d] = node_index<T>(c, m[d], comp, d); ok = ok && id[d] >= 0; }
    if (!ok) continue;
    int xa[2], xb[2], ya[2], yb[2], za[2], zb[2];
    const int nxi = cell_intervals(id[0], n[0], bd[0], xa, xb);
    const int nyi = cell_intervals(id[1], n[1], bd[1], ya, yb);
    const int nzi = cell_intervals(id[2], n[2], bd[2], za, zb);
    double acc = 0.0; bool hit = false;
    for (int zi = 0; zi < nzi; ++zi) for (int kc = za[zi]; kc <= zb[zi]; ++kc)
      for (int yi = 0; yi < nyi; ++yi) for (int jc = ya[yi]; jc <= yb[yi]; ++jc)
        for (int xi = 0; xi < nxi; ++xi) {
          const int row = c.nx * (jc + c.ny * kc);
          const int kend = row + xb[xi];
          for (int s = lower_bound_key(ib.keys, nl, row + xa[xi]); s < nl && ib.keys[s] <= kend; ++s) {
            const int l = ib.perm[s];
            const int* base = ib.base + ((size_t)comp * nl + l) * 3;
            const double* wt = ib.wts + ((size_t)comp * nl + l) * 12;
            double wgt = 1.0; bool in = true;
            for (int d = 0; d < 3; ++d) {
              int a = -1;                                       // support offset whose node is this one
              for (int q = 0; q < ib.sw; ++q) if (node_index<T>(c, base[d] + q, comp, d) == id[d]) { a = q; break; }
              if (a < 0) { in = false; break; }
              wgt *= wt[4 * d + a];
            }
            if (!in) continue;
            acc += ((F[3 * l + comp] * wgt) * ib.dV[l]) * ib.ivol;
            hit = true;
          }
        }
    if (hit) {
      T* f = comp == 0 ? u : (comp == 1 ? v : w);
      const size_t q = comp_index<T>(c, comp, id[0], id[1], id[2]);
      f[q] = T((double)f[q] + scale * acc);
    }
  }
}
template <class T> int launch_ibm_spread(const Ctx<T>& c, const IbmCtx& ib, const double* F, T* u, T* v, T* w, double scale, const Launch& L) {
  if (ib.n <= 0) return 0;
  FS_LAUNCH(L, "ibm_spread", 6.0 * ib.sw * ib.sw * ib.sw * ib.n * sizeof(T), k_ibm_spread<T><<<148 * 4, 128, 0, L.s>>>(c, ib, F, u, v, w, scale));
  return 1;
}

// =====================================================================================================
// The paper's eps-mask IBM (NEXT-1; Eq. 5, Eq. 8-9, Eq. 18-19, Eq. 23).
// =====================================================================================================
// Face classes from the cell mask: a face is solid (1) when either cell it separates is solid, an IB point (2) when it
// is fluid and one of its six same-component neighbours is solid (L74); prescribed boundary-normal faces and faces
// outside a bounded box count as fluid and are never forced.  Integer work: compared bit-exact with the oracle.
template <class T> __device__ __forceinline__ int mask_cell(const Ctx<T>& c, const unsigned char* __restrict__ eps, int i, int j, int k) {
  if (c.bx) { if (i < 0 || i >= c.nx) return 0; } else i = wrapi(i, c.nx);
  if (c.by) { if (j < 0 || j >= c.ny) return 0; } else j = wrapi(j, c.ny);
  if (c.bz) { if (k < 0 || k >= c.nz) return 0; } else k = wrapi(k, c.nz);
  return eps[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * k)] ? 1 : 0;
}
template <class T> __device__ __forceinline__ int face_solid(const Ctx<T>& c, const unsigned char* __restrict__ eps, int comp, int i, int j, int k) {
  int id[3] = {i, j, k};
  const int n[3] = {c.nx, c.ny, c.nz}, bd[3] = {c.bx, c.by, c.bz};
  for (int d = 0; d < 3; ++d) {
    if (!bd[d]) { id[d] = wrapi(id[d], n[d]); continue; }
    if (d == comp) { if (id[d] <= 0 || id[d] >= n[d]) return 0; }
    else if (id[d] < 0 || id[d] >= n[d]) return 0;
  }
  int lo[3] = {id[0], id[1], id[2]}; lo[comp] -= 1;
  return (mask_cell<T>(c, eps, id[0], id[1], id[2]) || mask_cell<T>(c, eps, lo[0], lo[1], lo[2])) ? 1 : 0;
}
template <class T> __global__ void __launch_bounds__(256) k_mask_classify(const Ctx<T> c, const IbmCtx ib) {
  const long long nU = (long long)c.nxu * c.ny * c.nz, nV = (long long)c.nx * c.nyv * c.nz, nW = (long long)c.nx * c.ny * c.nzw;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < nU + nV + nW; t += (long long)gridDim.x * blockDim.x) {
    const int comp = t < nU ? 0 : (t < nU + nV ? 1 : 2);
    const long long q = t - (comp == 0 ? 0 : (comp == 1 ? nU : nU + nV));
    const int ex = comp == 0 ? c.nxu : c.nx, ey = comp == 1 ? c.nyv : c.ny;
    const int i = (int)(q % ex), j = (int)((q / ex) % ey), k = (int)(q / ((long long)ex * ey));
    const int id[3] = {i, j, k}, n[3] = {c.nx, c.ny, c.nz}, bd[3] = {c.bx, c.by, c.bz};
    unsigned char cls = 0;
    if (!(bd[comp] && (id[comp] == 0 || id[comp] == n[comp]))) {
      if (face_solid<T>(c, ib.eps, comp, i, j, k)) cls = 1;
      else if (face_solid<T>(c, ib.eps, comp, i + 1, j, k) || face_solid<T>(c, ib.eps, comp, i - 1, j, k) ||
               face_solid<T>(c, ib.eps, comp, i, j + 1, k) || face_solid<T>(c, ib.eps, comp, i, j - 1, k) ||
               face_solid<T>(c, ib.eps, comp, i, j, k + 1) || face_solid<T>(c, ib.eps, comp, i, j, k - 1)) cls = 2;
    }
    (comp == 0 ? ib.mu : (comp == 1 ? ib.mv : ib.mw))[q] = cls;
  }
}
template <class T> int launch_mask_classify(const Ctx<T>& c, const IbmCtx& ib, const Launch& L) {
  FS_LAUNCH(L, "mask_classify", 0.0, k_mask_classify<T><<<148 * 8, 256, 0, L.s>>>(c, ib));
  return 1;
}

// Eq. 19: F_Ni = sum over the support nodes of marker i that are NOT solid of delta_h dv (one thread per marker
// component); the marker's contribution to Eq. 18 is then spread with the weight wdot_i / F_Ni (stored in Fl).
template <class T> __global__ void __launch_bounds__(128) k_mask_fn(const Ctx<T> c, const IbmCtx ib) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 3 * ib.n) return;
  const int l = t / 3, comp = t - 3 * l;
  const unsigned char* __restrict__ m = comp == 0 ? ib.mu : (comp == 1 ? ib.mv : ib.mw);
  const int* base = ib.base + ((size_t)comp * ib.n + l) * 3;
  const double* wt = ib.wts + ((size_t)comp * ib.n + l) * 12;
  double FN = 0.0;
  for (int cc = 0; cc < ib.sw; ++cc) {
    const int kk = node_index<T>(c, base[2] + cc, comp, 2);
    for (int b = 0; b < ib.sw; ++b) {
      const int jj = node_index<T>(c, base[1] + b, comp, 1);
      for (int a = 0; a < ib.sw; ++a) {
        const int ii = node_index<T>(c, base[0] + a, comp, 0);
        if (ii < 0 || jj < 0 || kk < 0) continue;
        if (m[comp_index<T>(c, comp, ii, jj, kk)] != 1) FN += (wt[a] * wt[4 + b]) * wt[8 + cc];
      }
    }
  }
  ib.Fl[t] = FN > 0.0 ? ib.Ub[t] / FN : 0.0;
}

// Eq. 4 + Eq. 5 (u* = (1 - eps) u~ + eps u_s), Eq. 23 (u_s = u_c in the solid, u_IB at the IB points) and the force on the
// body, -rho sum_x f dv with f = (u* - u~)/dt (Eq. 20 summed).  The forced value is also Eq. 9's field
// (1 - eps) u* + eps u_c: on a solid face u* = u_c, so the combination returns u_c bit for bit.
template <class T> __global__ void __launch_bounds__(256) k_mask_apply(const Ctx<T> c, const IbmCtx ib, int with_ib) {
  __shared__ double sh[3 * 32]; __shared__ int flag;
  const long long nU = (long long)c.nxu * c.ny * c.nz, nV = (long long)c.nx * c.nyv * c.nz, nW = (long long)c.nx * c.ny * c.nzw;
  double uc[3];
  for (int a = 0; a < 3; ++a) uc[a] = ib.has_body ? c.S->body_vel[a] : ib.uc[a];
  double v[3] = {0.0, 0.0, 0.0};
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < nU + nV + nW; t += (long long)gridDim.x * blockDim.x) {
    const int comp = t < nU ? 0 : (t < nU + nV ? 1 : 2);
    const long long q = t - (comp == 0 ? 0 : (comp == 1 ? nU : nU + nV));
    const int cls = (comp == 0 ? ib.mu : (comp == 1 ? ib.mv : ib.mw))[q];
    if (cls == 0 || (cls == 2 && !with_ib)) continue;
    T* f = comp == 0 ? c.us : (comp == 1 ? c.vs : c.ws);
    const T target = cls == 1 ? T(uc[comp]) : reinterpret_cast<const T*>(comp == 0 ? ib.ibu : (comp == 1 ? ib.ibv : ib.ibw))[q];
    v[comp] += ((double)target - (double)f[q]) / c.S->dt;
    f[q] = target;
  }
  if (grid_sum<3>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0) for (int a = 0; a < 3; ++a) c.S->body_force[a] = -c.rho * (v[a] * (c.hx * c.hy * c.hz));
  }
}
template <class T> int launch_mask_forcing(const Ctx<T>& c, const IbmCtx& ib, const Launch& L) {
  int n = 0;
  const int with_ib = ib.n > 0;
  if (with_ib) {
    const size_t nU = (size_t)c.nxu * c.ny * c.nz, nV = (size_t)c.nx * c.nyv * c.nz, nW = (size_t)c.nx * c.ny * c.nzw;
    FS_LAUNCH(L, "mask_ib_points", 0.0, {
      k_mask_fn<T><<<(3 * ib.n + 127) / 128, 128, 0, L.s>>>(c, ib);
      cudaMemsetAsync(ib.ibu, 0, nU * sizeof(T), L.s); cudaMemsetAsync(ib.ibv, 0, nV * sizeof(T), L.s); cudaMemsetAsync(ib.ibw, 0, nW * sizeof(T), L.s);
    });
    n += 4;
    n += launch_ibm_spread<T>(c, ib, ib.Fl, (T*)ib.ibu, (T*)ib.ibv, (T*)ib.ibw, 1.0, L);
  }
  FS_LAUNCH(L, "mask_forcing", 0.0, k_mask_apply<T><<<148 * 8, 256, 0, L.s>>>(c, ib, with_ib));
  return n + 1;
}

#define INST(T)                                                                                                             \
  template int launch_mask_classify<T>(const Ctx<T>&, const IbmCtx&, const Launch&);                                        \
  template int launch_mask_forcing<T>(const Ctx<T>&, const IbmCtx&, const Launch&);                                         \
  template int launch_ibm_index<T>(const Ctx<T>&, const IbmCtx&, const Launch&);                                            \
  template int launch_ibm_interpolate<T>(const Ctx<T>&, const IbmCtx&, const T*, const T*, const T*, double*, const Launch&); \
  template int launch_ibm_force<T>(const Ctx<T>&, const IbmCtx&, const Launch&);                                            \
  template int launch_ibm_spread<T>(const Ctx<T>&, const IbmCtx&, const double*, T*, T*, T*, double, const Launch&);
INST(float)
INST(double)

}  // namespace fs
