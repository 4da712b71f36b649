// fs_kernels_fluid.cu -- momentum RHS + predictor (S0+S1), open-boundary flux correction (O5),
// Poisson right-hand side (S6), projection + divergence diagnostics (S8), step bookkeeping (S9/S10).
// Hand-written for sm_100a; shares nothing with oracle/.
#include "fs_internal.cuh"
#include <cstring>
#include <cstdlib>

namespace fs {

static int tune_pf() { const char* e = getenv("FS_TUNE_PF2"); return e ? atoi(e) : 1; }   // experiments: FS_TUNE_PF2=0 turns the TMA prefetches off


constexpr int kFlatBlocks = 148 * 8;
static inline int flat_blocks(long long n) { long long b = (n + 255) / 256; return (int)(b < kFlatBlocks ? (b < 1 ? 1 : b) : kFlatBlocks); }

// ---------------------------------------------------------------------------------------------------
// Boundary-aware velocity access (S0): see col_setup / col_fix below.
// Component C at (i,j,k), at most one layer outside the stored range in a direction tangential to C:
//   periodic      : index wrap
//   no-slip/inflow: ghost = 2*u_wall - u_interior      slip/outflow: ghost = u_interior
// Along its own normal a bounded component stores faces 0..n, so no ghost is needed there.
// ---------------------------------------------------------------------------------------------------

// Counter-based inflow noise (O1): SplitMix64 finaliser chained over (seed, face, step, a, b) and
// mapped to [0,1) by (x >> 11) * 2^-53.  The oracle implements the same generator independently.
__device__ __forceinline__ uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
__device__ __forceinline__ double inflow_rand(uint64_t seed, long long step, int face, int a, int b) {
  uint64_t h = mix64(seed + 0x632BE59BD9B4E019ULL * (uint64_t)(face + 1));
  h = mix64(h + (uint64_t)step);
  h = mix64(h + (((uint64_t)(uint32_t)b << 32) | (uint64_t)(uint32_t)a));
  return (double)(h >> 11) * (1.0 / 9007199254740992.0);
}

// Value of a prescribed boundary-normal face of the predicted field (O1/O3).
//   old = u^n of that component, q = index of the face, qi = index of its interior neighbour face.
template <class T> __device__ __forceinline__ T boundary_normal(const Ctx<T>& c, const T* __restrict__ old, int d, int side,
                                                               int a, int b, size_t q, size_t qi, int jedge, double dtc) {
  const int face = 2 * d + side, t = c.bc[face];
  const double Ub = c.bcv[face][d];
  if (t == FS_BC_NOSLIP) return T(Ub);
  if (t == FS_BC_SLIP) return T(0);
  if (t == FS_BC_INFLOW) {
    double r = inflow_rand(c.seed, c.S->step, face, a, b);
    return T(Ub * (1.0 + c.inflow_noise * (2.0 * r - 1.0)));
  }
  // convective outflow (reading): du/dt + Uc du/dn = 0, first-order upwind
  const double dn = d == 0 ? c.hx : (d == 1 ? (double)c.dy64[jedge] : c.hz);
  const double o = (double)old[q], oi = (double)old[qi];
  const double grad = side ? (o - oi) / dn : (oi - o) / dn;
  return T(o - Ub * dtc * grad);
}

// ---------------------------------------------------------------------------------------------------
// S1: H^n = -div(u u) + nu lap(u) + g (central / central, Eq. 4) and the explicit
// predictor u~ = u^n + dt (a0 H^n + a1 H^{n-1}); prescribed boundary-normal faces get their O1 values.
//
// 2.5-D halo-tiled streaming kernel: a CTA owns a 30 x 8 column of cells of the extended box
// (nxu x nyv x nzw) plus a one-cell halo (32 x 10 threads, one thread per extended-tile cell) and marches
// in z.  Every plane of u, v, w is read once per CTA through the boundary-aware accessor (S0 folded into
// the tile load: wrap / ghost reflection are resolved when the value enters shared memory), kept in a
// four-slot ring of shared-memory planes (planes k-1, k, k+1 are live, the fourth slot takes the prefetch
// without a second barrier) and in a register queue for the thread's own column.  One __syncthreads per
// plane; H^{n-1} is read and H^n, u~ are written straight from / to global memory, coalesced.
// ---------------------------------------------------------------------------------------------------
constexpr int kMomTX = 32, kMomTY = 10;

// transported face value of a convective flux a * phi: central interpolation, or (first-order upwind, PAPER.md L100;
// DESIGN.md reading N3-1) the value on the upwind side of the face
template <class T> __device__ __forceinline__ T transported(bool upwind, T a, T minus, T plus, T central) {
  return upwind ? (a > T(0) ? minus : plus) : central;
}

template <class T> struct ColRef { unsigned off, pl; T A, B; };   // 32-bit element offsets: every field has < 2^32 entries (validated)   // value = A f[off + pl kz] + B  (x, y ghosts resolved)

template <class T, int C> __device__ __forceinline__ ColRef<T> col_setup(const Ctx<T>& c, int i, int j) {
  T A = T(1), B = T(0);
  if (!c.bx) i = wrapi(i, c.nx);
  else if (C != 0) {
    int face = -1;
    if (i < 0) { face = 0; i = -1 - i; } else if (i >= c.nx) { face = 1; i = 2 * c.nx - 1 - i; }
    if (face >= 0 && (c.bc[face] == FS_BC_NOSLIP || c.bc[face] == FS_BC_INFLOW)) { B = T(2.0 * c.bcv[face][C]) - B; A = -A; }
  } else i = min(max(i, 0), c.nx);
  if (!c.by) j = wrapi(j, c.ny);
  else if (C != 1) {
    int face = -1;
    if (j < 0) { face = 2; j = -1 - j; } else if (j >= c.ny) { face = 3; j = 2 * c.ny - 1 - j; }
    if (face >= 0 && (c.bc[face] == FS_BC_NOSLIP || c.bc[face] == FS_BC_INFLOW)) { B = T(2.0 * c.bcv[face][C]) - B; A = -A; }
  } else j = min(max(j, 0), c.ny);
  const int ex = C == 0 ? c.nxu : c.nx, ey = C == 1 ? c.nyv : c.ny;
  ColRef<T> r;
  r.off = (unsigned)i + (unsigned)ex * (unsigned)j; r.pl = (unsigned)ex * (unsigned)ey; r.A = A; r.B = B;
  return r;
}
// plane kk in [-1, nzw] of component C for this thread's column: the raw load and, separately, the ghost
// fix-up (so that the load can stay in flight for a whole plane before its value is touched)
template <class T, int C> __device__ __forceinline__ int col_plane(const Ctx<T>& c, int kk) {
  if (!c.bz) return kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk);
  if (C != 2) return kk < 0 ? -1 - kk : (kk >= c.nz ? 2 * c.nz - 1 - kk : kk);
  return min(max(kk, 0), c.nz);
}
template <class T, int C> __device__ __forceinline__ T col_raw(const Ctx<T>& c, const T* __restrict__ f, const ColRef<T>& r, int kk) {
  return f[r.off + r.pl * (unsigned)col_plane<T, C>(c, kk)];
}
template <class T, int C> __device__ __forceinline__ T col_fix(const Ctx<T>& c, const ColRef<T>& r, int kk, T raw) {
  T A = r.A, B = r.B;
  if (c.bz && C != 2) {
    const int face = kk < 0 ? 4 : (kk >= c.nz ? 5 : -1);
    if (face >= 0 && (c.bc[face] == FS_BC_NOSLIP || c.bc[face] == FS_BC_INFLOW)) { B = T(2.0 * c.bcv[face][C]) - B; A = -A; }
  }
  return A * raw + B;
}
template <class T, int C> __device__ __forceinline__ T col_load(const Ctx<T>& c, const T* __restrict__ f, const ColRef<T>& r, int kk) {
  return col_fix<T, C>(c, r, kk, col_raw<T, C>(c, f, r, kk));
}

// ---- LES closures (NEXT-4; section 3.4.5) -------------------------------------------
// Spalding's law (Eq. 27, kappa = 0.4, B = 5): u_tau for the wall-parallel speed U at distance y, Newton-Raphson on
// g(u_tau) = u+ + e^{-kappa B}[e^{kappa u+} - 1 - kappa u+ - (kappa u+)^2/2 - (kappa u+)^3/6] - y+ (convex, decreasing:
// monotone convergence from the left); start u+ = min(sqrt(Re_y), max(12.5, ln(1.182 Re_y)/kappa)), 30 iterations.
__device__ __forceinline__ double wall_utau(double U, double y, double nu) {
  if (!(U > 0.0)) return 0.0;
  const double kap = 0.4, eB = exp(-kap * 5.0);
  const double Rey = U * y / nu;
  const double up0 = fmin(sqrt(Rey), fmax(12.5, log(1.182 * Rey) / kap));
  double ut = U / up0;
  for (int it = 0; it < 30; ++it) {
    const double up = U / ut, yp = y * ut / nu, ku = kap * up, e = exp(ku);
    const double gval = up + eB * (e - 1.0 - ku - 0.5 * ku * ku - ku * ku * ku / 6.0) - yp;
    const double dgdup = 1.0 + eB * kap * (e - 1.0 - ku - 0.5 * ku * ku);
    const double dg = dgdup * (-up / ut) - y / nu;
    ut = ut - gval / dg;
  }
  return ut;
}
// Eq. 28-29: nu_t on the wall face that makes the flux of the tangential component (rel; the other one: other; both
// relative to the wall, first off-wall point at distance y) equal to tau_wi / rho = u_tau^2 rel / |U|
__device__ __forceinline__ double wall_nut(double rel, double other, double y, double nu) {
  const double U = sqrt(rel * rel + other * other);
  if (!(U > 0.0)) return 0.0;
  const double ut = wall_utau(U, y, nu);
  return (ut * ut * rel / U) / (rel / y + 1e-6) - nu;
}

// Constant Smagorinsky eddy viscosity at the cell centres (reading N4-1), nu_t = (C_s Delta)^2 sqrt(2 S_ij S_ij): diagonal
// gradients from the cell's own faces, cross gradients as central differences of face values averaged to the centres.
// One cell per thread through the boundary-aware accessors (not on the benchmarked path).
template <class T> __global__ void __launch_bounds__(256) k_eddy_viscosity(const Ctx<T> c, T* __restrict__ nut) {
  const long long N = (long long)c.nx * c.ny * c.nz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % c.nx); const long long t = q / c.nx; const int j = (int)(t % c.ny), k = (int)(t / c.ny);
    auto U = [&](int ii, int jj, int kk) { return (double)col_load<T, 0>(c, c.u, col_setup<T, 0>(c, ii, jj), kk); };
    auto V = [&](int ii, int jj, int kk) { return (double)col_load<T, 1>(c, c.v, col_setup<T, 1>(c, ii, jj), kk); };
    auto W = [&](int ii, int jj, int kk) { return (double)col_load<T, 2>(c, c.w, col_setup<T, 2>(c, ii, jj), kk); };
    auto ux = [&](int jj, int kk) { return 0.5 * (U(i, jj, kk) + U(i + 1, jj, kk)); };
    auto vy = [&](int ii, int kk) { return 0.5 * (V(ii, j, kk) + V(ii, j + 1, kk)); };
    auto wz = [&](int ii, int jj) { return 0.5 * (W(ii, jj, k) + W(ii, jj, k + 1)); };
    const double dyj = c.dy64[j];
    const double dyc2 = 1.0 / (double)c.idyc[j + 1] + 1.0 / (double)c.idyc[j];
    const double dudx = (U(i + 1, j, k) - U(i, j, k)) / c.hx, dvdy = (V(i, j + 1, k) - V(i, j, k)) / dyj, dwdz = (W(i, j, k + 1) - W(i, j, k)) / c.hz;
    const double dudy = (ux(j + 1, k) - ux(j - 1, k)) / dyc2, dudz = (ux(j, k + 1) - ux(j, k - 1)) / (2.0 * c.hz);
    const double dvdx = (vy(i + 1, k) - vy(i - 1, k)) / (2.0 * c.hx), dvdz = (vy(i, k + 1) - vy(i, k - 1)) / (2.0 * c.hz);
    const double dwdx = (wz(i + 1, j) - wz(i - 1, j)) / (2.0 * c.hx), dwdy = (wz(i, j + 1) - wz(i, j - 1)) / dyc2;
    const double S2 = 2.0 * (dudx * dudx + dvdy * dvdy + dwdz * dwdz)
                    + (dudy + dvdx) * (dudy + dvdx) + (dudz + dwdx) * (dudz + dwdx) + (dvdz + dwdy) * (dvdz + dwdy);
    const double delta = cbrt(c.hx * dyj * c.hz);
    nut[q] = T((c.cs * delta) * (c.cs * delta) * sqrt(S2));
  }
}

// LES variant of the kernel (template flag): the diffusive term becomes div[(nu + nu_t) grad u_i] with nu_t (array `nut`,
// cell centred) at the flux locations -- cell centres natively, edges as the mean of the four surrounding cells -- through
// a fourth shared-memory ring; on the wall faces of no-slip y walls nu_t is the wall model's (Eq. 28).
// ADT (CFL-adaptive dt): the step size and the variable-step AB2 coefficients are read from device memory; the fixed-step
// variant keeps them as constant-bank operands / immediates (the kernel sits at its register limit: three more live
// doubles cost it a third of its speed).
template <class T, bool UPW, bool LES, bool ADT> __global__ void __launch_bounds__(kMomTX * kMomTY, LES ? 1 : 2) k_momentum(const Ctx<T> c, int kz, const T* __restrict__ nut) {
  __shared__ T SU[4][kMomTY][kMomTX], SV[4][kMomTY][kMomTX], SW[4][kMomTY][kMomTX];
  __shared__ T SN[LES ? 4 : 1][LES ? kMomTY : 1][LES ? kMomTX : 1];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int iu = blockIdx.x * (kMomTX - 2) + tx - 1, ju = blockIdx.y * (kMomTY - 2) + ty - 1;   // may be -1 or past the box
  const int i = min(iu, c.nxu), j = min(ju, c.nyv);
  const bool own = tx >= 1 && tx <= kMomTX - 2 && ty >= 1 && ty <= kMomTY - 2 && iu < c.nxu && ju < c.nyv;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nzw);
  const bool ab2 = c.time_scheme == FS_TIME_AB2 && c.S->have_hist;
  // AB2 with the step-size ratio r = dt_n / dt_{n-1}: a0 = 1 + r/2, a1 = -r/2 (3/2, -1/2 for a fixed step)
  const double rdt = (ADT && ab2) ? c.S->dt / c.S->dt_prev : 1.0;
  const T a0 = ab2 ? (ADT ? T(1.0 + 0.5 * rdt) : T(1.5)) : T(1), a1 = ab2 ? (ADT ? T(-0.5 * rdt) : T(-0.5)) : T(0);
  const T dt = ADT ? T(c.S->dt) : T(c.dt), nu = T(c.nu);
  constexpr bool upw = UPW;                // convective scheme: compile-time, so the central path carries no selects
  const T* __restrict__ U = c.u; const T* __restrict__ V = c.v; const T* __restrict__ W = c.w;
  const ColRef<T> ru = col_setup<T, 0>(c, i, j), rv = col_setup<T, 1>(c, i, j), rw = col_setup<T, 2>(c, i, j);
  // y metrics of the tile rows, in shared memory (j clamped into the tables; unused rows never store)
  __shared__ T MY[8][kMomTY];
  if (tx < 8) {
    const int jc = min(max(j, 0), c.ny - 1);
    const T* tab = tx == 0 ? c.wyl + jc : tx == 1 ? c.wyh + jc : tx == 2 ? c.wyl + jc + 1 : tx == 3 ? c.wyh + jc + 1
                 : tx == 4 ? c.idy + jc + 1 : tx == 5 ? c.idy + jc : tx == 6 ? c.idyc + jc : c.idyc + jc + 1;
    MY[tx][ty] = *tab;
  }
  // nu_t of the own column: cell index wrapped (periodic) or clamped to the boundary cell (bounded)
  unsigned nq0 = 0; const unsigned npl = (unsigned)c.nx * (unsigned)c.ny;
  auto nplane = [&](int kk) { return (unsigned)(c.bz ? min(max(kk, 0), c.nz - 1) : (kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk))); };
  if (LES) {
    const int ic = c.bx ? min(max(iu, 0), c.nx - 1) : wrapi(iu, c.nx), jc = c.by ? min(max(ju, 0), c.ny - 1) : wrapi(ju, c.ny);
    nq0 = (unsigned)ic + (unsigned)c.nx * (unsigned)jc;
    SN[(k0 - 1) & 3][ty][tx] = nut[nq0 + npl * nplane(k0 - 1)];
    SN[k0 & 3][ty][tx] = nut[nq0 + npl * nplane(k0)];
  }
  const bool wm_lo = LES && c.wall_model && c.by && c.bc[2] == FS_BC_NOSLIP, wm_hi = LES && c.wall_model && c.by && c.bc[3] == FS_BC_NOSLIP;
  // register queue of the own column: B = k-1, c = k, T = k+1
  T uB = col_load<T, 0>(c, U, ru, k0 - 1), vB = col_load<T, 1>(c, V, rv, k0 - 1), wB = col_load<T, 2>(c, W, rw, k0 - 1);
  T uc = col_load<T, 0>(c, U, ru, k0), vc = col_load<T, 1>(c, V, rv, k0), wc = col_load<T, 2>(c, W, rw, k0);
  T un = col_raw<T, 0>(c, U, ru, k0 + 1), vn = col_raw<T, 1>(c, V, rv, k0 + 1), wn = col_raw<T, 2>(c, W, rw, k0 + 1);   // raw, in flight
  SU[(k0 - 1) & 3][ty][tx] = uB; SV[(k0 - 1) & 3][ty][tx] = vB; SW[(k0 - 1) & 3][ty][tx] = wB;
  SU[k0 & 3][ty][tx] = uc; SV[k0 & 3][ty][tx] = vc; SW[k0 & 3][ty][tx] = wc;
  const int txm = max(tx - 1, 0), txp = min(tx + 1, kMomTX - 1), tym = max(ty - 1, 0), typ = min(ty + 1, kMomTY - 1);
  // H^{n-1} of the own faces, prefetched one plane ahead (zero where the face does not exist)
  const bool hasu = own && j < c.ny, hasv = own && i < c.nx, hasw = own && i < c.nx && j < c.ny;
  const unsigned qu0 = (unsigned)i + (unsigned)c.nxu * (unsigned)j, plu = (unsigned)c.nxu * (unsigned)c.ny;
  const unsigned qv0 = (unsigned)i + (unsigned)c.nx * (unsigned)j, plv = (unsigned)c.nx * (unsigned)c.nyv;
  const unsigned qw0 = qv0, plw = (unsigned)c.nx * (unsigned)c.ny;
  T hun = (hasu && k0 < c.nz) ? c.hu[qu0 + plu * k0] : T(0);
  T hvn = (hasv && k0 < c.nz) ? c.hv[qv0 + plv * k0] : T(0);
  T hwn = hasw ? c.hw[qw0 + plw * k0] : T(0);
  for (int k = k0; k < k1; ++k) {
    const T uT = col_fix<T, 0>(c, ru, k + 1, un), vT = col_fix<T, 1>(c, rv, k + 1, vn), wT = col_fix<T, 2>(c, rw, k + 1, wn);
    const T huo = hun, hvo = hvn, hwo = hwn;
    if (k + 1 < k1) {
      hun = (hasu && k + 1 < c.nz) ? c.hu[qu0 + plu * (k + 1)] : T(0);
      hvn = (hasv && k + 1 < c.nz) ? c.hv[qv0 + plv * (k + 1)] : T(0);
      hwn = hasw ? c.hw[qw0 + plw * (k + 1)] : T(0);
    }
    const int s0 = (k - 1) & 3, s1 = k & 3, s2 = (k + 1) & 3;
    SU[s2][ty][tx] = uT; SV[s2][ty][tx] = vT; SW[s2][ty][tx] = wT;
    if (LES) SN[s2][ty][tx] = nut[nq0 + npl * nplane(k + 1)];
    if (k + 1 < k1) { un = col_raw<T, 0>(c, U, ru, k + 2); vn = col_raw<T, 1>(c, V, rv, k + 2); wn = col_raw<T, 2>(c, W, rw, k + 2); }
    __syncthreads();
    if (own) {
      const T wyl0 = MY[0][ty], wyh0 = MY[1][ty], wyl1 = MY[2][ty], wyh1 = MY[3][ty];
      const T idyj = MY[4][ty], idyjm = MY[5][ty], idyc0 = MY[6][ty], idyc1 = MY[7][ty];
      // ---- u face ----
      if (j < c.ny && k < c.nz) {
        const size_t q = qu0 + plu * (unsigned)k;
        if (c.bx && (i == 0 || i == c.nx)) {
          const int side = i == 0 ? 0 : 1;
          const size_t qi = side ? q - 1 : q + 1;
          c.us[q] = boundary_normal<T>(c, U, 0, side, j, k, q, qi, 0, (double)dt);
          c.hu[q] = T(0);
        } else {
          const T uE = SU[s1][ty][txp], uW = SU[s1][ty][txm], uN = SU[s1][typ][tx], uS = SU[s1][tym][tx];
          const T ue = T(0.5) * (uc + uE), uw = T(0.5) * (uW + uc);
          const T cx = (ue * transported<T>(upw, ue, uc, uE, ue) - uw * transported<T>(upw, uw, uW, uc, uw)) * c.ihx;
          const T vnn = T(0.5) * (SV[s1][typ][txm] + SV[s1][typ][tx]), unn = transported<T>(upw, vnn, uc, uN, wyl1 * uc + wyh1 * uN);
          const T vss = T(0.5) * (SV[s1][ty][txm] + vc),                uss = transported<T>(upw, vss, uS, uc, wyl0 * uS + wyh0 * uc);
          const T cy = (vnn * unn - vss * uss) * idyj;
          const T wt = T(0.5) * (SW[s2][ty][txm] + wT), ut = transported<T>(upw, wt, uc, uT, T(0.5) * (uc + uT));
          const T wb = T(0.5) * (SW[s1][ty][txm] + wc), ub = transported<T>(upw, wb, uB, uc, T(0.5) * (uB + uc));
          const T cz = (wt * ut - wb * ub) * c.ihz;
          const T dxx = (uE - T(2) * uc + uW) * c.ihx2;
          const T dyy = ((uN - uc) * idyc1 - (uc - uS) * idyc0) * idyj;
          const T dzz = (uT - T(2) * uc + uB) * c.ihz2;
          T H;
          if (LES) {
            const T nC = SN[s1][ty][tx], nW = SN[s1][ty][txm];
            const T fxe = (nu + nC) * (uE - uc) * c.ihx, fxw = (nu + nW) * (uc - uW) * c.ihx;
            T nn = T(0.25) * (((nW + nC) + SN[s1][typ][txm]) + SN[s1][typ][tx]), ns = T(0.25) * (((SN[s1][tym][txm] + SN[s1][tym][tx]) + nW) + nC);
            if ((wm_lo && j == 0) || (wm_hi && j == c.ny - 1)) {     // Eq. 28: u relative to the wall, w interpolated to the u face
              const int f = j == 0 ? 2 : 3;
              const double wf = 0.25 * ((((double)SW[s1][ty][txm] + (double)wc) + (double)SW[s2][ty][txm]) + (double)wT);
              const T nw = T(wall_nut((double)uc - c.bcv[f][0], wf - c.bcv[f][2], 0.5 * c.dy64[j], c.nu));
              if (j == 0) ns = nw; else nn = nw;
            }
            const T fyn = (nu + nn) * (uN - uc) * idyc1, fys = (nu + ns) * (uc - uS) * idyc0;
            const T nzt = T(0.25) * (((nW + nC) + SN[s2][ty][txm]) + SN[s2][ty][tx]), nzb = T(0.25) * (((SN[s0][ty][txm] + SN[s0][ty][tx]) + nW) + nC);
            const T fzt = (nu + nzt) * (uT - uc) * c.ihz, fzb = (nu + nzb) * (uc - uB) * c.ihz;
            const T visc = (fxe - fxw) * c.ihx + (fyn - fys) * idyj + (fzt - fzb) * c.ihz;
            H = -(cx + cy + cz) + visc + T(c.g[0]);
          } else H = -(cx + cy + cz) + nu * (dxx + dyy + dzz) + T(c.g[0]);
          c.us[q] = uc + dt * (a0 * H + a1 * huo);
          c.hu[q] = H;
        }
      }
      // ---- v face (control volume between y_c(j-1) and y_c(j)) ----
      if (i < c.nx && k < c.nz) {
        const size_t q = qv0 + plv * (unsigned)k;
        if (c.by && (j == 0 || j == c.ny)) {
          const int side = j == 0 ? 0 : 1;
          const size_t qi = side ? q - c.nx : q + c.nx;
          c.vs[q] = boundary_normal<T>(c, V, 1, side, i, k, q, qi, side ? c.ny - 1 : 0, (double)dt);
          c.hv[q] = T(0);
        } else {
          const T vE = SV[s1][ty][txp], vW = SV[s1][ty][txm], vN = SV[s1][typ][tx], vS = SV[s1][tym][tx];
          const T wl = wyl0, wh = wyh0;
          const T ue = wl * SU[s1][tym][txp] + wh * SU[s1][ty][txp], ve = transported<T>(upw, ue, vc, vE, T(0.5) * (vc + vE));
          const T uw = wl * SU[s1][tym][tx] + wh * uc,               vw = transported<T>(upw, uw, vW, vc, T(0.5) * (vW + vc));
          const T cx = (ue * ve - uw * vw) * c.ihx;
          const T vnn = T(0.5) * (vc + vN), vss = T(0.5) * (vS + vc);
          const T cy = (vnn * transported<T>(upw, vnn, vc, vN, vnn) - vss * transported<T>(upw, vss, vS, vc, vss)) * idyc0;
          const T wt = wl * SW[s2][tym][tx] + wh * wT, vt = transported<T>(upw, wt, vc, vT, T(0.5) * (vc + vT));
          const T wb = wl * SW[s1][tym][tx] + wh * wc, vb = transported<T>(upw, wb, vB, vc, T(0.5) * (vB + vc));
          const T cz = (wt * vt - wb * vb) * c.ihz;
          const T dxx = (vE - T(2) * vc + vW) * c.ihx2;
          const T dyy = ((vN - vc) * idyj - (vc - vS) * idyjm) * idyc0;
          const T dzz = (vT - T(2) * vc + vB) * c.ihz2;
          T H;
          if (LES) {
            const T nC = SN[s1][ty][tx], nS = SN[s1][tym][tx];
            const T fxe = (nu + T(0.25) * (((nS + SN[s1][tym][txp]) + nC) + SN[s1][ty][txp])) * (vE - vc) * c.ihx;
            const T fxw = (nu + T(0.25) * (((SN[s1][tym][txm] + nS) + SN[s1][ty][txm]) + nC)) * (vc - vW) * c.ihx;
            const T fyn = (nu + nC) * (vN - vc) * idyj, fys = (nu + nS) * (vc - vS) * idyjm;
            const T fzt = (nu + T(0.25) * (((nS + nC) + SN[s2][tym][tx]) + SN[s2][ty][tx])) * (vT - vc) * c.ihz;
            const T fzb = (nu + T(0.25) * (((SN[s0][tym][tx] + SN[s0][ty][tx]) + nS) + nC)) * (vc - vB) * c.ihz;
            const T visc = (fxe - fxw) * c.ihx + (fyn - fys) * idyc0 + (fzt - fzb) * c.ihz;
            H = -(cx + cy + cz) + visc + T(c.g[1]);
          } else H = -(cx + cy + cz) + nu * (dxx + dyy + dzz) + T(c.g[1]);
          c.vs[q] = vc + dt * (a0 * H + a1 * hvo);
          c.hv[q] = H;
        }
      }
      // ---- w face ----
      if (i < c.nx && j < c.ny) {
        const size_t q = qw0 + plw * (unsigned)k;
        if (c.bz && (k == 0 || k == c.nz)) {
          const int side = k == 0 ? 0 : 1;
          const size_t pl = (size_t)c.nx * c.ny;
          const size_t qi = side ? q - pl : q + pl;
          c.ws[q] = boundary_normal<T>(c, W, 2, side, i, j, q, qi, 0, (double)dt);
          c.hw[q] = T(0);
        } else {
          const T wE = SW[s1][ty][txp], wW = SW[s1][ty][txm], wN = SW[s1][typ][tx], wS = SW[s1][tym][tx];
          const T ue = T(0.5) * (SU[s0][ty][txp] + SU[s1][ty][txp]), we = transported<T>(upw, ue, wc, wE, T(0.5) * (wc + wE));
          const T uw = T(0.5) * (uB + uc),                           ww = transported<T>(upw, uw, wW, wc, T(0.5) * (wW + wc));
          const T cx = (ue * we - uw * ww) * c.ihx;
          const T vnn = T(0.5) * (SV[s0][typ][tx] + SV[s1][typ][tx]), wnn = transported<T>(upw, vnn, wc, wN, wyl1 * wc + wyh1 * wN);
          const T vss = T(0.5) * (vB + vc),                           wss = transported<T>(upw, vss, wS, wc, wyl0 * wS + wyh0 * wc);
          const T cy = (vnn * wnn - vss * wss) * idyj;
          const T wt = T(0.5) * (wc + wT), wb = T(0.5) * (wB + wc);
          const T cz = (wt * transported<T>(upw, wt, wc, wT, wt) - wb * transported<T>(upw, wb, wB, wc, wb)) * c.ihz;
          const T dxx = (wE - T(2) * wc + wW) * c.ihx2;
          const T dyy = ((wN - wc) * idyc1 - (wc - wS) * idyc0) * idyj;
          const T dzz = (wT - T(2) * wc + wB) * c.ihz2;
          T H;
          if (LES) {
            const T nC = SN[s1][ty][tx], nB = SN[s0][ty][tx];
            const T fxe = (nu + T(0.25) * (((nB + SN[s0][ty][txp]) + nC) + SN[s1][ty][txp])) * (wE - wc) * c.ihx;
            const T fxw = (nu + T(0.25) * (((SN[s0][ty][txm] + nB) + SN[s1][ty][txm]) + nC)) * (wc - wW) * c.ihx;
            T nn = T(0.25) * (((nB + SN[s0][typ][tx]) + nC) + SN[s1][typ][tx]), ns = T(0.25) * (((SN[s0][tym][tx] + nB) + SN[s1][tym][tx]) + nC);
            if ((wm_lo && j == 0) || (wm_hi && j == c.ny - 1)) {     // Eq. 28 for i = 3: u interpolated to the w face
              const int f = j == 0 ? 2 : 3;
              const double uf = 0.25 * ((((double)uB + (double)SU[s0][ty][txp]) + (double)uc) + (double)SU[s1][ty][txp]);
              const T nw = T(wall_nut((double)wc - c.bcv[f][2], uf - c.bcv[f][0], 0.5 * c.dy64[j], c.nu));
              if (j == 0) ns = nw; else nn = nw;
            }
            const T fyn = (nu + nn) * (wN - wc) * idyc1, fys = (nu + ns) * (wc - wS) * idyc0;
            const T fzt = (nu + nC) * (wT - wc) * c.ihz, fzb = (nu + nB) * (wc - wB) * c.ihz;
            const T visc = (fxe - fxw) * c.ihx + (fyn - fys) * idyj + (fzt - fzb) * c.ihz;
            H = -(cx + cy + cz) + visc + T(c.g[2]);
          } else H = -(cx + cy + cz) + nu * (dxx + dyy + dzz) + T(c.g[2]);
          c.ws[q] = wc + dt * (a0 * H + a1 * hwo);
          c.hw[q] = H;
        }
      }
    }
    uB = uc; uc = uT; vB = vc; vc = vT; wB = wc; wc = wT;
  }
}

template <class T> int launch_momentum(const Ctx<T>& c, const Launch& L) {
  if (momentumv_applies<T>(c)) return launch_momentumv<T>(c, L);
  const int bxn = (c.nxu + kMomTX - 3) / (kMomTX - 2), byn = (c.nyv + kMomTY - 3) / (kMomTY - 2);
  const bool les = c.nu > 0.0 && (c.cs > 0.0 || c.wall_model);
  // z chunks: whole waves of resident CTAs (2 CTAs of 320 threads per SM; the LES variant: 1) while chunks stay >= 16 planes
  const int kz = pick_kz((long long)bxn * byn, c.nzw, (les ? 1LL : 2LL) * 148, 2, 16);
  dim3 b(kMomTX, kMomTY, 1), g(bxn, byn, (c.nzw + kz - 1) / kz);
  const double bytes = 12.0 * sizeof(T) * c.nx * c.ny * c.nz;
  int n = 1;
  const bool adt = c.cfl > 0.0, upw = c.convection == FS_CONV_UPWIND;
  T* nut = nullptr;
  if (les) {
    const long long N = (long long)c.nx * c.ny * c.nz;
    nut = c.q;                           // PCG scratch, free until the Poisson solve of this step
    if (c.cs > 0.0) FS_LAUNCH(L, "eddy_viscosity", 4.0 * sizeof(T) * N, k_eddy_viscosity<T><<<flat_blocks(N), 256, 0, L.s>>>(c, nut));
    else FS_LAUNCH(L, "eddy_viscosity", 1.0 * sizeof(T) * N, cudaMemsetAsync(nut, 0, sizeof(T) * (size_t)N, L.s));
    ++n;
  }
  static const char* names[2][2][2] = {{{"k_momentum<f32,central>", "k_momentum<f32,upwind>"}, {"k_momentum<f32,central,LES>", "k_momentum<f32,upwind,LES>"}},
                                       {{"k_momentum<f64,central>", "k_momentum<f64,upwind>"}, {"k_momentum<f64,central,LES>", "k_momentum<f64,upwind,LES>"}}};
  const double tot = bytes + (les ? sizeof(T) * (double)c.nx * c.ny * c.nz : 0.0);
  FS_LAUNCHI(L, "momentum_predictor", names[sizeof(T) == 8][les][upw], tot, {
    if (les) {
      if (upw) { if (adt) k_momentum<T, true, true, true><<<g, b, 0, L.s>>>(c, kz, nut); else k_momentum<T, true, true, false><<<g, b, 0, L.s>>>(c, kz, nut); }
      else { if (adt) k_momentum<T, false, true, true><<<g, b, 0, L.s>>>(c, kz, nut); else k_momentum<T, false, true, false><<<g, b, 0, L.s>>>(c, kz, nut); }
    } else {
      if (upw) { if (adt) k_momentum<T, true, false, true><<<g, b, 0, L.s>>>(c, kz, nut); else k_momentum<T, true, false, false><<<g, b, 0, L.s>>>(c, kz, nut); }
      else { if (adt) k_momentum<T, false, false, true><<<g, b, 0, L.s>>>(c, kz, nut); else k_momentum<T, false, false, false><<<g, b, 0, L.s>>>(c, kz, nut); }
    }
  });
  return n;
}

// ---------------------------------------------------------------------------------------------------
// O5 outflow flux correction (reading; the paper is silent): the net outward flux Phi through all
// boundary-normal faces is removed by a uniform shift of the outflow faces, u_n(out) -= Phi / A_out.
// ---------------------------------------------------------------------------------------------------
template <class T> struct FaceIt {   // enumerates the boundary-normal faces of the bounded directions
  const Ctx<T>& c;
  __device__ FaceIt(const Ctx<T>& cc) : c(cc) {}
  __device__ long long count() const {
    long long n = 0;
    if (c.bx) n += 2LL * c.ny * c.nz;
    if (c.by) n += 2LL * c.nx * c.nz;
    if (c.bz) n += 2LL * c.nx * c.ny;
    return n;
  }
  // decode face id -> (d, side, a, b); returns the storage index, area, outward sign, and field
  __device__ void decode(long long f, int& d, int& side, size_t& q, double& area, T*& fld) const {
    long long nxf = c.bx ? 2LL * c.ny * c.nz : 0, nyf = c.by ? 2LL * c.nx * c.nz : 0;
    if (f < nxf) {
      d = 0; long long pl = (long long)c.ny * c.nz; side = f >= pl; long long r = f - side * pl;
      int j = (int)(r % c.ny), k = (int)(r / c.ny);
      q = (size_t)(side ? c.nx : 0) + (size_t)c.nxu * ((size_t)j + (size_t)c.ny * k);
      area = c.dy64[j] * c.hz; fld = c.us;
    } else if (f < nxf + nyf) {
      f -= nxf; d = 1; long long pl = (long long)c.nx * c.nz; side = f >= pl; long long r = f - side * pl;
      int i = (int)(r % c.nx), k = (int)(r / c.nx);
      q = (size_t)i + (size_t)c.nx * ((size_t)(side ? c.ny : 0) + (size_t)c.nyv * k);
      area = c.hx * c.hz; fld = c.vs;
    } else {
      f -= nxf + nyf; d = 2; long long pl = (long long)c.nx * c.ny; side = f >= pl; long long r = f - side * pl;
      int i = (int)(r % c.nx), j = (int)(r / c.nx);
      q = (size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * (size_t)(side ? c.nz : 0));
      area = c.hx * c.dy64[j]; fld = c.ws;
    }
  }
};

template <class T> __global__ void __launch_bounds__(256) k_flux_sum(const Ctx<T> c) {
  __shared__ double sh[2 * 32]; __shared__ int flag;
  FaceIt<T> it(c);
  const long long nf = it.count();
  double v[2] = {0.0, 0.0};
  for (long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x; f < nf; f += (long long)gridDim.x * blockDim.x) {
    int d, side; size_t q; double area; T* fld;
    it.decode(f, d, side, q, area, fld);
    const double sgn = side ? 1.0 : -1.0;
    v[0] += sgn * (double)fld[q] * area;
    if (c.bc[2 * d + side] == FS_BC_OUTFLOW_CONVECTIVE) v[1] += area;
  }
  if (grid_sum<2>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0) { c.S->flux_phi = v[0]; c.S->flux_aout = v[1]; }
  }
}
template <class T> __global__ void __launch_bounds__(256) k_flux_apply(const Ctx<T> c) {
  FaceIt<T> it(c);
  const long long nf = it.count();
  const double shift = c.S->flux_phi / c.S->flux_aout;
  for (long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x; f < nf; f += (long long)gridDim.x * blockDim.x) {
    int d, side; size_t q; double area; T* fld;
    it.decode(f, d, side, q, area, fld);
    if (c.bc[2 * d + side] == FS_BC_OUTFLOW_CONVECTIVE) {
      const double sgn = side ? 1.0 : -1.0;
      fld[q] = T((double)fld[q] - sgn * shift);
    }
  }
}
template <class T> int launch_flux_correction(const Ctx<T>& c, const Launch& L) {
  bool any = false;
  for (int f = 0; f < 6; ++f) any |= c.bc[f] == FS_BC_OUTFLOW_CONVECTIVE;
  if (!any) return 0;
  FS_LAUNCH(L, "flux_sum", 0.0, k_flux_sum<T><<<64, 256, 0, L.s>>>(c));
  FS_LAUNCH(L, "flux_apply", 0.0, k_flux_apply<T><<<64, 256, 0, L.s>>>(c));
  return 2;
}

// ---------------------------------------------------------------------------------------------------
// S6: raw right-hand side of the symmetrised system, bhat_raw = -dy_j (rho/dt) D(u*)  (Eq. 7;
// SURVEY O6), and its sum for the compatibility shift.  Written into r; pcg_init finishes the job.
// ---------------------------------------------------------------------------------------------------

template <class T> __global__ void __launch_bounds__(256) k_div_rhs(const Ctx<T> c, const T* __restrict__ bsrc) {
  __shared__ double sh[32]; __shared__ int flag;
  const long long N = (long long)c.nx * c.ny * c.nz;
  const T sc = T(c.rho / c.S->dt);
  double v[1] = {0.0};
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % c.nx); const long long t = q / c.nx; const int j = (int)(t % c.ny), k = (int)(t / c.ny);
    T b;
    if (bsrc) b = bsrc[q];
    else {
      const int ip = c.bx ? i + 1 : (i + 1 == c.nx ? 0 : i + 1);
      const int jp = c.by ? j + 1 : (j + 1 == c.ny ? 0 : j + 1);
      const int kp = c.bz ? k + 1 : (k + 1 == c.nz ? 0 : k + 1);
      const T ue = c.us[(size_t)ip + (size_t)c.nxu * ((size_t)j + (size_t)c.ny * k)], uw = c.us[(size_t)i + (size_t)c.nxu * ((size_t)j + (size_t)c.ny * k)];
      const T vn = c.vs[(size_t)i + (size_t)c.nx * ((size_t)jp + (size_t)c.nyv * k)], vs = c.vs[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.nyv * k)];
      const T wt = c.ws[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * kp)], wb = c.ws[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * k)];
      const T div = (ue - uw) * c.ihx + (vn - vs) * c.idy[j + 1] + (wt - wb) * c.ihz;
      b = div * sc;
    }
    const T bh = -c.dy[j + 1] * b;
    c.r[q] = bh;
    v[0] += (double)bh;
  }
  if (grid_sum<1>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0) {
      c.S->mean_coef = v[0] / c.S->sum_dy;
      c.S->max_div = 0.0; c.S->nan_flag = 0; c.S->true_rr = 0.0;
    }
  }
}
// Same pass for grids periodic in x with nx a multiple of the vector width: one 16-byte vector of cells per
// thread, 32 x 8 threads per CTA marching a z chunk (the top w face of one plane is the bottom of the next),
// no integer division.
template <class T> __global__ void __launch_bounds__(256) k_div_rhsv(const Ctx<T> c, int kz) {
  constexpr int VX = Vec16<T>::VX;
  using W = Vec16<T>;
  __shared__ double sh[32]; __shared__ int flag;
  const int gx = (blockIdx.x * 32 + threadIdx.x) * VX, gy = blockIdx.y * 8 + threadIdx.y;
  const bool valid = gx < c.nx && gy < c.ny;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  double sum = 0.0;
  if (valid) {
    const int jp = c.by ? gy + 1 : (gy + 1 == c.ny ? 0 : gy + 1);
    const int xe = gx + VX == c.nx ? 0 : gx + VX;
    const unsigned plc = (unsigned)c.nx * c.ny, plv = (unsigned)c.nx * c.nyv;
    const unsigned oc = (unsigned)gx + (unsigned)c.nx * gy, oe = (unsigned)xe + (unsigned)c.nx * gy;
    const unsigned ov = (unsigned)gx + (unsigned)c.nx * gy, ovp = (unsigned)gx + (unsigned)c.nx * jp;
    const T ihx = c.ihx, ihz = c.ihz, idy = c.idy[gy + 1], sc = T(c.rho / c.S->dt), mdy = -c.dy[gy + 1];
    W wb = ld16<T>(c.ws + (oc + plc * (unsigned)k0));
#pragma unroll 2
    for (int k = k0; k < k1; ++k) {
      const int kp = c.bz ? k + 1 : (k + 1 == c.nz ? 0 : k + 1);
      const W u = ld16<T>(c.us + (oc + plc * (unsigned)k));
      const T uE = c.us[oe + plc * (unsigned)k];
      const W vs = ld16<T>(c.vs + (ov + plv * (unsigned)k)), vn = ld16<T>(c.vs + (ovp + plv * (unsigned)k));
      const W wt = ld16<T>(c.ws + (oc + plc * (unsigned)kp));
      W r;
      T s = T(0);
#pragma unroll
      for (int a = 0; a < VX; ++a) {
        const T ue = a < VX - 1 ? u.a[a < VX - 1 ? a + 1 : a] : uE;
        const T div = (ue - u.a[a]) * ihx + (vn.a[a] - vs.a[a]) * idy + (wt.a[a] - wb.a[a]) * ihz;
        r.a[a] = mdy * (div * sc);
        s += r.a[a];
      }
      st16<T>(c.r + (oc + plc * (unsigned)k), r);
      sum += (double)s;
      wb = wt;
    }
  }
  double v[1] = {sum};
  if (grid_sum<1>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0 && threadIdx.y == 0) {
      c.S->mean_coef = v[0] / c.S->sum_dy;
      c.S->max_div = 0.0; c.S->nan_flag = 0; c.S->true_rr = 0.0;
    }
  }
}

template <class T> int launch_div_rhs(const Ctx<T>& c, const Launch& L) {
  const long long N = (long long)c.nx * c.ny * c.nz;
  if (!c.bx && c.nx % Vec16<T>::VX == 0) {
    const int bxn = (c.nx + 32 * Vec16<T>::VX - 1) / (32 * Vec16<T>::VX), byn = (c.ny + 7) / 8;
    int kz = c.nz;
    while (kz > 16 && (long long)bxn * byn * ((c.nz + kz - 1) / kz) < 8LL * 148 * 8) kz = (kz + 1) / 2;
    while ((long long)bxn * byn * ((c.nz + kz - 1) / kz) > kMaxPartials) kz *= 2;
    FS_LAUNCHI(L, "div_rhs", sizeof(T) == 8 ? "k_div_rhsv<f64>" : "k_div_rhsv<f32>", 4.0 * sizeof(T) * N, k_div_rhsv<T><<<dim3(bxn, byn, (c.nz + kz - 1) / kz), dim3(32, 8), 0, L.s>>>(c, kz));
    return 1;
  }
  FS_LAUNCHI(L, "div_rhs", sizeof(T) == 8 ? "k_div_rhs<f64>" : "k_div_rhs<f32>", 4.0 * sizeof(T) * N, k_div_rhs<T><<<flat_blocks(N), 256, 0, L.s>>>(c, nullptr));
  return 1;
}
template <class T> int launch_rhs_from_b(const Ctx<T>& c, const T* b, const Launch& L) {
  const long long N = (long long)c.nx * c.ny * c.nz;
  FS_LAUNCH(L, "div_rhs", 2.0 * sizeof(T) * N, k_div_rhs<T><<<flat_blocks(N), 256, 0, L.s>>>(c, b));
  return 1;
}

// plain staggered divergence of (u,v,w) (FS_DIV on demand)
template <class T> __global__ void __launch_bounds__(256) k_divergence(const Ctx<T> c, const T* __restrict__ u, const T* __restrict__ v,
                                                                     const T* __restrict__ w, T* __restrict__ out) {
  const long long N = (long long)c.nx * c.ny * c.nz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < N; q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % c.nx); const long long t = q / c.nx; const int j = (int)(t % c.ny), k = (int)(t / c.ny);
    const int ip = c.bx ? i + 1 : (i + 1 == c.nx ? 0 : i + 1);
    const int jp = c.by ? j + 1 : (j + 1 == c.ny ? 0 : j + 1);
    const int kp = c.bz ? k + 1 : (k + 1 == c.nz ? 0 : k + 1);
    const T ue = u[(size_t)ip + (size_t)c.nxu * ((size_t)j + (size_t)c.ny * k)], uw = u[(size_t)i + (size_t)c.nxu * ((size_t)j + (size_t)c.ny * k)];
    const T vn = v[(size_t)i + (size_t)c.nx * ((size_t)jp + (size_t)c.nyv * k)], vs = v[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.nyv * k)];
    const T wt = w[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * kp)], wb = w[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * k)];
    out[q] = (ue - uw) * c.ihx + (vn - vs) * c.idy[j + 1] + (wt - wb) * c.ihz;
  }
}
template <class T> int launch_divergence(const Ctx<T>& c, const T* u, const T* v, const T* w, T* out, const Launch& L) {
  const long long N = (long long)c.nx * c.ny * c.nz;
  FS_LAUNCH(L, "divergence", 4.0 * sizeof(T) * N, k_divergence<T><<<flat_blocks(N), 256, 0, L.s>>>(c, u, v, w, out));
  return 1;
}

// ---------------------------------------------------------------------------------------------------
// S8: projection u^{n+1} = u* - (dt/rho) G p at non-boundary faces (Eq. 6/10, L114, L131), fused with
// the diagnostics of the projected field: max |D u^{n+1}|, NaN flag, and the true Poisson residual
// (since D G = L:  bhat - A p = -dy_j (rho/dt) D u^{n+1} - mean_coef dy_j).
// One thread per cell of the extended box.
// ---------------------------------------------------------------------------------------------------
template <class T> __device__ __forceinline__ T proj_u(const Ctx<T>& c, int i, int j, int k, T dtr) {
  const size_t q = (size_t)i + (size_t)c.nxu * ((size_t)j + (size_t)c.ny * k);
  if (c.bx && (i == 0 || i == c.nx)) return c.us[q];
  const int im = i == 0 ? c.nx - 1 : i - 1;
  const size_t row = (size_t)c.nx * ((size_t)j + (size_t)c.ny * k);
  return c.us[q] - dtr * ((c.p[row + i] - c.p[row + im]) * c.ihx);
}
template <class T> __device__ __forceinline__ T proj_v(const Ctx<T>& c, int i, int j, int k, T dtr) {
  const size_t q = (size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.nyv * k);
  if (c.by && (j == 0 || j == c.ny)) return c.vs[q];
  const int jm = j == 0 ? c.ny - 1 : j - 1;
  return c.vs[q] - dtr * ((c.p[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * k)] -
                           c.p[(size_t)i + (size_t)c.nx * ((size_t)jm + (size_t)c.ny * k)]) * c.idyc[j]);
}
template <class T> __device__ __forceinline__ T proj_w(const Ctx<T>& c, int i, int j, int k, T dtr) {
  const size_t q = (size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * k);
  if (c.bz && (k == 0 || k == c.nz)) return c.ws[q];
  const int km = k == 0 ? c.nz - 1 : k - 1;
  return c.ws[q] - dtr * ((c.p[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * k)] -
                           c.p[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * km)]) * c.ihz);
}

template <class T> __global__ void __launch_bounds__(256) k_project(const Ctx<T> c, int kz) {
  __shared__ double sh[32]; __shared__ int flag;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k0 = blockIdx.z * kz;
  const T dtr = T(c.S->dt / c.rho);
  const double sc = c.rho / c.S->dt, mc = c.S->mean_coef;
  double v[1] = {0.0}; double md = 0.0; int nan = 0;
  if (i < c.nxu && j < c.nyv) {
    const int k1 = min(k0 + kz, c.nzw);
    for (int k = k0; k < k1; ++k) {
      T un = T(0), vn = T(0), wn = T(0);
      if (j < c.ny && k < c.nz) { un = proj_u<T>(c, i, j, k, dtr); c.u[(size_t)i + (size_t)c.nxu * ((size_t)j + (size_t)c.ny * k)] = un; }
      if (i < c.nx && k < c.nz) { vn = proj_v<T>(c, i, j, k, dtr); c.v[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.nyv * k)] = vn; }
      if (i < c.nx && j < c.ny) { wn = proj_w<T>(c, i, j, k, dtr); c.w[(size_t)i + (size_t)c.nx * ((size_t)j + (size_t)c.ny * k)] = wn; }
      if (i < c.nx && j < c.ny && k < c.nz) {
        const T ue = proj_u<T>(c, c.bx ? i + 1 : (i + 1 == c.nx ? 0 : i + 1), j, k, dtr);
        const T vt = proj_v<T>(c, i, c.by ? j + 1 : (j + 1 == c.ny ? 0 : j + 1), k, dtr);
        const T wt = proj_w<T>(c, i, j, c.bz ? k + 1 : (k + 1 == c.nz ? 0 : k + 1), dtr);
        const T div = (ue - un) * c.ihx + (vt - vn) * c.idy[j + 1] + (wt - wn) * c.ihz;
        const double a = fabs((double)div);
        if (a != a) nan = 1;
        md = fmax(md, a);
        const double dyj = c.dy64[j];
        const double e = -dyj * sc * (double)div - mc * dyj;
        v[0] += e * e;
      }
    }
  }
  // max and NaN flag are order-independent: plain atomics keep them deterministic
  md = warp_max(md);
  nan = __any_sync(0xffffffffu, nan);
  if (((threadIdx.x + blockDim.x * threadIdx.y) & 31) == 0) {
    if (md > 0.0) atomicMax((unsigned long long*)&c.S->max_div, (unsigned long long)__double_as_longlong(md));
    if (nan) atomicOr(&c.S->nan_flag, 1);
  }
  if (grid_sum<1>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (threadIdx.x == 0 && threadIdx.y == 0) c.S->true_rr = v[0];
  }
}

// Same pass for grids that are periodic in x with nx a multiple of the vector width: 2.5-D streaming kernel,
// one 16-byte vector of cells per thread, 32 VX x TY extended tile -> 30 VX x (TY - 2) results, z march.  A thread
// projects its own u, v, w faces of plane k (p of the west / south neighbours through a shared plane, p of
// the plane below from a register) and publishes the projected u, v in shared memory; the divergence of
// plane k-1 is formed one plane later from the east / north neighbours' projected faces of that plane and
// the w faces of planes k-1 and k.  Raw loads stay in flight for two planes.
// rows of the extended tile: 12 in fp32 (80 registers), 8 in fp64 (114 registers, no spills)
template <class T> struct PjTile { static constexpr int TY = sizeof(T) == 4 ? 12 : 8; };

template <class T> __global__ void __launch_bounds__(32 * PjTile<T>::TY, 2) k_projectv(const Ctx<T> c, int kz, const __grid_constant__ TmapSet tm) {
  constexpr int kPjTY = PjTile<T>::TY;
  constexpr int VX = Vec16<T>::VX, ROWE = 32 * VX, PLN = kPjTY * ROWE;
  using W = Vec16<T>;
  __shared__ __align__(16) T SP[2 * PLN], SU[2 * PLN], SV[2 * PLN];
  __shared__ double sh[32]; __shared__ int flag;
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = (blockIdx.x * 30 - 1 + lane) * VX, gy = blockIdx.y * (kPjTY - 2) - 1 + ty;
  const int sx = wrapi(gx, c.nx);
  const int syc = c.by ? min(max(gy, 0), c.ny - 1) : wrapi(gy, c.ny);      // row of cell-shaped arrays
  const int syv = c.by ? min(max(gy, 0), c.ny) : wrapi(gy, c.ny);          // row of v
  const bool own = lane >= 1 && lane <= 30 && ty >= 1 && ty <= kPjTY - 2 && gx < c.nx && gy < c.nyv;
  const bool rowc = gy < c.ny;                                            // the row has cells / u / w faces
  const bool vbnd = c.by && (gy <= 0 || gy >= c.ny);                       // v face on a wall: not projected
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nzw);
  const unsigned plc = (unsigned)c.nx * c.ny, plv = (unsigned)c.nx * c.nyv;
  const unsigned rowc_o = (unsigned)sx + (unsigned)c.nx * syc, rowv_o = (unsigned)sx + (unsigned)c.nx * syv;
  const T dtr = T(c.S->dt / c.rho), ihx = c.ihx, ihz = c.ihz;
  const T idycj = c.idyc[syv], idyj = c.idy[syc + 1];
  const double sc = c.rho / c.S->dt, mc = c.S->mean_coef, dyj = c.dy64[syc];
  const int o_own = ty * ROWE + lane * VX;
  const int o_s = (ty > 0 ? ty - 1 : 0) * ROWE + lane * VX, o_n = (ty < kPjTY - 1 ? ty + 1 : ty) * ROWE + lane * VX;
  const int o_w = ty * ROWE + (lane > 0 ? lane * VX - 1 : 0), o_e = ty * ROWE + (lane < 31 ? lane * VX + VX : 32 * VX - 1);
  auto kcell = [&](int k) { return c.bz ? min(max(k, 0), c.nz - 1) : (k < 0 ? k + c.nz : (k >= c.nz ? k - c.nz : k)); };
  auto kwf = [&](int k) { return c.bz ? min(max(k, 0), c.nz) : (k < 0 ? k + c.nz : (k >= c.nz ? k - c.nz : k)); };
  struct Raw { W p, us, vs, ws; };
  auto fetch = [&](int k, Raw& r) {
    const unsigned kc = (unsigned)kcell(k);
    r.p = ld16<T>(c.p + (rowc_o + plc * kc));
    r.us = ld16<T>(c.us + (rowc_o + plc * kc));
    r.vs = ld16<T>(c.vs + (rowv_o + plv * kc));
    r.ws = ld16<T>(c.ws + (rowc_o + plc * (unsigned)kwf(k)));
  };
  // tile planes of p, u*, v*, w* go to L2 kPfAhead planes before the register loads ask for them (one TMA prefetch per field
  // and plane, issued by one thread; the loads then have L2 latency, which the two planes in flight cover)
  const bool pf_on = tm.n > 0 && lane == 0 && ty == 0;
  const int pf_x = (blockIdx.x * 30 - 1) * VX, pf_y = blockIdx.y * (kPjTY - 2) - 1;
  auto prefetch = [&](int k) {
    if (!pf_on || k > k1) return;
    const int kc = kcell(k), kw = kwf(k);
    tma_prefetch_plane(tm.m[0], pf_x, pf_y, kc); tma_prefetch_plane(tm.m[1], pf_x, pf_y, kc);
    tma_prefetch_plane(tm.m[2], pf_x, pf_y, kc); tma_prefetch_plane(tm.m[3], pf_x, pf_y, kw);
  };
  for (int k = k0 + 2; k < k0 + 2 + kPfAhead; ++k) prefetch(k);
  Raw r0, r1;
  W pB = ld16<T>(c.p + (rowc_o + plc * (unsigned)kcell(k0 - 1)));
  fetch(k0, r0);
  fetch(k0 + 1, r1);
  W wnP;                                    // projected w faces of plane k-1
#pragma unroll
  for (int a = 0; a < VX; ++a) wnP.a[a] = T(0);
  double ss = 0.0, md = 0.0; int nan = 0;
  int b = 0;
  // one plane; r holds its raw loads and is refilled with plane k+2 at the end (the two Raw buffers alternate)
  auto body = [&](int k, Raw& r) {
    st16<T>(SP + b + o_own, r.p);
    __syncthreads();
    const W pS = ld16<T>(SP + b + o_s);
    const T pW0 = SP[b + o_w];
    const bool wbnd = c.bz && (k == 0 || k >= c.nz);
    W un, vn, wn;
#pragma unroll
    for (int a = 0; a < VX; ++a) {
      const T pc = r.p.a[a], pw = a > 0 ? r.p.a[a > 0 ? a - 1 : 0] : pW0;
      un.a[a] = r.us.a[a] - dtr * ((pc - pw) * ihx);
      vn.a[a] = vbnd ? r.vs.a[a] : r.vs.a[a] - dtr * ((pc - pS.a[a]) * idycj);
      wn.a[a] = wbnd ? r.ws.a[a] : r.ws.a[a] - dtr * ((pc - pB.a[a]) * ihz);
    }
    if (own && k < k1) {
      if (rowc && k < c.nz) st16<T>(c.u + (rowc_o + plc * (unsigned)k), un);
      if (k < c.nz) st16<T>(c.v + (rowv_o + plv * (unsigned)k), vn);
      if (rowc) st16<T>(c.w + (rowc_o + plc * (unsigned)k), wn);
    }
    // divergence of plane k-1 (its projected u, v faces were published one iteration ago)
    if (k > k0 && own && rowc && k - 1 < c.nz) {
      const int pb = PLN - b;
      const W vN = ld16<T>(SV + pb + o_n), vO = ld16<T>(SV + pb + o_own), uO = ld16<T>(SU + pb + o_own);
      const T uE0 = SU[pb + o_e];
#pragma unroll
      for (int a = 0; a < VX; ++a) {
        const T ue = a < VX - 1 ? uO.a[a < VX - 1 ? a + 1 : a] : uE0;
        const T div = (ue - uO.a[a]) * ihx + (vN.a[a] - vO.a[a]) * idyj + (wn.a[a] - wnP.a[a]) * ihz;
        const double ad = fabs((double)div);
        if (ad != ad) nan = 1;
        md = fmax(md, ad);
        const double e = -dyj * sc * (double)div - mc * dyj;
        ss += e * e;
      }
    }
    st16<T>(SU + b + o_own, un); st16<T>(SV + b + o_own, vn);
    wnP = wn; pB = r.p;
    prefetch(k + 2 + kPfAhead);
    if (k + 2 <= k1) fetch(k + 2, r);
    b = PLN - b;
  };
  for (int k = k0;;) {
    body(k, r0); if (++k > k1) break;
    body(k, r1); if (++k > k1) break;
  }
  md = warp_max(md);
  nan = __any_sync(0xffffffffu, nan);
  if (lane == 0) {
    if (md > 0.0) atomicMax((unsigned long long*)&c.S->max_div, (unsigned long long)__double_as_longlong(md));
    if (nan) atomicOr(&c.S->nan_flag, 1);
  }
  double v[1] = {ss};
  if (grid_sum<1>(v, c.partials, &c.S->ticket[0], sh, &flag)) {
    if (lane == 0 && ty == 0) c.S->true_rr = v[0];
  }
}

struct ColGeom { dim3 grid, block; int kz; };
ColGeom col_geom(int nx, int ny, int nz);
ColGeom col_geom(int nx, int ny, int nz) {
  ColGeom g;
  const int tx = nx >= 64 ? 64 : 32, ty = 256 / tx;
  g.block = dim3(tx, ty, 1);
  const int bxn = (nx + tx - 1) / tx, byn = (ny + ty - 1) / ty;
  // z chunk: aim at >= 4 waves of 148 blocks but keep chunks >= 8 planes and partials <= kMaxPartials
  int kz = nz;
  while (kz > 8 && (long long)bxn * byn * ((nz + kz - 1) / kz) < 4 * 148) kz = (kz + 1) / 2;
  while ((long long)bxn * byn * ((nz + kz - 1) / kz) > kMaxPartials) kz *= 2;
  g.kz = kz;
  g.grid = dim3(bxn, byn, (nz + kz - 1) / kz);
  return g;
}

template <class T> int launch_project(const Ctx<T>& c, const Launch& L) {
  if (!c.bx && c.nx % Vec16<T>::VX == 0) {
    const int bxn = (c.nx + 30 * Vec16<T>::VX - 1) / (30 * Vec16<T>::VX), byn = (c.nyv + PjTile<T>::TY - 3) / (PjTile<T>::TY - 2);
    const int kz = pick_kz((long long)bxn * byn, c.nzw, 2LL * 148, 1, 16);
    TmapSet tm; memset(&tm, 0, sizeof tm);
    const int bw = 32 * Vec16<T>::VX, bh = PjTile<T>::TY;
    static const int pf = tune_pf();
    if (pf && tmap_encode(&tm.m[0], c.p, sizeof(T), c.nx, c.ny, c.nz, bw, bh) && tmap_encode(&tm.m[1], c.us, sizeof(T), c.nx, c.ny, c.nz, bw, bh) &&
        tmap_encode(&tm.m[2], c.vs, sizeof(T), c.nx, c.nyv, c.nz, bw, bh) && tmap_encode(&tm.m[3], c.ws, sizeof(T), c.nx, c.ny, c.nzw, bw, bh)) tm.n = 4;
    FS_LAUNCHI(L, "project", sizeof(T) == 8 ? "k_projectv<f64>" : "k_projectv<f32>", 7.0 * sizeof(T) * c.nx * c.ny * c.nz,
              k_projectv<T><<<dim3(bxn, byn, (c.nzw + kz - 1) / kz), dim3(32, PjTile<T>::TY), 0, L.s>>>(c, kz, tm));
    return 1;
  }
  ColGeom g = col_geom(c.nxu, c.nyv, c.nzw);
  FS_LAUNCHI(L, "project", sizeof(T) == 8 ? "k_project<f64>" : "k_project<f32>", 7.0 * sizeof(T) * c.nx * c.ny * c.nz, k_project<T><<<g.grid, g.block, 0, L.s>>>(c, g.kz));
  return 1;
}

// ---------------------------------------------------------------------------------------------------
// S9 + S10: rigid-body oscillator m w'' + c w' + k w = F (Eq. 12) advanced by one classical
// RK4 step with the force frozen over the step (weak coupling, L212); markers translate with the body;
// AB2 history flag and step counter.  One block.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double body_acc(double F, double cc, double kk, double m, double a, double b) { return (F - cc * b - kk * a) / m; }

template <class T> __global__ void k_step_end(const Ctx<T> c, const IbmCtx ib) {
  __shared__ double dw[3], nv[3];
  Scalars* S = c.S;
  if (threadIdx.x == 0) {
    for (int a = 0; a < 3; ++a) { dw[a] = 0.0; nv[a] = S->body_vel[a]; }
    if (ib.has_body) {
      const double dt = S->dt, m = ib.bm, cc = ib.bc, kk = ib.bk;
      for (int a = 0; a < 3; ++a) if (ib.dof & (1 << a)) {
        // strong coupling: every sweep advances the structure from time level n; the markers reflect the previous iterate
        const double F = S->body_force[a], y0 = ib.strong ? S->body_disp0[a] : S->body_disp[a], y1 = ib.strong ? S->body_vel0[a] : S->body_vel[a];
        const double k1a = y1,                  k1b = body_acc(F, cc, kk, m, y0, y1);
        const double k2a = y1 + 0.5 * dt * k1b, k2b = body_acc(F, cc, kk, m, y0 + 0.5 * dt * k1a, y1 + 0.5 * dt * k1b);
        const double k3a = y1 + 0.5 * dt * k2b, k3b = body_acc(F, cc, kk, m, y0 + 0.5 * dt * k2a, y1 + 0.5 * dt * k2b);
        const double k4a = y1 + dt * k3b,       k4b = body_acc(F, cc, kk, m, y0 + dt * k3a, y1 + dt * k3b);
        const double w1 = y0 + dt / 6.0 * (k1a + 2.0 * k2a + 2.0 * k3a + k4a);
        const double v1 = y1 + dt / 6.0 * (k1b + 2.0 * k2b + 2.0 * k3b + k4b);
        dw[a] = w1 - S->body_disp[a]; nv[a] = v1;
        S->body_disp[a] = w1; S->body_vel[a] = v1;
      }
    }
    if (c.time_scheme == FS_TIME_RK3) {     // what the step reports: sums over the three stage solves
      S->iter = S->iter_acc; S->converged = S->conv_acc; S->body_runs = S->body_acc;
    }
    S->dt_prev = S->dt; S->time += S->dt;
    S->have_hist = 1; S->step += 1; S->total_iters += S->iter; S->total_body += S->body_runs;
    S->unconverged_steps += S->converged ? 0 : 1; S->nan_steps += S->nan_flag ? 1 : 0;
  }
  __syncthreads();
  if (ib.has_body) {
    for (int l = threadIdx.x; l < ib.n; l += blockDim.x)
      for (int a = 0; a < 3; ++a) {
        if (ib.dof & (1 << a)) ib.X[3 * l + a] = __dadd_rn(ib.X[3 * l + a], dw[a]);
        ib.Ub[3 * l + a] = nv[a];
      }
  }
}
template <class T> int launch_step_end(const Ctx<T>& c, const IbmCtx& ib, const Launch& L) {
  FS_LAUNCH(L, "step_end", 0.0, k_step_end<T><<<1, 256, 0, L.s>>>(c, ib));
  return 1;
}

// ---------------------------------------------------------------------------------------------------
// Step begin.  CFL-adaptive step size (reading N3-2): dt = min(dt_max, cfl h_min / max|u, v, w|) over all
// stored faces of the field at time level n; the maximum is order independent (atomicMax on the bit pattern of a
// non-negative double), the last CTA turns it into S->dt.  Runge-Kutta: u^n is kept for the stage combinations.
// ---------------------------------------------------------------------------------------------------
template <class T> __global__ void __launch_bounds__(256) k_dt_begin(const Ctx<T> c) {
  __shared__ int last;
  const long long nU = (long long)c.nxu * c.ny * c.nz, nV = (long long)c.nx * c.nyv * c.nz, nW = (long long)c.nx * c.ny * c.nzw;
  double m = 0.0;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < nU + nV + nW; q += (long long)gridDim.x * blockDim.x) {
    const T x = q < nU ? c.u[q] : (q < nU + nV ? c.v[q - nU] : c.w[q - nU - nV]);
    m = fmax(m, fabs((double)x));
  }
  m = warp_max(m);
  if ((threadIdx.x & 31) == 0 && m > 0.0) atomicMax((unsigned long long*)&c.S->umax, (unsigned long long)__double_as_longlong(m));
  __syncthreads();
  if (threadIdx.x == 0) { __threadfence(); last = atomicAdd(&c.S->ticket[1], 1u) == gridDim.x - 1; }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    const double um = __longlong_as_double((long long)atomicAdd((unsigned long long*)&c.S->umax, 0ULL));
    c.S->dt = um > 0.0 ? fmin(c.dt, c.cfl * c.hmin / um) : c.dt;
    c.S->umax = 0.0; c.S->ticket[1] = 0u;
  }
}
template <class T> __global__ void k_rk_begin(const Ctx<T> c) { c.S->iter_acc = 0; c.S->conv_acc = 1; c.S->body_acc = 0; }
template <class T> int launch_step_begin(const Ctx<T>& c, const Launch& L) {
  int n = 0;
  if (c.cfl > 0.0) {
    const long long N = (long long)c.nxu * c.ny * c.nz + (long long)c.nx * c.nyv * c.nz + (long long)c.nx * c.ny * c.nzw;
    FS_LAUNCH(L, "dt_cfl", 3.0 * sizeof(T) * c.nx * c.ny * c.nz, k_dt_begin<T><<<flat_blocks(N), 256, 0, L.s>>>(c)); ++n;
  }
  if (c.time_scheme == FS_TIME_RK3) {
    FS_LAUNCH(L, "rk_save", 6.0 * sizeof(T) * c.nx * c.ny * c.nz, {
      k_rk_begin<T><<<1, 1, 0, L.s>>>(c);
      cudaMemcpyAsync(c.q0u, c.u, sizeof(T) * (size_t)c.nxu * c.ny * c.nz, cudaMemcpyDeviceToDevice, L.s);
      cudaMemcpyAsync(c.q0v, c.v, sizeof(T) * (size_t)c.nx * c.nyv * c.nz, cudaMemcpyDeviceToDevice, L.s);
      cudaMemcpyAsync(c.q0w, c.w, sizeof(T) * (size_t)c.nx * c.ny * c.nzw, cudaMemcpyDeviceToDevice, L.s);
    });
    n += 4;
  }
  return n;
}
// Runge-Kutta stage end: u <- c0 u^n + c1 u (stages 1, 2; Shu-Osher weights 3/4, 1/4 and 1/3, 2/3), and the per-step sums
template <class T> __global__ void __launch_bounds__(256) k_rk_combine(const Ctx<T> c, T c0, T c1, int combine) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    Scalars* S = c.S;
    S->iter_acc += S->iter; S->conv_acc = S->conv_acc && S->converged; S->body_acc += S->body_runs;
  }
  if (!combine) return;
  const long long nU = (long long)c.nxu * c.ny * c.nz, nV = (long long)c.nx * c.nyv * c.nz, nW = (long long)c.nx * c.ny * c.nzw;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < nU + nV + nW; q += (long long)gridDim.x * blockDim.x) {
    if (q < nU) c.u[q] = c0 * c.q0u[q] + c1 * c.u[q];
    else if (q < nU + nV) c.v[q - nU] = c0 * c.q0v[q - nU] + c1 * c.v[q - nU];
    else c.w[q - nU - nV] = c0 * c.q0w[q - nU - nV] + c1 * c.w[q - nU - nV];
  }
}
template <class T> int launch_stage_end(const Ctx<T>& c, int stage, const Launch& L) {
  const double c0[3] = {0.0, 0.75, 1.0 / 3.0}, c1[3] = {1.0, 0.25, 2.0 / 3.0};
  const long long N = (long long)c.nxu * c.ny * c.nz + (long long)c.nx * c.nyv * c.nz + (long long)c.nx * c.ny * c.nzw;
  FS_LAUNCH(L, "rk_combine", (stage > 0 ? 9.0 : 0.0) * sizeof(T) * c.nx * c.ny * c.nz,
            k_rk_combine<T><<<stage > 0 ? flat_blocks(N) : 1, 256, 0, L.s>>>(c, T(c0[stage]), T(c1[stage]), stage > 0));
  return 1;
}

// ---------------------------------------------------------------------------------------------------
// dtype conversion / constant shift helpers for fs_fields_set / fs_fields_get
// ---------------------------------------------------------------------------------------------------
template <class TS, class TD> __global__ void k_convert(const TS* __restrict__ s, TD* __restrict__ d, long long n) {
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x) d[q] = (TD)s[q];
}
template <class TS, class TD> void launch_convert(const TS* src, TD* dst, long long n, cudaStream_t s) {
  if (n <= 0) return;
  k_convert<TS, TD><<<flat_blocks(n), 256, 0, s>>>(src, dst, n);
}
template <class T> __global__ void k_scale(T* __restrict__ x, T a, long long n) {
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x) x[q] *= a;
}
template <class T> void launch_scale(T* x, double a, long long n, cudaStream_t s) {
  if (n <= 0) return;
  k_scale<T><<<flat_blocks(n), 256, 0, s>>>(x, (T)a, n);
}

#define INST(T)                                                                                        \
  template int launch_momentum<T>(const Ctx<T>&, const Launch&);                                       \
  template int launch_flux_correction<T>(const Ctx<T>&, const Launch&);                                \
  template int launch_div_rhs<T>(const Ctx<T>&, const Launch&);                                        \
  template int launch_rhs_from_b<T>(const Ctx<T>&, const T*, const Launch&);                           \
  template int launch_project<T>(const Ctx<T>&, const Launch&);                                        \
  template int launch_divergence<T>(const Ctx<T>&, const T*, const T*, const T*, T*, const Launch&);   \
  template int launch_step_end<T>(const Ctx<T>&, const IbmCtx&, const Launch&);                        \
  template int launch_step_begin<T>(const Ctx<T>&, const Launch&);                                     \
  template int launch_stage_end<T>(const Ctx<T>&, int, const Launch&);                                 \
  template void launch_scale<T>(T*, double, long long, cudaStream_t);
INST(float)
INST(double)
template void launch_convert<float, double>(const float*, double*, long long, cudaStream_t);
template void launch_convert<double, float>(const double*, float*, long long, cudaStream_t);
template void launch_convert<float, float>(const float*, float*, long long, cudaStream_t);
template void launch_convert<double, double>(const double*, double*, long long, cudaStream_t);

}  // namespace fs
