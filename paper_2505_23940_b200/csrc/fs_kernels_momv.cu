// fs_kernels_momv.cu -- S0 + S1 for grids that are periodic in x with nx a multiple of the vector width: the
// momentum right-hand side H^n = -div(u u) + nu lap(u) + g (Eq. 4) and the explicit predictor
// u~ = u^n + dt (a0 H^n + a1 H^{n-1}), one 16-byte vector of x-adjacent faces per thread (2 fp64 / 4 fp32).
//
// Same 2.5-D scheme as k_momentum (fs_kernels_fluid.cu): a CTA owns an xy tile, marches in z, keeps the planes k-1,
// k, k+1 of u, v, w in a four-slot ring of shared-memory planes (the fourth slot takes plane k+2 without a second
// barrier) and its own column in a register queue; y / z ghosts (walls) are resolved when a value enters shared
// memory.  What changes is the work per thread: a vector of cells shares the y / z neighbours' loads (16-byte
// shared-memory reads), takes its x neighbours from its own registers except for one scalar per side, shares the
// index arithmetic and predicates, and reads / writes global memory in 16-byte pieces: 18 shared-memory loads per
// 2 (4) cells instead of 36 per cell, 32 VX x 16 extended tile -> 30 VX x 14 results (82 % instead of 75 %).
// The arithmetic per face is that of k_momentum, operation for operation (same parity route against the oracle).
// fp64 feeds the ring with cp.async (ASY): no register holds a load in flight, ghosts are fixed in place after arrival.
// Boundary types: x periodic; y and z periodic, no-slip or slip (inflow / outflow faces, the LES closures and odd
// sizes go through k_momentum).
#include "fs_internal.cuh"
#include <cstring>
#include <cstdlib>

namespace fs {


template <class T> __device__ __forceinline__ T mv_tr(bool upwind, T a, T minus, T plus, T central) {
  return upwind ? (a > T(0) ? minus : plus) : central;
}

// column of component C for a thread whose vector starts at cell sx (in range: x is periodic) in row j (may be one
// row outside: wall ghost = A f + B with the mirrored row, periodic: wrapped)
template <class T> struct MvCol { unsigned off, pl; T A, B; };
template <class T, int C> __device__ __forceinline__ MvCol<T> mv_col(const Ctx<T>& c, int sx, int j) {
  T A = T(1), B = T(0);
  if (!c.by) j = wrapi(j, c.ny);
  else if (C != 1) {
    int face = -1;
    if (j < 0) { face = 2; j = -1 - j; } else if (j >= c.ny) { face = 3; j = 2 * c.ny - 1 - j; }
    if (face >= 0 && c.bc[face] == FS_BC_NOSLIP) { B = T(2.0 * c.bcv[face][C]); A = T(-1); }
  } else j = min(max(j, 0), c.ny);
  const int ey = C == 1 ? c.nyv : c.ny;
  MvCol<T> r;
  r.off = (unsigned)sx + (unsigned)c.nx * (unsigned)j; r.pl = (unsigned)c.nx * (unsigned)ey; r.A = A; r.B = B;
  return r;
}
template <class T, int C> __device__ __forceinline__ int mv_plane(const Ctx<T>& c, int kk) {
  if (!c.bz) return kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk);
  if (C != 2) return kk < 0 ? -1 - kk : (kk >= c.nz ? 2 * c.nz - 1 - kk : kk);
  return min(max(kk, 0), c.nz);
}
template <class T, int C> __device__ __forceinline__ Vec16<T> mv_raw(const Ctx<T>& c, const T* __restrict__ f, const MvCol<T>& r, int kk) {
  return ld16<T>(f + (r.off + r.pl * (unsigned)mv_plane<T, C>(c, kk)));
}
template <class T, int C> __device__ __forceinline__ Vec16<T> mv_fix(const Ctx<T>& c, const MvCol<T>& r, int kk, const Vec16<T>& raw) {
  T A = r.A, B = r.B;
  if (c.bz && C != 2) {
    const int face = kk < 0 ? 4 : (kk >= c.nz ? 5 : -1);
    if (face >= 0 && c.bc[face] == FS_BC_NOSLIP) { B = T(2.0 * c.bcv[face][C]) - B; A = -A; }
  }
  Vec16<T> o;
#pragma unroll
  for (int a = 0; a < Vec16<T>::VX; ++a) o.a[a] = A * raw.a[a] + B;
  return o;
}

// ghost transform of plane kk for a column (the A, B of mv_fix), applied in place to a vector that a cp.async has put in shared memory
template <class T, int C> __device__ __forceinline__ void mv_fix_smem(const Ctx<T>& c, const MvCol<T>& r, int kk, T* slot) {
  T A = r.A, B = r.B;
  if (c.bz && C != 2) {
    const int face = kk < 0 ? 4 : (kk >= c.nz ? 5 : -1);
    if (face >= 0 && c.bc[face] == FS_BC_NOSLIP) { B = T(2.0 * c.bcv[face][C]) - B; A = -A; }
  }
  if (A != T(1) || B != T(0)) {
    Vec16<T> v = ld16<T>(slot);
#pragma unroll
    for (int a = 0; a < Vec16<T>::VX; ++a) v.a[a] = A * v.a[a] + B;
    st16<T>(slot, v);
  }
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// TY: rows of the extended tile.  ASY: planes of u, v, w go from global memory straight into the shared-memory ring with
// cp.async (no register holds a load in flight; the thread's own values of planes k-1 and k+1 are read back from the ring)
template <class T, bool UPW, bool ADT, int TY, bool ASY> __global__ void __launch_bounds__(32 * TY, 1)
k_momentumv(const Ctx<T> c, int kz, const __grid_constant__ TmapSet tm) {
  constexpr int kMvTY = TY;
  constexpr int VX = Vec16<T>::VX, ROWE = 32 * VX, PLN = kMvTY * ROWE;
  using W = Vec16<T>;
  extern __shared__ __align__(16) unsigned char mv_smem[];
  T* SU = reinterpret_cast<T*>(mv_smem); T* SV = SU + 4 * PLN; T* SW = SV + 4 * PLN;
  __shared__ T MY[8][kMvTY];
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int gx = (blockIdx.x * 30 - 1 + lane) * VX, ju = blockIdx.y * (kMvTY - 2) - 1 + ty;
  const int sx = wrapi(gx, c.nx), j = min(ju, c.nyv);
  const bool own = lane >= 1 && lane <= 30 && ty >= 1 && ty <= kMvTY - 2 && gx < c.nx && ju < c.nyv;
  const int k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nzw);
  const bool ab2 = c.time_scheme == FS_TIME_AB2 && c.S->have_hist;
  const double rdt = (ADT && ab2) ? c.S->dt / c.S->dt_prev : 1.0;
  const T a0 = ab2 ? (ADT ? T(1.0 + 0.5 * rdt) : T(1.5)) : T(1), a1 = ab2 ? (ADT ? T(-0.5 * rdt) : T(-0.5)) : T(0);
  const T dt = ADT ? T(c.S->dt) : T(c.dt), nu = T(c.nu);
  constexpr bool upw = UPW;
  const T* __restrict__ U = c.u; const T* __restrict__ V = c.v; const T* __restrict__ Wf = c.w;
  const MvCol<T> ru = mv_col<T, 0>(c, sx, j), rv = mv_col<T, 1>(c, sx, j), rw = mv_col<T, 2>(c, sx, j);
  if (lane < 8) {
    const int jc = min(max(j, 0), c.ny - 1);
    const T* tab = lane == 0 ? c.wyl + jc : lane == 1 ? c.wyh + jc : lane == 2 ? c.wyl + jc + 1 : lane == 3 ? c.wyh + jc + 1
                 : lane == 4 ? c.idy + jc + 1 : lane == 5 ? c.idy + jc : lane == 6 ? c.idyc + jc : c.idyc + jc + 1;
    MY[lane][ty] = *tab;
  }
  // shared-memory offsets inside one plane: own vector, the rows above / below, and the scalars next to the vector
  const int o_own = ty * ROWE + lane * VX;
  const int tym = ty > 0 ? ty - 1 : 0, typ = ty < kMvTY - 1 ? ty + 1 : ty;
  const int o_s = tym * ROWE + lane * VX, o_n = typ * ROWE + lane * VX;
  const int dw = lane > 0 ? -1 : 0, de = lane < 31 ? VX : VX - 1;          // west / east scalar relative to a vector start
  // register queue of the own column: B = k-1, c = k, T = k+1; n = raw loads of plane k+1 (k+2 after the store) in flight
  W uB, vB, wB, uc, vc, wc, un, vn, wn, uTq, vTq, wTq;
  auto issue = [&](int kk) {                // ASY: plane kk of u, v, w -> ring slot kk & 3 (this thread's vector)
    const int sl = (kk & 3) * PLN + o_own;
    cp_async16(SU + sl, U + (ru.off + ru.pl * (unsigned)mv_plane<T, 0>(c, kk)));
    cp_async16(SV + sl, V + (rv.off + rv.pl * (unsigned)mv_plane<T, 1>(c, kk)));
    cp_async16(SW + sl, Wf + (rw.off + rw.pl * (unsigned)mv_plane<T, 2>(c, kk)));
    cp_async_commit();
  };
  auto fixup = [&](int kk) {
    const int sl = (kk & 3) * PLN + o_own;
    mv_fix_smem<T, 0>(c, ru, kk, SU + sl); mv_fix_smem<T, 1>(c, rv, kk, SV + sl); mv_fix_smem<T, 2>(c, rw, kk, SW + sl);
  };
  if (ASY) {
    issue(k0 - 1); issue(k0); issue(k0 + 1);
    cp_async_wait_all();
    fixup(k0 - 1); fixup(k0); fixup(k0 + 1);
    __syncthreads();
    uc = ld16<T>(SU + (k0 & 3) * PLN + o_own); vc = ld16<T>(SV + (k0 & 3) * PLN + o_own); wc = ld16<T>(SW + (k0 & 3) * PLN + o_own);
    uTq = ld16<T>(SU + ((k0 + 1) & 3) * PLN + o_own); vTq = ld16<T>(SV + ((k0 + 1) & 3) * PLN + o_own); wTq = ld16<T>(SW + ((k0 + 1) & 3) * PLN + o_own);
  } else {
    uB = mv_fix<T, 0>(c, ru, k0 - 1, mv_raw<T, 0>(c, U, ru, k0 - 1)); vB = mv_fix<T, 1>(c, rv, k0 - 1, mv_raw<T, 1>(c, V, rv, k0 - 1));
    wB = mv_fix<T, 2>(c, rw, k0 - 1, mv_raw<T, 2>(c, Wf, rw, k0 - 1));
    uc = mv_fix<T, 0>(c, ru, k0, mv_raw<T, 0>(c, U, ru, k0)); vc = mv_fix<T, 1>(c, rv, k0, mv_raw<T, 1>(c, V, rv, k0));
    wc = mv_fix<T, 2>(c, rw, k0, mv_raw<T, 2>(c, Wf, rw, k0));
    un = mv_raw<T, 0>(c, U, ru, k0 + 1); vn = mv_raw<T, 1>(c, V, rv, k0 + 1); wn = mv_raw<T, 2>(c, Wf, rw, k0 + 1);
    st16<T>(SU + ((k0 - 1) & 3) * PLN + o_own, uB); st16<T>(SV + ((k0 - 1) & 3) * PLN + o_own, vB); st16<T>(SW + ((k0 - 1) & 3) * PLN + o_own, wB);
    st16<T>(SU + (k0 & 3) * PLN + o_own, uc); st16<T>(SV + (k0 & 3) * PLN + o_own, vc); st16<T>(SW + (k0 & 3) * PLN + o_own, wc);
  }
  // H^{n-1} of the own faces, one plane ahead (zero where the face does not exist)
  const bool hasu = own && j < c.ny, hasv = own, hasw = own && j < c.ny;
  const unsigned qu0 = (unsigned)sx + (unsigned)c.nx * (unsigned)j, plu = (unsigned)c.nx * (unsigned)c.ny;
  const unsigned qv0 = qu0, plv = (unsigned)c.nx * (unsigned)c.nyv;
  W zero;
#pragma unroll
  for (int a = 0; a < VX; ++a) zero.a[a] = T(0);
  W hun = zero, hvn = zero, hwn = zero;
  if (!ASY) {
    hun = (hasu && k0 < c.nz) ? ld16<T>(c.hu + (qu0 + plu * k0)) : zero;
    hvn = (hasv && k0 < c.nz) ? ld16<T>(c.hv + (qv0 + plv * k0)) : zero;
    hwn = hasw ? ld16<T>(c.hw + (qu0 + plu * k0)) : zero;
  }
  // boundary-normal faces of bounded y / z: no-slip keeps the wall velocity, slip has no normal flow
  const bool vwall = c.by && (j == 0 || j == c.ny);
  const T vwv = vwall ? (c.bc[j == 0 ? 2 : 3] == FS_BC_NOSLIP ? T(c.bcv[j == 0 ? 2 : 3][1]) : T(0)) : T(0);
  // tile planes of u, v, w and H^{n-1} go to L2 kPfAhead planes before the register loads (TMA, one thread)
  const bool pf_on = tm.n > 0 && lane == 0 && ty == 0;
  const int pf_x = (blockIdx.x * 30 - 1) * VX, pf_y = blockIdx.y * (kMvTY - 2) - 1;
  auto prefetch = [&](int k) {
    if (!pf_on || k > k1) return;
    tma_prefetch_plane(tm.m[0], pf_x, pf_y, mv_plane<T, 0>(c, k)); tma_prefetch_plane(tm.m[1], pf_x, pf_y, mv_plane<T, 1>(c, k));
    tma_prefetch_plane(tm.m[2], pf_x, pf_y, mv_plane<T, 2>(c, k));
    // H^{n-1} is only read on the tile's own faces: its boxes are the 30 VX x (TY - 2) interior
    if (k < k1 && k < c.nz) { tma_prefetch_plane(tm.m[3], pf_x + VX, pf_y + 1, k); tma_prefetch_plane(tm.m[4], pf_x + VX, pf_y + 1, k); }
    if (k < k1) tma_prefetch_plane(tm.m[5], pf_x + VX, pf_y + 1, k);
  };
  for (int k = k0 + 2; k < k0 + 2 + kPfAhead; ++k) prefetch(k);
  for (int k = k0; k < k1; ++k) {
    const int s0 = ((k - 1) & 3) * PLN, s1 = (k & 3) * PLN, s2 = ((k + 1) & 3) * PLN;
    W uT, vT, wT, huo, hvo, hwo;
    if (ASY) {
      // planes k-1, k, k+1 are in the ring and visible (barrier at the end of the previous plane); plane k+2 starts its way now
      if (k + 1 < k1) issue(k + 2);
      prefetch(k + 2 + kPfAhead);
      uT = uTq; vT = vTq; wT = wTq;
      huo = (hasu && k < c.nz) ? ld16<T>(c.hu + (qu0 + plu * k)) : zero;
      hvo = (hasv && k < c.nz) ? ld16<T>(c.hv + (qv0 + plv * k)) : zero;
      hwo = hasw ? ld16<T>(c.hw + (qu0 + plu * k)) : zero;
    } else {
      uT = mv_fix<T, 0>(c, ru, k + 1, un); vT = mv_fix<T, 1>(c, rv, k + 1, vn); wT = mv_fix<T, 2>(c, rw, k + 1, wn);
      huo = hun; hvo = hvn; hwo = hwn;
      if (k + 1 < k1) {
        hun = (hasu && k + 1 < c.nz) ? ld16<T>(c.hu + (qu0 + plu * (k + 1))) : zero;
        hvn = (hasv && k + 1 < c.nz) ? ld16<T>(c.hv + (qv0 + plv * (k + 1))) : zero;
        hwn = hasw ? ld16<T>(c.hw + (qu0 + plu * (k + 1))) : zero;
      }
      st16<T>(SU + s2 + o_own, uT); st16<T>(SV + s2 + o_own, vT); st16<T>(SW + s2 + o_own, wT);
      prefetch(k + 2 + kPfAhead);
      if (k + 1 < k1) { un = mv_raw<T, 0>(c, U, ru, k + 2); vn = mv_raw<T, 1>(c, V, rv, k + 2); wn = mv_raw<T, 2>(c, Wf, rw, k + 2); }
      __syncthreads();
    }
    if (own) {
      const T wyl0 = MY[0][ty], wyh0 = MY[1][ty], wyl1 = MY[2][ty], wyh1 = MY[3][ty];
      const T idyj = MY[4][ty], idyjm = MY[5][ty], idyc0 = MY[6][ty], idyc1 = MY[7][ty];
      // neighbours: rows above / below as vectors, one scalar west / east of the own vector; each component loads what it
      // needs inside its own block (the compiler barriers keep the three blocks' shared-memory loads from being hoisted
      // to the top together: that would hold 8 vectors + 10 scalars live on top of the register queue)
      const bool kin = k < c.nz;
      if (ASY) { uB = ld16<T>(SU + s0 + o_own); vB = ld16<T>(SV + s0 + o_own); wB = ld16<T>(SW + s0 + o_own); }
      // ---- u faces ----
      if (j < c.ny && kin) {
        const W uN = ld16<T>(SU + s1 + o_n), uS = ld16<T>(SU + s1 + o_s), vN = ld16<T>(SV + s1 + o_n);
        const T uWs = SU[s1 + o_own + dw], uEs = SU[s1 + o_own + de], vWs = SV[s1 + o_own + dw], vNWs = SV[s1 + o_n + dw];
        const T wWs = SW[s1 + o_own + dw], wTWs = SW[s2 + o_own + dw];
        W us, H;
#pragma unroll
        for (int a = 0; a < VX; ++a) {
          const T ucc = uc.a[a], uE = a < VX - 1 ? uc.a[a < VX - 1 ? a + 1 : a] : uEs, uW = a > 0 ? uc.a[a > 0 ? a - 1 : 0] : uWs;
          const T ue = T(0.5) * (ucc + uE), uw = T(0.5) * (uW + ucc);
          const T cx = (ue * mv_tr<T>(upw, ue, ucc, uE, ue) - uw * mv_tr<T>(upw, uw, uW, ucc, uw)) * c.ihx;
          const T vNw = a > 0 ? vN.a[a > 0 ? a - 1 : 0] : vNWs, vCw = a > 0 ? vc.a[a > 0 ? a - 1 : 0] : vWs;
          const T vnn = T(0.5) * (vNw + vN.a[a]), unn = mv_tr<T>(upw, vnn, ucc, uN.a[a], wyl1 * ucc + wyh1 * uN.a[a]);
          const T vss = T(0.5) * (vCw + vc.a[a]), uss = mv_tr<T>(upw, vss, uS.a[a], ucc, wyl0 * uS.a[a] + wyh0 * ucc);
          const T cy = (vnn * unn - vss * uss) * idyj;
          const T wTw = a > 0 ? wT.a[a > 0 ? a - 1 : 0] : wTWs, wCw = a > 0 ? wc.a[a > 0 ? a - 1 : 0] : wWs;
          const T wt = T(0.5) * (wTw + wT.a[a]), ut = mv_tr<T>(upw, wt, ucc, uT.a[a], T(0.5) * (ucc + uT.a[a]));
          const T wb = T(0.5) * (wCw + wc.a[a]), ub = mv_tr<T>(upw, wb, uB.a[a], ucc, T(0.5) * (uB.a[a] + ucc));
          const T cz = (wt * ut - wb * ub) * c.ihz;
          const T dxx = (uE - T(2) * ucc + uW) * c.ihx2;
          const T dyy = ((uN.a[a] - ucc) * idyc1 - (ucc - uS.a[a]) * idyc0) * idyj;
          const T dzz = (uT.a[a] - T(2) * ucc + uB.a[a]) * c.ihz2;
          const T h = -(cx + cy + cz) + nu * (dxx + dyy + dzz) + T(c.g[0]);
          H.a[a] = h; us.a[a] = ucc + dt * (a0 * h + a1 * huo.a[a]);
        }
        const unsigned q = qu0 + plu * (unsigned)k;
        st16<T>(c.us + q, us); st16<T>(c.hu + q, H);
      }
      asm volatile("" ::: "memory");
      // ---- v faces (control volume between y_c(j-1) and y_c(j)) ----
      if (kin) {
        const W vN = ld16<T>(SV + s1 + o_n), vS = ld16<T>(SV + s1 + o_s), uS = ld16<T>(SU + s1 + o_s);
        const W wS = ld16<T>(SW + s1 + o_s), wS2 = ld16<T>(SW + s2 + o_s);
        const T vWs = SV[s1 + o_own + dw], vEs = SV[s1 + o_own + de], uEs = SU[s1 + o_own + de], uSEs = SU[s1 + o_s + de];
        W vs, H;
        if (vwall) {
#pragma unroll
          for (int a = 0; a < VX; ++a) { vs.a[a] = vwv; H.a[a] = T(0); }
        } else {
#pragma unroll
          for (int a = 0; a < VX; ++a) {
            const T vcc = vc.a[a], vE = a < VX - 1 ? vc.a[a < VX - 1 ? a + 1 : a] : vEs, vW = a > 0 ? vc.a[a > 0 ? a - 1 : 0] : vWs;
            const T uSe = a < VX - 1 ? uS.a[a < VX - 1 ? a + 1 : a] : uSEs, uCe = a < VX - 1 ? uc.a[a < VX - 1 ? a + 1 : a] : uEs;
            const T ue = wyl0 * uSe + wyh0 * uCe, ve = mv_tr<T>(upw, ue, vcc, vE, T(0.5) * (vcc + vE));
            const T uw = wyl0 * uS.a[a] + wyh0 * uc.a[a], vw = mv_tr<T>(upw, uw, vW, vcc, T(0.5) * (vW + vcc));
            const T cx = (ue * ve - uw * vw) * c.ihx;
            const T vnn = T(0.5) * (vcc + vN.a[a]), vss = T(0.5) * (vS.a[a] + vcc);
            const T cy = (vnn * mv_tr<T>(upw, vnn, vcc, vN.a[a], vnn) - vss * mv_tr<T>(upw, vss, vS.a[a], vcc, vss)) * idyc0;
            const T wt = wyl0 * wS2.a[a] + wyh0 * wT.a[a], vt = mv_tr<T>(upw, wt, vcc, vT.a[a], T(0.5) * (vcc + vT.a[a]));
            const T wb = wyl0 * wS.a[a] + wyh0 * wc.a[a], vb = mv_tr<T>(upw, wb, vB.a[a], vcc, T(0.5) * (vB.a[a] + vcc));
            const T cz = (wt * vt - wb * vb) * c.ihz;
            const T dxx = (vE - T(2) * vcc + vW) * c.ihx2;
            const T dyy = ((vN.a[a] - vcc) * idyj - (vcc - vS.a[a]) * idyjm) * idyc0;
            const T dzz = (vT.a[a] - T(2) * vcc + vB.a[a]) * c.ihz2;
            const T h = -(cx + cy + cz) + nu * (dxx + dyy + dzz) + T(c.g[1]);
            H.a[a] = h; vs.a[a] = vcc + dt * (a0 * h + a1 * hvo.a[a]);
          }
        }
        const unsigned q = qv0 + plv * (unsigned)k;
        st16<T>(c.vs + q, vs); st16<T>(c.hv + q, H);
      }
      asm volatile("" ::: "memory");
      // ---- w faces ----
      if (j < c.ny) {
        const W wN = ld16<T>(SW + s1 + o_n), wS = ld16<T>(SW + s1 + o_s), vN = ld16<T>(SV + s1 + o_n), vN0 = ld16<T>(SV + s0 + o_n);
        const T wWs = SW[s1 + o_own + dw], wEs = SW[s1 + o_own + de], uEs = SU[s1 + o_own + de], uB_Es = SU[s0 + o_own + de];
        W ws, H;
        if (c.bz && (k == 0 || k == c.nz)) {
          const T wv = c.bc[k == 0 ? 4 : 5] == FS_BC_NOSLIP ? T(c.bcv[k == 0 ? 4 : 5][2]) : T(0);
#pragma unroll
          for (int a = 0; a < VX; ++a) { ws.a[a] = wv; H.a[a] = T(0); }
        } else {
#pragma unroll
          for (int a = 0; a < VX; ++a) {
            const T wcc = wc.a[a], wE = a < VX - 1 ? wc.a[a < VX - 1 ? a + 1 : a] : wEs, wW = a > 0 ? wc.a[a > 0 ? a - 1 : 0] : wWs;
            const T uBe = a < VX - 1 ? uB.a[a < VX - 1 ? a + 1 : a] : uB_Es, uCe = a < VX - 1 ? uc.a[a < VX - 1 ? a + 1 : a] : uEs;
            const T ue = T(0.5) * (uBe + uCe), we = mv_tr<T>(upw, ue, wcc, wE, T(0.5) * (wcc + wE));
            const T uw = T(0.5) * (uB.a[a] + uc.a[a]), ww = mv_tr<T>(upw, uw, wW, wcc, T(0.5) * (wW + wcc));
            const T cx = (ue * we - uw * ww) * c.ihx;
            const T vnn = T(0.5) * (vN0.a[a] + vN.a[a]), wnn = mv_tr<T>(upw, vnn, wcc, wN.a[a], wyl1 * wcc + wyh1 * wN.a[a]);
            const T vss = T(0.5) * (vB.a[a] + vc.a[a]), wss = mv_tr<T>(upw, vss, wS.a[a], wcc, wyl0 * wS.a[a] + wyh0 * wcc);
            const T cy = (vnn * wnn - vss * wss) * idyj;
            const T wt = T(0.5) * (wcc + wT.a[a]), wb = T(0.5) * (wB.a[a] + wcc);
            const T cz = (wt * mv_tr<T>(upw, wt, wcc, wT.a[a], wt) - wb * mv_tr<T>(upw, wb, wB.a[a], wcc, wb)) * c.ihz;
            const T dxx = (wE - T(2) * wcc + wW) * c.ihx2;
            const T dyy = ((wN.a[a] - wcc) * idyc1 - (wcc - wS.a[a]) * idyc0) * idyj;
            const T dzz = (wT.a[a] - T(2) * wcc + wB.a[a]) * c.ihz2;
            const T h = -(cx + cy + cz) + nu * (dxx + dyy + dzz) + T(c.g[2]);
            H.a[a] = h; ws.a[a] = wcc + dt * (a0 * h + a1 * hwo.a[a]);
          }
        }
        const unsigned q = qu0 + plu * (unsigned)k;
        st16<T>(c.ws + q, ws); st16<T>(c.hw + q, H);
      }
    }
    if (ASY) {
      cp_async_wait_all();
      if (k + 1 < k1) fixup(k + 2);
      __syncthreads();
      uc = uT; vc = vT; wc = wT;
      const int s3 = ((k + 2) & 3) * PLN + o_own;
      uTq = ld16<T>(SU + s3); vTq = ld16<T>(SV + s3); wTq = ld16<T>(SW + s3);
    } else { uB = uc; uc = uT; vB = vc; vc = vT; wB = wc; wc = wT; }
  }
}

// Load path per precision (profiles/r2_momentum.md, 512^3): fp64 with register loads sat at its 128-register cap with 16 warps
// per SM (4.25 ms against k_momentum's 3.45); with cp.async the loads in flight and the k-1 / k+1 copies of the own column live
// in the ring, the kernel needs 121 registers without spills and runs at 3.27 ms.  fp32 (four cells per thread, enough
// independent work) is faster with register loads: 1.55 ms against 1.76 with cp.async.  Tile heights 14 / 18 / 20 rows were
// slower in fp64 (3.40 / 4.47 / 3.85 ms: fewer warps, or spills at the lower register caps).
template <class T> struct MvCfg { static constexpr int TY = 16; static constexpr bool ASY = sizeof(T) == 8; };
template <class T> static size_t momv_smem() { return 12 * (size_t)MvCfg<T>::TY * 32 * Vec16<T>::VX * sizeof(T); }

template <class T> bool momentumv_applies(const Ctx<T>& c) {
  if (c.bx || c.nx % Vec16<T>::VX != 0) return false;
  if (c.nu > 0.0 && (c.cs > 0.0 || c.wall_model)) return false;
  for (int f = 2; f < 6; ++f) if (c.bc[f] != FS_BC_PERIODIC && c.bc[f] != FS_BC_NOSLIP && c.bc[f] != FS_BC_SLIP) return false;
  // FS_TUNE_MOMV=0 (read at every launch: a parity test switches it) routes these grids through k_momentum as well
  const char* e = getenv("FS_TUNE_MOMV");
  return !(e && atoi(e) == 0);
}

template <class T> cudaError_t momv_configure_device() {
  const int bytes = (int)momv_smem<T>();
  constexpr int TY = MvCfg<T>::TY; constexpr bool A = MvCfg<T>::ASY;
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(k_momentumv<T, false, false, TY, A>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(k_momentumv<T, false, true, TY, A>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(k_momentumv<T, true, false, TY, A>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_momentumv<T, true, true, TY, A>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

template <class T> int launch_momentumv(const Ctx<T>& c, const Launch& L) {
  constexpr int VX = Vec16<T>::VX, TY = MvCfg<T>::TY; constexpr bool A = MvCfg<T>::ASY;
  const int bxn = (c.nx + 30 * VX - 1) / (30 * VX), byn = (c.nyv + TY - 3) / (TY - 2);
  const int kz = pick_kz((long long)bxn * byn, c.nzw, 148, 2, 16);
  const dim3 b(32, TY, 1), g(bxn, byn, (c.nzw + kz - 1) / kz);
  const bool adt = c.cfl > 0.0, upw = c.convection == FS_CONV_UPWIND;
  TmapSet tm; memset(&tm, 0, sizeof tm);
  static const int pf = [] { const char* e = getenv("FS_TUNE_PF2"); return e ? atoi(e) : 1; }();
  const int bw = 32 * VX, bh = TY;
  // the cp.async variant already has a whole plane of lead on its loads: the L2 prefetch changes nothing there (3.28 vs 3.28 ms)
  if (pf && !A && tmap_encode(&tm.m[0], c.u, sizeof(T), c.nx, c.ny, c.nz, bw, bh) && tmap_encode(&tm.m[1], c.v, sizeof(T), c.nx, c.nyv, c.nz, bw, bh) &&
      tmap_encode(&tm.m[2], c.w, sizeof(T), c.nx, c.ny, c.nzw, bw, bh) && tmap_encode(&tm.m[3], c.hu, sizeof(T), c.nx, c.ny, c.nz, bw - 2 * VX, bh - 2) &&
      tmap_encode(&tm.m[4], c.hv, sizeof(T), c.nx, c.nyv, c.nz, bw - 2 * VX, bh - 2) && tmap_encode(&tm.m[5], c.hw, sizeof(T), c.nx, c.ny, c.nzw, bw - 2 * VX, bh - 2)) tm.n = 6;
  static const char* names[2][2] = {{"k_momentumv<f32,central>", "k_momentumv<f32,upwind>"}, {"k_momentumv<f64,central>", "k_momentumv<f64,upwind>"}};
  const size_t smem = momv_smem<T>();
  FS_LAUNCHI(L, "momentum_predictor", names[sizeof(T) == 8][upw], 12.0 * sizeof(T) * c.nx * c.ny * c.nz, {
    if (upw) { if (adt) k_momentumv<T, true, true, TY, A><<<g, b, smem, L.s>>>(c, kz, tm); else k_momentumv<T, true, false, TY, A><<<g, b, smem, L.s>>>(c, kz, tm); }
    else { if (adt) k_momentumv<T, false, true, TY, A><<<g, b, smem, L.s>>>(c, kz, tm); else k_momentumv<T, false, false, TY, A><<<g, b, smem, L.s>>>(c, kz, tm); }
  });
  return 1;
}

template bool momentumv_applies<float>(const Ctx<float>&);
template bool momentumv_applies<double>(const Ctx<double>&);
template cudaError_t momv_configure_device<float>();
template cudaError_t momv_configure_device<double>();
template int launch_momentumv<float>(const Ctx<float>&, const Launch&);
template int launch_momentumv<double>(const Ctx<double>&, const Launch&);

}  // namespace fs
