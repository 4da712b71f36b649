// fs_beam.cu -- flexible structure: Euler-Bernoulli beam elements + Newmark-beta (Eq. 11, Eq. 13-17
// L155-177, L177; reading N2-2 in DESIGN.md 3).
//
// Host (fs_set_beam, once): element matrices of Eq. 13-14 assembled into band storage (node 0 clamped: its two degrees of
// freedom are dropped; half bandwidth 3), the two lowest frequencies of Eq. 17 by a Cholesky reduction of the pencil to a
// standard symmetric problem + cyclic Jacobi rotations, Rayleigh damping (Eq. 15-16), and the banded Cholesky factor of
// the effective stiffness K_eff = K + a0 M + a1 C of the Newmark scheme (the step size is fixed when a beam is present).
// Device (every step, one CTA): nodal loads gathered from the marker forces in ascending marker id (Eq. 20), banded
// matrix-vector products, the banded triangular solves (one thread: <= 256 unknowns, bandwidth 3), the state update,
// xi of Algorithm 1, and the marker update X = X^ref + w n, U^b = dw/dt n.  All of it in fp64 whatever the grid's dtype
// (marker arrays are fp64).
#include "fs_internal.cuh"
#include <cmath>
#include <vector>

namespace fs {

// ---- host ---------------------------------------------------------------------------------------------------------
bool beam_build(int nb, const double* xy, double EI, double mus, double zeta, double dt,
                double* Lb, double* Mb, double* Cb, double* nk, double* coef) {
  const int n = 2 * (nb - 1);
  std::vector<double> K((size_t)n * n, 0.0), M((size_t)n * n, 0.0);
  auto add = [&](std::vector<double>& A, int r, int c, double v) { if (r >= 2 && c >= 2) A[(size_t)(r - 2) * n + (c - 2)] += v; };
  for (int e = 0; e + 1 < nb; ++e) {
    const double L = std::hypot(xy[2 * (e + 1)] - xy[2 * e], xy[2 * (e + 1) + 1] - xy[2 * e + 1]), L2 = L * L;
    const double k0 = EI / (L2 * L), m0 = mus * L / 420.0;
    const double ke[4][4] = {{12, 6 * L, -12, 6 * L}, {6 * L, 4 * L2, -6 * L, 2 * L2}, {-12, -6 * L, 12, -6 * L}, {6 * L, 2 * L2, -6 * L, 4 * L2}};       // Eq. 13
    const double me[4][4] = {{156, 22 * L, 54, -13 * L}, {22 * L, 4 * L2, 13 * L, -3 * L2}, {54, 13 * L, 156, -22 * L}, {-13 * L, -3 * L2, -22 * L, 4 * L2}}; // Eq. 14
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) { add(K, 2 * e + a, 2 * e + b, k0 * ke[a][b]); add(M, 2 * e + a, 2 * e + b, m0 * me[a][b]); }
  }
  // Eq. 17: M = G G^T, A = G^-1 K G^-T, eigenvalues of A by cyclic Jacobi; the two smallest are omega_1^2, omega_2^2
  std::vector<double> G((size_t)n * n, 0.0);
  for (int j = 0; j < n; ++j) {
    double d = M[(size_t)j * n + j];
    for (int k = 0; k < j; ++k) d -= G[(size_t)j * n + k] * G[(size_t)j * n + k];
    if (!(d > 0.0)) return false;
    G[(size_t)j * n + j] = std::sqrt(d);
    for (int i = j + 1; i < n; ++i) {
      double t = M[(size_t)i * n + j];
      for (int k = 0; k < j; ++k) t -= G[(size_t)i * n + k] * G[(size_t)j * n + k];
      G[(size_t)i * n + j] = t / G[(size_t)j * n + j];
    }
  }
  std::vector<double> A = K;
  for (int c = 0; c < n; ++c)                 // A <- G^-1 A  (forward substitution, column by column)
    for (int i = 0; i < n; ++i) {
      double t = A[(size_t)i * n + c];
      for (int k = 0; k < i; ++k) t -= G[(size_t)i * n + k] * A[(size_t)k * n + c];
      A[(size_t)i * n + c] = t / G[(size_t)i * n + i];
    }
  for (int r = 0; r < n; ++r)                 // A <- A G^-T  (row by row)
    for (int i = 0; i < n; ++i) {
      double t = A[(size_t)r * n + i];
      for (int k = 0; k < i; ++k) t -= G[(size_t)i * n + k] * A[(size_t)r * n + k];
      A[(size_t)r * n + i] = t / G[(size_t)i * n + i];
    }
  for (int r = 0; r < n; ++r) for (int c = r + 1; c < n; ++c) { const double t = 0.5 * (A[(size_t)r * n + c] + A[(size_t)c * n + r]); A[(size_t)r * n + c] = A[(size_t)c * n + r] = t; }
  for (int sweep = 0; sweep < 60; ++sweep) {
    double off = 0.0, dia = 0.0;
    for (int r = 0; r < n; ++r) for (int c = 0; c < n; ++c) (r == c ? dia : off) += A[(size_t)r * n + c] * A[(size_t)r * n + c];
    if (off <= 1e-30 * dia) break;
    for (int p = 0; p < n; ++p) for (int q = p + 1; q < n; ++q) {
      const double apq = A[(size_t)p * n + q];
      if (apq == 0.0) continue;
      const double th = (A[(size_t)q * n + q] - A[(size_t)p * n + p]) / (2.0 * apq);
      const double t = (th >= 0 ? 1.0 : -1.0) / (std::fabs(th) + std::sqrt(th * th + 1.0)), cs = 1.0 / std::sqrt(t * t + 1.0), sn = t * cs;
      for (int k = 0; k < n; ++k) { const double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q]; A[(size_t)k * n + p] = cs * akp - sn * akq; A[(size_t)k * n + q] = sn * akp + cs * akq; }
      for (int k = 0; k < n; ++k) { const double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k]; A[(size_t)p * n + k] = cs * apk - sn * aqk; A[(size_t)q * n + k] = sn * apk + cs * aqk; }
    }
  }
  double l1 = 1e300, l2 = 1e300;
  for (int r = 0; r < n; ++r) { const double v = A[(size_t)r * n + r]; if (v < l1) { l2 = l1; l1 = v; } else if (v < l2) l2 = v; }
  if (!(l1 > 0.0) || !(l2 > 0.0)) return false;
  const double om1 = std::sqrt(l1), om2 = std::sqrt(l2);
  const double alpha = 2.0 * zeta * om1 * om2 / (om1 + om2), beta = 2.0 * zeta / (om1 + om2);       // Eq. 16
  coef[0] = alpha; coef[1] = beta; coef[2] = om1; coef[3] = om2;
  // Newmark-beta, gamma = 1/2, beta_N = 1/4
  const double gam = 0.5, bet = 0.25;
  nk[0] = 1.0 / (bet * dt * dt); nk[1] = gam / (bet * dt); nk[2] = 1.0 / (bet * dt); nk[3] = 1.0 / (2.0 * bet) - 1.0;
  nk[4] = gam / bet - 1.0; nk[5] = 0.5 * dt * (gam / bet - 2.0);
  // band storage of M, C (Eq. 15) and the banded Cholesky factor of K_eff
  std::vector<double> Ke((size_t)n * 7, 0.0);
  for (int r = 0; r < n; ++r) for (int d = -3; d <= 3; ++d) {
    const int c = r + d; double m = 0.0, k = 0.0;
    if (c >= 0 && c < n) { m = M[(size_t)r * n + c]; k = K[(size_t)r * n + c]; }
    const double cc = alpha * m + beta * k;
    Mb[(size_t)r * 7 + d + 3] = m; Cb[(size_t)r * 7 + d + 3] = cc; Ke[(size_t)r * 7 + d + 3] = k + nk[0] * m + nk[1] * cc;
  }
  for (int r = 0; r < n; ++r) {               // L[r][c], c = r-3..r, stored at Lb[r*4 + (c - r + 3)]
    for (int c = r - 3; c <= r; ++c) {
      if (c < 0) { Lb[(size_t)r * 4 + (c - r + 3)] = 0.0; continue; }
      double t = Ke[(size_t)r * 7 + (c - r + 3)];
      for (int k = (r - 3 > 0 ? r - 3 : 0); k < c; ++k) if (k >= c - 3) t -= Lb[(size_t)r * 4 + (k - r + 3)] * Lb[(size_t)c * 4 + (k - c + 3)];
      if (c == r) { if (!(t > 0.0)) return false; Lb[(size_t)r * 4 + 3] = std::sqrt(t); }
      else Lb[(size_t)r * 4 + (c - r + 3)] = t / Lb[(size_t)c * 4 + 3];
    }
  }
  return true;
}

// ---- device -------------------------------------------------------------------------------------------------------
template <class T> __global__ void __launch_bounds__(256) k_beam_step(const Ctx<T> c, const IbmCtx ib) {
  __shared__ double Q[2 * kMaxBeamNodes], rhs[2 * kMaxBeamNodes], tm[2 * kMaxBeamNodes], tc[2 * kMaxBeamNodes], wn[2 * kMaxBeamNodes];
  const int n = ib.ndof, tid = threadIdx.x;
  const double* w0 = ib.strong ? ib.bw0 : ib.bw; const double* v0 = ib.strong ? ib.bv0 : ib.bv; const double* a0 = ib.strong ? ib.ba0 : ib.ba;
  const double rho = c.rho;
  // Eq. 20 gathered per node and projected on the axis normal; markers in ascending id; no nodal moments
  for (int r = tid; r < n; r += blockDim.x) {
    double q = 0.0;
    if (!(r & 1)) {
      const int node = (r >> 1) + 1;
      for (int k = ib.nstart[node]; k < ib.nstart[node + 1]; ++k) {
        const int l = ib.nlist[k];
        const double qx = -rho * ib.Fl[3 * l] * ib.dV[l], qy = -rho * ib.Fl[3 * l + 1] * ib.dV[l];
        q += qx * ib.bnrm[0] + qy * ib.bnrm[1];
      }
    }
    Q[r] = q;
    tm[r] = ib.nk[0] * w0[r] + ib.nk[2] * v0[r] + ib.nk[3] * a0[r];
    tc[r] = ib.nk[1] * w0[r] + ib.nk[4] * v0[r] + ib.nk[5] * a0[r];
  }
  __syncthreads();
  for (int r = tid; r < n; r += blockDim.x) {
    double mt = 0.0, ct = 0.0;
    for (int d = 0; d < 7; ++d) { const int k = r + d - 3; if (k >= 0 && k < n) { mt += ib.bM[r * 7 + d] * tm[k]; ct += ib.bC[r * 7 + d] * tc[k]; } }
    rhs[r] = Q[r] + mt + ct;
  }
  __syncthreads();
  if (tid == 0) {                            // K_eff w = rhs with K_eff = L L^T (half bandwidth 3)
    for (int r = 0; r < n; ++r) {
      double t = rhs[r];
      for (int k = (r - 3 > 0 ? r - 3 : 0); k < r; ++k) t -= ib.bL[r * 4 + (k - r + 3)] * wn[k];
      wn[r] = t / ib.bL[r * 4 + 3];
    }
    for (int r = n - 1; r >= 0; --r) {
      double t = wn[r];
      for (int k = r + 1; k <= r + 3 && k < n; ++k) t -= ib.bL[k * 4 + (r - k + 3)] * wn[k];
      wn[r] = t / ib.bL[r * 4 + 3];
    }
    double xi = 0.0;                         // Algorithm 1: || (w^k - w^(k-1)) / w^(k-1) ||^2, the markers reflect w^(k-1) = ib.bw
    for (int r = 0; r < n; ++r) { const double prev = ib.bw[r], dw = wn[r] - prev; if (!(dw == 0.0 && prev == 0.0)) xi += (dw / prev) * (dw / prev); }
    c.S->beam_xi = xi;
  }
  __syncthreads();
  for (int r = tid; r < n; r += blockDim.x) {
    const double an = ib.nk[0] * (wn[r] - w0[r]) - ib.nk[2] * v0[r] - ib.nk[3] * a0[r];
    const double vn = v0[r] + c.S->dt * (0.5 * a0[r] + 0.5 * an);
    ib.bQ[r] = Q[r];
    tm[r] = vn;                              // velocity of the new state, for the marker update below
    ib.bw[r] = wn[r]; ib.bv[r] = vn; ib.ba[r] = an;
  }
  __syncthreads();
  for (int l = tid; l < ib.n; l += blockDim.x) {
    const int node = ib.mnode[l];
    const double w = node > 0 ? wn[2 * (node - 1)] : 0.0, wd = node > 0 ? tm[2 * (node - 1)] : 0.0;
    ib.X[3 * l] = ib.Xref[3 * l] + w * ib.bnrm[0]; ib.X[3 * l + 1] = ib.Xref[3 * l + 1] + w * ib.bnrm[1]; ib.X[3 * l + 2] = ib.Xref[3 * l + 2];
    ib.Ub[3 * l] = wd * ib.bnrm[0]; ib.Ub[3 * l + 1] = wd * ib.bnrm[1]; ib.Ub[3 * l + 2] = 0.0;
  }
}
template <class T> int launch_beam_step(const Ctx<T>& c, const IbmCtx& ib, const Launch& L) {
  FS_LAUNCH(L, "beam_newmark", 0.0, k_beam_step<T><<<1, 256, 0, L.s>>>(c, ib));
  return 1;
}
template int launch_beam_step<float>(const Ctx<float>&, const IbmCtx&, const Launch&);
template int launch_beam_step<double>(const Ctx<double>&, const IbmCtx&, const Launch&);

}  // namespace fs
