// fs_oracle.cpp -- CPU ORACLE (test infrastructure, NOT the product; see fs_oracle.h).
//
// Plain single-threaded fp64 restatement of one fractional step of Diff-FlowFSI's fluid solver
// (section 2.3.1, Eq. 4-10) with marker-based direct-forcing IBM (Eq. 3, 5, 20-22) and
// the rigid-body oscillator (Eq. 12), following SURVEY.md 8(c) steps O1..O9 in that order.
// Triple loops, explicit index wrapping, sums in index order, no blocking / fusion / threads.
// Compile: g++ -O2 -ffp-contract=off (no FMA contraction, so index arithmetic is reproducible).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): P1..P17 of SURVEY.md 8(c) / DESIGN.md 4 and P18..P23
// (tests/test_oracle_boundary.py): slip / no-slip / inflow / outflow tangential ghosts, the convective outflow
// update, the direct-forcing scale of I-3 / I-4, the uniform outflow flux shift, rejection of supports that reach a
// non-periodic boundary, and the inflow-noise hash (published SplitMix64 vectors + frozen table).
// Parity unpinned: no function.  The convective-outflow formula, the flux correction and the hash chaining are
// READINGS of what the paper leaves open: the pins fix what the oracle computes, not the paper's intent.
#include "fs_oracle.h"
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>

typedef std::vector<double> vec;

struct orc_sim {
  orc_params P;
  int nx, ny, nz, bx, by, bz;          // bounded flags
  int nxu, nyv, nzw;                   // stored extent of each component along its own normal
  double hx, hy, hz;
  bool uniform_y;
  vec yf, dy, yc;                      // faces (ny+1), cell heights (ny), centres (ny)
  vec u, v, w, p, hu, hv, hw, divu;
  bool have_hist; long long step;
  double dt, dt_prev, time;            // step size of the current / previous step (CFL-adaptive dt), elapsed time
  // markers (always fp64)
  int nl; vec X, Ub, dV, Fl, Ul;       // positions, target vel, volumes, force, interpolated vel
  std::vector<int> base, perm, keys, seg; int nseg;
  bool oob;                            // a support reached a prescribed face / left a bounded box (unsupported)
  // body (Eq. 12)
  bool has_body; double bm, bc_, bk; int dof; double bdisp[3], bvel[3], bforce[3];
  // flexible beam (Eq. 11, 13-17, Newmark-beta; reading N2-2 in DESIGN.md 3)
  bool has_beam; int nb, ndof;         // nodes; degrees of freedom = 2 (nb - 1): (deflection, rotation) of nodes 1..nb-1, node 0 clamped
  vec bX0; std::vector<int> mnode;     // reference node positions (x, y); node of every marker
  double bnrm[2];                      // unit normal of the straight reference axis: markers move along it
  double EI, mus, zeta, ralpha, rbeta, om1, om2;   // Eq. 13-16: stiffness, mass per length, damping ratio, Rayleigh coefficients, omega_1, omega_2
  vec BK, BM, BC;                      // global matrices (ndof x ndof, dense, row major)
  vec bw, bv, ba, bQ;                  // displacement, velocity, acceleration of the DOFs; load vector of the last step
  vec Xref;                            // marker positions of the undeformed beam
  // GMG levels
  int nlev;
  // volume-of-solid mask (eps-mask IBM, Eq. 5, 8-9, 18-19, 23; reading E1 in DESIGN.md 3)
  bool has_mask; double uc[3];         // exact velocity of the immersed solid u_c (Eq. 8); a rigid body overrides it with its velocity
  std::vector<unsigned char> eps, mu, mv, mw;   // cell mask; per-face class of u, v, w: 0 fluid, 1 solid, 2 IB point
};

static inline int wrapi(int i, int n) { i %= n; return i < 0 ? i + n : i; }

// ---- grid metrics (SURVEY 8(c) "Grid") -------------------------------------------------
// DY(j) for j in [-1, ny]: mirrored ghost at a bounded end, wrapped when periodic.
static inline double DY(const orc_sim* s, int j) {
  if (j < 0)       return s->by ? s->dy[0]         : s->dy[wrapi(j, s->ny)];
  if (j >= s->ny)  return s->by ? s->dy[s->ny - 1] : s->dy[wrapi(j, s->ny)];
  return s->dy[j];
}
// distance between centres j-1 and j (across face j), j in [0, ny]
static inline double DYC(const orc_sim* s, int j) { return 0.5 * (DY(s, j - 1) + DY(s, j)); }

// ---- O1: velocity access with boundary rules ----------------------------------------------
// comp c (0=u,1=v,2=w); index (i,j,k) may be one layer outside in a tangential direction.
// Periodic: wrap.  Own normal direction, bounded: faces 0..n are stored.  Tangential, bounded:
// ghost = A*interior + B  with  no-slip/inflow: (-1, 2*bc_vel)  slip/outflow: (+1, 0).
static double getvel(const orc_sim* s, const vec& f, int c, int i, int j, int k) {
  const int n[3] = {s->nx, s->ny, s->nz};
  const int bd[3] = {s->bx, s->by, s->bz};
  int idx[3] = {i, j, k};
  double A = 1.0, B = 0.0;
  for (int d = 0; d < 3; ++d) {
    if (!bd[d]) { idx[d] = wrapi(idx[d], n[d]); continue; }
    if (d == c) continue;                       // stored 0..n
    int face = -1;
    if (idx[d] < 0)       { face = 2 * d;     idx[d] = -1 - idx[d]; }
    else if (idx[d] >= n[d]) { face = 2 * d + 1; idx[d] = 2 * n[d] - 1 - idx[d]; }
    if (face >= 0) {
      int t = s->P.bc[face];
      if (t == ORC_BC_NOSLIP || t == ORC_BC_INFLOW) { B = B * -1.0 + 2.0 * s->P.bc_vel[face][c]; A = -A; }
      // slip / outflow: zero gradient, A,B unchanged
    }
  }
  int ex = s->nx + (c == 0 ? s->bx : 0), ey = s->ny + (c == 1 ? s->by : 0);
  return A * f[(size_t)idx[0] + (size_t)ex * (idx[1] + (size_t)ey * idx[2])] + B;
}
#define U_(i,j,k) getvel(s, uu, 0, i, j, k)
#define V_(i,j,k) getvel(s, vv, 1, i, j, k)
#define W_(i,j,k) getvel(s, ww, 2, i, j, k)

static inline size_t IU(const orc_sim* s, int i, int j, int k) { return (size_t)i + (size_t)s->nxu * (j + (size_t)s->ny * k); }
static inline size_t IV(const orc_sim* s, int i, int j, int k) { return (size_t)i + (size_t)s->nx * (j + (size_t)s->nyv * k); }
static inline size_t IW(const orc_sim* s, int i, int j, int k) { return (size_t)i + (size_t)s->nx * (j + (size_t)s->ny * k); }
static inline size_t IP(const orc_sim* s, int i, int j, int k) { return (size_t)i + (size_t)s->nx * (j + (size_t)s->ny * k); }

// linear interpolation in y to face jf from centre values a (at jf-1) and b (at jf)   [O2]
static inline double interpY(const orc_sim* s, double a, double b, int jf) {
  double dm = DY(s, jf - 1), dp = DY(s, jf);
  return (dp * a + dm * b) / (dm + dp);
}

// ---- O2: momentum right-hand side H = -C + nu*Lap(u) + g -----------------------------------
// (Eq. 4: divergence form; central convection and diffusion, L100)
// Convection variant of L100 / Table 1 (L444-447), "first-order upwind" (reading N3-1): in every
// convective flux a*phi the advecting face velocity a keeps its central / linear interpolation and the
// transported value phi is the one on the upwind side of the face, phi = a > 0 ? phi_minus : phi_plus
// (ghost values come from the same boundary accessors as in the central scheme).
static inline double TR(const orc_sim* s, double a, double minus, double plus, double central) {
  return s->P.convection == ORC_CONV_UPWIND ? (a > 0.0 ? minus : plus) : central;
}
// ---- LES closures (NEXT-4; section 3.4.5) ---------------------------------------------
// Constant Smagorinsky model (reading N4-1): nu_t = (C_s Delta)^2 |S| at cell centres, Delta = (hx dy_j hz)^(1/3),
// |S| = sqrt(2 S_ij S_ij) with the diagonal gradients from the cell's own faces and the cross gradients as central
// differences of the face values averaged to the cell centres (ghost values from the O1 accessors).
static void eddy_viscosity(const orc_sim* s, const vec& uu, const vec& vv, const vec& ww, vec& nut) {
  const double hx = s->hx, hz = s->hz, cs = s->P.cs;
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i) {
    auto ux = [&](int jj, int kk) { return 0.5 * (U_(i, jj, kk) + U_(i + 1, jj, kk)); };     // u at the centres of column i
    auto vy = [&](int ii, int kk) { return 0.5 * (V_(ii, j, kk) + V_(ii, j + 1, kk)); };
    auto wz = [&](int ii, int jj) { return 0.5 * (W_(ii, jj, k) + W_(ii, jj, k + 1)); };
    const double dyc2 = DYC(s, j + 1) + DYC(s, j);                                           // y_c(j+1) - y_c(j-1)
    const double dudx = (U_(i + 1, j, k) - U_(i, j, k)) / hx, dvdy = (V_(i, j + 1, k) - V_(i, j, k)) / s->dy[j];
    const double dwdz = (W_(i, j, k + 1) - W_(i, j, k)) / hz;
    const double dudy = (ux(j + 1, k) - ux(j - 1, k)) / dyc2, dudz = (ux(j, k + 1) - ux(j, k - 1)) / (2.0 * hz);
    const double dvdx = (vy(i + 1, k) - vy(i - 1, k)) / (2.0 * hx), dvdz = (vy(i, k + 1) - vy(i, k - 1)) / (2.0 * hz);
    const double dwdx = (wz(i + 1, j) - wz(i - 1, j)) / (2.0 * hx), dwdy = (wz(i, j + 1) - wz(i, j - 1)) / dyc2;
    const double S2 = 2.0 * (dudx * dudx + dvdy * dvdy + dwdz * dwdz)
                    + (dudy + dvdx) * (dudy + dvdx) + (dudz + dwdx) * (dudz + dwdx) + (dvdz + dwdy) * (dvdz + dwdy);
    const double delta = std::cbrt(hx * s->dy[j] * hz);
    nut[IP(s, i, j, k)] = (cs * delta) * (cs * delta) * std::sqrt(S2);
  }
}
// nu_t of cell (i,j,k): wrapped in periodic directions, the boundary cell's value beyond a bounded end
static inline double NT(const orc_sim* s, const vec& nut, int i, int j, int k) {
  i = s->bx ? std::min(std::max(i, 0), s->nx - 1) : wrapi(i, s->nx);
  j = s->by ? std::min(std::max(j, 0), s->ny - 1) : wrapi(j, s->ny);
  k = s->bz ? std::min(std::max(k, 0), s->nz - 1) : wrapi(k, s->nz);
  return nut[IP(s, i, j, k)];
}
// Equilibrium wall model (Eq. 27, Spalding's law, kappa = 0.4, B = 5): friction velocity u_tau for the wall-parallel
// speed U at the distance y from the wall, by Newton-Raphson on
//   g(u_tau) = u+ + e^{-kappa B} [e^{kappa u+} - 1 - kappa u+ - (kappa u+)^2/2 - (kappa u+)^3/6] - y+,  u+ = U/u_tau, y+ = y u_tau/nu.
// g is convex and decreasing in u_tau, so Newton's iterates rise monotonically to the root from any start on its left
// (g >= 0).  Start: u+_0 = min( sqrt(Re_y), max(12.5, ln(1.182 Re_y) / kappa) ), Re_y = U y / nu = u+ y+ -- the viscous
// sublayer value (exact for small Re_y) capped by an upper bound of the root that follows from
// Re_y >= u+ e^{-kappa B} e^{kappa u+} / 2 for kappa u+ >= 5; both are >= the root's u+, i.e. u_tau,0 <= the root.
// A fixed 30 iterations (convergence is quadratic after two or three; no data-dependent exit).
extern "C" double orc_wall_utau(double U, double y, double nu) {
  if (!(U > 0.0)) return 0.0;
  const double kap = 0.4, eB = std::exp(-kap * 5.0);
  const double Rey = U * y / nu;
  const double up0 = std::min(std::sqrt(Rey), std::max(12.5, std::log(1.182 * Rey) / kap));
  double ut = U / up0;
  for (int it = 0; it < 30; ++it) {
    const double up = U / ut, yp = y * ut / nu, ku = kap * up, e = std::exp(ku);
    const double gval = up + eB * (e - 1.0 - ku - 0.5 * ku * ku - ku * ku * ku / 6.0) - yp;
    const double dgdup = 1.0 + eB * kap * (e - 1.0 - ku - 0.5 * ku * ku);
    const double dg = dgdup * (-up / ut) - y / nu;
    ut = ut - gval / dg;
  }
  return ut;
}
// Eq. 28-29: eddy viscosity that makes the wall flux of the tangential component `comp` (velocity rel, other tangential
// component other, both relative to the wall, at the first off-wall point, distance y) equal to the modelled stress:
//   tau_w = rho u_tau^2,  tau_wi = tau_w u_i / sqrt(u^2 + w^2),  nu_ti = (tau_wi / rho) / (du_i/dy + eps) - nu,  eps = 1e-6,
// with du_i/dy = u_i / y (the one-sided gradient the no-slip ghost value produces at the wall face).
static double wall_nut(const orc_sim* s, double rel, double other, double y) {
  const double U = std::sqrt(rel * rel + other * other);
  if (!(U > 0.0)) return 0.0;
  const double ut = orc_wall_utau(U, y, s->P.nu);
  const double tau_i = ut * ut * rel / U;                     // tau_wi / rho
  return tau_i / (rel / y + 1e-6) - s->P.nu;
}

static void momentum(const orc_sim* s, const vec& uu, const vec& vv, const vec& ww,
                     double nu, const double g[3], vec& HU, vec& HV, vec& HW) {
  const int nx = s->nx, ny = s->ny, nz = s->nz;
  const double hx = s->hx, hz = s->hz;
  std::fill(HU.begin(), HU.end(), 0.0); std::fill(HV.begin(), HV.end(), 0.0); std::fill(HW.begin(), HW.end(), 0.0);
  // LES: diffusive term div[(nu + nu_t) grad u_i] with nu_t at the flux locations (cell centres natively, edges as the
  // mean of the four surrounding cells); wall model: nu_t of Eq. 28 on the wall face of no-slip y walls (i = 1, 3)
  const bool les = nu > 0.0 && (s->P.cs > 0.0 || s->P.wall_model);
  vec nut;
  if (les) { nut.assign(s->p.size(), 0.0); if (s->P.cs > 0.0) eddy_viscosity(s, uu, vv, ww, nut); }
  auto Exy = [&](int i0, int i1, int j0, int j1, int k) { return 0.25 * (NT(s, nut, i0, j0, k) + NT(s, nut, i1, j0, k) + NT(s, nut, i0, j1, k) + NT(s, nut, i1, j1, k)); };
  auto Exz = [&](int i0, int i1, int j, int k0, int k1) { return 0.25 * (NT(s, nut, i0, j, k0) + NT(s, nut, i1, j, k0) + NT(s, nut, i0, j, k1) + NT(s, nut, i1, j, k1)); };
  auto Eyz = [&](int i, int j0, int j1, int k0, int k1) { return 0.25 * (NT(s, nut, i, j0, k0) + NT(s, nut, i, j1, k0) + NT(s, nut, i, j0, k1) + NT(s, nut, i, j1, k1)); };
  const bool wm_lo = les && s->P.wall_model && s->by && s->P.bc[2] == ORC_BC_NOSLIP;
  const bool wm_hi = les && s->P.wall_model && s->by && s->P.bc[3] == ORC_BC_NOSLIP;
  // u faces (boundary-normal faces i=0, nx of a bounded direction are prescribed, not advanced)
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = s->bx; i < nx; ++i) {
    double uc = U_(i, j, k);
    double ue = 0.5 * (uc + U_(i + 1, j, k)), uw = 0.5 * (U_(i - 1, j, k) + uc);
    double cx = (ue * TR(s, ue, uc, U_(i + 1, j, k), ue) - uw * TR(s, uw, U_(i - 1, j, k), uc, uw)) / hx;
    double vn = 0.5 * (V_(i - 1, j + 1, k) + V_(i, j + 1, k)), un = TR(s, vn, uc, U_(i, j + 1, k), interpY(s, uc, U_(i, j + 1, k), j + 1));
    double vs = 0.5 * (V_(i - 1, j, k) + V_(i, j, k)),         us = TR(s, vs, U_(i, j - 1, k), uc, interpY(s, U_(i, j - 1, k), uc, j));
    double cy = (vn * un - vs * us) / s->dy[j];
    double wt = 0.5 * (W_(i - 1, j, k + 1) + W_(i, j, k + 1)), ut = TR(s, wt, uc, U_(i, j, k + 1), 0.5 * (uc + U_(i, j, k + 1)));
    double wb = 0.5 * (W_(i - 1, j, k) + W_(i, j, k)),         ub = TR(s, wb, U_(i, j, k - 1), uc, 0.5 * (U_(i, j, k - 1) + uc));
    double cz = (wt * ut - wb * ub) / hz;
    double dxx = (U_(i + 1, j, k) - 2.0 * uc + U_(i - 1, j, k)) / (hx * hx);
    double dyy = ((U_(i, j + 1, k) - uc) / DYC(s, j + 1) - (uc - U_(i, j - 1, k)) / DYC(s, j)) / s->dy[j];
    double dzz = (U_(i, j, k + 1) - 2.0 * uc + U_(i, j, k - 1)) / (hz * hz);
    double visc = nu * (dxx + dyy + dzz);
    if (les) {
      const double fxe = (nu + NT(s, nut, i, j, k)) * (U_(i + 1, j, k) - uc) / hx, fxw = (nu + NT(s, nut, i - 1, j, k)) * (uc - U_(i - 1, j, k)) / hx;
      double nn = Exy(i - 1, i, j, j + 1, k), ns = Exy(i - 1, i, j - 1, j, k);
      if ((wm_lo && j == 0) || (wm_hi && j == ny - 1)) {          // Eq. 28: u is relative to the wall, w interpolated to the u face
        const int f = j == 0 ? 2 : 3;
        const double wf = 0.25 * (W_(i - 1, j, k) + W_(i, j, k) + W_(i - 1, j, k + 1) + W_(i, j, k + 1));
        const double nw = wall_nut(s, uc - s->P.bc_vel[f][0], wf - s->P.bc_vel[f][2], 0.5 * s->dy[j]);
        if (j == 0) ns = nw; else nn = nw;
      }
      const double fyn = (nu + nn) * (U_(i, j + 1, k) - uc) / DYC(s, j + 1), fys = (nu + ns) * (uc - U_(i, j - 1, k)) / DYC(s, j);
      const double fzt = (nu + Exz(i - 1, i, j, k, k + 1)) * (U_(i, j, k + 1) - uc) / hz, fzb = (nu + Exz(i - 1, i, j, k - 1, k)) * (uc - U_(i, j, k - 1)) / hz;
      visc = (fxe - fxw) / hx + (fyn - fys) / s->dy[j] + (fzt - fzb) / hz;
    }
    HU[IU(s, i, j, k)] = -(cx + cy + cz) + visc + g[0];
  }
  // v faces (control volume between y_c(j-1) and y_c(j), height DYC(j))
  for (int k = 0; k < nz; ++k) for (int j = s->by; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    double vc = V_(i, j, k);
    double ue = interpY(s, U_(i + 1, j - 1, k), U_(i + 1, j, k), j), ve = TR(s, ue, vc, V_(i + 1, j, k), 0.5 * (vc + V_(i + 1, j, k)));
    double uw = interpY(s, U_(i, j - 1, k), U_(i, j, k), j),         vw = TR(s, uw, V_(i - 1, j, k), vc, 0.5 * (V_(i - 1, j, k) + vc));
    double cx = (ue * ve - uw * vw) / hx;
    double vn = 0.5 * (vc + V_(i, j + 1, k)), vs = 0.5 * (V_(i, j - 1, k) + vc);
    double cy = (vn * TR(s, vn, vc, V_(i, j + 1, k), vn) - vs * TR(s, vs, V_(i, j - 1, k), vc, vs)) / DYC(s, j);
    double wt = interpY(s, W_(i, j - 1, k + 1), W_(i, j, k + 1), j), vt = TR(s, wt, vc, V_(i, j, k + 1), 0.5 * (vc + V_(i, j, k + 1)));
    double wb = interpY(s, W_(i, j - 1, k), W_(i, j, k), j),         vb = TR(s, wb, V_(i, j, k - 1), vc, 0.5 * (V_(i, j, k - 1) + vc));
    double cz = (wt * vt - wb * vb) / hz;
    double dxx = (V_(i + 1, j, k) - 2.0 * vc + V_(i - 1, j, k)) / (hx * hx);
    double dyy = ((V_(i, j + 1, k) - vc) / DY(s, j) - (vc - V_(i, j - 1, k)) / DY(s, j - 1)) / DYC(s, j);
    double dzz = (V_(i, j, k + 1) - 2.0 * vc + V_(i, j, k - 1)) / (hz * hz);
    double visc = nu * (dxx + dyy + dzz);
    if (les) {
      const double fxe = (nu + Exy(i, i + 1, j - 1, j, k)) * (V_(i + 1, j, k) - vc) / hx, fxw = (nu + Exy(i - 1, i, j - 1, j, k)) * (vc - V_(i - 1, j, k)) / hx;
      const double fyn = (nu + NT(s, nut, i, j, k)) * (V_(i, j + 1, k) - vc) / DY(s, j), fys = (nu + NT(s, nut, i, j - 1, k)) * (vc - V_(i, j - 1, k)) / DY(s, j - 1);
      const double fzt = (nu + Eyz(i, j - 1, j, k, k + 1)) * (V_(i, j, k + 1) - vc) / hz, fzb = (nu + Eyz(i, j - 1, j, k - 1, k)) * (vc - V_(i, j, k - 1)) / hz;
      visc = (fxe - fxw) / hx + (fyn - fys) / DYC(s, j) + (fzt - fzb) / hz;
    }
    HV[IV(s, i, j, k)] = -(cx + cy + cz) + visc + g[1];
  }
  // w faces
  for (int k = s->bz; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    double wc = W_(i, j, k);
    double ue = 0.5 * (U_(i + 1, j, k - 1) + U_(i + 1, j, k)), we = TR(s, ue, wc, W_(i + 1, j, k), 0.5 * (wc + W_(i + 1, j, k)));
    double uw = 0.5 * (U_(i, j, k - 1) + U_(i, j, k)),         wwst = TR(s, uw, W_(i - 1, j, k), wc, 0.5 * (W_(i - 1, j, k) + wc));
    double cx = (ue * we - uw * wwst) / hx;
    double vn = 0.5 * (V_(i, j + 1, k - 1) + V_(i, j + 1, k)), wn = TR(s, vn, wc, W_(i, j + 1, k), interpY(s, wc, W_(i, j + 1, k), j + 1));
    double vs = 0.5 * (V_(i, j, k - 1) + V_(i, j, k)),         ws = TR(s, vs, W_(i, j - 1, k), wc, interpY(s, W_(i, j - 1, k), wc, j));
    double cy = (vn * wn - vs * ws) / s->dy[j];
    double wt = 0.5 * (wc + W_(i, j, k + 1)), wb = 0.5 * (W_(i, j, k - 1) + wc);
    double cz = (wt * TR(s, wt, wc, W_(i, j, k + 1), wt) - wb * TR(s, wb, W_(i, j, k - 1), wc, wb)) / hz;
    double dxx = (W_(i + 1, j, k) - 2.0 * wc + W_(i - 1, j, k)) / (hx * hx);
    double dyy = ((W_(i, j + 1, k) - wc) / DYC(s, j + 1) - (wc - W_(i, j - 1, k)) / DYC(s, j)) / s->dy[j];
    double dzz = (W_(i, j, k + 1) - 2.0 * wc + W_(i, j, k - 1)) / (hz * hz);
    double visc = nu * (dxx + dyy + dzz);
    if (les) {
      const double fxe = (nu + Exz(i, i + 1, j, k - 1, k)) * (W_(i + 1, j, k) - wc) / hx, fxw = (nu + Exz(i - 1, i, j, k - 1, k)) * (wc - W_(i - 1, j, k)) / hx;
      double nn = Eyz(i, j, j + 1, k - 1, k), ns = Eyz(i, j - 1, j, k - 1, k);
      if ((wm_lo && j == 0) || (wm_hi && j == ny - 1)) {          // Eq. 28 for i = 3: u interpolated to the w face
        const int f = j == 0 ? 2 : 3;
        const double uf = 0.25 * (U_(i, j, k - 1) + U_(i + 1, j, k - 1) + U_(i, j, k) + U_(i + 1, j, k));
        const double nw = wall_nut(s, wc - s->P.bc_vel[f][2], uf - s->P.bc_vel[f][0], 0.5 * s->dy[j]);
        if (j == 0) ns = nw; else nn = nw;
      }
      const double fyn = (nu + nn) * (W_(i, j + 1, k) - wc) / DYC(s, j + 1), fys = (nu + ns) * (wc - W_(i, j - 1, k)) / DYC(s, j);
      const double fzt = (nu + NT(s, nut, i, j, k)) * (W_(i, j, k + 1) - wc) / hz, fzb = (nu + NT(s, nut, i, j, k - 1)) * (wc - W_(i, j, k - 1)) / hz;
      visc = (fxe - fxw) / hx + (fyn - fys) / s->dy[j] + (fzt - fzb) / hz;
    }
    HW[IW(s, i, j, k)] = -(cx + cy + cz) + visc + g[2];
  }
}

// ---- counter-based inflow noise (O1; the GPU path implements the same generator independently) --
static inline uint64_t sm64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
extern "C" double orc_inflow_rand(uint64_t seed, long long step, int face, int a, int b) {
  uint64_t h = sm64(seed + 0x632BE59BD9B4E019ULL * (uint64_t)(face + 1));
  h = sm64(h + (uint64_t)step);
  h = sm64(h + (((uint64_t)(uint32_t)b << 32) | (uint64_t)(uint32_t)a));
  return (double)(h >> 11) * (1.0 / 9007199254740992.0);   // [0,1), exact
}

// ---- O3 (boundary part): prescribed boundary-normal faces of the predicted field -------------
// us/vs/ws hold u~; un* hold u^n (needed by the convective outflow update).
static void set_boundary_normal(const orc_sim* s, vec& us, vec& vs, vec& ws,
                                const vec& un, const vec& vn, const vec& wn) {
  const int n[3] = {s->nx, s->ny, s->nz};
  const int bd[3] = {s->bx, s->by, s->bz};
  const double h[3] = {s->hx, s->hy, s->hz};
  for (int d = 0; d < 3; ++d) {
    if (!bd[d]) continue;
    vec& dst = d == 0 ? us : d == 1 ? vs : ws;
    const vec& old = d == 0 ? un : d == 1 ? vn : wn;
    int d1 = (d + 1) % 3, d2 = (d + 2) % 3;           // tangential directions
    if (d1 > d2) std::swap(d1, d2);                   // (a,b) = lower, higher axis
    for (int side = 0; side < 2; ++side) {
      int face = 2 * d + side, t = s->P.bc[face];
      int fidx = side ? n[d] : 0, inner = side ? n[d] - 1 : 1;
      double Ub = s->P.bc_vel[face][d];
      for (int b = 0; b < n[d2]; ++b) for (int a = 0; a < n[d1]; ++a) {
        int id[3], in[3]; id[d] = fidx; id[d1] = a; id[d2] = b; in[d] = inner; in[d1] = a; in[d2] = b;
        size_t q, qi;
        if (d == 0) { q = IU(s, id[0], id[1], id[2]); qi = IU(s, in[0], in[1], in[2]); }
        else if (d == 1) { q = IV(s, id[0], id[1], id[2]); qi = IV(s, in[0], in[1], in[2]); }
        else { q = IW(s, id[0], id[1], id[2]); qi = IW(s, in[0], in[1], in[2]); }
        double val;
        if (t == ORC_BC_NOSLIP) val = Ub;
        else if (t == ORC_BC_SLIP) val = 0.0;
        else if (t == ORC_BC_INFLOW) {
          double r = orc_inflow_rand(s->P.seed, s->step, face, a, b);
          val = Ub * (1.0 + s->P.inflow_noise * (2.0 * r - 1.0));
        } else {  // convective outflow (reading): d(u)/dt + Uc d(u)/dn = 0, first-order upwind
          double dn = d == 1 ? (side ? s->dy[s->ny - 1] : s->dy[0]) : h[d];
          double grad = side ? (old[q] - old[qi]) / dn : (old[qi] - old[q]) / dn;
          val = old[q] - Ub * s->dt * grad;
        }
        dst[q] = val;
      }
    }
  }
}

// ---- O4: IBM -----------------------------------------------------------------------------------
// 1-D kernels with h factored out.  Roma 3-point and the paper's 4-point Eq. 22 (L204).
extern "C" double orc_delta_phi(int kind, double r) {
  double a = std::fabs(r);
  if (kind == ORC_DELTA_ROMA3) {
    if (a <= 0.5) return (1.0 + std::sqrt(1.0 - 3.0 * a * a)) / 3.0;
    if (a <= 1.5) { double q = 1.0 - a; return (5.0 - 3.0 * a - std::sqrt(1.0 - 3.0 * q * q)) / 6.0; }
    return 0.0;
  }
  if (a <= 1.0) return (3.0 - 2.0 * a + std::sqrt(1.0 + 4.0 * a - 4.0 * a * a)) / 8.0;
  if (a <= 2.0) return (5.0 - 2.0 * a - std::sqrt(-7.0 + 12.0 * a - 4.0 * a * a)) / 8.0;
  return 0.0;
}

// node offset of component c along direction d: faces for d==c, centres otherwise
static inline double node_origin(const orc_sim* s, int c, int d) {
  const double o[3] = {s->P.x0, s->P.y0, s->P.z0}, h[3] = {s->hx, s->hy, s->hz};
  return d == c ? o[d] : o[d] + 0.5 * h[d];
}
static inline int support_width(const orc_sim* s) { return s->P.delta == ORC_DELTA_ROMA3 ? 3 : 4; }

// I-1: scaled coordinate and lowest support index (operations individually rounded; build uses
// -ffp-contract=off so no FMA is formed).
static inline double scaled_coord(const orc_sim* s, double X, int c, int d) {
  const double inv[3] = {1.0 / s->hx, 1.0 / s->hy, 1.0 / s->hz};
  double t = X - node_origin(s, c, d);
  return t * inv[d];
}
static inline int support_base(const orc_sim* s, double sc) {
  if (s->P.delta == ORC_DELTA_ROMA3) { double q = sc + 0.5; return (int)std::floor(q) - 1; }
  return (int)std::floor(sc) - 1;
}
// map a support node index to a storage index, or -1 if it must be skipped:
// periodic: wrap; bounded face-located: only interior faces 1..n-1; bounded centre-located: 0..n-1
static inline int node_index(const orc_sim* s, int m, int c, int d) {
  const int n[3] = {s->nx, s->ny, s->nz}; const int bd[3] = {s->bx, s->by, s->bz};
  if (!bd[d]) return wrapi(m, n[d]);
  if (d == c) return (m >= 1 && m <= n[d] - 1) ? m : -1;
  return (m >= 0 && m <= n[d] - 1) ? m : -1;
}

extern "C" void orc_ibm_index(orc_sim* s) {
  const int nl = s->nl;
  const int n[3] = {s->nx, s->ny, s->nz}; const int bd[3] = {s->bx, s->by, s->bz};
  const double o[3] = {s->P.x0, s->P.y0, s->P.z0};
  const double inv[3] = {1.0 / s->hx, 1.0 / s->hy, 1.0 / s->hz};
  s->base.assign((size_t)9 * nl, 0); s->keys.assign(nl, 0); s->perm.assign(nl, 0);
  std::vector<int> key_of(nl);
  for (int l = 0; l < nl; ++l) {
    for (int c = 0; c < 3; ++c) for (int d = 0; d < 3; ++d)
      s->base[((size_t)c * nl + l) * 3 + d] = support_base(s, scaled_coord(s, s->X[3 * l + d], c, d));
    // a support that reaches a non-periodic boundary is unsupported (the delta-kernel moment
    // identities P8-P10 do not hold for a truncated support); flagged here, reported by orc_set_markers / orc_step
    for (int c = 0; c < 3; ++c) for (int d = 0; d < 3; ++d) for (int a = 0; a < support_width(s); ++a)
      if (node_index(s, s->base[((size_t)c * nl + l) * 3 + d] + a, c, d) < 0) s->oob = true;
    int ic[3];
    for (int d = 0; d < 3; ++d) {
      double t = s->X[3 * l + d] - o[d];
      int q = (int)std::floor(t * inv[d]);
      ic[d] = bd[d] ? std::min(std::max(q, 0), n[d] - 1) : wrapi(q, n[d]);
    }
    key_of[l] = ic[0] + s->nx * (ic[1] + s->ny * ic[2]);
    s->perm[l] = l;
  }
  std::stable_sort(s->perm.begin(), s->perm.end(), [&](int a, int b) { return key_of[a] < key_of[b]; });
  s->seg.assign(nl + 1, 0); s->nseg = 0;
  for (int r = 0; r < nl; ++r) {
    s->keys[r] = key_of[s->perm[r]];
    if (r == 0 || s->keys[r] != s->keys[r - 1]) s->seg[s->nseg++] = r;
  }
  s->seg[s->nseg] = nl;
}

// weight of support node (a,b,cc) offsets for marker l / component c; returns storage index or -1
static inline long long ibm_node(const orc_sim* s, int l, int c, int a, int b, int cc, double* wgt) {
  int off[3] = {a, b, cc}, id[3]; double wt = 1.0;
  for (int d = 0; d < 3; ++d) {
    double sc = scaled_coord(s, s->X[3 * l + d], c, d);
    int m = s->base[((size_t)c * s->nl + l) * 3 + d] + off[d];
    double r = sc - (double)m;
    wt *= orc_delta_phi(s->P.delta, r);
    id[d] = node_index(s, m, c, d);
    if (id[d] < 0) return -1;
  }
  *wgt = wt;
  if (c == 0) return (long long)IU(s, id[0], id[1], id[2]);
  if (c == 1) return (long long)IV(s, id[0], id[1], id[2]);
  return (long long)IW(s, id[0], id[1], id[2]);
}

// I-2: U_l = sum_x u(x) delta_h(x - X_l) dv  = sum u * phi phi phi   (Eq. 3b / Eq. 20 operator)
static void interpolate(const orc_sim* s, const vec& us, const vec& vs, const vec& ws, vec& out) {
  const int sw = support_width(s);
  for (int l = 0; l < s->nl; ++l) for (int c = 0; c < 3; ++c) {
    const vec& f = c == 0 ? us : c == 1 ? vs : ws;
    double acc = 0.0;
    for (int cc = 0; cc < sw; ++cc) for (int b = 0; b < sw; ++b) for (int a = 0; a < sw; ++a) {
      double wt; long long q = ibm_node(s, l, c, a, b, cc, &wt);
      if (q >= 0) acc += f[(size_t)q] * wt;
    }
    out[3 * l + c] = acc;
  }
}
// I-4: f(x) += F_l delta_h(x - X_l) dV_l  (Eq. 3a), markers visited in cell-list (perm) order
static void spread(const orc_sim* s, const vec& F, vec& fu, vec& fv, vec& fw) {
  const int sw = support_width(s);
  const double ivol = 1.0 / (s->hx * s->hy * s->hz);
  for (int r = 0; r < s->nl; ++r) { int l = s->perm[r];
    for (int c = 0; c < 3; ++c) {
      vec& f = c == 0 ? fu : c == 1 ? fv : fw;
      for (int cc = 0; cc < sw; ++cc) for (int b = 0; b < sw; ++b) for (int a = 0; a < sw; ++a) {
        double wt; long long q = ibm_node(s, l, c, a, b, cc, &wt);
        if (q >= 0) f[(size_t)q] += F[3 * l + c] * wt * s->dV[l] * ivol;
      }
    }
  }
}

// ---- O5: outflow flux correction (reading; paper silent) ---------------------------------------
// net outward flux Phi through all boundary-normal faces is removed by a uniform shift of the
// outflow faces:  u_n(out) -= Phi / A_out.
static void flux_correction(const orc_sim* s, vec& us, vec& vs, vec& ws) {
  const int n[3] = {s->nx, s->ny, s->nz}; const int bd[3] = {s->bx, s->by, s->bz};
  double Phi = 0.0, Aout = 0.0; bool any = false;
  for (int pass = 0; pass < 2; ++pass) {
    for (int d = 0; d < 3; ++d) {
      if (!bd[d]) continue;
      vec& f = d == 0 ? us : d == 1 ? vs : ws;
      int d1 = (d + 1) % 3, d2 = (d + 2) % 3; if (d1 > d2) std::swap(d1, d2);
      for (int side = 0; side < 2; ++side) {
        int face = 2 * d + side; bool out = s->P.bc[face] == ORC_BC_OUTFLOW;
        double sgn = side ? 1.0 : -1.0;
        for (int b = 0; b < n[d2]; ++b) for (int a = 0; a < n[d1]; ++a) {
          int id[3]; id[d] = side ? n[d] : 0; id[d1] = a; id[d2] = b;
          double area = d == 0 ? s->dy[id[1]] * s->hz : d == 1 ? s->hx * s->hz : s->hx * s->dy[id[1]];
          size_t q = d == 0 ? IU(s, id[0], id[1], id[2]) : d == 1 ? IV(s, id[0], id[1], id[2]) : IW(s, id[0], id[1], id[2]);
          if (pass == 0) { Phi += sgn * f[q] * area; if (out) { Aout += area; any = true; } }
          else if (out) f[q] -= sgn * Phi / Aout;
        }
      }
    }
    if (!any) return;
  }
}

// ---- O6: staggered divergence, gradient, Laplacian -------------------------------------------
static void divergence(const orc_sim* s, const vec& uu, const vec& vv, const vec& ww, vec& out) {
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i) {
    double ue = uu[IU(s, s->bx ? i + 1 : wrapi(i + 1, s->nx), j, k)], uw = uu[IU(s, i, j, k)];
    double vn = vv[IV(s, i, s->by ? j + 1 : wrapi(j + 1, s->ny), k)], vs = vv[IV(s, i, j, k)];
    double wt = ww[IW(s, i, j, s->bz ? k + 1 : wrapi(k + 1, s->nz))], wb = ww[IW(s, i, j, k)];
    out[IP(s, i, j, k)] = (ue - uw) / s->hx + (vn - vs) / s->dy[j] + (wt - wb) / s->hz;
  }
}
// L p with the flux through every non-periodic boundary face dropped (homogeneous Neumann)
static void laplacian(const orc_sim* s, const double* p, double* out) {
  const int nx = s->nx, ny = s->ny, nz = s->nz;
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    double pc = p[IP(s, i, j, k)], acc = 0.0;
    if (!s->bx || i + 1 < nx) acc += (p[IP(s, wrapi(i + 1, nx), j, k)] - pc) / (s->hx * s->hx);
    if (!s->bx || i > 0)      acc -= (pc - p[IP(s, wrapi(i - 1, nx), j, k)]) / (s->hx * s->hx);
    double fy = 0.0;
    if (!s->by || j + 1 < ny) fy += (p[IP(s, i, wrapi(j + 1, ny), k)] - pc) / DYC(s, j + 1);
    if (!s->by || j > 0)      fy -= (pc - p[IP(s, i, wrapi(j - 1, ny), k)]) / DYC(s, j);
    acc += fy / s->dy[j];
    if (!s->bz || k + 1 < nz) acc += (p[IP(s, i, j, wrapi(k + 1, nz))] - pc) / (s->hz * s->hz);
    if (!s->bz || k > 0)      acc -= (pc - p[IP(s, i, j, wrapi(k - 1, nz))]) / (s->hz * s->hz);
    out[IP(s, i, j, k)] = acc;
  }
}
// A = -dy_j * L  (symmetric positive semi-definite, null space = constants)
static void apply_A(const orc_sim* s, const double* x, double* out) {
  laplacian(s, x, out);
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i)
    out[IP(s, i, j, k)] *= -s->dy[j];
}
static void jacobi_diag(const orc_sim* s, double* dg) {
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i) {
    double a = 0.0;
    if (!s->bx || i + 1 < s->nx) a += 1.0 / (s->hx * s->hx);
    if (!s->bx || i > 0)         a += 1.0 / (s->hx * s->hx);
    double fy = 0.0;
    if (!s->by || j + 1 < s->ny) fy += 1.0 / DYC(s, j + 1);
    if (!s->by || j > 0)         fy += 1.0 / DYC(s, j);
    a += fy / s->dy[j];
    if (!s->bz || k + 1 < s->nz) a += 1.0 / (s->hz * s->hz);
    if (!s->bz || k > 0)         a += 1.0 / (s->hz * s->hz);
    dg[IP(s, i, j, k)] = a * s->dy[j];
  }
}

// ---- O7g: geometric multigrid V-cycle on (-L) e = g, uniform isotropic grids -----------------------------------
// level arrays are nx x ny x nz-shaped with spacing h; operator rediscretised on every level.  bd[d] != 0: direction d is
// bounded -- the flux through a boundary face is dropped (homogeneous Neumann, as in the fine operator O6), so a cell has
// nnb <= 6 neighbours and the diagonal is nnb / h^2 (reading G1 in DESIGN.md 3: SURVEY O7g names triply periodic boxes
// only; restriction, prolongation and the damped-Jacobi smoother with the TRUE diagonal carry over unchanged, and the
// cycle stays a symmetric operator).  All periodic: nnb = 6 everywhere, the original formulas bit for bit.
static inline double mg_nnb(int nx, int ny, int nz, const int bd[3], int i, int j, int k) {
  double n = 6.0;
  if (bd[0]) n -= (i == 0) + (i == nx - 1);
  if (bd[1]) n -= (j == 0) + (j == ny - 1);
  if (bd[2]) n -= (k == 0) + (k == nz - 1);
  return n;
}
static void mg_neg_lap(int nx, int ny, int nz, double h, const int bd[3], const vec& e, vec& out) {
  double ih2 = 1.0 / (h * h);
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t c = (size_t)i + (size_t)nx * (j + (size_t)ny * k);
    auto at = [&](int ii, int jj, int kk) -> double {          // neighbour value; 0 beyond a bounded end (counted out by nnb)
      if (bd[0] ? (ii < 0 || ii >= nx) : false) return 0.0;
      if (bd[1] ? (jj < 0 || jj >= ny) : false) return 0.0;
      if (bd[2] ? (kk < 0 || kk >= nz) : false) return 0.0;
      return e[(size_t)wrapi(ii, nx) + (size_t)nx * (wrapi(jj, ny) + (size_t)ny * wrapi(kk, nz))];
    };
    double nb = at(i + 1, j, k) + at(i - 1, j, k) + at(i, j + 1, k) + at(i, j - 1, k) + at(i, j, k + 1) + at(i, j, k - 1);
    out[c] = (mg_nnb(nx, ny, nz, bd, i, j, k) * e[c] - nb) * ih2;
  }
}
// one damped-Jacobi sweep  e <- e + omega D^-1 (g - (-L) e),  D = nnb/h^2
static void mg_sweep(int nx, int ny, int nz, double h, double omega, const int bd[3], const vec& g, vec& e, vec& tmp, bool zero_guess) {
  if (!zero_guess) mg_neg_lap(nx, ny, nz, h, bd, e, tmp);
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t q = (size_t)i + (size_t)nx * (j + (size_t)ny * k);
    double c = omega * h * h / mg_nnb(nx, ny, nz, bd, i, j, k);
    e[q] = zero_guess ? c * g[q] : e[q] + c * (g[q] - tmp[q]);
  }
}
static int mg_levels(int nx, int ny, int nz) {
  int L = 1;
  while (nx % 2 == 0 && ny % 2 == 0 && nz % 2 == 0 && std::min(nx, std::min(ny, nz)) / 2 >= 4) { nx /= 2; ny /= 2; nz /= 2; ++L; }
  return L;
}
static void mg_vcycle(const orc_sim* s, int lev, int nx, int ny, int nz, double h, const vec& g, vec& e) {
  size_t N = (size_t)nx * ny * nz; vec tmp(N);
  const int bd[3] = {s->bx, s->by, s->bz};
  e.assign(N, 0.0);
  if (lev == s->nlev - 1) {                                    // coarsest: fixed sweeps from zero
    for (int it = 0; it < s->P.mg_coarse_sweeps; ++it) mg_sweep(nx, ny, nz, h, s->P.mg_omega, bd, g, e, tmp, it == 0);
    return;
  }
  for (int it = 0; it < s->P.mg_nu1; ++it) mg_sweep(nx, ny, nz, h, s->P.mg_omega, bd, g, e, tmp, it == 0);
  vec res(N);
  if (s->P.mg_nu1 > 0) { mg_neg_lap(nx, ny, nz, h, bd, e, tmp); for (size_t q = 0; q < N; ++q) res[q] = g[q] - tmp[q]; }
  else res = g;
  int cx = nx / 2, cy = ny / 2, cz = nz / 2; size_t Nc = (size_t)cx * cy * cz;
  vec gc(Nc), ec;
  for (int k = 0; k < cz; ++k) for (int j = 0; j < cy; ++j) for (int i = 0; i < cx; ++i) {   // restriction: mean of 8 children
    double a = 0.0;
    for (int dk = 0; dk < 2; ++dk) for (int dj = 0; dj < 2; ++dj) for (int di = 0; di < 2; ++di)
      a += res[(size_t)(2 * i + di) + (size_t)nx * ((2 * j + dj) + (size_t)ny * (2 * k + dk))];
    gc[(size_t)i + (size_t)cx * (j + (size_t)cy * k)] = 0.125 * a;
  }
  mg_vcycle(s, lev + 1, cx, cy, cz, 2.0 * h, gc, ec);
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i)      // piecewise-constant prolongation
    e[(size_t)i + (size_t)nx * (j + (size_t)ny * k)] += ec[(size_t)(i / 2) + (size_t)cx * ((j / 2) + (size_t)cy * (k / 2))];
  for (int it = 0; it < s->P.mg_nu2; ++it) mg_sweep(nx, ny, nz, h, s->P.mg_omega, bd, g, e, tmp, false);
}
// z = M^-1 r : A = -h L = h(-L)  =>  z = Vcycle(r / h)
static void precond_gmg(const orc_sim* s, const vec& r, vec& z) {
  vec g(r.size());
  for (size_t q = 0; q < r.size(); ++q) g[q] = r[q] / s->hy;
  mg_vcycle(s, 0, s->nx, s->ny, s->nz, s->hx, g, z);
}

// ---- O7: preconditioned conjugate gradients (textbook Hestenes-Stiefel) -----------------------
static double dot(const vec& a, const vec& b) { double t = 0.0; for (size_t q = 0; q < a.size(); ++q) t += a[q] * b[q]; return t; }
static void apply_precond(const orc_sim* s, const vec& dg, const vec& r, vec& z) {
  if (s->P.precond == ORC_PC_NONE) z = r;
  else if (s->P.precond == ORC_PC_JACOBI) { for (size_t q = 0; q < r.size(); ++q) z[q] = r[q] / dg[q]; }
  else precond_gmg(s, r, z);
}
// solves A x = bh (bh already compatible); x holds the initial guess
static void pcg(const orc_sim* s, const vec& bh, vec& x, orc_info* info) {
  size_t N = bh.size(); vec r(N), z(N), d(N), q(N), dg;
  if (s->P.precond == ORC_PC_JACOBI) { dg.resize(N); jacobi_diag(s, dg.data()); }
  apply_A(s, x.data(), q.data());
  for (size_t i = 0; i < N; ++i) r[i] = bh[i] - q[i];
  double bnorm = std::sqrt(dot(bh, bh)), rnorm = std::sqrt(dot(r, r));
  int it = 0, conv = 0;
  if (bnorm == 0.0 || rnorm <= s->P.rtol * bnorm) conv = 1;
  else {
    apply_precond(s, dg, r, z); d = z; double rho = dot(r, z);
    for (it = 1; it <= s->P.max_iter; ++it) {
      apply_A(s, d.data(), q.data());
      double alpha = rho / dot(d, q);
      for (size_t i = 0; i < N; ++i) x[i] += alpha * d[i];
      for (size_t i = 0; i < N; ++i) r[i] -= alpha * q[i];
      rnorm = std::sqrt(dot(r, r));
      if (rnorm <= s->P.rtol * bnorm) { conv = 1; break; }
      if (it == s->P.max_iter) break;
      apply_precond(s, dg, r, z);
      double rho2 = dot(r, z), beta = rho2 / rho;
      for (size_t i = 0; i < N; ++i) d[i] = z[i] + beta * d[i];
      rho = rho2;
    }
  }
  info->pcg_iters = it > s->P.max_iter ? s->P.max_iter : it; info->converged = conv;
  info->rel_residual = bnorm > 0.0 ? rnorm / bnorm : 0.0;
  apply_A(s, x.data(), q.data());
  double t = 0.0; for (size_t i = 0; i < N; ++i) { double e = bh[i] - q[i]; t += e * e; }
  info->true_rel_residual = bnorm > 0.0 ? std::sqrt(t) / bnorm : 0.0;
}
// O6: rhs = Laplacian right-hand side b (Eq. 7);  solves L p = b  as  A p = -dy*b, zero-mean p
static void poisson(const orc_sim* s, const vec& b, vec& p, orc_info* info) {
  size_t N = b.size(); vec bh(N);
  double sb = 0.0, sd = 0.0;
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i) {
    size_t q = IP(s, i, j, k); bh[q] = -s->dy[j] * b[q]; sb += bh[q]; sd += s->dy[j];
  }
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i)
    bh[IP(s, i, j, k)] -= (sb / sd) * s->dy[j];
  if (!s->P.warm_start) std::fill(p.begin(), p.end(), 0.0);
  pcg(s, bh, p, info);
  double sp = 0.0;
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i) sp += p[IP(s, i, j, k)] * s->dy[j];
  double mean = sp / sd;
  for (size_t q = 0; q < N; ++q) p[q] -= mean;
}

// ---- O8: projection  u = u* - (dt/rho) G p  at non-boundary faces (Eq. 10) ---------------
static void gradient(const orc_sim* s, const vec& p, vec& gu, vec& gv, vec& gw) {
  std::fill(gu.begin(), gu.end(), 0.0); std::fill(gv.begin(), gv.end(), 0.0); std::fill(gw.begin(), gw.end(), 0.0);
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = s->bx; i < s->nx; ++i)
    gu[IU(s, i, j, k)] = (p[IP(s, i, j, k)] - p[IP(s, wrapi(i - 1, s->nx), j, k)]) / s->hx;
  for (int k = 0; k < s->nz; ++k) for (int j = s->by; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i)
    gv[IV(s, i, j, k)] = (p[IP(s, i, j, k)] - p[IP(s, i, wrapi(j - 1, s->ny), k)]) / DYC(s, j);
  for (int k = s->bz; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i)
    gw[IW(s, i, j, k)] = (p[IP(s, i, j, k)] - p[IP(s, i, j, wrapi(k - 1, s->nz))]) / s->hz;
}

// ---- O9: rigid body, one classical RK4 step of  m w'' + c w' + k w = F  (Eq. 12), F frozen ------
extern "C" void orc_rk4_body(double m, double c, double k, double F, double dt, double* w, double* wd) {
  double y0 = *w, y1 = *wd;
  #define ACC(a, b) ((F - c * (b) - k * (a)) / m)
  double k1a = y1,                   k1b = ACC(y0, y1);
  double k2a = y1 + 0.5 * dt * k1b,  k2b = ACC(y0 + 0.5 * dt * k1a, y1 + 0.5 * dt * k1b);
  double k3a = y1 + 0.5 * dt * k2b,  k3b = ACC(y0 + 0.5 * dt * k2a, y1 + 0.5 * dt * k2b);
  double k4a = y1 + dt * k3b,        k4b = ACC(y0 + dt * k3a, y1 + dt * k3b);
  #undef ACC
  *w  = y0 + dt / 6.0 * (k1a + 2.0 * k2a + 2.0 * k3a + k4a);
  *wd = y1 + dt / 6.0 * (k1b + 2.0 * k2b + 2.0 * k3b + k4b);
}

// ---- O4': the paper-literal eps-mask direct forcing (NEXT-1) -------------------------
// Reading E1.  eps is given per pressure cell (1 in solid cells, 0 in fluid cells, L110).  A velocity
// face belongs to the solid when either of the two cells it separates is solid (its control volume intersects the
// immersed region, L106); prescribed boundary-normal faces are never forced.  IB points (L74): fluid faces with at
// least one of their six same-component neighbours in the solid.
static inline int mask_cell(const orc_sim* s, int i, int j, int k) {
  const int n[3] = {s->nx, s->ny, s->nz}; const int bd[3] = {s->bx, s->by, s->bz}; int id[3] = {i, j, k};
  for (int d = 0; d < 3; ++d) { if (bd[d]) { if (id[d] < 0 || id[d] >= n[d]) return 0; } else id[d] = wrapi(id[d], n[d]); }
  return s->eps[IP(s, id[0], id[1], id[2])] ? 1 : 0;
}
static void build_face_masks(orc_sim* s) {
  const int n[3] = {s->nx, s->ny, s->nz}; const int bd[3] = {s->bx, s->by, s->bz};
  std::vector<unsigned char>* M[3] = {&s->mu, &s->mv, &s->mw};
  const size_t sz[3] = {s->u.size(), s->v.size(), s->w.size()};
  for (int c = 0; c < 3; ++c) {
    M[c]->assign(sz[c], 0);
    const int e[3] = {n[0] + (c == 0 ? bd[0] : 0), n[1] + (c == 1 ? bd[1] : 0), n[2] + (c == 2 ? bd[2] : 0)};
    auto idx = [&](int i, int j, int k) { return (size_t)i + (size_t)e[0] * (j + (size_t)e[1] * k); };
    auto solid = [&](int i, int j, int k) -> int {            // face (i,j,k) of component c: outside the box / prescribed -> 0
      int id[3] = {i, j, k};
      for (int d = 0; d < 3; ++d) {
        if (!bd[d]) { id[d] = wrapi(id[d], n[d]); continue; }
        if (d == c) { if (id[d] <= 0 || id[d] >= n[d]) return 0; }
        else if (id[d] < 0 || id[d] >= n[d]) return 0;
      }
      int lo[3] = {id[0], id[1], id[2]}; lo[c] -= 1;
      return (mask_cell(s, id[0], id[1], id[2]) || mask_cell(s, lo[0], lo[1], lo[2])) ? 1 : 0;
    };
    for (int k = 0; k < e[2]; ++k) for (int j = 0; j < e[1]; ++j) for (int i = 0; i < e[0]; ++i) {
      const int id[3] = {i, j, k};
      if (bd[c] && (id[c] == 0 || id[c] == n[c])) continue;   // prescribed boundary-normal face
      if (solid(i, j, k)) { (*M[c])[idx(i, j, k)] = 1; continue; }
      if (solid(i + 1, j, k) || solid(i - 1, j, k) || solid(i, j + 1, k) || solid(i, j - 1, k) || solid(i, j, k + 1) || solid(i, j, k - 1))
        (*M[c])[idx(i, j, k)] = 2;
    }
  }
}
// Eq. 18-19: velocity at the IB points from the structure's markers with the half-distribution normalisation,
//   u_IB(x) = sum_i (1 / F_Ni) wdot(X_i) delta_h(x - X_i) dV_i,   F_Ni = sum_{x in gamma'} delta_h(x - X_i) dv(x)
// gamma' = the nodes of marker i's support that are NOT in the solid (Eq. 19 as printed has no dv: it would carry units
// of 1 / volume); a marker whose support holds no such node contributes nothing.
static void ib_point_velocity(orc_sim* s, vec& fu, vec& fv, vec& fw) {
  const int sw = support_width(s);
  vec G((size_t)3 * s->nl, 0.0);
  for (int l = 0; l < s->nl; ++l) for (int c = 0; c < 3; ++c) {
    const std::vector<unsigned char>& m = c == 0 ? s->mu : c == 1 ? s->mv : s->mw;
    double FN = 0.0;
    for (int cc = 0; cc < sw; ++cc) for (int b = 0; b < sw; ++b) for (int a = 0; a < sw; ++a) {
      double wt; long long q = ibm_node(s, l, c, a, b, cc, &wt);
      if (q >= 0 && m[(size_t)q] != 1) FN += wt;
    }
    G[3 * l + c] = FN > 0.0 ? s->Ub[3 * l + c] / FN : 0.0;
  }
  spread(s, G, fu, fv, fw);
  s->Fl = G;                              // reported as the markers' "force" array: wdot_i / F_Ni
}
// Eq. 4 + Eq. 5: with f = eps [ -(explicit right-hand side) + (u_s - u^t) / dt ] the predictor becomes
//   u* = (1 - eps) u~ + eps u_s,   u_s = u_c in the solid (Eq. 23, third branch), u_IB at the IB points (second branch,
// only when markers carry the structure's velocity).  Returns the force on the body, -rho sum_x f(x) dv (Eq. 20 summed).
static void mask_forcing(orc_sim* s, vec& us, vec& vs, vec& ws) {
  const double dt = s->dt, rho = s->P.rho, dv = s->hx * s->hy * s->hz;
  double uc[3]; for (int c = 0; c < 3; ++c) uc[c] = s->has_body ? s->bvel[c] : s->uc[c];
  vec ib[3];
  const bool with_ib = s->nl > 0;
  if (with_ib) {
    orc_ibm_index(s);
    ib[0].assign(us.size(), 0.0); ib[1].assign(vs.size(), 0.0); ib[2].assign(ws.size(), 0.0);
    ib_point_velocity(s, ib[0], ib[1], ib[2]);
  }
  vec* F[3] = {&us, &vs, &ws};
  const std::vector<unsigned char>* M[3] = {&s->mu, &s->mv, &s->mw};
  for (int c = 0; c < 3; ++c) {
    double acc = 0.0;
    for (size_t q = 0; q < F[c]->size(); ++q) {
      const int m = (*M[c])[q];
      if (m == 0 || (m == 2 && !with_ib)) continue;
      const double target = m == 1 ? uc[c] : ib[c][q];
      acc += (target - (*F[c])[q]) / dt * dv;                 // f dv
      (*F[c])[q] = target;
    }
    s->bforce[c] = -rho * acc;
  }
}
// Eq. 9: the field whose divergence drives the Poisson equation, (1 - eps) u* + eps u_c.
static void poisson_source_field(const orc_sim* s, vec& us, vec& vs, vec& ws) {
  double uc[3]; for (int c = 0; c < 3; ++c) uc[c] = s->has_body ? s->bvel[c] : s->uc[c];
  vec* F[3] = {&us, &vs, &ws};
  const std::vector<unsigned char>* M[3] = {&s->mu, &s->mv, &s->mw};
  for (int c = 0; c < 3; ++c) for (size_t q = 0; q < F[c]->size(); ++q) {
    const double e = (*M[c])[q] == 1 ? 1.0 : 0.0;
    (*F[c])[q] = (1.0 - e) * (*F[c])[q] + e * uc[c];
  }
}

// ---- O1..O5: the predicted field ----------------------------------------------------------------
// upto = 0: after O3 (explicit predictor + prescribed boundary-normal faces), 1: after O4 (IBM direct forcing),
// 2: after O5 (outflow flux correction).  one_step uses upto = 2; orc_predict exposes the intermediate stages so the
// tests can pin O1 (convective outflow), I-3/I-4 (forcing scale) and O5 (uniform shift) one by one.
static void predictor(orc_sim* s, int upto, vec& us, vec& vs, vec& ws, vec& HU, vec& HV, vec& HW) {
  const double dt = s->dt, rho = s->P.rho;
  momentum(s, s->u, s->v, s->w, s->P.nu, s->P.body_force, HU, HV, HW);                 // O1+O2
  double a0 = 1.0, a1 = 0.0;
  // AB2 with the step-size ratio r = dt_n / dt_{n-1} (CFL-adaptive dt, L431): a0 = 1 + r/2, a1 = -r/2; r = 1 exactly for
  // a fixed step, i.e. (3/2, -1/2).  Euler and the stages of the Runge-Kutta scheme use (1, 0) = Eq. 4 as printed.
  if (s->P.time_scheme == ORC_TIME_AB2 && s->have_hist) { const double r = dt / s->dt_prev; a0 = 1.0 + 0.5 * r; a1 = -0.5 * r; }
  us = s->u; vs = s->v; ws = s->w;                                                     // O3
  for (int k = 0; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = s->bx; i < s->nx; ++i) {
    size_t q = IU(s, i, j, k); us[q] = s->u[q] + dt * (a0 * HU[q] + a1 * s->hu[q]); }
  for (int k = 0; k < s->nz; ++k) for (int j = s->by; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i) {
    size_t q = IV(s, i, j, k); vs[q] = s->v[q] + dt * (a0 * HV[q] + a1 * s->hv[q]); }
  for (int k = s->bz; k < s->nz; ++k) for (int j = 0; j < s->ny; ++j) for (int i = 0; i < s->nx; ++i) {
    size_t q = IW(s, i, j, k); ws[q] = s->w[q] + dt * (a0 * HW[q] + a1 * s->hw[q]); }
  set_boundary_normal(s, us, vs, ws, s->u, s->v, s->w);
  for (int c = 0; c < 3; ++c) s->bforce[c] = 0.0;
  if (upto < 1) return;
  if (s->has_mask) mask_forcing(s, us, vs, ws);                                        // O4' (eps-mask IBM, Eq. 4-5, 18-19, 23)
  else if (s->nl > 0) {                                                                // O4
    orc_ibm_index(s);                                                                  // I-1
    interpolate(s, us, vs, ws, s->Ul);                                                 // I-2
    for (int l = 0; l < s->nl; ++l) for (int c = 0; c < 3; ++c)                        // I-3 (Eq. 5 at markers)
      s->Fl[3 * l + c] = (s->Ub[3 * l + c] - s->Ul[3 * l + c]) / dt;
    for (int l = 0; l < s->nl; ++l) for (int c = 0; c < 3; ++c) s->bforce[c] += s->Fl[3 * l + c] * s->dV[l];
    for (int c = 0; c < 3; ++c) s->bforce[c] *= -rho;
    vec fu(us.size(), 0.0), fv(vs.size(), 0.0), fw(ws.size(), 0.0);
    spread(s, s->Fl, fu, fv, fw);                                                      // I-4
    for (size_t q = 0; q < us.size(); ++q) us[q] += dt * fu[q];
    for (size_t q = 0; q < vs.size(); ++q) vs[q] += dt * fv[q];
    for (size_t q = 0; q < ws.size(); ++q) ws[q] += dt * fw[q];
  }
  if (upto < 2) return;
  flux_correction(s, us, vs, ws);                                                      // O5
}

// ---- the fluid part of one fractional step (O1..O8) from the current u, v, w, p with step size s->dt ---------------
static void fluid_substep(orc_sim* s, orc_info* info, vec& HU, vec& HV, vec& HW) {
  const double dt = s->dt, rho = s->P.rho;
  vec us, vs, ws;
  predictor(s, 2, us, vs, ws, HU, HV, HW);                                             // O1..O5
  if (s->has_mask) poisson_source_field(s, us, vs, ws);                                // Eq. 9 (Eq. 7 when eps = 0, L129)
  vec b(s->p.size());
  divergence(s, us, vs, ws, b);                                                        // O6
  for (size_t q = 0; q < b.size(); ++q) b[q] *= rho / dt;
  poisson(s, b, s->p, info);                                                           // O7
  vec gu(us.size()), gv(vs.size()), gw(ws.size());
  gradient(s, s->p, gu, gv, gw);                                                       // O8
  for (size_t q = 0; q < us.size(); ++q) s->u[q] = us[q] - dt / rho * gu[q];
  for (size_t q = 0; q < vs.size(); ++q) s->v[q] = vs[q] - dt / rho * gv[q];
  for (size_t q = 0; q < ws.size(); ++q) s->w[q] = ws[q] - dt / rho * gw[q];
}

// CFL-adaptive step size ("governed by the CFL condition based on the instantaneous maximum velocity";
// reading N3-2): dt = min(dt_max, CFL h_min / max(|u|, |v|, |w|)) over all stored faces at time level n, with
// dt_max = the configured dt and h_min the smallest cell extent.  cfl <= 0: fixed dt.
static double choose_dt(const orc_sim* s) {
  if (!(s->P.cfl > 0.0)) return s->P.dt;
  double umax = 0.0;
  for (double x : s->u) umax = std::max(umax, std::fabs(x));
  for (double x : s->v) umax = std::max(umax, std::fabs(x));
  for (double x : s->w) umax = std::max(umax, std::fabs(x));
  double hmin = std::min(s->hx, s->hz);
  for (double d : s->dy) hmin = std::min(hmin, d);
  if (!(umax > 0.0)) return s->P.dt;
  return std::min(s->P.dt, s->P.cfl * hmin / umax);
}

// ---- flexible beam (NEXT-2; Eq. 11, Eq. 13-17, Newmark-beta L177, Table 1) -------------------
// Reading N2-2.  A straight beam of nb nodes in the x-y plane, clamped at node 0 (both flexible benchmarks
// of section 3.3 are clamped plates, L544, L560).  "Only bending deformations are considered, and axial or shear effects
// are neglected" (L149): every free node carries the two degrees of freedom of the 4 x 4 element matrices of Eq. 13-14,
// the deflection w along the fixed normal n of the reference axis and the rotation theta; there is no axial motion.
// Markers sit at the nodes (any number per node, e.g. one per span plane): X_l = X_l^ref + w_node n, U^b_l = wdot_node n.
// Load: Q_w,i = n . q_i with q_i = -rho sum_{l in node i} F_l dV_l (Eq. 20 gathered per node), no nodal moments.
// Damping: C = alpha M + beta K (Eq. 15) with alpha, beta from the two LOWEST modal frequencies of Eq. 17 (Eq. 16).
// Time integration: Newmark-beta in its unconditionally stable second-order form (average acceleration, gamma = 1/2,
// beta_N = 1/4), started from rest with zero acceleration.

// Solves the dense n x n system A x = b by Gaussian elimination with partial pivoting (A and b by value: overwritten).
static vec dense_solve(vec A, vec b, int n) {
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r) if (std::fabs(A[(size_t)r * n + c]) > std::fabs(A[(size_t)piv * n + c])) piv = r;
    if (piv != c) { for (int k = 0; k < n; ++k) std::swap(A[(size_t)c * n + k], A[(size_t)piv * n + k]); std::swap(b[c], b[piv]); }
    for (int r = c + 1; r < n; ++r) {
      const double f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
      for (int k = c; k < n; ++k) A[(size_t)r * n + k] -= f * A[(size_t)c * n + k];
      b[r] -= f * b[c];
    }
  }
  vec x(n);
  for (int r = n - 1; r >= 0; --r) {
    double t = b[r];
    for (int k = r + 1; k < n; ++k) t -= A[(size_t)r * n + k] * x[k];
    x[r] = t / A[(size_t)r * n + r];
  }
  return x;
}
static vec matvec(const vec& A, const vec& x, int n) {
  vec y(n, 0.0);
  for (int r = 0; r < n; ++r) { double t = 0.0; for (int k = 0; k < n; ++k) t += A[(size_t)r * n + k] * x[k]; y[r] = t; }
  return y;
}
static double dotv(const vec& a, const vec& b) { double t = 0.0; for (size_t i = 0; i < a.size(); ++i) t += a[i] * b[i]; return t; }

// Assembles K and M from the element matrices of Eq. 13 and Eq. 14 (local DOF order: w_i, theta_i, w_{i+1}, theta_{i+1}),
// drops the clamped node's rows and columns, finds omega_1, omega_2 of Eq. 17 by inverse iteration (x <- K^-1 M x, the
// second vector kept M-orthogonal to the first) and builds C by Eq. 15-16.
static void beam_assemble(orc_sim* s) {
  const int nb = s->nb, nfull = 2 * nb, n = s->ndof;
  vec Kf((size_t)nfull * nfull, 0.0), Mf((size_t)nfull * nfull, 0.0);
  for (int e = 0; e + 1 < nb; ++e) {
    const double dx = s->bX0[2 * (e + 1)] - s->bX0[2 * e], dy = s->bX0[2 * (e + 1) + 1] - s->bX0[2 * e + 1];
    const double L = std::sqrt(dx * dx + dy * dy);
    const double ke[4][4] = {{12, 6 * L, -12, 6 * L}, {6 * L, 4 * L * L, -6 * L, 2 * L * L}, {-12, -6 * L, 12, -6 * L}, {6 * L, 2 * L * L, -6 * L, 4 * L * L}};
    const double me[4][4] = {{156, 22 * L, 54, -13 * L}, {22 * L, 4 * L * L, 13 * L, -3 * L * L}, {54, 13 * L, 156, -22 * L}, {-13 * L, -3 * L * L, -22 * L, 4 * L * L}};
    const double kf = s->EI / (L * L * L), mf = s->mus * L / 420.0;
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
      Kf[(size_t)(2 * e + a) * nfull + (2 * e + b)] += kf * ke[a][b];
      Mf[(size_t)(2 * e + a) * nfull + (2 * e + b)] += mf * me[a][b];
    }
  }
  s->BK.assign((size_t)n * n, 0.0); s->BM.assign((size_t)n * n, 0.0);
  for (int r = 0; r < n; ++r) for (int c = 0; c < n; ++c) {
    s->BK[(size_t)r * n + c] = Kf[(size_t)(r + 2) * nfull + (c + 2)];
    s->BM[(size_t)r * n + c] = Mf[(size_t)(r + 2) * nfull + (c + 2)];
  }
  vec phi[2]; double lam[2] = {0.0, 0.0};
  for (int m = 0; m < 2 && m < n; ++m) {
    vec x(n);
    for (int i = 0; i < n; ++i) x[i] = 1.0 + 0.37 * i + (m ? ((i / 2) % 2 ? -1.0 : 1.0) : 0.0);   // any start with a component along the mode
    for (int it = 0; it < 400; ++it) {
      if (m == 1) { const double c0 = dotv(phi[0], matvec(s->BM, x, n)); for (int i = 0; i < n; ++i) x[i] -= c0 * phi[0][i]; }
      x = dense_solve(s->BK, matvec(s->BM, x, n), n);
      if (m == 1) { const double c0 = dotv(phi[0], matvec(s->BM, x, n)); for (int i = 0; i < n; ++i) x[i] -= c0 * phi[0][i]; }
      const double nm = std::sqrt(dotv(x, matvec(s->BM, x, n)));
      for (int i = 0; i < n; ++i) x[i] /= nm;
    }
    lam[m] = dotv(x, matvec(s->BK, x, n)) / dotv(x, matvec(s->BM, x, n));      // Rayleigh quotient = omega^2
    phi[m] = x;
  }
  s->om1 = std::sqrt(lam[0]); s->om2 = std::sqrt(lam[1]);
  s->ralpha = 2.0 * s->zeta * s->om1 * s->om2 / (s->om1 + s->om2);              // Eq. 16
  s->rbeta = 2.0 * s->zeta / (s->om1 + s->om2);
  s->BC.assign((size_t)n * n, 0.0);
  for (size_t q = 0; q < s->BC.size(); ++q) s->BC[q] = s->ralpha * s->BM[q] + s->rbeta * s->BK[q];   // Eq. 15
}

// One Newmark-beta step (gamma = 1/2, beta_N = 1/4) of M a + C v + K w = Q from (w, v, a) with the load Q at the new time.
static void beam_newmark(const orc_sim* s, const vec& Q, double dt, vec& w, vec& v, vec& a) {
  const int n = s->ndof;
  const double gam = 0.5, bet = 0.25;
  const double a0 = 1.0 / (bet * dt * dt), a1 = gam / (bet * dt), a2 = 1.0 / (bet * dt), a3 = 1.0 / (2.0 * bet) - 1.0;
  const double a4 = gam / bet - 1.0, a5 = 0.5 * dt * (gam / bet - 2.0);
  vec Keff((size_t)n * n), tm(n), tc(n);
  for (size_t q = 0; q < Keff.size(); ++q) Keff[q] = s->BK[q] + a0 * s->BM[q] + a1 * s->BC[q];
  for (int i = 0; i < n; ++i) { tm[i] = a0 * w[i] + a2 * v[i] + a3 * a[i]; tc[i] = a1 * w[i] + a4 * v[i] + a5 * a[i]; }
  const vec Mt = matvec(s->BM, tm, n), Ct = matvec(s->BC, tc, n);
  vec rhs(n);
  for (int i = 0; i < n; ++i) rhs[i] = Q[i] + Mt[i] + Ct[i];
  const vec wn = dense_solve(Keff, rhs, n);
  for (int i = 0; i < n; ++i) {
    const double an = a0 * (wn[i] - w[i]) - a2 * v[i] - a3 * a[i];
    v[i] = v[i] + dt * ((1.0 - gam) * a[i] + gam * an);
    a[i] = an; w[i] = wn[i];
  }
}
// load vector from the marker forces of the last fluid step (Eq. 20 gathered per node, projected on the beam normal)
static void beam_load(orc_sim* s) {
  s->bQ.assign(s->ndof, 0.0);
  for (int l = 0; l < s->nl; ++l) {
    const int i = s->mnode[l];
    if (i <= 0) continue;                                      // markers of the clamped node load nothing
    const double qx = -s->P.rho * s->Fl[3 * l] * s->dV[l], qy = -s->P.rho * s->Fl[3 * l + 1] * s->dV[l];
    s->bQ[2 * (i - 1)] += qx * s->bnrm[0] + qy * s->bnrm[1];
  }
}
// markers follow their node: X = X^ref + w n, U^b = wdot n
static void beam_place_markers(orc_sim* s) {
  for (int l = 0; l < s->nl; ++l) {
    const int i = s->mnode[l];
    const double w = i > 0 ? s->bw[2 * (i - 1)] : 0.0, wd = i > 0 ? s->bv[2 * (i - 1)] : 0.0;
    s->X[3 * l] = s->Xref[3 * l] + w * s->bnrm[0]; s->X[3 * l + 1] = s->Xref[3 * l + 1] + w * s->bnrm[1]; s->X[3 * l + 2] = s->Xref[3 * l + 2];
    s->Ub[3 * l] = wd * s->bnrm[0]; s->Ub[3 * l + 1] = wd * s->bnrm[1]; s->Ub[3 * l + 2] = 0.0;
  }
}

// ---- the fluid part of one time step: a single fractional step, or the stages of the Runge-Kutta scheme ---------------
static void fluid_step(orc_sim* s, orc_info* info, vec& HU, vec& HV, vec& HW) {
  if (s->P.time_scheme == ORC_TIME_RK3) {
    // Explicit Runge-Kutta (L100, L431, Table 1; the paper names no tableau -- reading N3-3): the three-stage
    // third-order strong-stability-preserving scheme in Shu-Osher form, every stage a complete fractional step
    // E(u) = P[u + dt H(u) + IBM] (Eq. 4-10 with the Euler coefficients):
    //   u1 = E(u^n),  u2 = 3/4 u^n + 1/4 E(u1),  u^{n+1} = 1/3 u^n + 2/3 E(u2).
    // Convex combinations of projected fields stay divergence free.  p is the last stage's pressure (each solve
    // starts from the previous one), IBM force / body update use the last stage, iterations are summed.
    const vec u0 = s->u, v0 = s->v, w0 = s->w;
    const double c0[3] = {0.0, 0.75, 1.0 / 3.0}, c1[3] = {1.0, 0.25, 2.0 / 3.0};
    int iters = 0, conv = 1;
    for (int st = 0; st < 3; ++st) {
      fluid_substep(s, info, HU, HV, HW);
      iters += info->pcg_iters; conv = conv && info->converged;
      if (st > 0) {
        for (size_t q = 0; q < s->u.size(); ++q) s->u[q] = c0[st] * u0[q] + c1[st] * s->u[q];
        for (size_t q = 0; q < s->v.size(); ++q) s->v[q] = c0[st] * v0[q] + c1[st] * s->v[q];
        for (size_t q = 0; q < s->w.size(); ++q) s->w[q] = c0[st] * w0[q] + c1[st] * s->w[q];
      }
    }
    info->pcg_iters = iters; info->converged = conv;
  } else {
    fluid_substep(s, info, HU, HV, HW);
  }
}

// ---- one time step (O1..O9 in order), with the strong-coupling loop of Algorithm 1 (L212, L218-237) ------------------
// Reading N2-1 (the tail of Algorithm 1 is garbled in PAPER.md): sub-iteration k = 1..N restarts the fluid from time level
// n (u^{t-1}, p^{t-1}) with the structure's latest iterate -- markers at X^n + (w^(k-1) - w^n) moving with wdot^(k-1) --
// gathers the force, advances the structure from (w^n, wdot^n) with it (RK4, Eq. 12), and stops when
//   xi = || (w^(k) - w^(k-1)) / w^(k-1) ||_2^2 < tol  (1e-5 in the paper)   or k = N (100 in the paper).
// N = 1 is the weakly coupled scheme (L212).  A component with w^(k-1) = 0 = w^(k) contributes 0 to xi.
static void one_step(orc_sim* s, orc_info* info) {
  s->dt = choose_dt(s);
  const double dt = s->dt;
  vec HU(s->u.size()), HV(s->v.size()), HW(s->w.size());
  const int N = ((s->has_body || s->has_beam) && s->P.coupling_max_iters > 1) ? s->P.coupling_max_iters : 1;
  const vec bw0 = s->bw, bv0 = s->bv, ba0 = s->ba;             // beam state of time level n
  vec u0, v0, w0, p0, X0;
  double d0[3], vel0[3];
  for (int c = 0; c < 3; ++c) { d0[c] = s->bdisp[c]; vel0[c] = s->bvel[c]; }
  if (N > 1) { u0 = s->u; v0 = s->v; w0 = s->w; p0 = s->p; X0 = s->X; }
  int k = 0, iters = 0; double xi = 0.0;
  for (k = 1; k <= N; ++k) {
    if (k > 1) { s->u = u0; s->v = v0; s->w = w0; s->p = p0; }
    fluid_step(s, info, HU, HV, HW);
    iters += info->pcg_iters;
    if (s->has_body) {                                                                 // O9
      xi = 0.0;
      for (int c = 0; c < 3; ++c) if (s->dof & (1 << c)) {
        const double prev = s->bdisp[c];                       // w^(k-1): what the markers reflect during this sub-iteration
        double wn = d0[c], vn = vel0[c];
        orc_rk4_body(s->bm, s->bc_, s->bk, s->bforce[c], dt, &wn, &vn);
        const double dw = wn - prev;
        for (int l = 0; l < s->nl; ++l) s->X[3 * l + c] += dw;
        s->bdisp[c] = wn; s->bvel[c] = vn;
        if (!(dw == 0.0 && prev == 0.0)) xi += (dw / prev) * (dw / prev);
      }
      for (int l = 0; l < s->nl; ++l) for (int c = 0; c < 3; ++c) s->Ub[3 * l + c] = s->bvel[c];
    }
    if (s->has_beam) {                                                                 // O9': Newmark-beta on Eq. 11
      const vec prev = s->bw;                                  // w^(k-1): what the markers reflect during this sub-iteration
      beam_load(s);
      vec wn = bw0, vn = bv0, an = ba0;
      beam_newmark(s, s->bQ, dt, wn, vn, an);
      xi = 0.0;
      for (int i = 0; i < s->ndof; ++i) {
        const double dw = wn[i] - prev[i];
        if (!(dw == 0.0 && prev[i] == 0.0)) xi += (dw / prev[i]) * (dw / prev[i]);
      }
      s->bw = wn; s->bv = vn; s->ba = an;
      beam_place_markers(s);
    }
    if (N > 1 && xi < s->P.coupling_tol) break;
  }
  if (k > N) k = N;
  if (N > 1) info->pcg_iters = iters;
  info->coupling_iters = k; info->coupling_xi = xi;
  divergence(s, s->u, s->v, s->w, s->divu);
  double md = 0.0; int nan = 0;
  for (size_t q = 0; q < s->divu.size(); ++q) { double a = std::fabs(s->divu[q]); if (a > md) md = a; if (a != a) nan = 1; }
  info->max_abs_div = md; info->nan_flag = nan;
  s->hu = HU; s->hv = HV; s->hw = HW; s->have_hist = true; s->step += 1;
  s->dt_prev = dt; s->time += dt;
  for (int c = 0; c < 3; ++c) { info->body_force[c] = s->bforce[c]; info->body_disp[c] = s->bdisp[c]; info->body_vel[c] = s->bvel[c]; }
  info->step = s->step; info->dt = dt; info->time = s->time;
}

// ---- C interface --------------------------------------------------------------------------------
extern "C" orc_sim* orc_create(const orc_params* p) {
  if (!p || p->nx < 2 || p->ny < 2 || p->nz < 2 || p->dt <= 0 || p->rho <= 0 || p->lx <= 0 || p->ly <= 0 || p->lz <= 0) return nullptr;
  for (int d = 0; d < 3; ++d) {
    bool a = p->bc[2 * d] == ORC_BC_PERIODIC, b = p->bc[2 * d + 1] == ORC_BC_PERIODIC;
    if (a != b) return nullptr;
  }
  orc_sim* s = new orc_sim();
  s->P = *p; s->nx = p->nx; s->ny = p->ny; s->nz = p->nz;
  s->bx = p->bc[0] != ORC_BC_PERIODIC; s->by = p->bc[2] != ORC_BC_PERIODIC; s->bz = p->bc[4] != ORC_BC_PERIODIC;
  s->nxu = s->nx + s->bx; s->nyv = s->ny + s->by; s->nzw = s->nz + s->bz;
  s->hx = p->lx / p->nx; s->hy = p->ly / p->ny; s->hz = p->lz / p->nz;
  s->yf.resize(s->ny + 1); s->dy.resize(s->ny); s->yc.resize(s->ny);
  s->uniform_y = (p->yf == nullptr);
  for (int j = 0; j <= s->ny; ++j) s->yf[j] = p->yf ? p->yf[j] : p->y0 + j * s->hy;
  for (int j = 0; j < s->ny; ++j) {
    s->dy[j] = p->yf ? s->yf[j + 1] - s->yf[j] : s->hy;
    s->yc[j] = 0.5 * (s->yf[j] + s->yf[j + 1]);
    if (!(s->dy[j] > 0)) { delete s; return nullptr; }
  }
  s->P.yf = nullptr;
  if (p->precond == ORC_PC_GMG) {
    bool ok = s->uniform_y && std::fabs(s->hx - s->hy) <= 1e-12 * s->hx && std::fabs(s->hx - s->hz) <= 1e-12 * s->hx;
    if (!ok) { delete s; return nullptr; }
    s->nlev = mg_levels(s->nx, s->ny, s->nz);
  } else s->nlev = 0;
  size_t N = (size_t)s->nx * s->ny * s->nz;
  s->u.assign((size_t)s->nxu * s->ny * s->nz, 0.0); s->v.assign((size_t)s->nx * s->nyv * s->nz, 0.0);
  s->w.assign((size_t)s->nx * s->ny * s->nzw, 0.0); s->p.assign(N, 0.0); s->divu.assign(N, 0.0);
  s->hu = s->u; s->hv = s->v; s->hw = s->w;
  s->have_hist = false; s->step = 0; s->nl = 0; s->nseg = 0; s->has_body = false; s->dof = 0; s->oob = false; s->has_beam = false; s->nb = 0; s->ndof = 0;
  s->has_mask = false; s->uc[0] = s->uc[1] = s->uc[2] = 0.0;
  s->dt = s->dt_prev = p->dt; s->time = 0.0;
  for (int c = 0; c < 3; ++c) s->bdisp[c] = s->bvel[c] = s->bforce[c] = 0.0;
  return s;
}
extern "C" void orc_destroy(orc_sim* s) { delete s; }
static vec* field_ptr(orc_sim* s, int f) {
  switch (f) { case ORC_U: return &s->u; case ORC_V: return &s->v; case ORC_W: return &s->w; case ORC_P: return &s->p;
    case ORC_HU: return &s->hu; case ORC_HV: return &s->hv; case ORC_HW: return &s->hw; case ORC_DIV: return &s->divu; }
  return nullptr;
}
extern "C" long long orc_field_size(orc_sim* s, int f) { vec* v = field_ptr(s, f); return v ? (long long)v->size() : -1; }
extern "C" int orc_set_field(orc_sim* s, int f, const double* src) { vec* v = field_ptr(s, f); if (!v || !src) return 1; std::copy(src, src + v->size(), v->begin()); return 0; }
extern "C" int orc_get_field(orc_sim* s, int f, double* dst) { vec* v = field_ptr(s, f); if (!v || !dst) return 1; std::copy(v->begin(), v->end(), dst); return 0; }
extern "C" int orc_set_history(orc_sim* s, int have, long long step) { s->have_hist = have != 0; s->step = step; return 0; }
extern "C" int orc_set_markers(orc_sim* s, int n, const double* xyz, const double* vel, const double* dvol) {
  if (n < 0 || (n > 0 && !xyz)) return 1;
  if (n > 0 && (!s->uniform_y)) return 1;   // IBM needs uniform spacing
  s->nl = n; s->X.assign(xyz, xyz + (size_t)3 * n);
  s->Ub.assign((size_t)3 * n, 0.0); if (vel) s->Ub.assign(vel, vel + (size_t)3 * n);
  s->dV.assign(n, s->hx * s->hy * s->hz); if (dvol) s->dV.assign(dvol, dvol + n);
  s->Fl.assign((size_t)3 * n, 0.0); s->Ul.assign((size_t)3 * n, 0.0);
  s->oob = false;
  orc_ibm_index(s);
  if (s->oob) { s->nl = 0; s->oob = false; return 2; }   // unsupported: marker support touches a non-periodic boundary
  return 0;
}
extern "C" int orc_set_solid_mask(orc_sim* s, const unsigned char* eps_cells, const double* uc) {
  if (!eps_cells) { s->has_mask = false; return 0; }
  if (!s->uniform_y) return 1;
  s->eps.assign(eps_cells, eps_cells + s->p.size());
  for (int c = 0; c < 3; ++c) s->uc[c] = uc ? uc[c] : 0.0;
  s->has_mask = true;
  build_face_masks(s);
  return 0;
}
extern "C" void orc_get_face_masks(orc_sim* s, unsigned char* mu, unsigned char* mv, unsigned char* mw) {
  std::copy(s->mu.begin(), s->mu.end(), mu); std::copy(s->mv.begin(), s->mv.end(), mv); std::copy(s->mw.begin(), s->mw.end(), mw);
}
extern "C" int orc_set_body(orc_sim* s, double m, double c, double k, int dof) {
  if (!(m > 0)) return 1;
  s->has_body = true; s->bm = m; s->bc_ = c; s->bk = k; s->dof = dof; return 0;
}
extern "C" int orc_set_beam(orc_sim* s, int n_nodes, const double* node_xy, const int* marker_node, double EI, double mu_s, double zeta_s) {
  if (n_nodes < 2 || !node_xy || !marker_node || !(EI > 0) || !(mu_s > 0) || zeta_s < 0 || s->nl <= 0 || s->has_body || s->has_mask) return 1;
  const double tx = node_xy[2 * (n_nodes - 1)] - node_xy[0], ty = node_xy[2 * (n_nodes - 1) + 1] - node_xy[1];
  const double len = std::sqrt(tx * tx + ty * ty);
  if (!(len > 0)) return 1;
  for (int i = 1; i < n_nodes; ++i) {                          // straight, ordered along the axis
    const double ax = node_xy[2 * i] - node_xy[0], ay = node_xy[2 * i + 1] - node_xy[1];
    const double bx_ = node_xy[2 * i] - node_xy[2 * (i - 1)], by_ = node_xy[2 * i + 1] - node_xy[2 * (i - 1) + 1];
    if (std::fabs(ax * ty - ay * tx) > 1e-12 * len * len || !(bx_ * tx + by_ * ty > 0)) return 1;
  }
  for (int l = 0; l < s->nl; ++l) if (marker_node[l] < 0 || marker_node[l] >= n_nodes) return 1;
  s->nb = n_nodes; s->ndof = 2 * (n_nodes - 1);
  s->bX0.assign(node_xy, node_xy + (size_t)2 * n_nodes);
  s->mnode.assign(marker_node, marker_node + s->nl);
  s->bnrm[0] = -ty / len; s->bnrm[1] = tx / len;
  s->EI = EI; s->mus = mu_s; s->zeta = zeta_s;
  s->bw.assign(s->ndof, 0.0); s->bv.assign(s->ndof, 0.0); s->ba.assign(s->ndof, 0.0); s->bQ.assign(s->ndof, 0.0);
  s->Xref = s->X;
  s->has_beam = true;
  beam_assemble(s);
  return 0;
}
extern "C" int orc_beam_ndof(orc_sim* s) { return s->has_beam ? s->ndof : 0; }
extern "C" void orc_beam_matrices(orc_sim* s, double* K, double* M, double* C, double* coef /* alpha, beta, omega_1, omega_2 */) {
  if (K) std::copy(s->BK.begin(), s->BK.end(), K);
  if (M) std::copy(s->BM.begin(), s->BM.end(), M);
  if (C) std::copy(s->BC.begin(), s->BC.end(), C);
  if (coef) { coef[0] = s->ralpha; coef[1] = s->rbeta; coef[2] = s->om1; coef[3] = s->om2; }
}
extern "C" void orc_get_beam_state(orc_sim* s, double* w, double* v, double* a, double* Q) {
  if (w) std::copy(s->bw.begin(), s->bw.end(), w);
  if (v) std::copy(s->bv.begin(), s->bv.end(), v);
  if (a) std::copy(s->ba.begin(), s->ba.end(), a);
  if (Q) std::copy(s->bQ.begin(), s->bQ.end(), Q);
}
extern "C" void orc_set_beam_state(orc_sim* s, const double* w, const double* v, const double* a) {
  s->bw.assign(w, w + s->ndof); s->bv.assign(v, v + s->ndof); s->ba.assign(a, a + s->ndof);
  beam_place_markers(s);
}
extern "C" void orc_beam_newmark(orc_sim* s, const double* Q, double dt) {
  vec q(Q, Q + s->ndof);
  beam_newmark(s, q, dt, s->bw, s->bv, s->ba);
  s->bQ = q;
  beam_place_markers(s);
}
extern "C" int orc_step(orc_sim* s, int nsteps, orc_info* last, int* iters) {
  orc_info info; std::memset(&info, 0, sizeof info);
  for (int n = 0; n < nsteps; ++n) { one_step(s, &info); if (iters) iters[n] = info.pcg_iters; }
  if (last) *last = info;
  return s->oob ? 2 : 0;                                  // a moving body carried a support into a boundary
}
extern "C" int orc_poisson_solve(orc_sim* s, const double* rhs, double* p, orc_info* info) {
  size_t N = s->p.size(); vec b(rhs, rhs + N), x(p, p + N); orc_info I; std::memset(&I, 0, sizeof I);
  poisson(s, b, x, &I); std::copy(x.begin(), x.end(), p); if (info) *info = I; return 0;
}
extern "C" void orc_laplacian(orc_sim* s, const double* p, double* out) { laplacian(s, p, out); }
extern "C" void orc_apply_A(orc_sim* s, const double* x, double* out) { apply_A(s, x, out); }
extern "C" void orc_jacobi_diag(orc_sim* s, double* d) { jacobi_diag(s, d); }
extern "C" void orc_divergence(orc_sim* s, const double* u, const double* v, const double* w, double* out) {
  vec uu(u, u + s->u.size()), vv(v, v + s->v.size()), ww(w, w + s->w.size()), o(s->p.size());
  divergence(s, uu, vv, ww, o); std::copy(o.begin(), o.end(), out);
}
extern "C" void orc_gradient(orc_sim* s, const double* p, double* gu, double* gv, double* gw) {
  vec pp(p, p + s->p.size()), a(s->u.size()), b(s->v.size()), c(s->w.size());
  gradient(s, pp, a, b, c);
  std::copy(a.begin(), a.end(), gu); std::copy(b.begin(), b.end(), gv); std::copy(c.begin(), c.end(), gw);
}
extern "C" void orc_momentum_rhs(orc_sim* s, double* hu, double* hv, double* hw) {
  vec a(s->u.size()), b(s->v.size()), c(s->w.size());
  momentum(s, s->u, s->v, s->w, s->P.nu, s->P.body_force, a, b, c);
  std::copy(a.begin(), a.end(), hu); std::copy(b.begin(), b.end(), hv); std::copy(c.begin(), c.end(), hw);
}
extern "C" int orc_predict(orc_sim* s, int stage, double* us, double* vs, double* ws) {
  if (stage < 0 || stage > 2) return 1;
  s->dt = choose_dt(s);
  vec HU(s->u.size()), HV(s->v.size()), HW(s->w.size()), a, b, c;
  predictor(s, stage, a, b, c, HU, HV, HW);
  std::copy(a.begin(), a.end(), us); std::copy(b.begin(), b.end(), vs); std::copy(c.begin(), c.end(), ws);
  return 0;
}
extern "C" void orc_eddy_viscosity(orc_sim* s, double* out) {
  vec nut(s->p.size(), 0.0);
  if (s->P.cs > 0.0) eddy_viscosity(s, s->u, s->v, s->w, nut);
  std::copy(nut.begin(), nut.end(), out);
}
extern "C" void orc_convection(orc_sim* s, double* cu, double* cv, double* cw) {
  vec a(s->u.size()), b(s->v.size()), c(s->w.size()); const double g0[3] = {0, 0, 0};
  momentum(s, s->u, s->v, s->w, 0.0, g0, a, b, c);
  for (size_t q = 0; q < a.size(); ++q) cu[q] = -a[q];
  for (size_t q = 0; q < b.size(); ++q) cv[q] = -b[q];
  for (size_t q = 0; q < c.size(); ++q) cw[q] = -c[q];
}
extern "C" void orc_vcycle(orc_sim* s, const double* r, double* z) {
  vec rr(r, r + s->p.size()), zz(s->p.size()); precond_gmg(s, rr, zz); std::copy(zz.begin(), zz.end(), z);
}
extern "C" int orc_marker_count(orc_sim* s) { return s->nl; }
extern "C" void orc_get_cell_list(orc_sim* s, int* base, int* perm, int* keys, int* seg, int* nseg) {
  if (base) std::copy(s->base.begin(), s->base.end(), base);
  if (perm) std::copy(s->perm.begin(), s->perm.end(), perm);
  if (keys) std::copy(s->keys.begin(), s->keys.end(), keys);
  if (seg)  std::copy(s->seg.begin(), s->seg.end(), seg);
  if (nseg) *nseg = s->nseg;
}
extern "C" void orc_interpolate(orc_sim* s, const double* u, const double* v, const double* w, double* out) {
  vec uu(u, u + s->u.size()), vv(v, v + s->v.size()), ww(w, w + s->w.size()), o((size_t)3 * s->nl);
  interpolate(s, uu, vv, ww, o); std::copy(o.begin(), o.end(), out);
}
extern "C" void orc_spread(orc_sim* s, const double* F, double* fu, double* fv, double* fw) {
  vec FF(F, F + (size_t)3 * s->nl), a(fu, fu + s->u.size()), b(fv, fv + s->v.size()), c(fw, fw + s->w.size());
  spread(s, FF, a, b, c);
  std::copy(a.begin(), a.end(), fu); std::copy(b.begin(), b.end(), fv); std::copy(c.begin(), c.end(), fw);
}
extern "C" void orc_get_markers(orc_sim* s, double* xyz, double* vel, double* force) {
  if (xyz) std::copy(s->X.begin(), s->X.end(), xyz);
  if (vel) std::copy(s->Ub.begin(), s->Ub.end(), vel);
  if (force) std::copy(s->Fl.begin(), s->Fl.end(), force);
}
extern "C" void orc_set_body_state(orc_sim* s, const double* disp, const double* vel) {
  for (int c = 0; c < 3; ++c) { s->bdisp[c] = disp[c]; s->bvel[c] = vel[c]; }
}
extern "C" void orc_get_body_state(orc_sim* s, double* disp, double* vel, double* force) {
  for (int c = 0; c < 3; ++c) { disp[c] = s->bdisp[c]; vel[c] = s->bvel[c]; if (force) force[c] = s->bforce[c]; }
}
