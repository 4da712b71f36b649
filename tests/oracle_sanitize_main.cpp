// Driver for tests/test_oracle_fluid.py::test_oracle_runs_clean_under_address_and_undefined_behaviour_sanitizers: exercises
// every branch family of oracle/fs_oracle.cpp on tiny grids (periodic GMG, stretched channel with the LES closures, open box
// with markers + rigid body + strong coupling, eps mask, flexible beam, Runge-Kutta, CFL-adaptive dt, upwind) under
// -fsanitize=address,undefined.  Test infrastructure: links only the oracle.
#include "../oracle/fs_oracle.h"
#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>

static orc_params base(int nx, int ny, int nz, double lx, double ly, double lz) {
  orc_params p; std::memset(&p, 0, sizeof p);
  p.nx = nx; p.ny = ny; p.nz = nz; p.lx = lx; p.ly = ly; p.lz = lz;
  p.nu = 0.01; p.rho = 1.0; p.dt = 1e-3; p.time_scheme = ORC_TIME_AB2; p.precond = ORC_PC_JACOBI; p.rtol = 1e-8; p.max_iter = 500;
  p.warm_start = 1; p.mg_nu1 = 2; p.mg_nu2 = 2; p.mg_coarse_sweeps = 4; p.mg_omega = 6.0 / 7.0; p.coupling_max_iters = 1; p.coupling_tol = 1e-5;
  return p;
}
static void fill(orc_sim* s, double amp) {
  for (int f = ORC_U; f <= ORC_W; ++f) {
    std::vector<double> a((size_t)orc_field_size(s, f));
    for (size_t q = 0; q < a.size(); ++q) a[q] = amp * std::sin(0.37 * (double)q + f);
    orc_set_field(s, f, a.data());
  }
}
static int run(orc_sim* s, int n) { orc_info I; int rc = orc_step(s, n, &I, nullptr); return rc != 0 || I.nan_flag; }

int main() {
  int bad = 0;
  {  // periodic, GMG, Runge-Kutta, upwind, adaptive dt
    orc_params p = base(16, 16, 16, 6.28, 6.28, 6.28); p.precond = ORC_PC_GMG; p.time_scheme = ORC_TIME_RK3; p.convection = ORC_CONV_UPWIND; p.cfl = 0.4;
    orc_sim* s = orc_create(&p); fill(s, 0.5); bad |= run(s, 2); orc_destroy(s);
  }
  {  // stretched channel, LES + wall model
    std::vector<double> yf(13); for (int j = 0; j <= 12; ++j) yf[j] = std::tanh(2.0 * (2.0 * j / 12 - 1.0)) / std::tanh(2.0);
    orc_params p = base(10, 12, 8, 3.0, 2.0, 2.0); p.y0 = -1.0; p.yf = yf.data(); p.bc[2] = p.bc[3] = ORC_BC_NOSLIP; p.cs = 0.1; p.wall_model = 1; p.body_force[0] = 1.0;
    orc_sim* s = orc_create(&p); fill(s, 0.3); bad |= run(s, 2); orc_destroy(s);
  }
  const double h = 1.0 / 8.0;
  std::vector<double> X; std::vector<int> node;
  for (int k = 0; k < 4; ++k) for (int i = 0; i < 5; ++i) { X.push_back(1.01); X.push_back(0.77 + 0.1 * i); X.push_back((k + 0.5) * h); node.push_back(i); }
  const int nm = (int)node.size();
  for (int variant = 0; variant < 3; ++variant) {  // open box: rigid body with strong coupling / eps mask / flexible beam
    orc_params p = base(24, 16, 4, 3.0, 2.0, 0.5); p.dt = 5e-3;
    p.bc[0] = ORC_BC_INFLOW; p.bc[1] = ORC_BC_OUTFLOW; p.bc[2] = p.bc[3] = ORC_BC_SLIP; p.bc_vel[0][0] = 1.0; p.bc_vel[1][0] = 1.0; p.inflow_noise = 0.01; p.seed = 7;
    if (variant != 1) p.coupling_max_iters = 4;
    orc_sim* s = orc_create(&p);
    std::vector<double> u((size_t)orc_field_size(s, ORC_U), 1.0); orc_set_field(s, ORC_U, u.data());
    bad |= orc_set_markers(s, nm, X.data(), nullptr, nullptr);
    if (variant == 0) bad |= orc_set_body(s, 1.0, 0.1, 5.0, 3);
    if (variant == 1) {
      std::vector<unsigned char> eps((size_t)orc_field_size(s, ORC_P), 0);
      for (int k = 0; k < 4; ++k) for (int j = 6; j < 10; ++j) for (int i = 7; i < 9; ++i) eps[i + 24 * (j + 16 * k)] = 1;
      const double uc[3] = {0.0, 0.1, 0.0};
      bad |= orc_set_solid_mask(s, eps.data(), uc);
    }
    if (variant == 2) {
      double xy[10]; for (int i = 0; i < 5; ++i) { xy[2 * i] = 1.01; xy[2 * i + 1] = 0.77 + 0.1 * i; }
      bad |= orc_set_beam(s, 5, xy, node.data(), 0.05, 0.2, 0.02);
    }
    bad |= run(s, 2);
    orc_destroy(s);
  }
  std::printf("oracle sanitizer run: %s\n", bad ? "FAILED" : "ok");
  return bad;
}
