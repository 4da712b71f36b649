// fs_kernels_pcgc.cu -- the whole PCG solve (S7, point preconditioners) as ONE persistent cooperative
// kernel, for grids whose fields are small enough to live in (or near) the 126 MB L2: the FSI configurations c2-c4.
//
// On such grids the streaming kernels of fs_kernels_pcg.cu are latency bound: a z march of 16-32 planes costs 1-2 us
// per plane whatever the plane holds, a step is 10^3 iterations of two launches, and each iteration pays the graph's
// WHILE-node turnaround.  Here every CTA is resident for the whole solve (cooperative launch), every phase is flat --
// a thread owns the same 16-byte vectors of cells in every phase, neighbours of the 7-point operator are read straight
// from L1 / L2 -- and the two global reductions of textbook CG plus the halo dependence of q = A d are grid-wide
// barriers (one atomic per CTA on a counter + spin; co-residency is what the cooperative launch guarantees):
//     P1  d = z + beta d,  z = M^-1 r                          | grid.sync
//     P2  q = A d,  partial d.q                                 | grid.sync, every CTA sums the partials in the same order
//     P3  x += alpha d,  r -= alpha q,  partial r.r, r.z, sum r | grid.sync, every CTA sums, tests ||r|| <= rtol ||b||
// The recurrences, the operator and the order of floating-point operations per cell are those of k_pcg_dirapply /
// k_pcg_update (and of the oracle); only the partition of the reductions differs.  x is updated in place (no deferred
// update), so the zero-mean pass after the solve is the plain mean + shift.
// Tried and dropped (profiles/r2_small_configs.md): merging P1 into P2 by recomputing d on the six neighbours of every cell from r
// and the old d (10 words, two barriers: the barrier floor drops from 11.4 to 9.9 us per iteration) -- the fourteen loads per
// vector instead of seven thrash L2 on the 25-34 MB fields of c3 / c4 and the step gets 17-25 % slower.
#include "fs_internal.cuh"
#include <cstdlib>

namespace fs {

constexpr int kCoopThreads = 256;

// Sums NV arrays of n partials (array a at p + a * n) in a fixed order -- lane l of warp 0 adds partials l, l + 32, ..., then
// a butterfly over the lanes -- so every CTA gets bit-identical totals; returned to all threads through shared memory.
template <int NV> __device__ __forceinline__ void coop_sum(const double* __restrict__ p, int n, double (&out)[NV], double* sh) {
  const int tid = threadIdx.x;
  if (tid < 32) {
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      double t = 0.0;
#pragma unroll 8
      for (int b = tid; b < n; b += 32) t += __ldcg(p + (size_t)a * n + b);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      if (tid == 0) sh[a] = t;
    }
  }
  __syncthreads();
#pragma unroll
  for (int a = 0; a < NV; ++a) out[a] = sh[a];
  __syncthreads();
}

// Grid-wide barrier on a monotonically increasing counter (zeroed before the launch): arrive with one atomic per CTA, spin
// until all G CTAs of this round have arrived.  All CTAs are co-resident (cooperative launch), so the spin cannot deadlock.
// The fences order the CTA's global writes before its arrival and its later reads after the release.
__device__ __forceinline__ void coop_barrier(unsigned* counter, unsigned target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(counter, 1u);
    while (*reinterpret_cast<volatile unsigned*>(counter) < target) __nanosleep(40);
    __threadfence();
  }
  __syncthreads();
}

template <class T, int PC> __global__ void __launch_bounds__(kCoopThreads, 4) k_pcg_coop(const Ctx<T> c, double* __restrict__ part) {
  constexpr int VX = Vec16<T>::VX;
  using W = Vec16<T>;
  unsigned* bar = &c.S->ticket[4]; unsigned round = 0;
  __shared__ double sh[3 * 32];
  Scalars* S = c.S;
  if (S->done) return;                       // converged at the start: the same answer in every CTA (written by the start kernel)
  const int G = gridDim.x, bid = blockIdx.x, tid = threadIdx.x;
  const unsigned nvx = (unsigned)c.nx / VX, nrow = nvx * (unsigned)c.ny, NV = nrow * (unsigned)c.nz;
  const unsigned stride = (unsigned)G * kCoopThreads, v0 = (unsigned)bid * kCoopThreads + tid;
  const unsigned pl = (unsigned)c.nx * c.ny;
  double* pA = part; double* pB = part + 4 * (size_t)G;      // two sets of partials (P2 / P3), see the header of the loop
  const double bnorm = sqrt(S->bnorm2), rtol = S->rtol, Ncells = (double)c.nx * c.ny * c.nz;
  const int max_iter = S->max_iter;
  double rho = S->rho_cur, rho_prev = 1.0, rr = S->rr, rmean = S->rmean, alpha_d = 0.0;
  int iter = 0, conv = 0;
  bool first = true;
  // 1 / diag A of a cell: (x + y + z parts) * dy_j, the association of jacobi_diag / k_pcg_dirapply
  auto diag = [&](int i, int j, int k) {
    const T dxy = T((c.bx && i == 0 ? 0 : 1) + (c.bx && i == c.nx - 1 ? 0 : 1)) * c.ihx2;
    const T dyy = (c.cyh[j] + c.cyl[j]) * c.idy[j + 1];
    const T dzz = T((c.bz && k == 0 ? 0 : 1) + (c.bz && k == c.nz - 1 ? 0 : 1)) * c.ihz2;
    return (dxy + dyy + dzz) * c.dy[j + 1];
  };
  for (;;) {
    // ---- P1: direction -------------------------------------------------------------------------------------------
    const T beta = first ? T(0) : T(rho / rho_prev);
    for (unsigned v = v0; v < NV; v += stride) {
      const unsigned iv = v % nvx, t = v / nvx; const int j = (int)(t % (unsigned)c.ny), k = (int)(t / (unsigned)c.ny), i0 = (int)iv * VX;
      const unsigned o = (unsigned)i0 + (unsigned)c.nx * j + pl * (unsigned)k;
      const W r = ld16<T>(c.r + o);
      W d;
      if (!first) d = ld16<T>(c.d + o);
#pragma unroll
      for (int a = 0; a < VX; ++a) {
        const T z = PC == 1 ? r.a[a] / diag(i0 + a, j, k) : r.a[a];
        d.a[a] = first ? z : z + beta * d.a[a];
      }
      st16<T>(c.d + o, d);
    }
    coop_barrier(bar, (unsigned)G * ++round);
    // ---- P2: q = A d, d.q ------------------------------------------------------------------------------------------
    double dot = 0.0;
    for (unsigned v = v0; v < NV; v += stride) {
      const unsigned iv = v % nvx, t = v / nvx; const int j = (int)(t % (unsigned)c.ny), k = (int)(t / (unsigned)c.ny), i0 = (int)iv * VX;
      const unsigned row = (unsigned)c.nx * j + pl * (unsigned)k, o = (unsigned)i0 + row;
      // neighbour cells: wrapped (periodic) or clamped (bounded: zero difference = dropped Neumann flux)
      const int iw = i0 > 0 ? i0 - 1 : (c.bx ? 0 : c.nx - 1), ie = i0 + VX < c.nx ? i0 + VX : (c.bx ? c.nx - 1 : 0);
      const int js = j > 0 ? j - 1 : (c.by ? 0 : c.ny - 1), jn = j + 1 < c.ny ? j + 1 : (c.by ? c.ny - 1 : 0);
      const int kb = k > 0 ? k - 1 : (c.bz ? 0 : c.nz - 1), kt = k + 1 < c.nz ? k + 1 : (c.bz ? c.nz - 1 : 0);
      const W dC = ld16<T>(c.d + o);
      const W dS = ld16<T>(c.d + ((unsigned)i0 + (unsigned)c.nx * js + pl * (unsigned)k));
      const W dN = ld16<T>(c.d + ((unsigned)i0 + (unsigned)c.nx * jn + pl * (unsigned)k));
      const W dB = ld16<T>(c.d + ((unsigned)i0 + (unsigned)c.nx * j + pl * (unsigned)kb));
      const W dT = ld16<T>(c.d + ((unsigned)i0 + (unsigned)c.nx * j + pl * (unsigned)kt));
      const T dWs = c.d[row + (unsigned)iw], dEs = c.d[row + (unsigned)ie];
      const T cyl = c.cyl[j], cyh = c.cyh[j], idy = c.idy[j + 1], ndy = -c.dy[j + 1];
      W q;
      T sdot = T(0);
#pragma unroll
      for (int a = 0; a < VX; ++a) {
        const T xc = dC.a[a];
        const T xw = a > 0 ? dC.a[a > 0 ? a - 1 : 0] : dWs, xe = a < VX - 1 ? dC.a[a < VX - 1 ? a + 1 : a] : dEs;
        T acc = (xe - xc) * c.ihx2 - (xc - xw) * c.ihx2;
        const T fy = (dN.a[a] - xc) * cyh - (xc - dS.a[a]) * cyl;
        acc += fy * idy;
        acc += (dT.a[a] - xc) * c.ihz2 - (xc - dB.a[a]) * c.ihz2;
        q.a[a] = acc * ndy;
        sdot += xc * q.a[a];
      }
      st16<T>(c.q + o, q);
      dot += (double)sdot;
    }
    {
      double v1[1] = {dot};
      block_sum<1>(v1, sh);
      if (tid == 0) __stcg(pA + bid, v1[0]);
    }
    coop_barrier(bar, (unsigned)G * ++round);
    double dqv[1];
    coop_sum<1>(pA, G, dqv, sh);
    alpha_d = rho / dqv[0];
    const T alpha = T(alpha_d), rm = sizeof(T) == 4 ? T(rmean) : T(0);
    // ---- P3: x += alpha d, r -= alpha q, r.r, r.z, sum r -------------------------------------------------------------
    double s_rr = 0.0, s_rz = 0.0, s_r = 0.0;
    for (unsigned v = v0; v < NV; v += stride) {
      const unsigned iv = v % nvx, t = v / nvx; const int j = (int)(t % (unsigned)c.ny), k = (int)(t / (unsigned)c.ny), i0 = (int)iv * VX;
      const unsigned o = (unsigned)i0 + (unsigned)c.nx * j + pl * (unsigned)k;
      W r = ld16<T>(c.r + o), x = ld16<T>(c.p + o);
      const W q = ld16<T>(c.q + o), d = ld16<T>(c.d + o);
      T a0 = T(0), a1 = T(0), a2 = T(0);
#pragma unroll
      for (int a = 0; a < VX; ++a) {
        x.a[a] += alpha * d.a[a];
        T tt = r.a[a] - alpha * q.a[a];
        if (sizeof(T) == 4) tt -= rm;
        r.a[a] = tt;
        const T z = PC == 1 ? tt / diag(i0 + a, j, k) : tt;
        a0 += tt * tt; a1 += tt * z; a2 += tt;
      }
      st16<T>(c.p + o, x); st16<T>(c.r + o, r);
      s_rr += (double)a0; s_rz += (double)a1; s_r += (double)a2;
    }
    {
      double v3[3] = {s_rr, s_rz, s_r};
      block_sum<3>(v3, sh);
      if (tid == 0) { __stcg(pB + bid, v3[0]); __stcg(pB + G + bid, v3[1]); __stcg(pB + 2 * G + bid, v3[2]); }
    }
    coop_barrier(bar, (unsigned)G * ++round);
    double tot[3];
    coop_sum<3>(pB, G, tot, sh);
    rr = tot[0];
    const double rz = tot[1];
    rmean = tot[2] / Ncells;
    iter += 1; first = false;
    rho_prev = rho; rho = rz;
    conv = sqrt(rr) <= rtol * bnorm;
    if (conv || iter >= max_iter) break;
  }
  if (bid == 0 && tid == 0) {
    S->rr = rr; S->rmean = rmean; S->rho_cur = rho; S->rho_prev = rho_prev; S->alpha_prev = alpha_d;
    S->iter = iter; S->first = 0; S->converged = conv; S->done = 1;
    S->pending = 0; S->need_update = 0; S->dsel = 0;
  }
}

template <class T> static int coop_blocks(int pc, unsigned nv) {
  int per_sm = 0, dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (pc == 1) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_pcg_coop<T, 1>, kCoopThreads, 0);
  else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_pcg_coop<T, 0>, kCoopThreads, 0);
  long long g = (long long)per_sm * sms;
  const long long need = ((long long)nv + kCoopThreads - 1) / kCoopThreads;
  if (g > need) g = need;
  if (g > kMaxPartials / 2) g = kMaxPartials / 2;
  return (int)(g > 0 ? g : 1);
}

// Applies to the point preconditioners on grids with nx a multiple of the vector width whose fields are at most
// kCoopMaxBytes each (L2-sized: above that the streaming kernels run at the HBM roofline and win).
template <class T> bool pcg_coop_applies(const Ctx<T>& c) {
  constexpr long long kCoopMaxBytes = 64LL << 20;
  if (c.precond == FS_PC_GMG || c.nx % Vec16<T>::VX != 0) return false;
  if ((long long)c.nx * c.ny * c.nz * (long long)sizeof(T) > kCoopMaxBytes) return false;
  const char* e = getenv("FS_TUNE_COOP");
  if (e && atoi(e) == 0) return false;
  int dev = 0, coop = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  return coop != 0;
}

template <class T> int launch_pcg_coop(const Ctx<T>& c, const Launch& L) {
  const unsigned nv = (unsigned)(c.nx / Vec16<T>::VX) * c.ny * c.nz;
  const int pc = c.precond == FS_PC_JACOBI ? 1 : 0;
  const int G = coop_blocks<T>(pc, nv);
  Ctx<T> cc = c;
  double* part = c.partials;
  void* args[2] = {&cc, &part};
  const double N = (double)c.nx * c.ny * c.nz;
  FS_LAUNCHI(L, "pcg_solve_coop", sizeof(T) == 8 ? "k_pcg_coop<f64>" : "k_pcg_coop<f32>", 11.0 * sizeof(T) * N, {
    cudaMemsetAsync(&c.S->ticket[4], 0, sizeof(unsigned), L.s);          // the barrier counter of coop_barrier
    if (pc == 1) cudaLaunchCooperativeKernel((const void*)k_pcg_coop<T, 1>, dim3(G), dim3(kCoopThreads), args, 0, L.s);
    else cudaLaunchCooperativeKernel((const void*)k_pcg_coop<T, 0>, dim3(G), dim3(kCoopThreads), args, 0, L.s);
  });
  return 1;
}

template bool pcg_coop_applies<float>(const Ctx<float>&);
template bool pcg_coop_applies<double>(const Ctx<double>&);
template int launch_pcg_coop<float>(const Ctx<float>&, const Launch&);
template int launch_pcg_coop<double>(const Ctx<double>&, const Launch&);

}  // namespace fs
