/*
 * csrc/totals.cuh — step a9: conserved totals (§5.6.5 :1049-1063; DESIGN §"Totals", readings 14).
 *   S_tot = sum m S;  Q_q = sum m (N_q + J~^0_q/gamma);  P_i = sum m (C u_i + pi~^0_i/gamma), C = (w + Pi)/sigma;
 *   E = sum (m/sigma*) sqrt(-g) T^{00} (Cartesian, 2+1D hyperbolic per unit rapidity),
 *   E = sum (m/sigma*) tau (T^{tau tau} cosh eta + tau T^{tau eta} sinh eta) (3+1D hyperbolic).
 * Deterministic: fixed grid, warp-shuffle tree inside a block, partials reduced in block order by one block.
 */
#pragma once
#include "common.cuh"
#include "thermo_eos.cuh"

namespace ccake {

constexpr int TOT_THREADS = 256;
constexpr int TOT_NV = 14;   /* E, P1..3, S, NB, NS, NQ, M, work, npairs, (unused) x2, trace(max) at [13] */

__global__ void __launch_bounds__(TOT_THREADS)
totals_partial_kernel(int64_t n, KParams kp, Geom gm, const double* __restrict__ Y, int64_t npad, Sorted so,
                      double* __restrict__ partial, const uint32_t* __restrict__ orig, int64_t n_own) {
  double acc[TOT_NV];
  for (int k = 0; k < TOT_NV; ++k) acc[k] = 0.0;
  const int D = kp.D;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t a = so.perm[i];
    if ((int64_t)orig[a] >= n_own) continue;        /* ghost of a slab context: counted by its owner */
    double u[4];
    load_u(kp, gm, Y, npad, a, u);
    const double gam = u[0], sig = so.sigma[i], m = Y[CCAKE_MASS * npad + a];
    Dissip ds;
    if (D == 3) load_dissip<3>(kp, gm, Y, npad, a, u, ds);
    else load_dissip<2>(kp, gm, Y, npad, a, u, ds);
    const double p = so.p[i], w = so.e[i] + p, Pi = ds.bulkt * sig;
    const double Cc = (w + Pi) / sig;
    const double glo[4] = {1.0, -1.0, -1.0, -gm.G3};
    acc[4] += m * Y[CCAKE_S * npad + a];
    for (int q = 0; q < NQ; ++q) acc[5 + q] += m * (Y[(CCAKE_NB + q) * npad + a] + ds.Jt[q][0] / gam);
    for (int k = 1; k <= D; ++k) acc[k] += m * (Cc * glo[k] * u[k] + glo[k] * ds.pit[0][k] / gam);
    const double T00 = (w + Pi) * gam * gam - (p + Pi) + sig * ds.pit[0][0];
    const double vol = m / so.sigma_star[i];
    if (gm.hyper && D == 3) {
      const double eta = Y[CCAKE_R3 * npad + a];
      const double T03 = (w + Pi) * gam * u[3] + sig * ds.pit[0][3];
      acc[0] += vol * gm.sqrtg * (T00 * cosh(eta) + gm.tau * T03 * sinh(eta));
    } else {
      acc[0] += vol * gm.sqrtg * T00;
    }
    acc[8] += m;
    acc[9] += Y[CCAKE_WORK * npad + a];
    acc[10] += (double)so.nnb[i];
    double tr = ds.pit[0][0];
    for (int k = 1; k <= 3; ++k) tr += glo[k] * ds.pit[k][k];
    acc[13] = fmax(acc[13], fabs(tr * sig));
  }
  __shared__ double sm[TOT_NV][TOT_THREADS / 32];
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  for (int k = 0; k < TOT_NV; ++k) {
    double v = acc[k];
    for (int o = 16; o > 0; o >>= 1) {
      const double t = __shfl_xor_sync(0xffffffffu, v, o);
      v = (k == 13) ? fmax(v, t) : v + t;
    }
    if (lane == 0) sm[k][wp] = v;
  }
  __syncthreads();
  if (threadIdx.x < TOT_NV) {
    double v = sm[threadIdx.x][0];
    for (int j = 1; j < TOT_THREADS / 32; ++j) v = (threadIdx.x == 13) ? fmax(v, sm[threadIdx.x][j]) : v + sm[threadIdx.x][j];
    partial[blockIdx.x * TOT_NV + threadIdx.x] = v;
  }
}

__global__ void totals_final_kernel(const double* __restrict__ partial, int nblocks, double* __restrict__ out) {
  if (threadIdx.x < TOT_NV) {
    double v = partial[threadIdx.x];
    for (int b = 1; b < nblocks; ++b) {
      const double t = partial[b * TOT_NV + threadIdx.x];
      v = (threadIdx.x == 13) ? fmax(v, t) : v + t;
    }
    out[threadIdx.x] = v;
  }
}

}  // namespace ccake
