/*
 * csrc/pair_v1.cuh — steps a4 (smoothing sums) and a6 (gradient sums), first correct version: one thread per
 * particle a walking the 3^D neighbour cells of the traversal grid.  Kept as the simple cross-check of the tiled
 * kernels in pair_tiled.cuh (selected with CCAKE_PAIR_IMPL=1).
 *
 *   a4  sigma*_a = sum_b m_b W_ab,  s*_a = sum_b m_b S_b W_ab,  rho*_{q,a} = sum_b m_b N_{q,b} W_ab
 *       (Eq. 71-72 :877-882), b over r_ab^2 < (2h)^2 including b = a; W = cubic spline (Eq. 77 :910).
 *   a6  n = -1 and n = +1 SPH derivatives (Eq. 81-82 :934-938; DESIGN reading 3) with dW_ab of Eq. 79 :920.
 *
 * The neighbour decision is r2 = (dx*dx + dy*dy) + dz*dz < (2h)^2, strictly, evaluated with round-to-nearest
 * multiplies and adds and no FMA contraction (DESIGN reading 8), so neighbour sets are reproducible bit by bit.
 */
#pragma once
#include "common.cuh"

namespace ccake {

__device__ __forceinline__ double dist2_exact(double dx, double dy, double dz, int D) {
  double r2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
  if (D == 3) r2 = __dadd_rn(r2, __dmul_rn(dz, dz));
  return r2;
}

/* cubic spline, Eq. 77: W = sigma_D (1 - 3/2 q^2 + 3/4 q^3) [q <= 1], sigma_D/4 (2 - q)^3 [q <= 2] */
__device__ __forceinline__ double kernel_W(double r, double inv_h, double sigma_d) {
  const double q = r * inv_h;
  if (q <= 1.0) return sigma_d * (1.0 - 1.5 * q * q + 0.75 * q * q * q);
  if (q <= 2.0) { const double t = 2.0 - q; return sigma_d * 0.25 * t * t * t; }
  return 0.0;
}

/* Eq. 79: dW/dr / r  (so that grad_i W = fac * dr_i); 0 at r = 0 */
__device__ __forceinline__ double kernel_dW_over_r(double r, double inv_h, double sigma_d) {
  if (r == 0.0) return 0.0;
  const double q = r * inv_h;
  double f;
  if (q <= 1.0) f = -3.0 * q + 2.25 * q * q;
  else if (q <= 2.0) { const double t = 2.0 - q; f = -0.75 * t * t; }
  else return 0.0;
  return sigma_d * inv_h * f / r;
}

template <int D>
__global__ void __launch_bounds__(128)
smoothing_v1_kernel(int64_t n, KParams kp, const Grid* __restrict__ grid, Sorted so) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Grid g = *grid;
  const uint32_t cid = so.key[i];
  const int cx = cid % g.nc[0], cy = (cid / g.nc[0]) % g.nc[1], cz = cid / (g.nc[0] * g.nc[1]);
  const double xa = so.x[0][i], ya = so.x[1][i], za = (D == 3) ? so.x[2][i] : 0.0;
  double sg = 0.0, ss = 0.0, rq0 = 0.0, rq1 = 0.0, rq2 = 0.0;
  uint32_t cnt = 0;
  const int z0 = (D == 3) ? -1 : 0, z1 = (D == 3) ? 1 : 0;
  for (int dz = z0; dz <= z1; ++dz) {
    const int zz = cz + dz;
    if (zz < 0 || zz >= g.nc[2]) continue;
    for (int dy = -1; dy <= 1; ++dy) {
      const int yy = cy + dy;
      if (yy < 0 || yy >= g.nc[1]) continue;
      const int xlo = max(cx - 1, 0), xhi = min(cx + 1, g.nc[0] - 1);
      const int row = g.nc[0] * (yy + g.nc[1] * zz);
      const uint32_t b0 = so.cell_start[row + xlo], b1 = so.cell_start[row + xhi + 1];
      for (uint32_t b = b0; b < b1; ++b) {
        const double dx = xa - so.x[0][b], dyv = ya - so.x[1][b], dzv = (D == 3) ? za - so.x[2][b] : 0.0;
        const double r2 = dist2_exact(dx, dyv, dzv, D);
        if (r2 < kp.cut2) {
          const double W = kernel_W(sqrt(r2), kp.inv_h, kp.sigma_d);
          const double mW = so.m[b] * W;
          sg += mW;
          ss += mW * so.S[b];
          rq0 += mW * so.Nq[0][b];
          rq1 += mW * so.Nq[1][b];
          rq2 += mW * so.Nq[2][b];
          cnt += (b != (uint32_t)i);
        }
      }
    }
  }
  so.sigma_star[i] = sg;
  so.s_star[i] = ss;
  so.rho_star[0][i] = rq0;
  so.rho_star[1][i] = rq1;
  so.rho_star[2][i] = rq2;
  so.nnb[i] = cnt;
}

template <int D, bool VISC, bool DIFF>
__global__ void __launch_bounds__(128)
gradient_v1_kernel(int64_t n, KParams kp, const Grid* __restrict__ grid, Sorted so) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Grid g = *grid;
  const uint32_t cid = so.key[i];
  const int cx = cid % g.nc[0], cy = (cid / g.nc[0]) % g.nc[1], cz = cid / (g.nc[0] * g.nc[1]);
  const double xa = so.x[0][i], ya = so.x[1][i], za = (D == 3) ? so.x[2][i] : 0.0;
  double ua[D], va[D], Ba[D * D], Ka[3 * D], ala[3];
  const double Pa = so.Ppair[i];
  for (int k = 0; k < D; ++k) { ua[k] = so.u[k][i]; va[k] = so.v[k][i]; }
  if (VISC) for (int j = 0; j < D; ++j) for (int k = 0; k < D; ++k) Ba[j * D + k] = so.Bpair[j * 3 + k][i];
  if (DIFF) {
    for (int q = 0; q < 3; ++q) { ala[q] = so.alpha[q][i]; for (int j = 0; j < D; ++j) Ka[q * D + j] = so.Kpair[q * 3 + j][i]; }
  }
  double FP[D], FB[D], FK[3], DU[D * D], DA[3 * D], dv = 0.0;
  for (int k = 0; k < D; ++k) { FP[k] = 0.0; FB[k] = 0.0; }
  for (int k = 0; k < D * D; ++k) DU[k] = 0.0;
  for (int k = 0; k < 3 * D; ++k) DA[k] = 0.0;
  FK[0] = FK[1] = FK[2] = 0.0;
  const int z0 = (D == 3) ? -1 : 0, z1 = (D == 3) ? 1 : 0;
  for (int dz = z0; dz <= z1; ++dz) {
    const int zz = cz + dz;
    if (zz < 0 || zz >= g.nc[2]) continue;
    for (int dy = -1; dy <= 1; ++dy) {
      const int yy = cy + dy;
      if (yy < 0 || yy >= g.nc[1]) continue;
      const int xlo = max(cx - 1, 0), xhi = min(cx + 1, g.nc[0] - 1);
      const int row = g.nc[0] * (yy + g.nc[1] * zz);
      const uint32_t b0 = so.cell_start[row + xlo], b1 = so.cell_start[row + xhi + 1];
      for (uint32_t b = b0; b < b1; ++b) {
        double dr[3];
        dr[0] = xa - so.x[0][b]; dr[1] = ya - so.x[1][b]; dr[2] = (D == 3) ? za - so.x[2][b] : 0.0;
        const double r2 = dist2_exact(dr[0], dr[1], dr[2], D);
        if (r2 < kp.cut2 && b != (uint32_t)i) {
          const double fac = so.m[b] * kernel_dW_over_r(sqrt(r2), kp.inv_h, kp.sigma_d);
          double gW[D];
          for (int k = 0; k < D; ++k) gW[k] = fac * dr[k];
          const double Ps = Pa + so.Ppair[b];
          for (int k = 0; k < D; ++k) {
            FP[k] += Ps * gW[k];
            const double du = so.u[k][b] - ua[k];
            for (int j = 0; j < D; ++j) DU[j * D + k] += du * gW[j];
            dv += (so.v[k][b] - va[k]) * gW[k];
          }
          if (VISC)
            for (int k = 0; k < D; ++k)
              for (int j = 0; j < D; ++j) FB[k] += (Ba[j * D + k] + so.Bpair[j * 3 + k][b]) * gW[j];
          if (DIFF)
            for (int q = 0; q < 3; ++q) {
              const double da = so.alpha[q][b] - ala[q];
              for (int j = 0; j < D; ++j) {
                DA[q * D + j] += da * gW[j];
                FK[q] += (Ka[q * D + j] + so.Kpair[q * 3 + j][b]) * gW[j];
              }
            }
        }
      }
    }
  }
  const double inv = 1.0 / so.sigma_star[i];
  for (int k = 0; k < 3; ++k) {
    so.FP[k][i] = (k < D) ? FP[k] : 0.0;
    so.FB[k][i] = (k < D) ? FB[k] : 0.0;
    so.FK[k][i] = FK[k];
  }
  for (int j = 0; j < 3; ++j)
    for (int k = 0; k < 3; ++k) {
      so.DU[j * 3 + k][i] = (j < D && k < D) ? DU[j * D + k] * inv : 0.0;
      so.DA[j * 3 + k][i] = (k < D) ? DA[j * D + k] * inv : 0.0;   /* DA[q][i] = d_i alpha_q */
    }
  so.divv[i] = dv * inv;
}

}  // namespace ccake
