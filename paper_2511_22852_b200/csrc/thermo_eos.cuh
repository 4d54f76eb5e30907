/*
 * csrc/thermo_eos.cuh — step a5: rest-frame densities, equation of state, pair inputs.
 *
 *   X_a = X*_a / (gamma_a sqrt(-g))                              PAPER.md Eq. 68 :864 (DESIGN reading 2)
 *   table: per-axis cell search + quadrilinear blend of 16 nodes  :583-593 (log-decade axes :593)
 *   closed form: p = c0 T^4 + c2 T^2 sum mu^2 + c4 sum mu^4       App. A Eq. A.5-A.7 :2115-2122, cubic A.11-A.14
 *   pair inputs: (p + Pi)/sigma*^2, B^j_i/sigma*^2, K^j_q/sigma*^2, alpha_q = mu_q/T, v^i   (DESIGN §"EoM")
 */
#pragma once
#include "common.cuh"
#include "pair_mma.cuh"

namespace ccake {

struct ThermoOut { double T, mu[NQ], p, e, cs2, ws, wq[NQ]; int oob; };

/* last node <= x by comparisons only (binary search); the cell is clamped to [0, n-2] */
__device__ inline int axis_cell(const double* __restrict__ ax, int n, double x) {
  int lo = 0, hi = n;              /* first index with ax[idx] > x, in [lo, hi] */
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (ax[mid] <= x) lo = mid + 1; else hi = mid;
  }
  int i = lo - 1;
  if (i > n - 2) i = n - 2;
  if (i < 0) i = 0;
  return i;
}

/* caller's table [node][ncols] -> resident copy [node][TB_STRIDE] (TableDev) */
__global__ void table_pack_kernel(const double* __restrict__ src, int ncols, int64_t nodes, TableDev tb, double* __restrict__ dst) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nodes * TB_STRIDE) return;
  const int64_t node = i / TB_STRIDE;
  const int c = (int)(i - node * TB_STRIDE);
  const int k = (c < CCAKE_NCOLS_MAX) ? tb.col_of[c] : -1;
  dst[i] = (k >= 0) ? src[node * ncols + k] : 0.0;
}

__device__ inline ThermoOut eos_table_lookup(const TableDev& tb, double s, const double n[NQ]) {
  ThermoOut th;
  th.oob = 0;
  double x[4];
  x[0] = s;
  for (int k = 1; k < 4; ++k) x[k] = (tb.kind[k] == 1) ? n[k - 1] / s : n[k - 1];
  int i0[4];
  double t[4];
  for (int k = 0; k < 4; ++k) {
    const double* ax = tb.ax[k];
    const int nn = tb.dims[k];
    double xv = x[k];
    const double a0 = ax[0], a1 = ax[nn - 1];
    if (!(xv >= a0)) { xv = a0; th.oob = 1; }
    if (!(xv <= a1)) { xv = a1; th.oob = 1; }
    const int i = axis_cell(ax, nn, xv);
    i0[k] = i;
    const double lo = ax[i], hi = ax[i + 1];
    t[k] = (xv - lo) / (hi - lo);
  }
  double out[TB_STRIDE];
  for (int c = 0; c < TB_STRIDE; ++c) out[c] = 0.0;
  /* 16 nodes; the two nodes along the innermost axis are adjacent in memory (2 * TB_STRIDE doubles, 16-byte loads) */
  for (int b0 = 0; b0 < 2; ++b0)
    for (int b1 = 0; b1 < 2; ++b1)
      for (int b2 = 0; b2 < 2; ++b2) {
        const double w0 = b0 ? t[0] : 1.0 - t[0];
        const double w1 = b1 ? t[1] : 1.0 - t[1];
        const double w2 = b2 ? t[2] : 1.0 - t[2];
        const double w012 = (w0 * w1) * w2;
        const int64_t node = (((int64_t)(i0[0] + b0) * tb.dims[1] + (i0[1] + b1)) * tb.dims[2] + (i0[2] + b2)) * tb.dims[3] + i0[3];
        const double2* __restrict__ p0 = reinterpret_cast<const double2*>(tb.data + node * TB_STRIDE);
        const double wl = w012 * (1.0 - t[3]), wh = w012 * t[3];
#if CCAKE_V4
        static_assert(TB_STRIDE % 4 == 0, "32-byte loads");
#pragma unroll
        for (int u = 0; u < TB_STRIDE / 4; ++u) {
          double lo[4], hi[4];
          ldg_nc_v4(reinterpret_cast<const double*>(p0) + 4 * u, lo[0], lo[1], lo[2], lo[3]);
          ldg_nc_v4(reinterpret_cast<const double*>(p0) + TB_STRIDE + 4 * u, hi[0], hi[1], hi[2], hi[3]);
#pragma unroll
          for (int c = 0; c < 4; ++c) { out[4 * u + c] += wl * lo[c]; out[4 * u + c] += wh * hi[c]; }
        }
#else
#pragma unroll
        for (int u = 0; u < TB_STRIDE / 2; ++u) {
          const double2 lo = __ldg(p0 + u), hi = __ldg(p0 + TB_STRIDE / 2 + u);
          out[2 * u] += wl * lo.x; out[2 * u] += wh * hi.x;
          out[2 * u + 1] += wl * lo.y; out[2 * u + 1] += wh * hi.y;
        }
#endif
      }
  th.T = out[CCAKE_COL_T];
  for (int q = 0; q < NQ; ++q) { th.mu[q] = out[CCAKE_COL_MUB + q]; th.wq[q] = out[CCAKE_COL_WB + q]; }
  th.p = out[CCAKE_COL_P]; th.cs2 = out[CCAKE_COL_CS2]; th.e = out[CCAKE_COL_E]; th.ws = out[CCAKE_COL_WS];
  return th;
}

/* single real root of 4 c4 mu^3 + 2 c2 T^2 mu = n: depressed cubic chi^3 + a1 chi - a2 = 0, closed form of
   Eq. A.13-A.14 (:2146-2152) */
__device__ inline double mu_of_T(const KParams& kp, double T, double n) {
  if (n == 0.0) return 0.0;
  if (kp.c4 == 0.0) return n / (2.0 * kp.c2 * T * T);
  const double sgn = (n < 0.0) ? -1.0 : 1.0;
  const double a1 = kp.c2 * T * T / (2.0 * kp.c4);
  const double a2 = fabs(n) / (4.0 * kp.c4);
  const double delta = sqrt(12.0 * a1 * a1 * a1 + 81.0 * a2 * a2) + 9.0 * a2;
  const double d13 = cbrt(delta);
  const double chi = (1.2599210498948732 * d13 * d13 - 2.0 * 1.4422495703074083 * a1) / (3.3019272488946263 * d13);
  return sgn * chi;
}

/* (s, n_q) -> (T, mu_q): cubic for mu_q(T), monotone 1-D solve in T by bisection (analogue of Eq. A.15 with s as
   the key, :587); then p, e = 3p, c_s^2 = 1/3 and dw/ds, dw/dn_q from the Hessian of p (Eq. A.8-A.10) */
__device__ inline ThermoOut eos_closed_form(const KParams& kp, double s, const double n[NQ]) {
  ThermoOut th;
  th.oob = 0;
  double T;
  const double Tmax = cbrt(s / (4.0 * kp.c0));
  if (n[0] == 0.0 && n[1] == 0.0 && n[2] == 0.0) {
    T = Tmax;
  } else {
    double lo = 0.0, hi = Tmax;
    for (int it = 0; it < 200; ++it) {
      const double mid = 0.5 * (lo + hi);
      if (mid <= lo || mid >= hi) break;
      double m2 = 0.0;
      for (int q = 0; q < NQ; ++q) { const double m = mu_of_T(kp, mid, n[q]); m2 += m * m; }
      const double f = 4.0 * kp.c0 * mid * mid * mid + 2.0 * kp.c2 * mid * m2 - s;
      if (f > 0.0) hi = mid; else lo = mid;
    }
    T = 0.5 * (lo + hi);
  }
  th.T = T;
  double m2 = 0.0, m4 = 0.0;
  for (int q = 0; q < NQ; ++q) {
    const double m = mu_of_T(kp, T, n[q]);
    th.mu[q] = m;
    m2 += m * m;
    m4 += m * m * m * m;
  }
  th.p = kp.c0 * T * T * T * T + kp.c2 * T * T * m2 + kp.c4 * m4;
  th.e = 3.0 * th.p;
  th.cs2 = 1.0 / 3.0;
  /* H = Hessian of p in (T, mu): arrow matrix [[a, b^T], [b, diag(d)]]; z = H^-1 (s, n) by the Schur complement;
     dw/ds = T + z_0, dw/dn_q = mu_q + z_q */
  const double a = 12.0 * kp.c0 * T * T + 2.0 * kp.c2 * m2;
  double b[NQ], d[NQ];
  bool ok = true;
  for (int q = 0; q < NQ; ++q) {
    b[q] = 4.0 * kp.c2 * T * th.mu[q];
    d[q] = 2.0 * kp.c2 * T * T + 12.0 * kp.c4 * th.mu[q] * th.mu[q];
    if (d[q] == 0.0) ok = false;
  }
  if (ok) {
    double schur = a, rhs0 = s;
    for (int q = 0; q < NQ; ++q) { schur -= b[q] * b[q] / d[q]; rhs0 -= b[q] * n[q] / d[q]; }
    const double z0 = rhs0 / schur;
    th.ws = T + z0;
    for (int q = 0; q < NQ; ++q) th.wq[q] = th.mu[q] + (n[q] - b[q] * z0) / d[q];
  } else {               /* c2 = 0 and mu = 0: charges decouple */
    th.ws = T + T / 3.0;
    for (int q = 0; q < NQ; ++q) th.wq[q] = 0.0;
  }
  return th;
}

/* NEXT-1: the offline inversion of the EoS table on the device — one thread per node of the
   (s, B, S, Q) grid; axes 1..3 hold n_q (kind 0) or n_q / s (kind 1).  PAPER.md :576-593, App. A. */
struct InvertArgs {
  int dims[4], kind[4], ncols;
  int col_of[CCAKE_NCOLS_MAX];
  const double* ax[4];
};
__global__ void __launch_bounds__(128)
eos_invert_kernel(KParams kp, InvertArgs a, int64_t nodes, double* __restrict__ data) {
  const int64_t node = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (node >= nodes) return;
  int64_t r = node;
  const int i3 = (int)(r % a.dims[3]); r /= a.dims[3];
  const int i2 = (int)(r % a.dims[2]); r /= a.dims[2];
  const int i1 = (int)(r % a.dims[1]); r /= a.dims[1];
  const int i0 = (int)r;
  const double s = a.ax[0][i0];
  const double y[NQ] = {a.ax[1][i1], a.ax[2][i2], a.ax[3][i3]};
  double n[NQ];
  for (int q = 0; q < NQ; ++q) n[q] = (a.kind[q + 1] == 1) ? y[q] * s : y[q];
  const ThermoOut th = eos_closed_form(kp, s, n);
  double v[CCAKE_NCOLS_MAX];
  v[CCAKE_COL_T] = th.T;
  for (int q = 0; q < NQ; ++q) { v[CCAKE_COL_MUB + q] = th.mu[q]; v[CCAKE_COL_WB + q] = th.wq[q]; }
  v[CCAKE_COL_P] = th.p; v[CCAKE_COL_CS2] = th.cs2; v[CCAKE_COL_E] = th.e; v[CCAKE_COL_WS] = th.ws;
  double* __restrict__ o = data + node * a.ncols;
#pragma unroll
  for (int c = 0; c < CCAKE_NCOLS_MAX; ++c)
    if (a.col_of[c] >= 0) o[a.col_of[c]] = v[c];
}

/* Rest of NEXT-1: the offline inverter on a TABULATED forward EoS (PAPER.md :576-593; DESIGN reading 21) — what the paper
   runs on the host because "root-finding for non-linear functions is not tractable on GPUs" (:585).  One thread per
   node of the (s, B, S, Q) target grid: damped 4-D Newton on the quadrilinear interpolant of the forward table
   (p, s, n_B, n_S, n_Q)(T, mu_B, mu_S, mu_Q); a node the root-finder does not reach takes the backup EoS (:572), the
   closed-form conformal family of the context, and is flagged. */
struct FwdDev {
  int dims[4];
  const double* ax[4];
  const double* data;      /* [node][5] */
};

/* interpolant and its Jacobian by successive 1-D reductions (axis 3 first): v = lo + t (hi - lo); the slope along the
   reduced axis is (hi - lo) / width, slopes along axes reduced earlier are blended like the values.
   Y[0..4] = p, s, n_q; J[i][k] = d Y[1 + i] / d X_k. */
__device__ inline void fwd_eval(const FwdDev& f, const double X[4], double Y[5], double J[4][4]) {
  int i0[4];
  double t[4], iw[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const double* ax = f.ax[k];
    const int nn = f.dims[k];
    double xv = X[k];
    if (!(xv >= ax[0])) xv = ax[0];
    if (!(xv <= ax[nn - 1])) xv = ax[nn - 1];
    const int i = axis_cell(ax, nn, xv);
    i0[k] = i;
    const double lo = ax[i], w = ax[i + 1] - lo;
    t[k] = (xv - lo) / w;
    iw[k] = 1.0 / w;
  }
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    /* level 3 -> 8 values + slope along axis 3 */
    double v3[8], d3[8];
#pragma unroll
    for (int b = 0; b < 8; ++b) {
      const int64_t node = (((int64_t)(i0[0] + (b >> 2)) * f.dims[1] + (i0[1] + ((b >> 1) & 1))) * f.dims[2] + (i0[2] + (b & 1))) * f.dims[3] + i0[3];
      const double lo = __ldg(f.data + node * 5 + c), hi = __ldg(f.data + (node + 1) * 5 + c);
      const double df = hi - lo;
      v3[b] = fma(t[3], df, lo);
      d3[b] = df * iw[3];
    }
    double v2[4], d32[4], d2[4];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const double df = v3[2 * b + 1] - v3[2 * b];
      v2[b] = fma(t[2], df, v3[2 * b]);
      d2[b] = df * iw[2];
      d32[b] = fma(t[2], d3[2 * b + 1] - d3[2 * b], d3[2 * b]);
    }
    double v1[2], d31[2], d21[2], d1[2];
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const double df = v2[2 * b + 1] - v2[2 * b];
      v1[b] = fma(t[1], df, v2[2 * b]);
      d1[b] = df * iw[1];
      d21[b] = fma(t[1], d2[2 * b + 1] - d2[2 * b], d2[2 * b]);
      d31[b] = fma(t[1], d32[2 * b + 1] - d32[2 * b], d32[2 * b]);
    }
    const double df = v1[1] - v1[0];
    Y[c] = fma(t[0], df, v1[0]);
    if (c >= 1) {
      J[c - 1][0] = df * iw[0];
      J[c - 1][1] = fma(t[0], d1[1] - d1[0], d1[0]);
      J[c - 1][2] = fma(t[0], d21[1] - d21[0], d21[0]);
      J[c - 1][3] = fma(t[0], d31[1] - d31[0], d31[0]);
    }
  }
}

/* x = A^-1 b (transpose = false) or A^-T b, 4 x 4, elimination with partial pivoting; false if singular */
__device__ inline bool solve4(const double Ain[4][4], const double bin[4], bool transpose, double x[4]) {
  double A[4][5];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
#pragma unroll
    for (int k = 0; k < 4; ++k) A[i][k] = transpose ? Ain[k][i] : Ain[i][k];
    A[i][4] = bin[i];
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    int piv = c;
#pragma unroll
    for (int r = c + 1; r < 4; ++r) if (fabs(A[r][c]) > fabs(A[piv][c])) piv = r;
    if (A[piv][c] == 0.0) return false;
#pragma unroll
    for (int r = c + 1; r < 4; ++r)
      if (r == piv) {
#pragma unroll
        for (int k = 0; k < 5; ++k) { const double tmp = A[c][k]; A[c][k] = A[r][k]; A[r][k] = tmp; }
      }
    const double inv = 1.0 / A[c][c];
#pragma unroll
    for (int r = c + 1; r < 4; ++r) {
      const double fct = A[r][c] * inv;
#pragma unroll
      for (int k = c; k < 5; ++k) A[r][k] = fma(-fct, A[c][k], A[r][k]);
    }
  }
#pragma unroll
  for (int r = 3; r >= 0; --r) {
    double acc = A[r][4];
#pragma unroll
    for (int k = r + 1; k < 4; ++k) acc = fma(-A[r][k], x[k], acc);
    x[r] = acc / A[r][r];
  }
  return true;
}

__device__ inline ThermoOut eos_invert_forward(const KParams& kp, const FwdDev& f, double s, const double n[NQ], int& flag) {
  const double Ys[4] = {s, n[0], n[1], n[2]};
  const double inv_s = 1.0 / s;
  double X[4], Y[5], J[4][4];
  auto clampX = [&](double* x) {
#pragma unroll
    for (int k = 0; k < 4; ++k) x[k] = fmin(fmax(x[k], f.ax[k][0]), f.ax[k][f.dims[k] - 1]);
  };
  auto res2 = [&](const double* y) {
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i) { const double d = (y[1 + i] - Ys[i]) * inv_s; r = fma(d, d, r); }
    return r;
  };
  auto rmax = [&](const double* y) {
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i) r = fmax(r, fabs(y[1 + i] - Ys[i]));
    return r;
  };
  X[0] = X[1] = X[2] = X[3] = 0.0;
  clampX(X);
  {
    double lo = f.ax[0][0], hi = f.ax[0][f.dims[0] - 1];
    for (int it = 0; it < 60; ++it) {
      X[0] = 0.5 * (lo + hi);
      fwd_eval(f, X, Y, J);
      if (Y[1] > s) hi = X[0]; else lo = X[0];
    }
    X[0] = 0.5 * (lo + hi);
  }
  fwd_eval(f, X, Y, J);
  bool ok = false;
  const double tol = 1e-13 * s;
  for (int it = 0; it < 40; ++it) {
    if (rmax(Y) <= tol) { ok = true; break; }
    double rhs[4], d[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) rhs[i] = -(Y[1 + i] - Ys[i]);
    if (!solve4(J, rhs, false, d)) break;
    const double r0 = res2(Y);
    double lam = 1.0;
    bool acc = false;
    for (int hv = 0; hv <= 12; ++hv) {
      double Xn[4], Yn[5], Jn[4][4];
#pragma unroll
      for (int k = 0; k < 4; ++k) Xn[k] = X[k] + lam * d[k];       /* no contraction: as the oracle steps */
      clampX(Xn);
      fwd_eval(f, Xn, Yn, Jn);
      if (res2(Yn) < r0) {
#pragma unroll
        for (int k = 0; k < 4; ++k) X[k] = Xn[k];
#pragma unroll
        for (int c = 0; c < 5; ++c) Y[c] = Yn[c];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int k = 0; k < 4; ++k) J[i][k] = Jn[i][k];
        acc = true;
        break;
      }
      lam *= 0.5;
    }
    if (!acc) break;
  }
  if (!ok) ok = rmax(Y) <= tol;
  double z[4], v[4];
  if (ok) ok = solve4(J, Ys, true, z);
  if (ok) ok = solve4(J, Ys, false, v);
  if (!ok) {
    flag = 1;
    return eos_closed_form(kp, s, n);
  }
  flag = 0;
  ThermoOut th;
  th.oob = 0;
  th.T = X[0];
  for (int q = 0; q < NQ; ++q) { th.mu[q] = X[1 + q]; th.wq[q] = X[1 + q] + z[1 + q]; }
  th.p = Y[0];
  th.e = X[0] * s - Y[0] + (X[1] * n[0] + X[2] * n[1] + X[3] * n[2]);
  th.ws = X[0] + z[0];
  double num = 0.0, den = 0.0;
#pragma unroll
  for (int i = 0; i < 4; ++i) { num += Ys[i] * v[i]; den += X[i] * Ys[i]; }
  th.cs2 = num / den;
  return th;
}

__global__ void __launch_bounds__(128)
eos_invert_fwd_kernel(KParams kp, InvertArgs a, FwdDev f, int64_t nodes, double* __restrict__ data, int* __restrict__ flags,
                      unsigned long long* __restrict__ n_backup) {
  const int64_t node = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (node >= nodes) return;
  int64_t r = node;
  const int i3 = (int)(r % a.dims[3]); r /= a.dims[3];
  const int i2 = (int)(r % a.dims[2]); r /= a.dims[2];
  const int i1 = (int)(r % a.dims[1]); r /= a.dims[1];
  const int i0 = (int)r;
  const double s = a.ax[0][i0];
  const double y[NQ] = {a.ax[1][i1], a.ax[2][i2], a.ax[3][i3]};
  double n[NQ];
  for (int q = 0; q < NQ; ++q) n[q] = (a.kind[q + 1] == 1) ? y[q] * s : y[q];
  int flag = 0;
  const ThermoOut th = eos_invert_forward(kp, f, s, n, flag);
  if (flags) flags[node] = flag;
  if (flag) atomicAdd(n_backup, 1ULL);
  double v[CCAKE_NCOLS_MAX];
  v[CCAKE_COL_T] = th.T;
  for (int q = 0; q < NQ; ++q) { v[CCAKE_COL_MUB + q] = th.mu[q]; v[CCAKE_COL_WB + q] = th.wq[q]; }
  v[CCAKE_COL_P] = th.p; v[CCAKE_COL_CS2] = th.cs2; v[CCAKE_COL_E] = th.e; v[CCAKE_COL_WS] = th.ws;
  double* __restrict__ o = data + node * a.ncols;
#pragma unroll
  for (int c = 0; c < CCAKE_NCOLS_MAX; ++c)
    if (a.col_of[c] >= 0) o[a.col_of[c]] = v[c];
}

/* dissipative tensors of one particle: evolved spatial components from the store, time components from
   u_mu pi^{mu nu} = 0 and u_mu J^mu = 0 (never evolved; DESIGN reading 13) */
struct Dissip { double pit[4][4], Jt[NQ][4], bulkt; };

template <int D>
__device__ __forceinline__ void load_dissip(const KParams& kp, const Geom& gm, const double* Y, int64_t npad,
                                            int64_t a, const double u[4], Dissip& ds) {
  const double gam = u[0];
  const double G[4] = {0.0, 1.0, 1.0, gm.G3};
#pragma unroll
  for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) ds.pit[m][n] = 0.0;
#pragma unroll
  for (int q = 0; q < NQ; ++q) for (int m = 0; m < 4; ++m) ds.Jt[q][m] = 0.0;
  ds.bulkt = kp.bulk ? Y[CCAKE_BULK * npad + a] : 0.0;
  if (kp.shear) {
    ds.pit[1][1] = Y[CCAKE_PI11 * npad + a];
    ds.pit[1][2] = ds.pit[2][1] = Y[CCAKE_PI12 * npad + a];
    ds.pit[2][2] = Y[CCAKE_PI22 * npad + a];
    ds.pit[3][3] = Y[CCAKE_PI33 * npad + a];
    if (D == 3) {
      ds.pit[1][3] = ds.pit[3][1] = Y[CCAKE_PI13 * npad + a];
      ds.pit[2][3] = ds.pit[3][2] = Y[CCAKE_PI23 * npad + a];
    }
#pragma unroll
    for (int i = 1; i <= 3; ++i) {
      double acc = 0.0;
#pragma unroll
      for (int j = 1; j <= 3; ++j) acc += G[j] * u[j] * ds.pit[j][i];
      ds.pit[0][i] = ds.pit[i][0] = acc / gam;
    }
    double acc = 0.0;
#pragma unroll
    for (int j = 1; j <= 3; ++j) acc += G[j] * u[j] * ds.pit[j][0];
    ds.pit[0][0] = acc / gam;
  }
  if (kp.diff) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
#pragma unroll
      for (int i = 1; i <= D; ++i) ds.Jt[q][i] = Y[(CCAKE_JB1 + 3 * q + (i - 1)) * npad + a];
      double acc = 0.0;
#pragma unroll
      for (int j = 1; j <= 3; ++j) acc += G[j] * u[j] * ds.Jt[q][j];
      ds.Jt[q][0] = acc / gam;
    }
  }
}

__device__ inline void load_u(const KParams& kp, const Geom& gm, const double* Y, int64_t npad, int64_t a,
                              double u[4]) {
  u[1] = Y[CCAKE_U1 * npad + a];
  u[2] = Y[CCAKE_U2 * npad + a];
  u[3] = (kp.D == 3) ? Y[CCAKE_U3 * npad + a] : 0.0;
  u[0] = sqrt(1.0 + u[1] * u[1] + u[2] * u[2] + gm.G3 * u[3] * u[3]);
}

/* TD, TV, TF: dimension, shear, diffusion as template constants, so that the element array of the gradient record is indexed
   at compile time and lives in registers (with run-time indices it sat in local memory: 656 bytes of stack per thread).
   6 resident blocks per SM: 0.97 -> 0.85 ms per substep on C4 (4: 0.91, 8: 0.87). */
#ifndef CCAKE_THERMO_MINB
#define CCAKE_THERMO_MINB 6
#endif
#ifndef CCAKE_THERMO_AX_SMEM
#define CCAKE_THERMO_AX_SMEM 512        /* doubles; 0 = axes read from global memory */
#endif
template <int TD, bool TV, bool TF>
__global__ void __launch_bounds__(128, CCAKE_THERMO_MINB)
thermo_kernel(int64_t n, KParams kp, const double* __restrict__ x0_dev, double x0_off, TableDev tb, const double* __restrict__ Y,
              int64_t npad, Sorted so, Status* __restrict__ status, int on_step, const uint32_t* __restrict__ orig, int64_t n_own) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
#if CCAKE_THERMO_AX_SMEM
  /* the table axes (one array, TableDev) go to shared memory: the per-axis binary searches are ~22 dependent loads per
     particle at lane-divergent indices */
  __shared__ double s_ax[CCAKE_THERMO_AX_SMEM];
  if (kp.eos_kind == 1) {
    const int nax = tb.dims[0] + tb.dims[1] + tb.dims[2] + tb.dims[3];
    if (nax <= CCAKE_THERMO_AX_SMEM) {
      const double* __restrict__ ax0 = tb.ax[0];
      for (int j = threadIdx.x; j < nax; j += blockDim.x) s_ax[j] = ax0[j];
      __syncthreads();
      int off = 0;
      for (int k = 0; k < 4; ++k) { tb.ax[k] = s_ax + off; off += tb.dims[k]; }
    }
  }
#endif
  if (i >= n) return;
  const Geom gm = make_geom(kp.coords, *x0_dev + x0_off);      /* the time lives on the device: a captured step replays */
  constexpr int D = TD;
  const int64_t a = so.perm[i];
  double u[4];
  load_u(kp, gm, Y, npad, a, u);
  const double gam = u[0];
  const double lab = gam * gm.sqrtg;
  const double sst = so.sigma_star[i];
  const double sig = sst / lab, s = so.s_star[i] / lab;
  double nq[NQ];
  for (int q = 0; q < NQ; ++q) nq[q] = so.rho_star[q][i] / lab;
  const ThermoOut th = (kp.eos_kind == 0) ? eos_closed_form(kp, s, nq) : eos_table_lookup(tb, s, nq);
  if (th.oob && (int64_t)orig[a] < n_own) {   /* clamped to the table (ghosts of a slab context, whose sums are incomplete, do
                                                  not count): latest pass, and all substeps of steps since the load */
    atomicAdd(&status->n_oob, 1ULL);
    if (on_step) atomicAdd(&status->n_oob_total, 1ULL);
  }
  so.gamma[i] = gam; so.sigma[i] = sig; so.s[i] = s;
  so.T[i] = th.T; so.p[i] = th.p; so.e[i] = th.e; so.cs2[i] = th.cs2; so.ws[i] = th.ws;
  for (int q = 0; q < NQ; ++q) {
    so.n[q][i] = nq[q]; so.mu[q][i] = th.mu[q]; so.wq[q][i] = th.wq[q];
  }
  Dissip ds;
  load_dissip<D>(kp, gm, Y, npad, a, u, ds);
  const double sst2 = sst * sst;
  const double glo[4] = {1.0, -1.0, -1.0, -gm.G3};
  /* AoS payload record of the gradient pass (pair_mma.cuh): the elements m, m P, m u[D], m v[D],
     m B[D*D], m K[3*D], m alpha[3] stored per MMA column — the pair pass multiplies a column of b by the pair weight
     without m_b */
  constexpr GLayout L = make_glayout(TD, TV, TF);
  double el[32];
#pragma unroll
  for (int k = 0; k < 32; ++k) el[k] = 0.0;
  const double mb = Y[CCAKE_MASS * npad + a];
  el[L.M] = mb;
  el[L.P] = mb * ((th.p + ds.bulkt * sig) / sst2);
#pragma unroll
  for (int j = 1; j <= D; ++j) { el[L.U + j - 1] = mb * u[j]; el[L.V + j - 1] = mb * (u[j] / gam); }
  if (TV)
#pragma unroll
    for (int j = 1; j <= D; ++j)
#pragma unroll
      for (int k = 1; k <= D; ++k) {
        const double pi_j_k = sig * ds.pit[j][k] * glo[k];
        const double pi_0_k = sig * ds.pit[0][k] * glo[k];
        el[L.B + (j - 1) * D + (k - 1)] = mb * ((pi_j_k - (u[j] / gam) * pi_0_k) / sst2);
      }
  if (TF) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      el[L.AL + q] = mb * (th.mu[q] / th.T);
#pragma unroll
      for (int j = 1; j <= D; ++j)
        el[L.K + q * D + (j - 1)] = mb * ((sig * ds.Jt[q][j] - (u[j] / gam) * sig * ds.Jt[q][0]) / sst2);
    }
  }
  double* __restrict__ rg = so.rec_g + i * GREC_D;
  const double xyz[3] = {so.x[0][i], so.x[1][i], so.x[2][i]};
  write_grad_record<TD, TV, TF>(rg, el, xyz);                /* the position goes into the free slots of block 7 */
}

}  // namespace ccake
